// A5: interaction-partner search.
//
// The paper walks the tree once per particle, one thread each, descending while the particle lies
// within s/2 + h of a cell (eq. 69) and testing "distance < smoothing length" at the leaves.
// Here one WARP owns 32 particles that are consecutive in Morton order.  The warp walks the tree
// once for the group's bounding box grown by the reach (lanes test 2^D children of several nodes
// in parallel against the nodes' tight bounding boxes and hmax), collects candidate particles in
// shared memory, stages 32 candidates at a time (coalesced loads), and every lane applies the
// exact membership test of the paper to its own particle:
//     r^2 = (dx*dx + dy*dy) + dz*dz  <  H*H,   H = h_a, or (h_a + h_b)/2 with variable h (eq. 72)
// with every operation rounded separately, so the sets equal the oracle's bit for bit.
// Lists are written group-transposed, nb[(group*cap + k)*32 + lane], so that the pair-sum kernel
// reads them fully coalesced.
#include "sph_internal.cuh"

#define NB_WARPS 4
#define NB_STACK 1024

template <int D, bool VARH, bool COUNT_ONLY>
__global__ void __launch_bounds__(NB_WARPS * 32) k_neigh(Dev d) {
    constexpr int NC = 1 << D;
    __shared__ int s_stack[NB_WARPS][NB_STACK];
    __shared__ int s_cand[NB_WARPS][64];
    __shared__ double s_c[NB_WARPS][4][32];
    __shared__ int s_ci[NB_WARPS][32];

    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = blockIdx.x * NB_WARPS + w;
    const int n = d.n;
    if (g * 32 >= n) return;
    const int i = g * 32 + lane;
    const bool valid = i < n;
    const int ii = valid ? i : n - 1;
    const unsigned FULL = 0xffffffffu, lt = (1u << lane) - 1u;

    const double xi = d.sx[0][ii], yi = d.sx[1][ii], zi = (D == 3) ? d.sx[2][ii] : 0.0;
    const double Hi = d.sh[ii];
    const double Hi2 = __dmul_rn(Hi, Hi);
    double gmin[3] = {xi, yi, zi}, gmax[3] = {xi, yi, zi}, Hg = Hi;
    for (int o = 16; o > 0; o >>= 1) {
        for (int a = 0; a < D; ++a) {
            gmin[a] = fmin(gmin[a], __shfl_xor_sync(FULL, gmin[a], o));
            gmax[a] = fmax(gmax[a], __shfl_xor_sync(FULL, gmax[a], o));
        }
        Hg = fmax(Hg, __shfl_xor_sync(FULL, Hg, o));
    }

    int cnt = 0, own = 0, top = 0, ncand = 0;
    int *stack = s_stack[w], *cand = s_cand[w];
    int *nbw = d.nb + (size_t)g * d.cap * 32 + lane;

    auto flush = [&](int take) {
        const int cj = (lane < take) ? cand[lane] : -1;
        if (cj >= 0) {
            s_c[w][0][lane] = d.sx[0][cj];
            s_c[w][1][lane] = d.sx[1][cj];
            s_c[w][2][lane] = (D == 3) ? d.sx[2][cj] : 0.0;
            s_c[w][3][lane] = d.sh[cj];
            s_ci[w][lane] = cj;
        }
        __syncwarp();
        for (int j = 0; j < take; ++j) {
            const int b = s_ci[w][j];
            const double dx = __dsub_rn(xi, s_c[w][0][j]);
            const double dy = __dsub_rn(yi, s_c[w][1][j]);
            const double dz = (D == 3) ? __dsub_rn(zi, s_c[w][2][j]) : 0.0;
            const double r2 = sph_r2_exact(dx, dy, dz, D);
            if (COUNT_ONLY) {
                if (valid && b != i && r2 < Hi2) ++own;
            } else {
                double H2 = Hi2;
                if (VARH) {
                    const double Hab = __dmul_rn(0.5, __dadd_rn(Hi, s_c[w][3][j]));
                    H2 = __dmul_rn(Hab, Hab);
                }
                if (valid && b != i && r2 < H2) {
                    if (cnt < d.cap) nbw[(size_t)cnt * 32] = b;
                    ++cnt;
                }
            }
        }
        __syncwarp();
        // keep what is left
        const int rest = ncand - take;
        int keep = (lane < rest) ? cand[take + lane] : 0;
        __syncwarp();
        if (lane < rest) cand[lane] = keep;
        ncand = rest;
        __syncwarp();
    };

    const int nn = d.status->n_nodes;
    if (nn == 0) {
        // no internal node (n == 1 or all keys equal): every particle is a candidate
        for (int p0 = 0; p0 < n; p0 += 32) {
            if (p0 + lane < n) cand[lane] = p0 + lane;
            ncand = min(32, n - p0);
            __syncwarp();
            flush(ncand);
        }
    } else {
        if (lane == 0) stack[0] = 0;
        top = 1;
        __syncwarp();
        bool fail = false;
        while (top > 0) {
            const int npop = min(top, 32 / NC);
            const int j = lane / NC, c = lane % NC;
            const int node = (j < npop) ? stack[top - 1 - j] : -1;
            __syncwarp();
            top -= npop;
            int push = -1, c0 = 0, c1 = 0;
            if (node >= 0) {
                const int code = d.child[(size_t)node * NC + c];
                if (code >= 0) {
                    double reach = (VARH && !COUNT_ONLY) ? 0.5 * (Hg + d.nhmax[code]) : Hg;
                    reach *= (1.0 + 1e-9);
                    bool ov = true;
                    for (int a = 0; a < D; ++a)
                        ov = ov && (__dsub_rn(d.nbmin[a][code], gmax[a]) <= reach) &&
                             (__dsub_rn(gmin[a], d.nbmax[a][code]) <= reach);
                    if (ov) push = code;
                } else if (code == -2) {
                    c0 = d.child_lo[(size_t)node * (NC + 1) + c];
                    c1 = d.child_lo[(size_t)node * (NC + 1) + c + 1];
                    if (c1 - c0 == 1) {
                        double reach = (VARH && !COUNT_ONLY) ? 0.5 * (Hg + d.sh[c0]) : Hg;
                        reach *= (1.0 + 1e-9);
                        bool in = true;
                        for (int a = 0; a < D; ++a) {
                            const double xb = d.sx[a][c0];
                            in = in && (__dsub_rn(xb, gmax[a]) <= reach) && (__dsub_rn(gmin[a], xb) <= reach);
                        }
                        if (!in) c1 = c0;
                    }
                }
            }
            const unsigned pm = __ballot_sync(FULL, push >= 0);
            if (top + __popc(pm) > NB_STACK) { fail = true; break; }
            if (push >= 0) stack[top + __popc(pm & lt)] = push;
            top += __popc(pm);
            const unsigned sm_ = __ballot_sync(FULL, c1 - c0 == 1);
            if (c1 - c0 == 1) cand[ncand + __popc(sm_ & lt)] = c0;
            ncand += __popc(sm_);
            __syncwarp();
            while (ncand >= 32) flush(32);
            unsigned mm = __ballot_sync(FULL, c1 - c0 > 1);
            while (mm) {   // leaves holding several particles with one key (degenerate, rare)
                const int src = __ffs(mm) - 1;
                mm &= mm - 1;
                const int r0 = __shfl_sync(FULL, c0, src), r1 = __shfl_sync(FULL, c1, src);
                for (int p = r0; p < r1; p += 32) {
                    if (p + lane < r1) cand[ncand + lane] = p + lane;
                    ncand += min(32, r1 - p);
                    __syncwarp();
                    while (ncand >= 32) flush(32);
                }
            }
        }
        if (fail && lane == 0) atomicExch(&d.status->err_stack, 1);
        if (ncand > 0) flush(ncand);
    }

    if (COUNT_ONLY) {
        if (valid) d.own_cnt[i] = own;
    } else {
        if (valid) d.nb_cnt[i] = min(cnt, d.cap);
        int mx = cnt;
        for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(FULL, mx, o));
        int tot = valid ? min(cnt, d.cap) : 0;
        for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(FULL, tot, o);
        if (lane == 0) {
            if (mx > d.cap) atomicExch(&d.status->err_nb_overflow, 1);
            atomicMax(&d.status->nb_max, mx);
            atomicAdd(&d.status->n_pairs, (u64)tot);
        }
    }
}

// eq. 73: h_new = h * 1/2 * (1 + (n_des / n_a)^(1/D)), n_a >= 1 (reading U5)
__global__ void k_h_update(Dev d) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    double ratio = (double)d.n_des / (double)max(d.own_cnt[i], 1);
    double root = (d.D == 3) ? cbrt(ratio) : sqrt(ratio);
    d.sh[i] = d.sh[i] * 0.5 * (1.0 + root);
}

__global__ void k_writeback_h(Dev d) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    d.h[d.perm[i]] = d.sh[i];
}

// hmax of every node must follow the new h: recompute the moments pass cheaply (hmax only)
__global__ void k_hmax(Dev d, int level) {
    const int nd = blockIdx.x * blockDim.x + threadIdx.x;
    if (nd >= d.status->n_nodes) return;
    if (d.nlevel[nd] != level) return;
    const int NC = 1 << d.D;
    const int *cl = d.child_lo + (size_t)nd * (NC + 1);
    const int *ch = d.child + (size_t)nd * NC;
    double hmax = 0.0;
    for (int c = 0; c < NC; ++c) {
        const int code = ch[c];
        if (code >= 0) hmax = fmax(hmax, d.nhmax[code]);
        else if (code == -2) for (int p = cl[c]; p < cl[c + 1]; ++p) hmax = fmax(hmax, d.sh[p]);
    }
    d.nhmax[nd] = hmax;
}

template <int D>
static void launch_neigh(sph_ctx *ctx, bool varh, bool count_only) {
    Dev &d = ctx->d;
    const int groups = sph_ceil_div(d.n, 32);
    const int blocks = sph_ceil_div(groups, NB_WARPS);
    if (count_only) k_neigh<D, false, true><<<blocks, NB_WARPS * 32, 0, ctx->stream>>>(d);
    else if (varh) k_neigh<D, true, false><<<blocks, NB_WARPS * 32, 0, ctx->stream>>>(d);
    else k_neigh<D, false, false><<<blocks, NB_WARPS * 32, 0, ctx->stream>>>(d);
    ctx->launches += 1;
}

void sph_stage_writeback_h(sph_ctx *ctx) {
    k_writeback_h<<<sph_ceil_div(ctx->d.n, 256), 256, 0, ctx->stream>>>(ctx->d);
    ctx->launches += 1;
}

void sph_stage_neigh(sph_ctx *ctx) {
    Dev &d = ctx->d;
    StageTimer tm(ctx, SPH_T_NEIGHBOURS);
    const bool varh = (d.flags & SPH_F_VARIABLE_H) != 0;
    if (varh && ctx->cfg.h_iters > 0) {
        for (int it = 0; it < ctx->cfg.h_iters; ++it) {
            if (d.D == 3) launch_neigh<3>(ctx, varh, true); else launch_neigh<2>(ctx, varh, true);
            k_h_update<<<sph_ceil_div(d.n, 256), 256, 0, ctx->stream>>>(d);
            ctx->launches += 1;
            for (int lvl = d.L - 1; lvl >= 0; --lvl) {
                k_hmax<<<sph_ceil_div(d.n, 128), 128, 0, ctx->stream>>>(d, lvl);
                ctx->launches += 1;
            }
        }
        sph_stage_writeback_h(ctx);
    }
    if (d.D == 3) launch_neigh<3>(ctx, varh, false); else launch_neigh<2>(ctx, varh, false);
}
