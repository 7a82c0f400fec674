// A5: interaction-partner search.
//
// The paper walks the tree once per particle, one thread each, descending while the particle lies
// within s/2 + h of a cell (eq. 69) and testing "distance < smoothing length" at the leaves.
// Here one WARP owns 32 particles that are consecutive in Morton order and walks ONE stream for
// all of them, but every lane prunes for its own particle:
//
//   * The search stream (built by sph_build_search_items below) holds, in depth-first pre-order,
//     the octree cells with more than SPH_BUCKET particles and BUCKETS of <= SPH_BUCKET particles
//     that are consecutive in Morton order (runs of small sibling cells / leaves).  Every record
//     carries the bounding box and the largest h of the particles below it, rounded OUTWARD to
//     FP32: pruning runs on the FP32 pipe with directed rounding (a box that holds a partner is
//     never cut), the FP64 pipe is kept for the exact membership tests.
//   * Every lane keeps the index of the next record IT has to look at: a cell whose box is out
//     of the lane's reach is skipped (next = skip index), otherwise entered (next = cur + 1).
//     The warp visits min over lanes(next) (one redux.sync), so the records a warp touches are
//     the union of 32 single-particle walks -- bounded even where the Morton curve jumps and a
//     group's bounding box spans half a body (profiles/r1a_c5_first_path.md: that tail cost 96 %).
//   * A bucket within reach of any lane is staged through shared memory with one coalesced load
//     per coordinate, and every lane applies the exact membership test of the paper to its own
//     particle:   r^2 = (dx*dx + dy*dy) + dz*dz  <  H*H,   H = h_a, or (h_a + h_b)/2 with variable
//     h (eq. 72), every operation rounded separately, so the sets equal the oracle's bit for bit.
// Lists are written group-transposed, nb[(group*cap + k)*32 + lane], so that the pair-sum kernel
// reads them fully coalesced; within a list partners come in ascending Morton order.
#include "sph_internal.cuh"

#define NB_WARPS 2

// ------------------------------------------------------------------------------------------
// search stream layout
// ------------------------------------------------------------------------------------------
// bmark[i]: low word 1 = a bucket starts at sorted particle i; high word = number of big cells
// whose range starts at i.
__global__ void k_mark_buckets(Dev d) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int nn = d.status->n_nodes, n = d.n;
    if (nn == 0) {   // n == 1 or all keys equal: plain runs of SPH_BUCKET
        if (t < n && (t % SPH_BUCKET) == 0) d.bmark[t] = 1ull;
        return;
    }
    if (t >= nn) return;
    const int NC = 1 << d.D;
    const int lo = d.nlo[t], hi = d.nhi_s[t];
    if (hi - lo <= SPH_BUCKET) {
        if (t == 0) d.bmark[0] = 1ull;          // the whole set is one bucket
        return;
    }
    atomicAdd(&d.bmark[lo], 1ull << 32);
    const int *cl = d.child_lo + (size_t)t * (NC + 1);
    const int *ch = d.child + (size_t)t * NC;
    bool open = false;
    int run = 0;
    for (int c = 0; c < NC; ++c) {
        const int r0 = cl[c], r1 = cl[c + 1], sz = r1 - r0;
        if (sz == 0) continue;
        if (sz > SPH_BUCKET) {
            // a big child cell lays itself out; a leaf of > SPH_BUCKET coincident particles is cut into runs
            if (ch[c] == -2) for (int p = r0; p < r1; p += SPH_BUCKET) atomicAdd(&d.bmark[p], 1ull);
            open = false;
            continue;
        }
        if (open && run + sz <= SPH_BUCKET) run += sz;           // merge small siblings
        else { atomicAdd(&d.bmark[r0], 1ull); open = true; run = sz; }
    }
}

__global__ void k_emit_items(Dev d) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int n = d.n, nn = d.status->n_nodes;
    const int D = d.D;
    if (t == 0) {
        const u64 tot = d.bscan[n];
        d.status->n_items = (int)(tot & 0xffffffffu) + (int)(tot >> 32);
    }
    {   // buckets: the warp handles the bucket starts among its 32 positions one after the other,
        // all lanes loading the (<= SPH_BUCKET) members together (one thread per bucket with a serial loop
        // cost 0.5 ms on C5: profiles/r1d_c5.md)
        const unsigned FULL = 0xffffffffu;
        const int lane = threadIdx.x & 31, base = t - lane;
        const u64 mk = (t < n) ? d.bmark[t] : 0ull;
        unsigned starts = __ballot_sync(FULL, (mk & 1ull) != 0ull);
        while (starts) {
            const int j = __ffs(starts) - 1;
            starts &= starts - 1;
            const int s0 = base + j;
            const int q = s0 + 1 + lane;                       // a bucket has at most SPH_BUCKET <= 32 members
            const bool stop = (q >= n) || ((d.bmark[q] & 1ull) != 0ull);
            const int len = __ffs(__ballot_sync(FULL, stop));  // members: s0 .. s0 + len - 1
            const bool have = lane < len;
            const int p = s0 + (have ? lane : 0);
            double mn[3], mx[3], hm = have ? d.sh[p] : 0.0;
            for (int a = 0; a < 3; ++a) {
                const double x = (a < D) ? d.sx[a][p] : 0.0;
                mn[a] = x; mx[a] = x;
            }
            for (int o = 16; o > 0; o >>= 1) {
                for (int a = 0; a < 3; ++a) {
                    mn[a] = fmin(mn[a], __shfl_xor_sync(FULL, mn[a], o));
                    mx[a] = fmax(mx[a], __shfl_xor_sync(FULL, mx[a], o));
                }
                hm = fmax(hm, __shfl_xor_sync(FULL, hm, o));
            }
            if (lane == 0) {
                const u64 sc = d.bscan[s0], m0 = d.bmark[s0];
                const int pos = (int)(sc & 0xffffffffu) + (int)(sc >> 32) + (int)(m0 >> 32);
                SearchItem it;
                for (int a = 0; a < 3; ++a) { it.bmin[a] = __double2float_rd(mn[a]); it.bmax[a] = __double2float_ru(mx[a]); }
                it.hmax = __double2float_ru(hm); it.pad = 0.f; it.skip = -len; it.lo = s0; it.pad2[0] = it.pad2[1] = 0;
                d.items[pos] = it;
            }
        }
    }
    if (t < nn) {
        const int lo = d.nlo[t], hi = d.nhi_s[t];
        if (hi - lo > SPH_BUCKET) {              // big cell
            int k = 0;
            while (t - 1 - k >= 0 && d.nlo[t - 1 - k] == lo) ++k;     // ancestors sharing lo precede it
            const u64 sl = d.bscan[lo], sh_ = d.bscan[hi];
            SearchItem it;
            for (int a = 0; a < 3; ++a) { it.bmin[a] = __double2float_rd(d.nbmin[a][t]); it.bmax[a] = __double2float_ru(d.nbmax[a][t]); }
            it.hmax = __double2float_ru(d.nhmax[t]); it.pad = 0.f; it.pad2[0] = it.pad2[1] = 0;
            it.skip = (int)(sh_ & 0xffffffffu) + (int)(sh_ >> 32);
            it.lo = lo;
            d.items[(int)(sl & 0xffffffffu) + (int)(sl >> 32) + k] = it;
        }
    }
}

static void emit_items(sph_ctx *ctx) {
    k_emit_items<<<sph_ceil_div(ctx->d.n, 128), 128, 0, ctx->stream>>>(ctx->d);
    ctx->launches += 1;
}

void sph_build_search_items(sph_ctx *ctx) {
    Dev &d = ctx->d;
    cudaMemsetAsync(d.bmark, 0, ((size_t)d.n + 1) * sizeof(u64), ctx->stream);
    k_mark_buckets<<<sph_ceil_div(d.n, 128), 128, 0, ctx->stream>>>(d);
    ctx->launches += 1;
    sph_scan_u64(ctx, d.bmark, d.bscan, (i64)d.n + 1, d.scan_tmp);
    emit_items(ctx);
}

// ------------------------------------------------------------------------------------------
// the walk
// ------------------------------------------------------------------------------------------
template <int D, bool VARH, bool COUNT_ONLY>
__global__ void __launch_bounds__(NB_WARPS * 32) k_neigh(Dev d) {
    __shared__ double s_c[NB_WARPS][4][32];

    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = d.r_lo / 32 + blockIdx.x * NB_WARPS + w;   // groups of the rank's slice [r_lo, r_hi) (all of them on one GPU)
    const int n = d.n;
    if (g * 32 >= d.r_hi) return;
    const int i = g * 32 + lane;
    const bool valid = i < d.r_hi;
    const int ii = valid ? i : n - 1;
    const unsigned FULL = 0xffffffffu;

    const double xi = d.sx[0][ii], yi = d.sx[1][ii], zi = (D == 3) ? d.sx[2][ii] : 0.0;
    const double Hi = d.sh[ii];
    const double Hi2 = __dmul_rn(Hi, Hi);
    constexpr bool VH = VARH && !COUNT_ONLY;   // pair criterion (h_a + h_b)/2, eq. 72
    const float xlo = __double2float_rd(xi), xhi = __double2float_ru(xi), ylo = __double2float_rd(yi), yhi = __double2float_ru(yi);
    const float zlo = __double2float_rd(zi), zhi = __double2float_ru(zi);
    const float Hf = __double2float_ru(Hi) * 1.000001f;      // the pruning test must never cut a true partner

    int cnt = 0;
    int *nbw = d.nb + (size_t)g * d.cap * 32 + lane;
    const int cap = d.cap;
    const int nitems = d.status->n_items;
    const SearchItem *__restrict__ items = d.items;

    int next = valid ? 0 : 0x7fffffff;
    int cur = 0;
    while (cur < nitems) {
        // pruning in FP32 with directed rounding: the boxes are rounded outward, the particle towards
        // the box, the differences down and the reach up, so a box that a partner lies in is never cut
        const float4 *rec = reinterpret_cast<const float4 *>(items + cur);
        const float4 r0 = __ldg(rec), r1 = __ldg(rec + 1);            // bmin xyz bmax x | bmax yz hmax pad
        const int2 sl = __ldg(reinterpret_cast<const int2 *>(rec + 2));
        const int skip = sl.x, lo = sl.y;
        const bool act = (next == cur);
        const float reach = VH ? __fmul_ru(0.5f, __fadd_ru(Hf, r1.z)) * 1.000001f : Hf;
        // squared distance from the particle to the box, a LOWER bound (differences and products rounded down),
        // against reach^2 rounded up: the ball around the particle, not the cube around it (the corners of the
        // cube admit a quarter more boxes)
        const float ex = fmaxf(fmaxf(__fsub_rd(r0.x, xhi), __fsub_rd(xlo, r0.w)), 0.0f);
        const float ey = fmaxf(fmaxf(__fsub_rd(r0.y, yhi), __fsub_rd(ylo, r1.x)), 0.0f);
        float d2 = __fmaf_rd(ey, ey, __fmul_rd(ex, ex));
        if (D == 3) {
            const float ez = fmaxf(fmaxf(__fsub_rd(r0.z, zhi), __fsub_rd(zlo, r1.y)), 0.0f);
            d2 = __fmaf_rd(ez, ez, d2);
        }
        const bool ov = act && (d2 <= __fmul_ru(reach, reach));
        if (skip >= 0) {
            if (act) next = ov ? cur + 1 : skip;
        } else {
            if (act) next = cur + 1;
            if (__any_sync(FULL, ov)) {
                const int m = -skip;
                if (lane < m) {
                    const int p = lo + lane;
                    s_c[w][0][lane] = d.sx[0][p];
                    s_c[w][1][lane] = d.sx[1][p];
                    if (D == 3) s_c[w][2][lane] = d.sx[2][p];
                    if (VARH && !COUNT_ONLY) s_c[w][3][lane] = d.sh[p];
                }
                __syncwarp();
                for (int j = 0; j < m; ++j) {
                    const double dx = __dsub_rn(xi, s_c[w][0][j]);
                    const double dy = __dsub_rn(yi, s_c[w][1][j]);
                    const double dz = (D == 3) ? __dsub_rn(zi, s_c[w][2][j]) : 0.0;
                    const double r2 = sph_r2_exact(dx, dy, dz, D);
                    double H2 = Hi2;
                    if (VARH && !COUNT_ONLY) {
                        const double Hab = __dmul_rn(0.5, __dadd_rn(Hi, s_c[w][3][j]));
                        H2 = __dmul_rn(Hab, Hab);
                    }
                    if (valid && (lo + j != i) && r2 < H2) {
                        if (!COUNT_ONLY && cnt < cap) nbw[(size_t)cnt * 32] = lo + j;
                        ++cnt;
                    }
                }
                __syncwarp();
            }
        }
        cur = __reduce_min_sync(FULL, next);
    }

    if (COUNT_ONLY) {
        if (valid) d.own_cnt[i] = cnt;
    } else {
        if (valid) d.nb_cnt[i] = min(cnt, cap);
        int mx = cnt;
        for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(FULL, mx, o));
        int tot = valid ? min(cnt, cap) : 0;
        for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(FULL, tot, o);
        if (lane == 0) {
            if (mx > cap) atomicExch(&d.status->err_nb_overflow, 1);
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

// With a partition set (sph_set_partition) the walk covers the rank's slice only -- unless every particle's list is
// needed on every rank: the density sum (eq. 28) and the eq.-73 update feed the partners' sums.
static bool lists_replicated(const sph_ctx *ctx) {
    return (ctx->d.flags & SPH_F_DENSITY_SUM) || ((ctx->d.flags & SPH_F_VARIABLE_H) && ctx->cfg.h_iters > 0);
}

template <int D>
static void launch_neigh(sph_ctx *ctx, bool varh, bool count_only) {
    Dev d = ctx->d;
    if (lists_replicated(ctx)) { d.r_lo = 0; d.r_hi = d.n; }
    const int groups = sph_ceil_div(d.r_hi - d.r_lo, 32);
    if (groups == 0) return;
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
    sph_build_search_items(ctx);
    if (varh && ctx->cfg.h_iters > 0) {
        for (int it = 0; it < ctx->cfg.h_iters; ++it) {
            if (d.D == 3) launch_neigh<3>(ctx, varh, true); else launch_neigh<2>(ctx, varh, true);
            k_h_update<<<sph_ceil_div(d.n, 256), 256, 0, ctx->stream>>>(d);
            ctx->launches += 1;
            sph_launch_moments(ctx, 1);      // hmax of every cell follows the new h (the boxes are unchanged)
            emit_items(ctx);                 // refresh hmax of the records
        }
        sph_stage_writeback_h(ctx);
    }
    if (d.D == 3) launch_neigh<3>(ctx, varh, false); else launch_neigh<2>(ctx, varh, false);
}
