// A3 + A4: octree topology from the sorted Morton keys, then pseudo-particles bottom-up.
//
// The tree is the paper's Barnes-Hut octree (cubic cells, 2^D
// sub-cells, one particle per leaf) without the chains of single-child cells its insertion
// creates (reading U14).  An internal node is a cell in which two particles that are
// adjacent in Morton order first separate.  Instead of the paper's lock-based top-down insertion
// every node is found independently from the sorted keys:
//   k_find_nodes : one thread per adjacent pair; binary search for the start of the pair's cell;
//                  the pair that closes the FIRST occupied sub-cell emits the node (lo, level, hi)
//   radix sort   : nodes sorted by (lo, level)  == depth-first (pre-order) numbering
//   k_fill_nodes : child boundaries by binary search in the node's key range; child node ids by
//                  binary search in the sorted node keys
//   k_moments    : ONE launch, threads climb from the deepest cells: mass, centre of mass (monopole
//                  only), tight bounding box and hmax.  Children are
//                  summed in octant order, every operation rounded separately (reading U15), so
//                  that the opening decisions of the gravity walk are reproducible bit for bit.
#include <cuda/atomic>

#include "sph_internal.cuh"

__device__ __forceinline__ int lower_bound_key(const u64 *__restrict__ k, int lo, int hi, u64 v) {
    while (lo < hi) {   // first index in [lo,hi) with k[i] >= v
        int mid = (lo + hi) >> 1;
        if (k[mid] < v) lo = mid + 1; else hi = mid;
    }
    return lo;
}

__global__ void k_find_nodes(Dev d) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int DL = d.D * d.L;
    bool emit = false;
    u64 nk = 0;
    int hi = 0;
    if (i < d.n - 1) {
        const u64 ka = d.keys[i], kb = d.keys[i + 1];
        const u64 x = ka ^ kb;
        if (x != 0) {
            const int common = DL - (64 - __clzll((long long)x));   // common leading bits of the DL-bit keys
            const int lvl = common / d.D;
            const int shift = d.D * (d.L - lvl);                    // low bits below the cell prefix
            int lo;
            u64 cell0;
            if (lvl == 0) { lo = 0; cell0 = 0; }
            else {
                cell0 = (ka >> shift) << shift;
                lo = lower_bound_key(d.keys, 0, i, cell0);
            }
            // representative pair: i closes the first occupied sub-cell of the node
            if ((d.keys[lo] >> (shift - d.D)) == (ka >> (shift - d.D))) {
                emit = true;
                hi = (lvl == 0) ? d.n : lower_bound_key(d.keys, i + 1, d.n, cell0 + (1ull << shift));
                nk = ((u64)lo << 5) | (u64)lvl;                             // level 0..21 in 5 bits
            }
        }
    }
    unsigned m = __ballot_sync(0xffffffffu, emit);
    if (m) {
        int lane = threadIdx.x & 31, base = 0;
        if (lane == __ffs(m) - 1) base = atomicAdd(&d.status->n_nodes, __popc(m));
        base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
        if (emit) {
            int slot = base + __popc(m & ((1u << lane) - 1u));
            d.nkey[0][slot] = nk;
            d.nhi[0][slot] = hi;
        }
    }
}

__global__ void k_fill_nodes(Dev d, const u64 *__restrict__ nkey, const int *__restrict__ nhi) {
    const int nd = blockIdx.x * blockDim.x + threadIdx.x;
    const int nn = d.status->n_nodes;
    if (nd >= nn) return;
    const int D = d.D, NC = 1 << D;
    const u64 nk = nkey[nd];
    const int lo = (int)(nk >> 5), lvl = (int)(nk & 31u), hi = nhi[nd];
    d.nlo[nd] = lo; d.nhi_s[nd] = hi; d.nlevel[nd] = lvl;
    const double s = ldexp(d.root->s0, -lvl);               // eq. 68 (exact)
    d.ns2[nd] = __dmul_rn(s, s);
    {   // skip index: first node whose range starts at or after hi (nodes are sorted by (lo, level))
        const u64 want = (u64)hi << 5;
        int l2 = nd + 1, h2 = nn;
        while (l2 < h2) { int mid = (l2 + h2) >> 1; if (nkey[mid] < want) l2 = mid + 1; else h2 = mid; }
        d.nskip[nd] = l2;
    }
    const int shift = D * (d.L - lvl);
    const u64 prefix = (lvl == 0) ? 0ull : (d.keys[lo] >> shift);
    int b = lo;
    int *cl = d.child_lo + (size_t)nd * (NC + 1);
    int *ch = d.child + (size_t)nd * NC;
    cl[0] = lo;
    int ncc = 0;
    if (nd == 0) d.nparent[0] = -1;
    d.nready[nd] = 0;
    for (int c = 0; c < NC; ++c) {
        int e = (c == NC - 1) ? hi : lower_bound_key(d.keys, b, hi, ((prefix << D) | (u64)(c + 1)) << (shift - D));
        cl[c + 1] = e;
        int code;
        if (e == b) code = -1;
        else if (e - b == 1 || d.keys[b] == d.keys[e - 1]) code = -2;
        else {
            u64 x = d.keys[b] ^ d.keys[e - 1];
            int common = D * d.L - (64 - __clzll((long long)x));
            int clvl = common / D;
            u64 want = ((u64)b << 5) | (u64)clvl;
            int l2 = nd + 1, h2 = nn;                       // children follow their parent in pre-order
            while (l2 < h2) { int mid = (l2 + h2) >> 1; if (nkey[mid] < want) l2 = mid + 1; else h2 = mid; }
            code = l2;
            d.nparent[l2] = nd;
            ++ncc;
        }
        ch[c] = code;
        b = e;
    }
    d.ncc[nd] = ncc;
}

// Pseudo-particle of one cell from its children, children in octant order, every
// operation rounded separately (reading U15).  Child cells are read with ld.global.cg: they were
// written by other threads of the same launch.
__device__ __forceinline__ void cell_moments(const Dev &d, int nd, bool hmax_only) {
    const int D = d.D, NC = 1 << D;
    const int *cl = d.child_lo + (size_t)nd * (NC + 1);
    const int *ch = d.child + (size_t)nd * NC;
    double M = 0.0, S[3] = {0, 0, 0};
    double bmin[3] = {INFINITY, INFINITY, INFINITY}, bmax[3] = {-INFINITY, -INFINITY, -INFINITY}, hmax = 0.0;
    for (int c = 0; c < NC; ++c) {
        const int code = ch[c];
        if (code == -1) continue;
        if (code >= 0) {
            hmax = fmax(hmax, __ldcg(&d.nhmax[code]));
            if (hmax_only) continue;
            const double mc = __ldcg(&d.nmass[code]);
            M = __dadd_rn(M, mc);
            for (int a = 0; a < D; ++a) {
                S[a] = __dadd_rn(S[a], __dmul_rn(mc, __ldcg(&d.ncom[a][code])));
                bmin[a] = fmin(bmin[a], __ldcg(&d.nbmin[a][code]));
                bmax[a] = fmax(bmax[a], __ldcg(&d.nbmax[a][code]));
            }
        } else {
            for (int p = cl[c]; p < cl[c + 1]; ++p) {
                hmax = fmax(hmax, d.sh[p]);
                if (hmax_only) continue;
                const double mp = d.sm[p];
                M = __dadd_rn(M, mp);
                for (int a = 0; a < D; ++a) {
                    const double xp = d.sx[a][p];
                    S[a] = __dadd_rn(S[a], __dmul_rn(mp, xp));
                    bmin[a] = fmin(bmin[a], xp);
                    bmax[a] = fmax(bmax[a], xp);
                }
            }
        }
    }
    d.nhmax[nd] = hmax;
    if (hmax_only) return;
    d.nmass[nd] = M;
    for (int a = 0; a < 3; ++a) {
        d.ncom[a][nd] = (a < D) ? __ddiv_rn(S[a], M) : 0.0;
        d.nbmin[a][nd] = (a < D) ? bmin[a] : 0.0;
        d.nbmax[a][nd] = (a < D) ? bmax[a] : 0.0;
    }
}

// cell_moments with the loads of four children in flight at once (the serial form waits for one child after the
// other: the launch was bound by the latency of those loads, 0.45 ms on C5).  The sums run in the same order on the same
// values: same bits.  Returns false, with nothing written, when a leaf of several particles is among the children
// (the caller then takes cell_moments).
template <int D, bool HONLY>
__device__ __forceinline__ bool cell_moments_batched(const Dev &d, int nd) {
    constexpr int NC = 1 << D, HB = (NC < 4) ? NC : 4;
    const int *cl = d.child_lo + (size_t)nd * (NC + 1);
    const int *ch = d.child + (size_t)nd * NC;
    int code[NC], lo[NC + 1];
#pragma unroll
    for (int c = 0; c < NC; ++c) { code[c] = ch[c]; lo[c] = cl[c]; }
    lo[NC] = cl[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c)
        if (code[c] == -2 && lo[c + 1] - lo[c] != 1) return false;
    double M = 0.0, S[3] = {0, 0, 0};
    double bmin[3] = {INFINITY, INFINITY, INFINITY}, bmax[3] = {-INFINITY, -INFINITY, -INFINITY}, hmax = 0.0;
#pragma unroll
    for (int c0 = 0; c0 < NC; c0 += HB) {
        double w[HB], hm[HB], x[HB][3], mn[HB][3], mx[HB][3];
#pragma unroll
        for (int k = 0; k < HB; ++k) {                        // all loads of the batch first
            const int cd = code[c0 + k];
            w[k] = 0.0; hm[k] = 0.0;
#pragma unroll
            for (int a = 0; a < 3; ++a) { x[k][a] = 0.0; mn[k][a] = INFINITY; mx[k][a] = -INFINITY; }
            if (cd >= 0) {
                hm[k] = __ldcg(&d.nhmax[cd]);
                if (!HONLY) {
                    w[k] = __ldcg(&d.nmass[cd]);
#pragma unroll
                    for (int a = 0; a < D; ++a) {
                        x[k][a] = __ldcg(&d.ncom[a][cd]);
                        mn[k][a] = __ldcg(&d.nbmin[a][cd]);
                        mx[k][a] = __ldcg(&d.nbmax[a][cd]);
                    }
                }
            } else if (cd == -2) {
                const int p = lo[c0 + k];
                hm[k] = d.sh[p];
                if (!HONLY) {
                    w[k] = d.sm[p];
#pragma unroll
                    for (int a = 0; a < D; ++a) { x[k][a] = d.sx[a][p]; mn[k][a] = x[k][a]; mx[k][a] = x[k][a]; }
                }
            }
        }
#pragma unroll
        for (int k = 0; k < HB; ++k) {                        // then the sums, in octant order
            if (code[c0 + k] == -1) continue;
            hmax = fmax(hmax, hm[k]);
            if (HONLY) continue;
            M = __dadd_rn(M, w[k]);
#pragma unroll
            for (int a = 0; a < D; ++a) {
                S[a] = __dadd_rn(S[a], __dmul_rn(w[k], x[k][a]));
                bmin[a] = fmin(bmin[a], mn[k][a]);
                bmax[a] = fmax(bmax[a], mx[k][a]);
            }
        }
    }
    d.nhmax[nd] = hmax;
    if (HONLY) return true;
    d.nmass[nd] = M;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        d.ncom[a][nd] = (a < D) ? __ddiv_rn(S[a < D ? a : 0], M) : 0.0;
        d.nbmin[a][nd] = (a < D) ? bmin[a < D ? a : 0] : 0.0;
        d.nbmax[a][nd] = (a < D) ? bmax[a < D ? a : 0] : 0.0;
    }
    return true;
}

// Bottom-up in ONE launch (the first version launched once per level: 21 launches, 0.75 ms on C5).  A thread starts at
// a cell without child cells and climbs: after finishing a cell it increments the parent's counter; the thread that
// brings the counter to the parent's number of child cells computes the parent (all its children are complete and
// visible: release / acquire on the counter), the others retire.  The arithmetic of a cell does not depend on which
// thread performs it.  (2^D lanes per cell with the ordered sums done by shuffles were measured too: faster than the
// serial loop over the children for small sets, slower than the batched loads everywhere; profiles/r2_c5.md.)
template <int D, bool HONLY>
__global__ void k_moments(Dev d) {
    int nd = blockIdx.x * blockDim.x + threadIdx.x;
    if (nd >= d.status->n_nodes) return;
    if (d.ncc[nd] != 0) return;
    while (true) {
        if (!cell_moments_batched<D, HONLY>(d, nd)) cell_moments(d, nd, HONLY);
        const int parent = d.nparent[nd];
        if (parent < 0) return;
        // release my cell, acquire the siblings' cells: one acq_rel read-modify-write at device scope
        cuda::atomic_ref<int, cuda::thread_scope_device> ready(d.nready[parent]);
        const int done = ready.fetch_add(1, cuda::std::memory_order_acq_rel) + 1;
        if (done != d.ncc[parent]) return;
        nd = parent;
    }
}

__global__ void k_reset_ready(Dev d) {
    const int nd = blockIdx.x * blockDim.x + threadIdx.x;
    if (nd < d.status->n_nodes) d.nready[nd] = 0;
}

void sph_launch_moments(sph_ctx *ctx, int hmax_only) {
    Dev &d = ctx->d;
    if (hmax_only) {            // a second climb over the same tree: the counters start from zero again
        k_reset_ready<<<sph_ceil_div(d.n, 256), 256, 0, ctx->stream>>>(d);
        ctx->launches += 1;
    }
    const int blocks = sph_ceil_div(d.n, 128);
    if (d.D == 3) { if (hmax_only) k_moments<3, true><<<blocks, 128, 0, ctx->stream>>>(d); else k_moments<3, false><<<blocks, 128, 0, ctx->stream>>>(d); }
    else { if (hmax_only) k_moments<2, true><<<blocks, 128, 0, ctx->stream>>>(d); else k_moments<2, false><<<blocks, 128, 0, ctx->stream>>>(d); }
    ctx->launches += 1;
}

__global__ void k_zero_status(Dev d) {
    d.status->n_nodes = 0;
    d.status->n_pairs = 0; d.status->n_inter = 0; d.status->n_visit = 0; d.status->n_open = 0;
}

void sph_stage_tree(sph_ctx *ctx) {
    Dev &d = ctx->d;
    const int n = d.n;
    StageTimer *tt = new StageTimer(ctx, SPH_T_TREE);
    k_zero_status<<<1, 1, 0, ctx->stream>>>(d);
    k_find_nodes<<<sph_ceil_div(n, 256), 256, 0, ctx->stream>>>(d);
    ctx->launches += 2;
    int bits = 5, t = n;                     // key = first particle << 5 | level: one radix pass less for n < 2^19
    while (t > 0) { ++bits; t >>= 1; }
    int cur = 0;
    sph_radix_sort(ctx, d.nkey, d.nhi, n, &d.status->n_nodes, bits, &cur);
    k_fill_nodes<<<sph_ceil_div(n, 128), 128, 0, ctx->stream>>>(d, d.nkey[cur], d.nhi[cur]);
    ctx->launches += 1;
    delete tt;
    StageTimer tm(ctx, SPH_T_MOMENTS);
    sph_launch_moments(ctx, 0);
}
