// A1 + A2: root cube, Morton keys, LSD radix sort, SoA reorder.
//   root cube:  PAPER.md:463-465 (eq. 67); min-corner anchored (reading U12)
//   keys:       L bits per dimension, x lowest bit of each group (U13); ties by original index
//   sort:       hand-written 8-bit LSD radix sort, one kernel per pass (digit counts of all passes up front, stable
//               scatter with decoupled look-back over the tiles)
//   reorder:    every state array gathered into Morton order so that the tree walks, the partner
//               search and the pair sums read neighbouring particles from neighbouring addresses.
#include <cuda/atomic>

#include "sph_internal.cuh"

#define SORT_THREADS 256
#define SORT_ITEMS 8                    // measured on C5: 16 -> 0.556 ms, 12 -> 0.520, 8 -> 0.517 (shorter ranking chains, 6 blocks per SM)
#define SORT_TILE (SORT_THREADS * SORT_ITEMS)
#define SORT_WARPS (SORT_THREADS / 32)

// ------------------------------------------------------------------------------------------
// bounding box: per-block partial min/max; the last block to finish reduces them and derives s0 and scale
// ------------------------------------------------------------------------------------------
// min / max as integers: the bit pattern of a double with the sign bit flipped (positive) or all bits flipped (negative)
// orders like the value, and integer min / max cost one instruction where fmin / fmax of doubles cost four
__device__ __forceinline__ u64 dbl_key(double v) {
    const u64 b = (u64)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double key_dbl(u64 k) {
    return __longlong_as_double((long long)((k >> 63) ? (k & 0x7fffffffffffffffull) : ~k));
}

// The last block to finish (counter in d.partial's tail) reduces the per-block partials and derives s0 and scale.
__global__ void __launch_bounds__(256) k_bbox(Dev d, int nblocks, unsigned *done) {
    __shared__ u64 smin[3][8], smax[3][8];
    __shared__ bool last;
    u64 lo[3] = {~0ull, ~0ull, ~0ull}, hi[3] = {0ull, 0ull, 0ull};
    const int stride = gridDim.x * blockDim.x;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < d.n; i += 4 * stride) {           // four loads per axis in flight
        for (int a = 0; a < d.D; ++a) {
            const u64 k0 = dbl_key(d.x[a][i]), k1 = dbl_key(d.x[a][i + stride]), k2 = dbl_key(d.x[a][i + 2 * stride]),
                      k3 = dbl_key(d.x[a][i + 3 * stride]);
            lo[a] = min(min(lo[a], k0), min(k1, min(k2, k3)));
            hi[a] = max(max(hi[a], k0), max(k1, max(k2, k3)));
        }
    }
    for (; i < d.n; i += stride)
        for (int a = 0; a < d.D; ++a) { const u64 k = dbl_key(d.x[a][i]); lo[a] = min(lo[a], k); hi[a] = max(hi[a], k); }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    for (int a = 0; a < 3; ++a) {
        for (int o = 16; o > 0; o >>= 1) {
            lo[a] = min(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = max(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
        if (l == 0) { smin[a][w] = lo[a]; smax[a][w] = hi[a]; }
    }
    __syncthreads();
    u64 *part = reinterpret_cast<u64 *>(d.partial);
    if (threadIdx.x < 6) {
        const int a = threadIdx.x >> 1, isx = threadIdx.x & 1;
        u64 v = isx ? smax[a][0] : smin[a][0];
        for (int k = 1; k < 8; ++k) v = isx ? max(v, smax[a][k]) : min(v, smin[a][k]);
        part[(blockIdx.x * 3 + a) * 2 + isx] = v;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = (atomicAdd(done, 1u) == (unsigned)(nblocks - 1));
    __syncthreads();
    if (!last) return;
    __threadfence();
    for (int a = 0; a < 3; ++a) { lo[a] = ~0ull; hi[a] = 0ull; }
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x)
        for (int a = 0; a < 3; ++a) {
            lo[a] = min(lo[a], __ldcg(&part[(b * 3 + a) * 2 + 0]));
            hi[a] = max(hi[a], __ldcg(&part[(b * 3 + a) * 2 + 1]));
        }
    for (int a = 0; a < 3; ++a) {
        for (int o = 16; o > 0; o >>= 1) {
            lo[a] = min(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = max(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
        if (l == 0) { smin[a][w] = lo[a]; smax[a][w] = hi[a]; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double mn[3], mx[3];
        for (int a = 0; a < 3; ++a) {
            u64 l2 = smin[a][0], h2 = smax[a][0];
            for (int k = 1; k < 8; ++k) { l2 = min(l2, smin[a][k]); h2 = max(h2, smax[a][k]); }
            mn[a] = key_dbl(l2); mx[a] = key_dbl(h2);
        }
        double s0 = 0.0;
        for (int a = 0; a < d.D; ++a) s0 = fmax(s0, __dsub_rn(mx[a], mn[a]));   // eq. 67
        if (!(s0 > 0.0)) s0 = 1.0;
        for (int a = 0; a < 3; ++a) d.root->xmin[a] = (a < d.D) ? mn[a] : 0.0;
        d.root->s0 = s0;
        d.root->scale = __ddiv_rn(ldexp(1.0, d.L), s0);
        *done = 0u;                                             // for the next launch
    }
}

__device__ __forceinline__ u64 spread3(u64 v) {   // 21 bits -> every third bit
    v &= 0x1fffffull;
    v = (v | (v << 32)) & 0x1f00000000ffffull;
    v = (v | (v << 16)) & 0x1f0000ff0000ffull;
    v = (v | (v << 8)) & 0x100f00f00f00f00full;
    v = (v | (v << 4)) & 0x10c30c30c30c30c3ull;
    v = (v | (v << 2)) & 0x1249249249249249ull;
    return v;
}
__device__ __forceinline__ u64 spread2(u64 v) {   // 21 bits -> every second bit
    v &= 0x1fffffull;
    v = (v | (v << 16)) & 0x0000ffff0000ffffull;
    v = (v | (v << 8)) & 0x00ff00ff00ff00ffull;
    v = (v | (v << 4)) & 0x0f0f0f0f0f0f0f0full;
    v = (v | (v << 2)) & 0x3333333333333333ull;
    v = (v | (v << 1)) & 0x5555555555555555ull;
    return v;
}

__global__ void k_keys(Dev d) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    const double scale = d.root->scale;
    const u64 gmax = (1ull << d.L) - 1ull;
    u64 g[3] = {0, 0, 0};
    for (int a = 0; a < d.D; ++a) {
        double t = __dmul_rn(__dsub_rn(d.x[a][i], d.root->xmin[a]), scale);
        u64 gi = (u64)t;                       // truncation; t >= 0
        g[a] = gi < gmax ? gi : gmax;
    }
    u64 key = (d.D == 3) ? (spread3(g[0]) | (spread3(g[1]) << 1) | (spread3(g[2]) << 2))
                         : (spread2(g[0]) | (spread2(g[1]) << 1));
    d.key[0][i] = key;
    d.idx[0][i] = i;
}

// ------------------------------------------------------------------------------------------
// radix sort
// ------------------------------------------------------------------------------------------
// One pass = ONE kernel ("onesweep": Adinets & Merrill 2022, restated).  The counts of every digit of every pass over
// the whole input are taken once up front (k_sort_hist_all) and turned into the global start of every digit
// (k_sort_bases).  In a pass a block takes the next tile (a ticket, so that tiles start in order), ranks its keys,
// publishes the tile's digit counts and obtains the number of equal digits in all earlier tiles by looking back over the
// published counts of its predecessors: a word holds a count and a state, AGGREGATE (this tile alone) or PREFIX (this tile
// and everything before it); the walk back stops at the first PREFIX.  A tile waits only for tiles with smaller tickets,
// which are resident or finished, so the chain always ends (tile 0 publishes a PREFIX at once).  Round 1's pass was a
// histogram kernel, a three-kernel scan and the scatter: 40 launches for 8 passes, 11 now.
#define SORT_MAX_PASSES 8
#define SORT_LOOK 8                     // predecessors inspected per step of the look-back
#define SORT_FLAG_A 0x40000000u
#define SORT_FLAG_P 0x80000000u
#define SORT_CNT_MASK 0x3fffffffu       // n <= 0x3fffffff (cfg_ok)

// workspace (unsigned words): tickets [8, padded to 64] | digit counts / bases [8][256] | tile states [passes][tiles][256]
__host__ __device__ inline size_t sort_ws_words(i64 n) { return 64 + SORT_MAX_PASSES * 256 + (size_t)SORT_MAX_PASSES * 256 * ((n + SORT_TILE - 1) / SORT_TILE); }
size_t sph_sort_ws_words(i64 n) { return sort_ws_words(n); }

__global__ void __launch_bounds__(256) k_sort_hist_all(const u64 *__restrict__ kin, int n_host, const int *n_dev, int shift0,
                                                       int passes, unsigned *ghist) {
    __shared__ unsigned h[SORT_MAX_PASSES][256];
    const int n = n_dev ? *n_dev : n_host;
    for (int k = threadIdx.x; k < SORT_MAX_PASSES * 256; k += 256) (&h[0][0])[k] = 0;
    __syncthreads();
    for (i64 i = (i64)blockIdx.x * 256 + threadIdx.x; i < n; i += (i64)gridDim.x * 256) {
        const u64 key = kin[i] >> shift0;
        for (int p = 0; p < passes; ++p) atomicAdd(&h[p][(unsigned)(key >> (8 * p)) & 255u], 1u);
    }
    __syncthreads();
    for (int p = 0; p < passes; ++p) {
        const unsigned c = h[p][threadIdx.x];
        if (c) atomicAdd(&ghist[p * 256 + threadIdx.x], c);
    }
}

// exclusive scan of the 256 counts of every pass, in place (one block, thread = digit)
__global__ void __launch_bounds__(256) k_sort_bases(unsigned *ghist, int passes) {
    __shared__ unsigned wsum[8];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int p = 0; p < passes; ++p) {
        const unsigned c = ghist[p * 256 + threadIdx.x];
        unsigned inc = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { unsigned t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
        if (lane == 31) wsum[w] = inc;
        __syncthreads();
        unsigned off = 0;
        for (int k = 0; k < w; ++k) off += wsum[k];
        ghist[p * 256 + threadIdx.x] = off + inc - c;
        __syncthreads();
    }
}

// Stable scatter of one 8-bit digit.  Ranks inside a warp come from match_any; the tile is first
// put into digit order in shared memory, so that consecutive threads write consecutive addresses
// of the output (runs of one digit) instead of 256 scattered streams.
struct SortSmem {
    u64 key[SORT_TILE];
    int val[SORT_TILE];
    unsigned wc[SORT_WARPS][256];
    unsigned gbase[256];        // global start of the tile's run of every digit
    unsigned lstart[256];       // start of the digit inside the tile
};

__global__ void __launch_bounds__(SORT_THREADS)
k_sort_pass(const u64 *__restrict__ kin, const int *__restrict__ vin, u64 *__restrict__ kout,
            int *__restrict__ vout, int n_host, const int *n_dev, int shift,
            const unsigned *__restrict__ base, unsigned *state, unsigned *ticket) {
    extern __shared__ __align__(16) unsigned char sort_raw[];
    SortSmem &sm = *reinterpret_cast<SortSmem *>(sort_raw);
    __shared__ int s_tile;
    const int n = n_dev ? *n_dev : n_host;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) s_tile = (int)atomicAdd(ticket, 1u);
    for (int k = threadIdx.x; k < SORT_WARPS * 256; k += SORT_THREADS) (&sm.wc[0][0])[k] = 0;
    __syncthreads();
    const int tile = s_tile;
    const i64 tile0 = (i64)tile * SORT_TILE;
    if (tile0 >= n) return;                                     // (tiles beyond a device-side n: nobody looks at them)
    const i64 wbase = tile0 + (i64)w * (32 * SORT_ITEMS);
    u64 key[SORT_ITEMS];
    int val[SORT_ITEMS];
    unsigned rank[SORT_ITEMS];
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int j = 0; j < SORT_ITEMS; ++j) {
        i64 i = wbase + j * 32 + lane;
        bool valid = i < n;
        key[j] = valid ? kin[i] : 0ull;
        val[j] = valid ? vin[i] : 0;
        unsigned dg = (unsigned)(key[j] >> shift) & 255u;
        unsigned m = __match_any_sync(0xffffffffu, valid ? dg : 256u);
        unsigned prev = valid ? sm.wc[w][dg] : 0u;
        __syncwarp();
        if (valid && (m & lt) == 0) sm.wc[w][dg] = prev + __popc(m);
        __syncwarp();
        rank[j] = prev + __popc(m & lt);
    }
    __syncthreads();
    unsigned tot;
    {   // exclusive scan over warps, one digit per thread
        unsigned run = 0;
        for (int k = 0; k < SORT_WARPS; ++k) { unsigned t = sm.wc[k][threadIdx.x]; sm.wc[k][threadIdx.x] = run; run += t; }
        tot = run;
    }
    {   // equal digits in all earlier tiles: publish, look back, publish the inclusive prefix
        cuda::atomic_ref<unsigned, cuda::thread_scope_device> mine(state[(size_t)tile * 256 + threadIdx.x]);
        unsigned excl = 0;
        if (tile == 0) mine.store(SORT_FLAG_P | tot, cuda::std::memory_order_relaxed);
        else {
            mine.store(SORT_FLAG_A | tot, cuda::std::memory_order_relaxed);
            // a window of SORT_LOOK predecessors is read at once (independent loads), then consumed in order
            int t = tile - 1;
            bool done = false;
            while (!done) {
                unsigned v[SORT_LOOK];
#pragma unroll
                for (int q = 0; q < SORT_LOOK; ++q) {
                    cuda::atomic_ref<unsigned, cuda::thread_scope_device> prev(state[(size_t)max(t - q, 0) * 256 + threadIdx.x]);
                    v[q] = prev.load(cuda::std::memory_order_relaxed);
                }
                int used = 0;
#pragma unroll
                for (int q = 0; q < SORT_LOOK; ++q) {
                    if (!done && used == q && (v[q] >> 30) != 0u) {      // ready, and everything nearer was ready too
                        excl += v[q] & SORT_CNT_MASK;
                        ++used;
                        if (v[q] & SORT_FLAG_P) done = true;          // (tile 0 always ends the walk: t - q >= 0 here)
                    }
                }
                t -= used;
                if (used == 0) __nanosleep(20);
            }
            mine.store(SORT_FLAG_P | (excl + tot), cuda::std::memory_order_relaxed);
        }
        sm.gbase[threadIdx.x] = base[threadIdx.x] + excl;
    }
    {   // start of every digit inside the tile
        unsigned inc = tot;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { unsigned t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
        __shared__ unsigned wsum[SORT_WARPS];
        if (lane == 31) wsum[w] = inc;
        __syncthreads();
        unsigned off = 0;
        for (int k = 0; k < w; ++k) off += wsum[k];
        sm.lstart[threadIdx.x] = off + inc - tot;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < SORT_ITEMS; ++j) {
        i64 i = wbase + j * 32 + lane;
        if (i < n) {
            unsigned dg = (unsigned)(key[j] >> shift) & 255u;
            unsigned lp = sm.lstart[dg] + sm.wc[w][dg] + rank[j];
            sm.key[lp] = key[j];
            sm.val[lp] = val[j];
        }
    }
    __syncthreads();
    const int cnt = (int)min((i64)SORT_TILE, (i64)n - tile0);
    for (int k = threadIdx.x; k < cnt; k += SORT_THREADS) {
        const u64 kk = sm.key[k];
        const unsigned dg = (unsigned)(kk >> shift) & 255u;
        const unsigned pos = sm.gbase[dg] + ((unsigned)k - sm.lstart[dg]);
        kout[pos] = kk;
        vout[pos] = sm.val[k];
    }
}

// one-time kernel attributes (called by sph_create, outside any stream capture)
void sph_sort_init() {
    cudaFuncSetAttribute(k_sort_pass, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem));
}

void sph_radix_sort(sph_ctx *ctx, u64 *key[2], int *val[2], int n_host, const int *n_dev, int bits, int *cur) {
    const int nblocks = sph_ceil_div(n_host, SORT_TILE);
    const int passes = (bits + 7) / 8;
    unsigned *ws = ctx->d.hist, *ticket = ws, *ghist = ws + 64, *state = ws + 64 + SORT_MAX_PASSES * 256;
    cudaMemsetAsync(ws, 0, (64 + SORT_MAX_PASSES * 256 + (size_t)passes * 256 * nblocks) * sizeof(unsigned), ctx->stream);
    int c = *cur;
    k_sort_hist_all<<<min(sph_ceil_div(n_host, 2048), 148 * 8), 256, 0, ctx->stream>>>(key[c], n_host, n_dev, 0, passes, ghist);
    k_sort_bases<<<1, 256, 0, ctx->stream>>>(ghist, passes);
    for (int p = 0; p < passes; ++p) {
        k_sort_pass<<<nblocks, SORT_THREADS, sizeof(SortSmem), ctx->stream>>>(key[c], val[c], key[c ^ 1], val[c ^ 1], n_host, n_dev, 8 * p,
                                                                 ghist + p * 256, state + (size_t)p * 256 * nblocks, ticket + p);
        c ^= 1;
    }
    ctx->launches += 2 + passes;
    *cur = c;
}

// ------------------------------------------------------------------------------------------
// SoA gather into sorted order
// ------------------------------------------------------------------------------------------
// Two kernels: what the tree, the partner search and the walk read (positions, masses, h), and the rest of the
// state.  sph_step_host (api.cu) runs the second one only when the later part of its upload has arrived.
__global__ void k_gather_geom(Dev d) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    int o = d.perm[i];
    d.iperm[o] = i;
    for (int a = 0; a < 3; ++a) d.sx[a][i] = (a < d.D) ? d.x[a][o] : 0.0;
    d.sm[i] = d.m[o];
    d.sh[i] = d.h[o];
}

__global__ void k_gather_rest(Dev d) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    int o = d.perm[i];
    for (int a = 0; a < 3; ++a) d.sv[a][i] = (a < d.D) ? d.v[a][o] : 0.0;
    d.srho[i] = d.rho[o];
    d.su[i] = d.u[o];
    d.smat[i] = d.mat[o];
    if (d.flags & SPH_F_SOLID)
        for (int k = 0; k < 6; ++k) d.sS[k][i] = d.S[k][o];
    if (d.flags & SPH_F_DAMAGE) d.sdmg[i] = d.dmg[o];
}

void sph_stage_gather_rest(sph_ctx *ctx) {
    StageTimer tm(ctx, SPH_T_REORDER);
    k_gather_rest<<<sph_ceil_div(ctx->d.n, 256), 256, 0, ctx->stream>>>(ctx->d);
    ctx->launches += 1;
}

void sph_stage_order(sph_ctx *ctx) {
    Dev &d = ctx->d;
    const int n = d.n;
    int nb = min(sph_ceil_div(n, 256), 1024);
    {
        StageTimer tm(ctx, SPH_T_KEYS);
        k_bbox<<<nb, 256, 0, ctx->stream>>>(d, nb, d.bbox_done);
        k_keys<<<sph_ceil_div(n, 256), 256, 0, ctx->stream>>>(d);
        ctx->launches += 2;
    }
    int cur = 0;
    {
        StageTimer tm(ctx, SPH_T_SORT);
        sph_radix_sort(ctx, d.key, d.idx, n, nullptr, d.D * d.L, &cur);
    }
    d.keys = d.key[cur];
    d.perm = d.idx[cur];
    ctx->sort_cur = cur;
    {
        StageTimer tm(ctx, SPH_T_REORDER);
        k_gather_geom<<<sph_ceil_div(n, 256), 256, 0, ctx->stream>>>(d);
        ctx->launches += 1;
    }
    if (!ctx->split_gather) sph_stage_gather_rest(ctx);
}
