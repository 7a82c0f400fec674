// Device-wide exclusive prefix sum (hand-written, three small kernels): per-block reduce ->
// one block scans the block sums -> per-block scan with the block offset added.
// Used by the radix sort (digit offsets) and by the search-item layout of the partner search.
#include "sph_internal.cuh"

#define SCAN_THREADS 256
#define SCAN_ITEMS 8
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)

template <class T>
__device__ __forceinline__ T warp_incl_scan(T v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        T t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

// exclusive scan of one value per thread over the block; returns the exclusive prefix, total in *tot
template <class T>
__device__ __forceinline__ T block_excl_scan(T v, T *s_warp, T *tot) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const T inc = warp_incl_scan(v, lane);
    if (lane == 31) s_warp[w] = inc;
    __syncthreads();
    if (w == 0) {
        T x = (lane < (int)(blockDim.x >> 5)) ? s_warp[lane] : (T)0;
        T xi = warp_incl_scan(x, lane);
        s_warp[lane] = xi - x;
        if (lane == 31) s_warp[32] = xi;
    }
    __syncthreads();
    const T res = s_warp[w] + inc - v;
    *tot = s_warp[32];
    __syncthreads();
    return res;
}

template <class T>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const T *__restrict__ in, T *__restrict__ bsum, i64 n) {
    __shared__ T s_warp[33];
    const i64 base = (i64)blockIdx.x * SCAN_TILE;
    T s = 0;
#pragma unroll
    for (int j = 0; j < SCAN_ITEMS; ++j) {
        const i64 i = base + j * SCAN_THREADS + threadIdx.x;
        if (i < n) s += in[i];
    }
    T tot;
    block_excl_scan(s, s_warp, &tot);
    if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}

// one block: exclusive scan of nb block sums in place; the grand total goes to bsum[nb]
template <class T>
__global__ void __launch_bounds__(1024) k_scan_sums(T *bsum, int nb) {
    __shared__ T s_warp[33];
    __shared__ T s_run;
    if (threadIdx.x == 0) s_run = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nb; b0 += 1024) {
        const int i = b0 + threadIdx.x;
        const T v = (i < nb) ? bsum[i] : (T)0;
        T tot;
        const T ex = block_excl_scan(v, s_warp, &tot);
        const T run = s_run;
        if (i < nb) bsum[i] = run + ex;
        __syncthreads();
        if (threadIdx.x == 0) s_run = run + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) bsum[nb] = s_run;
}

template <class T>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const T *in, T *out, const T *__restrict__ bsum, i64 n) {
    __shared__ T s_warp[33];
    const i64 base = (i64)blockIdx.x * SCAN_TILE + (i64)threadIdx.x * SCAN_ITEMS;   // blocked arrangement
    T v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int j = 0; j < SCAN_ITEMS; ++j) { v[j] = (base + j < n) ? in[base + j] : (T)0; s += v[j]; }
    T tot;
    T run = block_excl_scan(s, s_warp, &tot) + bsum[blockIdx.x];
#pragma unroll
    for (int j = 0; j < SCAN_ITEMS; ++j) {
        if (base + j < n) out[base + j] = run;
        run += v[j];
    }
}

// small inputs (the digit tables of the radix sort for the small workloads): one block, one launch
#define SCAN_SMALL 16384
template <class T>
__global__ void __launch_bounds__(1024) k_scan_small(const T *in, T *out, T *bsum, int n, int nb) {
    __shared__ T s_warp[33];
    __shared__ T s_run;
    if (threadIdx.x == 0) s_run = 0;
    __syncthreads();
    for (int b0 = 0; b0 < n; b0 += 1024) {
        const int i = b0 + threadIdx.x;
        const T v = (i < n) ? in[i] : (T)0;
        T tot;
        const T ex = block_excl_scan(v, s_warp, &tot);
        const T run = s_run;
        if (i < n) out[i] = run + ex;
        __syncthreads();
        if (threadIdx.x == 0) s_run = run + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) bsum[nb] = s_run;
}

template <class T>
static void scan_impl(sph_ctx *ctx, const T *in, T *out, i64 n, T *bsum) {
    const int nb = sph_ceil_div(n, SCAN_TILE);
    if (n <= SCAN_SMALL) {
        k_scan_small<T><<<1, 1024, 0, ctx->stream>>>(in, out, bsum, (int)n, nb);
        ctx->launches += 1;
        return;
    }
    k_scan_reduce<T><<<nb, SCAN_THREADS, 0, ctx->stream>>>(in, bsum, n);
    k_scan_sums<T><<<1, 1024, 0, ctx->stream>>>(bsum, nb);
    k_scan_apply<T><<<nb, SCAN_THREADS, 0, ctx->stream>>>(in, out, bsum, n);
    ctx->launches += 3;
}

// out[i] = sum_{j<i} in[j]; in == out allowed. scratch: sph_scan_scratch_elems(n) elements of T;
// scratch[ceil(n / 2048)] receives the grand total.
void sph_scan_u32(sph_ctx *ctx, const unsigned *in, unsigned *out, i64 n, unsigned *scratch) { scan_impl<unsigned>(ctx, in, out, n, scratch); }
void sph_scan_u64(sph_ctx *ctx, const u64 *in, u64 *out, i64 n, u64 *scratch) { scan_impl<u64>(ctx, in, out, n, scratch); }
size_t sph_scan_scratch_elems(i64 n) { return (size_t)sph_ceil_div(n, SCAN_TILE) + 2; }
