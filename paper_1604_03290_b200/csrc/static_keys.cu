// sph_morton_keys_static: root cube (eq. 67) and Morton keys of a set of particles
// WITHOUT any device workspace from the caller and without any allocation by the library.
//
// Who this is for.  Every other compute call of this library needs a context, and a context needs a device workspace of
// sph_workspace_bytes() bytes that the caller obtains somewhere.  Some callers have no way to obtain device memory when
// they want the keys:
//   * a plug-in (in-situ analysis, a visualisation filter, a load balancer) that a host application hands DEVICE pointers
//     to its particles and a DEVICE output buffer: the application owns the memory pool, and the plug-in is not
//     allowed to go around it with cudaMalloc;
//   * code on a latency-critical path: cudaMalloc and cudaFree synchronise the whole device and take an unbounded time,
//     so a time loop that must not stall (or must not disturb the other streams of the process) cannot call them;
//   * a process that runs close to its memory limit (a fixed MPS / MIG share, a simulation that fills the HBM): an
//     allocation may fail exactly when the keys are needed.
// Such a caller still has its inputs (the positions) and its outputs (the key array); what it lacks is the scratch memory
// the bounding-box reduction needs (per-block partial boxes, an arrival counter, the root cube handed to the key kernel).
// Here that scratch is a fixed array inside the library's device image, g_static_scratch below: every GPU that loads
// libsph_b200.so holds its SPH_STATIC_SCRATCH_BYTES (49 408 bytes) from the first use of the library on that GPU until the
// process exits, whether or not this entry point is ever called.
//
// Rules that follow from one shared array (also in include/sph.h):
//   * all calls on one GPU use the same scratch.  Calls that may overlap on the GPU (different streams without an
//     ordering between them, or different host threads on different streams) race on it and give wrong keys; calls on one
//     stream, or on streams ordered by events, are fine;
//   * the scratch keeps what the last call left.  The only word that must start at zero is the arrival counter of the
//     reduction; the call clears it on the stream before every launch (the partial boxes and the root cube are fully
//     overwritten before they are read);
//   * the FIRST call on a GPU looks up the device address of the array (cudaGetSymbolAddress, which may also load the
//     module onto that GPU).  Make that first call during set-up, with that GPU current, and before any stream capture.
//
// The kernels are variants of k_bbox / k_keys (order.cu) that take plain pointers instead of a context's pointer block:
// the same arithmetic in the same order, hence the same root cube and the same keys bit for bit
// (tests/test_zz_no_alloc.py).  order.cu itself is untouched and shares no state with this file.
#include <cuda_runtime.h>
#include <stdarg.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/sph.h"

typedef unsigned long long u64;

#define SK_THREADS 256
#define SK_MAX_BLOCKS 1024      // blocks of the reduction = partial boxes in the scratch
#define SK_MAX_DEVICES 64

// Layout of the scratch.  Host code never reads or writes it; it only obtains its device address.
struct StaticScratch {
    u64 part[SK_MAX_BLOCKS][6];     // per block: (min, max) of x, y, z as ordered bit patterns
    double xmin[3];                 // root cube: min corner, edge, 2^L / edge (eq. 67)
    double s0;
    double scale;
    unsigned done;                  // blocks that have stored their partial box; MUST be 0 at launch
    unsigned pad[53];
};
static_assert(sizeof(StaticScratch) == SPH_STATIC_SCRATCH_BYTES, "include/sph.h states the size of the scratch");
static_assert(SPH_STATIC_SCRATCH_BYTES % 256 == 0, "whole 256-byte lines");

// In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address, and a kernel that was
// handed `g_static_scratch` itself would fault or scribble over host memory.
static __device__ __align__(256) unsigned char g_static_scratch[SPH_STATIC_SCRATCH_BYTES];

// device address of the array on every GPU this process has used the entry point on (looked up once per GPU)
static std::mutex g_lookup_mutex;
static StaticScratch *g_scratch_of_device[SK_MAX_DEVICES];

static int fail(char *errbuf, size_t errbuf_len, int code, const char *fmt, ...) {
    if (errbuf && errbuf_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, errbuf_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// a double's bit pattern, mapped so that unsigned integer order equals floating-point order
__device__ __forceinline__ u64 sk_ordered(double v) {
    const u64 b = (u64)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double sk_value(u64 k) {
    return __longlong_as_double((long long)((k >> 63) ? (k & 0x7fffffffffffffffull) : ~k));
}

// block-wide min / max of three axes; the result is valid in thread 0's smin / smax rows [a][0..7]
__device__ __forceinline__ void sk_block_reduce(u64 lo[3], u64 hi[3], u64 (*smin)[8], u64 (*smax)[8]) {
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        for (int o = 16; o > 0; o >>= 1) {
            lo[a] = min(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = max(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
        if (l == 0) { smin[a][w] = lo[a]; smax[a][w] = hi[a]; }
    }
    __syncthreads();
}

// Bounding box of the particles, then the root cube of eq. 67: the cube is anchored at the min corner and its edge is
// the largest extent over the axes (reading U12), 1 when all particles coincide.  Every block stores a partial
// box into the scratch; the block that arrives last folds them.
__global__ void __launch_bounds__(SK_THREADS)
k_bbox_static(const double *__restrict__ x0, const double *__restrict__ x1, const double *__restrict__ x2, int n, int D, int L,
              StaticScratch *s) {
    __shared__ u64 smin[3][8], smax[3][8];
    __shared__ bool last;
    const double *x[3] = {x0, x1, x2};
    u64 lo[3] = {~0ull, ~0ull, ~0ull}, hi[3] = {0ull, 0ull, 0ull};
    const int stride = gridDim.x * blockDim.x;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (a < D) {
                const u64 k = sk_ordered(x[a][i]);
                lo[a] = min(lo[a], k);
                hi[a] = max(hi[a], k);
            }
    }
    sk_block_reduce(lo, hi, smin, smax);
    if (threadIdx.x < 6) {
        const int a = threadIdx.x >> 1, is_max = threadIdx.x & 1;
        u64 v = is_max ? smax[a][0] : smin[a][0];
        for (int k = 1; k < 8; ++k) v = is_max ? max(v, smax[a][k]) : min(v, smin[a][k]);
        s->part[blockIdx.x][threadIdx.x] = v;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = (atomicAdd(&s->done, 1u) == gridDim.x - 1u);
    __syncthreads();
    if (!last) return;
    __threadfence();
#pragma unroll
    for (int a = 0; a < 3; ++a) { lo[a] = ~0ull; hi[a] = 0ull; }
    for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = min(lo[a], __ldcg(&s->part[b][2 * a]));
            hi[a] = max(hi[a], __ldcg(&s->part[b][2 * a + 1]));
        }
    sk_block_reduce(lo, hi, smin, smax);
    if (threadIdx.x == 0) {
        double mn[3], mx[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            u64 l2 = smin[a][0], h2 = smax[a][0];
            for (int k = 1; k < 8; ++k) { l2 = min(l2, smin[a][k]); h2 = max(h2, smax[a][k]); }
            mn[a] = sk_value(l2);
            mx[a] = sk_value(h2);
        }
        double s0 = 0.0;
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (a < D) s0 = fmax(s0, __dsub_rn(mx[a], mn[a]));                  // eq. 67
        if (!(s0 > 0.0)) s0 = 1.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) s->xmin[a] = (a < D) ? mn[a] : 0.0;
        s->s0 = s0;
        s->scale = __ddiv_rn(ldexp(1.0, L), s0);
        s->done = 0u;                       // leave the counter as the next launch needs it
    }
}

__device__ __forceinline__ u64 sk_every_third_bit(u64 v) {
    v &= 0x1fffffull;
    v = (v | (v << 32)) & 0x1f00000000ffffull;
    v = (v | (v << 16)) & 0x1f0000ff0000ffull;
    v = (v | (v << 8)) & 0x100f00f00f00f00full;
    v = (v | (v << 4)) & 0x10c30c30c30c30c3ull;
    v = (v | (v << 2)) & 0x1249249249249249ull;
    return v;
}
__device__ __forceinline__ u64 sk_every_second_bit(u64 v) {
    v &= 0x1fffffull;
    v = (v | (v << 16)) & 0x0000ffff0000ffffull;
    v = (v | (v << 8)) & 0x00ff00ff00ff00ffull;
    v = (v | (v << 4)) & 0x0f0f0f0f0f0f0f0full;
    v = (v | (v << 2)) & 0x3333333333333333ull;
    v = (v | (v << 1)) & 0x5555555555555555ull;
    return v;
}

// Grid coordinates by truncation of (x - xmin) * 2^L / s0, clamped to 2^L - 1; bits interleaved with x lowest in
// every group (reading U13).  Also copies the root cube to the caller's buffer.
__global__ void __launch_bounds__(SK_THREADS)
k_keys_static(const double *__restrict__ x0, const double *__restrict__ x1, const double *__restrict__ x2, int n, int D, int L,
              const StaticScratch *__restrict__ s, u64 *__restrict__ keys, double *__restrict__ root) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0 && root) {
        root[0] = s->xmin[0]; root[1] = s->xmin[1]; root[2] = s->xmin[2]; root[3] = s->s0;
    }
    if (i >= n) return;
    const double *x[3] = {x0, x1, x2};
    const double scale = s->scale;
    const u64 gmax = (1ull << L) - 1ull;
    u64 g[3] = {0, 0, 0};
#pragma unroll
    for (int a = 0; a < 3; ++a)
        if (a < D) {
            const double t = __dmul_rn(__dsub_rn(x[a][i], s->xmin[a]), scale);
            const u64 gi = (u64)t;
            g[a] = gi < gmax ? gi : gmax;
        }
    keys[i] = (D == 3) ? (sk_every_third_bit(g[0]) | (sk_every_third_bit(g[1]) << 1) | (sk_every_third_bit(g[2]) << 2))
                       : (sk_every_second_bit(g[0]) | (sk_every_second_bit(g[1]) << 1));
}

extern "C" int sph_morton_keys_static(const double *x, const double *y, const double *z, int64_t n, int32_t dim,
                                      int32_t morton_bits, void *cuda_stream, uint64_t *keys, double *root, char *errbuf,
                                      size_t errbuf_len) {
    if (errbuf && errbuf_len) errbuf[0] = 0;
    // ---- arguments (before any CUDA call, so that a bad size is reported as such on every machine) ----
    if (dim != 2 && dim != 3) return fail(errbuf, errbuf_len, SPH_ERR_ARG, "dim = %d: must be 2 or 3", (int)dim);
    if (n < 1) return fail(errbuf, errbuf_len, SPH_ERR_ARG, "n = %lld: must be at least 1", (long long)n);
    if (n > (int64_t)SPH_STATIC_MAX_N)
        return fail(errbuf, errbuf_len, SPH_ERR_ARG,
                    "n = %lld is beyond SPH_STATIC_MAX_N = %lld, the largest set the fixed scratch of sph_morton_keys_static "
                    "serves: split the set, or use a context (sph_create) with a workspace",
                    (long long)n, (long long)SPH_STATIC_MAX_N);
    if (morton_bits < 0 || morton_bits > 21)
        return fail(errbuf, errbuf_len, SPH_ERR_ARG, "morton_bits = %d: must be 1..21 (0 = 21)", (int)morton_bits);
    if (!x || !y || (dim == 3 && !z) || !keys) return fail(errbuf, errbuf_len, SPH_ERR_ARG, "x, y, z (3-D) and keys must not be NULL");
    const int L = morton_bits ? morton_bits : 21;

    // ---- device address of the scratch on the current GPU (looked up on the first call per GPU) ----
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(errbuf, errbuf_len, SPH_ERR_CUDA, "no CUDA device: %s (there is no CPU fallback)", cudaGetErrorString(e));
    }
    if (dev < 0 || dev >= SK_MAX_DEVICES) return fail(errbuf, errbuf_len, SPH_ERR_CUDA, "device ordinal %d not supported", dev);
    StaticScratch *s = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_lookup_mutex);
        if (!g_scratch_of_device[dev]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, g_static_scratch);
            if (e != cudaSuccess || !p) {
                cudaGetLastError();
                return fail(errbuf, errbuf_len, SPH_ERR_CUDA, "cudaGetSymbolAddress(scratch) on device %d: %s", dev,
                            cudaGetErrorString(e));
            }
            g_scratch_of_device[dev] = static_cast<StaticScratch *>(p);
        }
        s = g_scratch_of_device[dev];
    }

    // ---- two launches and one 4-byte clear, nothing else ----
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int ni = (int)n;
    const int blocks_all = (ni + SK_THREADS - 1) / SK_THREADS;
    const int blocks_box = blocks_all < SK_MAX_BLOCKS ? blocks_all : SK_MAX_BLOCKS;
    // a launch that failed half way (or a call that raced with this one) may have left the counter non-zero
    e = cudaMemsetAsync(&s->done, 0, sizeof(unsigned), st);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(errbuf, errbuf_len, SPH_ERR_CUDA, "clearing the arrival counter: %s", cudaGetErrorString(e));
    }
    k_bbox_static<<<blocks_box, SK_THREADS, 0, st>>>(x, y, dim == 3 ? z : nullptr, ni, dim, L, s);
    k_keys_static<<<blocks_all, SK_THREADS, 0, st>>>(x, y, dim == 3 ? z : nullptr, ni, dim, L, s, (u64 *)keys, root);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(errbuf, errbuf_len, SPH_ERR_CUDA, "kernel launch: %s", cudaGetErrorString(e));
    return SPH_OK;
}
