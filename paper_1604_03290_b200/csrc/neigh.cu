// A5: interaction-partner search.
//
// The paper walks the tree once per particle, one thread each, descending while the particle lies
// within s/2 + h of a cell (eq. 69) and testing "distance < smoothing length" at the leaves.
// Here one WARP owns 32 particles that are consecutive in Morton order (a "group") and the walk has
// two granularities:
//
//   * The SEARCH TREE (sph_build_search_items below) holds the octree cells with more than SPH_BUCKET
//     particles and BUCKETS of <= SPH_BUCKET particles that are consecutive in Morton order (runs of
//     small sibling cells / leaves); the children of a cell are contiguous.  Every item carries the
//     bounding box and the largest h of the particles below it, rounded OUTWARD to FP32: pruning
//     runs on the FP32 pipe with directed rounding (a box that holds a partner is never cut), the FP64
//     pipe is kept for the exact membership tests.
//   * Descent: lane = item.  A round takes the children of up to four cells from a small stack of ranges; every
//     lane tests ITS item against the bounding box of the whole group (one test per item, not one per
//     item and particle) and cells within reach push their children.
//   * Buckets within reach of the group box are then looked at by lane = particle: every lane tests
//     the bucket's box against the ball around ITS particle, and only if some lane's ball touches it
//     the bucket is staged through shared memory and every lane applies the exact membership test of
//     the paper to its own particle:  r^2 = (dx*dx + dy*dy) + dz*dz  <  H*H,  H = h_a, or (h_a + h_b)/2
//     with variable h (eq. 72), every operation rounded separately, so the sets equal the oracle's bit
//     for bit.  Where the Morton curve jumps and a group's box spans a large region, the group box
//     admits many buckets, but each costs only the per-lane box test (about 20 instructions), never
//     the member loop: the exact tests a warp runs are those of the union of 32 single-particle walks.
//
// Round 1 walked a pre-order stream of the same items with one "next item" index per lane (the warp
// visited the minimum): every item cost about 40 instructions for all 32 lanes, 60 % of the kernel
// (profiles/r2_c5.md).  The descent above costs one lane one test per item.
// Lists are written group-transposed, nb[(group*cap + k)*32 + lane], so that the pair-sum kernel
// reads them fully coalesced.
#include <algorithm>
#include <type_traits>

#include "sph_internal.cuh"

#define NB_WARPS 2
#define NB_STACK 384            // ranges of child items per warp
#define NB_RESERVE 168          // a depth-first descent keeps <= 8 pending siblings per tree level (21 levels)
#define NB_RANGES 4             // ranges (cells) whose child items one round tests

// ------------------------------------------------------------------------------------------
// search tree
// ------------------------------------------------------------------------------------------
// One thread per octree cell with more than SPH_BUCKET particles ("big"): counts its child items -- a big child cell is
// one item, small children (cells or leaves) are merged into runs of <= SPH_BUCKET particles, a leaf of more coincident
// particles is cut into runs -- and notes for every child where it goes: nord[child cell] = ordinal among the parent's
// items; bmark[first particle of a run] = parent (32 bits) | ordinal (24) | length (8).
__global__ void k_count_kids(Dev d, unsigned *kcnt) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int nn = d.status->n_nodes, n = d.n;
    if (t >= n) return;
    unsigned cnt = 0;
    if (nn == 0) {
        // n == 1 or all keys equal: a virtual root (item 0) over plain runs of SPH_BUCKET
        if (t == 0) cnt = (unsigned)((n + SPH_BUCKET - 1) / SPH_BUCKET);
        if ((t % SPH_BUCKET) == 0) d.bmark[t] = (u64)(unsigned)min(SPH_BUCKET, n - t) | ((u64)(t / SPH_BUCKET) << 8);
        kcnt[t] = cnt;
        return;
    }
    if (t >= nn) { kcnt[t] = 0; return; }
    const int NC = 1 << d.D;
    const int lo = d.nlo[t], hi = d.nhi_s[t];
    if (hi - lo <= SPH_BUCKET) {
        if (t == 0) { d.bmark[0] = (u64)(unsigned)(hi - lo); cnt = 1; }      // the whole set is one bucket below the root item
        kcnt[t] = cnt;
        return;
    }
    const int *cl = d.child_lo + (size_t)t * (NC + 1);
    const int *ch = d.child + (size_t)t * NC;
    int run0 = -1, run = 0;                     // open run of small children: first particle, particles so far
    auto close_run = [&]() {
        if (run0 >= 0) { d.bmark[run0] = (u64)(unsigned)run | ((u64)cnt << 8) | ((u64)(unsigned)t << 32); ++cnt; run0 = -1; run = 0; }
    };
    for (int c = 0; c < NC; ++c) {
        const int r0 = cl[c], r1 = cl[c + 1], sz = r1 - r0;
        if (sz == 0) continue;
        if (sz > SPH_BUCKET) {
            close_run();
            if (ch[c] >= 0) { d.nord[ch[c]] = (int)cnt; ++cnt; }             // a big child cell lays itself out
            else for (int p = r0; p < r1; p += SPH_BUCKET) {                  // a leaf of > SPH_BUCKET coincident particles
                d.bmark[p] = (u64)(unsigned)min(SPH_BUCKET, r1 - p) | ((u64)cnt << 8) | ((u64)(unsigned)t << 32);
                ++cnt;
            }
            continue;
        }
        if (run0 >= 0 && run + sz > SPH_BUCKET) close_run();
        if (run0 < 0) run0 = r0;
        run += sz;                                                            // merge small siblings
    }
    close_run();
    kcnt[t] = cnt;
}

// Item 0 is the root; the children of cell t are items kfirst[t] + 1 ... + kcnt[t].
__global__ void k_emit_items(Dev d, const unsigned *kcnt, const unsigned *kfirst) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int n = d.n, nn = d.status->n_nodes;
    const int D = d.D;
    if (t == 0) {
        d.status->n_items = 1 + (int)kfirst[n - 1] + (int)kcnt[n - 1];
        if (nn == 0 || d.nhi_s[0] - d.nlo[0] <= SPH_BUCKET) {       // virtual / small root: never pruned
            SearchItem it;
            for (int a = 0; a < 3; ++a) { it.bmin[a] = -3.0e38f; it.bmax[a] = 3.0e38f; }
            it.hmax = 3.0e38f; it.pad = 0.f; it.skip = 1; it.lo = (int)kcnt[0]; it.pad2[0] = it.pad2[1] = 0;
            d.items[0] = it;
        }
    }
    {   // buckets: the warp handles the bucket starts among its 32 positions one after the other, all lanes loading the
        // (<= SPH_BUCKET) members together (one thread per bucket with a serial loop cost 0.5 ms on C5: profiles/r1d_c5.md)
        const unsigned FULL = 0xffffffffu;
        const int lane = threadIdx.x & 31, base = t - lane;
        const u64 mk = (t < n) ? d.bmark[t] : 0ull;
        unsigned starts = __ballot_sync(FULL, (mk & 0xffull) != 0ull);
        while (starts) {
            const int j = __ffs(starts) - 1;
            starts &= starts - 1;
            const int s0 = base + j;
            const u64 m0 = __shfl_sync(FULL, mk, j);
            const int len = (int)(m0 & 0xffull), ord = (int)((m0 >> 8) & 0xffffffull), par = (int)(m0 >> 32);
            const bool have = lane < len;
            const int p = s0 + (have ? lane : 0);
            // rounded outward to FP32 BEFORE the reduction: rounding is monotone, so min / max of the rounded values are
            // the rounded min / max, and FP32 min / max is one instruction where FP64 costs four
            float mn[3], mx[3], hm = have ? __double2float_ru(d.sh[p]) : 0.0f;
            for (int a = 0; a < 3; ++a) {
                const double x = (a < D) ? d.sx[a][p] : 0.0;
                mn[a] = __double2float_rd(x); mx[a] = __double2float_ru(x);
            }
            for (int o = 16; o > 0; o >>= 1) {
                for (int a = 0; a < 3; ++a) {
                    mn[a] = fminf(mn[a], __shfl_xor_sync(FULL, mn[a], o));
                    mx[a] = fmaxf(mx[a], __shfl_xor_sync(FULL, mx[a], o));
                }
                hm = fmaxf(hm, __shfl_xor_sync(FULL, hm, o));
            }
            if (lane == 0) {
                SearchItem it;
                for (int a = 0; a < 3; ++a) { it.bmin[a] = mn[a]; it.bmax[a] = mx[a]; }
                it.hmax = hm; it.pad = 0.f; it.skip = -len; it.lo = s0; it.pad2[0] = it.pad2[1] = 0;
                d.items[1 + (int)kfirst[par] + ord] = it;
            }
        }
    }
    if (t < nn) {
        const int lo = d.nlo[t], hi = d.nhi_s[t];
        if (hi - lo > SPH_BUCKET) {              // big cell: skip = first child item, lo = number of child items
            SearchItem it;
            for (int a = 0; a < 3; ++a) { it.bmin[a] = __double2float_rd(d.nbmin[a][t]); it.bmax[a] = __double2float_ru(d.nbmax[a][t]); }
            it.hmax = __double2float_ru(d.nhmax[t]); it.pad = 0.f; it.pad2[0] = it.pad2[1] = 0;
            it.skip = 1 + (int)kfirst[t];
            it.lo = (int)kcnt[t];
            d.items[t == 0 ? 0 : 1 + (int)kfirst[d.nparent[t]] + d.nord[t]] = it;
        }
    }
}

static unsigned *kcnt_of(Dev &d) { return reinterpret_cast<unsigned *>(d.bscan); }
static unsigned *kfirst_of(Dev &d) { return reinterpret_cast<unsigned *>(d.bscan) + ((size_t)d.n + 1); }

static void emit_items(sph_ctx *ctx) {
    Dev &d = ctx->d;
    k_emit_items<<<sph_ceil_div(d.n, 128), 128, 0, ctx->stream>>>(d, kcnt_of(d), kfirst_of(d));
    ctx->launches += 1;
}

void sph_build_search_items(sph_ctx *ctx) {
    Dev &d = ctx->d;
    cudaMemsetAsync(d.bmark, 0, ((size_t)d.n + 1) * sizeof(u64), ctx->stream);
    k_count_kids<<<sph_ceil_div(d.n, 128), 128, 0, ctx->stream>>>(d, kcnt_of(d));
    ctx->launches += 1;
    sph_scan_u32(ctx, kcnt_of(d), kfirst_of(d), (i64)d.n, (unsigned *)d.scan_tmp);
    emit_items(ctx);
}

// ------------------------------------------------------------------------------------------
// the walk
// ------------------------------------------------------------------------------------------
template <int D, bool VARH, bool COUNT_ONLY>
__global__ void __launch_bounds__(NB_WARPS * 32) k_neigh(Dev d) {
    __shared__ double s_c[NB_WARPS][4][32];
    __shared__ int2 s_stack[NB_WARPS][NB_STACK];

    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = d.r_lo / 32 + blockIdx.x * NB_WARPS + w;   // groups of the rank's slice [r_lo, r_hi) (all of them on one GPU)
    if (g * 32 >= d.r_hi) return;
    const int i = g * 32 + lane;
    const bool valid = i < d.r_hi;
    const int ii = valid ? i : d.r_hi - 1;                   // a tail lane repeats the last particle (keeps the group box tight)
    const unsigned FULL = 0xffffffffu, lt = (1u << lane) - 1u;

    const double xi = d.sx[0][ii], yi = d.sx[1][ii], zi = (D == 3) ? d.sx[2][ii] : 0.0;
    const double Hi = d.sh[ii];
    const double Hi2 = __dmul_rn(Hi, Hi);
    const double xq = valid ? xi : __longlong_as_double(0x7ff8000000000000ll);   // membership tests of a tail lane compare NaN: never a partner
    constexpr bool VH = VARH && !COUNT_ONLY;   // pair criterion (h_a + h_b)/2, eq. 72
    const float xlo = __double2float_rd(xi), xhi = __double2float_ru(xi), ylo = __double2float_rd(yi), yhi = __double2float_ru(yi);
    const float zlo = __double2float_rd(zi), zhi = __double2float_ru(zi);
    const float Hf = __double2float_ru(Hi) * 1.000001f;      // the pruning test must never cut a true partner
    // The group: its largest reach and TWO bounding boxes (outward), split where the Morton curve makes its largest
    // jump inside the group (the most significant bit in which two consecutive keys differ).  The particles before the
    // jump are the last ones of one octree cell, those after it the first ones of the next: each half is compact even
    // when the jump crosses half a body (one box for the group was round 1's 71.9 ms tail: a few warps looked at every
    // bucket of the workload).
    int split;
    {
        const u64 kx = (lane < 31 && i + 1 < d.r_hi) ? (d.keys[ii] ^ d.keys[ii + 1]) : 0ull;
        const int msb = kx ? 64 - __clzll((long long)kx) : 0;                 // 0 = equal keys / no right neighbour
        split = __reduce_max_sync(FULL, (unsigned)(msb << 5) | (unsigned)lane) & 31;   // box A = lanes <= split
    }
    const bool inA = lane <= split;
    const float big = 3.0e38f;
    float ax0 = inA ? xlo : big, ax1 = inA ? xhi : -big, ay0 = inA ? ylo : big, ay1 = inA ? yhi : -big;
    float az0 = inA ? zlo : big, az1 = inA ? zhi : -big;
    float bx0 = inA ? big : xlo, bx1 = inA ? -big : xhi, by0 = inA ? big : ylo, by1 = inA ? -big : yhi;
    float bz0 = inA ? big : zlo, bz1 = inA ? -big : zhi, gH = Hf;
    for (int o = 16; o > 0; o >>= 1) {
        ax0 = fminf(ax0, __shfl_xor_sync(FULL, ax0, o)); ax1 = fmaxf(ax1, __shfl_xor_sync(FULL, ax1, o));
        ay0 = fminf(ay0, __shfl_xor_sync(FULL, ay0, o)); ay1 = fmaxf(ay1, __shfl_xor_sync(FULL, ay1, o));
        bx0 = fminf(bx0, __shfl_xor_sync(FULL, bx0, o)); bx1 = fmaxf(bx1, __shfl_xor_sync(FULL, bx1, o));
        by0 = fminf(by0, __shfl_xor_sync(FULL, by0, o)); by1 = fmaxf(by1, __shfl_xor_sync(FULL, by1, o));
        if (D == 3) {
            az0 = fminf(az0, __shfl_xor_sync(FULL, az0, o)); az1 = fmaxf(az1, __shfl_xor_sync(FULL, az1, o));
            bz0 = fminf(bz0, __shfl_xor_sync(FULL, bz0, o)); bz1 = fmaxf(bz1, __shfl_xor_sync(FULL, bz1, o));
        }
        gH = fmaxf(gH, __shfl_xor_sync(FULL, gH, o));
    }
    // (an empty box B -- split = 31 -- has min = +big, max = -big: its distance to anything is huge)

    int cnt = 0;
    int *nbw = d.nb + (size_t)g * d.cap * 32 + SPH_NB_POS(lane);
    const int cap = d.cap;
    const SearchItem *__restrict__ items = d.items;
    int2 *stack = s_stack[w];

    int top = 1;
    if (lane == 0) { const int2 root = __ldg(reinterpret_cast<const int2 *>(reinterpret_cast<const float4 *>(items) + 2)); stack[0] = root; }
    __syncwarp();
    while (top > 0) {
        // ---- lane = item: the children of up to NB_RANGES cells against the box of the group ----
        // (a cell has at most 2^D child items, so one range fills a quarter of the warp: several ranges per round while the
        // stack has room for the ranges their cells may push, one range -- a plain depth-first descent -- otherwise)
        int it = 0, take = 0;
        {
            const int nrmax = (top + 32 <= NB_STACK - NB_RESERVE) ? NB_RANGES : 1;
            int2 rgs[NB_RANGES];
            int nr = 0;
#pragma unroll
            for (int r = 0; r < NB_RANGES; ++r) {
                rgs[r] = make_int2(0, 0);
                if (r < nrmax && top - r > 0) rgs[r] = stack[top - 1 - r];
            }
            __syncwarp();
            int newtop = top;
#pragma unroll
            for (int r = 0; r < NB_RANGES; ++r) {
                if (rgs[r].y > 0 && take < 32 && nr == r) {
                    const int tk = min(32 - take, rgs[r].y);
                    if (lane >= take && lane < take + tk) it = rgs[r].x + (lane - take);
                    take += tk;
                    if (tk < rgs[r].y) { if (lane == 0) stack[top - 1 - r] = make_int2(rgs[r].x + tk, rgs[r].y - tk); }   // the rest stays (it is the top entry then)
                    else --newtop;
                    ++nr;
                }
            }
            top = newtop;
            __syncwarp();
        }
        const float4 *rec = reinterpret_cast<const float4 *>(items + it);
        const float4 r0 = __ldg(rec), r1 = __ldg(rec + 1);            // bmin xyz bmax x | bmax yz hmax pad
        const int2 ab = __ldg(reinterpret_cast<const int2 *>(rec + 2));
        bool adm;
        {
            // squared distance between the item's box and the nearer of the group's two boxes, a LOWER bound, against
            // the largest reach
            const float reach = VH ? __fmul_ru(0.5f, __fadd_ru(gH, r1.z)) * 1.000001f : gH;
            const float ex = fmaxf(fmaxf(__fsub_rd(r0.x, ax1), __fsub_rd(ax0, r0.w)), 0.0f);
            const float ey = fmaxf(fmaxf(__fsub_rd(r0.y, ay1), __fsub_rd(ay0, r1.x)), 0.0f);
            const float fx = fmaxf(fmaxf(__fsub_rd(r0.x, bx1), __fsub_rd(bx0, r0.w)), 0.0f);
            const float fy = fmaxf(fmaxf(__fsub_rd(r0.y, by1), __fsub_rd(by0, r1.x)), 0.0f);
            float dA = __fmaf_rd(ey, ey, __fmul_rd(ex, ex)), dB = __fmaf_rd(fy, fy, __fmul_rd(fx, fx));
            if (D == 3) {
                const float ez = fmaxf(fmaxf(__fsub_rd(r0.z, az1), __fsub_rd(az0, r1.y)), 0.0f);
                const float fz = fmaxf(fmaxf(__fsub_rd(r0.z, bz1), __fsub_rd(bz0, r1.y)), 0.0f);
                dA = __fmaf_rd(ez, ez, dA); dB = __fmaf_rd(fz, fz, dB);
            }
            adm = (lane < take) && (fminf(dA, dB) <= __fmul_ru(reach, reach));
        }
        const unsigned cells = __ballot_sync(FULL, adm && ab.x >= 0);
        unsigned buckets = __ballot_sync(FULL, adm && ab.x < 0);
        if (adm && ab.x >= 0) {
            const int pos = top + __popc(cells & lt);
            if (pos < NB_STACK) stack[pos] = ab;
        }
        top += __popc(cells);
        if (top > NB_STACK) { if (lane == 0) atomicOr(&d.status->err_stack, 2); break; }   // unreachable: <= 8 pending siblings per level
        __syncwarp();
        // ---- lane = particle: the admitted buckets, in Morton order ----
        while (buckets) {
            const int src = __ffs(buckets) - 1;
            buckets &= buckets - 1;
            const float4 *brec = reinterpret_cast<const float4 *>(items + __shfl_sync(FULL, it, src));
            const float4 b0 = __ldg(brec), b1 = __ldg(brec + 1);
            const int2 bl = __ldg(reinterpret_cast<const int2 *>(brec + 2));
            const int m = -bl.x, lo = bl.y;
            // the ball around MY particle against the bucket's box (lower bound of the squared distance)
            const float reach = VH ? __fmul_ru(0.5f, __fadd_ru(Hf, b1.z)) * 1.000001f : Hf;
            const float ex = fmaxf(fmaxf(__fsub_rd(b0.x, xhi), __fsub_rd(xlo, b0.w)), 0.0f);
            const float ey = fmaxf(fmaxf(__fsub_rd(b0.y, yhi), __fsub_rd(ylo, b1.x)), 0.0f);
            float d2 = __fmaf_rd(ey, ey, __fmul_rd(ex, ex));
            if (D == 3) {
                const float ez = fmaxf(fmaxf(__fsub_rd(b0.z, zhi), __fsub_rd(zlo, b1.y)), 0.0f);
                d2 = __fmaf_rd(ez, ez, d2);
            }
            const bool ov = valid && (d2 <= __fmul_ru(reach, reach));
            if (!__any_sync(FULL, ov)) continue;
            if (lane < m) {
                const int p = lo + lane;
                s_c[w][0][lane] = d.sx[0][p];
                s_c[w][1][lane] = d.sx[1][p];
                if (D == 3) s_c[w][2][lane] = d.sx[2][p];
                if (VARH && !COUNT_ONLY) s_c[w][3][lane] = d.sh[p];
            }
            __syncwarp();
            // The exact test of every member, a predicated store and a predicated count per member (no branch).  Two things
            // are settled per bucket instead of per member: whether the bucket holds a particle of the group (only then a
            // member can be the lane's own particle) and whether every lane has room for all members (only otherwise the
            // capacity is checked per store).
            const int jself = i - lo;
            const bool own = __any_sync(FULL, (unsigned)jself < (unsigned)m);
            const bool tight = __any_sync(FULL, cnt + m > cap);
            auto members = [&](auto own_c, auto tight_c) {
                constexpr bool OWN = decltype(own_c)::value, TIGHT = decltype(tight_c)::value;
#pragma unroll 4
                for (int j = 0; j < m; ++j) {
                    const double dx = __dsub_rn(xq, s_c[w][0][j]);
                    const double dy = __dsub_rn(yi, s_c[w][1][j]);
                    const double dz = (D == 3) ? __dsub_rn(zi, s_c[w][2][j]) : 0.0;
                    const double r2 = sph_r2_exact(dx, dy, dz, D);
                    double H2 = Hi2;
                    if (VARH && !COUNT_ONLY) {
                        const double Hab = __dmul_rn(0.5, __dadd_rn(Hi, s_c[w][3][j]));
                        H2 = __dmul_rn(Hab, Hab);
                    }
                    if (TIGHT || COUNT_ONLY) {
                        const bool hit = (!OWN || j != jself) && r2 < H2;      // (a lane beyond the slice compares NaN: never a hit)
                        if (!COUNT_ONLY && hit && cnt < cap) nbw[(size_t)cnt * 32] = lo + j;
                        cnt += hit ? 1 : 0;
                    } else if (OWN) {
                        // compare, store and count under ONE predicate
                        asm volatile("{ .reg .pred p, q; setp.ne.s32 q, %5, %6; setp.lt.and.f64 p, %3, %4, q;\n"
                                     "  @p st.global.s32 [%1], %2; @p add.s32 %0, %0, 1; }"
                                     : "+r"(cnt) : "l"(nbw + (size_t)cnt * 32), "r"(lo + j), "d"(r2), "d"(H2), "r"(jself), "r"(j) : "memory");
                    } else {
                        asm volatile("{ .reg .pred p; setp.lt.f64 p, %3, %4;\n"
                                     "  @p st.global.s32 [%1], %2; @p add.s32 %0, %0, 1; }"
                                     : "+r"(cnt) : "l"(nbw + (size_t)cnt * 32), "r"(lo + j), "d"(r2), "d"(H2) : "memory");
                    }
                }
            };
            if (!own && !tight) members(std::false_type{}, std::false_type{});
            else if (!tight) members(std::true_type{}, std::false_type{});
            else members(std::true_type{}, std::true_type{});
            __syncwarp();
        }
    }

    if (COUNT_ONLY) {
        if (valid) d.own_cnt[i] = cnt;
    } else {
        if (valid) d.nb_cnt[i] = min(cnt, cap);
        int mx = cnt;
        for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(FULL, mx, o));
        for (int k = cnt; k < min(mx, cap); ++k) nbw[(size_t)k * 32] = ii;   // complete rows (SPH_NB_POS)
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
