// Internal declarations shared by the CUDA translation units of libsph_b200.so.
// (Nothing here is shared with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/sph.h"

typedef unsigned long long u64;
typedef long long i64;


#define SPH_MAX_MAT 16
#define SPH_MAX_WORLD 64
#define SPH_RATE_PAD (32 * SPH_MAX_WORLD)   // rate arrays are world * slice <= n + 32 * world long (sph_set_partition)
#define SPH_WARP 32

// Device-side status block (one per context, in the workspace).
struct DevStatus {
    int n_nodes;        // internal octree nodes found by the last build
    int err_nb_overflow;
    int err_stack;      // bit 0: the gravity walk's stack guard fired, bit 1: the partner search's
    int nb_max;         // largest partner count seen
    // work counters of the last evaluation (algorithmic units for the roofline)
    u64 n_pairs;        // sum over particles of |N(a)|               (A5)
    u64 n_inter;        // accepted pseudo-particles + direct particles, per particle, summed (A11)
    u64 n_visit;        // nodes whose opening test a particle evaluated, summed               (A11)
    u64 n_open;         // of those, the cells the particle opened (did not accept), summed   (A11)
    int n_items;        // items of the search tree (neigh.cu)
    int pad;
    u64 rkerr;          // bit pattern of the error estimate of eq. 63 (sph_step_rk3)
    u64 dtlim[3];       // bit patterns of the three time-step limits (positive doubles order like integers)
};

// Root cube of the last build (device).
struct DevRoot {
    double xmin[3];
    double s0;
    double scale;       // 2^L / s0
    double pad[3];
};

// One item of the search tree (neigh.cu): the octree cells that hold more than SPH_BUCKET particles
// ("big" cells) and buckets of <= SPH_BUCKET Morton-consecutive particles; the child items of a cell are
// contiguous, item 0 is the root.  skip >= 0: big cell, skip = index of its first child item, lo = number
// of child items; skip < 0: bucket of -skip particles starting at sorted index lo.
#define PR_REC 16
#define SPH_BUCKET 16       // <= 32 (one lane stages one member); 16 measured best on C4/C5 (32: +11 %, 8: +14 %)
struct __align__(16) SearchItem {
    float bmin[3], bmax[3];     // box of the particles below, rounded OUTWARD to FP32 (pruning only)
    float hmax;                 // largest smoothing length below, rounded up
    float pad;
    int skip, lo;
    int pad2[2];
};

// Gravity records (gravity.cu): one per octree cell and per leaf, the children of a cell contiguous.
// GravRec: centre of mass (or particle position) and G * mass.  GravMeta: first = index of the first
// child record (cell), or first sorted particle (multi-particle leaf); info = count << 8 | kind,
// kind (5 bits) = level of the cell (0..21), GR_LEAF1 = single particle, GR_LEAFN = several particles in one
// leaf (equal keys at the deepest level).
struct __align__(32) GravRec {
    double x, y, z, gm;
};
struct __align__(8) GravMeta {
    int first, info;
};
#define GR_LEAF1 30
#define GR_LEAFN 31

struct Mats {
    sph_material m[SPH_MAX_MAT];
};

// All device pointers of one context. Passed by value to kernels (plain POD).
struct Dev {
    int D, L, flags, cap;       // cap = max_neighbours
    int n;
    int n_des;
    int r_lo, r_hi;             // sorted range whose partner lists, pair sums and walks THIS rank computes (0, n on one GPU)
    double theta2, G, eps2, av_alpha, av_beta, av_eps;
    double as_eps, as_n, as_mpd, xsph;
    // ---- master state, original order ----
    double *x[3], *v[3], *m, *rho, *u, *S[6], *dmg, *h;
    int *mat, *n_act;
    i64 *flaw_off;
    double *flaw_eps;
    // ---- RK2 base copy (x v rho u S dmg: 15 arrays contiguous) ----
    double *q0;
    double *rk[3];              // k1, k2, k3 of sph_step_rk3, original order, 15 arrays each (SPH_F_RK3)
    double *ag_keep[3];         // last walked gravitational acceleration, original order (gravity_every > 1)
    int *rk_nact, *rk_nmax;     // activated flaws of the newest evaluation / maximum over the step
    double *h0;                 // smoothing lengths at the start of sph_step_rk3 (given back when the step is rejected)
    // ---- sorted working copies ----
    double *sx[3], *sv[3], *sm, *srho, *su, *sS[6], *sdmg, *sh;
    int *smat;
    // ---- order ----
    u64 *key[2];
    int *idx[2];                // idx[cur][i] = original index of sorted i (perm)
    u64 *keys;                  // sorted keys (alias of key[cur] after the sort)
    int *perm;                  // alias of idx[cur]
    int *iperm;                 // inverse: iperm[original] = sorted index (written by the reorder)
    unsigned *hist;             // radix histograms
    double *partial;            // bbox partials
    DevRoot *root;
    DevStatus *status;
    // ---- tree (depth-first order) ----
    u64 *nkey[2];
    int *nhi[2];
    int *nlevel, *nlo, *nhi_s;  // per node
    int *nskip;                 // first node after the subtree (pre-order)
    int *nparent, *ncc, *nready; // parent cell (-1 root), number of child CELLS, children finished (k_moments)
    int *nord;                  // search tree: ordinal of a big cell among its parent's items
    int *child;                 // NC per node: >=0 node, -1 empty, -2 leaf
    int *child_lo;              // NC+1 per node
    double *nmass, *ncom[3], *nbmin[3], *nbmax[3], *nhmax, *ns2;
    // ---- search tree of the partner search ----
    SearchItem *items;          // up to 2n records
    GravRec *grec;              // n + n_nodes records
    GravMeta *gmeta;
    unsigned *gcnt, *gfirst;    // per cell: number of child records, index of the first
    double *gthr;               // 32 acceptance thresholds on r^2 (eq. 50), by record kind
    unsigned *bbox_done;        // blocks of k_bbox that have finished (0 between launches)
    u64 *bmark, *bscan;         // n+1 each: bucket starts (parent | ordinal | length); child-item counts and their scan
    u64 *scan_tmp;              // scratch of the prefix sums
    // ---- partner lists: group-transposed, nb[(g*cap + k)*32 + SPH_NB_POS(lane)] (sorted indices) ----
    int *nb;
    int *nb_cnt;
    int *own_cnt;               // n_a of eq. 73
    // ---- pre-pass ----
    double *p, *cs;             // pressure, sound speed
    double *prec;               // PR_REC doubles per particle: x3 v3 rho m/rho cs h sigma/rho^2 (6)
    // ---- rates, sorted order ----
    double *drho, *dv[3], *du, *dS[6], *ddmg, *ag[3], *strain;
    double *dxs[3];             // XSPH term of eq. 40 (only with SPH_F_XSPH)
    double *gradv[9], *Cten[9]; // velocity gradient (eq. 42) and correction tensor (eq. 43), row-major (only with SPH_F_EXPORT_GRADV)
    int *n_act_new;
    // ---- sharding: the ranks' failure flags travel with the rates (api.cu exchange_rates) ----
    unsigned char *xstat;       // world * slice bytes; rank r's slot = 3 ints at byte r * slice
    unsigned char *xbuf;        // pack buffer of the ONE all-gather per exchange: world blocks of slice * (bytes per particle)
};

struct SphTiming;   // api.cu: CUDA-event pairs around the stages (sph_timing_*)

struct sph_ctx {
    sph_config cfg;
    Dev d;
    Mats mats;
    cudaStream_t stream;
    void *ws;
    size_t ws_bytes;
    int have_state, have_tree, have_lists, have_rates;
    i64 launches;
    int count_work;             // sph_counters_enable: the gravity walk keeps its work counters
    // Morton-range sharding over the GPUs of a node (sph_set_partition): rank, ranks, slice length, the caller's
    // all-gather, and whether an evaluation is collecting its arrays for ONE exchange at its end
    int rank, world;
    i64 slice;
    sph_exchange_fn xfn;
    void *xuser;
    int in_evaluate;
    int q0_live;                // inside sph_step / sph_step_host / sph_step_rk3: Dev::q0 holds the base copy (no host download)
    int sort_cur;
    SphTiming *timing;          // NULL unless sph_timing_enable(ctx, 1)
    // sph_step as a CUDA graph: captured when the same dt is asked for twice in a row, replayed after
    cudaGraphExec_t step_graph;
    double graph_dt, last_dt;
    i64 graph_launches;
    int graphs_off;
    i64 step_no;                // sph_step calls since the last upload (gravity_every)
    int grav_reuse;             // set by sph_step: sph_evaluate takes the stored accelerations
    // sph_step_host: the upload runs on a second stream beside the geometric stages of the first evaluation
    cudaStream_t copy_stream;
    cudaEvent_t ev_fork, ev_geom, ev_rest;
    int split_gather;           // sph_stage_order gathers positions, masses and h only (sph_stage_gather_rest follows later)
    cudaGraphExec_t hstep_graph;
    double hgraph_dt, hlast_dt;
    i64 hgraph_launches;
    sph_state_in hgraph_src, hlast_src;
    char err[512];
};

// RAII bracket of one stage: two event records on ctx->stream when timing is enabled, nothing otherwise.
void sph_timing_begin(sph_ctx *ctx, int stage);
void sph_timing_end(sph_ctx *ctx, int stage);
struct StageTimer {
    sph_ctx *c; int stage;
    StageTimer(sph_ctx *ctx, int st) : c(ctx), stage(st) { if (c->timing) sph_timing_begin(c, stage); }
    ~StageTimer() { if (c->timing) sph_timing_end(c, stage); }
};

// Position of a lane's entry inside the 32 entries of a list row: lanes 0, 4, 8, ... 28 first, then 1, 5, ..., so that the
// 8 lanes that stage one quarter of a row's records in the pair kernel (lanes r = q + 4 t) find their 8 partner indices in
// 32 contiguous bytes.  Rows k < (largest count of the group) are complete: lanes with fewer partners hold their own
// index there (a valid record that is read and ignored).
#define SPH_NB_POS(lane) ((((lane) & 3) << 3) | ((lane) >> 2))

static inline int sph_ceil_div(i64 a, i64 b) { return (int)((a + b - 1) / b); }

// ---- sort.cu ----
// LSD radix sort of (key, val) pairs, `bits` low key bits significant. n is read on the host
// (n_host) or, if n_dev != NULL, from device memory (kernels early-exit; grids sized for n_host).
// Result ends in key[*cur], val[*cur].
void sph_radix_sort(sph_ctx *ctx, u64 *key[2], int *val[2], int n_host, const int *n_dev, int bits, int *cur);
void sph_sort_init();
size_t sph_sort_ws_words(i64 n);   // words of Dev::hist the sort needs for n keys

// ---- scan.cu ---- exclusive prefix sums (in == out allowed); scratch[ceil(n/2048)] = grand total
void sph_scan_u32(sph_ctx *ctx, const unsigned *in, unsigned *out, i64 n, unsigned *scratch);
void sph_scan_u64(sph_ctx *ctx, const u64 *in, u64 *out, i64 n, u64 *scratch);
size_t sph_scan_scratch_elems(i64 n);

// ---- per-stage entry points (each enqueues kernels on ctx->stream) ----
void sph_stage_order(sph_ctx *ctx);     // A1 + A2
void sph_stage_gather_rest(sph_ctx *ctx);   // second half of A2 when ctx->split_gather was set for sph_stage_order
void sph_stage_tree(sph_ctx *ctx);      // A3 + A4
void sph_stage_neigh(sph_ctx *ctx);     // A5
void sph_stage_rhs(sph_ctx *ctx);       // A6-A10
void sph_stage_gravity(sph_ctx *ctx);   // A11
void sph_stage_writeback_h(sph_ctx *ctx);
void sph_launch_moments(sph_ctx *ctx, int hmax_only);   // tree.cu: pseudo-particles bottom-up, one launch

// ---- exact-order arithmetic for the floating-point decisions (never contracted to FMA) ----
__device__ __forceinline__ double sph_r2_exact(double dx, double dy, double dz, int D) {
    double r2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
    if (D == 3) r2 = __dadd_rn(r2, __dmul_rn(dz, dz));
    return r2;
}
