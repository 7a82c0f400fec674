/*
 * sph.h -- C ABI of the B200-native SPH right-hand-side library (libsph_b200.so).
 *
 * The library evaluates, on one NVIDIA B200 (sm_100a), the per-timestep right-hand side of
 * the solid-body SPH method with Barnes-Hut self-gravity of Schaefer et al.,
 * arXiv:1604.03290 ("PAPER.md" below = /root/reference/PAPER.md of the build):
 *
 *   tree build -> pseudo-particles -> interaction-partner search -> SPH sums -> self-gravity
 *   (the sub-step list of PAPER.md:693, section 6.2), plus the predictor-corrector step of
 *   PAPER.md:388-394.
 *
 * Conventions
 *   - All real data are FP64, indices int32, Morton keys uint64.  Arrays are structure-of-arrays,
 *     one contiguous array per quantity, length n unless stated otherwise.
 *   - Users see ORIGINAL particle order everywhere.  The Morton-sorted order is internal.
 *   - `h` is the paper's smoothing length: the kernel vanishes for r/h > 1 (eq. 25).
 *   - Stress components are stored as S[6] = (xx, xy, xz, yy, yz, zz); in 2-D only xx, xy, yy are used.
 *   - The damage state variable is dmg = d^(1/3) in [0, 1] (eq. 46).
 *   - Every pointer argument is documented as HOST or DEVICE.  The library never allocates device
 *     memory: the caller passes one device workspace of sph_workspace_bytes() bytes and owns it.
 *   - All calls return an int status (0 = SPH_OK, negative = error); nothing throws or aborts.
 *     Work is enqueued asynchronously on the stream given to sph_create; calls that return data to
 *     the HOST (sph_download with dst_is_device = 0, the sph_get_* calls, sph_sync) synchronise that
 *     stream and also report device-side failures (list overflow, stack overflow) recorded earlier.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns SPH_ERR_CUDA.
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sph_ctx sph_ctx; /* opaque; host object created by sph_create */

enum {
    SPH_OK = 0,
    SPH_ERR_ARG = -1,                /* bad argument (NULL, n < 1, dim not 2/3, theta >= 1/sqrt(dim), ...) */
    SPH_ERR_STATE = -2,              /* call order: e.g. sph_rhs before sph_find_neighbours */
    SPH_ERR_WORKSPACE = -3,          /* workspace too small or misaligned (256 B) */
    SPH_ERR_NEIGHBOUR_OVERFLOW = -4, /* a particle has more than max_neighbours partners */
    SPH_ERR_TREE_DEPTH = -5,         /* a traversal stack was exhausted: the gravity walk's or the partner search's (guards: the
                                        pop policies bound both stacks for every theta and particle distribution, see
                                        csrc/gravity.cu and csrc/neigh.cu); sph_last_error names the kernel */
    SPH_ERR_CUDA = -6                /* CUDA runtime error or no device; see sph_last_error */
};

enum {
    SPH_F_SOLID = 1,         /* deviatoric stress S, correction tensor, dS/dt */
    SPH_F_PLASTIC = 2,       /* von Mises limiter */
    SPH_F_DAMAGE = 4,        /* Grady-Kipp damage */
    SPH_F_GRAVITY = 8,       /* Barnes-Hut self-gravity */
    SPH_F_VARIABLE_H = 16,   /* mean smoothing length per pair + eq. 73 update */
    SPH_F_DENSITY_SUM = 32,  /* rho by kernel sum, eq. 28, instead of continuity */
    SPH_F_ART_STRESS = 64,   /* artificial stress against the tensile instability (eqs. 35-38) */
    SPH_F_XSPH = 128,        /* particles move with the XSPH-smoothed velocity (eq. 40) */
    SPH_F_RK3 = 256,         /* reserve the rate buffers of the embedded Runge-Kutta step (sph_step_rk3) */
    SPH_F_EXPORT_GRADV = 512 /* keep the velocity gradient of eq. 42 and the correction tensor of eqs. 43-44 of the last
                                evaluation (18 n doubles more workspace) so that sph_download can return them */
};

enum { SPH_EOS_IDEAL_GAS = 0, SPH_EOS_MURNAGHAN = 1, SPH_EOS_TILLOTSON = 2 };

/* Material parameters. Murnaghan: PAPER.md:120 (eq. 13). Tillotson: PAPER.md:128-137 (eqs. 14-15).
 * mu: shear modulus (eq. 7); Y0: von Mises yield stress (eq. 17), 0 = no limiter for this material;
 * brittle: 1 = damage model applies to this material. */
typedef struct {
    int32_t eos;
    int32_t brittle;
    double rho0, K0, nM, gamma;
    double tA, tB, tE0, tEiv, tEcv, ta, tb, talpha, tbeta;
    double mu, Y0;
} sph_material;

typedef struct {
    int32_t dim;            /* 2 or 3 */
    int32_t flags;          /* SPH_F_* */
    int32_t n_materials;
    int32_t morton_bits;    /* bits per dimension of the Morton key, 1..21; 0 = default 21 */
    int32_t max_neighbours; /* capacity of one interaction list (PAPER.md:481 interactionsList); 0 = 128 */
    int32_t n_des;          /* desired partner count of eq. 73 */
    int32_t h_iters;        /* eq.-73 updates per sph_find_neighbours (only with SPH_F_VARIABLE_H) */
    int32_t gravity_every;  /* gravity/hydro decoupling: sph_step walks the tree for self-gravity only in
                               every gravity_every-th step and reuses the stored accelerations in between; 0 or 1 =
                               every step.  sph_gravity and sph_evaluate always walk. */
    int64_t n;              /* particles */
    int64_t n_flaws;        /* total flaw thresholds (length of flaw_eps); 0 without damage */
    double theta;           /* opening angle of eq. 50; must be < 1/sqrt(dim) */
    double G;               /* gravitational constant */
    double eps_soft;        /* Plummer softening length added in eq. 51 */
    double av_alpha, av_beta, av_eps; /* artificial viscosity, eqs. 32-33 */
    double as_eps, as_n, as_mpd;      /* artificial stress: factor eps_s (eq. 37), exponent n and mean particle
                                         distance dmpd of f = W(r)/W(dmpd) (eq. 38); used with SPH_F_ART_STRESS */
    double xsph;                      /* XSPH factor x_sph of eq. 40; used with SPH_F_XSPH */
} sph_config;

/* Input state, original order.  NULL members are left unchanged (or zero on first upload).
 * x[2], v[2] and the z components of S are ignored when dim == 2.
 * flaw_off has n+1 entries (CSR into flaw_eps, thresholds ascending per particle; eq. 45). */
typedef struct {
    const double *x[3], *v[3], *m, *rho, *u, *S[6], *dmg, *h;
    const int32_t *mat, *n_act;
    const int64_t *flaw_off;
    const double *flaw_eps;
} sph_state_in;

/* Output buffers, original order, each of length n; NULL members are skipped.
 * State: x, v, rho, u, S, dmg, h, n_act.  Rates of the LAST evaluation: drho (eq. 29), dv (eqs. 30/34,
 * SPH part only), du (eq. 31), dS (eqs. 7-10), ddmg (eq. 46, rate of dmg = d^(1/3)), ag (eq. 51,
 * gravitational acceleration), p and cs (equation of state), strain (eq. 48), n_act_new (activated
 * flaws found by the last evaluation, latched with the committed count), nb_count (partners),
 * dxs (eq. 40: the XSPH term x_sph sum_b 2 m_b/(rho_a+rho_b) (v_b - v_a) W_ab, so that dx/dt = v + dxs;
 * zero without SPH_F_XSPH); gradv[3*alpha+beta] = d v^alpha / d x^beta of eq. 42 and C[3*gamma+beta] = the
 * correction tensor of eqs. 43-44 (identity where reading U17 applies), both only with
 * SPH_F_SOLID | SPH_F_EXPORT_GRADV, zero otherwise.
 * With HOST buffers the rates are un-sorted by one kernel into workspace that sph_step and sph_rhs also use,
 * copied out, and the call synchronises once. */
typedef struct {
    double *x[3], *v[3], *rho, *u, *S[6], *dmg, *h;
    double *drho, *dv[3], *du, *dS[6], *ddmg, *ag[3], *p, *cs, *strain;
    int32_t *n_act, *n_act_new, *nb_count;
    double *dxs[3];
    double *gradv[9], *C[9];
} sph_state_out;

/* Bytes of device workspace sph_create needs for this configuration (0 on invalid config). */
size_t sph_workspace_bytes(const sph_config *cfg);

/* cfg, materials: HOST.  d_workspace: DEVICE, 256-byte aligned, >= sph_workspace_bytes(cfg).
 * cuda_stream: a cudaStream_t (NULL = default stream).  *out receives the context. */
int sph_create(const sph_config *cfg, const sph_material *materials, void *d_workspace,
               size_t workspace_bytes, void *cuda_stream, sph_ctx **out);
void sph_destroy(sph_ctx *ctx);

/* Copy particle state into the context (original order). src_is_device: 1 = DEVICE pointers,
 * 0 = HOST pointers (pinned memory makes the copy asynchronous). Invalidates tree and lists and clears
 * the device-side failures latched by evaluations of the previous state. */
int sph_upload(sph_ctx *ctx, const sph_state_in *src, int src_is_device);

/* A1-A4: bounding cube (eq. 67) -> Morton keys -> radix sort + SoA reorder -> octree topology ->
 * pseudo-particles (mass, centre of mass) with bounding boxes and hmax. */
int sph_build_tree(sph_ctx *ctx);

/* A5: interaction partners b != a with r_ab < h, or r_ab < (h_a+h_b)/2 with
 * SPH_F_VARIABLE_H (eq. 72), preceded by h_iters updates of eq. 73. Needs sph_build_tree. */
int sph_find_neighbours(sph_ctx *ctx);

/* A6-A10: [density sum eq. 28] -> EoS, limiter, damaged stress -> pair sums eqs. 29-34, 41-44 ->
 * dS/dt (eqs. 7-10) and damage rate (eqs. 46-49). Needs tree and lists. */
int sph_rhs(sph_ctx *ctx);

/* A11: Barnes-Hut walk, eqs. 50-51, monopoles only. Needs sph_build_tree. Zero without SPH_F_GRAVITY. */
int sph_gravity(sph_ctx *ctx);

/* One complete right-hand-side evaluation: build_tree, find_neighbours, rhs, gravity. */
int sph_evaluate(sph_ctx *ctx);

/* A12: predictor-corrector step (eqs. 52-53): two complete evaluations and two updates.
 * The launch sequence of a step depends only on the configuration and dt: when the same dt is asked
 * for twice in a row the library captures the sequence into a CUDA graph and replays it on later
 * calls with that dt (same results bit for bit).  This needs a capturable stream (not the legacy
 * default stream) and no stage timing; otherwise, or with SPH_NO_GRAPH set in the environment at
 * sph_create, the kernels are launched one by one. */
int sph_step(sph_ctx *ctx, double dt);

/* sph_upload(ctx, src, 0) followed by sph_step(ctx, dt) as ONE call, for a caller that feeds every step from HOST
 * memory: the same state afterwards, bit for bit.  A second stream copies src while the first stream works: positions,
 * h and masses go first, the order, the tree, the partner search and the walk (eqs. 50-51) -- which
 * read nothing else -- run beside the copy of the other members, then those are gathered, the base copy of eq. 52 is
 * taken and the SPH sums follow (the stages of the first evaluation are independent of one another apart from that
 * order).  src: HOST pointers as for sph_upload (NULL members keep their device values); page-locked buffers are needed
 * for the copies to overlap.  The call returns when everything is enqueued: src must stay unchanged until a call
 * that synchronises (sph_sync, sph_download to host buffers).  The same src pointers and dt twice in a row: the whole
 * sequence, copies included, is captured into a CUDA graph and replayed on later calls.  With stage timing, decoupled
 * gravity or a partition set it is exactly sph_upload + sph_step. */
int sph_step_host(sph_ctx *ctx, const sph_state_in *src, double dt);

/* One step of the embedded Runge-Kutta scheme (eqs. 58-65): three complete
 * evaluations k1 = f(q), k2 = f(q + dt/2 k1), k3 = f(q - dt k1 + 2 dt k2); third-order result
 * q + dt (k1 + 4 k2 + k3)/6 (eq. 58), midpoint result q + dt k2 (eq. 62), error estimate
 * eps_err = max |q_mm - q_rk3| / |q + dt k1| over all particles and integrated quantities with a
 * non-zero denominator (eq. 63).  eps_err <= eps_des: the state becomes the third-order result and
 * dt_new = dt |eps_des/eps_err|^0.3 (eq. 64); otherwise the state is left unchanged and
 * dt_new = 0.9 dt |eps_des/eps_err|^(1/4) (eq. 65).  Stage states get the post-update rules of
 * sph_step; n_act is committed (maximum over the three evaluations) only on acceptance.
 * A rejected step gives back the whole state, including the smoothing lengths that eq. 73 rewrote during the
 * three evaluations.  A state or rate that is not finite gives eps_err = +inf: rejected, dt_new = 0.
 * A device-side failure of one of the evaluations (list overflow) is returned and nothing is accepted.
 * out (HOST double[3]) = eps_err, dt_new, accepted (1.0 / 0.0).  Needs SPH_F_RK3.  Synchronises. */
int sph_step_rk3(sph_ctx *ctx, double dt, double eps_des, double *out);

/* Upper limits of the next time step from the rates of the LAST complete evaluation:
 *   out[0] = min_a 0.2 h_a / |dv_a/dt|       (eq. 54; the acceleration includes self-gravity)
 *   out[1] = min_a 0.7 h_a / c_s,a           (eq. 55, Courant)
 *   out[2] = min_a,q 0.7 |q_a| / |dq_a/dt|   (eq. 57) over q = rho (not with SPH_F_DENSITY_SUM), u, the
 *            components of S (SPH_F_SOLID) and dmg (SPH_F_DAMAGE); entries with q = 0 or dq/dt = 0 are skipped
 *   out[3] = the smallest of the three       (eq. 56 with eq. 57)
 * A limit that no particle sets is +infinity; a NaN state or rate gives the limit 0.  Without SPH_F_GRAVITY
 * (or before sph_gravity) eq. 54 takes the SPH acceleration alone.  out: HOST double[4].  Synchronises and
 * reports device-side failures of the evaluation. */
int sph_timestep(sph_ctx *ctx, double *out);

/* Copy state and/or the rates of the last evaluation out, original order.
 * dst_is_device: 1 = DEVICE buffers (asynchronous), 0 = HOST buffers (synchronises). */
int sph_download(sph_ctx *ctx, const sph_state_out *dst, int dst_is_device);

/* ---- Morton-range sharding over the GPUs of one node (the paper: "future work") ----
 * One process and one context per GPU; every rank uploads the SAME full state.  The cheap global stages (keys, sort,
 * reorder, octree, pseudo-particles, pre-pass, update) run replicated on every rank; the expensive per-particle stages
 * (partner search, pair sums, gravity walk) run only for the rank's contiguous slice of the Morton order; then ONE
 * all-gather per evaluation completes the rate arrays on every rank (no reduction: every rate is written by exactly one
 * rank, and a particle's arithmetic does not depend on the rank that does it, so the sharded result equals the
 * single-GPU result bit for bit).
 *
 * sph_partition (host only): slice = ceil(n / world) rounded up to a multiple of 32 (warp groups never straddle two
 * ranks); rank r owns the sorted indices [lo, hi) = [min(n, r slice), min(n, (r + 1) slice)).  Any pointer may be NULL.
 *
 * sph_exchange_fn: the caller's in-place all-gather, called by the library at the end of sph_evaluate (or of sph_rhs /
 * sph_gravity when called alone) with n_arrays DEVICE arrays of world * slice_elems elements of elem_bytes[k] bytes each;
 * rank r has filled elements [r slice_elems, (r + 1) slice_elems) of every array; on return (stream-ordered on
 * cuda_stream) every array must be complete on every rank.  Return 0, or non-zero to fail the call with SPH_ERR_CUDA.
 * paper_1604_03290_b200/binding.py supplies one built on torch.distributed (NCCL over NVLink).
 *
 * sph_set_partition: before the next evaluation; world = 1 (or fn = NULL with world = 1) switches sharding off.
 * With SPH_F_DENSITY_SUM, or SPH_F_VARIABLE_H with h_iters > 0, the partner search and the density sum stay replicated
 * (every particle's density and smoothing length feed its partners' sums); the pair sums and the walk are still sharded.
 * sph_get_neighbours then returns the lists of the rank's own slice only; the work counters are per rank.  sph_step does
 * not capture CUDA graphs while a partition is set.
 * The library packs the rank's slices of all exchanged arrays into one contiguous block first (one kernel), so the
 * function is called with n_arrays = 1 -- ONE collective per evaluation, elem_bytes[0] = the bytes per particle of all
 * arrays together (137 for a solid, damaged, self-gravitating run) -- and copies the other ranks' blocks back into the
 * arrays afterwards (one kernel); a conforming function still handles any n_arrays.
 * The device-side failure flags (list overflow, stack guards, largest partner count) are collective: the packed block also
 * carries one byte per particle in which each rank's slot holds its flags, and after the all-gather every rank folds all
 * slots into its own, so that all ranks return the same error from the same call and sph_step_rk3 accepts or gives back a
 * step on all ranks alike. */
typedef int (*sph_exchange_fn)(void *user, void *cuda_stream, int n_arrays, void *const *arrays, const int32_t *elem_bytes,
                               int64_t slice_elems);
int sph_partition(int64_t n, int world, int rank, int64_t *lo, int64_t *hi, int64_t *slice);
int sph_set_partition(sph_ctx *ctx, int rank, int world, sph_exchange_fn fn, void *user);

/* Wait for all enqueued work; returns the first device-side failure if any. */
int sph_sync(sph_ctx *ctx);

/* ---- inspection for parity tests (HOST buffers; synchronise) ---- */
/* keys[n]: sorted Morton keys; perm[n]: perm[i] = original index of the i-th sorted particle.
 * root[4]: xmin, ymin, zmin of the root cube and its edge s0 (eq. 67). Any pointer may be NULL. */
int sph_get_order(sph_ctx *ctx, uint64_t *keys, int32_t *perm, double *root);
/* Number of internal octree nodes. */
int sph_get_tree_size(sph_ctx *ctx, int32_t *n_nodes);
/* Node list in the library's depth-first order (sorted by (lo, level)); each array n_nodes long,
 * com/bmin/bmax 3*n_nodes (node-major). child: (2^dim)*n_nodes entries: >= 0 node index,
 * -1 empty, -2 leaf; child_lo: (2^dim+1)*n_nodes boundaries into the sorted order. NULL = skip. */
int sph_get_tree(sph_ctx *ctx, int32_t *level, uint64_t *prefix, int32_t *lo, int32_t *hi,
                 double *mass, double *com, double *bmin, double *bmax, double *hmax,
                 int32_t *child, int32_t *child_lo);
/* CSR partner lists in ORIGINAL indices, ascending per particle. off[n+1]; idx[cap]. Returns
 * SPH_ERR_ARG if cap is too small (off is still filled, so off[n] tells the needed size). */
int sph_get_neighbours(sph_ctx *ctx, int64_t *off, int32_t *idx, int64_t cap);
/* Number of kernels launched by this context so far. */
int64_t sph_launch_count(sph_ctx *ctx);

/* ---- measurement ---- */
/* Stages of one right-hand-side evaluation, in the sub-step order of PAPER.md:693. */
enum {
    SPH_T_KEYS = 0,     /* A1  bounding cube (eq. 67) + Morton keys                         */
    SPH_T_SORT,         /* A2  radix sort of (key, index)                                  */
    SPH_T_REORDER,      /* A2  SoA gather into Morton order                                */
    SPH_T_TREE,         /* A3  octree topology (node discovery, node sort, child tables)   */
    SPH_T_MOMENTS,      /* A4  pseudo-particles: mass, centre of mass, boxes, hmax         */
    SPH_T_NEIGHBOURS,   /* A5  interaction-partner search (+ eq. 73)                       */
    SPH_T_DENSITY,      /* A6  density sum, eq. 28                                         */
    SPH_T_PREPASS,      /* A7  EoS, limiter, damaged stress                                */
    SPH_T_PAIRS,        /* A8-A10 pair sums + correction tensor + dS/dt + damage epilogue  */
    SPH_T_GRAVITY,      /* A11 Barnes-Hut walk                                             */
    SPH_T_UPDATE,       /* A12 predictor / corrector update                                */
    SPH_T_COUNT
};
/* on != 0: bracket every stage with a pair of CUDA events on the context's stream (two event
 * records per stage, no synchronisation); on == 0: stop and drop pending records. */
int sph_timing_enable(sph_ctx *ctx, int on);
/* Synchronises the stream and ADDS the device time [ms] and the number of kernel launches of every
 * stage bracket recorded since the last read into ms[SPH_T_COUNT] / launches[SPH_T_COUNT] (HOST). */
int sph_timing_read(sph_ctx *ctx, double *ms, int64_t *launches);
const char *sph_timing_name(int stage);
/* on != 0: the gravity walk also counts its interactions and opening tests (entries [2]-[4] of sph_get_counters;
 * the counting variant of the walk is about 15 % slower, so off by default; without it those entries read 0).  Drops a captured step graph. */
int sph_counters_enable(sph_ctx *ctx, int on);
/* Work counters of the LAST evaluation (HOST out[5]; synchronises): [0] internal nodes; [1] sum over
 * particles of the partner count; [2] sum over particles of gravity interactions (accepted pseudo-
 * particles + directly summed particles, eq. 51); [3] sum over particles of opening tests (eq. 50:
 * accepted and opened cells); [4] of those, the opened cells.  Also reports device-side failures. */
int sph_get_counters(sph_ctx *ctx, int64_t *out);
/* Dependency-free FP64 FMA throughput of the device [TFLOP/s] (the ALU roofline denominator;
 * MEASURED_PEAKS.json has no FP64 figure). stream: cudaStream_t. Synchronises. */
int sph_measure_fp64_peak(void *cuda_stream, double *tflops);
/* Streaming FP64 copy bandwidth [GB/s, read + write bytes] over `bytes` of the workspace-free
 * scratch the caller provides (DEVICE src, dst). Synchronises. */
int sph_measure_copy_bw(void *cuda_stream, const double *src, double *dst, size_t bytes, double *gbs);

/* ---- Morton keys for callers that cannot allocate device memory (root cube eq. 67) ----
 * Everything above needs a context, and a context needs a workspace the caller allocates.  A caller that has only the
 * buffers it was given -- a plug-in inside a host application that owns the GPU memory pool, a time loop that must not
 * pay the device-wide synchronisation of cudaMalloc / cudaFree, a process at its memory limit -- cannot get one.  This one
 * call serves it: root cube and Morton keys (stages A1 of sph_build_tree, the same bits) with NO workspace argument.  It
 * never calls cudaMalloc, cudaFree or any allocating routine: the scratch of the bounding-box reduction is a fixed array
 * of SPH_STATIC_SCRATCH_BYTES inside the library's device image, which every GPU that loads the library holds until the
 * process exits.
 *
 *   x, y, z   DEVICE, n doubles each, the caller's (z is ignored and may be NULL when dim == 2); read only.
 *   n         1 .. SPH_STATIC_MAX_N; anything larger is rejected with SPH_ERR_ARG and a message (the kernels index with
 *             int32 like the rest of the library, and the fixed scratch holds the partial boxes of at most 1024 blocks).
 *   dim       2 or 3.   morton_bits   bits per dimension, 1..21; 0 = 21.
 *   keys      DEVICE, n uint64, the caller's; keys[i] = key of particle i (ORIGINAL order, not sorted).
 *   root      DEVICE double[4] or NULL: xmin, ymin, zmin (0 in 2-D) and the edge s0 of the root cube.
 *   errbuf    HOST char[errbuf_len] or NULL: receives a one-line message when the call fails (empty on success).
 * Asynchronous: two kernels and a 4-byte clear are enqueued on cuda_stream (a cudaStream_t, NULL = default stream); the
 * buffers must stay valid until they have run.  Returns SPH_OK, SPH_ERR_ARG, or SPH_ERR_CUDA (no device, launch failure).
 *
 * Because the scratch is ONE array per GPU, shared by every call and every thread of the process:
 *   - calls that can overlap on the GPU (streams with no ordering between them) race on it and produce wrong keys; keep the
 *     calls on one stream or order them with events.  It shares nothing with contexts, so it may overlap with those;
 *   - it keeps the last call's contents; the call clears the one word that has to start at zero (the arrival counter of
 *     the reduction) on the stream before it launches, everything else is rewritten before it is read;
 *   - the first call on a GPU looks up the array's device address (cudaGetSymbolAddress), which may load the library's
 *     kernels onto that GPU: make that first call at set-up, with that GPU current on the calling thread, and before any
 *     stream capture begins.  The GPU that is current must be the one the stream and the buffers belong to. */
#define SPH_STATIC_MAX_N 0x3fffffff      /* 2^30 - 1 particles per call */
#define SPH_STATIC_SCRATCH_BYTES 49408   /* device memory the library's image reserves on every GPU for this call */
int sph_morton_keys_static(const double *x, const double *y, const double *z, int64_t n, int32_t dim, int32_t morton_bits,
                           void *cuda_stream, uint64_t *keys, double *root, char *errbuf, size_t errbuf_len);

const char *sph_last_error(sph_ctx *ctx);
const char *sph_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
