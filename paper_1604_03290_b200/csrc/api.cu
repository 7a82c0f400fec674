// C ABI of libsph_b200.so (declared in include/sph.h): context, workspace layout, upload/download,
// call-order checks, the predictor-corrector update (A12) and the inspection calls used by the
// parity tests.  Every compute step runs in the kernels of order.cu / tree.cu / neigh.cu / rhs.cu /
// gravity.cu; this file holds host logic and three small per-particle kernels (update, unsort).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "sph_internal.cuh"

// ------------------------------------------------------------------------------------------------
// workspace layout: one bump allocation pass, used both to size and to carve
// ------------------------------------------------------------------------------------------------
namespace {

struct Bump {
    char *base;
    size_t off;
    template <class T> T *take(size_t count) {
        off = (off + 255) & ~(size_t)255;
        T *p = base ? (T *)(base + off) : (T *)nullptr;
        off += count * sizeof(T);
        return p;
    }
};

int cfg_cap(const sph_config *c) { return c->max_neighbours > 0 ? c->max_neighbours : 128; }
int cfg_L(const sph_config *c) { return c->morton_bits > 0 ? c->morton_bits : 21; }

bool cfg_ok(const sph_config *c) {
    if (!c) return false;
    if (c->dim != 2 && c->dim != 3) return false;
    if (c->n < 1 || c->n > (int64_t)0x3fffffff) return false;
    if (c->n_materials < 1 || c->n_materials > SPH_MAX_MAT) return false;
    if (c->morton_bits < 0 || c->morton_bits > 21) return false;
    if (c->max_neighbours < 0 || c->max_neighbours > 4096) return false;
    if (c->n_flaws < 0 || c->gravity_every < 0) return false;
    if ((c->flags & SPH_F_GRAVITY) && !(c->theta >= 0.0 && c->theta * c->theta * c->dim < 1.0)) return false;
    if ((c->flags & SPH_F_VARIABLE_H) && c->h_iters > 0 && c->n_des < 1) return false;
    if ((c->flags & SPH_F_ART_STRESS) && !(c->as_mpd > 0.0 && c->as_n > 0.0 && c->as_eps >= 0.0)) return false;
    if ((c->flags & SPH_F_XSPH) && !(c->xsph >= 0.0 && c->xsph <= 1.0)) return false;
    return true;
}

// Bytes per particle of everything a sharded evaluation exchanges (the list of exchange_rates with which = 3): the
// ranks' flag slots (1), drho du (16), dv (24), dS (48, solid), ddmg strain n_act_new (20, damage), dxs (24, XSPH),
// grad v and C (144, exported), nb_cnt (4), ag (24, gravity).  Sizes the pack buffer Dev::xbuf.
int exchange_bytes_per_particle(int flags) {
    int b = 1 + 16 + 24 + 4;
    if (flags & SPH_F_SOLID) b += 48;
    if (flags & SPH_F_DAMAGE) b += 20;
    if (flags & SPH_F_XSPH) b += 24;
    if ((flags & SPH_F_SOLID) && (flags & SPH_F_EXPORT_GRADV)) b += 144;
    if (flags & SPH_F_GRAVITY) b += 24;
    return b;
}

// Fills d with pointers into base (or only measures when base == nullptr). Returns bytes used.
size_t carve(const sph_config *c, char *base, Dev *d, Mats **mats_dev) {
    Bump b{base, 0};
    const size_t n = (size_t)c->n;
    const int D = c->dim, NC = 1 << D;
    const size_t groups = (n + 31) / 32;
    Dev z;
    memset(&z, 0, sizeof(z));
    // master state: x3 v3 rho u S6 dmg contiguous (the RK2 base copy mirrors these 15 arrays)
    double *st = b.take<double>(15 * n);
    for (int a = 0; a < 3; ++a) { z.x[a] = st ? st + (size_t)a * n : nullptr; z.v[a] = st ? st + (size_t)(3 + a) * n : nullptr; }
    z.rho = st ? st + 6 * n : nullptr;
    z.u = st ? st + 7 * n : nullptr;
    for (int k = 0; k < 6; ++k) z.S[k] = st ? st + (size_t)(8 + k) * n : nullptr;
    z.dmg = st ? st + 14 * n : nullptr;
    z.m = b.take<double>(n);
    z.h = b.take<double>(n);
    z.mat = b.take<int>(n);
    z.n_act = b.take<int>(n);
    z.flaw_off = b.take<i64>(n + 1);
    z.flaw_eps = b.take<double>((size_t)std::max<int64_t>(c->n_flaws, 1));
    z.q0 = b.take<double>(15 * n);
    for (int k = 0; k < 3; ++k) z.rk[k] = b.take<double>((c->flags & SPH_F_RK3) ? 15 * n : 1);
    for (int a = 0; a < 3; ++a) z.ag_keep[a] = b.take<double>((c->gravity_every > 1) ? n : 1);
    z.rk_nact = b.take<int>((c->flags & SPH_F_RK3) ? n : 1);
    z.rk_nmax = b.take<int>((c->flags & SPH_F_RK3) ? n : 1);
    z.h0 = b.take<double>((c->flags & SPH_F_RK3) ? n : 1);
    for (int a = 0; a < 3; ++a) { z.sx[a] = b.take<double>(n); z.sv[a] = b.take<double>(n); }
    z.sm = b.take<double>(n); z.srho = b.take<double>(n); z.su = b.take<double>(n);
    for (int k = 0; k < 6; ++k) z.sS[k] = b.take<double>(n);
    z.sdmg = b.take<double>(n); z.sh = b.take<double>(n);
    z.smat = b.take<int>(n);
    for (int k = 0; k < 2; ++k) { z.key[k] = b.take<u64>(n); z.idx[k] = b.take<int>(n); }
    z.iperm = b.take<int>(n);
    z.hist = b.take<unsigned>(sph_sort_ws_words((i64)n));
    z.partial = b.take<double>(1024 * 6);
    z.root = b.take<DevRoot>(1);
    z.status = b.take<DevStatus>(1);
    for (int k = 0; k < 2; ++k) { z.nkey[k] = b.take<u64>(n); z.nhi[k] = b.take<int>(n); }
    z.nlevel = b.take<int>(n); z.nlo = b.take<int>(n); z.nhi_s = b.take<int>(n); z.nskip = b.take<int>(n);
    z.nparent = b.take<int>(n); z.ncc = b.take<int>(n); z.nready = b.take<int>(n); z.nord = b.take<int>(n);
    z.child = b.take<int>(n * NC);
    z.child_lo = b.take<int>(n * (NC + 1));
    z.nmass = b.take<double>(n);
    for (int a = 0; a < 3; ++a) { z.ncom[a] = b.take<double>(n); z.nbmin[a] = b.take<double>(n); z.nbmax[a] = b.take<double>(n); }
    z.nhmax = b.take<double>(n); z.ns2 = b.take<double>(n);
    z.items = b.take<SearchItem>(2 * n + 2);
    const size_t ngr = (c->flags & SPH_F_GRAVITY) ? 2 * n + 2 : 1;
    z.grec = b.take<GravRec>(ngr);
    z.gmeta = b.take<GravMeta>(ngr);
    z.gcnt = b.take<unsigned>((c->flags & SPH_F_GRAVITY) ? n + 1 : 1);
    z.gfirst = b.take<unsigned>((c->flags & SPH_F_GRAVITY) ? n + 1 : 1);
    z.gthr = b.take<double>(32);
    z.bbox_done = b.take<unsigned>(1);
    z.bmark = b.take<u64>(n + 1); z.bscan = b.take<u64>(n + 1);
    z.scan_tmp = b.take<u64>(sph_scan_scratch_elems((i64)n + 1) + 2);
    z.nb = b.take<int>(groups * (size_t)cfg_cap(c) * 32);
    const size_t np_ = n + SPH_RATE_PAD;                 // arrays the ranks exchange: world * slice <= n + 32 * world elements
    z.nb_cnt = b.take<int>(np_); z.own_cnt = b.take<int>(n);
    z.p = b.take<double>(n); z.cs = b.take<double>(n);
    z.prec = b.take<double>(n * PR_REC);
    z.drho = b.take<double>(np_); z.du = b.take<double>(np_); z.ddmg = b.take<double>(np_); z.strain = b.take<double>(np_);
    for (int a = 0; a < 3; ++a) { z.dv[a] = b.take<double>(np_); z.ag[a] = b.take<double>(np_); }
    for (int k = 0; k < 6; ++k) z.dS[k] = b.take<double>(np_);
    z.n_act_new = b.take<int>(np_);
    for (int a = 0; a < 3; ++a) z.dxs[a] = b.take<double>((c->flags & SPH_F_XSPH) ? np_ : 1);
    for (int k = 0; k < 9; ++k) { z.gradv[k] = b.take<double>((c->flags & SPH_F_EXPORT_GRADV) ? np_ : 1); z.Cten[k] = b.take<double>((c->flags & SPH_F_EXPORT_GRADV) ? np_ : 1); }
    z.xstat = b.take<unsigned char>(np_);
    z.xbuf = b.take<unsigned char>(np_ * (size_t)exchange_bytes_per_particle(c->flags));
    Mats *md = b.take<Mats>(1);
    if (mats_dev) *mats_dev = md;
    if (d) *d = z;
    return (b.off + 255) & ~(size_t)255;
}

int fail(sph_ctx *ctx, int code, const char *msg) {
    if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s", msg);
    return code;
}

int check_cuda(sph_ctx *ctx, const char *where) {
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) return SPH_OK;
    snprintf(ctx->err, sizeof(ctx->err), "%s: %s", where, cudaGetErrorString(e));
    return SPH_ERR_CUDA;
}

// Device-side failures latched by the kernels of the evaluations since the last sph_upload (which
// clears them): every call that has the status block on the host reports them.
int status_flags(sph_ctx *ctx, const DevStatus &st, const char *where) {
    if (st.err_nb_overflow) {
        snprintf(ctx->err, sizeof(ctx->err), "interaction list overflow: %d partners > max_neighbours %d", st.nb_max, ctx->d.cap);
        return SPH_ERR_NEIGHBOUR_OVERFLOW;
    }
    if (st.err_stack)
        return fail(ctx, SPH_ERR_TREE_DEPTH, (st.err_stack & 2) ? "partner search: descent stack exhausted (internal bound violated)"
                                                                : "gravity walk: traversal stack exhausted (internal bound violated)");
    return check_cuda(ctx, where);
}

}  // namespace

struct sph_ctx_ext {
    sph_ctx c;
    Mats *mats_dev;
};

// ------------------------------------------------------------------------------------------------
// stage timing: event pairs on the context's stream, resolved by sph_timing_read
// ------------------------------------------------------------------------------------------------
struct SphTiming {
    struct Rec { int stage; cudaEvent_t e0, e1; i64 l0, l1; };
    std::vector<Rec> pending;
    std::vector<cudaEvent_t> pool;
    cudaEvent_t get() {
        if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
        cudaEvent_t e; cudaEventCreate(&e); return e;
    }
    ~SphTiming() {
        for (auto &r : pending) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
        for (auto e : pool) cudaEventDestroy(e);
    }
};

void sph_timing_begin(sph_ctx *ctx, int stage) {
    SphTiming *t = ctx->timing;
    SphTiming::Rec r{stage, t->get(), t->get(), ctx->launches, 0};
    cudaEventRecord(r.e0, ctx->stream);
    t->pending.push_back(r);
}
void sph_timing_end(sph_ctx *ctx, int stage) {
    SphTiming *t = ctx->timing;
    for (size_t k = t->pending.size(); k-- > 0;)
        if (t->pending[k].stage == stage && t->pending[k].l1 == 0) {
            cudaEventRecord(t->pending[k].e1, ctx->stream);
            t->pending[k].l1 = ctx->launches + 1;   // +1 so that 0 means "open"
            return;
        }
}

static inline sph_ctx_ext *ext(sph_ctx *c) { return (sph_ctx_ext *)c; }

// Dev::q0 holds the base copy of a step while one of the step calls is between its first and its last enqueue.  Host
// downloads stage through q0 (sph_download), which stream order makes safe AFTER a step call has returned; a call that
// arrived while the flag is up (a future split-step API, a second thread) would overwrite the base copy, so it is refused.
struct Q0Live {
    sph_ctx *c;
    explicit Q0Live(sph_ctx *ctx) : c(ctx) { c->q0_live += 1; }
    ~Q0Live() { c->q0_live -= 1; }
};

const sph_material *sph_dev_mats(sph_ctx *ctx) { return ext(ctx)->mats_dev->m; }

// ------------------------------------------------------------------------------------------------
// small per-particle kernels
// ------------------------------------------------------------------------------------------------
// Un-sort up to UJ_MAX arrays in one launch (blockIdx.y = array): dst[perm[i]] = src[i].
#define UJ_MAX 48
struct UJob { const void *src; void *dst; int is_int; int pad; };
struct UJobs { UJob j[UJ_MAX]; };
__global__ void k_unsort_many(UJobs jobs, const int *__restrict__ perm, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const UJob jb = jobs.j[blockIdx.y];
    const int o = perm[i];
    if (jb.is_int) ((int *)jb.dst)[o] = ((const int *)jb.src)[i];
    else ((double *)jb.dst)[o] = ((const double *)jb.src)[i];
}
__global__ void k_fill_d(double *dst, double v, size_t n) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = v;
}

// A12, PAPER.md:388-394 (eqs. 52-53): q <- q0 + c * f, f = rates of the last evaluation (sorted
// order, scattered through perm), dx/dt = v of the evaluated state (eq. 39), plus the XSPH term of
// eq. 40 with SPH_F_XSPH.
// Every product and sum is rounded separately (reading O6).  After the update: dmg clamped to
// [0, (n_act/n_tot)^(1/3)] (eq. 47), S <- f_Y S (eq. 16); n_act committed only when commit != 0.
__global__ void k_update(Dev d, const sph_material *mats, double c, int commit) {
    // One thread per particle in ORIGINAL order: the base copy and the state (30 arrays) are read and written
    // coalesced, the rates of the last evaluation (Morton order) are gathered through the inverse permutation.
    // (Round 1 ran in Morton order and scattered the 30: 0.56 -> 0.4x ms on C5.)
    const int o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= d.n) return;
    const size_t n = (size_t)d.n;
    const int i = d.iperm[o];
    const double *q0 = d.q0;
    const int D = d.D;
    for (int a = 0; a < 3; ++a) {
        if (a < D) {
            double vel = d.v[a][o];
            if (d.flags & SPH_F_XSPH) vel = __dadd_rn(vel, d.dxs[a][i]);      // eq. 40
            d.x[a][o] = __dadd_rn(q0[(size_t)a * n + o], __dmul_rn(c, vel));
            d.v[a][o] = __dadd_rn(q0[(size_t)(3 + a) * n + o], __dmul_rn(c, __dadd_rn(d.dv[a][i], d.ag[a][i])));
        } else {
            d.x[a][o] = 0.0;
            d.v[a][o] = 0.0;
        }
    }
    if (!(d.flags & SPH_F_DENSITY_SUM)) d.rho[o] = __dadd_rn(q0[6 * n + o], __dmul_rn(c, d.drho[i]));
    d.u[o] = __dadd_rn(q0[7 * n + o], __dmul_rn(c, d.du[i]));
    const sph_material &mt = mats[d.mat[o]];
    if (d.flags & SPH_F_SOLID) {
        double S[6];
        for (int k = 0; k < 6; ++k) S[k] = __dadd_rn(q0[(size_t)(8 + k) * n + o], __dmul_rn(c, d.dS[k][i]));
        if ((d.flags & SPH_F_PLASTIC) && mt.Y0 > 0.0) {
            double SS;
            if (D == 3) {
                const double dg = __dadd_rn(__dadd_rn(__dmul_rn(S[0], S[0]), __dmul_rn(S[3], S[3])), __dmul_rn(S[5], S[5]));
                const double of = __dadd_rn(__dadd_rn(__dmul_rn(S[1], S[1]), __dmul_rn(S[2], S[2])), __dmul_rn(S[4], S[4]));
                SS = __dadd_rn(dg, __dmul_rn(2.0, of));
            } else {
                SS = __dadd_rn(__dadd_rn(__dmul_rn(S[0], S[0]), __dmul_rn(S[3], S[3])), __dmul_rn(2.0, __dmul_rn(S[1], S[1])));
            }
            const double J2 = __dmul_rn(0.5, SS), Y2 = __dmul_rn(mt.Y0, mt.Y0), J3 = __dmul_rn(3.0, J2);
            if (J3 > Y2) {
                const double fY = __ddiv_rn(Y2, J3);
                for (int k = 0; k < 6; ++k) S[k] = __dmul_rn(S[k], fY);
            }
        }
        for (int k = 0; k < 6; ++k) d.S[k][o] = S[k];
    }
    if (d.flags & SPH_F_DAMAGE) {
        const i64 ntot = d.flaw_off[o + 1] - d.flaw_off[o];
        const int nact = d.n_act_new[i];
        const double dmax = (ntot > 0) ? cbrt((double)nact / (double)ntot) : 0.0;
        double g = __dadd_rn(q0[14 * n + o], __dmul_rn(c, d.ddmg[i]));
        g = fmin(fmax(g, 0.0), dmax);
        d.dmg[o] = g;
        if (commit) d.n_act[o] = nact;
    }
}

// ------------------------------------------------------------------------------------------------
// embedded Runge-Kutta step, PAPER.md:416-451 (eqs. 58-65)
// ------------------------------------------------------------------------------------------------
// rates of the last evaluation -> K (original order, the 15-array layout of the state block):
// dx/dt = v (+ XSPH term, eq. 40), dv/dt = SPH + gravity, drho/dt, du/dt, dS/dt, d(dmg)/dt
__global__ void k_rk_rates(Dev d, double *K, int first) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    const size_t n = (size_t)d.n;
    const int o = d.perm[i];
    for (int a = 0; a < 3; ++a) {
        double vel = 0.0, acc = 0.0;
        if (a < d.D) {
            vel = d.v[a][o];
            if (d.flags & SPH_F_XSPH) vel = __dadd_rn(vel, d.dxs[a][i]);
            acc = __dadd_rn(d.dv[a][i], d.ag[a][i]);
        }
        K[(size_t)a * n + o] = vel;
        K[(size_t)(3 + a) * n + o] = acc;
    }
    K[6 * n + o] = (d.flags & SPH_F_DENSITY_SUM) ? 0.0 : d.drho[i];
    K[7 * n + o] = d.du[i];
    for (int k = 0; k < 6; ++k) K[(size_t)(8 + k) * n + o] = (d.flags & SPH_F_SOLID) ? d.dS[k][i] : 0.0;
    K[14 * n + o] = (d.flags & SPH_F_DAMAGE) ? d.ddmg[i] : 0.0;
    if (d.flags & SPH_F_DAMAGE) {
        const int na = d.n_act_new[i];
        d.rk_nact[o] = na;
        d.rk_nmax[o] = first ? na : max(d.rk_nmax[o], na);
    }
}

// state <- q0 + dt (c1 k1 + c2 k2 + c3 k3), term by term, every product and sum rounded separately;
// then the post-update rules of the predictor-corrector (eq. 47 clamp, eq. 16 limiter).  nterms = 1
// (eq. 60), 2 (eq. 61) or 3 (eq. 58, commit: n_act <- maximum over the three evaluations).
__global__ void k_rk_stage(Dev d, const sph_material *mats, double dt, double c1, double c2, double c3, int nterms) {
    const int o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= d.n) return;
    const size_t n = (size_t)d.n;
    const double cc[3] = {__dmul_rn(dt, c1), __dmul_rn(dt, c2), __dmul_rn(dt, c3)};
    auto comb = [&](int q) {
        double val = d.q0[(size_t)q * n + o];
        for (int t = 0; t < nterms; ++t) val = __dadd_rn(val, __dmul_rn(cc[t], d.rk[t][(size_t)q * n + o]));
        return val;
    };
    const int D = d.D;
    for (int a = 0; a < 3; ++a) {
        d.x[a][o] = (a < D) ? comb(a) : 0.0;
        d.v[a][o] = (a < D) ? comb(3 + a) : 0.0;
    }
    if (!(d.flags & SPH_F_DENSITY_SUM)) d.rho[o] = comb(6);
    d.u[o] = comb(7);
    const sph_material &mt = mats[d.mat[o]];
    if (d.flags & SPH_F_SOLID) {
        double S[6];
        for (int k = 0; k < 6; ++k) S[k] = comb(8 + k);
        if ((d.flags & SPH_F_PLASTIC) && mt.Y0 > 0.0) {
            double SS;
            if (D == 3) {
                const double dg = __dadd_rn(__dadd_rn(__dmul_rn(S[0], S[0]), __dmul_rn(S[3], S[3])), __dmul_rn(S[5], S[5]));
                const double of = __dadd_rn(__dadd_rn(__dmul_rn(S[1], S[1]), __dmul_rn(S[2], S[2])), __dmul_rn(S[4], S[4]));
                SS = __dadd_rn(dg, __dmul_rn(2.0, of));
            } else {
                SS = __dadd_rn(__dadd_rn(__dmul_rn(S[0], S[0]), __dmul_rn(S[3], S[3])), __dmul_rn(2.0, __dmul_rn(S[1], S[1])));
            }
            const double J2 = __dmul_rn(0.5, SS), Y2 = __dmul_rn(mt.Y0, mt.Y0), J3 = __dmul_rn(3.0, J2);
            if (J3 > Y2) {
                const double fY = __ddiv_rn(Y2, J3);
                for (int k = 0; k < 6; ++k) S[k] = __dmul_rn(S[k], fY);
            }
        }
        for (int k = 0; k < 6; ++k) d.S[k][o] = S[k];
    }
    if (d.flags & SPH_F_DAMAGE) {
        const i64 ntot = d.flaw_off[o + 1] - d.flaw_off[o];
        const int nact = (nterms == 3) ? d.rk_nmax[o] : d.rk_nact[o];
        const double dmax = (ntot > 0) ? cbrt((double)nact / (double)ntot) : 0.0;
        d.dmg[o] = fmin(fmax(comb(14), 0.0), dmax);
        if (nterms == 3) d.n_act[o] = nact;
    }
}

// eq. 63: max over particles and integrated quantities of |q_mm - q_rk3| / |q + dt k1| (non-zero
// denominators only); positive doubles order like their bit patterns -> atomicMax on u64
__global__ void k_rk_err_init(Dev d) { d.status->rkerr = 0ull; }
__global__ void __launch_bounds__(256) k_rk_err(Dev d, double dt) {
    const int o = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t n = (size_t)d.n;
    const double inf = __longlong_as_double(0x7ff0000000000000ll);
    double e = 0.0;
    if (o < d.n) {
        for (int q = 0; q < 15; ++q) {
            if ((q < 3 && q >= d.D) || (q >= 3 && q < 6 && q - 3 >= d.D)) continue;
            if (q == 6 && (d.flags & SPH_F_DENSITY_SUM)) continue;
            if (q >= 8 && q < 14 && !(d.flags & SPH_F_SOLID)) continue;
            if (d.D == 2 && (q == 10 || q == 12 || q == 13)) continue;
            if (q == 14 && !(d.flags & SPH_F_DAMAGE)) continue;
            const double q0 = d.q0[(size_t)q * n + o], k1 = d.rk[0][(size_t)q * n + o];
            const double k2 = d.rk[1][(size_t)q * n + o], k3 = d.rk[2][(size_t)q * n + o];
            const double s = __dadd_rn(__dadd_rn(__ddiv_rn(k1, 6.0), __ddiv_rn(__dmul_rn(4.0, k2), 6.0)), __ddiv_rn(k3, 6.0));
            const double q3 = __dadd_rn(q0, __dmul_rn(dt, s));                       // eq. 58
            const double qm = __dadd_rn(q0, __dmul_rn(dt, k2));                      // eq. 62
            const double den = fabs(__dadd_rn(q0, __dmul_rn(dt, k1)));
            const double num = fabs(__dsub_rn(qm, q3));
            if (!(den == den) || !(num == num) || isinf(den) || isinf(num)) e = inf;  // a state or rate that blew up: reject
            else if (den > 0.0) e = fmax(e, __ddiv_rn(num, den));                      // eq. 63
        }
    }
    for (int off = 16; off > 0; off >>= 1) e = fmax(e, __shfl_xor_sync(0xffffffffu, e, off));
    __shared__ double s_e[8];
    if ((threadIdx.x & 31) == 0) s_e[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) e = fmax(e, s_e[w]);
        atomicMax(&d.status->rkerr, (u64)__double_as_longlong(e));
    }
}

// gravity/hydro decoupling (reading U31): keep / take the walked accelerations, original order
__global__ void k_ag_keep(Dev d) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    const int o = d.perm[i];
    for (int a = 0; a < 3; ++a) d.ag_keep[a][o] = d.ag[a][i];
}
__global__ void k_ag_take(Dev d) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    const int o = d.perm[i];
    for (int a = 0; a < 3; ++a) d.ag[a][i] = d.ag_keep[a][o];
}

// PAPER.md:396-414 (eqs. 54-57): time-step limits, one min-reduction over the particles (sorted order).
// Positive doubles order like their bit patterns, so the block minima are combined with atomicMin on u64.
__global__ void k_dtlim_init(Dev d) {
    if (threadIdx.x < 3) d.status->dtlim[threadIdx.x] = 0x7ff0000000000000ull;
}
__global__ void __launch_bounds__(256) k_dtlim(Dev d, int with_ag) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const double inf = __longlong_as_double(0x7ff0000000000000ll);
    double t[3] = {inf, inf, inf};
    if (i < d.n) {
        const double h = d.sh[i];
        double a2 = 0.0;
        for (int a = 0; a < d.D; ++a) { const double acc = with_ag ? d.dv[a][i] + d.ag[a][i] : d.dv[a][i]; a2 += acc * acc; }
        // a NaN state or rate gives the limit 0 (fmin would drop it and the blow-up would go unseen)
        if (!(a2 == a2)) t[0] = 0.0;
        else if (a2 > 0.0) t[0] = 0.2 * h / sqrt(a2);                  // eq. 54
        const double cs = d.cs[i];
        if (!(cs == cs)) t[1] = 0.0;
        else if (cs > 0.0) t[1] = 0.7 * h / cs;                         // eq. 55
        auto lim = [&](double q, double dq) {                          // eq. 57
            if (!(q == q) || !(dq == dq)) t[2] = 0.0;
            else if (q != 0.0 && dq != 0.0) t[2] = fmin(t[2], 0.7 * fabs(q) / fabs(dq));
        };
        if (!(d.flags & SPH_F_DENSITY_SUM)) lim(d.srho[i], d.drho[i]);
        lim(d.su[i], d.du[i]);
        if (d.flags & SPH_F_SOLID) {
            for (int k = 0; k < 6; ++k) {
                if (d.D == 2 && (k == 2 || k == 4 || k == 5)) continue;
                lim(d.sS[k][i], d.dS[k][i]);
            }
        }
        if (d.flags & SPH_F_DAMAGE) lim(d.sdmg[i], d.ddmg[i]);
    }
    __shared__ double s_min[3][8];
    for (int k = 0; k < 3; ++k) {
        double v = t[k];
        for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
        if ((threadIdx.x & 31) == 0) s_min[k][threadIdx.x >> 5] = v;
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        double v = s_min[threadIdx.x][0];
        for (int w = 1; w < 8; ++w) v = fmin(v, s_min[threadIdx.x][w]);
        atomicMin(&d.status->dtlim[threadIdx.x], (u64)__double_as_longlong(v));
    }
}

// ------------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------------
extern "C" {

size_t sph_workspace_bytes(const sph_config *cfg) {
    if (!cfg_ok(cfg)) return 0;
    return carve(cfg, nullptr, nullptr, nullptr);
}

// the captured steps no longer describe what a step launches
static void drop_graphs(sph_ctx *ctx) {
    if (ctx->step_graph) { cudaGraphExecDestroy(ctx->step_graph); ctx->step_graph = nullptr; }
    if (ctx->hstep_graph) { cudaGraphExecDestroy(ctx->hstep_graph); ctx->hstep_graph = nullptr; }
    ctx->last_dt = ctx->graph_dt = -1.0;
    ctx->hlast_dt = ctx->hgraph_dt = -1.0;
}

int sph_create(const sph_config *cfg, const sph_material *materials, void *d_workspace, size_t workspace_bytes,
               void *cuda_stream, sph_ctx **out) {
    if (!out) return SPH_ERR_ARG;
    *out = nullptr;
    if (!cfg_ok(cfg) || !materials) return SPH_ERR_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return SPH_ERR_CUDA; }
    if (!d_workspace || ((uintptr_t)d_workspace & 255)) return SPH_ERR_WORKSPACE;
    if (workspace_bytes < carve(cfg, nullptr, nullptr, nullptr)) return SPH_ERR_WORKSPACE;
    sph_ctx_ext *e = new (std::nothrow) sph_ctx_ext();
    if (!e) return SPH_ERR_ARG;
    memset(e, 0, sizeof(*e));
    sph_ctx *c = &e->c;
    c->cfg = *cfg;
    c->stream = (cudaStream_t)cuda_stream;
    c->ws = d_workspace;
    c->ws_bytes = workspace_bytes;
    carve(cfg, (char *)d_workspace, &c->d, &e->mats_dev);
    Dev &d = c->d;
    d.D = cfg->dim; d.L = cfg_L(cfg); d.flags = cfg->flags; d.cap = cfg_cap(cfg);
    d.n = (int)cfg->n; d.n_des = cfg->n_des;
    d.r_lo = 0; d.r_hi = d.n;
    c->rank = 0; c->world = 1; c->slice = cfg->n; c->xfn = nullptr; c->xuser = nullptr; c->in_evaluate = 0;
    d.theta2 = cfg->theta * cfg->theta;
    d.G = cfg->G;
    d.eps2 = cfg->eps_soft * cfg->eps_soft;
    d.av_alpha = cfg->av_alpha; d.av_beta = cfg->av_beta; d.av_eps = cfg->av_eps;
    d.as_eps = cfg->as_eps; d.as_n = cfg->as_n; d.as_mpd = cfg->as_mpd; d.xsph = cfg->xsph;
    memset(&c->mats, 0, sizeof(c->mats));
    for (int k = 0; k < cfg->n_materials; ++k) c->mats.m[k] = materials[k];
    cudaMemcpyAsync(e->mats_dev, &c->mats, sizeof(Mats), cudaMemcpyHostToDevice, c->stream);
    cudaMemsetAsync(d.status, 0, sizeof(DevStatus), c->stream);
    cudaMemsetAsync(d.bbox_done, 0, sizeof(unsigned), c->stream);
    // defaults for state members never uploaded
    const size_t n = (size_t)d.n;
    cudaMemsetAsync(d.x[0], 0, 15 * n * sizeof(double), c->stream);
    cudaMemsetAsync(d.m, 0, n * sizeof(double), c->stream);
    cudaMemsetAsync(d.h, 0, n * sizeof(double), c->stream);
    cudaMemsetAsync(d.mat, 0, n * sizeof(int), c->stream);
    cudaMemsetAsync(d.n_act, 0, n * sizeof(int), c->stream);
    cudaMemsetAsync(d.flaw_off, 0, (n + 1) * sizeof(i64), c->stream);
    for (int a = 0; a < 3; ++a) cudaMemsetAsync(d.ag[a], 0, n * sizeof(double), c->stream);   // read as 0 until a walk fills it
    cudaStreamSynchronize(c->stream);   // c->mats is pageable host memory: finish the copy now
    sph_sort_init();
    c->step_graph = nullptr;
    c->last_dt = c->graph_dt = -1.0;
    c->hstep_graph = nullptr;
    c->hlast_dt = c->hgraph_dt = -1.0;
    c->graphs_off = (getenv("SPH_NO_GRAPH") != nullptr);
    cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
    cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&c->ev_geom, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&c->ev_rest, cudaEventDisableTiming);
    int rc = check_cuda(c, "sph_create");
    if (rc != SPH_OK) { sph_destroy(c); return rc; }
    *out = c;
    return SPH_OK;
}

void sph_destroy(sph_ctx *ctx) {
    if (!ctx) return;
    cudaStreamSynchronize(ctx->stream);
    if (ctx->copy_stream) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamDestroy(ctx->copy_stream); }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_geom) cudaEventDestroy(ctx->ev_geom);
    if (ctx->ev_rest) cudaEventDestroy(ctx->ev_rest);
    drop_graphs(ctx);
    delete ctx->timing;
    delete ext(ctx);
}

int sph_timing_enable(sph_ctx *ctx, int on) {
    if (!ctx) return SPH_ERR_ARG;
    if (on && !ctx->timing) ctx->timing = new (std::nothrow) SphTiming();
    if (!on && ctx->timing) { cudaStreamSynchronize(ctx->stream); delete ctx->timing; ctx->timing = nullptr; }
    return SPH_OK;
}

int sph_timing_read(sph_ctx *ctx, double *ms, int64_t *launches) {
    if (!ctx || !ms || !launches) return SPH_ERR_ARG;
    if (!ctx->timing) return fail(ctx, SPH_ERR_STATE, "sph_timing_read before sph_timing_enable");
    if (cudaStreamSynchronize(ctx->stream) != cudaSuccess) return check_cuda(ctx, "sph_timing_read");
    SphTiming *t = ctx->timing;
    for (auto &r : t->pending) {
        if (r.l1 != 0) {
            float e = 0.f;
            if (cudaEventElapsedTime(&e, r.e0, r.e1) == cudaSuccess && r.stage >= 0 && r.stage < SPH_T_COUNT) {
                ms[r.stage] += (double)e;
                launches[r.stage] += (r.l1 - 1) - r.l0;
            }
        }
        t->pool.push_back(r.e0); t->pool.push_back(r.e1);
    }
    t->pending.clear();
    return check_cuda(ctx, "sph_timing_read");
}

const char *sph_timing_name(int stage) {
    static const char *names[SPH_T_COUNT] = {"keys", "sort", "reorder", "tree", "moments", "neighbours",
                                             "density", "prepass", "pairs", "gravity", "update"};
    return (stage >= 0 && stage < SPH_T_COUNT) ? names[stage] : "?";
}

int sph_counters_enable(sph_ctx *ctx, int on) {
    if (!ctx) return SPH_ERR_ARG;
    ctx->count_work = on ? 1 : 0;
    drop_graphs(ctx);                        // another kernel variant
    return SPH_OK;
}

int sph_get_counters(sph_ctx *ctx, int64_t *out) {
    if (!ctx || !out) return SPH_ERR_ARG;
    DevStatus st;
    cudaMemcpyAsync(&st, ctx->d.status, sizeof(st), cudaMemcpyDeviceToHost, ctx->stream);
    cudaStreamSynchronize(ctx->stream);
    out[0] = st.n_nodes; out[1] = (int64_t)st.n_pairs; out[2] = (int64_t)st.n_inter; out[3] = (int64_t)st.n_visit;
    out[4] = (int64_t)st.n_open;
    return status_flags(ctx, st, "sph_get_counters");
}

int sph_step_rk3(sph_ctx *ctx, double dt, double eps_des, double *out) {
    if (!ctx || !out) return SPH_ERR_ARG;
    if (!(ctx->d.flags & SPH_F_RK3)) return fail(ctx, SPH_ERR_STATE, "sph_step_rk3 needs SPH_F_RK3 at sph_create");
    if (!ctx->have_state) return fail(ctx, SPH_ERR_STATE, "sph_step_rk3 before sph_upload");
    Q0Live live(ctx);
    Dev &d = ctx->d;
    const size_t n = (size_t)d.n;
    const int gb = sph_ceil_div(d.n, 256);
    int rc;
    cudaMemcpyAsync(d.q0, d.x[0], 15 * n * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream);
    // eq. 73 rewrites the master h in every evaluation: a rejected step must give it back too
    const bool keep_h = (d.flags & SPH_F_VARIABLE_H) && ctx->cfg.h_iters > 0;
    if (keep_h) cudaMemcpyAsync(d.h0, d.h, n * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream);
    const double c[3][3] = {{0.5, 0.0, 0.0}, {-1.0, 2.0, 0.0}, {1.0 / 6.0, 4.0 / 6.0, 1.0 / 6.0}};
    for (int st = 0; st < 3; ++st) {
        if ((rc = sph_evaluate(ctx)) != SPH_OK) return rc;                                   // eqs. 59-61
        k_rk_rates<<<gb, 256, 0, ctx->stream>>>(d, d.rk[st], st == 0);
        ctx->launches += 1;
        if (st < 2) {
            k_rk_stage<<<gb, 256, 0, ctx->stream>>>(d, sph_dev_mats(ctx), dt, c[st][0], c[st][1], c[st][2], st + 1);
            ctx->launches += 1;
        }
    }
    k_rk_err_init<<<1, 1, 0, ctx->stream>>>(d);
    k_rk_err<<<gb, 256, 0, ctx->stream>>>(d, dt);
    ctx->launches += 2;
    DevStatus stt;
    cudaMemcpyAsync(&stt, d.status, sizeof(stt), cudaMemcpyDeviceToHost, ctx->stream);
    cudaStreamSynchronize(ctx->stream);
    if ((rc = status_flags(ctx, stt, "sph_step_rk3")) != SPH_OK) {          // truncated lists / walk: nothing is accepted
        cudaMemcpyAsync(d.x[0], d.q0, 15 * n * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream);
        if (keep_h) cudaMemcpyAsync(d.h, d.h0, n * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream);
        ctx->have_tree = ctx->have_lists = 0;
        return rc;
    }
    double err;
    memcpy(&err, &stt.rkerr, sizeof(double));
    const bool ok = err <= eps_des;                                          // false for +inf (a NaN state or rate)
    if (ok) {
        k_rk_stage<<<gb, 256, 0, ctx->stream>>>(d, sph_dev_mats(ctx), dt, c[2][0], c[2][1], c[2][2], 3);   // eq. 58
        ctx->launches += 1;
        out[1] = (err == 0.0) ? INFINITY : dt * pow(fabs(eps_des / err), 0.3);               // eq. 64
    } else {
        cudaMemcpyAsync(d.x[0], d.q0, 15 * n * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream);
        if (keep_h) cudaMemcpyAsync(d.h, d.h0, n * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream);
        out[1] = 0.9 * dt * pow(fabs(eps_des / err), 0.25);                                 // eq. 65 (0 when err = +inf)
    }
    out[0] = err;
    out[2] = ok ? 1.0 : 0.0;
    ctx->have_tree = ctx->have_lists = 0;
    return check_cuda(ctx, "sph_step_rk3");
}

int sph_timestep(sph_ctx *ctx, double *out) {
    if (!ctx || !out) return SPH_ERR_ARG;
    if ((ctx->have_rates & 1) == 0 || ((ctx->d.flags & SPH_F_GRAVITY) && (ctx->have_rates & 2) == 0))
        return fail(ctx, SPH_ERR_STATE, "sph_timestep before a complete evaluation");
    Dev &d = ctx->d;
    k_dtlim_init<<<1, 32, 0, ctx->stream>>>(d);
    k_dtlim<<<sph_ceil_div(d.n, 256), 256, 0, ctx->stream>>>(d, (ctx->have_rates & 2) ? 1 : 0);
    ctx->launches += 2;
    DevStatus st;
    cudaMemcpyAsync(&st, d.status, sizeof(st), cudaMemcpyDeviceToHost, ctx->stream);
    cudaStreamSynchronize(ctx->stream);
    for (int k = 0; k < 3; ++k) memcpy(&out[k], &st.dtlim[k], sizeof(double));
    out[3] = std::min(out[0], std::min(out[1], out[2]));
    return status_flags(ctx, st, "sph_timestep");
}

// ------------------------------------------------------------------------------------------------
// Morton-range sharding (include/sph.h): partition and the one all-gather per evaluation
// ------------------------------------------------------------------------------------------------
int sph_partition(int64_t n, int world, int rank, int64_t *lo, int64_t *hi, int64_t *slice) {
    if (n < 1 || world < 1 || world > SPH_MAX_WORLD || rank < 0 || rank >= world) return SPH_ERR_ARG;
    const int64_t per = (n + world - 1) / world;
    const int64_t sl = (per + 31) / 32 * 32;
    const int64_t l = std::min<int64_t>(n, (int64_t)rank * sl), h = std::min<int64_t>(n, l + sl);
    if (lo) *lo = l;
    if (hi) *hi = h;
    if (slice) *slice = sl;
    return SPH_OK;
}

int sph_set_partition(sph_ctx *ctx, int rank, int world, sph_exchange_fn fn, void *user) {
    if (!ctx) return SPH_ERR_ARG;
    int64_t lo, hi, sl;
    if (sph_partition(ctx->d.n, world, rank, &lo, &hi, &sl) != SPH_OK) return fail(ctx, SPH_ERR_ARG, "sph_set_partition: bad rank / world");
    if (world > 1 && !fn) return fail(ctx, SPH_ERR_ARG, "sph_set_partition: world > 1 needs an exchange function");
    ctx->rank = rank; ctx->world = world; ctx->slice = sl;
    ctx->xfn = (world > 1) ? fn : nullptr; ctx->xuser = user;
    ctx->d.r_lo = (int)lo; ctx->d.r_hi = (int)hi;
    ctx->have_tree = ctx->have_lists = ctx->have_rates = 0;
    drop_graphs(ctx);
    return SPH_OK;
}

// The failure flags steer control flow (sph_step_rk3 gives the state back, every synchronising call returns the error), so
// they must be the same on every rank: a rank writes its three words (err_nb_overflow, err_stack, nb_max) into its slot of
// a byte array that travels with the rates, and after the all-gather every rank folds all slots into its own status block
// (OR, OR, max).  The flags are latched until the next upload, so folding them again later changes nothing.
__global__ void k_status_pack(Dev d, int *slot) {
    slot[0] = d.status->err_nb_overflow; slot[1] = d.status->err_stack; slot[2] = d.status->nb_max;
}
__global__ void k_status_merge(Dev d, const unsigned char *xstat, i64 slice, int world) {
    int ov = 0, stk = 0, mx = 0;
    for (int r = 0; r < world; ++r) {
        const int *slot = reinterpret_cast<const int *>(xstat + (size_t)r * (size_t)slice);
        ov |= slot[0]; stk |= slot[1]; mx = max(mx, slot[2]);
    }
    d.status->err_nb_overflow = ov; d.status->err_stack = stk; d.status->nb_max = mx;
}

// ONE all-gather per exchange: the rank's slices of all arrays are packed into one contiguous block of Dev::xbuf
// (rank-major: block r = [array 0 slice | array 1 slice | ...] of rank r), the caller's function gathers that one array,
// and the other ranks' blocks are copied back into the arrays.  A slice of `slice` elements of 1, 4 or 8 bytes is a whole
// number of 32-byte pieces (slice is a multiple of 32) and every array starts on a 256-byte boundary, so both kernels
// move 16-byte words.
#define XJ_MAX 64
struct XJobs {
    unsigned char *arr[XJ_MAX];     // the array (element 0)
    unsigned off[XJ_MAX];           // bytes per particle of the arrays before it
    unsigned eb[XJ_MAX];            // its element size
};
// grid (pieces, arrays, ranks): unpack = 1 copies block q of xbuf into the arrays for every q but `rank`;
// unpack = 0 copies the arrays' slices of `rank` into its block (gridDim.z = 1).
__global__ void k_xcopy(XJobs jobs, unsigned char *xbuf, i64 slice, int sum_eb, int rank, int unpack) {
    const int k = blockIdx.y;
    const int q = unpack ? (int)blockIdx.z : rank;
    if (unpack && q == rank) return;
    const i64 words = slice * (i64)jobs.eb[k] / 16;
    const i64 j = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= words) return;
    uint4 *a = reinterpret_cast<uint4 *>(jobs.arr[k] + (size_t)q * (size_t)slice * jobs.eb[k]) + j;
    uint4 *x = reinterpret_cast<uint4 *>(xbuf + (size_t)q * (size_t)slice * (size_t)sum_eb + (size_t)jobs.off[k] * (size_t)slice) + j;
    if (unpack) *a = *x; else *x = *a;
}

// which: 1 = the arrays sph_rhs fills, 2 = the gravitational acceleration, 3 = both
static int exchange_rates(sph_ctx *ctx, int which) {
    if (ctx->world <= 1 || !ctx->xfn) return SPH_OK;
    Dev &d = ctx->d;
    XJobs jobs;
    int na = 0;
    unsigned sum_eb = 0;
    auto add = [&](void *p, int bytes) { jobs.arr[na] = (unsigned char *)p; jobs.eb[na] = (unsigned)bytes; jobs.off[na] = sum_eb; sum_eb += bytes; ++na; };
    // slice is a multiple of 32, so a slot of `slice` BYTES holds the three words and keeps them 4-byte aligned
    k_status_pack<<<1, 1, 0, ctx->stream>>>(d, reinterpret_cast<int *>(d.xstat + (size_t)ctx->rank * (size_t)ctx->slice));
    add(d.xstat, 1);
    if (which & 1) {
        add(d.drho, 8); add(d.du, 8);
        // all components, also the zero rows of a 2-D run: every array a download can return is complete on every rank
        for (int a = 0; a < 3; ++a) add(d.dv[a], 8);
        if (d.flags & SPH_F_SOLID) for (int k = 0; k < 6; ++k) add(d.dS[k], 8);
        if (d.flags & SPH_F_DAMAGE) { add(d.ddmg, 8); add(d.strain, 8); add(d.n_act_new, 4); }
        if (d.flags & SPH_F_XSPH) for (int a = 0; a < 3; ++a) add(d.dxs[a], 8);
        if ((d.flags & SPH_F_SOLID) && (d.flags & SPH_F_EXPORT_GRADV)) for (int k = 0; k < 9; ++k) { add(d.gradv[k], 8); add(d.Cten[k], 8); }
        add(d.nb_cnt, 4);
    }
    if ((which & 2) && (d.flags & SPH_F_GRAVITY)) for (int a = 0; a < 3; ++a) add(d.ag[a], 8);
    const int pieces = sph_ceil_div(ctx->slice * 8 / 16, 256);         // of the widest element; narrower arrays exit early
    k_xcopy<<<dim3(pieces, na, 1), 256, 0, ctx->stream>>>(jobs, d.xbuf, ctx->slice, (int)sum_eb, ctx->rank, 0);
    void *arr[1] = {d.xbuf};
    int32_t eb[1] = {(int32_t)sum_eb};
    if (ctx->xfn(ctx->xuser, (void *)ctx->stream, 1, arr, eb, (int64_t)ctx->slice) != 0)
        return fail(ctx, SPH_ERR_CUDA, "the caller's exchange function (all-gather of the rates) failed");
    k_xcopy<<<dim3(pieces, na, ctx->world), 256, 0, ctx->stream>>>(jobs, d.xbuf, ctx->slice, (int)sum_eb, ctx->rank, 1);
    k_status_merge<<<1, 1, 0, ctx->stream>>>(d, d.xstat, ctx->slice, ctx->world);
    ctx->launches += 4;
    return SPH_OK;
}

int sph_upload(sph_ctx *ctx, const sph_state_in *s, int src_is_device) {
    if (!ctx || !s) return SPH_ERR_ARG;
    Dev &d = ctx->d;
    const size_t n = (size_t)d.n;
    const cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    auto cp = [&](void *dst, const void *src, size_t bytes) {
        if (src && bytes) cudaMemcpyAsync(dst, src, bytes, kind, ctx->stream);
    };
    for (int a = 0; a < d.D; ++a) { cp(d.x[a], s->x[a], n * 8); cp(d.v[a], s->v[a], n * 8); }
    cp(d.m, s->m, n * 8); cp(d.rho, s->rho, n * 8); cp(d.u, s->u, n * 8); cp(d.dmg, s->dmg, n * 8); cp(d.h, s->h, n * 8);
    for (int k = 0; k < 6; ++k) cp(d.S[k], s->S[k], n * 8);
    cp(d.mat, s->mat, n * 4); cp(d.n_act, s->n_act, n * 4);
    cp(d.flaw_off, s->flaw_off, (n + 1) * 8);
    cp(d.flaw_eps, s->flaw_eps, (size_t)ctx->cfg.n_flaws * 8);
    // a new state: the failures latched by evaluations of the old one no longer apply
    cudaMemsetAsync(&d.status->err_nb_overflow, 0, 3 * sizeof(int), ctx->stream);   // err_nb_overflow, err_stack, nb_max
    if (!src_is_device) cudaStreamSynchronize(ctx->stream);   // caller may free or reuse its buffers
    ctx->have_state = 1; ctx->have_tree = ctx->have_lists = ctx->have_rates = 0;
    ctx->step_no = 0;
    return check_cuda(ctx, "sph_upload");
}

int sph_build_tree(sph_ctx *ctx) {
    if (!ctx) return SPH_ERR_ARG;
    if (!ctx->have_state) return fail(ctx, SPH_ERR_STATE, "sph_build_tree before sph_upload");
    sph_stage_order(ctx);
    sph_stage_tree(ctx);
    ctx->have_tree = 1; ctx->have_lists = 0; ctx->have_rates = 0;
    return check_cuda(ctx, "sph_build_tree");
}

int sph_find_neighbours(sph_ctx *ctx) {
    if (!ctx) return SPH_ERR_ARG;
    if (!ctx->have_tree) return fail(ctx, SPH_ERR_STATE, "sph_find_neighbours before sph_build_tree");
    sph_stage_neigh(ctx);
    ctx->have_lists = 1;
    return check_cuda(ctx, "sph_find_neighbours");
}

int sph_rhs(sph_ctx *ctx) {
    if (!ctx) return SPH_ERR_ARG;
    if (!ctx->have_tree || !ctx->have_lists) return fail(ctx, SPH_ERR_STATE, "sph_rhs before sph_find_neighbours");
    sph_stage_rhs(ctx);
    ctx->have_rates |= 1;
    if (!ctx->in_evaluate) { const int rc = exchange_rates(ctx, 1); if (rc != SPH_OK) return rc; }
    return check_cuda(ctx, "sph_rhs");
}

int sph_gravity(sph_ctx *ctx) {
    if (!ctx) return SPH_ERR_ARG;
    if (!ctx->have_tree) return fail(ctx, SPH_ERR_STATE, "sph_gravity before sph_build_tree");
    sph_stage_gravity(ctx);
    ctx->have_rates |= 2;
    if (!ctx->in_evaluate) { const int rc = exchange_rates(ctx, 2); if (rc != SPH_OK) return rc; }
    return check_cuda(ctx, "sph_gravity");
}

int sph_evaluate(sph_ctx *ctx) {
    if (!ctx) return SPH_ERR_ARG;
    int rc;
    if ((rc = sph_build_tree(ctx)) != SPH_OK) return rc;
    if ((rc = sph_find_neighbours(ctx)) != SPH_OK) return rc;
    ctx->in_evaluate = 1;                    // sharded: ONE all-gather for the whole evaluation, after the walk
    rc = sph_rhs(ctx);
    if (rc == SPH_OK) {
        if (ctx->grav_reuse) {               // decoupled step: the stored field (complete on every rank), brought into the new order
            StageTimer tm(ctx, SPH_T_GRAVITY);
            k_ag_take<<<sph_ceil_div(ctx->d.n, 256), 256, 0, ctx->stream>>>(ctx->d);
            ctx->launches += 1;
            ctx->have_rates |= 2;
        } else {
            rc = sph_gravity(ctx);
        }
    }
    ctx->in_evaluate = 0;
    if (rc != SPH_OK) return rc;
    if ((rc = exchange_rates(ctx, ctx->grav_reuse ? 1 : 3)) != SPH_OK) return rc;
    return check_cuda(ctx, "sph_evaluate");
}

// the launches of one predictor-corrector step, enqueued on ctx->stream
static int step_enqueue(sph_ctx *ctx, double dt) {
    Dev &d = ctx->d;
    const size_t n = (size_t)d.n;
    int rc;
    const int every = ctx->cfg.gravity_every;
    const bool decoupled = every > 1 && (d.flags & SPH_F_GRAVITY);
    ctx->grav_reuse = decoupled && (ctx->step_no % every) != 0;
    ctx->step_no += 1;
    {
        StageTimer tm(ctx, SPH_T_UPDATE);
        cudaMemcpyAsync(d.q0, d.x[0], 15 * n * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream);
    }
    if ((rc = sph_evaluate(ctx)) != SPH_OK) { ctx->grav_reuse = 0; return rc; }
    {
        StageTimer tm(ctx, SPH_T_UPDATE);
        k_update<<<sph_ceil_div(d.n, 256), 256, 0, ctx->stream>>>(d, sph_dev_mats(ctx), 0.5 * dt, 0);   // eq. 52
        ctx->launches += 1;
    }
    if ((rc = sph_evaluate(ctx)) != SPH_OK) { ctx->grav_reuse = 0; return rc; }
    if (decoupled && !ctx->grav_reuse) {     // the field the next gravity_every - 1 steps reuse
        k_ag_keep<<<sph_ceil_div(d.n, 256), 256, 0, ctx->stream>>>(d);
        ctx->launches += 1;
    }
    ctx->grav_reuse = 0;
    {
        StageTimer tm(ctx, SPH_T_UPDATE);
        k_update<<<sph_ceil_div(d.n, 256), 256, 0, ctx->stream>>>(d, sph_dev_mats(ctx), dt, 1);         // eq. 53
        ctx->launches += 1;
    }
    ctx->have_tree = ctx->have_lists = 0;   // the state moved on; the rates stay readable
    return check_cuda(ctx, "sph_step");
}

// A step is ~80 launches; for the small workloads (C1-C3) the GPU idles between them.  The launch
// sequence of a step depends only on the configuration and on dt, so it is captured into a CUDA
// graph the second time in a row a dt is asked for and replayed from then on (stage timing runs the
// plain launches: event brackets are not part of the graph).
int sph_step(sph_ctx *ctx, double dt) {
    if (!ctx) return SPH_ERR_ARG;
    if (!ctx->have_state) return fail(ctx, SPH_ERR_STATE, "sph_step before sph_upload");
    Q0Live live(ctx);
    if (ctx->timing || ctx->graphs_off || ctx->cfg.gravity_every > 1 || ctx->world > 1) return step_enqueue(ctx, dt);
    if (ctx->step_graph && ctx->graph_dt == dt) {
        if (cudaGraphLaunch(ctx->step_graph, ctx->stream) != cudaSuccess) return check_cuda(ctx, "sph_step (graph)");
        ctx->launches += ctx->graph_launches;
        ctx->have_tree = ctx->have_lists = 0;
        ctx->have_rates = 3;
        return SPH_OK;
    }
    const bool repeat = (ctx->last_dt == dt);
    ctx->last_dt = dt;
    if (!repeat) return step_enqueue(ctx, dt);
    if (cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
        cudaGetLastError();
        ctx->graphs_off = 1;
        return step_enqueue(ctx, dt);
    }
    const i64 l0 = ctx->launches;
    const int rc = step_enqueue(ctx, dt);
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(ctx->stream, &graph);
    cudaGraphExec_t exec = nullptr;
    if (rc != SPH_OK || ce != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
        cudaGetLastError();
        if (graph) cudaGraphDestroy(graph);
        ctx->launches = l0;
        ctx->graphs_off = 1;                 // nothing has run: do the step with plain launches
        return step_enqueue(ctx, dt);
    }
    cudaGraphDestroy(graph);
    if (ctx->step_graph) cudaGraphExecDestroy(ctx->step_graph);
    ctx->step_graph = exec;
    ctx->graph_dt = dt;
    ctx->graph_launches = ctx->launches - l0;
    if (cudaGraphLaunch(exec, ctx->stream) != cudaSuccess) return check_cuda(ctx, "sph_step (graph)");
    return SPH_OK;
}

// ---- sph_step_host: upload and step as one call, the copies beside the first evaluation ----
// part 0: what the tree, the partner search and the walk read; part 1: the rest of sph_upload's members
static void upload_part(sph_ctx *ctx, const sph_state_in *s, cudaStream_t st, int part) {
    Dev &d = ctx->d;
    const size_t n = (size_t)d.n;
    auto cp = [&](void *dst, const void *src, size_t bytes) {
        if (src && bytes) cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st);
    };
    if (part == 0) {
        for (int a = 0; a < d.D; ++a) cp(d.x[a], s->x[a], n * 8);
        cp(d.h, s->h, n * 8); cp(d.m, s->m, n * 8);
        cudaMemsetAsync(&d.status->err_nb_overflow, 0, 3 * sizeof(int), st);   // as sph_upload
    } else {
        for (int a = 0; a < d.D; ++a) cp(d.v[a], s->v[a], n * 8);
        cp(d.rho, s->rho, n * 8); cp(d.u, s->u, n * 8); cp(d.dmg, s->dmg, n * 8);
        for (int k = 0; k < 6; ++k) cp(d.S[k], s->S[k], n * 8);
        cp(d.mat, s->mat, n * 4); cp(d.n_act, s->n_act, n * 4);
        cp(d.flaw_off, s->flaw_off, (n + 1) * 8);
        cp(d.flaw_eps, s->flaw_eps, (size_t)ctx->cfg.n_flaws * 8);
    }
}

// The launches of sph_upload + sph_step with the first evaluation reordered: positions, h and masses arrive first and the
// order, the tree, the partner search and the walk (which read nothing else) run while the second stream copies the rest;
// then the remaining arrays are gathered, the base copy of eq. 52 is taken and the SPH sums follow.
static int host_step_enqueue(sph_ctx *ctx, const sph_state_in *s, double dt) {
    Dev &d = ctx->d;
    const size_t n = (size_t)d.n;
    int rc;
    cudaEventRecord(ctx->ev_fork, ctx->stream);                   // the copies overwrite what earlier launches may still read
    cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_fork, 0);
    upload_part(ctx, s, ctx->copy_stream, 0);
    cudaEventRecord(ctx->ev_geom, ctx->copy_stream);
    upload_part(ctx, s, ctx->copy_stream, 1);
    cudaEventRecord(ctx->ev_rest, ctx->copy_stream);
    cudaStreamWaitEvent(ctx->stream, ctx->ev_geom, 0);
    ctx->have_state = 1; ctx->have_tree = ctx->have_lists = ctx->have_rates = 0;
    ctx->step_no = 1; ctx->grav_reuse = 0;
    ctx->split_gather = 1;
    sph_stage_order(ctx);
    ctx->split_gather = 0;
    sph_stage_tree(ctx);
    ctx->have_tree = 1;
    sph_stage_neigh(ctx);
    ctx->have_lists = 1;
    sph_stage_gravity(ctx);
    ctx->have_rates |= 2;
    cudaStreamWaitEvent(ctx->stream, ctx->ev_rest, 0);
    sph_stage_gather_rest(ctx);
    cudaMemcpyAsync(d.q0, d.x[0], 15 * n * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream);
    sph_stage_rhs(ctx);
    ctx->have_rates |= 1;
    k_update<<<sph_ceil_div(d.n, 256), 256, 0, ctx->stream>>>(d, sph_dev_mats(ctx), 0.5 * dt, 0);   // eq. 52
    ctx->launches += 1;
    if ((rc = sph_evaluate(ctx)) != SPH_OK) return rc;
    k_update<<<sph_ceil_div(d.n, 256), 256, 0, ctx->stream>>>(d, sph_dev_mats(ctx), dt, 1);         // eq. 53
    ctx->launches += 1;
    ctx->have_tree = ctx->have_lists = 0;
    return check_cuda(ctx, "sph_step_host");
}

int sph_step_host(sph_ctx *ctx, const sph_state_in *s, double dt) {
    if (!ctx || !s) return SPH_ERR_ARG;
    Q0Live live(ctx);
    // stage timing, decoupled gravity and sharded runs take the plain sequence
    if (ctx->timing || ctx->cfg.gravity_every > 1 || ctx->world > 1 || !ctx->copy_stream) {
        const int rc = sph_upload(ctx, s, 0);
        return rc != SPH_OK ? rc : sph_step(ctx, dt);
    }
    const bool same = memcmp(&ctx->hlast_src, s, sizeof(*s)) == 0 && ctx->hlast_dt == dt;
    if (ctx->hstep_graph && ctx->hgraph_dt == dt && memcmp(&ctx->hgraph_src, s, sizeof(*s)) == 0) {
        if (cudaGraphLaunch(ctx->hstep_graph, ctx->stream) != cudaSuccess) return check_cuda(ctx, "sph_step_host (graph)");
        ctx->launches += ctx->hgraph_launches;
        ctx->have_state = 1; ctx->have_tree = ctx->have_lists = 0; ctx->have_rates = 3; ctx->step_no = 1;
        return SPH_OK;
    }
    ctx->hlast_src = *s; ctx->hlast_dt = dt;
    // the same buffers and dt twice in a row: capture the sequence (both streams) and replay it from then on
    if (!same || ctx->graphs_off || cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
        cudaGetLastError();
        return host_step_enqueue(ctx, s, dt);
    }
    const i64 l0 = ctx->launches;
    const int rc = host_step_enqueue(ctx, s, dt);
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(ctx->stream, &graph);
    cudaGraphExec_t exec = nullptr;
    if (rc != SPH_OK || ce != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
        cudaGetLastError();
        if (graph) cudaGraphDestroy(graph);
        ctx->launches = l0;
        ctx->graphs_off = 1;                     // nothing has run: do the step with plain launches
        return host_step_enqueue(ctx, s, dt);
    }
    cudaGraphDestroy(graph);
    if (ctx->hstep_graph) cudaGraphExecDestroy(ctx->hstep_graph);
    ctx->hstep_graph = exec;
    ctx->hgraph_dt = dt; ctx->hgraph_src = *s;
    ctx->hgraph_launches = ctx->launches - l0;
    if (cudaGraphLaunch(exec, ctx->stream) != cudaSuccess) return check_cuda(ctx, "sph_step_host (graph)");
    return SPH_OK;
}

static int device_flags(sph_ctx *ctx) {
    DevStatus st;
    if (cudaMemcpyAsync(&st, ctx->d.status, sizeof(st), cudaMemcpyDeviceToHost, ctx->stream) != cudaSuccess ||
        cudaStreamSynchronize(ctx->stream) != cudaSuccess) {
        check_cuda(ctx, "status");
        return SPH_ERR_CUDA;
    }
    return status_flags(ctx, st, "sync");
}

int sph_sync(sph_ctx *ctx) {
    if (!ctx) return SPH_ERR_ARG;
    return device_flags(ctx);
}

int sph_download(sph_ctx *ctx, const sph_state_out *o, int dst_is_device) {
    if (!ctx || !o) return SPH_ERR_ARG;
    if (!ctx->have_state) return fail(ctx, SPH_ERR_STATE, "sph_download before sph_upload");
    if (!dst_is_device && ctx->q0_live)
        return fail(ctx, SPH_ERR_STATE, "sph_download to host buffers while a step call is under way (its base copy is the staging area)");
    Dev &d = ctx->d;
    const int n = d.n;
    const size_t nb = (size_t)n * 8;
    const cudaMemcpyKind kind = dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    auto plain = [&](void *dst, const void *src, size_t bytes) {
        if (dst) cudaMemcpyAsync(dst, src, bytes, kind, ctx->stream);
    };
    for (int a = 0; a < 3; ++a) { plain(o->x[a], d.x[a], nb); plain(o->v[a], d.v[a], nb); }
    plain(o->rho, d.rho, nb); plain(o->u, d.u, nb); plain(o->dmg, d.dmg, nb); plain(o->h, d.h, nb);
    for (int k = 0; k < 6; ++k) plain(o->S[k], d.S[k], nb);
    plain(o->n_act, d.n_act, (size_t)n * 4);
    bool want_rates = o->drho || o->du || o->ddmg || o->p || o->cs || o->strain || o->n_act_new || o->nb_count;
    for (int a = 0; a < 3; ++a) want_rates = want_rates || o->dv[a] || o->ag[a] || o->dxs[a];
    for (int k = 0; k < 6; ++k) want_rates = want_rates || o->dS[k];
    for (int k = 0; k < 9; ++k) want_rates = want_rates || o->gradv[k] || o->C[k];
    if (want_rates && !ctx->have_rates) return fail(ctx, SPH_ERR_STATE, "sph_download of rates before an evaluation");
    const bool sph = (ctx->have_rates & 1) != 0, grav = (ctx->have_rates & 2) != 0;
    const bool solid = sph && (d.flags & SPH_F_SOLID), dam = sph && (d.flags & SPH_F_DAMAGE);
    const bool gexp = solid && (d.flags & SPH_F_EXPORT_GRADV);
    // The rates live in Morton order: ONE kernel un-sorts every requested array (straight into the
    // caller's DEVICE buffers, or into staging slots that are then copied to the HOST buffers), and a
    // host download synchronises once.  Staging = the RK2 base copy q0 (15 n doubles, live only inside
    // sph_step) followed by the pair records prec (16 n doubles, live only inside sph_rhs).
    UJobs jobs;
    struct Copy { void *dst; const void *src; size_t bytes; };
    Copy copies[UJ_MAX];
    int nj = 0;
    size_t slot = 0;
    auto stage_slot = [&](size_t k) -> double * {
        return (k < 15) ? d.q0 + k * (size_t)n : d.prec + (k - 15) * (size_t)n;
    };
    auto job = [&](void *dst, const void *src, bool present, bool is_int) {
        if (!dst) return;
        const size_t bytes = (size_t)n * (is_int ? 4 : 8);
        if (!present) {          // quantity not computed under the current flags: zeros
            if (dst_is_device) cudaMemsetAsync(dst, 0, bytes, ctx->stream);
            else memset(dst, 0, bytes);
            return;
        }
        void *target = dst;
        if (!dst_is_device) {
            target = stage_slot(slot++);
            copies[nj] = Copy{dst, target, bytes};
        }
        jobs.j[nj] = UJob{src, target, is_int ? 1 : 0, 0};
        ++nj;
    };
    job(o->drho, d.drho, sph, false); job(o->du, d.du, sph, false);
    for (int a = 0; a < 3; ++a) { job(o->dv[a], d.dv[a], sph, false); job(o->ag[a], d.ag[a], grav, false); }
    for (int a = 0; a < 3; ++a) job(o->dxs[a], d.dxs[a], sph && (d.flags & SPH_F_XSPH), false);
    for (int k = 0; k < 6; ++k) job(o->dS[k], d.dS[k], solid, false);
    job(o->ddmg, d.ddmg, dam, false); job(o->strain, d.strain, dam, false);
    job(o->p, d.p, sph, false); job(o->cs, d.cs, sph, false);
    job(o->n_act_new, d.n_act_new, dam, true);
    job(o->nb_count, d.nb_cnt, ctx->have_lists || sph, true);
    if (nj > 0) {
        dim3 grid(sph_ceil_div(n, 256), nj);
        k_unsort_many<<<grid, 256, 0, ctx->stream>>>(jobs, d.perm, n);
        ctx->launches += 1;
        if (!dst_is_device)
            for (int k = 0; k < nj; ++k) cudaMemcpyAsync(copies[k].dst, copies[k].src, copies[k].bytes, cudaMemcpyDeviceToHost, ctx->stream);
    }
    // second batch: velocity gradient and correction tensor (18 arrays; the staging slots are free again
    // only after the copies above, which are stream-ordered)
    nj = 0; slot = 0;
    for (int k = 0; k < 9; ++k) { job(o->gradv[k], d.gradv[k], gexp, false); job(o->C[k], d.Cten[k], gexp, false); }
    if (nj > 0) {
        dim3 grid(sph_ceil_div(n, 256), nj);
        k_unsort_many<<<grid, 256, 0, ctx->stream>>>(jobs, d.perm, n);
        ctx->launches += 1;
        if (!dst_is_device)
            for (int k = 0; k < nj; ++k) cudaMemcpyAsync(copies[k].dst, copies[k].src, copies[k].bytes, cudaMemcpyDeviceToHost, ctx->stream);
    }
    if (!dst_is_device) return device_flags(ctx);
    return check_cuda(ctx, "sph_download");
}

int64_t sph_launch_count(sph_ctx *ctx) { return ctx ? ctx->launches : 0; }
const char *sph_last_error(sph_ctx *ctx) { return ctx ? ctx->err : "null context"; }
const char *sph_version(void) { return "sph-b200 0.1 (sm_100a, FP64)"; }

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// inspection for the parity tests (HOST buffers; synchronise)
// ------------------------------------------------------------------------------------------------
extern "C" {

int sph_get_order(sph_ctx *ctx, uint64_t *keys, int32_t *perm, double *root) {
    if (!ctx) return SPH_ERR_ARG;
    if (!ctx->have_tree) return fail(ctx, SPH_ERR_STATE, "sph_get_order before sph_build_tree");
    Dev &d = ctx->d;
    const size_t n = (size_t)d.n;
    if (keys) cudaMemcpyAsync(keys, d.keys, n * 8, cudaMemcpyDeviceToHost, ctx->stream);
    if (perm) cudaMemcpyAsync(perm, d.perm, n * 4, cudaMemcpyDeviceToHost, ctx->stream);
    DevRoot r;
    cudaMemcpyAsync(&r, d.root, sizeof(r), cudaMemcpyDeviceToHost, ctx->stream);
    cudaStreamSynchronize(ctx->stream);
    if (root) { root[0] = r.xmin[0]; root[1] = r.xmin[1]; root[2] = r.xmin[2]; root[3] = r.s0; }
    return check_cuda(ctx, "sph_get_order");
}

int sph_get_tree_size(sph_ctx *ctx, int32_t *n_nodes) {
    if (!ctx || !n_nodes) return SPH_ERR_ARG;
    if (!ctx->have_tree) return fail(ctx, SPH_ERR_STATE, "sph_get_tree_size before sph_build_tree");
    DevStatus st;
    cudaMemcpyAsync(&st, ctx->d.status, sizeof(st), cudaMemcpyDeviceToHost, ctx->stream);
    cudaStreamSynchronize(ctx->stream);
    *n_nodes = st.n_nodes;
    return check_cuda(ctx, "sph_get_tree_size");
}

int sph_get_tree(sph_ctx *ctx, int32_t *level, uint64_t *prefix, int32_t *lo, int32_t *hi, double *mass, double *com,
                 double *bmin, double *bmax, double *hmax, int32_t *child, int32_t *child_lo) {
    int32_t nn = 0;
    int rc = sph_get_tree_size(ctx, &nn);
    if (rc != SPH_OK) return rc;
    Dev &d = ctx->d;
    const int D = d.D, NC = 1 << D;
    const size_t m = (size_t)nn;
    if (m == 0) return SPH_OK;
    auto get = [&](void *dst, const void *src, size_t bytes) {
        if (dst) cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, ctx->stream);
    };
    std::vector<int32_t> lv(m), l0(m);
    get(lv.data(), d.nlevel, m * 4);
    get(l0.data(), d.nlo, m * 4);
    get(hi, d.nhi_s, m * 4);
    get(mass, d.nmass, m * 8);
    get(hmax, d.nhmax, m * 8);
    get(child, d.child, m * NC * 4);
    get(child_lo, d.child_lo, m * (NC + 1) * 4);
    std::vector<double> t3[3][3];
    for (int a = 0; a < 3; ++a) {
        if (com) { t3[0][a].resize(m); get(t3[0][a].data(), d.ncom[a], m * 8); }
        if (bmin) { t3[1][a].resize(m); get(t3[1][a].data(), d.nbmin[a], m * 8); }
        if (bmax) { t3[2][a].resize(m); get(t3[2][a].data(), d.nbmax[a], m * 8); }
    }
    std::vector<u64> keys;
    if (prefix) { keys.resize((size_t)d.n); get(keys.data(), d.keys, (size_t)d.n * 8); }
    cudaStreamSynchronize(ctx->stream);
    for (size_t k = 0; k < m; ++k) {
        if (level) level[k] = lv[k];
        if (lo) lo[k] = l0[k];
        if (prefix) prefix[k] = (lv[k] == 0) ? 0ull : (keys[(size_t)l0[k]] >> (D * (d.L - lv[k])));
        for (int a = 0; a < 3; ++a) {
            if (com) com[3 * k + a] = t3[0][a][k];
            if (bmin) bmin[3 * k + a] = t3[1][a][k];
            if (bmax) bmax[3 * k + a] = t3[2][a][k];
        }
    }
    return check_cuda(ctx, "sph_get_tree");
}

int sph_get_neighbours(sph_ctx *ctx, int64_t *off, int32_t *idx, int64_t cap) {
    if (!ctx || !off) return SPH_ERR_ARG;
    if (!ctx->have_lists) return fail(ctx, SPH_ERR_STATE, "sph_get_neighbours before sph_find_neighbours");
    int rc = device_flags(ctx);
    if (rc != SPH_OK) return rc;
    Dev &d = ctx->d;
    const size_t n = (size_t)d.n;
    std::vector<int> cnt(n), perm(n);
    cudaMemcpyAsync(cnt.data(), d.nb_cnt, n * 4, cudaMemcpyDeviceToHost, ctx->stream);
    cudaMemcpyAsync(perm.data(), d.perm, n * 4, cudaMemcpyDeviceToHost, ctx->stream);
    cudaStreamSynchronize(ctx->stream);
    off[0] = 0;
    {
        std::vector<int> co(n);
        for (size_t i = 0; i < n; ++i) {       // sharded: only the rank's own slice has lists (the counts are complete)
            if ((int)i < d.r_lo || (int)i >= d.r_hi) cnt[i] = 0;
            co[(size_t)perm[i]] = cnt[i];
        }
        for (size_t o = 0; o < n; ++o) off[o + 1] = off[o] + co[o];
    }
    if (!idx) return SPH_OK;
    if (cap < off[n]) return fail(ctx, SPH_ERR_ARG, "sph_get_neighbours: idx too small");
    // lists are group-transposed on the device: fetch a block of groups at a time
    const size_t groups = (n + 31) / 32, gcap = (size_t)d.cap * 32;
    const size_t chunk = std::max<size_t>(1, (64u << 20) / (gcap * 4));
    std::vector<int> buf(chunk * gcap);
    for (size_t g0 = 0; g0 < groups; g0 += chunk) {
        const size_t g1 = std::min(groups, g0 + chunk);
        cudaMemcpyAsync(buf.data(), d.nb + g0 * gcap, (g1 - g0) * gcap * 4, cudaMemcpyDeviceToHost, ctx->stream);
        cudaStreamSynchronize(ctx->stream);
        for (size_t g = g0; g < g1; ++g)
            for (int lane = 0; lane < 32; ++lane) {
                const size_t i = g * 32 + lane;
                if (i >= n) break;
                int32_t *dst = idx + off[(size_t)perm[i]];
                const int *src = buf.data() + (g - g0) * gcap + SPH_NB_POS(lane);
                for (int k = 0; k < cnt[i]; ++k) dst[k] = perm[(size_t)src[(size_t)k * 32]];
                std::sort(dst, dst + cnt[i]);
            }
    }
    return check_cuda(ctx, "sph_get_neighbours");
}

}  // extern "C"
