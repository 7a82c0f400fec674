// =====================================================================================
// CPU ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, scalar FP64 restatement of the per-timestep right-hand side of
// Schaefer et al., "A smooth particle hydrodynamics code to model collisions between
// solid, self-gravitating objects" (arXiv:1604.03290; /root/reference/PAPER.md).
// It shares no code, header, table or helper with the CUDA path under
// paper_1604_03290_b200/ and neither imports the other.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
// this library.  Compile with -ffp-contract=off: every floating-point operation is
// rounded separately, in the order written, because neighbour membership, Morton
// quantisation and the tree opening test are floating-point decisions that the CUDA
// path must reproduce bit for bit.
//
// Citations are "PAPER.md:<line> (eq./section)".  Readings of ambiguous or garbled
// passages carry the U-numbers of SURVEY.md section 8(c) / DESIGN.md "Readings".
//
// Parity pins: every function here is pinned by tests/test_oracle_*.py (closed forms,
// invariants, brute force, golden values of tests/golden/; round 2 added the sign of S in
// eqs. 30/31, the (1-d) S factor of eq. 20, a hand value of Tillotson eq. 15, the density sum
// with the mean h, and the post-update rules of the step in tests/test_oracle_pins_r2.py)
// EXCEPT the readings the paper cannot pin:
//   * crack growth speed c_g and the length R_s in eqs. 24/46 (U16): "parity unpinned"
//     by the paper (pinned only by dimensional analysis and the hand-computed formula);
//   * the per-component tension criterion of the artificial stress, eq. 37 (U25): "parity
//     unpinned" by the paper (pinned by a two-particle closed form and the conservation identities).
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

typedef long long i64;
typedef unsigned long long u64;

extern "C" {

struct orc_mat {
    int eos;                       // 0 ideal gas, 1 Murnaghan (eq. 13), 2 Tillotson (eqs. 14-15)
    double rho0, K0, nM, gamma;
    double tA, tB, tE0, tEiv, tEcv, ta, tb, talpha, tbeta;
    double mu, Y0;
    int brittle;
};

struct orc_cfg {
    int dim, flags, L, n_materials;
    i64 n;
    double theta, G, eps_soft, av_alpha, av_beta, av_eps;
    double as_eps, as_n, as_mpd, xsph;   // artificial stress (eqs. 35-38) and XSPH factor (eq. 40)
};

struct orc_state {
    const double *x[3], *v[3], *m, *rho, *u, *S[6], *dmg, *h;
    const int *mat, *n_act;
    const i64 *flaw_off;
    const double *flaw_eps;
};

struct orc_rates {                  // all arrays have one entry per TARGET
    double *drho, *dv[3], *du, *gradv[9], *dS[6], *ddmg, *strain, *C[9];
    int *n_act;
    double *A_drho, *A_dv[3], *A_du, *A_gradv[9], *A_dS[6];   // sums of |pair terms| (T1)
    double *dxs[3], *A_dxs[3];      // XSPH velocity correction (eq. 40) and its sum of |terms|
};

enum { F_SOLID = 1, F_PLASTIC = 2, F_DAMAGE = 4, F_GRAVITY = 8, F_VARIABLE_H = 16, F_DENSITY_SUM = 32,
       F_ART_STRESS = 64, F_XSPH = 128 };

// -------------------------------------------------------------------------------------
// P1. Cubic B-spline kernel, PAPER.md:217 (eq. 25), :221 (eq. 26), :226 (eq. 27).
// h is the paper's h: W vanishes for r/h > 1.
// -------------------------------------------------------------------------------------
static double norm_s(int D) {
    const double pi = 3.14159265358979323846;
    if (D == 1) return 4.0 / 3.0;
    if (D == 2) return 40.0 / (7.0 * pi);
    return 8.0 / pi;
}

double orc_W(int D, double r, double h) {
    double q = r / h;
    double hD = (D == 1) ? h : (D == 2) ? h * h : h * h * h;
    double f;
    if (q < 0.5) f = 6.0 * q * q * q - 6.0 * q * q + 1.0;
    else if (q <= 1.0) f = 2.0 * (1.0 - q) * (1.0 - q) * (1.0 - q);
    else f = 0.0;
    return norm_s(D) / hD * f;
}

double orc_dW(int D, double r, double h) {          // dW/dr
    double q = r / h;
    double hD1 = (D == 1) ? h * h : (D == 2) ? h * h * h : h * h * h * h;
    double f;
    if (q < 0.5) f = 3.0 * q * q - 2.0 * q;
    else if (q <= 1.0) f = -(1.0 - q) * (1.0 - q);
    else f = 0.0;
    return 6.0 * norm_s(D) / hD1 * f;
}

// -------------------------------------------------------------------------------------
// P13-P15. Equations of state and sound speed.
//   ideal gas: p = (gamma-1) rho u (named at PAPER.md:505; textbook form), c = sqrt(gamma (gamma-1) u)
//   Murnaghan: PAPER.md:120 (eq. 13); c = sqrt(K0/rho0) (eq. 12)           (U11)
//   Tillotson: PAPER.md:128 (eq. 14), :132 (eq. 15), :137 (interpolation);               (U18)
//              c = sqrt(A_T/rho0) (Table 1 note: A_T is the bulk modulus)   (U11)
// -------------------------------------------------------------------------------------
void orc_eos(const orc_mat *mt, double rho, double u, double *p, double *cs) {
    if (mt->eos == 0) {
        *p = (mt->gamma - 1.0) * rho * u;
        *cs = std::sqrt(mt->gamma * (mt->gamma - 1.0) * u);
    } else if (mt->eos == 1) {
        *p = mt->K0 / mt->nM * (std::pow(rho / mt->rho0, mt->nM) - 1.0);
        *cs = std::sqrt(mt->K0 / mt->rho0);
    } else {
        double eta = rho / mt->rho0, chi = eta - 1.0;
        double om = u / (mt->tE0 * eta * eta) + 1.0;
        // eq. 14, compressed or cold
        double pc = (mt->ta + mt->tb / om) * rho * u + mt->tA * chi + mt->tB * chi * chi;
        // eq. 15, expanded and hot
        double z = mt->rho0 / rho - 1.0;
        double pe = mt->ta * rho * u +
                    (mt->tb * rho * u / om + mt->tA * chi * std::exp(-mt->tbeta * z)) *
                        std::exp(-mt->talpha * z * z);
        if (eta >= 1.0 || u <= mt->tEiv) *p = pc;
        else if (u >= mt->tEcv) *p = pe;
        else *p = ((u - mt->tEiv) * pe + (mt->tEcv - u) * pc) / (mt->tEcv - mt->tEiv);
        *cs = std::sqrt(mt->tA / mt->rho0);
    }
}

// -------------------------------------------------------------------------------------
// O1. Root cube (eq. 67), L-bit quantisation and Morton keys (U12, U13).
// -------------------------------------------------------------------------------------
u64 orc_interleave(int D, u64 gx, u64 gy, u64 gz, int L) {
    u64 key = 0;
    for (int b = 0; b < L; ++b) {
        key |= ((gx >> b) & 1ull) << (D * b + 0);
        key |= ((gy >> b) & 1ull) << (D * b + 1);
        if (D == 3) key |= ((gz >> b) & 1ull) << (D * b + 2);
    }
    return key;
}

void orc_order(int D, i64 n, const double *x, const double *y, const double *z, int L,
               u64 *key_sorted, int *perm, double *xmin3, double *s0_out) {
    const double *X[3] = {x, y, z};
    double lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    for (int a = 0; a < D; ++a) {
        lo[a] = hi[a] = X[a][0];
        for (i64 i = 1; i < n; ++i) { lo[a] = std::min(lo[a], X[a][i]); hi[a] = std::max(hi[a], X[a][i]); }
    }
    double s0 = 0.0;
    for (int a = 0; a < D; ++a) s0 = std::max(s0, hi[a] - lo[a]);         // eq. 67
    if (!(s0 > 0.0)) s0 = 1.0;                                             // all particles coincide
    double scale = std::ldexp(1.0, L) / s0;
    u64 gmax = (1ull << L) - 1ull;
    std::vector<u64> key(n);
    for (i64 i = 0; i < n; ++i) {
        u64 g[3] = {0, 0, 0};
        for (int a = 0; a < D; ++a) {
            double t = (X[a][i] - lo[a]) * scale;
            u64 gi = (u64)t;
            g[a] = std::min(gmax, gi);
        }
        key[i] = orc_interleave(D, g[0], g[1], g[2], L);
    }
    std::vector<int> p(n);
    for (i64 i = 0; i < n; ++i) p[i] = (int)i;
    std::stable_sort(p.begin(), p.end(), [&](int a, int b) { return key[a] < key[b]; });
    for (i64 i = 0; i < n; ++i) { perm[i] = p[i]; key_sorted[i] = key[p[i]]; }
    for (int a = 0; a < 3; ++a) xmin3[a] = lo[a];
    *s0_out = s0;
}

// -------------------------------------------------------------------------------------
// O3. Reference octree (PAPER.md:364-368 section 3.3, :459-475 section 3.5.1), built by
// recursive top-down partition of the sorted key range.  Cells with a single occupied
// child are not stored (U14): all cells of such a chain hold the same pseudo-particle.
// Pseudo-particles: total mass and centre of mass, monopole only,
// children summed in octant order, every operation rounded separately (U15).
// -------------------------------------------------------------------------------------
struct Node {
    int level; u64 prefix; int lo, hi;
    int child[8];      // >=0 internal node id, -1 empty, <=-2: leaf holding particles [plo, phi)
    int plo[8], phi[8];
    double mass, com[3], bmin[3], bmax[3], hmax;
};

struct Tree {
    int D, L; i64 n; double s0, xmin[3];
    std::vector<u64> key; std::vector<int> perm;
    std::vector<double> sx[3], sm, sh;     // particle data in sorted order
    std::vector<Node> nodes;               // nodes[0] = root (if n >= 2 distinct keys)
};

static int build_rec(Tree &T, int lo, int hi, int level) {
    // returns node id, or -2 if [lo,hi) is a leaf (1 particle, or all keys equal)
    const int D = T.D, L = T.L, NC = 1 << D;
    if (hi - lo == 1 || T.key[lo] == T.key[hi - 1]) return -2;
    for (;;) {   // skip chain cells
        int shift = D * (L - 1 - level);
        u64 d0 = (T.key[lo] >> shift) & (u64)(NC - 1), d1 = (T.key[hi - 1] >> shift) & (u64)(NC - 1);
        if (d0 != d1) break;
        ++level;
    }
    int id = (int)T.nodes.size();
    T.nodes.push_back(Node());
    {
        Node &nd = T.nodes[id];
        nd.level = level; nd.lo = lo; nd.hi = hi;
        nd.prefix = (level == 0) ? 0ull : (T.key[lo] >> (D * (L - level)));
    }
    int shift = D * (L - 1 - level);
    int start = lo;
    for (int c = 0; c < NC; ++c) {
        int end = start;
        while (end < hi && (int)((T.key[end] >> shift) & (u64)(NC - 1)) == c) ++end;
        int ch;
        if (end == start) ch = -1;
        else ch = build_rec(T, start, end, level + 1);
        Node &nd = T.nodes[id];
        nd.child[c] = ch; nd.plo[c] = start; nd.phi[c] = end;
        start = end;
    }
    return id;
}

static void moments_rec(Tree &T, int id) {
    const int D = T.D, NC = 1 << D;
    for (int c = 0; c < NC; ++c) if (T.nodes[id].child[c] >= 0) moments_rec(T, T.nodes[id].child[c]);
    Node &nd = T.nodes[id];
    double M = 0.0, S[3] = {0, 0, 0};
    double bmin[3] = {INFINITY, INFINITY, INFINITY}, bmax[3] = {-INFINITY, -INFINITY, -INFINITY}, hmax = 0.0;
    for (int c = 0; c < NC; ++c) {
        int ch = nd.child[c];
        if (ch == -1) continue;
        if (ch >= 0) {
            const Node &k = T.nodes[ch];
            M = M + k.mass;
            for (int a = 0; a < D; ++a) {
                S[a] = S[a] + k.mass * k.com[a];
                bmin[a] = std::min(bmin[a], k.bmin[a]); bmax[a] = std::max(bmax[a], k.bmax[a]);
            }
            hmax = std::max(hmax, k.hmax);
        } else {
            for (int p = nd.plo[c]; p < nd.phi[c]; ++p) {
                M = M + T.sm[p];
                for (int a = 0; a < D; ++a) {
                    S[a] = S[a] + T.sm[p] * T.sx[a][p];
                    bmin[a] = std::min(bmin[a], T.sx[a][p]); bmax[a] = std::max(bmax[a], T.sx[a][p]);
                }
                hmax = std::max(hmax, T.sh[p]);
            }
        }
    }
    nd.mass = M;
    for (int a = 0; a < 3; ++a) { nd.com[a] = (a < D) ? S[a] / M : 0.0; nd.bmin[a] = bmin[a]; nd.bmax[a] = bmax[a]; }
    nd.hmax = hmax;
}

void *orc_tree_build(int D, i64 n, int L, const double *x, const double *y, const double *z,
                     const double *m, const double *h) {
    Tree *T = new Tree();
    T->D = D; T->L = L; T->n = n;
    T->key.resize(n); T->perm.resize(n);
    orc_order(D, n, x, y, z, L, T->key.data(), T->perm.data(), T->xmin, &T->s0);
    const double *X[3] = {x, y, z};
    for (int a = 0; a < 3; ++a) { T->sx[a].resize(n); for (i64 i = 0; i < n; ++i) T->sx[a][i] = (a < D) ? X[a][T->perm[i]] : 0.0; }
    T->sm.resize(n); T->sh.resize(n);
    for (i64 i = 0; i < n; ++i) { T->sm[i] = m[T->perm[i]]; T->sh[i] = h[T->perm[i]]; }
    T->nodes.reserve((size_t)n);
    if (n >= 2) {
        int r = build_rec(*T, 0, (int)n, 0);
        if (r >= 0) moments_rec(*T, 0);
    }
    return T;
}

void orc_tree_free(void *t) { delete (Tree *)t; }
int orc_tree_nnodes(void *t) { return (int)((Tree *)t)->nodes.size(); }
double orc_tree_s0(void *t) { return ((Tree *)t)->s0; }
void orc_tree_order(void *t, u64 *key, int *perm) {
    Tree *T = (Tree *)t;
    std::memcpy(key, T->key.data(), sizeof(u64) * T->n);
    std::memcpy(perm, T->perm.data(), sizeof(int) * T->n);
}

// Canonical node list sorted by (level, prefix).  child entries are not exported (ids
// are build-order dependent); ranges are.
void orc_tree_get(void *t, int *level, u64 *prefix, int *lo, int *hi, double *mass, double *com,
                  double *bmin, double *bmax, double *hmax) {
    Tree *T = (Tree *)t;
    int nn = (int)T->nodes.size();
    std::vector<int> o(nn);
    for (int i = 0; i < nn; ++i) o[i] = i;
    std::sort(o.begin(), o.end(), [&](int a, int b) {
        const Node &A = T->nodes[a], &B = T->nodes[b];
        return A.level != B.level ? A.level < B.level : A.prefix < B.prefix;
    });
    for (int i = 0; i < nn; ++i) {
        const Node &N = T->nodes[o[i]];
        level[i] = N.level; prefix[i] = N.prefix; lo[i] = N.lo; hi[i] = N.hi; mass[i] = N.mass;
        for (int a = 0; a < 3; ++a) { com[3 * i + a] = N.com[a]; bmin[3 * i + a] = N.bmin[a]; bmax[3 * i + a] = N.bmax[a]; }
        hmax[i] = N.hmax;
    }
}

// -------------------------------------------------------------------------------------
// O2. Interaction partners ("distance ... smaller than the smoothing length";
// variable h: mean smoothing length, eq. 72; symmetric set, U4).
// Brute force over all particles IS the definition.
// -------------------------------------------------------------------------------------
static inline double dist2(const orc_state *s, int D, i64 a, i64 b) {
    double dx = s->x[0][a] - s->x[0][b];
    double dy = s->x[1][a] - s->x[1][b];
    double r2 = dx * dx + dy * dy;
    if (D == 3) { double dz = s->x[2][a] - s->x[2][b]; r2 = r2 + dz * dz; }
    return r2;
}

static inline bool is_partner(const orc_cfg *c, const orc_state *s, i64 a, i64 b) {
    if (a == b) return false;
    double r2 = dist2(s, c->dim, a, b);
    double H = (c->flags & F_VARIABLE_H) ? 0.5 * (s->h[a] + s->h[b]) : s->h[a];
    return r2 < H * H;
}

// Two-call protocol: idx == NULL -> only off[] is filled.  Returns total count.
i64 orc_neighbours_brute(const orc_cfg *c, const orc_state *s, i64 nt, const i64 *targets,
                         i64 *off, int *idx) {
    std::vector<i64> cnt(nt, 0);
#pragma omp parallel for schedule(dynamic, 16)
    for (i64 t = 0; t < nt; ++t) {
        i64 a = targets[t], k = 0;
        for (i64 b = 0; b < c->n; ++b) if (is_partner(c, s, a, b)) ++k;
        cnt[t] = k;
    }
    off[0] = 0;
    for (i64 t = 0; t < nt; ++t) off[t + 1] = off[t] + cnt[t];
    if (idx) {
#pragma omp parallel for schedule(dynamic, 16)
        for (i64 t = 0; t < nt; ++t) {
            i64 a = targets[t], k = off[t];
            for (i64 b = 0; b < c->n; ++b) if (is_partner(c, s, a, b)) idx[k++] = (int)b;
        }
    }
    return off[nt];
}

// n_a of eq. 73: partners within the particle's OWN h (U5).
void orc_count_own_h(const orc_cfg *c, const orc_state *s, i64 nt, const i64 *targets, int *n_a) {
#pragma omp parallel for schedule(dynamic, 16)
    for (i64 t = 0; t < nt; ++t) {
        i64 a = targets[t]; int k = 0;
        for (i64 b = 0; b < c->n; ++b) {
            if (b == a) continue;
            if (dist2(s, c->dim, a, b) < s->h[a] * s->h[a]) ++k;
        }
        n_a[t] = k;
    }
}

// eq. 73: h_new = h * 1/2 (1 + (n_des/n_a)^(1/D)), n_a clamped to >= 1 (U5)
void orc_h_update(int D, i64 n, const double *h, const int *n_a, int n_des, double *h_new) {
    for (i64 i = 0; i < n; ++i) {
        double ratio = (double)n_des / (double)std::max(n_a[i], 1);
        double root = (D == 3) ? std::cbrt(ratio) : (D == 2) ? std::sqrt(ratio) : ratio;
        h_new[i] = h[i] * 0.5 * (1.0 + root);
    }
}

// Tree-walk search of the paper (eq. 69): descend into a node when the
// particle lies inside the cube of half-edge s/2 + h around the node's centre; at a leaf
// apply the exact test above.  With variable h the reach is (h_a + hmax_node)/2.
// A small slack keeps the walk conservative; membership is decided by is_partner alone.
static void nb_walk(const Tree &T, const orc_cfg *c, const orc_state *s, i64 a, int id,
                    std::vector<int> &out, bool own_h) {
    const int D = T.D, NC = 1 << D;
    const Node &nd = T.nodes[id];
    for (int ch = 0; ch < NC; ++ch) {
        int k = nd.child[ch];
        if (k == -1) continue;
        if (k >= 0) {
            const Node &kn = T.nodes[k];
            double sl = std::ldexp(T.s0, -kn.level);
            double reach = ((c->flags & F_VARIABLE_H) && !own_h) ? 0.5 * (s->h[a] + kn.hmax) : s->h[a];
            double half = 0.5 * sl + reach * (1.0 + 1e-9) + sl * 1e-9;
            bool inside = true;
            u64 pf = kn.prefix;
            for (int ax = 0; ax < D && inside; ++ax) {
                u64 g = 0;                       // de-interleave the cell's integer coordinate
                for (int b = 0; b < kn.level; ++b) g |= ((pf >> (D * b + ax)) & 1ull) << b;
                double centre = T.xmin[ax] + ((double)g + 0.5) * sl;
                if (std::fabs(s->x[ax][a] - centre) > half) inside = false;
            }
            if (inside) nb_walk(T, c, s, a, k, out, own_h);
        } else {
            for (int p = nd.plo[ch]; p < nd.phi[ch]; ++p) {
                i64 b = T.perm[p];
                bool in = own_h ? (b != a && dist2(s, c->dim, a, b) < s->h[a] * s->h[a]) : is_partner(c, s, a, b);
                if (in) out.push_back((int)b);
            }
        }
    }
}

i64 orc_neighbours_tree(void *t, const orc_cfg *c, const orc_state *s, i64 nt, const i64 *targets,
                        i64 *off, int *idx, i64 cap, int own_h) {
    const Tree &T = *(Tree *)t;
    std::vector<std::vector<int>> lists(nt);
    if (!T.nodes.empty()) {
#pragma omp parallel for schedule(dynamic, 64)
        for (i64 k = 0; k < nt; ++k) {
            nb_walk(T, c, s, targets[k], 0, lists[k], own_h != 0);
            std::sort(lists[k].begin(), lists[k].end());
        }
    } else {
        // no internal node: n < 2 or all keys equal -> fall back to the definition
        for (i64 k = 0; k < nt; ++k)
            for (i64 b = 0; b < c->n; ++b) {
                i64 a = targets[k];
                bool in = own_h ? (b != a && dist2(s, c->dim, a, b) < s->h[a] * s->h[a]) : is_partner(c, s, a, b);
                if (in) lists[k].push_back((int)b);
            }
    }
    off[0] = 0;
    for (i64 k = 0; k < nt; ++k) off[k + 1] = off[k] + (i64)lists[k].size();
    if (idx && off[nt] <= cap)
        for (i64 k = 0; k < nt; ++k) std::copy(lists[k].begin(), lists[k].end(), idx + off[k]);
    return off[nt];
}

// -------------------------------------------------------------------------------------
// O4.1  Density by kernel sum, PAPER.md:236 (eq. 28), self term included (U7).
// -------------------------------------------------------------------------------------
void orc_density(const orc_cfg *c, const orc_state *s, i64 nt, const i64 *targets, const i64 *off,
                 const int *idx, double *rho_out) {
    const int D = c->dim;
#pragma omp parallel for schedule(dynamic, 64)
    for (i64 t = 0; t < nt; ++t) {
        i64 a = targets[t];
        double rho = s->m[a] * orc_W(D, 0.0, s->h[a]);
        for (i64 k = off[t]; k < off[t + 1]; ++k) {
            i64 b = idx[k];
            double H = (c->flags & F_VARIABLE_H) ? 0.5 * (s->h[a] + s->h[b]) : s->h[a];
            rho += s->m[b] * orc_W(D, std::sqrt(dist2(s, D, a, b)), H);
        }
        rho_out[t] = rho;
    }
}

// -------------------------------------------------------------------------------------
// O4.2  Per-particle pre-pass: EoS, von Mises limiter (eqs. 16-18, as
// printed: f_Y = min[Y0^2 / 3 J2, 1], U9), damaged stress (eqs. 20-21).
// The state variable dmg is d^(1/3) (eq. 46), so d = dmg^3.
// Outputs per particle: p, cs, sigma[6] (the stress entering eqs. 30/31), St[6] (limited S).
// -------------------------------------------------------------------------------------
static const int IX[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};   // S[6] = xx xy xz yy yz zz

void orc_prepass(const orc_cfg *c, const orc_mat *mats, const orc_state *s, double *p, double *cs,
                 double *sigma, double *St) {
    const int D = c->dim;
    const i64 n = c->n;
    for (i64 a = 0; a < n; ++a) {
        const orc_mat *mt = &mats[s->mat[a]];
        orc_eos(mt, s->rho[a], s->u[a], &p[a], &cs[a]);
        double Sl[6] = {0, 0, 0, 0, 0, 0};
        if (c->flags & F_SOLID) {
            for (int k = 0; k < 6; ++k) Sl[k] = s->S[k][a];
            if (D == 2) { Sl[2] = Sl[4] = Sl[5] = 0.0; }
            if ((c->flags & F_PLASTIC) && mt->Y0 > 0.0) {
                double SS = 0.0;
                for (int al = 0; al < D; ++al) for (int be = 0; be < D; ++be) SS += Sl[IX[al][be]] * Sl[IX[al][be]];
                double J2 = 0.5 * SS;                                   // eq. 18
                double fY = 1.0;
                if (3.0 * J2 > mt->Y0 * mt->Y0) fY = mt->Y0 * mt->Y0 / (3.0 * J2);   // eq. 17
                for (int k = 0; k < 6; ++k) Sl[k] = fY * Sl[k];        // eq. 16
            }
        }
        double d = 0.0;
        if ((c->flags & F_DAMAGE) && mt->brittle) d = s->dmg[a] * s->dmg[a] * s->dmg[a];
        double phat = (p[a] >= 0.0) ? p[a] : (1.0 - d) * p[a];         // eq. 21
        for (int k = 0; k < 6; ++k) { St[6 * a + k] = Sl[k]; sigma[6 * a + k] = (1.0 - d) * Sl[k]; }   // eq. 20
        for (int al = 0; al < D; ++al) sigma[6 * a + IX[al][al]] -= phat;
    }
}

// Largest eigenvalue of a symmetric DxD matrix by cyclic Jacobi rotations (textbook).
static double max_eig_sym(int D, const double A_in[3][3]) {
    double A[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) A[i][j] = (i < D && j < D) ? A_in[i][j] : 0.0;
    for (int sweep = 0; sweep < 64; ++sweep) {
        double offn = 0.0;
        for (int i = 0; i < D; ++i) for (int j = i + 1; j < D; ++j) offn += A[i][j] * A[i][j];
        if (offn == 0.0) break;
        for (int p = 0; p < D; ++p) for (int q = p + 1; q < D; ++q) {
            if (A[p][q] == 0.0) continue;
            double th = (A[q][q] - A[p][p]) / (2.0 * A[p][q]);
            double t = ((th >= 0.0) ? 1.0 : -1.0) / (std::fabs(th) + std::sqrt(th * th + 1.0));
            double cs = 1.0 / std::sqrt(t * t + 1.0), sn = t * cs;
            for (int k = 0; k < D; ++k) {           // A <- A J
                double akp = A[k][p], akq = A[k][q];
                A[k][p] = cs * akp - sn * akq; A[k][q] = sn * akp + cs * akq;
            }
            for (int k = 0; k < D; ++k) {           // A <- J^T A
                double apk = A[p][k], aqk = A[q][k];
                A[p][k] = cs * apk - sn * aqk; A[q][k] = sn * apk + cs * aqk;
            }
        }
    }
    double e = A[0][0];
    for (int i = 1; i < D; ++i) e = std::max(e, A[i][i]);
    return e;
}

double orc_max_eig(int D, const double *a9) {
    double A[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) A[i][j] = a9[3 * i + j];
    return max_eig_sym(D, A);
}

static bool invert(int D, const double N[3][3], double C[3][3], double *det_out) {
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) C[i][j] = (i == j) ? 1.0 : 0.0;
    if (D == 2) {
        double det = N[0][0] * N[1][1] - N[0][1] * N[1][0];
        *det_out = det;
        if (!(std::fabs(det) >= 1e-12)) return false;
        C[0][0] = N[1][1] / det; C[0][1] = -N[0][1] / det;
        C[1][0] = -N[1][0] / det; C[1][1] = N[0][0] / det;
        return true;
    }
    double c00 = N[1][1] * N[2][2] - N[1][2] * N[2][1];
    double c01 = N[1][2] * N[2][0] - N[1][0] * N[2][2];
    double c02 = N[1][0] * N[2][1] - N[1][1] * N[2][0];
    double det = N[0][0] * c00 + N[0][1] * c01 + N[0][2] * c02;
    *det_out = det;
    if (!(std::fabs(det) >= 1e-12)) return false;
    C[0][0] = c00 / det;
    C[0][1] = (N[0][2] * N[2][1] - N[0][1] * N[2][2]) / det;
    C[0][2] = (N[0][1] * N[1][2] - N[0][2] * N[1][1]) / det;
    C[1][0] = c01 / det;
    C[1][1] = (N[0][0] * N[2][2] - N[0][2] * N[2][0]) / det;
    C[1][2] = (N[0][2] * N[1][0] - N[0][0] * N[1][2]) / det;
    C[2][0] = c02 / det;
    C[2][1] = (N[0][1] * N[2][0] - N[0][0] * N[2][1]) / det;
    C[2][2] = (N[0][0] * N[1][1] - N[0][1] * N[1][0]) / det;
    return true;
}

// -------------------------------------------------------------------------------------
// O4.3-O4.5  SPH rates of one evaluation for the target particles, given their partner
// lists (CSR, original indices) and the pre-pass arrays of ALL particles.
//   continuity   PAPER.md:242 (eq. 29)            gradient w.r.t. x_a (U2)
//   momentum     PAPER.md:247, :276 (eqs. 30, 34) gradient w.r.t. x_a, -Pi* delta (U2, U3)
//   energy       PAPER.md:254 (eq. 31)            as printed (d/dx_b = -d/dx_a), AV included (U3)
//   viscosity    PAPER.md:263-278 (eqs. 32-33)    (U10)
//   grad v       PAPER.md:317-330 (eqs. 41-44)    C = inverse of the (x_b - x_a) matrix (U6, U17)
//   dS/dt        PAPER.md:83-96 (eqs. 7-10)       1/D in the trace term (U8)
//   damage       PAPER.md:344-360 (eqs. 46-49), :189 (eq. 24 repaired, U16), U18-U20
//   art. stress  PAPER.md:284-302 (eqs. 35-38)    zeta = -eps_s sigma/rho^2 per component in tension (U25),
//                                                 f = W_ab / W(dmpd), same term in the energy sum (U3)
//   XSPH         PAPER.md:311 (eq. 40)            2 m_b / (rho_a + rho_b) (U26)
// -------------------------------------------------------------------------------------
void orc_rhs(const orc_cfg *c, const orc_mat *mats, const orc_state *s, const double *p,
             const double *cs, const double *sigma, const double *St, i64 nt, const i64 *targets,
             const i64 *off, const int *idx, orc_rates *o) {
    const int D = c->dim;
    const bool solid = (c->flags & F_SOLID) != 0, varh = (c->flags & F_VARIABLE_H) != 0;
    const bool art = (c->flags & F_ART_STRESS) != 0, xsph = (c->flags & F_XSPH) != 0;
    (void)p;
#pragma omp parallel for schedule(dynamic, 64)
    for (i64 t = 0; t < nt; ++t) {
        const i64 a = targets[t];
        const i64 k0 = off[t], k1 = off[t + 1];
        const orc_mat *mt = &mats[s->mat[a]];
        const double rho_a = s->rho[a];

        // ---- correction tensor (eq. 43 with the sign of eq. 44, U6) ----
        double C[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
        if (solid) {
            double N[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
            for (i64 k = k0; k < k1; ++k) {
                i64 b = idx[k];
                double dx[3] = {0, 0, 0};
                for (int al = 0; al < D; ++al) dx[al] = s->x[al][a] - s->x[al][b];
                double r = std::sqrt(dist2(s, D, a, b));
                double H = varh ? 0.5 * (s->h[a] + s->h[b]) : s->h[a];
                double dW = orc_dW(D, r, H);
                double Vb = s->m[b] / s->rho[b];
                for (int al = 0; al < D; ++al) for (int ga = 0; ga < D; ++ga) {
                    double gW = (r > 0.0) ? dW * dx[ga] / r : 0.0;       // dW_ab/dx_a^gamma
                    N[al][ga] += Vb * (-dx[al]) * gW;                    // (x_b - x_a)^alpha
                }
            }
            double det;
            double Ci[3][3];
            if ((k1 - k0) >= D + 1 && invert(D, N, Ci, &det))            // U17
                for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) C[i][j] = Ci[i][j];
        }

        // ---- pair sums ----
        double drho = 0, dv[3] = {0, 0, 0}, du = 0, gv[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
        double xs[3] = {0, 0, 0}, Axs[3] = {0, 0, 0};
        double Adrho = 0, Adv[3] = {0, 0, 0}, Adu = 0, Agv[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
        for (i64 k = k0; k < k1; ++k) {
            i64 b = idx[k];
            double dx[3] = {0, 0, 0}, dvv[3] = {0, 0, 0};
            for (int al = 0; al < D; ++al) { dx[al] = s->x[al][a] - s->x[al][b]; dvv[al] = s->v[al][a] - s->v[al][b]; }
            double r2 = dist2(s, D, a, b);
            double r = std::sqrt(r2);
            double H = varh ? 0.5 * (s->h[a] + s->h[b]) : s->h[a];
            double dW = orc_dW(D, r, H);
            double gW[3] = {0, 0, 0};
            for (int be = 0; be < D; ++be) gW[be] = (r > 0.0) ? dW * dx[be] / r : 0.0;
            double Vb = s->m[b] / s->rho[b];
            double vr = 0.0, vgW = 0.0;
            for (int al = 0; al < D; ++al) { vr += dvv[al] * dx[al]; vgW += dvv[al] * gW[al]; }
            // eq. 29
            drho += Vb * vgW;  Adrho += std::fabs(Vb * vgW);
            // eqs. 32-33
            double Pi = 0.0;
            if (vr < 0.0) {
                double Hb = 0.5 * (s->h[a] + s->h[b]);
                double cb = 0.5 * (cs[a] + cs[b]);
                double rb = 0.5 * (rho_a + s->rho[b]);
                double nu = Hb * vr / (r2 + c->av_eps * Hb * Hb);
                Pi = (-c->av_alpha * cb * nu + c->av_beta * nu * nu) / rb;
            }
            // T_ab = sigma_a/rho_a^2 + sigma_b/rho_b^2 - Pi* delta  (eqs. 30, 34)
            double Tm[3][3];
            for (int al = 0; al < D; ++al) for (int be = 0; be < D; ++be) {
                Tm[al][be] = sigma[6 * a + IX[al][be]] / (rho_a * rho_a) + sigma[6 * b + IX[al][be]] / (s->rho[b] * s->rho[b]);
                if (al == be) Tm[al][be] -= Pi;
            }
            if (art) {                                                   // eqs. 35-38
                double f = orc_W(D, r, H) / orc_W(D, c->as_mpd, H);      // eq. 38
                double fn = std::pow(f, c->as_n);
                for (int al = 0; al < D; ++al) for (int be = 0; be < D; ++be) {
                    double sa = sigma[6 * a + IX[al][be]] / (rho_a * rho_a);
                    double sb = sigma[6 * b + IX[al][be]] / (s->rho[b] * s->rho[b]);
                    double za = (sa > 0.0) ? -c->as_eps * sa : 0.0;      // eq. 37: tension only (U25)
                    double zb = (sb > 0.0) ? -c->as_eps * sb : 0.0;
                    Tm[al][be] += (za + zb) * fn;                        // eqs. 35-36
                }
            }
            if (xsph) {                                                  // eq. 40 (U26)
                double wgt = c->xsph * 2.0 * s->m[b] / (rho_a + s->rho[b]) * orc_W(D, r, H);
                for (int al = 0; al < D; ++al) { xs[al] += wgt * (-dvv[al]); Axs[al] += std::fabs(wgt * dvv[al]); }
            }
            double e = 0.0;
            for (int al = 0; al < D; ++al) {
                double f = 0.0;
                for (int be = 0; be < D; ++be) f += Tm[al][be] * gW[be];
                dv[al] += s->m[b] * f;  Adv[al] += std::fabs(s->m[b] * f);
                e += f * dvv[al];
            }
            du += -0.5 * s->m[b] * e;  Adu += std::fabs(0.5 * s->m[b] * e);
            if (solid) {
                double gWC[3] = {0, 0, 0};
                for (int be = 0; be < D; ++be) for (int ga = 0; ga < D; ++ga) gWC[be] += gW[ga] * C[ga][be];   // eq. 42
                for (int al = 0; al < D; ++al) for (int be = 0; be < D; ++be) {
                    double term = Vb * (-dvv[al]) * gWC[be];              // (v_b - v_a)^alpha
                    gv[al][be] += term;  Agv[al][be] += std::fabs(term);
                }
            }
        }
        drho = rho_a * drho;  Adrho = std::fabs(rho_a) * Adrho;
        o->drho[t] = drho; o->du[t] = du; o->A_drho[t] = Adrho; o->A_du[t] = Adu;
        for (int al = 0; al < 3; ++al) { o->dv[al][t] = dv[al]; o->A_dv[al][t] = Adv[al]; }
        for (int al = 0; al < 3; ++al) { o->dxs[al][t] = xs[al]; o->A_dxs[al][t] = Axs[al]; }
        for (int al = 0; al < 3; ++al) for (int be = 0; be < 3; ++be) {
            o->gradv[3 * al + be][t] = gv[al][be]; o->A_gradv[3 * al + be][t] = Agv[al][be];
            o->C[3 * al + be][t] = C[al][be];
        }

        // ---- epilogue: dS/dt (eqs. 7-10) ----
        double dS[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, AdS[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
        if (solid) {
            double eps[3][3], R[3][3], Ae[3][3], Sm[3][3];
            double tr = 0.0, Atr = 0.0;
            for (int al = 0; al < 3; ++al) for (int be = 0; be < 3; ++be) {
                eps[al][be] = 0.5 * (gv[al][be] + gv[be][al]);            // eq. 8
                R[al][be] = 0.5 * (gv[al][be] - gv[be][al]);              // eq. 10
                Ae[al][be] = 0.5 * (Agv[al][be] + Agv[be][al]);
                Sm[al][be] = St[6 * a + IX[al][be]];
            }
            for (int al = 0; al < D; ++al) { tr += eps[al][al]; Atr += Ae[al][al]; }
            for (int al = 0; al < D; ++al) for (int be = 0; be < D; ++be) {
                double v = 2.0 * mt->mu * (eps[al][be] - ((al == be) ? tr / D : 0.0));   // eq. 7, 1/D (U8)
                double Av = 2.0 * mt->mu * (Ae[al][be] + ((al == be) ? Atr / D : 0.0));
                for (int ga = 0; ga < D; ++ga) {
                    v += Sm[al][ga] * R[ga][be] - R[al][ga] * Sm[ga][be];               // eq. 9
                    Av += std::fabs(Sm[al][ga]) * Ae[ga][be] + Ae[al][ga] * std::fabs(Sm[ga][be]);
                }
                dS[al][be] = v; AdS[al][be] = Av;
            }
        }
        for (int al = 0; al < 3; ++al) for (int be = al; be < 3; ++be) {
            o->dS[IX[al][be]][t] = dS[al][be]; o->A_dS[IX[al][be]][t] = AdS[al][be];
        }

        // ---- epilogue: Grady-Kipp damage ----
        double ddmg = 0.0, strain = 0.0;
        int nact = s->n_act ? s->n_act[a] : 0;
        if ((c->flags & F_DAMAGE) && mt->brittle) {
            double dm = s->dmg[a];
            double d = dm * dm * dm;
            i64 f0 = s->flaw_off[a], f1 = s->flaw_off[a + 1];
            i64 ntot = f1 - f0;
            if (d < 1.0 && ntot > 0) {
                double Sg[3][3];
                for (int al = 0; al < 3; ++al) for (int be = 0; be < 3; ++be) Sg[al][be] = sigma[6 * a + IX[al][be]];
                double smax = max_eig_sym(D, Sg);                         // principal stress
                double K = (mt->eos == 2) ? mt->tA : mt->K0;             // U18
                double E = 9.0 * K * mt->mu / (3.0 * K + mt->mu);        // eq. 49
                strain = smax / ((1.0 - d) * E);                          // eq. 48
                int cnt = 0;
                for (i64 j = f0; j < f1; ++j) if (s->flaw_eps[j] <= strain) ++cnt;
                nact = std::max(nact, cnt);                               // latched (U19)
                double cg = 0.4 * std::sqrt((K + 4.0 / 3.0 * (1.0 - d) * mt->mu) / rho_a);   // eq. 24 repaired (U16)
                if (d < (double)nact / (double)ntot) ddmg = (double)nact * cg / s->h[a];     // eqs. 46-47, R_s = h (U16, U20)
            }
        }
        o->ddmg[t] = ddmg; o->strain[t] = strain; o->n_act[t] = nact;
    }
}

// -------------------------------------------------------------------------------------
// O5. Gravity.  Tree walk with the opening criterion s/r < theta (eq. 50)
// taken as s*s < (theta*theta)*r2 on the unsoftened distance, monopoles only
// (PAPER.md:380); force PAPER.md:376 (eq. 51) with attractive sign and Plummer softening
// (U21).  Particles at zero distance contribute nothing (direction undefined).
// -------------------------------------------------------------------------------------
struct GravAcc { double a[3]; double A[3]; i64 n_inter; i64 n_test, n_open; };   // n_test: opening tests (eq. 50), n_open: of those, cells opened

static inline void grav_add(GravAcc &g, int D, double G, double M, const double dx[3], double r2, double eps2) {
    double r2e = r2 + eps2;
    double f = G * M / (r2e * std::sqrt(r2e));
    for (int al = 0; al < D; ++al) { g.a[al] -= f * dx[al]; g.A[al] += std::fabs(f * dx[al]); }
    g.n_inter++;
}

static void grav_walk(const Tree &T, const orc_cfg *c, int id, int psorted, GravAcc &g) {
    const int D = T.D, NC = 1 << D;
    const Node &nd = T.nodes[id];
    const double th2 = c->theta * c->theta, eps2 = c->eps_soft * c->eps_soft;
    for (int ch = 0; ch < NC; ++ch) {
        int k = nd.child[ch];
        if (k == -1) continue;
        if (k >= 0) {
            const Node &kn = T.nodes[k];
            double dx[3] = {0, 0, 0};
            for (int al = 0; al < D; ++al) dx[al] = T.sx[al][psorted] - kn.com[al];
            double r2 = dx[0] * dx[0] + dx[1] * dx[1];
            if (D == 3) r2 = r2 + dx[2] * dx[2];
            double sl = std::ldexp(T.s0, -kn.level);                      // eq. 68
            g.n_test++;
            if (sl * sl < th2 * r2) grav_add(g, D, c->G, kn.mass, dx, r2, eps2);
            else { g.n_open++; grav_walk(T, c, k, psorted, g); }
        } else {
            for (int p = nd.plo[ch]; p < nd.phi[ch]; ++p) {
                if (p == psorted) continue;
                double dx[3] = {0, 0, 0};
                for (int al = 0; al < D; ++al) dx[al] = T.sx[al][psorted] - T.sx[al][p];
                double r2 = dx[0] * dx[0] + dx[1] * dx[1];
                if (D == 3) r2 = r2 + dx[2] * dx[2];
                if (r2 > 0.0) grav_add(g, D, c->G, T.sm[p], dx, r2, eps2);
            }
        }
    }
}

// targets are ORIGINAL indices; ag is (3, nt) row-major; A_ag likewise; n_inter per target.
// n_test / n_open (may be NULL): opening tests evaluated and cells opened, per target (work counters only).
void orc_gravity_tree(void *t, const orc_cfg *c, i64 nt, const i64 *targets, double *ag, double *A_ag,
                      i64 *n_inter, i64 *n_test, i64 *n_open) {
    const Tree &T = *(Tree *)t;
    std::vector<int> inv(T.n);
    for (i64 i = 0; i < T.n; ++i) inv[T.perm[i]] = (int)i;
#pragma omp parallel for schedule(dynamic, 16)
    for (i64 k = 0; k < nt; ++k) {
        GravAcc g = {{0, 0, 0}, {0, 0, 0}, 0, 0, 0};
        int ps = inv[targets[k]];
        if (!T.nodes.empty()) {
            // the root itself is always opened: the particle lies inside it (s/r >= 1/sqrt(D) > theta)
            grav_walk(T, c, 0, ps, g);
        } else {
            const double eps2 = c->eps_soft * c->eps_soft;
            for (i64 p = 0; p < T.n; ++p) {
                if (p == ps) continue;
                double dx[3] = {0, 0, 0};
                for (int al = 0; al < T.D; ++al) dx[al] = T.sx[al][ps] - T.sx[al][p];
                double r2 = dx[0] * dx[0] + dx[1] * dx[1];
                if (T.D == 3) r2 = r2 + dx[2] * dx[2];
                if (r2 > 0.0) grav_add(g, T.D, c->G, T.sm[p], dx, r2, eps2);
            }
        }
        for (int al = 0; al < 3; ++al) { ag[al * nt + k] = g.a[al]; A_ag[al * nt + k] = g.A[al]; }
        n_inter[k] = g.n_inter;
        if (n_test) n_test[k] = g.n_test;
        if (n_open) n_open[k] = g.n_open;
    }
}

// Direct summation (the definition tree gravity approximates) and the softened potential.
void orc_gravity_direct(const orc_cfg *c, const orc_state *s, i64 nt, const i64 *targets, double *ag,
                        double *pot) {
    const int D = c->dim;
    const double eps2 = c->eps_soft * c->eps_soft;
#pragma omp parallel for schedule(dynamic, 16)
    for (i64 k = 0; k < nt; ++k) {
        i64 a = targets[k];
        double acc[3] = {0, 0, 0}, ph = 0.0;
        for (i64 b = 0; b < c->n; ++b) {
            if (b == a) continue;
            double dx[3] = {0, 0, 0};
            for (int al = 0; al < D; ++al) dx[al] = s->x[al][a] - s->x[al][b];
            double r2 = dist2(s, D, a, b);
            if (!(r2 > 0.0)) continue;
            double r2e = r2 + eps2;
            double f = c->G * s->m[b] / (r2e * std::sqrt(r2e));
            for (int al = 0; al < D; ++al) acc[al] -= f * dx[al];
            ph -= c->G * s->m[b] / std::sqrt(r2e);
        }
        for (int al = 0; al < 3; ++al) ag[al * nt + k] = acc[al];
        pot[k] = ph;
    }
}

}  // extern "C"
