// A6-A10: density sum, per-particle pre-pass, SPH pair sums and per-particle epilogue.
//
//   k_density : rho_a = sum_b m_b W_ab incl. self term              PAPER.md:236 (eq. 28)
//   k_prepass : EoS (eqs. 13-15), von Mises limiter (eqs. 16-18), damaged stress (eqs. 20-21);
//               stores p, c_s, V = m/rho and sigma/rho^2 so the pair loop has no division by rho
//   k_pairs   : one lane per particle, 32 Morton-consecutive particles per warp, lists read
//               coalesced (group-transposed), neighbour data gathered through L1 (Morton order
//               keeps a warp's k-th partners within a few cache lines):
//                 continuity eq. 29, momentum eqs. 30/34, energy eq. 31, viscosity eqs. 32-33,
//                 moment matrix of eqs. 43/44 and the uncorrected velocity-gradient sum.
//               The correction tensor C_a is constant per particle, so
//                 sum_b V_b dv^a (gradW . C) = (sum_b V_b dv^a gradW) . C
//               and ONE pass over the list yields both the matrix and the gradient (the paper's
//               formulation needs the inverse before the second sum, i.e. two passes).
//               Epilogue in the same kernel: C = N^-1 (eqs. 42-44), strain and rotation rates
//               (eqs. 8, 10), dS/dt (eqs. 7, 9), Grady-Kipp damage (eqs. 46-49, 24).
#include "sph_internal.cuh"

struct DevMats { const sph_material *m; };

__device__ __forceinline__ void eos_eval(const sph_material &mt, double rho, double u, double &p, double &cs) {
    if (mt.eos == SPH_EOS_IDEAL_GAS) {
        p = (mt.gamma - 1.0) * rho * u;
        cs = sqrt(mt.gamma * (mt.gamma - 1.0) * u);
    } else if (mt.eos == SPH_EOS_MURNAGHAN) {
        p = mt.K0 / mt.nM * (pow(rho / mt.rho0, mt.nM) - 1.0);
        cs = sqrt(mt.K0 / mt.rho0);
    } else {
        const double eta = rho / mt.rho0, chi = eta - 1.0;
        const double om = u / (mt.tE0 * eta * eta) + 1.0;
        const double pc = (mt.ta + mt.tb / om) * rho * u + mt.tA * chi + mt.tB * chi * chi;
        if (eta >= 1.0 || u <= mt.tEiv) p = pc;
        else {
            const double z = mt.rho0 / rho - 1.0;
            const double pe = mt.ta * rho * u + (mt.tb * rho * u / om + mt.tA * chi * exp(-mt.tbeta * z)) * exp(-mt.talpha * z * z);
            if (u >= mt.tEcv) p = pe;
            else p = ((u - mt.tEiv) * pe + (mt.tEcv - u) * pc) / (mt.tEcv - mt.tEiv);
        }
        cs = sqrt(mt.tA / mt.rho0);
    }
}

// S[6] = xx xy xz yy yz zz.  Returns f_Y of eq. 17 (as printed: Y0^2 / 3 J2, no square root).
template <int D>
__device__ __forceinline__ double yield_factor(const sph_material &mt, int flags, const double S[6]) {
    if (!(flags & SPH_F_PLASTIC) || !(mt.Y0 > 0.0)) return 1.0;
    double SS;
    if (D == 3) SS = S[0] * S[0] + S[3] * S[3] + S[5] * S[5] + 2.0 * (S[1] * S[1] + S[2] * S[2] + S[4] * S[4]);
    else SS = S[0] * S[0] + S[3] * S[3] + 2.0 * S[1] * S[1];
    const double J2 = 0.5 * SS;
    const double Y2 = mt.Y0 * mt.Y0;
    return (3.0 * J2 > Y2) ? Y2 / (3.0 * J2) : 1.0;
}

template <int D>
__global__ void k_prepass(Dev d, const sph_material *mats) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.n) return;
    const sph_material mt = mats[d.smat[i]];
    const double rho = d.srho[i], u = d.su[i];
    double p, cs;
    eos_eval(mt, rho, u, p, cs);
    double S[6] = {0, 0, 0, 0, 0, 0};
    if (d.flags & SPH_F_SOLID) {
        for (int k = 0; k < 6; ++k) S[k] = d.sS[k][i];
        if (D == 2) { S[2] = 0.0; S[4] = 0.0; S[5] = 0.0; }
        const double fY = yield_factor<D>(mt, d.flags, S);
        for (int k = 0; k < 6; ++k) S[k] *= fY;
    }
    double dd = 0.0;
    if ((d.flags & SPH_F_DAMAGE) && mt.brittle) { const double g = d.sdmg[i]; dd = g * g * g; }
    const double phat = (p >= 0.0) ? p : (1.0 - dd) * p;
    const double ir2 = 1.0 / (rho * rho);
    double sg[6];
    for (int k = 0; k < 6; ++k) sg[k] = (1.0 - dd) * S[k];
    sg[0] -= phat; sg[3] -= phat;
    if (D == 3) sg[5] -= phat;
    for (int k = 0; k < 6; ++k) d.sr2[k][i] = sg[k] * ir2;
    d.p[i] = p;
    d.cs[i] = cs;
    d.vol[i] = d.sm[i] / rho;
}

template <int D> struct KNorm;
template <> struct KNorm<2> { static constexpr double s = 40.0 / (7.0 * 3.14159265358979323846); };
template <> struct KNorm<3> { static constexpr double s = 8.0 / 3.14159265358979323846; };

template <int D, bool VARH>
__global__ void __launch_bounds__(128) k_density(Dev d) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const int g = i >> 5;
    if (g * 32 >= d.n) return;
    const bool valid = i < d.n;
    const int ii = valid ? i : d.n - 1;
    const double xi = d.sx[0][ii], yi = d.sx[1][ii], zi = (D == 3) ? d.sx[2][ii] : 0.0, Hi = d.sh[ii];
    const int cnt = valid ? d.nb_cnt[ii] : 0;
    int mx = cnt;
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    const int *nbw = d.nb + (size_t)g * d.cap * 32 + lane;
    const double iHi = 1.0 / Hi;
    double rho = d.sm[ii] * KNorm<D>::s * ((D == 3) ? iHi * iHi * iHi : iHi * iHi);   // self term (q = 0)
    for (int k = 0; k < mx; ++k) {
        if (k < cnt) {
            const int b = nbw[(size_t)k * 32];
            const double dx = xi - d.sx[0][b], dy = yi - d.sx[1][b], dz = (D == 3) ? zi - d.sx[2][b] : 0.0;
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double iH = VARH ? 1.0 / (0.5 * (Hi + d.sh[b])) : iHi;
            const double q = r * iH;
            double f;
            if (q < 0.5) f = 6.0 * q * q * q - 6.0 * q * q + 1.0;
            else { const double t = fmax(1.0 - q, 0.0); f = 2.0 * t * t * t; }
            rho += d.sm[b] * KNorm<D>::s * ((D == 3) ? iH * iH * iH : iH * iH) * f;
        }
    }
    if (valid) { d.srho[i] = rho; d.rho[d.perm[i]] = rho; }
}

// largest eigenvalue of a symmetric DxD matrix, cyclic Jacobi
template <int D>
__device__ double max_eig_jacobi(double A[3][3]) {
    for (int sweep = 0; sweep < 32; ++sweep) {
        double off = 0.0;
        for (int i = 0; i < D; ++i) for (int j = i + 1; j < D; ++j) off += A[i][j] * A[i][j];
        if (off == 0.0) break;
        for (int p = 0; p < D; ++p) for (int q = p + 1; q < D; ++q) {
            if (A[p][q] == 0.0) continue;
            const double th = (A[q][q] - A[p][p]) / (2.0 * A[p][q]);
            const double t = ((th >= 0.0) ? 1.0 : -1.0) / (fabs(th) + sqrt(th * th + 1.0));
            const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
            for (int k = 0; k < D; ++k) { const double a = A[k][p], b = A[k][q]; A[k][p] = c * a - s * b; A[k][q] = s * a + c * b; }
            for (int k = 0; k < D; ++k) { const double a = A[p][k], b = A[q][k]; A[p][k] = c * a - s * b; A[q][k] = s * a + c * b; }
        }
    }
    double e = A[0][0];
    for (int i = 1; i < D; ++i) e = fmax(e, A[i][i]);
    return e;
}

template <int D, bool SOLID, bool VARH>
__global__ void __launch_bounds__(128) k_pairs(Dev d, const sph_material *mats) {
    constexpr int NS = (D == 3) ? 6 : 3;                 // independent stress components
    constexpr int SI[6] = {0, 1, (D == 3) ? 2 : 3, 3, 4, 5};   // 2-D: xx xy yy -> 0 1 3
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const int g = i >> 5;
    if (g * 32 >= d.n) return;
    const bool valid = i < d.n;
    const int ii = valid ? i : d.n - 1;

    double xa[3], va[3], sa[NS];
    for (int a = 0; a < D; ++a) { xa[a] = d.sx[a][ii]; va[a] = d.sv[a][ii]; }
    for (int k = 0; k < NS; ++k) sa[k] = d.sr2[SI[k]][ii];
    const double Hi = d.sh[ii], rhoi = d.srho[ii], csi = d.cs[ii];
    const double iHi = 1.0 / Hi;
    const double fac_i = 6.0 * KNorm<D>::s * ((D == 3) ? (iHi * iHi) * (iHi * iHi) : iHi * iHi * iHi);
    const int cnt = valid ? d.nb_cnt[ii] : 0;
    int mx = cnt;
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    const int *nbw = d.nb + (size_t)g * d.cap * 32 + lane;

    double drho = 0.0, du = 0.0, dv[3] = {0, 0, 0};
    double G[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    double N[6] = {0, 0, 0, 0, 0, 0};                     // symmetric moment matrix xx xy xz yy yz zz

    for (int k = 0; k < mx; ++k) {
        if (k < cnt) {
            const int b = nbw[(size_t)k * 32];
            double dx[3], dvv[3];
            double r2 = 0.0, vr = 0.0;
            for (int a = 0; a < D; ++a) {
                dx[a] = xa[a] - d.sx[a][b];
                dvv[a] = va[a] - d.sv[a][b];
                r2 += dx[a] * dx[a];
                vr += dvv[a] * dx[a];
            }
            const double mb = d.sm[b], rhob = d.srho[b], volb = d.vol[b], hb = d.sh[b];
            const double rinv = (r2 > 0.0) ? rsqrt(r2) : 0.0;
            const double r = r2 * rinv;
            double iH = iHi, fac = fac_i;
            if (VARH) {
                iH = 1.0 / (0.5 * (Hi + hb));
                fac = 6.0 * KNorm<D>::s * ((D == 3) ? (iH * iH) * (iH * iH) : iH * iH * iH);
            }
            const double q = r * iH;
            const double t1 = 1.0 - q;
            const double f = (q < 0.5) ? (3.0 * q - 2.0) * q : -(t1 * t1);
            const double gf = fac * f * rinv;                 // (dW/dr) / r
            double gW[3], vg = 0.0;
            for (int a = 0; a < D; ++a) { gW[a] = gf * dx[a]; vg += dvv[a] * gW[a]; }
            drho += volb * vg;                                // eq. 29
            double Pi = 0.0;
            if (vr < 0.0) {                                   // eqs. 32-33, approaching pairs only
                const double Hb = 0.5 * (Hi + hb), cb = 0.5 * (csi + d.cs[b]), rb = 0.5 * (rhoi + rhob);
                const double den = r2 + d.av_eps * Hb * Hb;
                const double inv = 1.0 / (den * rb);
                const double nu = Hb * vr * rb * inv;
                Pi = nu * (d.av_beta * nu - d.av_alpha * cb) * den * inv;
            }
            double T[NS];
            for (int k2 = 0; k2 < NS; ++k2) T[k2] = sa[k2] + d.sr2[SI[k2]][b];
            double fv[3];
            if (D == 3) {
                T[0] -= Pi; T[3] -= Pi; T[5] -= Pi;
                fv[0] = T[0] * gW[0] + T[1] * gW[1] + T[2] * gW[2];
                fv[1] = T[1] * gW[0] + T[3] * gW[1] + T[4] * gW[2];
                fv[2] = T[2] * gW[0] + T[4] * gW[1] + T[5] * gW[2];
            } else {
                T[0] -= Pi; T[2] -= Pi;
                fv[0] = T[0] * gW[0] + T[1] * gW[1];
                fv[1] = T[1] * gW[0] + T[2] * gW[1];
            }
            double e = 0.0;
            for (int a = 0; a < D; ++a) { dv[a] += mb * fv[a]; e += fv[a] * dvv[a]; }   // eqs. 30/34
            du += mb * e;                                                             // eq. 31 (x -1/2 below)
            if (SOLID) {
                for (int a = 0; a < D; ++a) {
                    const double wa = -volb * dvv[a];         // V_b (v_b - v_a)^alpha
                    for (int c = 0; c < D; ++c) G[a][c] += wa * gW[c];
                }
                const double u0 = -volb * dx[0], u1 = -volb * dx[1];
                N[0] += u0 * gW[0]; N[1] += u0 * gW[1]; N[3] += u1 * gW[1];
                if (D == 3) { const double u2 = -volb * dx[2]; N[2] += u0 * gW[2]; N[4] += u1 * gW[2]; N[5] += u2 * gW[2]; }
            }
        }
    }
    if (!valid) return;

    d.drho[i] = rhoi * drho;
    d.du[i] = -0.5 * du;
    for (int a = 0; a < 3; ++a) d.dv[a][i] = (a < D) ? dv[a] : 0.0;

    const sph_material mt = mats[d.smat[i]];
    double St[6] = {0, 0, 0, 0, 0, 0};
    if (SOLID) {
        // ---- correction tensor, eqs. 42-44 (identity when singular / too few partners, U17) ----
        double C[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
        if (cnt >= D + 1) {
            if (D == 2) {
                const double det = N[0] * N[3] - N[1] * N[1];
                if (fabs(det) >= 1e-12) {
                    const double id = 1.0 / det;
                    C[0][0] = N[3] * id; C[0][1] = -N[1] * id; C[1][0] = -N[1] * id; C[1][1] = N[0] * id;
                }
            } else {
                const double c00 = N[3] * N[5] - N[4] * N[4];
                const double c01 = N[4] * N[2] - N[1] * N[5];
                const double c02 = N[1] * N[4] - N[3] * N[2];
                const double det = N[0] * c00 + N[1] * c01 + N[2] * c02;
                if (fabs(det) >= 1e-12) {
                    const double id = 1.0 / det;
                    C[0][0] = c00 * id; C[0][1] = c01 * id; C[0][2] = c02 * id;
                    C[1][0] = c01 * id; C[1][1] = (N[0] * N[5] - N[2] * N[2]) * id; C[1][2] = (N[2] * N[1] - N[0] * N[4]) * id;
                    C[2][0] = c02 * id; C[2][1] = C[1][2]; C[2][2] = (N[0] * N[3] - N[1] * N[1]) * id;
                }
            }
        }
        double gv[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
        for (int a = 0; a < D; ++a) for (int c = 0; c < D; ++c) {
            double s = 0.0;
            for (int e2 = 0; e2 < D; ++e2) s += G[a][e2] * C[e2][c];
            gv[a][c] = s;
        }
        // ---- dS/dt, eqs. 7-10 (1/D in the trace term, reading U8) ----
        double S[6];
        for (int k = 0; k < 6; ++k) S[k] = d.sS[k][i];
        if (D == 2) { S[2] = 0.0; S[4] = 0.0; S[5] = 0.0; }
        const double fY = yield_factor<D>(mt, d.flags, S);
        for (int k = 0; k < 6; ++k) St[k] = fY * S[k];
        const double Sm[3][3] = {{St[0], St[1], St[2]}, {St[1], St[3], St[4]}, {St[2], St[4], St[5]}};
        double eps[3][3], R[3][3], tr = 0.0;
        for (int a = 0; a < 3; ++a) for (int c = 0; c < 3; ++c) {
            eps[a][c] = 0.5 * (gv[a][c] + gv[c][a]);
            R[a][c] = 0.5 * (gv[a][c] - gv[c][a]);
        }
        for (int a = 0; a < D; ++a) tr += eps[a][a];
        double dS[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
        for (int a = 0; a < D; ++a) for (int c = a; c < D; ++c) {
            double v = 2.0 * mt.mu * (eps[a][c] - ((a == c) ? tr / D : 0.0));
            for (int e2 = 0; e2 < D; ++e2) v += Sm[a][e2] * R[e2][c] - R[a][e2] * Sm[e2][c];
            dS[a][c] = v;
        }
        d.dS[0][i] = dS[0][0]; d.dS[1][i] = dS[0][1]; d.dS[2][i] = dS[0][2];
        d.dS[3][i] = dS[1][1]; d.dS[4][i] = dS[1][2]; d.dS[5][i] = dS[2][2];
    }

    // ---- Grady-Kipp damage, eqs. 46-49, 24 (readings U16, U18-U20) ----
    if (d.flags & SPH_F_DAMAGE) {
        const int orig = d.perm[i];
        int nact = d.n_act[orig];
        double ddmg = 0.0, strain = 0.0;
        if (mt.brittle) {
            const double gdm = d.sdmg[i];
            const double dd = gdm * gdm * gdm;
            const i64 f0 = d.flaw_off[orig], f1 = d.flaw_off[orig + 1];
            const i64 ntot = f1 - f0;
            if (dd < 1.0 && ntot > 0) {
                const double p = d.p[i];
                const double phat = (p >= 0.0) ? p : (1.0 - dd) * p;
                double A[3][3];
                A[0][0] = (1.0 - dd) * St[0] - phat; A[0][1] = A[1][0] = (1.0 - dd) * St[1]; A[0][2] = A[2][0] = (1.0 - dd) * St[2];
                A[1][1] = (1.0 - dd) * St[3] - phat; A[1][2] = A[2][1] = (1.0 - dd) * St[4]; A[2][2] = (1.0 - dd) * St[5] - phat;
                const double smax = max_eig_jacobi<D>(A);
                const double K = (mt.eos == SPH_EOS_TILLOTSON) ? mt.tA : mt.K0;
                const double E = 9.0 * K * mt.mu / (3.0 * K + mt.mu);
                strain = smax / ((1.0 - dd) * E);
                int c = 0;
                for (i64 j = f0; j < f1; ++j) c += (d.flaw_eps[j] <= strain) ? 1 : 0;
                nact = max(nact, c);
                const double cg = 0.4 * sqrt((K + 4.0 / 3.0 * (1.0 - dd) * mt.mu) / rhoi);
                if (dd < (double)nact / (double)ntot) ddmg = (double)nact * cg / Hi;
            }
        }
        d.ddmg[i] = ddmg;
        d.strain[i] = strain;
        d.n_act_new[i] = nact;
    }
}

template <int D>
static void rhs_dim(sph_ctx *ctx, const sph_material *mats) {
    Dev &d = ctx->d;
    const int n = d.n;
    const bool varh = (d.flags & SPH_F_VARIABLE_H) != 0, solid = (d.flags & SPH_F_SOLID) != 0;
    const int gb = sph_ceil_div((i64)sph_ceil_div(n, 32) * 32, 128);
    if (d.flags & SPH_F_DENSITY_SUM) {
        StageTimer tm(ctx, SPH_T_DENSITY);
        if (varh) k_density<D, true><<<gb, 128, 0, ctx->stream>>>(d);
        else k_density<D, false><<<gb, 128, 0, ctx->stream>>>(d);
        ctx->launches += 1;
    }
    {
        StageTimer tm(ctx, SPH_T_PREPASS);
        k_prepass<D><<<sph_ceil_div(n, 256), 256, 0, ctx->stream>>>(d, mats);
        ctx->launches += 1;
    }
    StageTimer tm(ctx, SPH_T_PAIRS);
    if (solid) {
        if (varh) k_pairs<D, true, true><<<gb, 128, 0, ctx->stream>>>(d, mats);
        else k_pairs<D, true, false><<<gb, 128, 0, ctx->stream>>>(d, mats);
    } else {
        if (varh) k_pairs<D, false, true><<<gb, 128, 0, ctx->stream>>>(d, mats);
        else k_pairs<D, false, false><<<gb, 128, 0, ctx->stream>>>(d, mats);
    }
    ctx->launches += 1;
}

const sph_material *sph_dev_mats(sph_ctx *ctx);

void sph_stage_rhs(sph_ctx *ctx) {
    if (ctx->d.D == 3) rhs_dim<3>(ctx, sph_dev_mats(ctx));
    else rhs_dim<2>(ctx, sph_dev_mats(ctx));
}
