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

#define PP_WARPS 8
template <int D>
__global__ void __launch_bounds__(PP_WARPS * 32) k_prepass(Dev d, const sph_material *mats) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int n = d.n;
    const int ii = min(i, n - 1);                              // (a tail lane repeats the last particle and stores nothing)
    const sph_material mt = mats[d.smat[ii]];
    const double rho = d.srho[ii], u = d.su[ii];
    double p, cs;
    eos_eval(mt, rho, u, p, cs);
    double S[6] = {0, 0, 0, 0, 0, 0};
    if (d.flags & SPH_F_SOLID) {
        for (int k = 0; k < 6; ++k) S[k] = d.sS[k][ii];
        if (D == 2) { S[2] = 0.0; S[4] = 0.0; S[5] = 0.0; }
        const double fY = yield_factor<D>(mt, d.flags, S);
        for (int k = 0; k < 6; ++k) S[k] *= fY;
    }
    double dd = 0.0;
    if ((d.flags & SPH_F_DAMAGE) && mt.brittle) { const double g = d.sdmg[ii]; dd = g * g * g; }
    const double phat = (p >= 0.0) ? p : (1.0 - dd) * p;
    const double ir2 = 1.0 / (rho * rho);
    double sg[6];
    for (int k = 0; k < 6; ++k) sg[k] = (1.0 - dd) * S[k];
    sg[0] -= phat; sg[3] -= phat;
    if (D == 3) sg[5] -= phat;
    if (i < n) { d.p[i] = p; d.cs[i] = cs; }
    // packed 128-byte record read by the pair kernel (one cache line per partner).  The 32 records of a warp go through
    // shared memory (144-byte stride: conflict-free 16-byte accesses) and leave as 8 fully coalesced 512-byte stores;
    // one lane storing its own record 16 bytes at a time touched 32 lines per store instruction.
    __shared__ __align__(16) double s_rec[PP_WARPS][32 * 18];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (i < n) {
        double2 *rec = reinterpret_cast<double2 *>(&s_rec[w][lane * 18]);
        rec[0] = make_double2(d.sx[0][i], d.sx[1][i]);
        rec[1] = make_double2((D == 3) ? d.sx[2][i] : 0.0, d.sv[0][i]);
        rec[2] = make_double2(d.sv[1][i], (D == 3) ? d.sv[2][i] : 0.0);
        rec[3] = make_double2(rho, d.sm[i] / rho);
        rec[4] = make_double2(cs, d.sh[i]);
        rec[5] = make_double2(sg[0] * ir2, sg[1] * ir2);
        rec[6] = make_double2(sg[2] * ir2, sg[3] * ir2);
        rec[7] = make_double2(sg[4] * ir2, sg[5] * ir2);
    }
    __syncwarp();
    const int i0 = i - lane;                                   // first particle of the warp
    double2 *out = reinterpret_cast<double2 *>(d.prec + (size_t)i0 * PR_REC);
#pragma unroll
    for (int t = 0; t < 8; ++t) {
        const int q = t * 32 + lane, r = q >> 3, sub = q & 7;  // record r of the warp, 16-byte part sub
        if (i0 + r < n) out[q] = *reinterpret_cast<const double2 *>(&s_rec[w][r * 18 + sub * 2]);
    }
}

template <int D> struct KNorm;
template <> struct KNorm<2> { static constexpr double s = 40.0 / (7.0 * 3.14159265358979323846); };
template <> struct KNorm<3> { static constexpr double s = 8.0 / 3.14159265358979323846; };

template <int D, bool VARH>
__global__ void __launch_bounds__(128) k_density(Dev d) {
    const int i = d.r_lo + blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const int g = i >> 5;
    if (g * 32 >= d.r_hi) return;
    const bool valid = i < d.r_hi;
    const int ii = valid ? i : d.n - 1;
    const double xi = d.sx[0][ii], yi = d.sx[1][ii], zi = (D == 3) ? d.sx[2][ii] : 0.0, Hi = d.sh[ii];
    const int cnt = valid ? d.nb_cnt[ii] : 0;
    int mx = cnt;
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    const int *nbw = d.nb + (size_t)g * d.cap * 32 + SPH_NB_POS(lane);
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

// ---- fast FP64 helpers for positive, normal arguments (no zero / infinity / denormal branches) ----
__device__ __forceinline__ double rsqrt_fast(double x) {      // hardware seed + one third-order step: < 1 ulp
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y * y, 1.0);
    return fma(fma(e, 0.375, 0.5), y * e, y);
}
__device__ __forceinline__ double sqrt_fast(double x) {       // x * rsqrt(x) + one Newton correction
    const double y = rsqrt_fast(x);
    const double s = x * y;
    return fma(fma(-s, s, x), 0.5 * y, s);
}
__device__ __forceinline__ double div_fast(double n, double dn) {   // n / dn, dn normal and non-zero
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(dn));
    y = fma(y, fma(-dn, y, 1.0), y);
    y = fma(y, fma(-dn, y, 1.0), y);
    const double q = n * y;
    return fma(fma(-dn, q, n), y, q);
}

// One Jacobi rotation that annihilates apq (r = the third index); eigenvalues only.
__device__ __forceinline__ void jacobi_rot(double &app, double &aqq, double &apq, double &arp, double &arq) {
    const double tau = aqq - app;
    const double w2 = fma(tau, tau, 4.0 * apq * apq);
    const bool on = (apq != 0.0) && (w2 > 0.0);
    const double w = sqrt_fast(on ? w2 : 1.0);
    const double den = tau + ((tau >= 0.0) ? w : -w);
    const double t = on ? div_fast(2.0 * apq, den) : 0.0;
    const double c = rsqrt_fast(fma(t, t, 1.0)), sn = t * c;
    app = fma(-t, apq, app);
    aqq = fma(t, apq, aqq);
    apq = on ? 0.0 : apq;
    const double rp = arp, rq = arq;
    arp = c * rp - sn * rq;
    arq = sn * rp + c * rq;
}

// Largest eigenvalue of a symmetric DxD matrix (eq. 48: maximum principal stress).
// 3-D: cyclic Jacobi on the six independent components, the sweeps taken by the whole warp together
// (the per-lane data-dependent loop of the first version cost more instructions than the pair
// loop: profiles/r1b).  2-D: closed form.
template <int D>
__device__ __forceinline__ double max_eig_sym(double a00, double a01, double a02, double a11, double a12, double a22) {
    if constexpr (D == 2) {
        const double hm = 0.5 * (a00 - a11), w2 = fma(hm, hm, a01 * a01);
        return 0.5 * (a00 + a11) + ((w2 > 0.0) ? sqrt_fast(w2) : 0.0);
    } else {
    for (int sweep = 0; sweep < 12; ++sweep) {
        const double off = a01 * a01 + a02 * a02 + a12 * a12;
        const double dg = a00 * a00 + a11 * a11 + a22 * a22;
        if (__all_sync(__activemask(), off <= 1e-36 * dg)) break;      // also off == 0
        jacobi_rot(a00, a11, a01, a02, a12);      // (p, q, r) = (0, 1, 2)
        jacobi_rot(a00, a22, a02, a01, a12);      // (0, 2, 1)
        jacobi_rot(a11, a22, a12, a01, a02);      // (1, 2, 0)
    }
    return fmax(a00, fmax(a11, a22));
    }
}

#define PR_WARPS 1
#define PR_MINBLOCKS 1            // resident blocks per SM the register allocation must allow (1 = no cap)
#define PR_STRIDE 18            // doubles between staged records (144 B): 16-byte reads by lane are conflict-free

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem_src));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::); }
__device__ __forceinline__ void cp_async_wait1() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }

// One lane per particle, 32 Morton-consecutive particles per warp.  Round k handles the k-th partner
// of every lane: the 32 partner records (128 B each, written by k_prepass) are copied to shared
// memory by the whole warp -- 8 lanes fetch one record as 8 x 16 B, so a warp-wide copy touches 4
// cache lines instead of 32 -- with cp.async one round ahead of the arithmetic; then every lane
// reads ITS partner's record from shared memory (144-byte stride: conflict-free).
// EXTRA: artificial stress (eqs. 35-38, reading U25) and/or the XSPH sum (eq. 40, reading U26).
template <int D, bool SOLID, bool VARH, bool EXTRA>
__global__ void __launch_bounds__(PR_WARPS * 32, PR_MINBLOCKS) k_pairs(Dev d, const sph_material *mats) {
    constexpr int NS = (D == 3) ? 6 : 3;                 // independent stress components
    constexpr int SI[6] = {0, 1, (D == 3) ? 2 : 3, 3, 4, 5};   // 2-D: xx xy yy -> 0 1 3
    __shared__ __align__(16) double s_buf[PR_WARPS][2][32 * PR_STRIDE];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = d.r_lo / 32 + blockIdx.x * PR_WARPS + w;   // groups of the rank's slice (all of them on one GPU)
    if (g * 32 >= d.r_hi) return;
    const int i = g * 32 + lane;
    const bool valid = i < d.r_hi;
    const int ii = valid ? i : d.n - 1;
    const unsigned FULL = 0xffffffffu;
    const double *__restrict__ prec = d.prec;

    double xa[3], va[3], sa[NS];
    double Hi, rhoi, csi;
    {
        const double2 *rec = reinterpret_cast<const double2 *>(prec + (size_t)ii * PR_REC);
        const double2 c0 = rec[0], c1 = rec[1], c2 = rec[2], c3 = rec[3], c4 = rec[4], c5 = rec[5], c6 = rec[6], c7 = rec[7];
        xa[0] = c0.x; xa[1] = c0.y; xa[2] = c1.x; va[0] = c1.y; va[1] = c2.x; va[2] = c2.y;
        rhoi = c3.x; csi = c4.x; Hi = c4.y;
        const double sr[6] = {c5.x, c5.y, c6.x, c6.y, c7.x, c7.y};
        for (int k = 0; k < NS; ++k) sa[k] = sr[SI[k]];
    }
    const double iHi = 1.0 / Hi;
    const double fac_i = 6.0 * KNorm<D>::s * ((D == 3) ? (iHi * iHi) * (iHi * iHi) : iHi * iHi * iHi);
    const int cnt = valid ? d.nb_cnt[ii] : 0;
    int mx = cnt;
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(FULL, mx, o));
    // the partner indices of the 8 rows my lane group stages (rows row0 + 4 t): 32 contiguous bytes per round (SPH_NB_POS)
    const int4 *nbg = reinterpret_cast<const int4 *>(d.nb + (size_t)g * d.cap * 32 + (lane >> 3) * 8);

    double drho = 0.0, du = 0.0, dv[3] = {0, 0, 0};
    double G[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    double N[6] = {0, 0, 0, 0, 0, 0};                     // symmetric moment matrix xx xy xz yy yz zz
    double xs[3] = {0, 0, 0};                             // XSPH sum
    const bool art = EXTRA && (d.flags & SPH_F_ART_STRESS), xsph = EXTRA && (d.flags & SPH_F_XSPH);
    // kernel shape w(q) = W h^D / s (eq. 25): 6q^3 - 6q^2 + 1 below q = 1/2, 2 (1 - q)^3 above
    auto wshape = [](double q) { const double t = fmax(1.0 - q, 0.0); return (q < 0.5) ? fma(6.0 * q * q, q - 1.0, 1.0) : 2.0 * t * t * t; };
    const double wnorm_i = KNorm<D>::s * ((D == 3) ? iHi * iHi * iHi : iHi * iHi);
    const double wm_i = EXTRA ? wshape(d.as_mpd * iHi) : 1.0;

    // copy the records of partners `b` (one per lane) into buffer `buf`
    const int sub = lane & 7, row0 = lane >> 3;
    auto stage = [&](int4 ia, int4 ib, int buf) {
        double *dstb = &s_buf[w][buf][0];
        const int br[8] = {ia.x, ia.y, ia.z, ia.w, ib.x, ib.y, ib.z, ib.w};
#pragma unroll
        for (int t = 0; t < 8; ++t) {
            const int r = row0 + 4 * t;
            cp_async16(dstb + r * PR_STRIDE + sub * 2, prec + (size_t)br[t] * PR_REC + sub * 2);
        }
    };
    // (rows k < mx are complete: a lane with fewer partners holds its own index there)
    const int4 own4 = make_int4(ii, ii, ii, ii);
    int4 ia = (mx > 0) ? __ldg(nbg) : own4, ib = (mx > 0) ? __ldg(nbg + 1) : own4;
    if (mx > 0) stage(ia, ib, 0);
    cp_async_commit();
    if (mx > 1) { ia = __ldg(nbg + 8); ib = __ldg(nbg + 9); }

    for (int k = 0; k < mx; ++k) {
        if (k + 1 < mx) stage(ia, ib, (k + 1) & 1);
        cp_async_commit();
        if (k + 2 < mx) { ia = __ldg(nbg + (size_t)(k + 2) * 8); ib = __ldg(nbg + (size_t)(k + 2) * 8 + 1); }
        cp_async_wait1();
        __syncwarp();
        const double2 *rec = reinterpret_cast<const double2 *>(&s_buf[w][k & 1][lane * PR_STRIDE]);
        const double2 c0 = rec[0], c1 = rec[1], c2 = rec[2], c3 = rec[3], c4 = rec[4], c5 = rec[5], c6 = rec[6], c7 = rec[7];
        if (k < cnt) {
            const double xb[3] = {c0.x, c0.y, c1.x}, vb[3] = {c1.y, c2.x, c2.y};
            const double rhob = c3.x, volb = c3.y, csb = c4.x, hb = c4.y;
            const double sb6[6] = {c5.x, c5.y, c6.x, c6.y, c7.x, c7.y};
            const double mb = rhob * volb;
            double dx[3], dvv[3];
            double r2 = 0.0, vr = 0.0;
            for (int a = 0; a < D; ++a) {
                dx[a] = xa[a] - xb[a];
                dvv[a] = va[a] - vb[a];
                r2 += dx[a] * dx[a];
                vr += dvv[a] * dx[a];
            }
            const double rinv = (r2 > 0.0) ? rsqrt_fast(r2) : 0.0;     // a coincident partner contributes nothing
            const double r = r2 * rinv;
            double iH = iHi, fac = fac_i;
            if (VARH) {
                iH = div_fast(1.0, 0.5 * (Hi + hb));
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
                const double Hb = 0.5 * (Hi + hb), cb = 0.5 * (csi + csb), rb = 0.5 * (rhoi + rhob);
                const double den = r2 + d.av_eps * Hb * Hb;
                const double inv = div_fast(1.0, den * rb);
                const double nu = Hb * vr * rb * inv;
                Pi = nu * (d.av_beta * nu - d.av_alpha * cb) * den * inv;
            }
            double T[NS];
            for (int k2 = 0; k2 < NS; ++k2) T[k2] = sa[k2] + sb6[SI[k2]];
            if (EXTRA) {
                const double wq = wshape(q);
                if (art) {                                    // eqs. 35-38: repulsive stress in tension
                    const double wm = VARH ? wshape(d.as_mpd * iH) : wm_i;
                    const double fr = wq / wm;                // eq. 38
                    const double fn = (d.as_n == 4.0) ? (fr * fr) * (fr * fr) : pow(fr, d.as_n);
                    for (int k2 = 0; k2 < NS; ++k2) {
                        const double s1 = sa[k2], s2 = sb6[SI[k2]];
                        const double z = ((s1 > 0.0) ? s1 : 0.0) + ((s2 > 0.0) ? s2 : 0.0);   // eq. 37 (U25)
                        T[k2] -= d.as_eps * z * fn;
                    }
                }
                if (xsph) {                                   // eq. 40 (U26)
                    const double wn = VARH ? KNorm<D>::s * ((D == 3) ? iH * iH * iH : iH * iH) : wnorm_i;
                    const double wgt = d.xsph * 2.0 * mb / (rhoi + rhob) * (wn * wq);
                    for (int a = 0; a < D; ++a) xs[a] -= wgt * dvv[a];
                }
            }
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
            for (int a = 0; a < D; ++a) { dv[a] += mb * fv[a]; e += fv[a] * dvv[a]; }   // eqs. 30/34 (35 with artificial stress)
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
        __syncwarp();                                         // buffer k & 1 is refilled in round k + 1
    }
    if (!valid) return;

    d.drho[i] = rhoi * drho;
    d.du[i] = -0.5 * du;
    for (int a = 0; a < 3; ++a) d.dv[a][i] = (a < D) ? dv[a] : 0.0;
    if (xsph) for (int a = 0; a < 3; ++a) d.dxs[a][i] = (a < D) ? xs[a] : 0.0;

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
        if (d.flags & SPH_F_EXPORT_GRADV) {                   // A8 made visible: eqs. 42-44 compared directly by the parity tests
            for (int a = 0; a < 3; ++a) for (int c = 0; c < 3; ++c) { d.gradv[3 * a + c][i] = gv[a][c]; d.Cten[3 * a + c][i] = C[a][c]; }
        }
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
                const double od = 1.0 - dd;
                const double smax = max_eig_sym<D>(od * St[0] - phat, od * St[1], od * St[2], od * St[3] - phat,
                                                   od * St[4], od * St[5] - phat);
                const double K = (mt.eos == SPH_EOS_TILLOTSON) ? mt.tA : mt.K0;
                const double E = 9.0 * K * mt.mu / (3.0 * K + mt.mu);
                strain = smax / ((1.0 - dd) * E);
                // thresholds are ascending per particle (sph.h, eq. 45): the number of activated flaws is the
                // position of the first threshold above the strain (bisection: ~4 reads instead of ~15)
                i64 lo = f0, hi = f1;
                while (lo < hi) {
                    const i64 mid = (lo + hi) >> 1;
                    if (d.flaw_eps[mid] <= strain) lo = mid + 1; else hi = mid;
                }
                nact = max(nact, (int)(lo - f0));
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
    const int pb = sph_ceil_div(sph_ceil_div(d.r_hi - d.r_lo, 32), PR_WARPS);   // pair sums: the rank's slice
    if (d.flags & SPH_F_DENSITY_SUM) {
        StageTimer tm(ctx, SPH_T_DENSITY);
        Dev dd = d;                              // every particle's density on every rank (its partners read it)
        dd.r_lo = 0; dd.r_hi = n;
        if (varh) k_density<D, true><<<gb, 128, 0, ctx->stream>>>(dd);
        else k_density<D, false><<<gb, 128, 0, ctx->stream>>>(dd);
        ctx->launches += 1;
    }
    {
        StageTimer tm(ctx, SPH_T_PREPASS);
        k_prepass<D><<<sph_ceil_div(n, 256), 256, 0, ctx->stream>>>(d, mats);
        ctx->launches += 1;
    }
    StageTimer tm(ctx, SPH_T_PAIRS);
    const bool extra = (d.flags & (SPH_F_ART_STRESS | SPH_F_XSPH)) != 0;
#define SPH_PAIRS(S, V, E) k_pairs<D, S, V, E><<<pb, PR_WARPS * 32, 0, ctx->stream>>>(d, mats)
    if (pb == 0) return;                         // a rank without particles (more ranks than slices)
    if (solid) {
        if (varh) { if (extra) SPH_PAIRS(true, true, true); else SPH_PAIRS(true, true, false); }
        else { if (extra) SPH_PAIRS(true, false, true); else SPH_PAIRS(true, false, false); }
    } else {
        if (varh) { if (extra) SPH_PAIRS(false, true, true); else SPH_PAIRS(false, true, false); }
        else { if (extra) SPH_PAIRS(false, false, true); else SPH_PAIRS(false, false, false); }
    }
#undef SPH_PAIRS
    ctx->launches += 1;
}

const sph_material *sph_dev_mats(sph_ctx *ctx);

void sph_stage_rhs(sph_ctx *ctx) {
    if (ctx->d.D == 3) rhs_dim<3>(ctx, sph_dev_mats(ctx));
    else rhs_dim<2>(ctx, sph_dev_mats(ctx));
}
