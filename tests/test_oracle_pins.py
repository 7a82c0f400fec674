"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test names the passage it pins.  None of them re-types the oracle's own formula as
the expected value: expectations are closed forms, invariants, library routines
(scipy quadrature, numpy eigensolver, cKDTree), brute force, or golden values with a
citation in tests/golden/.
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate
from scipy.spatial import cKDTree

import sph_inputs as si
from oracle import oracle as orc

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "lattice_sums.txt")) as fh:
    for line in fh:
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            GOLD[k] = float(v)


# ------------------------------------------------------------------ kernel
@pytest.mark.parametrize("D", [1, 2, 3])
def test_kernel_normalisation_integral(D):
    h = 0.73
    surf = {1: lambda r: 2.0, 2: lambda r: 2 * math.pi * r, 3: lambda r: 4 * math.pi * r * r}[D]
    val = sum(integrate.quad(lambda r: orc.W(D, r, h) * surf(r), a, b, epsabs=1e-14, epsrel=1e-13)[0]
              for a, b in ((0, h / 2), (h / 2, h)))
    assert abs(val - 1.0) < 1e-11
    assert abs(orc.W(D, 0.0, 1.0) - GOLD[f"s_{D}d"]) < 1e-15       # eq. 26 as printed


@pytest.mark.parametrize("D", [1, 2, 3])
def test_kernel_derivative_and_branches(D):
    h = 1.7
    for r in np.linspace(0.01, 1.05, 41) * h:
        e = 1e-6 * h
        fd = (orc.W(D, r + e, h) - orc.W(D, r - e, h)) / (2 * e)
        assert abs(fd - orc.dW(D, r, h)) < 1e-7 * abs(orc.dW(D, 0.4 * h, h))
    # both branches meet at r/h = 1/2 with value 0.25 s / h^D, compact support at r = h
    lo, hi = orc.W(D, 0.5 * h * (1 - 1e-15), h), orc.W(D, 0.5 * h, h)
    assert abs(lo - hi) < 1e-14 * hi and abs(hi - 0.25 * GOLD[f"s_{D}d"] / h ** D) < 1e-15 * hi * 10
    assert orc.W(D, h * 1.0000001, h) == 0.0 and orc.dW(D, h * 1.0000001, h) == 0.0


def test_kernel_equals_textbook_m4_spline():
    # Monaghan & Lattanzio M4 in the "2h" convention with h_cfg = h_paper/2
    hp = 0.9
    hc = hp / 2
    for r in np.linspace(0, 1.1, 23) * hp:
        q = r / hc
        m4 = (1 - 1.5 * q * q + 0.75 * q ** 3) if q < 1 else (0.25 * (2 - q) ** 3 if q < 2 else 0.0)
        assert abs(orc.W(3, r, hp) - m4 / (math.pi * hc ** 3)) < 1e-13


# ------------------------------------------------------------------ lattice sums (golden)
def _lattice(D, k=7, dx=0.37):
    ax = np.arange(-k, k + 1) * dx
    g = np.meshgrid(*([ax] * D), indexing="ij")
    x = np.zeros((3, g[0].size))
    for a in range(D):
        x[a] = g[a].ravel()
    n = x.shape[1]
    off, eps = np.zeros(n + 1, np.int64), np.zeros(0)
    w = si.Workload(name="lattice", dim=D, flags=si.F_SOLID, materials=[si.RUBBER], x=x,
                    v=np.zeros((3, n)), m=np.full(n, 1.3 * dx ** D), rho=np.full(n, 1.3),
                    u=np.zeros(n), S=np.zeros((6, n)), dmg=np.zeros(n), h=np.full(n, 2.6 * dx),
                    mat=np.zeros(n, np.int32), n_act=np.zeros(n, np.int32), flaw_off=off, flaw_eps=eps)
    centre = int(np.argmin((x ** 2).sum(0)))
    return w, centre, dx


@pytest.mark.parametrize("D", [2, 3])
def test_lattice_neighbour_count_density_and_moment(D):
    w, c, dx = _lattice(D)
    off, idx = orc.neighbours(w, [c])
    assert off[1] == GOLD[f"neighbours_{D}d"]
    rho = orc.density(w, off, idx, [c])[0]
    assert abs(rho * dx ** D / w.m[c] - GOLD[f"density_{D}d"]) < 1e-13
    assert abs(rho / 1.3 - 1.0) < 3e-3
    r = orc.rhs(w, off, idx, [c])
    Cm = r["C"][:, 0].reshape(3, 3)[:D, :D]
    N = np.linalg.inv(Cm)
    assert abs(N[0, 0] - GOLD[f"moment00_{D}d"]) < 1e-12       # positive: fixes the sign of eq. 43/44 (U6)
    assert np.allclose(N, N[0, 0] * np.eye(D), atol=1e-13)


# ------------------------------------------------------------------ invariants of the pair sums
def _blob(n=700, D=3, seed=3, **kw):
    return si.random_blob(n, D, seed, **kw)


@pytest.mark.parametrize("D,varh", [(3, False), (3, True), (2, False)])
def test_momentum_and_energy_conservation(D, varh):
    w = _blob(600, D, 11, variable_h=varh, gravity=False)
    if not varh:
        w.h[:] = w.h[0]                # fixed common h: symmetric partner sets
    e = orc.evaluate(w, "brute", h_iters=0)
    P = (w.m[None, :] * e["dv"]).sum(1)
    scale = (w.m[None, :] * np.abs(e["dv"])).sum()
    assert np.abs(P).max() <= 1e-13 * scale                 # north_star: 1e-13 relative
    # sum_a m_a (v_a . dv_a/dt + du_a/dt) = 0: holds only with opposite gradients in eqs. 30/31 (U2, U3)
    rate = (w.m * ((w.v * e["dv"]).sum(0) + e["du"])).sum()
    assert abs(rate) <= 1e-12 * (w.m * (np.abs(w.v * e["dv"]).sum(0) + np.abs(e["du"]))).sum()
    # partner sets are symmetric
    off, idx = e["nb_off"], e["nb_idx"]
    pairs = {(a, int(b)) for a in range(w.n) for b in idx[off[a]:off[a + 1]]}
    assert all((b, a) in pairs for a, b in pairs)


def test_gas_limit_is_textbook_sph():
    # S = 0, no strength: eqs. 29-34 must reduce to the textbook gas form
    #   dv_a = -sum m_b (p_a/rho_a^2 + p_b/rho_b^2 + Pi_ab) grad_a W,  du_a = 1/2 sum m_b (...) v_ab.grad_a W
    w = _blob(400, 3, 5, solid=False, gravity=False)
    w.h[:] = w.h[0]
    e = orc.evaluate(w, "brute")
    g = w.materials[0]["gamma"]
    p = (g - 1) * w.rho * w.u
    cs = np.sqrt(g * (g - 1) * w.u)
    X, V = w.x.T, w.v.T
    kd = cKDTree(X)
    for a in range(0, w.n, 37):
        acc, du, drho = np.zeros(3), 0.0, 0.0
        for b in kd.query_ball_point(X[a], w.h[a]):
            if b == a:
                continue
            d = X[a] - X[b]
            r = np.linalg.norm(d)
            gW = orc.dW(3, r, w.h[a]) * d / r
            vab = V[a] - V[b]
            vr = vab @ d
            Pi = 0.0
            if vr < 0:
                nu = w.h[a] * vr / (r * r + w.av_eps * w.h[a] ** 2)
                Pi = (-w.av_alpha * 0.5 * (cs[a] + cs[b]) * nu + w.av_beta * nu * nu) / (0.5 * (w.rho[a] + w.rho[b]))
            P = p[a] / w.rho[a] ** 2 + p[b] / w.rho[b] ** 2 + Pi
            acc -= w.m[b] * P * gW
            du += 0.5 * w.m[b] * P * (vab @ gW)
            drho += w.rho[a] * w.m[b] / w.rho[b] * (vab @ gW)
        assert np.allclose(e["dv"][:, a], acc, rtol=1e-11, atol=1e-13 * np.abs(e["A_dv"][:, a]).max())
        assert abs(e["du"][a] - du) <= 1e-11 * abs(du) + 1e-13 * e["A_du"][a]
        assert abs(e["drho"][a] - drho) <= 1e-11 * abs(drho) + 1e-13 * e["A_drho"][a]


def test_uniform_pressure_blob_pushes_surface_outward_and_interior_balances():
    w, c, dx = _lattice(3, k=6)
    w.materials = [si.material(si.EOS_MURNAGHAN, rho0=1.0, K0=1.0, nM=4.0, mu=0.2)]
    w.rho[:] = 1.3                                   # p > 0 everywhere
    w.m[:] = 1.3 * dx ** 3
    e = orc.evaluate(w, "brute")
    assert np.abs(e["dv"][:, c]).max() < 1e-12 * e["A_dv"][:, c].max()      # interior: exact balance
    corner = int(np.argmax(w.x.sum(0)))
    assert (e["dv"][:, corner] > 0).all()            # positive pressure accelerates the corner outward (U2)


def test_artificial_viscosity_repels_approaching_pair_only():
    n = 2
    x = np.zeros((3, n)); x[0, 1] = 0.5
    mk = lambda v1: si.Workload(name="pair", dim=3, flags=0, materials=[si.GAS], x=x,
                                v=np.array([[0.0, v1], [0, 0], [0, 0]]), m=np.ones(n), rho=np.ones(n),
                                u=np.zeros(n), S=np.zeros((6, n)), dmg=np.zeros(n), h=np.ones(n),
                                mat=np.zeros(n, np.int32), n_act=np.zeros(n, np.int32),
                                flaw_off=np.zeros(n + 1, np.int64), flaw_eps=np.zeros(0),
                                av_alpha=1.0, av_beta=2.0)
    app = orc.evaluate(mk(-1.0), "brute")            # u = 0 -> p = 0, c_s = 0: only the beta term acts
    assert app["dv"][0, 0] < 0 < app["dv"][0, 1]     # pushed apart
    assert app["du"][0] > 0                          # dissipation heats
    rec = orc.evaluate(mk(+1.0), "brute")
    assert np.all(rec["dv"] == 0) and np.all(rec["du"] == 0)     # receding: Pi* = 0


def test_continuity_translation_and_linear_field():
    w = _blob(500, 3, 9, gravity=False)
    w.h[:] = w.h[0]
    w.v[:] = np.array([0.3, -0.2, 0.7])[:, None]     # rigid translation
    e = orc.evaluate(w, "brute")
    assert np.all(e["drho"] == 0.0) and np.all(e["gradv"] == 0.0)
    A = np.array([[0.2, -0.5, 0.1], [0.3, 0.05, -0.4], [-0.6, 0.2, -0.1]])
    w.v = A @ w.x + np.array([0.1, 0.2, 0.3])[:, None]
    e = orc.evaluate(w, "brute")
    cnt = e["nb_off"][1:] - e["nb_off"][:-1]
    for a in np.flatnonzero(cnt >= 12)[::25]:
        Cm = e["C"][:, a].reshape(3, 3)
        if np.allclose(Cm, np.eye(3)):
            continue
        N = np.linalg.inv(Cm)
        # eq. 29 with v = A x:  drho/dt = -rho A^{ab} N^{ba}  (N = eq. 44's moment matrix)
        assert abs(e["drho"][a] + w.rho[a] * np.trace(A @ N)) <= 1e-11 * e["A_drho"][a]
        # eq. 42: first-order consistency, grad v = A exactly
        assert np.allclose(e["gradv"][:, a].reshape(3, 3), A, atol=1e-11)


def test_correction_tensor_identity_eq44():
    w = _blob(400, 3, 21, gravity=False, variable_h=True)
    e = orc.evaluate(w, "brute", h_iters=0)
    off, idx = e["nb_off"], e["nb_idx"]
    for a in range(0, w.n, 29):
        nb = idx[off[a]:off[a + 1]]
        Cm = e["C"][:, a].reshape(3, 3)
        if nb.size < 8 or np.allclose(Cm, np.eye(3)):
            continue
        acc = np.zeros((3, 3))
        for b in nb:
            d = w.x[:, a] - w.x[:, b]
            r = np.linalg.norm(d)
            gW = orc.dW(3, r, 0.5 * (w.h[a] + w.h[b])) * d / r
            acc += w.m[b] / w.rho[b] * np.outer(-d, gW @ Cm)
        assert np.allclose(acc, np.eye(3), atol=1e-11)


def test_stress_rate_trace_shear_and_rotation():
    w = _blob(500, 3, 13, gravity=False, damage=False)
    w.h[:] = w.h[0]
    mu = np.array([m["mu"] for m in w.materials])[w.mat]
    e = orc.evaluate(w, "brute")
    tr = e["dS"][0] + e["dS"][3] + e["dS"][5]
    assert np.abs(tr).max() <= 1e-12 * np.abs(e["A_dS"]).max()           # deviatoric: trace 0 (U8)
    full = (e["nb_off"][1:] - e["nb_off"][:-1]) >= 12
    # pure shear v = (g y, 0, 0), S = 0:  dS^xy/dt = mu g, everything else 0   (eqs. 7-8)
    g = 0.37
    w2 = w.copy(); w2.S[:] = 0.0; w2.v[:] = 0.0; w2.v[0] = g * w2.x[1]
    e2 = orc.evaluate(w2, "brute")
    ok = full & ~np.all(np.isclose(e2["C"].T, np.eye(3).ravel()), axis=1)
    assert np.allclose(e2["dS"][1][ok], (mu * g)[ok], rtol=1e-10)
    assert np.abs(e2["dS"][[0, 2, 3, 4, 5]][:, ok]).max() < 1e-10 * mu.max() * g
    # rigid rotation v = Omega x X: strain rate 0, dS/dt = S R - R S with R_ab = dv_a/dx_b antisymmetric (eq. 9)
    Om = np.array([0.3, -0.7, 0.5])
    R = np.array([[0, -Om[2], Om[1]], [Om[2], 0, -Om[0]], [-Om[1], Om[0], 0]])
    w3 = w.copy(); w3.v = R @ w3.x
    for m_ in w3.materials:
        m_["Y0"] = 0.0                                                   # no limiter: S-tilde = S
    e3 = orc.evaluate(w3, "brute")
    for a in np.flatnonzero(ok)[::40]:
        S = np.array([[w3.S[0, a], w3.S[1, a], w3.S[2, a]], [w3.S[1, a], w3.S[3, a], w3.S[4, a]],
                      [w3.S[2, a], w3.S[4, a], w3.S[5, a]]])
        exp = S @ R - R @ S
        got = e3["dS"][:, a]
        assert np.allclose(got, [exp[0, 0], exp[0, 1], exp[0, 2], exp[1, 1], exp[1, 2], exp[2, 2]],
                           atol=1e-10 * np.abs(S).max())


# ------------------------------------------------------------------ equations of state
def test_murnaghan_closed_forms():
    m = si.material(si.EOS_MURNAGHAN, rho0=2.5, K0=7.0, nM=4.0)
    assert orc.eos(m, 2.5, 0.0)[0] == 0.0
    e = 1e-6
    slope = (orc.eos(m, 2.5 * (1 + e), 0)[0] - orc.eos(m, 2.5 * (1 - e), 0)[0]) / (2 * e * 2.5)
    assert abs(slope - 7.0 / 2.5) < 1e-6                                 # dp/drho = K0/rho0 = c_s^2 (eq. 12)
    assert abs(orc.eos(m, 2.5, 0)[1] - math.sqrt(7.0 / 2.5)) < 1e-15
    assert abs(orc.eos(m, 5.0, 0)[0] - 7.0 / 4 * 15.0) < 1e-13           # (2^4 - 1) K0/n


def test_tillotson_continuity_and_limits():
    m = si.BASALT
    r0 = m["rho0"]
    assert orc.eos(m, r0, 0.0)[0] == 0.0
    e = 1e-7
    K = (orc.eos(m, r0 * (1 + e), 0)[0] - orc.eos(m, r0 * (1 - e), 0)[0]) / (2 * e)
    assert abs(K / m["tA"] - 1.0) < 1e-6                                 # rho0 dp/drho = A_T at (rho0, 0)
    for rho in (0.7 * r0, 0.95 * r0):                                    # expanded states: interpolation is continuous
        for E in (m["tEiv"], m["tEcv"]):
            pl, pr = orc.eos(m, rho, E * (1 - 1e-12))[0], orc.eos(m, rho, E * (1 + 1e-12))[0]
            assert abs(pl - pr) <= 1e-9 * max(abs(pl), abs(pr), 1.0)
    # compressed states use eq. 14 whatever u is
    u = 2 * m["tEcv"]
    rho = 1.2 * r0
    eta, chi = 1.2, 0.2
    p14 = (m["ta"] + m["tb"] / (1 + u / (m["tE0"] * eta ** 2))) * rho * u + m["tA"] * chi + m["tB"] * chi ** 2
    assert abs(orc.eos(m, rho, u)[0] / p14 - 1) < 1e-14
    # far expansion at high energy tends to the ideal-gas-like term a rho u (eq. 15)
    rho = 1e-3 * r0
    assert abs(orc.eos(m, rho, u)[0] / (m["ta"] * rho * u) - 1) < 1e-3


def test_von_mises_limiter_idempotent_and_bounded():
    w = _blob(300, 3, 4, gravity=False, damage=False)
    p, cs, sig, St = orc.prepass(w)
    Y0 = np.array([m["Y0"] for m in w.materials])[w.mat]
    J2 = 0.5 * (St[:, 0] ** 2 + St[:, 3] ** 2 + St[:, 5] ** 2 + 2 * (St[:, 1] ** 2 + St[:, 2] ** 2 + St[:, 4] ** 2))
    lim = Y0 > 0
    # eq. 17 as printed (no square root): after limiting, Y0^2/(3 J2') >= 1, i.e. limiting again changes nothing
    assert np.all(3 * J2[lim] <= Y0[lim] ** 2 * (Y0[lim] ** 2 / np.minimum(Y0[lim] ** 2, 3 * J2[lim] + 1e-300) + 1e-12) ** 2 + 1e-12)
    w2 = w.copy(); w2.S = St.T.copy()
    St2 = orc.prepass(w2)[3]
    assert np.allclose(St2, St, rtol=1e-14, atol=0)
    J2in = 0.5 * (w.S[0] ** 2 + w.S[3] ** 2 + w.S[5] ** 2 + 2 * (w.S[1] ** 2 + w.S[2] ** 2 + w.S[4] ** 2))
    untouched = lim & (3 * J2in <= Y0 ** 2)
    assert untouched.any() and np.array_equal(St[untouched], w.S.T[untouched])


# ------------------------------------------------------------------ damage
def test_max_principal_stress_vs_library_eigensolver():
    rng = np.random.default_rng(5)
    for D in (2, 3):
        for _ in range(200):
            A = rng.normal(size=(3, 3)); A = A + A.T
            ref = np.linalg.eigvalsh(A[:D, :D]).max()
            assert abs(orc.max_eig(D, A) - ref) < 1e-13 * np.abs(A).max()
    assert orc.max_eig(3, np.diag([1.0, 5.0, -2.0])) == 5.0


def test_damage_rate_single_particle_by_hand():
    # one brittle particle under uniform tension sigma = s * I: strain = s/((1-d) E) (eq. 48)
    mat = si.material(si.EOS_MURNAGHAN, rho0=2.0, K0=3.0, nM=4.0, mu=1.5, Y0=0.0, brittle=1)
    n = 1
    rho = 2.0 * 0.9                                  # expanded -> p < 0 (tension)
    thr = np.array([0.001, 0.002, 0.05, 10.0])
    w = si.Workload(name="one", dim=3, flags=si.F_SOLID | si.F_DAMAGE, materials=[mat],
                    x=np.zeros((3, n)), v=np.zeros((3, n)), m=np.ones(n), rho=np.full(n, rho),
                    u=np.zeros(n), S=np.zeros((6, n)), dmg=np.full(n, 0.5), h=np.full(n, 0.25),
                    mat=np.zeros(n, np.int32), n_act=np.zeros(n, np.int32),
                    flaw_off=np.array([0, 4], np.int64), flaw_eps=thr)
    e = orc.evaluate(w, "brute")
    d = 0.125
    p = 3.0 / 4.0 * (0.9 ** 4 - 1)                   # eq. 13
    smax = -(1 - d) * p                              # eqs. 20-21: sigma = -(1-d) p delta
    E = 9 * 3.0 * 1.5 / (3 * 3.0 + 1.5)              # eq. 49
    strain = smax / ((1 - d) * E)
    assert abs(e["strain"][0] / strain - 1) < 1e-14
    nact = int((thr <= strain).sum())
    assert nact == 3 and e["n_act"][0] == nact
    cg = 0.4 * math.sqrt((3.0 + 4.0 / 3.0 * (1 - d) * 1.5) / rho)       # 40 % of the longitudinal wave speed (U16)
    assert abs(e["ddmg"][0] / (nact * cg / 0.25) - 1) < 1e-14           # eq. 46 with R_s = h
    w.dmg[:] = (3 / 4) ** (1 / 3) * 1.0000001                           # d just above n_act/n_tot: limiter (eq. 47)
    assert orc.evaluate(w, "brute")["ddmg"][0] == 0.0
    w.dmg[:] = 0.5; w.n_act[:] = 4                                      # latched count wins (U19)
    assert orc.evaluate(w, "brute")["n_act"][0] == 4


# ------------------------------------------------------------------ order and tree
def _naive_interleave(D, g, L):
    key = 0
    for b in range(L):
        for a in range(D):
            key |= ((g[a] >> b) & 1) << (D * b + a)
    return key


def test_morton_interleave_and_order():
    rng = np.random.default_rng(2)
    for D in (2, 3):
        for _ in range(100):
            g = [int(v) for v in rng.integers(0, 2 ** 21, 3)]
            assert orc.interleave(D, *g) == _naive_interleave(D, g, 21)
    w = _blob(3000, 3, 8, duplicates=7)
    t = orc.Tree(w)
    key, perm = t.order()
    assert np.array_equal(np.sort(perm), np.arange(w.n))
    assert np.all(key[1:] >= key[:-1])
    eq = key[1:] == key[:-1]
    assert eq.sum() >= 7 and np.all(perm[1:][eq] > perm[:-1][eq])          # ties by original index (U13)
    # keys re-derived with numpy from the printed recipe (eq. 67, min-corner anchoring U12)
    lo = w.x.min(1); s0 = (w.x.max(1) - lo).max()
    assert s0 == t.s0
    g = np.minimum(((w.x - lo[:, None]) * (2.0 ** 21 / s0)).astype(np.uint64), 2 ** 21 - 1)
    k2 = np.array([_naive_interleave(3, [int(g[0, i]), int(g[1, i]), int(g[2, i])], 21) for i in perm], dtype=np.uint64)
    assert np.array_equal(k2, key)


@pytest.mark.parametrize("D", [2, 3])
def test_tree_matches_adjacent_prefix_definition(D):
    w = _blob(2500, D, 17, duplicates=5)
    t = orc.Tree(w)
    key, perm = t.order()
    nd = t.nodes()
    L = 21
    # definition: cells in which adjacent sorted particles first separate
    want = set()
    for i in range(w.n - 1):
        x = int(key[i]) ^ int(key[i + 1])
        if x == 0:
            continue
        lvl = (D * L - x.bit_length()) // D
        want.add((lvl, int(key[i]) >> (D * (L - lvl))))
    got = set(zip(nd["level"].tolist(), [int(p) for p in nd["prefix"]]))
    assert got == want
    # ranges: every node covers exactly the keys carrying its prefix
    for i in range(0, len(nd["level"]), 37):
        lvl, pf = int(nd["level"][i]), int(nd["prefix"][i])
        member = np.array([(int(k) >> (D * (L - lvl))) == pf for k in key]) if lvl else np.ones(w.n, bool)
        idx = np.flatnonzero(member)
        assert idx[0] == nd["lo"][i] and idx[-1] + 1 == nd["hi"][i] and idx.size == nd["hi"][i] - nd["lo"][i]
        ms = w.m[perm[idx]]
        assert abs(nd["mass"][i] - ms.sum()) <= 1e-14 * ms.sum()
        cm = (w.x[:, perm[idx]] * ms).sum(1) / ms.sum()
        assert np.allclose(nd["com"][i][:D], cm[:D], rtol=0, atol=1e-14 * np.abs(w.x).max() * 10)
        assert np.array_equal(nd["bmin"][i][:D], w.x[:D, perm[idx]].min(1))
        assert np.array_equal(nd["bmax"][i][:D], w.x[:D, perm[idx]].max(1))
        assert nd["hmax"][i] == w.h[perm[idx]].max()
    root = np.flatnonzero(nd["level"] == 0)
    assert root.size == 1 and nd["lo"][root[0]] == 0 and nd["hi"][root[0]] == w.n


# ------------------------------------------------------------------ neighbours
@pytest.mark.parametrize("D,varh", [(3, False), (3, True), (2, True)])
def test_neighbour_sets_brute_tree_and_kdtree(D, varh):
    w = _blob(1500, D, 23, variable_h=varh, duplicates=4)
    ob, ib = orc.neighbours(w, mode="brute")
    ot, it = orc.neighbours(w, mode="tree")
    assert np.array_equal(ob, ot) and np.array_equal(ib, it)
    # independent library: pairs within the largest possible reach, then the printed criterion
    kd = cKDTree(w.x[:D].T)
    for a in range(0, w.n, 17):
        cand = kd.query_ball_point(w.x[:D, a], w.h.max() * 1.01)
        d2 = ((w.x[:, cand] - w.x[:, [a]]) ** 2).sum(0)
        H = 0.5 * (w.h[a] + w.h[cand]) if varh else np.full(len(cand), w.h[a])
        exp = sorted(int(b) for b, r2, hh in zip(cand, d2, H) if b != a and r2 < hh * hh * (1 - 1e-12))
        got = ib[ob[a]:ob[a + 1]].tolist()
        assert set(exp) <= set(got) and len(got) - len(exp) <= 1
    n_a = orc.count_own_h(w)
    assert np.array_equal(n_a, orc.count_own_h(w, mode="tree"))
    h2 = orc.h_update(D, w.h, n_a, 50)
    k = int(np.argmax(n_a))
    assert abs(h2[k] / w.h[k] - 0.5 * (1 + (50 / n_a[k]) ** (1 / D))) < 1e-15      # eq. 73


# ------------------------------------------------------------------ gravity
def test_gravity_theta_zero_is_direct_sum_and_theta_half_error():
    w = si.make("C2", scale=0.05)                   # 3277 particles, rho ~ 1/r
    t = orc.Tree(w)
    a0, _, n0 = orc.gravity_tree(w, t, theta=0.0)
    ad, _ = orc.gravity_direct(w)
    mag = np.linalg.norm(ad, axis=0)
    assert np.abs(a0 - ad).max() <= 1e-12 * mag.max()
    assert np.all(n0 == w.n - 1)
    a5, _, n5 = orc.gravity_tree(w, t, theta=0.5)
    a3, _, n3 = orc.gravity_tree(w, t, theta=0.3)
    rel5 = np.median(np.linalg.norm(a5 - ad, axis=0) / mag)
    rel3 = np.median(np.linalg.norm(a3 - ad, axis=0) / mag)
    # north_star asks for a median relative error <= 1e-3 at theta = 0.5.  The paper's method
    # (monopoles only, s/r < theta on the geometric cell edge) does not reach
    # that at 0.5: measured 3.3e-3 / 2.6e-3 / 2.3e-3 at N = 3277 / 16384 / 65536 (DESIGN.md,
    # reading U32).  It does at theta = 0.3, and the error grows like theta^2 or faster
    # ("The error scales with theta^2").
    assert rel3 <= 1e-3
    assert rel5 <= 5e-3
    assert 2.0 <= rel5 / rel3 <= 8.0
    assert n5.mean() < n3.mean() < 0.5 * w.n
    # M(<r) = M r^2/R^2  =>  |a| = G M / R^2 = 1 inside (sampling noise ~ N^-1/2, softening near r=0)
    r = np.linalg.norm(w.x, axis=0)
    sel = (r > 0.3) & (r < 0.9)
    ar = -(ad * w.x).sum(0) / r
    assert abs(np.mean(ar[sel]) - 1.0) < 0.05


def test_gravity_two_body_and_shell_theorem():
    x = np.zeros((3, 2)); x[0, 1] = 2.0
    w = si.Workload(name="2", dim=3, flags=si.F_GRAVITY, materials=[si.GAS], x=x, v=np.zeros((3, 2)),
                    m=np.array([3.0, 5.0]), rho=np.ones(2), u=np.ones(2), S=np.zeros((6, 2)),
                    dmg=np.zeros(2), h=np.ones(2), mat=np.zeros(2, np.int32), n_act=np.zeros(2, np.int32),
                    flaw_off=np.zeros(3, np.int64), flaw_eps=np.zeros(0), G=2.0, eps_soft=0.0)
    ag, _, _ = orc.gravity_tree(w)
    assert abs(ag[0, 0] - 2.0 * 5.0 / 4.0) < 1e-15 and abs(ag[0, 1] + 2.0 * 3.0 / 4.0) < 1e-15   # attractive (U21)
    w.eps_soft = 1.5
    ag, _, _ = orc.gravity_tree(w)
    assert abs(ag[0, 0] - 2.0 * 5.0 * 2.0 / (4.0 + 2.25) ** 1.5) < 1e-15                          # Plummer
    # shell theorem: test particles inside / outside a uniform thin shell
    rng = np.random.default_rng(0)
    ns = 20000
    u = rng.normal(size=(3, ns)); u /= np.linalg.norm(u, axis=0)
    xs = np.concatenate([u, np.array([[0.3, 0.0], [0.1, 0.0], [0.0, 2.5]]).T.reshape(3, 2)], axis=1)
    xs[:, -2] = [0.3, 0.1, 0.0]; xs[:, -1] = [0.0, 0.0, 2.5]
    n = ns + 2
    m = np.full(n, 1.0 / ns); m[-2:] = 1e-30
    ws = si.Workload(name="shell", dim=3, flags=si.F_GRAVITY, materials=[si.GAS], x=xs, v=np.zeros((3, n)),
                     m=m, rho=np.ones(n), u=np.ones(n), S=np.zeros((6, n)), dmg=np.zeros(n), h=np.ones(n),
                     mat=np.zeros(n, np.int32), n_act=np.zeros(n, np.int32),
                     flaw_off=np.zeros(n + 1, np.int64), flaw_eps=np.zeros(0), G=1.0, eps_soft=0.0, theta=0.3)
    ag, _, _ = orc.gravity_tree(ws, targets=[n - 2, n - 1])
    assert np.linalg.norm(ag[:, 0]) < 0.03           # inside: no force (sampling noise)
    assert abs(ag[2, 1] + 1.0 / 2.5 ** 2) < 0.01     # outside: point mass at the centre


def test_gravity_tree_order_independence_and_duplicates():
    w = _blob(1200, 3, 31, duplicates=6)
    ag, _, _ = orc.gravity_tree(w)
    p = np.random.default_rng(1).permutation(w.n)
    w2 = w.subset(p)
    ag2, _, _ = orc.gravity_tree(w2)
    # same particles in another input order: identical canonical tree; only tie order of duplicates may differ
    assert np.allclose(ag2, ag[:, p], rtol=1e-12, atol=1e-12 * np.abs(ag).max())


# ------------------------------------------------------------------ time step
def test_energy_drift_bounded_over_20_rk2_steps_c1_twin():
    # north_star invariant: total energy drift bounded over 20 steps (C1: no gravity).
    # Bound proposed in SURVEY 8(c): |dE| <= 1e-6 (E_kin + E_int)(0); the elastic energy stored in S is
    # not part of sum m (v^2/2 + u) -- du/dt (eq. 31) already contains the S : eps-dot work.
    w = si.make("C1", scale=0.12, twin=True)
    E = lambda q: float((q.m * (0.5 * (q.v ** 2).sum(0) + q.u)).sum())
    E0 = E(w)
    Eabs = float((w.m * (0.5 * (w.v ** 2).sum(0) + np.abs(w.u))).sum())
    q = w
    for _ in range(20):
        q, f1, f2 = orc.step(q, w.dt, "tree")
    assert abs(E(q) - E0) <= 1e-6 * Eabs
    assert np.isfinite(q.x).all() and np.abs(q.x - w.x).max() > 0
