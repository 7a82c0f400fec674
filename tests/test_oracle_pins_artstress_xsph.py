"""Pins of the oracle's artificial stress (eqs. 35-38) and XSPH (PAPER.md:305-311,
eq. 40) -- SURVEY.md 8(f) item 1.  Expectations are closed forms, invariants and an independent numpy
sum with the textbook M4 spline; none re-types the oracle's loop.  Readings U25-U27 of DESIGN.md."""
import math

import numpy as np
import pytest

import sph_inputs as si
from oracle import oracle as orc


def m4(D, r, hcfg):
    """Textbook Monaghan-Lattanzio M4 spline, support 2 h_cfg (not the oracle's form of eq. 25)."""
    q = r / hcfg
    sig = {2: 10.0 / (7.0 * math.pi), 3: 1.0 / math.pi}[D] / hcfg ** D
    return sig * np.where(q < 1.0, 1.0 - 1.5 * q * q + 0.75 * q ** 3, np.where(q < 2.0, 0.25 * (2.0 - q) ** 3, 0.0))


def _blob(n, D, seed, **kw):
    w = si.random_blob(n, D, seed, gravity=False, **kw)
    w.h[:] = w.h[0]
    w.as_mpd = (1.0 / n) ** (1.0 / D)
    return w


@pytest.mark.parametrize("D", [2, 3])
def test_xsph_matches_independent_sum_and_conserves_momentum(D):
    w = _blob(400, D, 5)
    w.flags |= si.F_XSPH
    w.xsph = 0.37
    e = orc.evaluate(w, "brute", h_iters=0)
    x, v = w.x[:D].T, w.v[:D].T
    r = np.linalg.norm(x[:, None, :] - x[None, :, :], axis=2)
    Wm = m4(D, r, 0.5 * w.h[0])
    np.fill_diagonal(Wm, 0.0)
    wgt = 2.0 * w.m[None, :] / (w.rho[:, None] + w.rho[None, :]) * Wm          # eq. 40 with (rho_a + rho_b), U26
    want = w.xsph * (wgt[:, :, None] * (v[None, :, :] - v[:, None, :])).sum(1)
    assert np.allclose(e["dxs"][:D].T, want, rtol=1e-11, atol=1e-14 * np.abs(want).max())
    # the smoothed velocity carries the same linear momentum as v (pair terms antisymmetric)
    tot = w.m[None, :] * e["dxs"]
    # sum_a m_a dxs_a = x_sph sum_ab 2 m_a m_b/(rho_a+rho_b) (v_b - v_a) W_ab = 0
    assert np.abs(tot.sum(1)).max() <= 1e-12 * np.abs(tot).sum()
    # rigid translation: no correction at all
    w2 = w.copy()
    w2.v[:] = 0.0
    w2.v[0] = 1.7
    assert not orc.evaluate(w2, "brute", h_iters=0)["dxs"].any()
    # without the flag the term is absent
    w3 = w.copy()
    w3.flags &= ~si.F_XSPH
    assert not orc.evaluate(w3, "brute", h_iters=0)["dxs"].any()


def test_xsph_moves_positions_in_the_step():
    w = si.make("C1x", scale=0.05, twin=True)
    qn, f1, f2 = orc.step(w, w.dt, mode="brute")
    w0 = w.copy()
    w0.flags &= ~si.F_XSPH
    q0, g1, g2 = orc.step(w0, w.dt, mode="brute")
    # eqs. 52-53 with eq. 40: the corrector moves x by dt (v_p + dxs_p); the velocities of the
    # predicted states differ between the two runs only through the predictor's positions
    assert np.allclose(qn.x[:2] - w.x[:2], w.dt * ((w.v + 0.5 * w.dt * (f1["dv"] + f1["ag"]))[:2] + f2["dxs"][:2]), rtol=1e-9, atol=1e-15)
    assert np.abs(qn.x - q0.x).max() > 0.0


def test_artificial_stress_two_particles_in_tension_closed_form():
    # two gas-free Murnaghan particles with rho < rho0 (p < 0, S = 0): sigma = -p delta > 0, so
    # T = (|p|/rho^2)_a + (|p|/rho^2)_b and eq. 35 scales it by (1 - eps_s (W(r)/W(dmpd))^n)
    for D in (2, 3):
        w = si.random_blob(2, D, 1, gravity=False, damage=False)
        w.flags = si.F_SOLID | si.F_ART_STRESS
        w.mat[:] = 1                                     # Murnaghan, no yield limit
        w.S[:] = 0.0
        w.v[:] = 0.0
        w.rho[:] = 0.9 * w.materials[1]["rho0"]
        w.x[:] = 0.0
        w.x[0, 1] = 0.31
        w.h[:] = 0.8
        w.as_eps, w.as_n, w.as_mpd = 0.2, 4.0, 0.5
        e1 = orc.evaluate(w, "brute")
        w0 = w.copy()
        w0.flags = si.F_SOLID
        e0 = orc.evaluate(w0, "brute")
        f = float(m4(D, np.array(0.31), 0.4) / m4(D, np.array(0.5), 0.4))
        assert e0["dv"][0, 0] > 0.0                      # tension pulls particle 0 towards particle 1
        assert np.allclose(e1["dv"], e0["dv"] * (1.0 - 0.2 * f ** 4), rtol=1e-12, atol=0.0)
        # compression: no artificial stress at all
        w.rho[:] = 1.1 * w.materials[1]["rho0"]
        w0.rho[:] = w.rho
        assert np.array_equal(orc.evaluate(w, "brute")["dv"], orc.evaluate(w0, "brute")["dv"])


@pytest.mark.parametrize("D", [2, 3])
def test_artificial_stress_keeps_momentum_and_energy_identities(D):
    w = _blob(500, D, 9)
    w.flags |= si.F_ART_STRESS | si.F_XSPH
    e = orc.evaluate(w, "brute", h_iters=0)
    w0 = w.copy()
    w0.flags &= ~(si.F_ART_STRESS | si.F_XSPH)
    e0 = orc.evaluate(w0, "brute", h_iters=0)
    assert np.abs(e["dv"] - e0["dv"]).max() > 1e-6 * np.abs(e0["dv"]).max()     # the term is active on this cloud
    P = (w.m[None, :] * e["dv"]).sum(1)
    assert np.abs(P).max() <= 1e-13 * (w.m[None, :] * np.abs(e["dv"])).sum()
    rate = (w.m * ((w.v * e["dv"]).sum(0) + e["du"])).sum()
    assert abs(rate) <= 1e-12 * (w.m * (np.abs(w.v * e["dv"]).sum(0) + np.abs(e["du"]))).sum()
    # continuity, velocity gradient and dS/dt do not see the artificial stress
    for k in ("drho", "dS", "gradv"):
        assert np.array_equal(e[k], e0[k]), k


# ------------------------------------------------------------------ time-step limits
def test_timestep_limits_hand_values_and_scaling():
    """eqs. 54-57 on hand-made rates: the planted particle sets each limit; h scales eqs. 54-55."""
    w = si.random_blob(50, 3, 2, gravity=False, damage=False)
    n = w.n
    e = dict(h=w.h.copy(), dv=np.full((3, n), 1e-3), ag=np.zeros((3, n)), cs=np.full(n, 2.0), rho=w.rho.copy(),
             drho=np.zeros(n), du=np.zeros(n), dS=np.zeros((6, n)), ddmg=np.zeros(n))
    e["dv"][:, 7] = (3.0, 4.0, 12.0)                       # |dv/dt| = 13
    e["cs"][11] = 50.0
    e["du"][5] = -4.0 * abs(w.u[5])                         # 0.7 |u|/|du/dt| = 0.175
    t = orc.timestep(w, e)
    assert t["acceleration"] == pytest.approx(0.2 * w.h[7] / 13.0, rel=1e-15)
    assert t["courant"] == pytest.approx(0.7 * w.h[11] / 50.0, rel=1e-15)
    assert t["change"] == pytest.approx(0.175, rel=1e-14)
    assert t["dt_max"] == min(t["acceleration"], t["courant"], t["change"])
    e2 = dict(e); e2["h"] = 2.0 * e["h"]
    t2 = orc.timestep(w, e2)
    assert t2["acceleration"] == pytest.approx(2.0 * t["acceleration"]) and t2["courant"] == pytest.approx(2.0 * t["courant"])
    assert t2["change"] == t["change"]
    # gravity enters eq. 54
    e3 = dict(e); e3["ag"] = -e["dv"]
    assert orc.timestep(w, e3)["acceleration"] == float("inf")
    # nobody limits: +inf
    e4 = dict(e); e4["du"] = np.zeros(n)
    assert orc.timestep(w, e4)["change"] == float("inf")


# ------------------------------------------------------------------ embedded RK3
def test_rk3_embedded_on_linear_ode_closed_forms():
    """dq/dt = lam q: eq. 58 reproduces the Taylor polynomial to third order, eq. 62 to second, so
    eq. 63 gives |z^3/6| / |1 + z| with z = lam dt; eqs. 64-65 by hand."""
    lam = np.array([-0.7, 0.3, 1.9, -2.2])
    q = np.array([1.3, -0.4, 2.5, 0.9])
    dt = 0.21
    z = lam * dt
    q_rk3, q_mm, err = orc.rk3_embedded(q, lambda y: lam * y, dt)
    assert np.allclose(q_rk3, q * (1 + z + z ** 2 / 2 + z ** 3 / 6), rtol=1e-14)
    assert np.allclose(q_mm, q * (1 + z + z ** 2 / 2), rtol=1e-14)
    assert err == pytest.approx(np.max(np.abs(z ** 3 / 6) / np.abs(1 + z)), rel=1e-12)
    # third order: halving dt divides the one-step error by ~16 (local error ~ dt^4)
    exact = lambda t: q * np.exp(lam * t)
    e1 = np.abs(orc.rk3_embedded(q, lambda y: lam * y, dt)[0] - exact(dt)).max()
    e2 = np.abs(orc.rk3_embedded(q, lambda y: lam * y, dt / 2)[0] - exact(dt / 2)).max()
    assert 12.0 < e1 / e2 < 20.0
    # zero denominators are skipped
    assert orc.rk3_embedded(np.zeros(3), lambda y: 0.0 * y, dt)[2] == 0.0
    # eqs. 64-65
    assert orc.rk3_new_dt(0.1, 1e-4, 1e-3) == (True, pytest.approx(0.1 * 10 ** 0.3))
    assert orc.rk3_new_dt(0.1, 1e-2, 1e-3) == (False, pytest.approx(0.9 * 0.1 * 0.1 ** 0.25))


def test_step_rk3_accepts_and_rejects():
    w = si.make("C1x", scale=0.05, twin=True)
    q, err, dt_new, ok, fs = orc.step_rk3(w, w.dt, 1e30)
    assert ok and err > 0.0 and dt_new > w.dt
    q2, err2, dt2, ok2, _ = orc.step_rk3(w, w.dt, 1e-30)
    assert not ok2 and err2 == err and dt2 < w.dt
    assert np.array_equal(q2.x, w.x) and np.array_equal(q2.v, w.v) and np.array_equal(q2.S, w.S)
    # the accepted state is close to the RK2 state (both at least second order)
    q_rk2, _, _ = orc.step(w, w.dt)
    assert np.abs(q.v - q_rk2.v).max() <= 1e-3 * np.abs(q_rk2.v).max()
