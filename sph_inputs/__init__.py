"""Seeded synthetic inputs for the five workloads of BASELINE.json (C1..C5).

This module serves BOTH the CPU oracle (oracle/) and the CUDA path
(paper_1604_03290_b200/). It holds none of the method's arithmetic: no SPH
kernel, no equation of state, no tree, no sums. It only lays particles out and
fills the per-particle state arrays and material parameter tables.  The paper
uses no public dataset; these inputs take the shapes, sizes and material values
of its experiments (PAPER.md:497-501 rubber rings, :503-552 collapsing cloud,
:554-566 Al impact, :568-578 basalt impact, :584-661 Ceres-mass collision) as
BASELINE.json configs[0..4] restate them, and stand in for them.

Conventions
-----------
* ``h`` is the PAPER's smoothing length: the kernel vanishes for r/h > 1
  (eq. 25), i.e. h is the support radius.  BASELINE.json's
  "h = 1.3 dx with a 2h cubic spline" is the same kernel with h_paper = 2.6 dx.
* Stress components are stored as S[6] = (xx, xy, xz, yy, yz, zz).
* Flaws (eq. 45) are input data: a CSR table of activation
  threshold strains per particle, ascending within a particle.

Every generator takes ``seed`` and ``scale`` (scale < 1 gives a smaller
instance of the same workload: same geometry and physics, fewer particles).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# flags (mirrored by include/sph.h and by oracle/; plain integers, no arithmetic)
F_SOLID = 1
F_PLASTIC = 2
F_DAMAGE = 4
F_GRAVITY = 8
F_VARIABLE_H = 16
F_DENSITY_SUM = 32
F_ART_STRESS = 64      # artificial stress, PAPER.md:284-302 (eqs. 35-38)
F_XSPH = 128           # XSPH velocity smoothing, PAPER.md:311 (eq. 40)
F_RK3 = 256            # library only: reserve the rate buffers of the embedded Runge-Kutta step

EOS_IDEAL_GAS = 0
EOS_MURNAGHAN = 1
EOS_TILLOTSON = 2


def material(eos, rho0=1.0, K0=0.0, nM=0.0, gamma=0.0, tA=0.0, tB=0.0, tE0=1.0,
             tEiv=0.0, tEcv=1.0, ta=0.0, tb=0.0, talpha=0.0, tbeta=0.0, mu=0.0,
             Y0=0.0, brittle=0):
    return dict(eos=int(eos), rho0=float(rho0), K0=float(K0), nM=float(nM),
                gamma=float(gamma), tA=float(tA), tB=float(tB), tE0=float(tE0),
                tEiv=float(tEiv), tEcv=float(tEcv), ta=float(ta), tb=float(tb),
                talpha=float(talpha), tbeta=float(tbeta), mu=float(mu),
                Y0=float(Y0), brittle=int(brittle))


# BASELINE.json configs[2]: aluminium (Tillotson)
AL = material(EOS_TILLOTSON, rho0=2700.0, tA=75.2e9, tB=65e9, tE0=5e6, tEiv=3e6,
              tEcv=13.9e6, ta=0.5, tb=1.63, talpha=5.0, tbeta=5.0, mu=26.7e9,
              Y0=0.3e9)
# BASELINE.json configs[3]: basalt; E_iv/E_cv from PAPER.md:615 (Table 1)
BASALT = material(EOS_TILLOTSON, rho0=2860.0, tA=26.7e9, tB=26.7e9, tE0=487e6,
                  tEiv=4.72e6, tEcv=18.2e6, ta=0.5, tb=1.5, talpha=5.0,
                  tbeta=5.0, mu=22.7e9, Y0=3.5e9, brittle=1)
NYLON = material(EOS_MURNAGHAN, rho0=1185.0, K0=2.5e9, nM=4.0, mu=1e9, Y0=0.0)
RUBBER = material(EOS_MURNAGHAN, rho0=1.0, K0=1.0, nM=4.0, mu=0.22, Y0=0.0)
GAS = material(EOS_IDEAL_GAS, gamma=5.0 / 3.0)


@dataclass
class Workload:
    name: str
    dim: int
    flags: int
    materials: list
    x: np.ndarray          # (3, n) float64 (row 2 is zero for dim 2)
    v: np.ndarray          # (3, n)
    m: np.ndarray          # (n,)
    rho: np.ndarray
    u: np.ndarray
    S: np.ndarray          # (6, n)
    dmg: np.ndarray        # d^(1/3) in [0, 1]
    h: np.ndarray          # paper's h = support radius
    mat: np.ndarray        # int32 material index
    n_act: np.ndarray      # int32 activated flaws (latched)
    flaw_off: np.ndarray   # int64 (n+1,)
    flaw_eps: np.ndarray   # float64 (n_flaws,), ascending per particle
    theta: float = 0.5
    G: float = 0.0
    eps_soft: float = 0.0
    av_alpha: float = 1.0
    av_beta: float = 0.0
    av_eps: float = 0.01
    as_eps: float = 0.2    # artificial stress factor, exponent n and mean particle distance (eqs. 37-38)
    as_n: float = 4.0
    as_mpd: float = 1.0
    xsph: float = 0.5      # XSPH factor of eq. 40
    n_des: int = 50
    h_iters: int = 0
    dt: float = 1e-3
    steps: int = 10
    max_neighbours: int = 128
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.m.shape[0])

    def copy(self) -> "Workload":
        kw = {}
        for k, val in self.__dict__.items():
            kw[k] = val.copy() if isinstance(val, np.ndarray) else (
                dict(val) if isinstance(val, dict) else val)
        return Workload(**kw)

    def subset(self, idx) -> "Workload":
        """Particles idx only (flaw table re-packed). For tiny test cases."""
        idx = np.asarray(idx, dtype=np.int64)
        w = self.copy()
        for k in ("x", "v", "S"):
            setattr(w, k, np.ascontiguousarray(getattr(self, k)[:, idx]))
        for k in ("m", "rho", "u", "dmg", "h", "mat", "n_act"):
            setattr(w, k, np.ascontiguousarray(getattr(self, k)[idx]))
        cnt = (self.flaw_off[1:] - self.flaw_off[:-1])[idx]
        off = np.zeros(len(idx) + 1, dtype=np.int64)
        np.cumsum(cnt, out=off[1:])
        eps = np.empty(int(off[-1]), dtype=np.float64)
        for j, a in enumerate(idx):
            eps[off[j]:off[j + 1]] = self.flaw_eps[self.flaw_off[a]:self.flaw_off[a + 1]]
        w.flaw_off, w.flaw_eps = off, eps
        return w


def _empty_flaws(n):
    return np.zeros(n + 1, dtype=np.int64), np.zeros(0, dtype=np.float64)


def _zeros_state(n):
    return dict(v=np.zeros((3, n)), u=np.zeros(n), S=np.zeros((6, n)),
                dmg=np.zeros(n), n_act=np.zeros(n, dtype=np.int32))


def weibull_flaws(rng, brittle_idx, n, k_w, m_w, volume):
    """Flaw assignment as the paper states it: flaw j = 1, 2, ...
    goes to a random brittle particle with threshold (j / (k V))^(1/m) until every
    brittle particle holds at least one.  Returns CSR (flaw_off[n+1], flaw_eps)."""
    nb = len(brittle_idx)
    off = np.zeros(n + 1, dtype=np.int64)
    if nb == 0:
        return off, np.zeros(0, dtype=np.float64)
    seen = np.zeros(nb, dtype=bool)
    n_seen = 0
    picks = []
    chunk = max(nb, 1024)
    while True:
        c = rng.integers(0, nb, size=chunk, dtype=np.int64)
        uniq, first = np.unique(c, return_index=True)
        needed = ~seen[uniq]
        if n_seen + int(np.count_nonzero(needed)) == nb:
            # coverage completes inside this chunk: cut at the position where it does
            last = int(first[needed].max())
            picks.append(c[:last + 1])
            break
        seen[uniq] = True
        n_seen += int(np.count_nonzero(needed))
        picks.append(c)
    who = np.concatenate(picks)
    T = who.shape[0]
    j = np.arange(1, T + 1, dtype=np.float64)
    eps_all = (j / (k_w * volume)) ** (1.0 / m_w)
    order = np.argsort(who, kind="stable")          # ascending j within a particle
    cnt = np.bincount(who, minlength=nb)
    cnt_full = np.zeros(n, dtype=np.int64)
    cnt_full[brittle_idx] = cnt
    np.cumsum(cnt_full, out=off[1:])
    # brittle_idx is ascending, so CSR order over all particles == order over brittle ones
    return off, np.ascontiguousarray(eps_all[order])


def _lattice_in_sphere(dx, radius, dim=3):
    k = int(math.ceil(radius / dx)) + 1
    ax = np.arange(-k, k + 1, dtype=np.float64) * dx
    if dim == 3:
        X, Y, Z = np.meshgrid(ax, ax, ax, indexing="ij")
        keep = (X * X + Y * Y + Z * Z) <= radius * radius
        return np.stack([X[keep], Y[keep], Z[keep]])
    X, Y = np.meshgrid(ax, ax, indexing="ij")
    keep = (X * X + Y * Y) <= radius * radius
    return np.stack([X[keep], Y[keep], np.zeros(int(keep.sum()))])


def _perturb(w: Workload, rng, cs_of_mat):
    """Parity twin: same geometry, every branch of the rate equations exercised on
    every particle (velocity noise, density spread, Tillotson regimes, stresses above
    the yield limit, partial damage)."""
    n, D = w.n, w.dim
    cs = np.array([cs_of_mat[int(k)] for k in w.mat])
    L = max(float(np.ptp(w.x[a])) for a in range(D)) or 1.0
    for a in range(D):
        phase = 2.0 * math.pi * w.x[(a + 1) % D] / L * 3.0
        w.v[a] += 0.02 * cs * (np.sin(phase) + rng.uniform(-1.0, 1.0, n))
    rho0 = np.array([w.materials[int(k)]["rho0"] for k in w.mat])
    gas = np.array([w.materials[int(k)]["eos"] == EOS_IDEAL_GAS for k in w.mat])
    xi = rng.uniform(0.0, 1.0, n)
    if not (w.flags & F_DENSITY_SUM):
        w.rho = np.where(gas, w.rho, rho0 * (1.0 + 0.04 * (xi - 0.5)))
    till = np.array([w.materials[int(k)]["eos"] == EOS_TILLOTSON for k in w.mat])
    if till.any():
        Ecv = np.array([w.materials[int(k)]["tEcv"] for k in w.mat])
        # u spread over (0, 1.5 E_cv): below E_iv, between, above E_cv all occur
        w.u = np.where(till, rng.uniform(0.0, 1.5, n) * Ecv, w.u)
    if w.flags & F_SOLID:
        mu = np.array([w.materials[int(k)]["mu"] for k in w.mat])
        Y0 = np.array([w.materials[int(k)]["Y0"] for k in w.mat])
        amp = np.where(Y0 > 0.0, 2.0 * Y0 / math.sqrt(3.0), 0.05 * mu)
        A = rng.uniform(-1.0, 1.0, (3, 3, n))
        A = 0.5 * (A + A.transpose(1, 0, 2))
        if D == 2:
            A[2, :, :] = 0.0
            A[:, 2, :] = 0.0
        tr = (A[0, 0] + A[1, 1] + A[2, 2]) / D
        for a in range(D):
            A[a, a] -= tr
        J2 = 0.5 * np.einsum("abn,abn->n", A, A)
        A *= (amp * rng.uniform(0.1, 1.0, n) / np.sqrt(np.maximum(J2, 1e-300)))[None, None, :]
        w.S = np.ascontiguousarray(np.stack([A[0, 0], A[0, 1], A[0, 2], A[1, 1], A[1, 2], A[2, 2]]))
    if w.flags & F_DAMAGE:
        brittle = np.array([w.materials[int(k)]["brittle"] == 1 for k in w.mat])
        w.dmg = np.where(brittle, rng.uniform(0.0, 0.9, n), 0.0)
        ntot = (w.flaw_off[1:] - w.flaw_off[:-1])
        w.n_act = np.minimum(rng.integers(0, 3, n), ntot).astype(np.int32)
    w.name += "-twin"
    return w


# ----------------------------------------------------------------------------------------
# C1: 2-D rubber rings (BASELINE.json configs[0])
# ----------------------------------------------------------------------------------------
def c1_rubber_rings(seed=1604, scale=1.0, twin=False):
    rng = np.random.default_rng(seed)
    dx = 0.1 / math.sqrt(scale)
    k = int(math.ceil(4.0 / dx)) + 1
    ax = np.arange(-k, k + 1, dtype=np.float64) * dx
    X, Y = np.meshgrid(ax, ax, indexing="ij")
    r2 = X * X + Y * Y
    keep = (r2 >= 9.0) & (r2 <= 16.0)
    ring = np.stack([X[keep], Y[keep]])
    nr = ring.shape[1]
    n = 2 * nr
    x = np.zeros((3, n))
    x[0, :nr] = ring[0] - 5.0
    x[0, nr:] = ring[0] + 5.0
    x[1, :nr] = ring[1]
    x[1, nr:] = ring[1]
    x[:2] += rng.uniform(-0.01 * dx, 0.01 * dx, (2, n))
    st = _zeros_state(n)
    st["v"][0, :nr] = +0.059
    st["v"][0, nr:] = -0.059
    off, eps = _empty_flaws(n)
    w = Workload(name="C1-rubber-rings-2d", dim=2, flags=F_SOLID, materials=[RUBBER],
                 x=x, m=np.full(n, 1.0 * dx * dx), rho=np.ones(n), h=np.full(n, 2.6 * dx),
                 mat=np.zeros(n, dtype=np.int32), flaw_off=off, flaw_eps=eps,
                 av_alpha=1.0, av_beta=0.0, dt=1e-3, steps=20, max_neighbours=48,
                 meta=dict(dx=dx), **st)
    if twin:
        _perturb(w, rng, {0: 1.0})
    return w


def c1x_rubber_rings_paper(seed=1604, scale=1.0, twin=False):
    """C1 with the settings of the paper's own ring test: artificial stress
    eps_s = 0.2, n = 4, dmpd = the lattice spacing, and XSPH with x_sph = 0.5."""
    w = c1_rubber_rings(seed=seed, scale=scale, twin=twin)
    w.name = w.name.replace("C1", "C1x")
    w.flags |= F_ART_STRESS | F_XSPH
    w.as_eps, w.as_n, w.as_mpd, w.xsph = 0.2, 4.0, w.meta["dx"], 0.5
    return w


# ----------------------------------------------------------------------------------------
# C2: 3-D self-gravitating gas sphere, rho ~ 1/r (BASELINE.json configs[1])
# ----------------------------------------------------------------------------------------
def c2_gas_sphere(seed=1605, scale=1.0, twin=False, n=None):
    from scipy.spatial import cKDTree
    rng = np.random.default_rng(seed)
    n = int(n if n is not None else max(256, round(65536 * scale)))
    rs = np.empty(0)
    while rs.size < n:                       # rejection: accept r with probability r
        r = rng.uniform(0.0, 1.0, 2 * n)
        a = rng.uniform(0.0, 1.0, 2 * n)
        rs = np.concatenate([rs, r[a < r]])
    rs = rs[:n]
    cth = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * math.pi, n)
    sth = np.sqrt(1.0 - cth * cth)
    x = np.stack([rs * sth * np.cos(phi), rs * sth * np.sin(phi), rs * cth])
    # h: midway between the 50th and 51st neighbour distance -> exactly 50 partners inside h
    kd = cKDTree(x.T)
    nd = min(52, n)
    d, _ = kd.query(x.T, k=nd)               # d[:,0] is the particle itself
    h = 0.5 * (d[:, nd - 2] + d[:, nd - 1])
    st = _zeros_state(n)
    st["u"][:] = 0.05
    off, eps = _empty_flaws(n)
    w = Workload(name="C2-gas-sphere-gravity", dim=3,
                 flags=F_GRAVITY | F_VARIABLE_H | F_DENSITY_SUM, materials=[GAS],
                 x=np.ascontiguousarray(x), m=np.full(n, 1.0 / n), rho=np.ones(n), h=h,
                 mat=np.zeros(n, dtype=np.int32), flaw_off=off, flaw_eps=eps,
                 theta=0.5, G=1.0, eps_soft=0.01, av_alpha=1.0, av_beta=2.0,
                 n_des=50, h_iters=1, dt=1e-3, steps=10, max_neighbours=192, **st)
    if twin:
        _perturb(w, rng, {0: math.sqrt(5.0 / 3.0 * 2.0 / 3.0 * 0.05)})
    return w


def _cube_lattice(edge, npts):
    dx = edge / npts
    ax = (np.arange(npts, dtype=np.float64) + 0.5) * dx - 0.5 * edge
    X, Y, Z = np.meshgrid(ax, ax, ax, indexing="ij")
    return dx, np.stack([X.ravel(), Y.ravel(), Z.ravel()])


def _impact(name, seed, scale, twin, edge, npts_full, proj_radius, speed, target_mat,
            proj_mat, flags, weibull, dt):
    rng = np.random.default_rng(seed)
    npts = max(6, int(round(npts_full * scale ** (1.0 / 3.0))))
    dx, cube = _cube_lattice(edge, npts)
    # projectile on the same lattice, touching the +z face, flying along -z
    sph = _lattice_in_sphere(dx, max(proj_radius, 1.01 * dx))
    z_top = 0.5 * edge - 0.5 * dx
    kz = math.ceil((max(proj_radius, 1.01 * dx)) / dx) + 1
    shift = np.array([0.5 * dx if npts % 2 == 0 else 0.0] * 2 + [0.0])
    sph = sph + shift[:, None]
    sph[2] += z_top + kz * dx
    x = np.ascontiguousarray(np.concatenate([cube, sph], axis=1))
    nt, npj = cube.shape[1], sph.shape[1]
    n = nt + npj
    mats = [target_mat, proj_mat]
    mat = np.zeros(n, dtype=np.int32)
    mat[nt:] = 1
    rho = np.where(mat == 0, target_mat["rho0"], proj_mat["rho0"]).astype(np.float64)
    st = _zeros_state(n)
    st["v"][2, nt:] = -speed
    if weibull is not None:
        k_w, m_w = weibull
        brittle_idx = np.flatnonzero(np.array([mats[k]["brittle"] for k in mat]) == 1)
        off, eps = weibull_flaws(rng, brittle_idx, n, k_w, m_w, edge ** 3)
    else:
        off, eps = _empty_flaws(n)
    w = Workload(name=name, dim=3, flags=flags, materials=mats, x=x, m=rho * dx ** 3,
                 rho=rho, h=np.full(n, 2.6 * dx), mat=mat, flaw_off=off, flaw_eps=eps,
                 av_alpha=0.5, av_beta=0.0, dt=dt, steps=10, max_neighbours=128,
                 meta=dict(dx=dx, n_target=nt, n_projectile=npj), **st)
    if twin:
        cs = {k: math.sqrt((mm["tA"] if mm["eos"] == EOS_TILLOTSON else mm["K0"]) / mm["rho0"])
              for k, mm in enumerate(mats)}
        _perturb(w, rng, cs)
    return w


# C3: aluminium sphere into aluminium cube (BASELINE.json configs[2])
def c3_al_impact(seed=1606, scale=1.0, twin=False):
    return _impact("C3-al-impact", seed, scale, twin, edge=0.1, npts_full=79,
                   proj_radius=0.005, speed=7000.0, target_mat=AL, proj_mat=AL,
                   flags=F_SOLID | F_PLASTIC, weibull=None, dt=1e-8)


# C4: nylon sphere into basalt cube with Weibull flaws (BASELINE.json configs[3])
def c4_basalt_impact(seed=1607, scale=1.0, twin=False):
    return _impact("C4-basalt-impact-damage", seed, scale, twin, edge=0.2, npts_full=126,
                   proj_radius=0.0032, speed=4000.0, target_mat=BASALT, proj_mat=NYLON,
                   flags=F_SOLID | F_PLASTIC | F_DAMAGE, weibull=(4e35, 9.0), dt=1e-8)


# C5: two self-gravitating basalt spheres (BASELINE.json configs[4])
def c5_ceres_collision(seed=1608, scale=1.0, twin=False):
    rng = np.random.default_rng(seed)
    R = 470e3
    n_each = 2.0e6 * scale
    dx = R * (4.0 / 3.0 * math.pi / n_each) ** (1.0 / 3.0)
    body = _lattice_in_sphere(dx, R)
    nb = body.shape[1]
    n = 2 * nb
    # centres in contact (distance 2R + dx) along a line at 45 deg to the relative velocity (x)
    sep = 2.0 * R + dx
    c = 0.5 * sep * np.array([math.cos(math.pi / 4), math.sin(math.pi / 4), 0.0])
    x = np.concatenate([body - c[:, None], body + c[:, None]], axis=1)
    x += rng.uniform(-0.01 * dx, 0.01 * dx, (3, n))
    x = np.ascontiguousarray(x)
    st = _zeros_state(n)
    st["v"][0, :nb] = +2500.0
    st["v"][0, nb:] = -2500.0
    rho = np.full(n, BASALT["rho0"])
    vol = 2.0 * (4.0 / 3.0) * math.pi * R ** 3
    off, eps = weibull_flaws(rng, np.arange(n, dtype=np.int64), n, 4e35, 9.0, vol)
    w = Workload(name="C5-ceres-collision-gravity", dim=3,
                 flags=F_SOLID | F_PLASTIC | F_DAMAGE | F_GRAVITY, materials=[BASALT],
                 x=x, m=rho * dx ** 3, rho=rho, h=np.full(n, 2.6 * dx),
                 mat=np.zeros(n, dtype=np.int32), flaw_off=off, flaw_eps=eps,
                 theta=0.5, G=6.674e-11, eps_soft=0.0, av_alpha=0.5, av_beta=0.0,
                 dt=0.05, steps=5, max_neighbours=128, meta=dict(dx=dx, n_each=nb), **st)
    if twin:
        _perturb(w, rng, {0: math.sqrt(BASALT["tA"] / BASALT["rho0"])})
    return w


# Table 1 of the paper (Benz & Asphaug 1999): basalt and water ice; Table 2 (the two k
# values printed on one line: basalt 1e61 m^-3 with m = 16, ice 1e46 m^-3 with m = 9.1)
BASALT_T1 = material(EOS_TILLOTSON, rho0=2700.0, tA=26.7e9, tB=26.7e9, tE0=487e6, tEiv=4.72e6, tEcv=18.2e6, ta=0.5,
                     tb=1.5, talpha=5.0, tbeta=5.0, mu=22.7e9, Y0=3.5e9, brittle=1)
ICE = material(EOS_TILLOTSON, rho0=917.0, tA=9.47e9, tB=9.47e9, tE0=10e6, tEiv=0.773e6, tEcv=3.04e6, ta=0.3, tb=0.1,
               talpha=10.0, tbeta=5.0, mu=2.8e9, Y0=1e9, brittle=1)
WEIBULL_T2 = {0: (1e61, 16.0), 1: (1e46, 9.1)}      # material index -> (k [m^-3], m)


# C6 (second workload): the two-material bodies of the paper's section 5.1:
# a target of one Ceres mass with a basalt core and a 30 wt-% water-ice mantle (R_T = 509 km) and a solid-basalt
# projectile of the same mass (R_P = 437 km), in contact at 45 degrees like C5, both brittle with their own Weibull sets.
def c6_ice_mantle(seed=1609, scale=1.0, twin=False):
    rng = np.random.default_rng(seed)
    M = 9.43e20
    v_core, v_ice = 0.7 * M / BASALT_T1["rho0"], 0.3 * M / ICE["rho0"]
    r_core = (3.0 * v_core / (4.0 * math.pi)) ** (1.0 / 3.0)
    r_t = (3.0 * (v_core + v_ice) / (4.0 * math.pi)) ** (1.0 / 3.0)            # 509 km
    r_p = (3.0 * (M / BASALT_T1["rho0"]) / (4.0 * math.pi)) ** (1.0 / 3.0)      # 437 km
    n_tot = 400_000.0 * scale                                                    # twice the paper's 200 000
    dx = ((4.0 / 3.0) * math.pi * (r_t ** 3 + r_p ** 3) / n_tot) ** (1.0 / 3.0)
    tgt, prj = _lattice_in_sphere(dx, r_t), _lattice_in_sphere(dx, r_p)
    nt, npj = tgt.shape[1], prj.shape[1]
    n = nt + npj
    mat = np.zeros(n, dtype=np.int32)
    mat[:nt] = (np.sqrt((tgt ** 2).sum(0)) > r_core).astype(np.int32)           # 1 = ice mantle
    sep = r_t + r_p + dx
    c = sep * np.array([math.cos(math.pi / 4), math.sin(math.pi / 4), 0.0])
    frac = r_p ** 3 / (r_t ** 3 + r_p ** 3)                                       # place the contact point near the origin
    x = np.concatenate([tgt - frac * c[:, None], prj + (1.0 - frac) * c[:, None]], axis=1)
    x += rng.uniform(-0.01 * dx, 0.01 * dx, (3, n))
    x = np.ascontiguousarray(x)
    mats = [BASALT_T1, ICE]
    rho = np.array([m_["rho0"] for m_ in mats])[mat]
    st = _zeros_state(n)
    v_imp = 877.0                                                                # 1.7 v_esc
    st["v"][0, :nt] = +0.5 * v_imp
    st["v"][0, nt:] = -0.5 * v_imp
    # flaws: every material with its own Weibull set over its own volume (eq. 45 per material)
    cnt = np.zeros(n, dtype=np.int64)
    parts = {}
    for k, (k_w, m_w) in WEIBULL_T2.items():
        idx = np.flatnonzero(mat == k)
        vol = idx.size * dx ** 3
        off_k, eps_k = weibull_flaws(rng, idx, n, k_w, m_w, vol)
        cnt += off_k[1:] - off_k[:-1]
        parts[k] = eps_k
    off = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(cnt, out=off[1:])
    eps = np.empty(int(off[-1]), dtype=np.float64)
    owner = np.repeat(mat, cnt)                                                  # material of every CSR slot
    for k in parts:
        eps[owner == k] = parts[k]
    w = Workload(name="C6-ice-mantle-collision-gravity", dim=3,
                 flags=F_SOLID | F_PLASTIC | F_DAMAGE | F_GRAVITY, materials=mats, x=x, m=rho * dx ** 3, rho=rho,
                 h=np.full(n, 2.6 * dx), mat=mat, flaw_off=off, flaw_eps=eps, theta=0.5, G=6.674e-11, eps_soft=0.0,
                 av_alpha=0.5, av_beta=0.0, dt=0.05, steps=5, max_neighbours=128,
                 meta=dict(dx=dx, n_target=nt, n_projectile=npj, r_core=r_core, r_target=r_t, r_projectile=r_p), **st)
    if twin:
        _perturb(w, rng, {k: math.sqrt(mm["tA"] / mm["rho0"]) for k, mm in enumerate(mats)})
    return w


def twin_of(w, seed=0):
    """Parity twin of an already generated nominal workload: a copy with the same geometry and flaw table and the
    seeded perturbations of _perturb (used by bench.py to time the state the kernels see in a running simulation
    without generating the particles and flaws a second time)."""
    q = w.copy()
    amp = {}
    for k, mm in enumerate(q.materials):            # velocity-noise amplitude per material (a scale, not the EoS)
        if mm["eos"] == EOS_TILLOTSON:
            amp[k] = math.sqrt(mm["tA"] / mm["rho0"])
        elif mm["eos"] == EOS_MURNAGHAN:
            amp[k] = math.sqrt(mm["K0"] / mm["rho0"])
        else:
            amp[k] = math.sqrt(mm["gamma"] * (mm["gamma"] - 1.0) * float(np.mean(q.u)))
    return _perturb(q, np.random.default_rng(seed), amp)


CONFIGS = {"C1": c1_rubber_rings, "C1x": c1x_rubber_rings_paper, "C2": c2_gas_sphere, "C3": c3_al_impact,
           "C4": c4_basalt_impact, "C5": c5_ceres_collision, "C6": c6_ice_mantle}


def make(name, scale=1.0, twin=False, seed=None):
    fn = CONFIGS[name]
    return fn(scale=scale, twin=twin) if seed is None else fn(seed=seed, scale=scale, twin=twin)


def random_blob(n, dim=3, seed=0, solid=True, gravity=True, variable_h=False, damage=True,
                duplicates=0):
    """Small disordered test cloud (not one of the five workloads) for tests: uniform
    random points in a unit box, every physics branch switched on, optional exactly
    duplicated positions (degenerate multi-particle leaves)."""
    rng = np.random.default_rng(seed)
    x = np.zeros((3, n))
    x[:dim] = rng.uniform(0.0, 1.0, (dim, n))
    if duplicates:
        src = rng.integers(0, n - duplicates, duplicates)
        x[:, n - duplicates:] = x[:, src]
    dxm = (1.0 / n) ** (1.0 / dim)
    h = np.full(n, 2.6 * dxm)
    if variable_h:
        h = h * rng.uniform(0.8, 1.25, n)
    mats = [material(EOS_TILLOTSON, rho0=2.0, tA=3.0, tB=2.0, tE0=4.0, tEiv=0.5, tEcv=1.5,
                     ta=0.5, tb=1.3, talpha=5.0, tbeta=5.0, mu=1.1, Y0=0.2, brittle=1),
            material(EOS_MURNAGHAN, rho0=1.5, K0=2.0, nM=4.0, mu=0.7, Y0=0.0),
            material(EOS_IDEAL_GAS, gamma=1.4)]
    if not solid:
        mats = [mats[2]]
    mat = rng.integers(0, len(mats), n).astype(np.int32)
    rho0 = np.array([mats[k]["rho0"] for k in mat])
    rho = rho0 * rng.uniform(0.9, 1.1, n)
    flags = (F_SOLID | F_PLASTIC if solid else 0) | (F_GRAVITY if gravity else 0) | \
            (F_VARIABLE_H if variable_h else 0) | (F_DAMAGE if (solid and damage) else 0)
    st = _zeros_state(n)
    st["v"][:dim] = rng.uniform(-0.3, 0.3, (dim, n))
    st["u"][:] = rng.uniform(0.0, 2.0, n)
    if solid and damage:
        bidx = np.flatnonzero(np.array([mats[k]["brittle"] for k in mat]) == 1)
        off, eps = weibull_flaws(rng, bidx, n, 1e4, 3.0, 1.0)
    else:
        off, eps = _empty_flaws(n)
    w = Workload(name=f"blob{dim}d-{n}", dim=dim, flags=flags, materials=mats, x=x,
                 m=rho * dxm ** dim * rng.uniform(0.8, 1.2, n), rho=rho, h=h, mat=mat,
                 flaw_off=off, flaw_eps=eps, theta=0.5, G=1.0 if gravity else 0.0,
                 eps_soft=0.01, av_alpha=1.0, av_beta=2.0, dt=1e-3, steps=2,
                 max_neighbours=256, **st)
    if solid:
        cs = {0: math.sqrt(3.0 / 2.0), 1: math.sqrt(2.0 / 1.5), 2: 1.0}
        name = w.name
        _perturb(w, rng, cs)
        w.name = name
        w.rho = rho
    return w
