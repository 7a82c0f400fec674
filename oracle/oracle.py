"""ctypes front end of the CPU oracle (oracle/sph_oracle.cpp).  TEST INFRASTRUCTURE ONLY:
imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs.  It never imports the CUDA package, and the CUDA package never imports it.

`evaluate()` composes one complete right-hand-side evaluation in the paper's order
(PAPER.md:693 substep list): tree build -> pseudo-particles -> interaction partners ->
[density sum] -> EoS / limiter / damaged stress -> SPH sums -> self-gravity.
`step()` is the predictor-corrector of PAPER.md:388-394 (eqs. 52-53).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

F_SOLID, F_PLASTIC, F_DAMAGE, F_GRAVITY, F_VARIABLE_H, F_DENSITY_SUM = 1, 2, 4, 8, 16, 32
F_ART_STRESS, F_XSPH = 64, 128

_P = C.POINTER
_dp = _P(C.c_double)
_ip = _P(C.c_int)
_lp = _P(C.c_longlong)


class Mat(C.Structure):
    _fields_ = [("eos", C.c_int)] + [(k, C.c_double) for k in
                ("rho0", "K0", "nM", "gamma", "tA", "tB", "tE0", "tEiv", "tEcv", "ta", "tb",
                 "talpha", "tbeta", "mu", "Y0")] + [("brittle", C.c_int)]


class Cfg(C.Structure):
    _fields_ = [("dim", C.c_int), ("flags", C.c_int), ("L", C.c_int), ("n_materials", C.c_int),
                ("n", C.c_longlong), ("theta", C.c_double), ("G", C.c_double),
                ("eps_soft", C.c_double), ("av_alpha", C.c_double), ("av_beta", C.c_double),
                ("av_eps", C.c_double), ("as_eps", C.c_double), ("as_n", C.c_double),
                ("as_mpd", C.c_double), ("xsph", C.c_double)]


class State(C.Structure):
    _fields_ = [("x", _dp * 3), ("v", _dp * 3), ("m", _dp), ("rho", _dp), ("u", _dp),
                ("S", _dp * 6), ("dmg", _dp), ("h", _dp), ("mat", _ip), ("n_act", _ip),
                ("flaw_off", _lp), ("flaw_eps", _dp)]


class Rates(C.Structure):
    _fields_ = [("drho", _dp), ("dv", _dp * 3), ("du", _dp), ("gradv", _dp * 9), ("dS", _dp * 6),
                ("ddmg", _dp), ("strain", _dp), ("C", _dp * 9), ("n_act", _ip),
                ("A_drho", _dp), ("A_dv", _dp * 3), ("A_du", _dp), ("A_gradv", _dp * 9),
                ("A_dS", _dp * 6), ("dxs", _dp * 3), ("A_dxs", _dp * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_W.restype = C.c_double
        L.orc_W.argtypes = [C.c_int, C.c_double, C.c_double]
        L.orc_dW.restype = C.c_double
        L.orc_dW.argtypes = [C.c_int, C.c_double, C.c_double]
        L.orc_eos.argtypes = [_P(Mat), C.c_double, C.c_double, _dp, _dp]
        L.orc_interleave.restype = C.c_ulonglong
        L.orc_interleave.argtypes = [C.c_int, C.c_ulonglong, C.c_ulonglong, C.c_ulonglong, C.c_int]
        L.orc_max_eig.restype = C.c_double
        L.orc_max_eig.argtypes = [C.c_int, _dp]
        L.orc_tree_build.restype = C.c_void_p
        L.orc_tree_build.argtypes = [C.c_int, C.c_longlong, C.c_int, _dp, _dp, _dp, _dp, _dp]
        L.orc_tree_free.argtypes = [C.c_void_p]
        L.orc_tree_nnodes.argtypes = [C.c_void_p]
        L.orc_tree_s0.restype = C.c_double
        L.orc_tree_s0.argtypes = [C.c_void_p]
        L.orc_tree_order.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_tree_get.argtypes = [C.c_void_p] + [C.c_void_p] * 9
        L.orc_neighbours_brute.restype = C.c_longlong
        L.orc_neighbours_brute.argtypes = [_P(Cfg), _P(State), C.c_longlong, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_neighbours_tree.restype = C.c_longlong
        L.orc_neighbours_tree.argtypes = [C.c_void_p, _P(Cfg), _P(State), C.c_longlong, C.c_void_p,
                                          C.c_void_p, C.c_void_p, C.c_longlong, C.c_int]
        L.orc_count_own_h.argtypes = [_P(Cfg), _P(State), C.c_longlong, C.c_void_p, C.c_void_p]
        L.orc_h_update.argtypes = [C.c_int, C.c_longlong, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.orc_density.argtypes = [_P(Cfg), _P(State), C.c_longlong, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_prepass.argtypes = [_P(Cfg), _P(Mat), _P(State)] + [C.c_void_p] * 4
        L.orc_rhs.argtypes = [_P(Cfg), _P(Mat), _P(State)] + [C.c_void_p] * 4 + \
                             [C.c_longlong, C.c_void_p, C.c_void_p, C.c_void_p, _P(Rates)]
        L.orc_gravity_tree.argtypes = [C.c_void_p, _P(Cfg), C.c_longlong, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_gravity_direct.argtypes = [_P(Cfg), _P(State), C.c_longlong, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _ptr(a, typ=_dp):
    return a.ctypes.data_as(typ)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def W(D, r, h):
    return lib().orc_W(int(D), float(r), float(h))


def dW(D, r, h):
    return lib().orc_dW(int(D), float(r), float(h))


def make_mats(materials):
    arr = (Mat * len(materials))()
    for i, m in enumerate(materials):
        for k, _ in Mat._fields_:
            setattr(arr[i], k, m[k])
    return arr


def eos(material, rho, u):
    m = make_mats([material])
    p, cs = C.c_double(), C.c_double()
    lib().orc_eos(m, float(rho), float(u), C.byref(p), C.byref(cs))
    return p.value, cs.value


def interleave(D, gx, gy, gz, L=21):
    return int(lib().orc_interleave(int(D), int(gx), int(gy), int(gz), int(L)))


def max_eig(D, A):
    A = _f64(np.asarray(A).reshape(9))
    return lib().orc_max_eig(int(D), _ptr(A))


class _Bound:
    """Keeps the numpy arrays a State/Cfg struct points into alive."""

    def __init__(self, w, L=21, h=None, rho=None, n_act=None):
        self.keep = []
        self.n = w.n
        self.cfg = Cfg(dim=w.dim, flags=w.flags, L=L, n_materials=len(w.materials), n=w.n,
                       theta=w.theta, G=w.G, eps_soft=w.eps_soft, av_alpha=w.av_alpha,
                       av_beta=w.av_beta, av_eps=w.av_eps, as_eps=w.as_eps, as_n=w.as_n,
                       as_mpd=w.as_mpd, xsph=w.xsph)
        self.mats = make_mats(w.materials)
        st = State()
        x, v, S = _f64(w.x), _f64(w.v), _f64(w.S)
        self.x, self.v, self.S = x, v, S
        self.m, self.u, self.dmg = _f64(w.m), _f64(w.u), _f64(w.dmg)
        self.rho = _f64(w.rho if rho is None else rho)
        self.h = _f64(w.h if h is None else h)
        self.mat = np.ascontiguousarray(w.mat, dtype=np.int32)
        self.n_act = np.ascontiguousarray(w.n_act if n_act is None else n_act, dtype=np.int32)
        self.flaw_off = np.ascontiguousarray(w.flaw_off, dtype=np.int64)
        self.flaw_eps = _f64(w.flaw_eps) if w.flaw_eps.size else np.zeros(1)
        for a in range(3):
            st.x[a] = _ptr(x[a]); st.v[a] = _ptr(v[a])
        for k in range(6):
            st.S[k] = _ptr(S[k])
        st.m, st.rho, st.u, st.dmg, st.h = map(_ptr, (self.m, self.rho, self.u, self.dmg, self.h))
        st.mat, st.n_act = _ptr(self.mat, _ip), _ptr(self.n_act, _ip)
        st.flaw_off, st.flaw_eps = _ptr(self.flaw_off, _lp), _ptr(self.flaw_eps)
        self.state = st


class Tree:
    """Reference octree + pseudo-particles."""

    def __init__(self, w, L=21, h=None):
        self.D, self.n, self.L = w.dim, w.n, L
        x = _f64(w.x)
        self._keep = (x, _f64(w.m), _f64(w.h if h is None else h))
        self.handle = lib().orc_tree_build(w.dim, w.n, L, _ptr(x[0]), _ptr(x[1]), _ptr(x[2]),
                                           _ptr(self._keep[1]), _ptr(self._keep[2]))

    def __del__(self):
        if getattr(self, "handle", None):
            lib().orc_tree_free(self.handle)
            self.handle = None

    @property
    def s0(self):
        return lib().orc_tree_s0(self.handle)

    def order(self):
        key = np.empty(self.n, dtype=np.uint64)
        perm = np.empty(self.n, dtype=np.int32)
        lib().orc_tree_order(self.handle, key.ctypes.data, perm.ctypes.data)
        return key, perm

    def nodes(self):
        nn = lib().orc_tree_nnodes(self.handle)
        out = dict(level=np.empty(nn, np.int32), prefix=np.empty(nn, np.uint64),
                   lo=np.empty(nn, np.int32), hi=np.empty(nn, np.int32), mass=np.empty(nn),
                   com=np.empty((nn, 3)), bmin=np.empty((nn, 3)), bmax=np.empty((nn, 3)),
                   hmax=np.empty(nn))
        lib().orc_tree_get(self.handle, *[out[k].ctypes.data for k in
                                          ("level", "prefix", "lo", "hi", "mass", "com", "bmin", "bmax", "hmax")])
        return out


def _targets(n, targets):
    return np.arange(n, dtype=np.int64) if targets is None else np.ascontiguousarray(targets, dtype=np.int64)


def neighbours(w, targets=None, mode="brute", tree=None, h=None, own_h=False):
    """CSR (off, idx) of interaction partners in original indices, ascending per particle."""
    b = _Bound(w, h=h)
    t = _targets(w.n, targets)
    off = np.zeros(t.size + 1, dtype=np.int64)
    if mode == "brute":
        assert not own_h
        tot = lib().orc_neighbours_brute(C.byref(b.cfg), C.byref(b.state), t.size, t.ctypes.data, off.ctypes.data, None)
        idx = np.empty(max(int(tot), 1), dtype=np.int32)
        lib().orc_neighbours_brute(C.byref(b.cfg), C.byref(b.state), t.size, t.ctypes.data, off.ctypes.data, idx.ctypes.data)
        return off, idx[:tot]
    tree = tree or Tree(w, h=h)
    tot = lib().orc_neighbours_tree(tree.handle, C.byref(b.cfg), C.byref(b.state), t.size, t.ctypes.data,
                                    off.ctypes.data, None, 0, int(own_h))
    idx = np.empty(max(int(tot), 1), dtype=np.int32)
    lib().orc_neighbours_tree(tree.handle, C.byref(b.cfg), C.byref(b.state), t.size, t.ctypes.data,
                              off.ctypes.data, idx.ctypes.data, idx.size, int(own_h))
    return off, idx[:tot]


def count_own_h(w, h=None, mode="brute"):
    if mode == "tree":
        off, _ = neighbours(w, mode="tree", h=h, own_h=True)
        return (off[1:] - off[:-1]).astype(np.int32)
    b = _Bound(w, h=h)
    t = _targets(w.n, None)
    n_a = np.empty(w.n, dtype=np.int32)
    lib().orc_count_own_h(C.byref(b.cfg), C.byref(b.state), t.size, t.ctypes.data, n_a.ctypes.data)
    return n_a


def h_update(D, h, n_a, n_des):
    h = _f64(h)
    out = np.empty_like(h)
    n_a = np.ascontiguousarray(n_a, dtype=np.int32)
    lib().orc_h_update(int(D), h.size, h.ctypes.data, n_a.ctypes.data, int(n_des), out.ctypes.data)
    return out


def density(w, off, idx, targets=None, h=None):
    b = _Bound(w, h=h)
    t = _targets(w.n, targets)
    rho = np.empty(t.size)
    idx = np.ascontiguousarray(idx, dtype=np.int32) if idx.size else np.zeros(1, np.int32)
    lib().orc_density(C.byref(b.cfg), C.byref(b.state), t.size, t.ctypes.data, off.ctypes.data,
                      idx.ctypes.data, rho.ctypes.data)
    return rho


def prepass(w, rho=None, h=None):
    b = _Bound(w, rho=rho, h=h)
    n = w.n
    p, cs, sigma, St = np.empty(n), np.empty(n), np.empty((n, 6)), np.empty((n, 6))
    lib().orc_prepass(C.byref(b.cfg), b.mats, C.byref(b.state), p.ctypes.data, cs.ctypes.data,
                      sigma.ctypes.data, St.ctypes.data)
    return p, cs, sigma, St


def rhs(w, off, idx, targets=None, rho=None, h=None, n_act=None):
    """SPH rates for the targets given their partner lists. Returns dict of (.., nt) arrays."""
    b = _Bound(w, rho=rho, h=h, n_act=n_act)
    t = _targets(w.n, targets)
    nt = t.size
    n = w.n
    p, cs, sigma, St = np.empty(n), np.empty(n), np.empty((n, 6)), np.empty((n, 6))
    lib().orc_prepass(C.byref(b.cfg), b.mats, C.byref(b.state), p.ctypes.data, cs.ctypes.data,
                      sigma.ctypes.data, St.ctypes.data)
    out = dict(drho=np.zeros(nt), dv=np.zeros((3, nt)), du=np.zeros(nt), gradv=np.zeros((9, nt)),
               dS=np.zeros((6, nt)), ddmg=np.zeros(nt), strain=np.zeros(nt), C=np.zeros((9, nt)),
               n_act=np.zeros(nt, np.int32), A_drho=np.zeros(nt), A_dv=np.zeros((3, nt)),
               A_du=np.zeros(nt), A_gradv=np.zeros((9, nt)), A_dS=np.zeros((6, nt)),
               dxs=np.zeros((3, nt)), A_dxs=np.zeros((3, nt)))
    r = Rates()
    for k, _ in Rates._fields_:
        arr = out[k]
        if arr.ndim == 2:
            for j in range(arr.shape[0]):
                getattr(r, k)[j] = _ptr(arr[j])
        else:
            setattr(r, k, _ptr(arr, _ip if arr.dtype == np.int32 else _dp))
    idx = np.ascontiguousarray(idx, dtype=np.int32) if idx.size else np.zeros(1, np.int32)
    lib().orc_rhs(C.byref(b.cfg), b.mats, C.byref(b.state), p.ctypes.data, cs.ctypes.data,
                  sigma.ctypes.data, St.ctypes.data, nt, t.ctypes.data, off.ctypes.data,
                  idx.ctypes.data, C.byref(r))
    out.update(p=p[t], cs=cs[t], sigma=sigma[t].T.copy(), St=St[t].T.copy())
    return out


def gravity_tree(w, tree=None, targets=None, theta=None, counts=None):
    """Barnes-Hut accelerations (3, nt), sums of |terms| and accepted interactions per target.  counts: a dict that
    receives the per-target work counters n_test (opening tests of eq. 50) and n_open (cells opened)."""
    tree = tree or Tree(w)
    b = _Bound(w)
    if theta is not None:
        b.cfg.theta = float(theta)
    t = _targets(w.n, targets)
    ag, A = np.zeros((3, t.size)), np.zeros((3, t.size))
    ni = np.zeros(t.size, dtype=np.int64)
    nt_, no_ = np.zeros(t.size, dtype=np.int64), np.zeros(t.size, dtype=np.int64)
    lib().orc_gravity_tree(tree.handle, C.byref(b.cfg), t.size, t.ctypes.data, ag.ctypes.data,
                           A.ctypes.data, ni.ctypes.data, nt_.ctypes.data, no_.ctypes.data)
    if counts is not None:
        counts["n_test"], counts["n_open"] = nt_, no_
    return ag, A, ni


def gravity_direct(w, targets=None):
    b = _Bound(w)
    t = _targets(w.n, targets)
    ag, pot = np.zeros((3, t.size)), np.zeros(t.size)
    lib().orc_gravity_direct(C.byref(b.cfg), C.byref(b.state), t.size, t.ctypes.data, ag.ctypes.data,
                             pot.ctypes.data)
    return ag, pot


def evaluate(w, mode="brute", targets=None, h_iters=None):
    """One complete RHS evaluation (O1-O5 of DESIGN.md) on workload state `w`.

    mode "brute": O(N^2) partner search (the definition).  mode "tree": the paper's tree walk.
    Returns a dict with the rates for `targets` (original indices; default all), the smoothing
    lengths after the eq.-73 updates, the density used, and the partner lists.
    """
    t = _targets(w.n, targets)
    h = _f64(w.h).copy()
    iters = w.h_iters if h_iters is None else h_iters
    if w.flags & F_VARIABLE_H:
        for _ in range(iters):                               # eq. 73
            n_a = count_own_h(w, h=h, mode=mode)
            h = h_update(w.dim, h, n_a, w.n_des)
    tree = Tree(w, h=h)
    rho = _f64(w.rho)
    if w.flags & F_DENSITY_SUM:                              # eq. 28 needs every particle's density
        off_all, idx_all = neighbours(w, None, mode, tree, h=h)
        rho = density(w, off_all, idx_all, None, h=h)
        if targets is None:
            off, idx = off_all, idx_all
        else:
            cnt = (off_all[1:] - off_all[:-1])[t]
            off = np.zeros(t.size + 1, np.int64)
            np.cumsum(cnt, out=off[1:])
            idx = np.concatenate([idx_all[off_all[a]:off_all[a + 1]] for a in t]) if t.size else idx_all[:0]
    else:
        off, idx = neighbours(w, t, mode, tree, h=h)
    out = rhs(w, off, idx, t, rho=rho, h=h)
    out["h"] = h
    out["rho"] = rho
    out["nb_off"], out["nb_idx"] = off, idx
    if w.flags & F_GRAVITY:
        cnt = {}
        ag, A, ni = gravity_tree(w, tree, t, counts=cnt)
        out["ag"], out["A_ag"], out["n_inter"] = ag, A, ni
        out["n_test"], out["n_open"] = cnt["n_test"], cnt["n_open"]
    else:
        out["ag"], out["A_ag"] = np.zeros((3, t.size)), np.zeros((3, t.size))
        out["n_inter"] = np.zeros(t.size, np.int64)
    out["tree"] = tree
    return out


def timestep(w, e):
    """Time-step limits of PAPER.md:396-414 from the workload state `w` and the rates `e` of one
    evaluation of ALL particles (evaluate(w, ...)):  eq. 54 (0.2 h/|dv/dt|, gravity included), eq. 55
    (0.7 h/c_s), eq. 57 (0.7 |q|/|dq/dt| over rho, u, the components of S and dmg; entries with q = 0
    or dq/dt = 0 are skipped: reading U28) and their minimum (eq. 56).  +inf where nobody sets a limit."""
    D, inf = w.dim, float("inf")
    h = e["h"]
    out = {}
    acc = np.sqrt(((e["dv"] + e["ag"])[:D] ** 2).sum(axis=0))
    out["acceleration"] = min([0.2 * h[a] / acc[a] for a in range(w.n) if acc[a] > 0.0], default=inf)
    cs = e["cs"]
    out["courant"] = min([0.7 * h[a] / cs[a] for a in range(w.n) if cs[a] > 0.0], default=inf)
    pairs = [(w.u, e["du"])]
    if not (w.flags & F_DENSITY_SUM):
        pairs.append((e["rho"], e["drho"]))
    if w.flags & F_SOLID:
        comps = (0, 1, 3) if D == 2 else range(6)
        pairs += [(w.S[k], e["dS"][k]) for k in comps]
    if w.flags & F_DAMAGE:
        pairs.append((w.dmg, e["ddmg"]))
    lim = inf
    for q, dq in pairs:
        for a in range(w.n):
            if q[a] != 0.0 and dq[a] != 0.0:
                lim = min(lim, 0.7 * abs(q[a]) / abs(dq[a]))
    out["change"] = lim
    out["dt_max"] = min(out.values())
    return out


def _limit(w):
    """S <- f_Y S after an update (eq. 16); dmg clamp (eq. 47)."""
    D = w.dim
    if (w.flags & F_SOLID) and (w.flags & F_PLASTIC):
        Y0 = np.array([m["Y0"] for m in w.materials])[w.mat]
        S = w.S
        if D == 3:
            SS = S[0] ** 2 + S[3] ** 2 + S[5] ** 2 + 2.0 * (S[1] ** 2 + S[2] ** 2 + S[4] ** 2)
        else:
            SS = S[0] ** 2 + S[3] ** 2 + 2.0 * S[1] ** 2
        J2 = 0.5 * SS
        with np.errstate(divide="ignore", invalid="ignore"):
            fY = np.where((Y0 > 0.0) & (3.0 * J2 > Y0 * Y0), Y0 * Y0 / (3.0 * J2), 1.0)
        w.S = S * fY[None, :]


def step(w, dt, mode="brute", ag_reuse=None):
    """Predictor-corrector, PAPER.md:388-394 (eqs. 52-53): two full RHS evaluations.
    Returns the new workload state (a copy) and the two evaluations.
    ag_reuse (3, n): gravity/hydro decoupling (reading U31) -- both evaluations take this
    stored gravitational acceleration instead of walking the tree."""
    D = w.dim

    def advance(base, vel, f, c, n_act_eval):
        q = base.copy()
        if w.flags & F_XSPH:
            q.x = base.x + c * (vel + f["dxs"])         # eq. 40
        else:
            q.x = base.x + c * vel                      # dx/dt = v (eq. 39)
        q.v = base.v + c * (f["dv"] + f["ag"])
        if w.flags & F_DENSITY_SUM:
            q.rho = f["rho"].copy()                     # not integrated: eq. 28 each evaluation
        else:
            q.rho = base.rho + c * f["drho"]
        q.u = base.u + c * f["du"]
        if w.flags & F_SOLID:
            q.S = base.S + c * f["dS"]
        if w.flags & F_DAMAGE:
            ntot = (base.flaw_off[1:] - base.flaw_off[:-1]).astype(np.float64)
            dmax = np.cbrt(np.where(ntot > 0, n_act_eval / np.maximum(ntot, 1.0), 0.0))
            q.dmg = np.minimum(np.maximum(base.dmg + c * f["ddmg"], 0.0), dmax)
        q.h = f["h"].copy()
        if D == 2:
            q.x[2] = 0.0
            q.v[2] = 0.0
        _limit(q)
        return q

    f1 = evaluate(w, mode)
    if ag_reuse is not None:
        f1["ag"] = np.array(ag_reuse, dtype=np.float64)
    qp = advance(w, w.v, f1, 0.5 * dt, f1["n_act"])
    qp.n_act = w.n_act.copy()                            # committed only after the corrector (U19)
    f2 = evaluate(qp, mode)
    if ag_reuse is not None:
        f2["ag"] = np.array(ag_reuse, dtype=np.float64)
    qn = advance(w, qp.v, f2, dt, f2["n_act"])
    qn.n_act = f2["n_act"].astype(np.int32)
    return qn, f1, f2


# -----------------------------------------------------------------------------------------
# Embedded Runge-Kutta integrator, PAPER.md:416-451 (eqs. 58-65)
# -----------------------------------------------------------------------------------------
def rk3_embedded(q, f, dt):
    """eqs. 58-63 for a plain vector quantity q and a rate function f(q): returns (q_rk3, q_mm,
    eps_err) with eps_err = max |q_mm - q_rk3| / |q + dt f(q)| over the entries whose denominator is
    not zero (0 when there is none).  Used by the pins; step_rk3 applies the same formulas."""
    k1 = f(q)                                            # eq. 59
    k2 = f(q + 0.5 * dt * k1)                            # eq. 60
    k3 = f(q - dt * k1 + 2.0 * dt * k2)                  # eq. 61
    q_rk3 = q + dt * (k1 / 6.0 + 4.0 * k2 / 6.0 + k3 / 6.0)   # eq. 58
    q_mm = q + dt * k2                                   # eq. 62
    den = np.abs(q + dt * k1)                            # eq. 63
    num = np.abs(q_mm - q_rk3)
    ok = den > 0.0
    return q_rk3, q_mm, (float(np.max(num[ok] / den[ok])) if ok.any() else 0.0)


def rk3_new_dt(dt, eps_err, eps_des):
    """eq. 64 (accepted: eps_err <= eps_des) and eq. 65 (rejected). Returns (accepted, dt_new)."""
    if eps_err <= eps_des:
        return True, (float("inf") if eps_err == 0.0 else dt * abs(eps_des / eps_err) ** 0.3)
    return False, 0.9 * dt * abs(eps_des / eps_err) ** 0.25


def _rk_fields(w):
    """integrated quantities and the names of their rates (reading U29: every integrated quantity
    enters the error estimate of eq. 63)"""
    names = [("x", None), ("v", None), ("u", "du")]
    if not (w.flags & F_DENSITY_SUM):
        names.append(("rho", "drho"))
    if w.flags & F_SOLID:
        names.append(("S", "dS"))
    if w.flags & F_DAMAGE:
        names.append(("dmg", "ddmg"))
    return names


def _rk_rate(w, q, f, name, rate):
    if name == "x":
        return q.v + f["dxs"] if (w.flags & F_XSPH) else q.v          # eqs. 39 / 40
    if name == "v":
        return f["dv"] + f["ag"]
    return f[rate]


def step_rk3(w, dt, eps_des, mode="brute"):
    """One step of the embedded Runge-Kutta scheme of PAPER.md:416-451 with the SPH right-hand side.
    Stage states get the same post-update rules as the predictor of the RK2 scheme (damage clamp of
    eq. 47 with the activated flaws of the evaluation that produced the newest rate, limiter of eq.
    16); n_act is committed (maximum over the three evaluations) only when the step is accepted
    (readings U29-U30).  Returns (state, eps_err, dt_new, accepted, [f1, f2, f3]); on rejection the
    state is the unchanged input."""
    D = w.dim
    fields = _rk_fields(w)

    def make_state(coeffs, ks, n_act_eval, f_last):
        q = w.copy()
        for name, _ in fields:
            val = getattr(w, name).copy()
            for c, k in zip(coeffs, ks):
                val = val + (dt * c) * k[name]
            setattr(q, name, val)
        if w.flags & F_DENSITY_SUM:
            q.rho = f_last["rho"].copy()
        if w.flags & F_DAMAGE:
            ntot = (w.flaw_off[1:] - w.flaw_off[:-1]).astype(np.float64)
            dmax = np.cbrt(np.where(ntot > 0, n_act_eval / np.maximum(ntot, 1.0), 0.0))
            q.dmg = np.minimum(np.maximum(q.dmg, 0.0), dmax)
        q.h = f_last["h"].copy()
        if D == 2:
            q.x[2] = 0.0
            q.v[2] = 0.0
        _limit(q)
        q.n_act = w.n_act.copy()
        return q

    def rates(q, f):
        return {name: _rk_rate(w, q, f, name, rate) for name, rate in fields}

    f1 = evaluate(w, mode)
    k1 = rates(w, f1)
    q2 = make_state([0.5], [k1], f1["n_act"], f1)                       # eq. 60
    f2 = evaluate(q2, mode)
    k2 = rates(q2, f2)
    q3 = make_state([-1.0, 2.0], [k1, k2], f2["n_act"], f2)             # eq. 61
    f3 = evaluate(q3, mode)
    k3 = rates(q3, f3)
    eps_err = 0.0
    for name, _ in fields:                                               # eqs. 58, 62, 63 on the raw sums
        q0 = getattr(w, name)
        q_rk3 = q0 + dt * (k1[name] / 6.0 + 4.0 * k2[name] / 6.0 + k3[name] / 6.0)
        q_mm = q0 + dt * k2[name]
        den = np.abs(q0 + dt * k1[name])
        ok = den > 0.0
        if ok.any():
            eps_err = max(eps_err, float(np.max(np.abs(q_mm - q_rk3)[ok] / den[ok])))
    accepted, dt_new = rk3_new_dt(dt, eps_err, eps_des)
    if not accepted:
        return w.copy(), eps_err, dt_new, False, [f1, f2, f3]
    n_act = np.maximum(np.maximum(f1["n_act"], f2["n_act"]), f3["n_act"]).astype(np.int32)
    qn = make_state([1.0 / 6.0, 4.0 / 6.0, 1.0 / 6.0], [k1, k2, k3], n_act, f3)
    qn.n_act = n_act
    return qn, eps_err, dt_new, True, [f1, f2, f3]
