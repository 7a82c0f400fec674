"""Thin ctypes binding of libsph_b200.so (include/sph.h).  Argument marshalling only: every step
of the path runs in the library's CUDA kernels.  PyTorch supplies device memory (the workspace and
optional device-resident inputs/outputs) and the stream.  There is no CPU fallback: importing works
anywhere (so the symbol table can be checked), but creating a context needs a CUDA device and the
compiled library, and fails loudly otherwise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsph_b200.so")

SPH_OK = 0
SPH_ERR_ARG, SPH_ERR_STATE, SPH_ERR_WORKSPACE = -1, -2, -3
SPH_ERR_NEIGHBOUR_OVERFLOW, SPH_ERR_TREE_DEPTH, SPH_ERR_CUDA = -4, -5, -6
SPH_F_SOLID, SPH_F_PLASTIC, SPH_F_DAMAGE, SPH_F_GRAVITY, SPH_F_VARIABLE_H, SPH_F_DENSITY_SUM = 1, 2, 4, 8, 16, 32
SPH_F_ART_STRESS, SPH_F_XSPH, SPH_F_RK3, SPH_F_EXPORT_GRADV = 64, 128, 256, 512

EXPORTS = ["sph_workspace_bytes", "sph_create", "sph_destroy", "sph_upload", "sph_build_tree",
           "sph_find_neighbours", "sph_rhs", "sph_gravity", "sph_evaluate", "sph_step", "sph_step_host", "sph_download",
           "sph_sync", "sph_get_order", "sph_get_tree_size", "sph_get_tree", "sph_get_neighbours",
           "sph_launch_count", "sph_last_error", "sph_version", "sph_timing_enable", "sph_timing_read",
           "sph_timing_name", "sph_get_counters", "sph_counters_enable", "sph_partition", "sph_set_partition", "sph_timestep", "sph_step_rk3", "sph_measure_fp64_peak", "sph_measure_copy_bw",
           "sph_morton_keys_static"]
SPH_T_COUNT = 11
SPH_STATIC_MAX_N = 0x3FFFFFFF          # include/sph.h: largest n of sph_morton_keys_static
SPH_STATIC_SCRATCH_BYTES = 49408

# the caller's in-place all-gather (include/sph.h: sph_exchange_fn)
EXCHANGE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_int32), C.c_int64)

_vp = C.c_void_p


class Material(C.Structure):
    _fields_ = [("eos", C.c_int32), ("brittle", C.c_int32)] + [(k, C.c_double) for k in (
        "rho0", "K0", "nM", "gamma", "tA", "tB", "tE0", "tEiv", "tEcv", "ta", "tb", "talpha", "tbeta", "mu", "Y0")]


class Config(C.Structure):
    _fields_ = [("dim", C.c_int32), ("flags", C.c_int32), ("n_materials", C.c_int32), ("morton_bits", C.c_int32),
                ("max_neighbours", C.c_int32), ("n_des", C.c_int32), ("h_iters", C.c_int32), ("gravity_every", C.c_int32),
                ("n", C.c_int64), ("n_flaws", C.c_int64), ("theta", C.c_double), ("G", C.c_double),
                ("eps_soft", C.c_double), ("av_alpha", C.c_double), ("av_beta", C.c_double), ("av_eps", C.c_double),
                ("as_eps", C.c_double), ("as_n", C.c_double), ("as_mpd", C.c_double), ("xsph", C.c_double)]


class StateIn(C.Structure):
    _fields_ = [("x", _vp * 3), ("v", _vp * 3), ("m", _vp), ("rho", _vp), ("u", _vp), ("S", _vp * 6),
                ("dmg", _vp), ("h", _vp), ("mat", _vp), ("n_act", _vp), ("flaw_off", _vp), ("flaw_eps", _vp)]


class StateOut(C.Structure):
    _fields_ = [("x", _vp * 3), ("v", _vp * 3), ("rho", _vp), ("u", _vp), ("S", _vp * 6), ("dmg", _vp), ("h", _vp),
                ("drho", _vp), ("dv", _vp * 3), ("du", _vp), ("dS", _vp * 6), ("ddmg", _vp), ("ag", _vp * 3),
                ("p", _vp), ("cs", _vp), ("strain", _vp), ("n_act", _vp), ("n_act_new", _vp), ("nb_count", _vp),
                ("dxs", _vp * 3), ("gradv", _vp * 9), ("C", _vp * 9)]


_OUT_SHAPES = dict(x=3, v=3, rho=0, u=0, S=6, dmg=0, h=0, drho=0, dv=3, du=0, dS=6, ddmg=0, ag=3, p=0, cs=0,
                   strain=0, n_act=0, n_act_new=0, nb_count=0, dxs=3, gradv=9, C=9)
_OUT_INT = ("n_act", "n_act_new", "nb_count")
STATE_FIELDS = ("x", "v", "rho", "u", "S", "dmg", "h", "n_act")
RATE_FIELDS = ("drho", "dv", "du", "dS", "ddmg", "ag", "p", "cs", "strain", "n_act_new", "nb_count", "dxs")

_lib = None


class SphError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"sph error {code}: {msg}")
        self.code = code


def load_library():
    """dlopen the compiled library and declare the signatures of include/sph.h."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1604_03290_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.sph_workspace_bytes.restype = C.c_size_t
    L.sph_workspace_bytes.argtypes = [C.POINTER(Config)]
    L.sph_create.argtypes = [C.POINTER(Config), C.POINTER(Material), _vp, C.c_size_t, _vp, C.POINTER(_vp)]
    L.sph_destroy.restype = None
    L.sph_destroy.argtypes = [_vp]
    L.sph_upload.argtypes = [_vp, C.POINTER(StateIn), C.c_int]
    for name in ("sph_build_tree", "sph_find_neighbours", "sph_rhs", "sph_gravity", "sph_evaluate", "sph_sync"):
        getattr(L, name).argtypes = [_vp]
    L.sph_step.argtypes = [_vp, C.c_double]
    L.sph_step_host.argtypes = [_vp, C.POINTER(StateIn), C.c_double]
    L.sph_download.argtypes = [_vp, C.POINTER(StateOut), C.c_int]
    L.sph_get_order.argtypes = [_vp, _vp, _vp, _vp]
    L.sph_get_tree_size.argtypes = [_vp, C.POINTER(C.c_int32)]
    L.sph_get_tree.argtypes = [_vp] + [_vp] * 11
    L.sph_get_neighbours.argtypes = [_vp, _vp, _vp, C.c_int64]
    L.sph_launch_count.restype = C.c_int64
    L.sph_launch_count.argtypes = [_vp]
    L.sph_last_error.restype = C.c_char_p
    L.sph_last_error.argtypes = [_vp]
    L.sph_version.restype = C.c_char_p
    L.sph_timing_enable.argtypes = [_vp, C.c_int]
    L.sph_timing_read.argtypes = [_vp, _vp, _vp]
    L.sph_timing_name.restype = C.c_char_p
    L.sph_timing_name.argtypes = [C.c_int]
    L.sph_get_counters.argtypes = [_vp, _vp]
    L.sph_counters_enable.argtypes = [_vp, C.c_int]
    L.sph_partition.argtypes = [C.c_int64, C.c_int, C.c_int, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.sph_set_partition.argtypes = [_vp, C.c_int, C.c_int, EXCHANGE_FN, _vp]
    L.sph_timestep.argtypes = [_vp, _vp]
    L.sph_step_rk3.argtypes = [_vp, C.c_double, C.c_double, _vp]
    L.sph_measure_fp64_peak.argtypes = [_vp, C.POINTER(C.c_double)]
    L.sph_measure_copy_bw.argtypes = [_vp, _vp, _vp, C.c_size_t, C.POINTER(C.c_double)]
    L.sph_morton_keys_static.argtypes = [_vp, _vp, _vp, C.c_int64, C.c_int32, C.c_int32, _vp, _vp, _vp, C.c_char_p, C.c_size_t]
    _lib = L
    return L


def make_config(dim, n, flags, n_materials=1, morton_bits=21, max_neighbours=128, n_des=50, h_iters=0,
                n_flaws=0, theta=0.5, G=0.0, eps_soft=0.0, av_alpha=1.0, av_beta=0.0, av_eps=0.01,
                as_eps=0.2, as_n=4.0, as_mpd=1.0, xsph=0.5, gravity_every=0):
    return Config(dim=dim, flags=flags, n_materials=n_materials, morton_bits=morton_bits,
                  max_neighbours=max_neighbours, n_des=n_des, h_iters=h_iters, gravity_every=gravity_every, n=n, n_flaws=n_flaws,
                  theta=theta, G=G, eps_soft=eps_soft, av_alpha=av_alpha, av_beta=av_beta, av_eps=av_eps,
                  as_eps=as_eps, as_n=as_n, as_mpd=as_mpd, xsph=xsph)


def make_materials(materials):
    arr = (Material * len(materials))()
    for i, m in enumerate(materials):
        for k, _ in Material._fields_:
            setattr(arr[i], k, m[k])
    return arr


def config_of(w, h_iters=None, max_neighbours=None, morton_bits=21, gravity_every=0):
    """sph_config + materials of a workload object from sph_inputs (plain field copy)."""
    cfg = make_config(w.dim, w.n, w.flags, len(w.materials), morton_bits,
                      w.max_neighbours if max_neighbours is None else max_neighbours, w.n_des,
                      w.h_iters if h_iters is None else h_iters, int(w.flaw_eps.size), w.theta, w.G, w.eps_soft,
                      w.av_alpha, w.av_beta, w.av_eps, w.as_eps, w.as_n, w.as_mpd, w.xsph, gravity_every)
    return cfg, make_materials(w.materials)


class Context:
    """Owns the device workspace (a torch uint8 tensor) and the sph_ctx handle."""

    def __init__(self, cfg, materials, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1604_03290_b200 needs a CUDA device (no CPU fallback)")
        L = load_library()
        self.torch = torch
        self.device = torch.device(device)
        self.cfg = cfg
        self.n, self.dim = int(cfg.n), int(cfg.dim)
        nbytes = L.sph_workspace_bytes(C.byref(cfg))
        if nbytes == 0:
            raise SphError(SPH_ERR_ARG, "invalid configuration")
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self.workspace.data_ptr() + 255) & ~255
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = _vp()
            rc = L.sph_create(C.byref(cfg), materials, _vp(base), nbytes, _vp(self.stream.cuda_stream), C.byref(h))
        if rc != SPH_OK:
            raise SphError(rc, "sph_create failed")
        self.handle = h
        self._keep = []

    def close(self):
        if getattr(self, "handle", None):
            load_library().sph_destroy(self.handle)
            self.handle = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != SPH_OK:
            raise SphError(rc, load_library().sph_last_error(self.handle).decode())

    # ---- marshalling helpers ----
    def _in_ptr(self, a, dtype, is_dev):
        if a is None:
            return None
        if is_dev:
            assert a.is_cuda and a.is_contiguous() and a.dtype == dtype[1], "device input must be contiguous CUDA"
            self._keep.append(a)
            return a.data_ptr()
        arr = np.ascontiguousarray(a, dtype=dtype[0])
        self._keep.append(arr)
        return arr.ctypes.data

    def _state_in(self, x=None, v=None, m=None, rho=None, u=None, S=None, dmg=None, h=None, mat=None, n_act=None,
                  flaw_off=None, flaw_eps=None, device=False):
        """sph_state_in of the given arrays (the arrays are kept alive in self._keep)."""
        t = self.torch
        f64, i32, i64 = (np.float64, t.float64), (np.int32, t.int32), (np.int64, t.int64)
        self._keep = []
        s = StateIn()
        if not device:
            conv = lambda a: a.numpy() if isinstance(a, t.Tensor) else a
            x, v, m, rho, u, S, dmg, h, mat, n_act, flaw_off, flaw_eps = map(
                lambda a: None if a is None else conv(a), (x, v, m, rho, u, S, dmg, h, mat, n_act, flaw_off, flaw_eps))
        for name, arr, cnt in (("x", x, 3), ("v", v, 3), ("S", S, 6)):
            if arr is not None:
                for k in range(cnt):
                    if cnt == 3 and k >= self.dim:
                        continue
                    getattr(s, name)[k] = self._in_ptr(arr[k], f64, device)
        for name, arr in (("m", m), ("rho", rho), ("u", u), ("dmg", dmg), ("h", h)):
            setattr(s, name, self._in_ptr(arr, f64, device))
        s.mat, s.n_act = self._in_ptr(mat, i32, device), self._in_ptr(n_act, i32, device)
        s.flaw_off = self._in_ptr(flaw_off, i64, device)
        if flaw_eps is not None and int(self.cfg.n_flaws) > 0:
            s.flaw_eps = self._in_ptr(flaw_eps, f64, device)
        return s

    def upload(self, device=False, **arrays):
        """sph_upload.  Arrays: x, v (3, n); S (6, n); others (n,); numpy/host-tensor (device=False) or CUDA
        torch tensors (device=True).  Pinned host tensors may be passed as numpy views."""
        s = self._state_in(device=device, **arrays)
        self._check(load_library().sph_upload(self.handle, C.byref(s), int(device)))
        if not device:
            self._keep = []

    def step_host(self, dt, **arrays):
        """sph_step_host: upload of HOST arrays (as for upload) and one step, the copies beside the first evaluation.
        The arrays are referenced until the next call that synchronises: do not change them before that."""
        s = self._state_in(device=False, **arrays)
        self._check(load_library().sph_step_host(self.handle, C.byref(s), float(dt)))

    def upload_workload(self, w):
        self.upload(x=w.x, v=w.v, m=w.m, rho=w.rho, u=w.u, S=w.S, dmg=w.dmg, h=w.h, mat=w.mat, n_act=w.n_act,
                    flaw_off=w.flaw_off, flaw_eps=w.flaw_eps)

    def build_tree(self):
        self._check(load_library().sph_build_tree(self.handle))

    def find_neighbours(self):
        self._check(load_library().sph_find_neighbours(self.handle))

    def rhs(self):
        self._check(load_library().sph_rhs(self.handle))

    def gravity(self):
        self._check(load_library().sph_gravity(self.handle))

    def evaluate(self):
        self._check(load_library().sph_evaluate(self.handle))

    def step(self, dt):
        self._check(load_library().sph_step(self.handle, float(dt)))

    def sync(self):
        self._check(load_library().sph_sync(self.handle))

    def download(self, fields=STATE_FIELDS + RATE_FIELDS, device=False, out=None):
        """sph_download into fresh (or caller-provided `out`) buffers; returns dict name -> array."""
        t = self.torch
        n = self.n
        res = {} if out is None else out
        s = StateOut()
        for name in fields:
            k = _OUT_SHAPES[name]
            shape = (k, n) if k else (n,)
            if name not in res:
                if device:
                    res[name] = t.zeros(shape, dtype=t.int32 if name in _OUT_INT else t.float64, device=self.device)
                else:
                    res[name] = np.zeros(shape, dtype=np.int32 if name in _OUT_INT else np.float64)
            a = res[name]
            base = a.data_ptr() if device else (a.data_ptr() if isinstance(a, t.Tensor) else a.ctypes.data)
            item = 4 if name in _OUT_INT else 8
            if k:
                for j in range(k):
                    getattr(s, name)[j] = base + j * n * item
            else:
                setattr(s, name, base)
        self._check(load_library().sph_download(self.handle, C.byref(s), int(device)))
        return res

    # ---- inspection ----
    def get_order(self):
        keys, perm, root = np.empty(self.n, np.uint64), np.empty(self.n, np.int32), np.empty(4)
        self._check(load_library().sph_get_order(self.handle, keys.ctypes.data, perm.ctypes.data, root.ctypes.data))
        return keys, perm, root

    def get_tree(self):
        nn = C.c_int32()
        self._check(load_library().sph_get_tree_size(self.handle, C.byref(nn)))
        m, NC = nn.value, 1 << self.dim
        out = dict(level=np.empty(m, np.int32), prefix=np.empty(m, np.uint64), lo=np.empty(m, np.int32),
                   hi=np.empty(m, np.int32), mass=np.empty(m), com=np.empty((m, 3)), bmin=np.empty((m, 3)),
                   bmax=np.empty((m, 3)), hmax=np.empty(m), child=np.empty((m, NC), np.int32),
                   child_lo=np.empty((m, NC + 1), np.int32))
        self._check(load_library().sph_get_tree(self.handle, *[out[k].ctypes.data for k in (
            "level", "prefix", "lo", "hi", "mass", "com", "bmin", "bmax", "hmax", "child", "child_lo")]))
        return out

    def get_neighbours(self):
        off = np.zeros(self.n + 1, np.int64)
        self._check(load_library().sph_get_neighbours(self.handle, off.ctypes.data, None, 0))
        idx = np.empty(max(int(off[-1]), 1), np.int32)
        self._check(load_library().sph_get_neighbours(self.handle, off.ctypes.data, idx.ctypes.data, idx.size))
        return off, idx[:int(off[-1])]

    def launch_count(self):
        return int(load_library().sph_launch_count(self.handle))

    def timing_enable(self, on=True):
        self._check(load_library().sph_timing_enable(self.handle, int(bool(on))))

    def timing_read(self):
        """dict stage name -> (device ms, kernel launches) accumulated since the previous read."""
        L = load_library()
        ms, ln = np.zeros(SPH_T_COUNT), np.zeros(SPH_T_COUNT, np.int64)
        self._check(L.sph_timing_read(self.handle, ms.ctypes.data, ln.ctypes.data))
        return {L.sph_timing_name(k).decode(): (float(ms[k]), int(ln[k])) for k in range(SPH_T_COUNT)}

    def step_rk3(self, dt, eps_des):
        """sph_step_rk3: returns (eps_err, dt_new, accepted)."""
        out = np.zeros(3)
        self._check(load_library().sph_step_rk3(self.handle, float(dt), float(eps_des), out.ctypes.data))
        return float(out[0]), float(out[1]), bool(out[2])

    def timestep(self):
        """sph_timestep: dict of the limits of eqs. 54, 55, 57 and their minimum (eq. 56)."""
        out = np.zeros(4)
        self._check(load_library().sph_timestep(self.handle, out.ctypes.data))
        return dict(acceleration=float(out[0]), courant=float(out[1]), change=float(out[2]), dt_max=float(out[3]))

    # ---- Morton-range sharding over the GPUs of a node (include/sph.h) ----
    def set_partition(self, rank, world, group=None, exchange=None):
        """sph_set_partition.  Every rank must have uploaded the same full state.  The all-gather of the rate arrays
        at the end of an evaluation is `exchange(tensors, slice_bytes)` if given (tests emulate ranks with it), else
        all_gather_slices over the torch.distributed group.  The library packs the slices of all rate arrays into one
        block before it calls back, so this is ONE in-place NCCL all-gather per evaluation over NVLink."""
        torch = self.torch
        if world <= 1:
            self._check(load_library().sph_set_partition(self.handle, 0, 1, EXCHANGE_FN(0), None))
            self._xfn = None
            return

        def hook(_user, _stream, n_arrays, arrays, elem_bytes, slice_elems):
            try:
                with torch.cuda.stream(self.stream):
                    sb = [int(elem_bytes[k]) * int(slice_elems) for k in range(n_arrays)]
                    ts = [device_bytes(torch, int(arrays[k]), world * sb[k], self.device) for k in range(n_arrays)]
                    if exchange is not None:
                        exchange(ts, sb)
                    else:
                        all_gather_slices(ts, sb, rank, group)
                return 0
            except Exception as e:                        # never let an exception cross the C boundary
                self._xerr = e
                return 1

        self._xfn = EXCHANGE_FN(hook)                     # keep the callback object alive
        self._check(load_library().sph_set_partition(self.handle, int(rank), int(world), self._xfn, None))

    def counters_enable(self, on=True):
        self._check(load_library().sph_counters_enable(self.handle, int(bool(on))))

    def get_counters(self):
        out = np.zeros(5, np.int64)
        self._check(load_library().sph_get_counters(self.handle, out.ctypes.data))
        return dict(n_nodes=int(out[0]), n_pairs=int(out[1]), n_inter=int(out[2]), n_visit=int(out[3]), n_open=int(out[4]))


def sph_partition(n, world, rank):
    """(lo, hi, slice) of sph_partition: the sorted indices rank `rank` of `world` owns and the slice length."""
    lo, hi, sl = C.c_int64(), C.c_int64(), C.c_int64()
    rc = load_library().sph_partition(int(n), int(world), int(rank), C.byref(lo), C.byref(hi), C.byref(sl))
    if rc != SPH_OK:
        raise SphError(rc, "sph_partition")
    return lo.value, hi.value, sl.value


class _DeviceBytes:
    def __init__(self, ptr, nbytes):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def device_bytes(torch, ptr, nbytes, device):
    """a uint8 torch tensor over `nbytes` of device memory at `ptr` (no copy; the library owns the memory)"""
    return torch.as_tensor(_DeviceBytes(ptr, nbytes), device=device)


def all_gather_slices(tensors, slice_bytes, rank, group=None):
    """In-place all-gather of flat byte tensors: rank r has filled bytes [r sb, (r + 1) sb) of every tensor; afterwards
    every tensor is complete on every rank.  Works on CUDA tensors (NCCL) and on CPU tensors (gloo, used by the tests)."""
    import torch.distributed as dist
    for t, sb in zip(tensors, slice_bytes):
        own = t[rank * sb:(rank + 1) * sb]
        if not t.is_cuda:
            own = own.clone()                             # gloo: no aliasing of input and output
        dist.all_gather_into_tensor(t, own, group=group)


# ---- module-level functions with the names of the C ABI ----
def sph_version():
    return load_library().sph_version().decode()


def sph_workspace_bytes(cfg):
    return int(load_library().sph_workspace_bytes(C.byref(cfg)))


def sph_create(cfg, materials, device="cuda:0", stream=None):
    return Context(cfg, materials, device, stream)


def sph_destroy(ctx):
    ctx.close()


def sph_upload(ctx, **arrays):
    ctx.upload(**arrays)


def sph_build_tree(ctx):
    ctx.build_tree()


def sph_find_neighbours(ctx):
    ctx.find_neighbours()


def sph_rhs(ctx):
    ctx.rhs()


def sph_gravity(ctx):
    ctx.gravity()


def sph_evaluate(ctx):
    ctx.evaluate()


def sph_step(ctx, dt):
    ctx.step(dt)


def sph_step_host(ctx, dt, **arrays):
    ctx.step_host(dt, **arrays)


def sph_download(ctx, fields=STATE_FIELDS + RATE_FIELDS, device=False, out=None):
    return ctx.download(fields, device, out)


def sph_step_rk3(ctx, dt, eps_des):
    return ctx.step_rk3(dt, eps_des)


def sph_timestep(ctx):
    return ctx.timestep()


def sph_sync(ctx):
    ctx.sync()


def sph_measure_fp64_peak(stream=None):
    """Dependency-free FP64 FMA throughput of the current device, TFLOP/s."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    v = C.c_double()
    rc = load_library().sph_measure_fp64_peak(_vp(st.cuda_stream), C.byref(v))
    if rc != SPH_OK:
        raise SphError(rc, "sph_measure_fp64_peak")
    return v.value


def sph_measure_copy_bw(nbytes=1 << 30, stream=None):
    """Streaming FP64 copy bandwidth (read + write bytes), GB/s."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    a = torch.zeros(nbytes // 8, dtype=torch.float64, device="cuda")
    b = torch.empty_like(a)
    v = C.c_double()
    rc = load_library().sph_measure_copy_bw(_vp(st.cuda_stream), _vp(a.data_ptr()), _vp(b.data_ptr()), nbytes, C.byref(v))
    if rc != SPH_OK:
        raise SphError(rc, "sph_measure_copy_bw")
    return v.value


def sph_morton_keys_static(x, y, z, keys, root=None, dim=3, morton_bits=21, stream=None):
    """Root cube and Morton keys of the particles at (x, y, z) for a caller that cannot allocate device memory
    (include/sph.h: sph_morton_keys_static): no context, no workspace; the library allocates nothing and uses its one
    fixed scratch array per GPU, so calls that may overlap on the GPU must be ordered by the caller.

    x, y, z: contiguous float64 CUDA tensors of equal length n (z may be None when dim == 2); keys: uint64 (or int64)
    CUDA tensor of length n, written in the particles' ORIGINAL order; root: float64 CUDA tensor of length 4 or None.
    Every buffer is the caller's: this wrapper, like the C call, creates none.  The work is enqueued on `stream`
    (default: torch's current stream); n > SPH_STATIC_MAX_N raises SphError(SPH_ERR_ARG)."""
    import torch
    n = int(x.numel())
    for t, dt in ((x, (torch.float64,)), (y, (torch.float64,)), (z, (torch.float64,)), (keys, (torch.uint64, torch.int64)),
                  (root, (torch.float64,))):
        if t is None:
            continue
        if not (t.is_cuda and t.is_contiguous() and t.dtype in dt and t.device == x.device):
            raise SphError(SPH_ERR_ARG, "sph_morton_keys_static: contiguous CUDA tensors of one device, float64 / uint64")
    if y.numel() != n or keys.numel() != n or (z is not None and z.numel() != n) or (root is not None and root.numel() != 4):
        raise SphError(SPH_ERR_ARG, "sph_morton_keys_static: x, y, z, keys need one length, root needs 4 entries")
    err = C.create_string_buffer(256)
    with torch.cuda.device(x.device):
        st = stream if stream is not None else torch.cuda.current_stream(x.device)
        rc = load_library().sph_morton_keys_static(
            _vp(x.data_ptr()), _vp(y.data_ptr()), _vp(z.data_ptr()) if z is not None else None, n, dim, morton_bits,
            _vp(st.cuda_stream), _vp(keys.data_ptr()), _vp(root.data_ptr()) if root is not None else None, err, len(err))
    if rc != SPH_OK:
        raise SphError(rc, err.value.decode())
