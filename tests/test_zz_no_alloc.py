"""sph_morton_keys_static: Morton keys for callers that cannot allocate device memory.

Why the call exists: every other compute call of the library works inside a context, and a context needs a device
workspace that the caller allocates.  A plug-in that is handed device pointers by an application which owns the GPU memory
pool, a time loop that must never pay the device-wide stall of cudaMalloc / cudaFree, or a process at its memory limit has
inputs and outputs but no way to get that workspace.  For them the library keeps the scratch of the bounding-box reduction
in a fixed array of its own device image (SPH_STATIC_SCRATCH_BYTES per GPU, sets of up to SPH_STATIC_MAX_N particles) and
allocates nothing (include/sph.h, csrc/static_keys.cu).

What is checked: root cube and keys are integer / bit-pattern work, so the bar is bit-exact agreement with the existing
path (sph_upload + sph_build_tree, read back with sph_get_order) -- on TWO calls in a row on one stream without a
synchronisation in between, the second on a smaller set in another dimension and another box, so that anything the first
call left in the shared scratch (partial boxes of blocks the second call does not launch, the old root cube, the arrival
counter) would show up as wrong keys.  The file is named to be collected last: `pytest -x` stops at the first failure,
and this test is an addition to the hot path's parity suite, not a gate in front of it.  It passes alone in a fresh process
(first call = the address look-up of the scratch) and after the other GPU tests (library already in use).
"""
import ctypes as C

import numpy as np
import pytest

import sph_inputs


@pytest.fixture(scope="module")
def P():
    import paper_1604_03290_b200 as P
    from paper_1604_03290_b200 import build
    build.build()
    return P


def _existing_path(P, w, morton_bits):
    """Root cube and keys through a context: sorted keys + permutation -> keys in original order."""
    cfg, mats = P.config_of(w, morton_bits=morton_bits)
    ctx = P.sph_create(cfg, mats)
    ctx.upload_workload(w)
    ctx.build_tree()
    keys_sorted, perm, root = ctx.get_order()
    ctx.close()
    keys = np.empty_like(keys_sorted)
    keys[perm] = keys_sorted
    return keys, root


def _device_inputs(torch, w):
    x = torch.from_numpy(np.ascontiguousarray(w.x)).cuda()
    return x[0].contiguous(), x[1].contiguous(), (x[2].contiguous() if w.dim == 3 else None)


@pytest.mark.gpu
def test_static_keys_equal_the_context_path_on_two_calls_in_a_row(P):
    import torch
    # A: 3-D, 300 000 particles (more 256-thread blocks than the 1024 partial boxes of the scratch: every slot is written),
    #    box with negative and positive coordinates.  B: 2-D, 5 000 particles (20 blocks), another box, 13 bits.
    wa = sph_inputs.random_blob(300_000, dim=3, seed=5, damage=False)
    wa.x[:3] = (wa.x[:3] - 0.37) * 3.1
    wb = sph_inputs.random_blob(5_000, dim=2, seed=6, damage=False)
    wb.x[:2] = wb.x[:2] * 0.25 + 7.0
    cases = [(wa, 21), (wb, 13)]
    expect = [_existing_path(P, w, bits) for w, bits in cases]

    # the caller's buffers: inputs and outputs only (torch stands in for the application that owns the memory)
    bufs = []
    for w, _ in cases:
        x, y, z = _device_inputs(torch, w)
        keys = torch.full((w.n,), -1, dtype=torch.int64, device="cuda")     # poisoned: every key must be written
        root = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
        bufs.append((x, y, z, keys, root))
    torch.cuda.synchronize()

    def both_calls():
        for (w, bits), (x, y, z, keys, root) in zip(cases, bufs):           # back to back, same stream, no sync between
            P.sph_morton_keys_static(x, y, z, keys, root, dim=w.dim, morton_bits=bits)
        torch.cuda.synchronize()

    def check():
        for (w, _), (x, y, z, keys, root), (ekeys, eroot) in zip(cases, bufs, expect):
            got = keys.cpu().numpy().view(np.uint64)
            assert np.array_equal(root.cpu().numpy(), eroot), (w.name, root.cpu().numpy(), eroot)
            assert np.array_equal(got, ekeys), f"{w.name}: {np.count_nonzero(got != ekeys)} keys differ"

    both_calls()
    check()

    # once more, now that the look-up of the first call on this GPU is behind us: the library must not have taken device
    # memory (an allocation would lower the free memory by at least one 2 MiB page)
    for _, _, _, keys, root in bufs:
        keys.fill_(-1)
        root.fill_(float("nan"))
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    both_calls()
    free_after, _ = torch.cuda.mem_get_info()
    check()
    assert free_after >= free_before, (free_before, free_after)


@pytest.mark.gpu
def test_static_keys_degenerate_sets(P):
    """One particle, and a set of coincident particles (edge 0 -> the root cube takes edge 1, as in the context path)."""
    import torch
    for n in (1, 700):
        x = torch.full((n,), -2.5, dtype=torch.float64, device="cuda")
        y = torch.full((n,), 0.125, dtype=torch.float64, device="cuda")
        z = torch.full((n,), 9.0, dtype=torch.float64, device="cuda")
        keys = torch.full((n,), -1, dtype=torch.int64, device="cuda")
        root = torch.empty(4, dtype=torch.float64, device="cuda")
        P.sph_morton_keys_static(x, y, z, keys, root, dim=3)
        assert root.cpu().tolist() == [-2.5, 0.125, 9.0, 1.0]
        assert (keys == 0).all().item()


def test_static_keys_reject_bad_sizes_before_touching_the_gpu(P):
    """Sizes beyond the stated maximum (and other bad arguments) are refused with a message; this runs without a GPU too,
    because the arguments are checked before the first CUDA call (the pointers are never followed)."""
    L = P.load_library()
    err = C.create_string_buffer(256)
    fake = C.c_void_p(256)
    call = lambda n, dim=3, bits=21, x=fake, keys=fake: L.sph_morton_keys_static(   # noqa: E731
        x, fake, fake, n, dim, bits, None, keys, None, err, len(err))
    assert call(P.binding.SPH_STATIC_MAX_N + 1) == P.SPH_ERR_ARG
    assert b"SPH_STATIC_MAX_N" in err.value and str(P.binding.SPH_STATIC_MAX_N).encode() in err.value
    assert call(1 << 40) == P.SPH_ERR_ARG
    assert call(0) == P.SPH_ERR_ARG and b"n = 0" in err.value
    assert call(10, dim=4) == P.SPH_ERR_ARG and b"dim" in err.value
    assert call(10, bits=22) == P.SPH_ERR_ARG and b"morton_bits" in err.value
    assert call(10, x=None) == P.SPH_ERR_ARG and b"NULL" in err.value
    assert call(10, keys=None) == P.SPH_ERR_ARG
    # the message buffer is optional
    assert L.sph_morton_keys_static(fake, fake, fake, 0, 3, 21, None, fake, None, None, 0) == P.SPH_ERR_ARG
    # the header's constants are the ones the binding repeats
    import os
    import re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "sph.h")).read()
    assert int(re.search(r"#define SPH_STATIC_MAX_N (0x[0-9a-f]+)", hdr).group(1), 16) == P.binding.SPH_STATIC_MAX_N
    assert int(re.search(r"#define SPH_STATIC_SCRATCH_BYTES (\d+)", hdr).group(1)) == P.binding.SPH_STATIC_SCRATCH_BYTES


def test_static_keys_without_a_device_fail_loudly(P):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    L = P.load_library()
    err = C.create_string_buffer(256)
    fake = C.c_void_p(256)
    assert L.sph_morton_keys_static(fake, fake, fake, 10, 3, 21, None, fake, None, err, len(err)) == P.SPH_ERR_CUDA
    assert b"no CUDA device" in err.value
