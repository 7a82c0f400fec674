"""CPU checks of the C-ABI boundary: the library builds, loads, exports every symbol include/sph.h
declares, validates configurations on the host, and refuses to compute without a CUDA device
(no CPU fallback).  No compute call is made here."""
import ctypes as C
import os
import re

import pytest

import paper_1604_03290_b200 as P
from paper_1604_03290_b200 import build as sph_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    sph_build.build()
    return P.load_library()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "sph.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 19
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/sph.h but not exported"
    assert sorted(P.EXPORTS) == names


def test_struct_layouts_match_header():
    # sizes implied by include/sph.h (LP64): material 2*int32 + 15 doubles; config 8*int32 + 2*int64 + 10 doubles
    assert C.sizeof(P.Material) == 8 + 15 * 8
    assert C.sizeof(P.Config) == 32 + 16 + 80
    assert C.sizeof(P.binding.StateIn) == 8 * (3 + 3 + 3 + 6 + 2 + 2 + 2)
    assert C.sizeof(P.binding.StateOut) == 8 * (3 + 3 + 2 + 6 + 2 + 1 + 3 + 1 + 6 + 1 + 3 + 3 + 3 + 3 + 9 + 9)


def test_workspace_sizing_and_config_validation(lib):
    ok = P.make_config(3, 100000, P.SPH_F_SOLID | P.SPH_F_GRAVITY)
    b1 = P.sph_workspace_bytes(ok)
    assert b1 > 0 and b1 % 256 == 0
    big = P.make_config(3, 200000, P.SPH_F_SOLID | P.SPH_F_GRAVITY)
    assert P.sph_workspace_bytes(big) > b1
    # C5 at full size fits a B200 many times over (DESIGN.md memory budget)
    c5 = P.make_config(3, 4_000_000, 15, n_flaws=61_000_000)
    assert P.sph_workspace_bytes(c5) < 16e9
    for bad in (P.make_config(4, 10, 0), P.make_config(3, 0, 0), P.make_config(3, 10, 0, n_materials=0),
                P.make_config(3, 10, 0, morton_bits=22), P.make_config(3, 10, 0, n_flaws=-1),
                # theta must stay below 1/sqrt(D) so that a cell containing the particle is always opened
                P.make_config(3, 10, P.SPH_F_GRAVITY, theta=0.58), P.make_config(2, 10, P.SPH_F_GRAVITY, theta=0.71)):
        assert P.sph_workspace_bytes(bad) == 0
    assert P.sph_workspace_bytes(P.make_config(2, 10, P.SPH_F_GRAVITY, theta=0.70)) > 0


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    cfg = P.make_config(3, 16, 0)
    mats = P.make_materials([dict(eos=0, brittle=0, rho0=1, K0=0, nM=0, gamma=1.4, tA=0, tB=0, tE0=1, tEiv=0,
                                  tEcv=1, ta=0, tb=0, talpha=0, tbeta=0, mu=0, Y0=0)])
    h = C.c_void_p()
    assert lib.sph_create(C.byref(cfg), mats, None, 0, None, C.byref(h)) == P.SPH_ERR_CUDA
    assert not h.value
    with pytest.raises(RuntimeError):
        P.sph_create(cfg, mats)
    assert lib.sph_upload(None, None, 0) == P.SPH_ERR_ARG
    assert lib.sph_launch_count(None) == 0


def test_product_and_oracle_share_nothing():
    pkg = os.path.join(ROOT, "paper_1604_03290_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                for needle in ("import oracle", "from oracle", "libsph_oracle", "sph_oracle", "orc_"):
                    assert needle not in txt, (f, needle)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            for needle in ("import paper_1604_03290_b200", "from paper_1604_03290_b200", "libsph_b200", "sph.h",
                           "sph_internal"):
                assert needle not in txt, (f, needle)
