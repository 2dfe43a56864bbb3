"""CPU-side checks of the CUDA library: it loads, exports every symbol the header declares, its host
logic (path enumeration, validation) is right, the plan kernels compile for sm_100a, and compute
calls fail loudly without a device (there is no CPU fallback)."""
import ctypes
import os
import re

import pytest
import torch

import oracle as O
from paper_2605_22698_b200 import binding as B
from paper_2605_22698_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_loads_and_exports_every_declared_symbol():
    L = B.lib()
    header = open(os.path.join(ROOT, "include", "e3b200.h")).read()
    declared = set(re.findall(r"\b(e3_[a-z_0-9]+)\s*\(", header))
    declared -= {"e3_plan", "e3_session"}
    assert declared == set(B.SYMBOLS), declared ^ set(B.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name
    assert L.e3_status_string(0) == b"ok"
    assert b"sorted" in L.e3_status_string(B.E3_ERR_UNSORTED)


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("natural", [False, True])
def test_all_paths_matches_oracle_enumerator(k, natural):
    cfg = W.CONFIGS[k]
    ii = [(l, p, cfg.channels) for l, p in cfg.irreps_in]
    io, pp = B.e3_all_paths(ii, cfg.sh_lmax, cfg.out_lmax, natural)
    io_ref, pp_ref = O.all_paths(ii, cfg.sh_lmax, cfg.out_lmax, natural)
    assert io == [tuple(t) for t in io_ref] and pp == [tuple(t) for t in pp_ref]
    expect = {1: (15, 11), 2: (13, 10), 3: (15, 11), 4: (34, 23), 5: (34, 23)}[k]
    assert len(pp) == expect[1 if natural else 0]


def test_jit_check_compiles_small_plans_without_real_spilling():
    for k in (1, 2, 3):
        cfg = W.CONFIGS[k]
        ii = [(l, p, cfg.channels) for l, p in cfg.irreps_in]
        io, pp = B.e3_all_paths(ii, cfg.sh_lmax, cfg.out_lmax)
        r = B.e3_jit_check(ii, cfg.sh_lmax, io, pp, B.E3_F32)
        # a few bytes of spill in a cold corner are tolerated; a spilling inner loop would show hundreds
        assert r["fwd_regs"] > 0 and r["bwd_regs"] > 0 and r["fwd_spill"] <= 64 and r["bwd_spill"] <= 64, r


def test_jit_check_rejects_bad_plans():
    C = 4
    with pytest.raises(B.E3Error) as e:        # triangle
        B.e3_jit_check([(0, 1, C)], 1, [(0, 1, C)], [(0, 1, 0)])
    assert e.value.status == B.E3_ERR_BAD_PATH
    with pytest.raises(B.E3Error) as e:        # parity
        B.e3_jit_check([(0, 1, C)], 1, [(1, 1, C)], [(0, 1, 0)])
    assert e.value.status == B.E3_ERR_BAD_PATH
    with pytest.raises(B.E3Error) as e:        # l > 3
        B.e3_jit_check([(4, 1, C)], 1, [(4, 1, C)], [(0, 0, 0)])
    assert e.value.status == B.E3_ERR_UNSUPPORTED
    with pytest.raises(B.E3Error) as e:        # unequal multiplicities that are not multiples of 4
        B.e3_jit_check([(0, 1, 8), (1, -1, 6)], 1, [(0, 1, 8), (1, -1, 6)], [(0, 0, 0), (1, 0, 1)])
    assert e.value.status == B.E3_ERR_UNSUPPORTED
    with pytest.raises(B.E3Error) as e:        # a channelwise path cannot change the multiplicity
        B.e3_jit_check([(0, 1, 8), (1, -1, 4)], 1, [(1, -1, 8)], [(0, 1, 0), (1, 0, 0)])
    assert e.value.status == B.E3_ERR_BAD_PATH


def test_jit_check_compiles_the_papers_nequip_irreps():
    """NEXT-4: PAPER.md L484-L485 `64x0e + 64x0o + 32x1o + 32x1e + 32x2e + 32x2o` (l_max 2, L486) is one kernel pair per
    multiplicity class; an input irrep that no path reads is allowed."""
    ii = [(0, 1, 64), (0, -1, 64), (1, -1, 32), (1, 1, 32), (2, 1, 32), (2, -1, 32)]
    io, pp = B.e3_all_paths(ii, 2, 2)
    assert len(pp) == 30 and all(io[k][2] == ii[p[0]][2] for k, p in enumerate(pp))
    r = B.e3_jit_check(ii, 2, io, pp, B.E3_F32)
    assert r["fwd_regs"] > 0 and r["bwd_regs"] > 0 and r["fwd_spill"] <= 64 and r["bwd_spill"] <= 64, r
    r = B.e3_jit_check([(0, 1, 4), (1, -1, 8)], 1, [(0, 1, 4)], [(0, 0, 0)])
    assert r["fwd_regs"] > 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device behaviour")
def test_plan_create_fails_loudly_without_a_device():
    with pytest.raises(B.E3Error) as e:
        B.e3_plan_create([(0, 1, 4)], 0, [(0, 1, 4)], [(0, 0, 0)])
    assert e.value.status == B.E3_ERR_CUDA
    assert "no CPU fallback" in str(e.value)


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2605_22698_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "e3_oracle" not in src, f


def test_symcon_jit_check_compiles_and_validates():
    """NEXT-3: the specialised symmetric-contraction kernels are generated and compiled for sm_100a without a device."""
    C = 8
    ii = [(0, 1, C), (1, -1, C), (2, 1, C)]
    io = [(0, 1, C), (1, -1, C), (2, 1, C), (0, 1, C), (2, 1, C), (1, -1, C)]
    pp = [(0, -1, 0), (1, -1, 1), (2, -1, 2), (1, 1, 3), (1, 1, 4), (1, 2, 5)]
    r = B.e3_symcon_jit_check(ii, io, pp)
    assert r["fwd_regs"] > 0 and r["fwd_spill"] == 0, r
    with pytest.raises(B.E3Error) as e:
        B.e3_symcon_jit_check([(0, 1, C)], [(3, -1, C)], [(0, 0, 0)])        # 0 x 0 -> 3: triangle rule
    assert e.value.status == B.E3_ERR_BAD_PATH
