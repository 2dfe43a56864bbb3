"""A tiny whole-hot-path case run under `compute-sanitizer` (tests/test_sanitizer.py spawns it; it is also the command named in
profiles/r02_sanitizer.md).  Not collected by pytest (no test_ prefix).

    python tests/sanitizer_case.py <case> [E3_TUNE string]

cases: smoke (config 1), ragged<C> (C channels, lmax 3, degrees 0..37, e.g. ragged64), ring (the small-stage bf16 plan of
test_forward_partial_sums_fit_the_warp_ring: two paths, fsplit 4), degenerate (E = 0, hub, duplicate, zero-length, self-loop edges).
Exits non-zero when the result misses the oracle's parity bars, so a sanitizer "0 errors" run is also a correct run."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np  # noqa: E402

case = sys.argv[1] if len(sys.argv) > 1 else "smoke"
if len(sys.argv) > 2 and sys.argv[2]:
    os.environ["E3_TUNE"] = sys.argv[2]
os.environ.setdefault("E3_JIT_CACHE", "0")

from helpers import TOL_BF16, compare, gpu_plan, make_case, plan_inputs, run_gpu, run_oracle  # noqa: E402
from paper_2605_22698_b200 import workloads as W  # noqa: E402


def ragged(C, storage="f32", irr=((0, 1), (1, -1), (2, 1), (3, -1)), lmax=3):
    rng = np.random.default_rng(7 + C)
    cfg = W.small_config(channels=C, irreps_in=irr, sh_lmax=lmax, out_lmax=lmax, storage=storage)
    pl = plan_inputs(cfg)
    n = 13
    deg = rng.integers(0, 9, size=n); deg[4] = 37; deg[9] = 0
    rcv = np.repeat(np.arange(n), deg); snd = rng.integers(0, n, size=rcv.size)
    o = np.lexsort((snd, rcv)); snd, rcv = snd[o].astype(np.int32), rcv[o].astype(np.int32)
    e = rcv.size
    in_dim, out_dim = sum(2 * l + 1 for l, _ in irr), sum(2 * l + 1 for l, _, _ in pl[2])
    g = W.Graph(n, np.zeros((n, 3)), snd, rcv, (rng.normal(size=(e, 3)) * 2).astype(np.float32), 0.0)
    x = W.round_to_storage(rng.normal(size=(n, in_dim * C)), storage)
    w = W.round_to_storage(rng.normal(size=(e, len(pl[3]) * C)), storage)
    G = rng.normal(size=(n, out_dim * C)).astype(np.float32)
    plan = gpu_plan(pl, storage)
    tol = dict(tol_fwd=TOL_BF16, tol_vjp=TOL_BF16, tol_sh=8e-3) if storage == "bf16" else {}
    return compare(run_gpu(plan, g, x, w, G), run_oracle(pl, g, x, w, G, storage=storage), **tol)


if case == "smoke":
    pl, g, x, w, G = make_case(W.CONFIGS[1])
    errs = compare(run_gpu(gpu_plan(pl), g, x, w, G), run_oracle(pl, g, x, w, G))
elif case.startswith("ragged"):
    errs = ragged(int(case[6:] or 64))
elif case.startswith("bf16_"):
    errs = ragged(int(case[5:] or 64), storage="bf16")
elif case == "ring":          # the plan of test_forward_partial_sums_fit_the_warp_ring (bf16, two paths, fsplit 4) on 40 atoms
    os.environ["E3_TUNE"] = "fwd_split=4,bwd_split=3"
    rng = np.random.default_rng(78)
    C = 128
    pl = ([(0, 1, C)], 3, [(1, -1, C), (3, -1, C)], [(0, 1, 0), (0, 3, 1)])
    n = 40
    deg = rng.integers(0, 13, size=n)
    rcv = np.repeat(np.arange(n), deg); snd = rng.integers(0, n, size=rcv.size)
    o = np.lexsort((snd, rcv)); snd, rcv = snd[o].astype(np.int32), rcv[o].astype(np.int32)
    e = rcv.size
    g = W.Graph(n, np.zeros((n, 3)), snd, rcv, (rng.normal(size=(e, 3)) * 2).astype(np.float32), 0.0)
    x = W.round_to_storage(rng.normal(size=(n, C)), "bf16")
    w = W.round_to_storage(rng.normal(size=(e, 2 * C)), "bf16")
    G = rng.normal(size=(n, 10 * C)).astype(np.float32)
    plan = gpu_plan(pl, "bf16")
    errs = compare(run_gpu(plan, g, x, w, G), run_oracle(pl, g, x, w, G, storage="bf16"), tol_fwd=TOL_BF16, tol_vjp=TOL_BF16, tol_sh=8e-3)
elif case == "degenerate":
    rng = np.random.default_rng(5)
    C = 64
    cfg = W.small_config(channels=C, irreps_in=((0, 1), (1, -1)), sh_lmax=3, out_lmax=3)
    pl = plan_inputs(cfg)
    plan = gpu_plan(pl)
    P, od = len(pl[3]), sum(2 * l + 1 for l, _, _ in pl[2])
    errs = {}
    for n, snd, rcv in ((6, [], []), (10, [0, 1, 2, 3], [7, 7, 7, 7]), (40, list(rng.integers(0, 40, 300)), [11] * 300),
                        (40, [5] * 300, list(rng.integers(0, 40, 300))), (4, [1, 1, 1, 2, 2], [0, 0, 0, 0, 3]), (3, [0, 1, 2], [0, 1, 2])):
        e = len(snd)
        o = np.lexsort((snd, rcv))
        snd, rcv = np.asarray(snd, np.int32)[o], np.asarray(rcv, np.int32)[o]
        vec = (rng.normal(size=(e, 3)) * 2).astype(np.float32)
        if e > 2:
            vec[2] = 0.0
        g = W.Graph(n, np.zeros((n, 3)), snd, rcv, vec, 0.0)
        x = rng.normal(size=(n, 4 * C)).astype(np.float32)
        w = rng.normal(size=(e, P * C)).astype(np.float32)
        G = rng.normal(size=(n, od * C)).astype(np.float32)
        errs = compare(run_gpu(plan, g, x, w, G), run_oracle(pl, g, x, w, G))
else:
    raise SystemExit(f"unknown case {case}")
print("sanitizer_case", case, os.environ.get("E3_TUNE", ""), {k: f"{v:.1e}" for k, v in errs.items()})
