"""GPU parity on RANDOM plans and graphs: random input irreps, path subsets, shared output blocks (reading A6), natural-parity
tables, channel counts (second- and first-generation kernels), fp32 / bf16 storage, ragged degrees (0..120), zero-length edges and
launch-shape knobs -- each against the fp64 oracle with the bars of reading A16, and run twice for bit-identical results."""
import os

import numpy as np
import pytest

import oracle as O
from helpers import TOL_BF16, compare, gpu_plan, run_gpu, run_oracle
from paper_2605_22698_b200 import workloads as W

pytestmark = pytest.mark.gpu

TUNES = ["", "fwd_split=2,bwd_split=2", "fwd_split=4,bwd_split=3", "bwd_depth=1", "bwd_depth=1,bwd_r=2", "bwd_role_cost=1",
         "bwd_role_cost=1000000", "rows=12", "chunk=2,bwd_chunk=3", "fwd_depth_max=2"]


def _random_case(rng, medium=False):
    C = int(rng.choice([32, 64, 128] if medium else [4, 8, 16, 32, 64, 128, 256, 12, 48]))
    lmax_in, sh_lmax, out_lmax = (int(rng.integers(0, 4)) for _ in range(3))
    storage = "bf16" if rng.random() < 0.3 else "f32"
    irr = [(l, (1 if rng.random() < 0.5 else -1)) for l in range(lmax_in + 1) if rng.random() < 0.85] or [(0, 1)]
    irreps_in = [(l, p, C) for l, p in irr]
    irreps_out, paths = O.all_paths(irreps_in, sh_lmax, out_lmax, bool(rng.random() < 0.3))
    if not paths:
        return None
    keep = [i for i in range(len(paths)) if rng.random() < 0.8] or [0]          # a random subset of the allowed paths
    paths = [paths[i] for i in keep]
    used = sorted(set(p[2] for p in paths))
    remap = {o: k for k, o in enumerate(used)}
    irreps_out = [irreps_out[o] for o in used]
    paths = [(a, b, remap[c]) for a, b, c in paths]
    if rng.random() < 0.4:                                                       # several paths adding into one output block
        first, new_out, m = {}, [], {}
        for k, io in enumerate(irreps_out):
            key = (io[0], io[1])
            if key in first and rng.random() < 0.7:
                m[k] = first[key]
            else:
                first.setdefault(key, len(new_out))
                m[k] = len(new_out)
                new_out.append(io)
        irreps_out, paths = new_out, [(a, b, m[c]) for a, b, c in paths]
    pl = (irreps_in, sh_lmax, irreps_out, paths)
    if medium:                                                                   # several CTA chunks, fsplit = 1 and > 1
        n = int(rng.integers(150, 2500))
        deg = rng.integers(0, int(rng.integers(8, 60)), size=n)
    else:
        n = int(rng.integers(1, 40))
        deg = rng.integers(0, 14, size=n)
    if rng.random() < 0.3:
        deg[rng.integers(0, n)] = int(rng.integers(30, 120))
    rcv = np.repeat(np.arange(n), deg)
    snd = rng.integers(0, n, size=rcv.size)
    o = np.lexsort((snd, rcv))
    snd, rcv = snd[o].astype(np.int32), rcv[o].astype(np.int32)
    e = rcv.size
    in_dim = sum(2 * l + 1 for l, _, _ in irreps_in)
    out_dim = sum(2 * l + 1 for l, _, _ in irreps_out)
    vec = (rng.normal(size=(e, 3)) * 2).astype(np.float32)
    if e and rng.random() < 0.2:
        vec[rng.integers(0, e)] = 0                                              # zero-length edge (reading A3)
    g = W.Graph(n, np.zeros((n, 3)), snd, rcv, vec, 0.0)
    x = W.round_to_storage(rng.normal(size=(n, in_dim * C)), storage)
    w = W.round_to_storage(rng.normal(size=(e, len(paths) * C)), storage)
    G = rng.normal(size=(n, out_dim * C)).astype(np.float32)
    return pl, storage, g, x, w, G, str(rng.choice(TUNES))


@pytest.mark.parametrize("block", range(5))
def test_random_plans_against_oracle(block, monkeypatch):
    done = 0
    medium = block == 4                  # block 4: graphs of 150-2500 nodes, up to ~60k edges
    for it in range(24 if medium else 40):
        rng = np.random.default_rng(777000 + 1000 * block + it)
        case = _random_case(rng, medium)
        if case is None:
            continue
        pl, storage, g, x, w, G, tune = case
        if tune:
            monkeypatch.setenv("E3_TUNE", tune)
        else:
            monkeypatch.delenv("E3_TUNE", raising=False)
        plan = gpu_plan(pl, storage)
        gpu = run_gpu(plan, g, x, w, G)
        ref = run_oracle(pl, g, x, w, G, storage=storage)
        ctx = f"block {block} it {it}: C={pl[0][0][2]} {storage} in={pl[0]} sh={pl[1]} out={pl[2]} paths={pl[3]} E={g.n_edges} tune={tune!r}"
        try:
            if storage == "bf16":
                compare(gpu, ref, tol_fwd=TOL_BF16, tol_vjp=TOL_BF16, tol_sh=8e-3)
            else:
                compare(gpu, ref)
        except AssertionError as ex:
            raise AssertionError(f"{ctx}: {ex}") from ex
        again = run_gpu(plan, g, x, w, G)
        for k in gpu:
            assert np.array_equal(gpu[k], again[k]), f"{ctx}: {k} differs between two runs"
        done += 1
    assert done >= (18 if medium else 30)


def test_forward_partial_sums_fit_the_warp_ring(monkeypatch):
    """Regression (found by the random soak): with bf16 storage and few paths a ring stage is small, and the per-warp ring must
    still hold the fsplit partial sums (rows x lanes x 16 B): 10 rows x 32 lanes here against 6 stages of 800 B."""
    rng = np.random.default_rng(78)
    C = 128
    pl = ([(0, 1, C)], 3, [(1, -1, C), (3, -1, C)], [(0, 1, 0), (0, 3, 1)])
    n = 292
    deg = rng.integers(0, 13, size=n)
    rcv = np.repeat(np.arange(n), deg)
    snd = rng.integers(0, n, size=rcv.size)
    o = np.lexsort((snd, rcv))
    snd, rcv = snd[o].astype(np.int32), rcv[o].astype(np.int32)
    e = rcv.size
    g = W.Graph(n, np.zeros((n, 3)), snd, rcv, (rng.normal(size=(e, 3)) * 2).astype(np.float32), 0.0)
    x = W.round_to_storage(rng.normal(size=(n, C)), "bf16")
    w = W.round_to_storage(rng.normal(size=(e, 2 * C)), "bf16")
    G = rng.normal(size=(n, 10 * C)).astype(np.float32)
    monkeypatch.setenv("E3_TUNE", "fwd_split=4,bwd_split=3")
    plan = gpu_plan(pl, "bf16")
    compare(run_gpu(plan, g, x, w, G), run_oracle(pl, g, x, w, G, storage="bf16"), tol_fwd=TOL_BF16, tol_vjp=TOL_BF16, tol_sh=8e-3)
