"""NEXT-4: plans with per-irrep multiplicities on the CUDA path (one generated kernel
pair per multiplicity class over the rows of the whole plan) against the fp64 oracle's orc_tp_mul_* on the same inputs."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import oracle as O
from helpers import TOL_BF16, TOL_FWD, TOL_VJP, relerr, to_dev
from paper_2605_22698_b200 import binding as B
from paper_2605_22698_b200 import workloads as W

pytestmark = pytest.mark.gpu

NEQUIP = [(0, 1, 64), (0, -1, 64), (1, -1, 32), (1, 1, 32), (2, 1, 32), (2, -1, 32)]


def _ragged_graph(rng, n, max_deg):
    rcv, snd = [], []
    for r in range(n):
        d = int(rng.integers(0, max_deg + 1)) if r % 7 else 0              # isolated receivers included
        s = np.sort(rng.integers(0, n, size=d))
        rcv += [r] * d
        snd += list(s)
    return np.asarray(snd, np.int32), np.asarray(rcv, np.int32)


def _case(irreps_in, sh_lmax, out_lmax, n, max_deg, seed, natural=False, drop_paths_of=None):
    rng = np.random.default_rng(seed)
    irreps_out, paths = O.all_paths(irreps_in, sh_lmax, out_lmax, natural)
    if drop_paths_of is not None:                                            # an input irrep that no path reads
        keep = [k for k, p in enumerate(paths) if p[0] != drop_paths_of]
        irreps_out = [irreps_out[paths[k][2]] for k in keep]
        paths = [(paths[k][0], paths[k][1], j) for j, k in enumerate(keep)]
    in_size, sh_dim, out_size, w_size = O.tp_mul_dims(irreps_in, sh_lmax, irreps_out, paths)
    snd, rcv = _ragged_graph(rng, n, max_deg)
    e = len(snd)
    vec = (rng.normal(size=(e, 3)) * 2).astype(np.float32)
    x = rng.normal(size=(n, in_size)).astype(np.float32)
    w = (rng.normal(size=(e, w_size)) / np.sqrt(len(paths))).astype(np.float32)
    G = rng.normal(size=(n, out_size)).astype(np.float32)
    return (irreps_in, sh_lmax, irreps_out, paths), (in_size, sh_dim, out_size, w_size), snd, rcv, vec, x, w, G


def _run_both(pl, sizes, snd, rcv, vec, x, w, G, storage="f32"):
    n = x.shape[0]
    plan = B.e3_plan_create(*pl, B.E3_BF16 if storage == "bf16" else B.E3_F32)
    assert (plan.feats_per_node, plan.sh_dim, plan.out_per_node, plan.weights_per_edge) == sizes
    st = plan.storage
    xs, ws = W.round_to_storage(x, storage), W.round_to_storage(w, storage)
    sd, rd, vd = to_dev(snd), to_dev(rcv), to_dev(vec)
    xd, wd, Gd = to_dev(xs, st), to_dev(ws, st), to_dev(G)
    row_ptr, perm_s, col_ptr = B.e3_graph_prepare(sd, rd, n, validate=True)
    sh = B.e3_sh_fwd(plan, vd)
    out = torch.full((n, plan.out_per_node), float("nan"), device="cuda")
    B.e3_tp_scatter_fwd(plan, xd, sh, wd, sd, rd, row_ptr, n, out=out)
    dx, dY, dw = B.e3_tp_scatter_bwd(plan, xd, sh, wd, sd, rd, row_ptr, perm_s, col_ptr, n, Gd)
    out2 = B.e3_tp_scatter_fwd(plan, xd, sh, wd, sd, rd, row_ptr, n)
    dx2, dY2, dw2 = B.e3_tp_scatter_bwd(plan, xd, sh, wd, sd, rd, row_ptr, perm_s, col_ptr, n, Gd)
    torch.cuda.synchronize()
    assert torch.equal(out, out2) and torch.equal(dx, dx2) and torch.equal(dY, dY2) and torch.equal(dw, dw2)    # run-to-run bit-identical
    Y = O.sh(pl[1], vec.astype(np.float64))
    Yin = W.round_to_storage(Y, storage).astype(np.float64) if storage == "bf16" else Y
    x64, w64 = np.asarray(xs, np.float64), np.asarray(ws, np.float64)
    ref_out = O.tp_mul_fwd(*pl, x64, Yin, w64, snd, rcv, n)
    ref = O.tp_mul_bwd(*pl, x64, Yin, w64, snd, rcv, n, G.astype(np.float64))
    got = [t.float().cpu().numpy() for t in (out, dx, dY, dw)]
    assert np.isfinite(got[0]).all()
    errs = dict(out=relerr(got[0], ref_out), dx=relerr(got[1], ref[0]), dY=relerr(got[2], ref[1]), dw=relerr(got[3], ref[2]))
    return plan, errs


@pytest.mark.parametrize("irreps_in,lmax", [
    (NEQUIP, 2),
    ([(0, 1, 8), (0, -1, 8), (1, -1, 4), (1, 1, 4), (2, 1, 4), (2, -1, 4)], 2),                 # class 4 runs on the first-generation kernels
    ([(0, 1, 128), (1, -1, 64), (2, 1, 32), (3, -1, 16)], 3),                                  # four classes, l up to 3
    ([(0, 1, 64), (1, -1, 32), (1, 1, 64), (2, 1, 32)], 2),                                    # classes interleaved in the row
])
def test_unequal_multiplicities_against_the_oracle(irreps_in, lmax):
    pl, sizes, *data = _case(irreps_in, lmax, lmax, n=37, max_deg=21, seed=len(irreps_in) + lmax)
    plan, errs = _run_both(pl, sizes, *data)
    print(plan.kernel_info(0), plan.kernel_info(1), {k: f"{v:.2e}" for k, v in errs.items()})
    assert errs["out"] <= TOL_FWD and max(errs["dx"], errs["dY"], errs["dw"]) <= TOL_VJP, errs


def test_unequal_multiplicities_bf16_storage():
    pl, sizes, *data = _case(NEQUIP, 2, 2, n=23, max_deg=15, seed=11)
    _, errs = _run_both(pl, sizes, *data, storage="bf16")
    assert max(errs.values()) <= TOL_BF16, errs


def test_input_irrep_without_paths_and_natural_parity():
    # the 2o block (index 5) is read by no path: its grad_feats rows must come out as exact zeros
    pl, sizes, *data = _case(NEQUIP, 2, 2, n=19, max_deg=9, seed=5, drop_paths_of=5)
    _, errs = _run_both(pl, sizes, *data)
    assert errs["out"] <= TOL_FWD and max(errs["dx"], errs["dY"], errs["dw"]) <= TOL_VJP, errs
    pl, sizes, *data = _case(NEQUIP, 2, 2, n=19, max_deg=9, seed=6, natural=True)
    _, errs = _run_both(pl, sizes, *data)
    assert errs["out"] <= TOL_FWD and max(errs["dx"], errs["dY"], errs["dw"]) <= TOL_VJP, errs


def test_composite_plan_rejections_and_cg_table():
    with pytest.raises(B.E3Error):                                           # a path may not change the multiplicity
        B.e3_plan_create([(0, 1, 8), (1, -1, 4)], 1, [(1, -1, 8)], [(0, 1, 0), (1, 0, 0)])
    with pytest.raises(B.E3Error):                                           # multiplicities must be multiples of 4
        B.e3_plan_create([(0, 1, 8), (1, -1, 6)], 1, [(0, 1, 8), (1, -1, 6)], [(0, 0, 0), (1, 0, 1)])
    irreps_out, paths = O.all_paths(NEQUIP, 2, 2)
    plan = B.e3_plan_create(NEQUIP, 2, irreps_out, paths)
    for p in (0, 7, len(paths) - 1):                                         # e3_plan_get_cg follows the caller's path numbering
        l1, l2, l3 = NEQUIP[paths[p][0]][0], paths[p][1], irreps_out[paths[p][2]][0]
        dense = np.zeros((2 * l1 + 1, 2 * l2 + 1, 2 * l3 + 1))
        for m1, m2, m3, c in plan.get_cg(p):
            dense[m1, m2, m3] = c
        assert np.abs(dense - O.cg_real(l1, l2, l3)).max() < 1e-14


def test_session_host_path_with_unequal_multiplicities():
    pl, sizes, snd, rcv, vec, x, w, G = _case(NEQUIP, 2, 2, n=41, max_deg=17, seed=9)
    n, e = x.shape[0], len(snd)
    plan = B.e3_plan_create(*pl)
    sess = B.Session(plan, e, n)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hout = torch.empty((n, plan.out_per_node), dtype=torch.float32).pin_memory()
    hdx = torch.empty((n, plan.feats_per_node), dtype=torch.float32).pin_memory()
    hdw = torch.empty((e, plan.weights_per_edge), dtype=torch.float32).pin_memory()
    hF = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    sess.run_host(pin(vec), pin(x), pin(w), pin(snd), pin(rcv), n, grad_out=pin(G), out=hout, grad_feats=hdx, grad_weights=hdw, forces=hF)
    Y = O.sh(2, vec.astype(np.float64))
    ref_out = O.tp_mul_fwd(*pl, x.astype(np.float64), Y, w.astype(np.float64), snd, rcv, n)
    dx, dY, dw = O.tp_mul_bwd(*pl, x.astype(np.float64), Y, w.astype(np.float64), snd, rcv, n, G.astype(np.float64))
    F = O.force_reduce(O.sh_bwd(2, vec.astype(np.float64), dY), snd, rcv, n)
    assert relerr(hout.numpy(), ref_out) <= TOL_FWD
    assert relerr(hdx.numpy(), dx) <= TOL_VJP and relerr(hdw.numpy(), dw) <= TOL_VJP
    assert relerr(hF.numpy(), F) <= TOL_VJP


def test_nequip_multiplicities_on_the_config2_graph():
    """The paper's NequIP irreps (L484-L485) on a benchmark-size graph (1536 atoms, 80 518 edges, several CTA waves and both
    multiplicity classes in the launch shapes the heuristics pick for it), whole tensors against the oracle."""
    g, _ = W.make_graph(W.CONFIGS[2])
    rng = np.random.default_rng(12)
    irreps_out, paths = O.all_paths(NEQUIP, 2, 2)
    pl = (NEQUIP, 2, irreps_out, paths)
    in_size, sh_dim, out_size, w_size = O.tp_mul_dims(*pl)
    n, e = g.n_nodes, g.n_edges
    x = rng.normal(size=(n, in_size)).astype(np.float32)
    w = (rng.normal(size=(e, w_size)) / np.sqrt(len(paths))).astype(np.float32)
    G = rng.normal(size=(n, out_size)).astype(np.float32)
    _, errs = _run_both(pl, (in_size, sh_dim, out_size, w_size), g.senders, g.receivers, g.vec, x, w, G)
    print({k: f"{v:.2e}" for k, v in errs.items()})
    assert errs["out"] <= TOL_FWD and max(errs["dx"], errs["dY"], errs["dw"]) <= TOL_VJP, errs


def _random_mul_case(rng):
    """Random plan with per-irrep multiplicities (multiples of 4): random irreps of both parities, a random subset of the allowed paths
    (some input irreps end up unread), sometimes several paths of one multiplicity adding into one output block (A6), ragged graph."""
    muls = [int(m) for m in rng.choice([4, 8, 12, 16, 32, 64, 128], size=int(rng.integers(2, 4)), replace=False)]
    irreps_in = []
    for l in range(int(rng.integers(1, 4)) + 1):
        for par in (1, -1):
            if rng.random() < 0.6:
                irreps_in.append((l, par, int(rng.choice(muls))))
    if len(set(t[2] for t in irreps_in)) < 2:
        irreps_in = [(0, 1, muls[0]), (1, -1, muls[1])]
    sh_lmax, out_lmax = int(rng.integers(1, 4)), int(rng.integers(0, 4))
    irreps_out, paths = O.all_paths(irreps_in, sh_lmax, out_lmax, bool(rng.random() < 0.3))
    keep = [i for i in range(len(paths)) if rng.random() < 0.75]
    if len(keep) < 2:
        return None
    paths = [paths[i] for i in keep]
    used = sorted(set(p[2] for p in paths))
    remap = {o: k for k, o in enumerate(used)}
    irreps_out = [irreps_out[o] for o in used]
    paths = [(a, b, remap[c]) for a, b, c in paths]
    if rng.random() < 0.4:                                                   # shared output blocks: same (l, parity, mul) only
        first, new_out, m = {}, [], {}
        for k, io in enumerate(irreps_out):
            if io in first and rng.random() < 0.7:
                m[k] = first[io]
            else:
                first.setdefault(io, len(new_out))
                m[k] = len(new_out)
                new_out.append(io)
        irreps_out, paths = new_out, [(a, b, m[c]) for a, b, c in paths]
    if len(set(irreps_in[p[0]][2] for p in paths)) < 1:
        return None
    in_size, sh_dim, out_size, w_size = O.tp_mul_dims(irreps_in, sh_lmax, irreps_out, paths)
    n = int(rng.integers(1, 60))
    snd, rcv = _ragged_graph(rng, n, int(rng.integers(1, 30)))
    e = len(snd)
    vec = (rng.normal(size=(e, 3)) * 2).astype(np.float32)
    x = rng.normal(size=(n, in_size)).astype(np.float32)
    w = (rng.normal(size=(e, w_size)) / np.sqrt(len(paths))).astype(np.float32)
    G = rng.normal(size=(n, out_size)).astype(np.float32)
    return (irreps_in, sh_lmax, irreps_out, paths), (in_size, sh_dim, out_size, w_size), snd, rcv, vec, x, w, G


@pytest.mark.parametrize("block", range(3))
def test_random_plans_with_unequal_multiplicities(block, monkeypatch):
    tunes = ["", "fwd_split=2,bwd_split=2", "bwd_role_cost=1", "v2=0", "rows=12", "bwd_overlap=3", "fwd_v3=1"]
    done = 0
    for it in range(16):
        rng = np.random.default_rng(991000 + 100 * block + it)
        case = _random_mul_case(rng)
        if case is None:
            continue
        pl, sizes, *data = case
        tune = tunes[int(rng.integers(0, len(tunes)))]
        if tune:
            monkeypatch.setenv("E3_TUNE", tune)
        else:
            monkeypatch.delenv("E3_TUNE", raising=False)
        storage = "bf16" if rng.random() < 0.25 else "f32"
        try:
            _, errs = _run_both(pl, sizes, *data, storage=storage)
        except Exception as ex:
            raise AssertionError(f"block {block} it {it}: in={pl[0]} sh={pl[1]} out={pl[2]} paths={pl[3]} tune={tune!r} {storage}: {ex}") from ex
        bar_f, bar_v = (TOL_BF16, TOL_BF16) if storage == "bf16" else (TOL_FWD, TOL_VJP)
        assert errs["out"] <= bar_f and max(errs["dx"], errs["dY"], errs["dw"]) <= bar_v, (block, it, pl, tune, storage, errs)
        done += 1
    assert done >= 10
