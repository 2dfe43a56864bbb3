"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on
identical seeded inputs.  Bars (BASELINE.json north_star, reading A16): indices bit-exact; forward
max|err|/max|ref| <= 1e-5; VJP and forces <= 1e-4; bf16 storage <= 2e-2."""
import numpy as np
import pytest
import torch

import oracle as O
from helpers import (TOL_BF16, compare, gpu_plan, make_case, plan_inputs, relerr, run_gpu, run_oracle, to_dev)
from paper_2605_22698_b200 import binding as B
from paper_2605_22698_b200 import workloads as W

pytestmark = pytest.mark.gpu


# ------------------------------------------------------------------ plan / CG planner kernel
@pytest.mark.parametrize("k", [1, 2, 4])
def test_planner_cg_matches_oracle(k):
    cfg = W.CONFIGS[k]
    pl = plan_inputs(cfg)
    plan = gpu_plan(pl)
    nnz = 0
    for p, (i_in, l2, i_out) in enumerate(pl[3]):
        l1, l3 = pl[0][i_in][0], pl[2][i_out][0]
        ref = O.cg_real(l1, l2, l3)
        got = np.zeros_like(ref)
        for m1, m2, m3, c in plan.get_cg(p):
            got[m1, m2, m3] = c
        assert np.abs(got - ref).max() < 1e-14
        assert np.count_nonzero(got) == int((np.abs(ref) > 1e-12).sum())
        nnz += np.count_nonzero(got)
    assert nnz == plan.nnz_total == {1: 137, 2: 134, 4: 611}[k]          # SURVEY 8(d) totals
    assert (plan.in_dim, plan.sh_dim, plan.out_dim) == O.plan_dims(*pl)


# ------------------------------------------------------------------ graph preparation (bit exact)
@pytest.mark.parametrize("n,e,kind", [(1, 0, "rand"), (7, 1, "rand"), (50, 400, "rand"), (2000, 60000, "rand"),
                                      (300, 9000, "hub"), (64, 500, "dup")])
def test_graph_prepare_bit_exact(n, e, kind):
    rng = np.random.default_rng(n + e)
    snd = rng.integers(0, n, size=e)
    rcv = rng.integers(0, n, size=e)
    if kind == "hub":
        snd[: e // 2] = 3                       # one sender with thousands of out-edges
        rcv[e // 2:] = 5
    if kind == "dup":
        snd[:100] = 1; rcv[:100] = 2            # duplicate edges
    o = np.lexsort((snd, rcv))
    snd, rcv = snd[o].astype(np.int32), rcv[o].astype(np.int32)
    row_ptr, perm_s, col_ptr = B.e3_graph_prepare(to_dev(snd), to_dev(rcv), n, validate=True)
    assert np.array_equal(row_ptr.cpu().numpy(), np.concatenate([[0], np.cumsum(np.bincount(rcv, minlength=n))]))
    assert np.array_equal(col_ptr.cpu().numpy(), np.concatenate([[0], np.cumsum(np.bincount(snd, minlength=n))]))
    assert np.array_equal(perm_s.cpu().numpy(), np.argsort(snd, kind="stable"))


def test_graph_prepare_validation_errors():
    snd = to_dev(np.array([0, 1, 2], np.int32))
    with pytest.raises(B.E3Error) as e:
        B.e3_graph_prepare(snd, to_dev(np.array([2, 1, 0], np.int32)), 3, validate=True)
    assert e.value.status == B.E3_ERR_UNSORTED
    with pytest.raises(B.E3Error) as e:
        B.e3_graph_prepare(snd, to_dev(np.array([0, 1, 7], np.int32)), 3, validate=True)
    assert e.value.status == B.E3_ERR_INVALID_ARG


# ------------------------------------------------------------------ spherical harmonics
@pytest.mark.parametrize("lmax", [0, 1, 2, 3])
def test_sh_fwd_bwd_parity(lmax):
    rng = np.random.default_rng(lmax)
    n = 5000 + 77                                # several 128-edge tiles and a ragged tail
    vec = (rng.normal(size=(n, 3)) * rng.uniform(0.05, 5.0, size=(n, 1))).astype(np.float32)
    vec[17] = 0.0                                # zero-length edge (reading A3)
    vec[18] = [0, 0, 2.5]
    vec[19] = [0, 0, -1e-3]
    C = 4
    plan = B.e3_plan_create([(0, 1, C)], lmax, [(0, 1, C)], [(0, 0, 0)])
    sh = B.e3_sh_fwd(plan, to_dev(vec)).cpu().numpy()
    ref = O.sh(lmax, vec.astype(np.float64))
    assert relerr(sh, ref) <= 2e-6
    assert sh[17, 0] == 1.0 and not sh[17, 1:].any()
    gsh = rng.normal(size=(n, (lmax + 1) ** 2)).astype(np.float32)
    gv = B.e3_sh_bwd(plan, to_dev(vec), to_dev(gsh)).cpu().numpy()
    gref = O.sh_bwd(lmax, vec.astype(np.float64), gsh.astype(np.float64))
    assert relerr(gv, gref) <= 1e-5
    assert not gv[17].any()
    assert B.e3_sh_fwd(plan, to_dev(vec[:0])).shape == (0, (lmax + 1) ** 2)


# ------------------------------------------------------------------ the five configs
@pytest.mark.parametrize("k", [1, 2, 3])
def test_full_path_parity_configs_1_2_3(k):
    cfg = W.CONFIGS[k]
    pl, g, x, w, G = make_case(cfg)
    plan = gpu_plan(pl)
    gpu = run_gpu(plan, g, x, w, G)
    ref = run_oracle(pl, g, x, w, G)
    errs = compare(gpu, ref)
    print(cfg.name, "E", g.n_edges, {k_: f"{v:.2e}" for k_, v in errs.items()})


def test_natural_parity_plan_config2():
    cfg = W.CONFIGS[2]
    pl, g, x, w, G = make_case(cfg, natural=True)
    assert len(pl[3]) == 10
    plan = gpu_plan(pl)
    compare(run_gpu(plan, g, x, w, G), run_oracle(pl, g, x, w, G))


# ------------------------------------------------------------------ tiny adversarial graphs / plans
def _tiny(rng, n, e):
    snd = rng.integers(0, n, size=e); rcv = rng.integers(0, n, size=e)
    o = np.lexsort((snd, rcv))
    return snd[o].astype(np.int32), rcv[o].astype(np.int32)


@pytest.mark.parametrize("C", [1, 3, 4, 8, 16, 32, 33, 64, 96, 128, 256])
def test_channel_counts_and_ragged_lanes(C):
    rng = np.random.default_rng(C)
    cfg = W.small_config(n_atoms=9, channels=C, irreps_in=((0, 1), (1, -1), (2, 1)), sh_lmax=2, out_lmax=2)
    pl = plan_inputs(cfg)
    n, e = 9, 40
    snd, rcv = _tiny(rng, n, e)
    g = W.Graph(n, np.zeros((n, 3)), snd, rcv, (rng.normal(size=(e, 3)) * 2).astype(np.float32), 0.0)
    x = rng.normal(size=(n, 9 * C)).astype(np.float32)
    w = rng.normal(size=(e, len(pl[3]) * C)).astype(np.float32)
    G = rng.normal(size=(n, 51 * C)).astype(np.float32)
    plan = gpu_plan(pl)
    compare(run_gpu(plan, g, x, w, G), run_oracle(pl, g, x, w, G))


def test_degenerate_graphs():
    rng = np.random.default_rng(5)
    C = 64
    cfg = W.small_config(channels=C, irreps_in=((0, 1), (1, -1)), sh_lmax=3, out_lmax=3)
    pl = plan_inputs(cfg)
    plan = gpu_plan(pl)
    P, od = len(pl[3]), sum(2 * l + 1 for l, _, _ in pl[2])

    def case(n, snd, rcv, vec=None):
        e = len(snd)
        o = np.lexsort((snd, rcv))
        snd, rcv = np.asarray(snd, np.int32)[o], np.asarray(rcv, np.int32)[o]
        vec = (rng.normal(size=(e, 3)) * 2).astype(np.float32) if vec is None else vec
        g = W.Graph(n, np.zeros((n, 3)), snd, rcv, vec, 0.0)
        x = rng.normal(size=(n, 4 * C)).astype(np.float32)
        w = rng.normal(size=(e, P * C)).astype(np.float32)
        G = rng.normal(size=(n, od * C)).astype(np.float32)
        gpu, ref = run_gpu(plan, g, x, w, G), run_oracle(pl, g, x, w, G)
        compare(gpu, ref)
        return gpu

    out = case(6, [], [])["out"]                                   # E = 0: every row written as zeros
    assert out.shape == (6, od * C) and not out.any()
    gpu = case(10, [0, 1, 2, 3], [7, 7, 7, 7])                      # isolated receivers 0..6, 8, 9
    assert not gpu["out"][:7].any() and not gpu["out"][8:].any() and not gpu["dx"][4:].any()
    case(40, list(rng.integers(0, 40, 300)), [11] * 300)            # one hub receiver with 300 in-edges
    case(40, [5] * 300, list(rng.integers(0, 40, 300)))             # one hub sender with 300 out-edges
    case(4, [1, 1, 1, 2, 2], [0, 0, 0, 0, 3])                       # duplicate edges
    v = (rng.normal(size=(5, 3))).astype(np.float32); v[2] = 0.0    # a zero-length edge (A3)
    case(4, [1, 2, 3, 0, 1], [0, 0, 0, 2, 3], v)
    case(3, [0, 1, 2], [0, 1, 2])                                   # self loops are legal input


def test_shared_output_block_and_partial_plans():
    rng = np.random.default_rng(6)
    C = 64
    irreps_in = [(0, 1, C), (1, -1, C), (2, 1, C)]
    # two + three paths adding into shared blocks (reading A6); input irrep 2 and SH l=1 partly unused
    irreps_out = [(1, -1, C), (2, 1, C)]
    paths = [(0, 1, 0), (1, 0, 0), (1, 2, 0), (2, 0, 1), (0, 2, 1), (1, 1, 1)]
    pl = (irreps_in, 2, irreps_out, paths)
    n, e = 12, 70
    snd, rcv = _tiny(rng, n, e)
    g = W.Graph(n, np.zeros((n, 3)), snd, rcv, (rng.normal(size=(e, 3)) * 2).astype(np.float32), 0.0)
    x = rng.normal(size=(n, 9 * C)).astype(np.float32)
    w = rng.normal(size=(e, len(paths) * C)).astype(np.float32)
    G = rng.normal(size=(n, 8 * C)).astype(np.float32)
    plan = gpu_plan(pl)
    compare(run_gpu(plan, g, x, w, G), run_oracle(pl, g, x, w, G))


def test_vjp_with_arbitrary_sh_input_and_no_grad_weights():
    rng = np.random.default_rng(7)
    cfg = W.small_config(channels=64, irreps_in=((0, 1), (1, -1), (2, 1), (3, -1)), sh_lmax=3, out_lmax=3)
    pl = plan_inputs(cfg)
    n, e = 20, 150
    snd, rcv = _tiny(rng, n, e)
    g = W.Graph(n, np.zeros((n, 3)), snd, rcv, rng.normal(size=(e, 3)).astype(np.float32), 0.0)
    x = rng.normal(size=(n, 16 * 64)).astype(np.float32)
    w = rng.normal(size=(e, 34 * 64)).astype(np.float32)
    G = rng.normal(size=(n, 156 * 64)).astype(np.float32)
    Y = rng.normal(size=(e, 16)).astype(np.float32)                # Y as a free input of the trilinear map
    plan = gpu_plan(pl)
    gpu = run_gpu(plan, g, x, w, G, sh_override=Y, want_forces=False)
    ref = run_oracle(pl, g, x, w, G, sh_override=Y, want_forces=False)
    gpu["sh"] = ref["sh"]                                          # SH kernel not involved here
    compare(gpu, ref)
    # grad_weights = NULL skips it and leaves the other gradients unchanged
    snd_d, rcv_d = to_dev(snd), to_dev(rcv)
    rp, ps, cp = B.e3_graph_prepare(snd_d, rcv_d, n)
    dx, dY, dw = B.e3_tp_scatter_bwd(plan, to_dev(x), to_dev(Y), to_dev(w), snd_d, rcv_d, rp, ps, cp, n, to_dev(G),
                                     want_grad_weights=False)
    assert dw is None
    assert np.array_equal(dx.cpu().numpy(), gpu["dx"]) and np.array_equal(dY.cpu().numpy(), gpu["dY"])


# ------------------------------------------------------------------ launch-shape variants of the generated kernels
@pytest.mark.parametrize("tune", [
    "fwd_split=1,bwd_split=1", "fwd_split=2,bwd_split=3", "fwd_split=4,bwd_split=4",       # warps / CTAs sharing a receiver
    "bwd_role_cost=1", "bwd_role_cost=1000000",                                               # one role per input irrep / a single role
    "bwd_depth=1", "bwd_depth=1,bwd_r=2", "bwd_depth=1,bwd_r=2,bwd_role_cost=1000000",        # ring stages, half-unit weights ring
    "fwd_depth_max=2", "rows=12", "rows=20,rows_hard=30,fwd_minb=2", "chunk=3,bwd_chunk=5",   # forward ring depth, role sizes, CTA order
    "bwd_v2=0", "v2=0",                                                                       # first-generation kernels
    # third-generation forward (opt-in; team CTAs, mbarrier ring): team shapes, ring depth / lag, CTA order, TMA bulk operand copies
    "fwd_v3=1", "fwd_v3=1,fwd_v3_lag=2", "fwd_v3=1,team=2", "fwd_v3=1,team=4,fwd_v3_depth=2", "fwd_v3=1,team=1,fwd_v3_chunk=5",
    "fwd_v3=1,fwd_v3_depth=8,fwd_split=2", "fwd_v3=1,fwd_v3_depth=3,fwd_v3_lag=2,fwd_split=4", "fwd_v3=1,fwd_v3_bulk=1", "fwd_v3=1,fwd_v3_bulk=1,fwd_split=2,team=2",
])
@pytest.mark.parametrize("C", [32, 64, 128])
def test_launch_shape_variants(tune, C, monkeypatch):
    """E3_TUNE only moves work between warps / CTAs / ring stages; every variant must meet the same parity bars.
    C = 32 / 64 / 128 gives 4 / 2 / 1 edges per warp step; degrees 0..90 give ragged steps and empty parts."""
    rng = np.random.default_rng(1000 + C)
    cfg = W.small_config(channels=C, irreps_in=((0, 1), (1, -1), (2, 1), (3, -1)), sh_lmax=3, out_lmax=3)
    pl = plan_inputs(cfg)
    n = 23
    deg = rng.integers(0, 12, size=n); deg[4] = 90; deg[9] = 0; deg[10] = 1; deg[11] = 33
    rcv = np.repeat(np.arange(n), deg)
    snd = rng.integers(0, n, size=rcv.size)
    o = np.lexsort((snd, rcv))
    snd, rcv = snd[o].astype(np.int32), rcv[o].astype(np.int32)
    e = rcv.size
    g = W.Graph(n, np.zeros((n, 3)), snd, rcv, (rng.normal(size=(e, 3)) * 2).astype(np.float32), 0.0)
    x = rng.normal(size=(n, 16 * C)).astype(np.float32)
    w = rng.normal(size=(e, 34 * C)).astype(np.float32)
    G = rng.normal(size=(n, 156 * C)).astype(np.float32)
    monkeypatch.setenv("E3_TUNE", tune)
    plan = gpu_plan(pl)
    monkeypatch.delenv("E3_TUNE")
    gpu = run_gpu(plan, g, x, w, G)
    compare(gpu, run_oracle(pl, g, x, w, G))
    again = run_gpu(plan, g, x, w, G)
    for k in gpu:
        assert np.array_equal(gpu[k], again[k]), k


# ------------------------------------------------------------------ bf16 storage (reading A12)
def test_bf16_storage_parity_and_fp32_recovers():
    cfg = W.small_config(n_atoms=200, channels=128, irreps_in=((0, 1), (1, -1), (2, 1), (3, -1)), sh_lmax=3, out_lmax=3,
                         box=12.0, storage="bf16", k=105)
    pl, g, x, w, G = make_case(cfg)
    assert g.n_edges > 3000
    plan16 = gpu_plan(pl, "bf16")
    gpu = run_gpu(plan16, g, x, w, G)
    ref = run_oracle(pl, g, x, w, G, storage="bf16")
    errs = compare(gpu, ref, tol_fwd=TOL_BF16, tol_vjp=TOL_BF16, tol_sh=8e-3)
    # same (bf16-representable) values supplied as fp32 storage: error drops to the fp32 level except for
    # the SH, which is then no longer rounded
    plan32 = gpu_plan(pl, "f32")
    e32 = compare(run_gpu(plan32, g, x, w, G), run_oracle(pl, g, x, w, G))
    assert e32["out"] < 1e-5 and e32["dw"] < 1e-4
    print("bf16", errs, "f32", e32)


@pytest.mark.parametrize("C,lmax", [(32, 3), (64, 3), (256, 3), (64, 2)])
def test_bf16_storage_channel_counts(C, lmax):
    """bf16 storage with 4 / 2 edges per warp step, two 128-channel blocks per edge (C = 256: grad_sh accumulates over the
    blocks), and lmax = 2 (odd SH row: the first-generation direct-load kernels)."""
    rng = np.random.default_rng(300 + C + lmax)
    irr = ((0, 1), (1, -1), (2, 1), (3, -1))[: lmax + 1]
    cfg = W.small_config(channels=C, irreps_in=irr, sh_lmax=lmax, out_lmax=lmax, storage="bf16")
    pl = plan_inputs(cfg)
    n = 17
    deg = rng.integers(0, 9, size=n); deg[3] = 41
    rcv = np.repeat(np.arange(n), deg)
    snd = rng.integers(0, n, size=rcv.size)
    o = np.lexsort((snd, rcv))
    snd, rcv = snd[o].astype(np.int32), rcv[o].astype(np.int32)
    e = rcv.size
    in_dim, out_dim = sum(2 * l + 1 for l, _ in irr), sum(2 * l + 1 for l, _, _ in pl[2])
    g = W.Graph(n, np.zeros((n, 3)), snd, rcv, (rng.normal(size=(e, 3)) * 2).astype(np.float32), 0.0)
    x = W.round_to_storage(rng.normal(size=(n, in_dim * C)), "bf16")
    w = W.round_to_storage(rng.normal(size=(e, len(pl[3]) * C)), "bf16")
    G = rng.normal(size=(n, out_dim * C)).astype(np.float32)
    plan = gpu_plan(pl, "bf16")
    compare(run_gpu(plan, g, x, w, G), run_oracle(pl, g, x, w, G, storage="bf16"), tol_fwd=TOL_BF16, tol_vjp=TOL_BF16, tol_sh=8e-3)


# ------------------------------------------------------------------ determinism
def test_run_to_run_bit_identical():
    cfg = W.CONFIGS[1]
    pl, g, x, w, G = make_case(cfg)
    plan = gpu_plan(pl)
    a = run_gpu(plan, g, x, w, G)
    b = run_gpu(plan, g, x, w, G)
    for k in a:
        assert np.array_equal(a[k], b[k]), k


# ------------------------------------------------------------------ host-buffer session == device path
def test_session_host_path_matches_device_path():
    cfg = W.CONFIGS[1]
    pl, g, x, w, G = make_case(cfg)
    plan = gpu_plan(pl)
    dev = run_gpu(plan, g, x, w, G)
    s = B.Session(plan, g.n_edges + 10, g.n_nodes + 3)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out = torch.empty((g.n_nodes, plan.out_dim * plan.channels)).pin_memory()
    dx = torch.empty((g.n_nodes, plan.in_dim * plan.channels)).pin_memory()
    dw = torch.empty((g.n_edges, plan.weights_per_edge)).pin_memory()
    dvec = torch.empty((g.n_edges, 3)).pin_memory()
    F = torch.empty((g.n_nodes, 3)).pin_memory()
    up, down = s.run_host(pin(g.vec), pin(x), pin(w), pin(g.senders), pin(g.receivers), g.n_nodes, pin(G), out, dx, dw, dvec, F)
    assert up == g.vec.nbytes + x.nbytes + w.nbytes + 2 * g.senders.nbytes + G.nbytes
    assert down == sum(t.numel() * 4 for t in (out, dx, dw, dvec, F))
    for name, t in (("out", out), ("dx", dx), ("dw", dw), ("dvec", dvec), ("F", F)):
        assert np.array_equal(t.numpy(), dev[name]), name


def test_session_pipelined_chunks_match_device_path():
    """154 MB of weights => the host path runs in 4 receiver-range chunks on three streams; every result must be
    bit-identical to the unchunked device entry points (and hence within the oracle bars checked elsewhere)."""
    cfg = W.small_config(n_atoms=1536, channels=32, irreps_in=((0, 1), (1, -1), (2, 1)), sh_lmax=2, out_lmax=2,
                         box=24.8579, k=107)
    pl, g, x, w, G = make_case(cfg)
    assert w.nbytes > 3 * (48 << 20)
    plan = gpu_plan(pl)
    dev = run_gpu(plan, g, x, w, G)
    s = B.Session(plan, g.n_edges, g.n_nodes)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out = torch.empty((g.n_nodes, plan.out_dim * plan.channels)).pin_memory()
    dx = torch.empty((g.n_nodes, plan.in_dim * plan.channels)).pin_memory()
    dw = torch.empty((g.n_edges, plan.weights_per_edge)).pin_memory()
    dvec = torch.empty((g.n_edges, 3)).pin_memory()
    F = torch.empty((g.n_nodes, 3)).pin_memory()
    for _ in range(2):
        up, down = s.run_host(pin(g.vec), pin(x), pin(w), pin(g.senders), pin(g.receivers), g.n_nodes, pin(G), out, dx, dw, dvec, F)
        assert up == g.vec.nbytes + x.nbytes + w.nbytes + 2 * g.senders.nbytes + G.nbytes
        for name, t in (("out", out), ("dx", dx), ("dw", dw), ("dvec", dvec), ("F", F)):
            assert np.array_equal(t.numpy(), dev[name]), name
    # forward only (no cotangent), and a VJP whose grad_weights are not requested: fewer copies, same numbers
    out.zero_()
    up, down = s.run_host(pin(g.vec), pin(x), pin(w), pin(g.senders), pin(g.receivers), g.n_nodes, None, out)
    assert down == out.numel() * 4 and np.array_equal(out.numpy(), dev["out"])
    dx.zero_(); F.zero_()
    up, down = s.run_host(pin(g.vec), pin(x), pin(w), pin(g.senders), pin(g.receivers), g.n_nodes, pin(G), None, dx, None, None, F)
    assert down == (dx.numel() + F.numel()) * 4
    assert np.array_equal(dx.numpy(), dev["dx"]) and np.array_equal(F.numpy(), dev["F"])


def test_fp32_peak_measurement_aid():
    """e3_measure_fp32_peak (bench.py's `alu_peak.measured_sustained_tflops`): a sane fraction of 148 x 128 x 2 x 1.965 GHz."""
    t = B.e3_measure_fp32_peak(30.0)
    assert 0.4 * 74.45 < t < 1.05 * 74.45, t
