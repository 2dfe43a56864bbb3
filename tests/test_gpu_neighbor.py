"""NEXT-4: the device neighbour list against the brute-force oracle (reading N1).
Everything is integer or a float32 value with one defined rounding sequence, so the comparison is bit-exact."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import oracle as O
from helpers import TOL_FWD, TOL_VJP, compare, gpu_plan, make_case, relerr, run_gpu, run_oracle, to_dev
from paper_2605_22698_b200 import binding as B
from paper_2605_22698_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _gpu(pos, box, rc, **kw):
    s, r, v, rp = B.e3_neighbor_build(to_dev(np.ascontiguousarray(pos, np.float32)), box, rc, **kw)
    torch.cuda.synchronize()
    return s.cpu().numpy(), r.cpu().numpy(), v.cpu().numpy(), rp.cpu().numpy()


def _same(pos, box, rc):
    got = _gpu(pos, box, rc)
    ref = O.neighbor_build(pos, box, rc)
    assert len(got[0]) == len(ref[0]), (len(got[0]), len(ref[0]))
    for g, q, name in zip(got, ref, ("senders", "receivers", "vec", "row_ptr")):
        assert np.array_equal(g, q), name                      # bit-exact, vec included
    return len(ref[0])


@pytest.mark.parametrize("k", [1, 2])
def test_neighbor_build_reproduces_the_benchmark_graphs(k):
    g, _ = W.make_graph(W.CONFIGS[k])
    pos = g.pos.astype(np.float32)
    E = _same(pos, (g.box,) * 3, W.CUTOFF)
    assert abs(E - g.n_edges) <= 2                               # the fp64 harness graph differs only at the cutoff, if at all
    s, r, v, rp = _gpu(pos, (g.box,) * 3, W.CUTOFF)
    if E == g.n_edges:
        assert np.array_equal(s, g.senders) and np.array_equal(r, g.receivers) and np.abs(v - g.vec).max() < 5e-6
    # the list is what the rest of the path expects: e3_graph_prepare on it returns the same row_ptr
    row_ptr, _, _ = B.e3_graph_prepare(to_dev(s), to_dev(r), g.n_nodes, validate=True)
    assert np.array_equal(row_ptr.cpu().numpy(), rp)


def test_neighbor_build_open_mixed_and_wrapped_geometries():
    rng = np.random.default_rng(0)
    _same(rng.normal(0, 8.0, size=(2000, 3)).astype(np.float32), (0, 0, 0), 5.0)                 # open cluster
    _same(rng.normal(0, 1.5, size=(300, 3)).astype(np.float32), (0, 0, 0), 5.0)                  # dense blob: degree ~ N (one or two cells)
    slab = np.stack([rng.uniform(0, 30, 1500), rng.uniform(0, 22, 1500), rng.normal(0, 3.0, 1500)], 1).astype(np.float32)
    _same(slab, (30.0, 22.0, 0.0), 5.0)                                                          # periodic in x, y only
    p = rng.uniform(-40, 55, size=(1200, 3)).astype(np.float32)
    _same(p, (17.0, 13.5, 10.0), 5.0)                                                            # atoms outside the box; 2-3 cells per axis
    _same(rng.uniform(0, 1, size=(50, 3)).astype(np.float32) * np.float32(400.0), (0, 0, 0), 5.0)   # sparse: almost no edges
    a = np.arange(8, dtype=np.float32) * 2.5
    lat = np.stack(np.meshgrid(a, a, a, indexing="ij"), -1).reshape(-1, 3)                       # lattice: many pairs EXACTLY at the cutoff (2 x 2.5)
    E = _same(lat, (20.0, 20.0, 20.0), 5.0)
    assert E == 512 * (6 + 12 + 8)                                                                # shells at 2.5, 3.54, 4.33; the 5.0 shell is excluded (strict)


def test_neighbor_build_edge_cases_and_errors():
    z = torch.zeros((0, 3), device="cuda")
    s, r, v, rp = B.e3_neighbor_build(z, (10, 10, 10), 5.0)
    assert s.numel() == 0 and rp.cpu().tolist() == [0]
    s, r, v, rp = _gpu(np.zeros((1, 3), np.float32), (0, 0, 0), 5.0)
    assert len(s) == 0 and rp.tolist() == [0, 0]
    two = np.array([[0, 0, 0], [0, 0, 0]], np.float32)                                          # coincident atoms: zero-length edges are kept
    s, r, v, rp = _gpu(two, (0, 0, 0), 5.0)
    assert s.tolist() == [1, 0] and r.tolist() == [0, 1] and not v.any()
    with pytest.raises(B.E3Error) as e:
        B.e3_neighbor_build(to_dev(two), (9.0, 20, 20), 5.0)
    assert e.value.status == B.E3_ERR_UNSUPPORTED
    rng = np.random.default_rng(1)
    pos = to_dev(rng.uniform(0, 12, size=(400, 3)).astype(np.float32))
    with pytest.raises(B.E3Error) as e:
        B.e3_neighbor_build(pos, (12, 12, 12), 5.0, max_edges=10)
    assert e.value.status == B.E3_ERR_WORKSPACE
    a = B.e3_neighbor_build(pos, (12, 12, 12), 5.0)              # capacity guess 64 per atom is too small here: second call inside
    b = B.e3_neighbor_build(pos, (12, 12, 12), 5.0)
    assert a[0].numel() > 64 * 400 and all(torch.equal(x, y) for x, y in zip(a, b))


def test_neighbor_build_full_size_sampled_rows():
    g, _ = W.make_graph(W.CONFIGS[4])                                                            # 100 000 atoms
    pos = g.pos.astype(np.float32)
    s, r, v, rp = _gpu(pos, (g.box,) * 3, W.CUTOFF)
    assert abs(len(s) - g.n_edges) <= 4 and rp[-1] == len(s)
    assert np.all(np.diff(r.astype(np.int64) * g.n_nodes + s) > 0)                               # strictly ascending (receiver, sender)
    pick = np.sort(np.random.default_rng(4).choice(g.n_nodes, 256, replace=False))
    so, ro, vo, _ = O.neighbor_build(pos, (g.box,) * 3, W.CUTOFF, only_receivers=pick)
    m = np.isin(r, pick)
    assert np.array_equal(s[m], so) and np.array_equal(r[m], ro) and np.array_equal(v[m], vo)
    key = r.astype(np.int64) * g.n_nodes + s                                                     # every edge has its reverse
    assert np.array_equal(np.sort(s.astype(np.int64) * g.n_nodes + r), key)


def test_whole_path_on_a_device_built_graph():
    """positions -> e3_neighbor_build -> SH -> TP fwd/VJP -> forces, against the oracle run on the ORACLE's own neighbour list."""
    cfg = W.CONFIGS[1]
    pl, g, x, w, G = make_case(cfg)
    pos = g.pos.astype(np.float32)
    s, r, v, rp = B.e3_neighbor_build(to_dev(pos), (g.box,) * 3, W.CUTOFF)
    so, ro, vo, _ = O.neighbor_build(pos, (g.box,) * 3, W.CUTOFF)
    assert len(so) == g.n_edges                                   # same count as the harness graph, so w (drawn per edge) fits
    g_gpu = W.Graph(g.n_nodes, g.pos, s.cpu().numpy(), r.cpu().numpy(), v.cpu().numpy(), g.box)
    g_orc = W.Graph(g.n_nodes, g.pos, so, ro, vo, g.box)
    compare(run_gpu(gpu_plan(pl), g_gpu, x, w, G), run_oracle(pl, g_orc, x, w, G))


# ------------------------------------------------------------------ SURVEY 8(e) / reading N2: receiver-range shards on the GPU
def test_shard_local_problems_on_the_gpu_reassemble_the_whole_graph():
    """The three shards of config 2 run ONE AFTER THE OTHER on this GPU (each is an ordinary local call on owned + halo rows, as
    planned by e3_shard_*); halo gradients are added back to their owners in rank order.  Equals the oracle on the whole graph."""
    cfg = W.CONFIGS[2]
    pl, g, x, w, G = make_case(cfg)
    plan = gpu_plan(pl)
    ref = run_oracle(pl, g, x, w, G, want_forces=False)
    sh_all = B.e3_sh_fwd(plan, to_dev(g.vec))
    world = 3
    b = B.e3_shard_ranges(g.receivers, g.n_nodes, world)
    out = np.zeros_like(ref["out"], dtype=np.float32); dx = np.zeros_like(ref["dx"], dtype=np.float32)
    dY = np.zeros_like(ref["dY"], dtype=np.float32); dw = np.zeros_like(ref["dw"], dtype=np.float32)
    for k in range(world):
        L = B.e3_shard_localize(g.senders, g.receivers, g.n_nodes, b[k], b[k + 1])
        ids = np.concatenate([np.arange(L["lo"], L["hi"]), L["halo"]])
        n_loc, n_own = len(ids), L["hi"] - L["lo"]
        assert len(L["halo"]) > 0
        e = slice(L["e_lo"], L["e_hi"])
        sd, rd = to_dev(L["senders_local"]), to_dev(L["receivers_local"])
        row_ptr, perm_s, col_ptr = B.e3_graph_prepare(sd, rd, n_loc, validate=True)
        xl, wl, shl = to_dev(x[ids]), to_dev(w[e]), sh_all[e].contiguous()
        Gl = np.zeros((n_loc, G.shape[1]), np.float32); Gl[:n_own] = G[L["lo"]:L["hi"]]
        o = B.e3_tp_scatter_fwd(plan, xl, shl, wl, sd, rd, row_ptr, n_loc)
        a, b_, c = B.e3_tp_scatter_bwd(plan, xl, shl, wl, sd, rd, row_ptr, perm_s, col_ptr, n_loc, to_dev(Gl))
        torch.cuda.synchronize()
        assert not o[n_own:].any()                                         # halo atoms receive nothing locally
        out[L["lo"]:L["hi"]] = o[:n_own].cpu().numpy()
        np.add.at(dx, ids, a.cpu().numpy())                                # reverse halo, rank order
        dY[e] = b_.cpu().numpy(); dw[e] = c.cpu().numpy()
    assert relerr(out, ref["out"]) <= TOL_FWD
    assert relerr(dx, ref["dx"]) <= TOL_VJP and relerr(dY, ref["dY"]) <= TOL_VJP and relerr(dw, ref["dw"]) <= TOL_VJP


def test_sharded_tp_single_rank_nccl():
    """ShardedTP's default (CUDA) local calls under a real NCCL process group of one rank: no halo, equals the plain calls bit for bit."""
    import os
    import torch.distributed as dist
    from paper_2605_22698_b200.sharded import ShardedTP
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(32500 + os.getpid() % 2000), RANK="0", WORLD_SIZE="1")
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        cfg = W.CONFIGS[1]
        pl, g, x, w, G = make_case(cfg)
        plan = gpu_plan(pl)
        st = ShardedTP(plan, g.senders, g.receivers, g.n_nodes, "cuda")
        assert (st.lo, st.hi, st.e_lo, st.e_hi, len(st.halo)) == (0, g.n_nodes, 0, g.n_edges, 0)
        sh = B.e3_sh_fwd(plan, to_dev(g.vec))
        xd, wd, Gd = to_dev(x), to_dev(w), to_dev(G)
        out = st.fwd(xd, sh, wd)
        dx, dY, dw = st.bwd(xd, sh, wd, Gd)
        ref = run_gpu(plan, g, x, w, G, want_forces=False)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), ref["out"]) and np.array_equal(dx.cpu().numpy(), ref["dx"])
        assert np.array_equal(dY.cpu().numpy(), ref["dY"]) and np.array_equal(dw.cpu().numpy(), ref["dw"])
    finally:
        dist.destroy_process_group()
