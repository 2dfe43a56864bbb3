"""Pins for the NEXT-4 oracle functions: neighbour list (reading N1) and receiver-range sharding (reading N2).
PAPER.md L66 (Graph: edge vectors from positions and connectivity), L82 (larger systems), L298 / L497 (5 A cutoff)."""
from __future__ import annotations

import numpy as np
import pytest
from scipy.spatial import cKDTree

import oracle as O
from paper_2605_22698_b200 import workloads as W


def _kdtree_edges(pos, box, rc):
    """Library routine on the same float32 positions (distances in fp64): directed pairs sorted by (receiver, sender)."""
    p = np.asarray(pos, np.float64)
    if all(b > 0 for b in box):
        assert box[0] == box[1] == box[2]
        t = cKDTree(np.mod(p, float(box[0])), boxsize=float(box[0]))
    else:
        assert not any(b > 0 for b in box)
        t = cKDTree(p)
    pr = t.query_pairs(rc, output_type="ndarray")
    s = np.concatenate([pr[:, 0], pr[:, 1]]); r = np.concatenate([pr[:, 1], pr[:, 0]])
    o = np.lexsort((s, r))
    return s[o], r[o]


def _true_d(pos, s, r, box):
    d = np.asarray(pos, np.float64)[r] - np.asarray(pos, np.float64)[s]
    for a in range(3):
        if box[a] > 0:
            d[:, a] -= float(box[a]) * np.round(d[:, a] / float(box[a]))
    return d


@pytest.mark.parametrize("n,box,seed", [(300, 14.0, 0), (500, 0.0, 1), (64, 10.0, 2)])
def test_neighbor_oracle_matches_kdtree_away_from_the_cutoff(n, box, seed):
    rng = np.random.default_rng(seed)
    pos = (rng.uniform(0, box, size=(n, 3)) if box > 0 else rng.normal(0, 4.0, size=(n, 3))).astype(np.float32)
    bx = (box, box, box)
    s, r, vec, row_ptr = O.neighbor_build(pos, bx, 5.0)
    ks, kr = _kdtree_edges(pos, bx, 5.0)
    a = set(zip(s.tolist(), r.tolist())); b = set(zip(ks.tolist(), kr.tolist()))
    for (ss, rr) in a ^ b:                                   # any disagreement must be a pair at the cutoff to fp32 rounding
        d = np.linalg.norm(_true_d(pos, np.array([ss]), np.array([rr]), bx))
        assert abs(d - 5.0) < 1e-5
    assert len(a ^ b) <= 1 and len(a) > 10 * n // 3
    assert np.abs(vec - _true_d(pos, s, r, bx)).max() < 5e-6
    assert np.all(np.diff(r) >= 0) and np.all((np.diff(s) > 0) | (np.diff(r) > 0))      # (receiver, sender) strictly ascending
    assert not np.any(s == r)
    assert np.array_equal(row_ptr, np.searchsorted(r, np.arange(n + 1), "left"))
    pick = np.array([0, 7, n // 2, n - 1])                    # the sampled form returns exactly those receivers' rows
    s1, r1, v1, _ = O.neighbor_build(pos, bx, 5.0, only_receivers=pick)
    m = np.isin(r, pick)
    assert np.array_equal(s1, s[m]) and np.array_equal(r1, r[m]) and np.array_equal(v1, vec[m])


def test_neighbor_oracle_simple_cubic_coordination_numbers():
    a, m = 2.0, 6                                            # 6^3 sites, box 12 = 2.4 * cutoff
    g = np.arange(m, dtype=np.float32) * a
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    for rc, z in ((2.5, 6), (3.0, 18), (3.6, 26), (4.1, 32)):                     # shells at a, a*sqrt2, a*sqrt3, 2a: 6, 12, 8, 6
        s, r, vec, row_ptr = O.neighbor_build(pos, (a * m,) * 3, rc) if a * m >= 2 * rc else (None,) * 4
        assert np.all(np.diff(row_ptr) == z)
        assert np.allclose(np.sort(np.unique(np.round(np.linalg.norm(vec, axis=1), 4)))[0], a)
    with pytest.raises(ValueError):
        O.neighbor_build(pos, (a * m,) * 3, 6.5)              # box < 2 * cutoff: a sender would have two images in range


def test_neighbor_oracle_pair_symmetry_and_python_brute_force():
    rng = np.random.default_rng(3)
    pos = rng.normal(0, 2.5, size=(40, 3)).astype(np.float32)
    s, r, vec, _ = O.neighbor_build(pos, (0, 0, 0), 5.0)
    idx = {(int(a), int(b)): k for k, (a, b) in enumerate(zip(s, r))}
    for (a, b), k in idx.items():
        assert (b, a) in idx and np.array_equal(vec[idx[(b, a)]], -vec[k])
    want = []
    for rr in range(40):
        for ss in range(40):
            if ss != rr and float(np.sum((pos[rr].astype(np.float64) - pos[ss]) ** 2)) < 25.0 - 1e-4:
                want.append((ss, rr))
    assert set(want) <= set(idx) and len(idx) - len(want) <= 1
    # mixed periodicity: periodic along x only
    s2, r2, vec2, _ = O.neighbor_build(pos, (12.0, 0, 0), 5.0)
    d = pos[r2] - pos[s2]
    d[:, 0] -= 12.0 * np.round(d[:, 0] / 12.0)
    assert np.abs(vec2 - d).max() < 1e-5 and len(s2) >= len(s)


def test_neighbor_oracle_reproduces_the_harness_graph_of_config_1():
    g, _ = W.make_graph(W.CONFIGS[1])                       # fp64 harness build (cKDTree), reading A11
    s, r, vec, _ = O.neighbor_build(g.pos.astype(np.float32), (g.box,) * 3, W.CUTOFF)
    assert np.array_equal(s, g.senders) and np.array_equal(r, g.receivers)
    assert np.abs(vec - g.vec).max() < 5e-6


# ------------------------------------------------------------------ N2: receiver-range sharding
def test_shard_ranges_cover_and_balance():
    g, _ = W.make_graph(W.CONFIGS[2])
    for world in (1, 2, 3, 8):
        b = O.shard_ranges(g.receivers, g.n_nodes, world)
        assert b[0] == 0 and b[-1] == g.n_nodes and all(x <= y for x, y in zip(b, b[1:]))
        cnt = [np.count_nonzero((g.receivers >= lo) & (g.receivers < hi)) for lo, hi in zip(b, b[1:])]
        assert sum(cnt) == g.n_edges and max(cnt) - min(cnt) <= 2 * 90          # within two receivers' worth of edges
    assert O.shard_ranges(np.zeros(0, np.int32), 5, 3) == [0, 5, 5, 5]


def test_shard_local_graphs_reassemble_the_global_problem():
    """Running the oracle on every rank's local graph (owned + halo rows) and adding the halo gradients back to their owners
    equals the oracle on the whole graph: the sharding needs one exchange each way and nothing else."""
    cfg = W.small_config(n_atoms=60, channels=4, irreps_in=((0, 1), (1, -1)), sh_lmax=2, out_lmax=2, box=11.0, k=7)
    g, rng = W.make_graph(cfg)
    irreps_in = [(l, p, cfg.channels) for l, p in cfg.irreps_in]
    irreps_out, paths = O.all_paths(irreps_in, 2, 2)
    pl = (irreps_in, 2, irreps_out, paths)
    od = sum(2 * l + 1 for l, _, _ in irreps_out)
    x = rng.normal(size=(60, 4 * 4)); w = rng.normal(size=(g.n_edges, len(paths) * 4)); G = rng.normal(size=(60, od * 4))
    Y = O.sh(2, g.vec.astype(np.float64))
    out = O.tp_scatter_fwd(*pl, x, Y, w, g.senders, g.receivers, 60)
    dx, dY, dw = O.tp_scatter_bwd(*pl, x, Y, w, g.senders, g.receivers, 60, G)
    world = 3
    out_s, dx_s, dY_s, dw_s = np.zeros_like(out), np.zeros_like(dx), np.zeros_like(dY), np.zeros_like(dw)
    seen = np.zeros(g.n_edges, int)
    for rank in range(world):
        L = O.shard_local_graph(g.senders, g.receivers, 60, world, rank)
        own = np.arange(L["lo"], L["hi"])
        ids = np.concatenate([own, L["halo"]])                                   # local -> global node ids
        assert len(np.unique(ids)) == len(ids) and np.array_equal(ids[L["senders_local"]], g.senders[L["e_lo"]:L["e_hi"]])
        n_loc = len(ids)
        Gl = np.zeros((n_loc, G.shape[1])); Gl[:len(own)] = G[own]
        e = slice(L["e_lo"], L["e_hi"])
        seen[e] += 1
        o = O.tp_scatter_fwd(*pl, x[ids], Y[e], w[e], L["senders_local"], L["receivers_local"], n_loc)
        a, b_, c = O.tp_scatter_bwd(*pl, x[ids], Y[e], w[e], L["senders_local"], L["receivers_local"], n_loc, Gl)
        assert np.all(o[len(own):] == 0)                                          # halo atoms receive nothing locally
        out_s[own] = o[:len(own)]
        np.add.at(dx_s, ids, a)                                                  # reverse halo: gradients return to their owners
        dY_s[e] = b_; dw_s[e] = c
    assert np.all(seen == 1)
    for p, q in ((out_s, out), (dx_s, dx), (dY_s, dY), (dw_s, dw)):
        assert np.abs(p - q).max() < 1e-12
