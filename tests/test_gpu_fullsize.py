"""GPU parity at BASELINE.json's full sizes (configs 4 and 5: 100 000 atoms, ~5.2 M edges), in the launch
configuration bench.py times.  The fp64 oracle cannot run 5.2 M edges x 34 paths in seconds, so outputs
are checked on seeded samples the oracle computes one by one:
  forward   : every output row of 48 sampled receivers (all their in-edges),
  grad_feats: every row of 48 sampled senders (all their out-edges),
  grad_sh / grad_weights / grad_vec: 2048 sampled edges,
plus properties that hold at any size: indices bit-exact against numpy, sum of forces = 0, Euler
identity <G, out> = <grad_weights, w> = <grad_feats, x>, every row written.
The weights (45.6 GB) are drawn on the device (workloads.draw_w_device); the oracle is fed rows copied
back from that very tensor, never anything computed by the CUDA path."""
import numpy as np
import pytest
import torch

import oracle as O
from helpers import TOL_BF16, TOL_FWD, TOL_VJP, plan_inputs, relerr
from paper_2605_22698_b200 import binding as B
from paper_2605_22698_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _compact(ids):
    uniq, inv = np.unique(ids, return_inverse=True)
    return uniq, inv.astype(np.int32)


@pytest.mark.parametrize("k", [4, 5])
def test_full_size_sampled_parity(k):
    import gc
    cfg = W.CONFIGS[k]
    gc.collect()
    torch.cuda.empty_cache()
    free, total = torch.cuda.mem_get_info()
    if total < 160e9:
        pytest.skip("needs a 180 GB device (B200); this one is smaller")
    # on a B200 a fragmented or occupied device must FAIL here, not silently turn cfg4/5 parity into "untested"
    assert free >= 150e9, f"only {free / 1e9:.0f} GB of {total / 1e9:.0f} GB free on a B200-class device: cannot run the full-size parity case"
    dev = torch.device("cuda")
    pl = plan_inputs(cfg)
    plan = B.e3_plan_create(pl[0], pl[1], pl[2], pl[3], B.E3_BF16 if cfg.storage == "bf16" else B.E3_F32)
    P, C, st = plan.n_paths, plan.channels, plan.storage
    tol_f, tol_v = (TOL_BF16, TOL_BF16) if cfg.storage == "bf16" else (TOL_FWD, TOL_VJP)
    g, rng = W.make_graph(cfg)
    E, N = g.n_edges, g.n_nodes
    x_h = W.draw_x(cfg, rng)
    G_h = W.draw_g(cfg, rng, plan.out_dim)
    w = W.draw_w_device(cfg, E, P, dev)
    x = torch.from_numpy(x_h).to(dev).to(st)
    G = torch.from_numpy(G_h).to(dev)
    snd, rcv, vec = (torch.from_numpy(a).to(dev) for a in (g.senders, g.receivers, g.vec))

    row_ptr, perm_s, col_ptr = B.e3_graph_prepare(snd, rcv, N, validate=True)
    assert np.array_equal(row_ptr.cpu().numpy(), np.concatenate([[0], np.cumsum(np.bincount(g.receivers, minlength=N))]))
    assert np.array_equal(col_ptr.cpu().numpy(), np.concatenate([[0], np.cumsum(np.bincount(g.senders, minlength=N))]))
    perm_ref = np.argsort(g.senders, kind="stable").astype(np.int32)
    assert np.array_equal(perm_s.cpu().numpy(), perm_ref)

    sh = B.e3_sh_fwd(plan, vec)
    out = torch.full((N, plan.out_dim * C), float("nan"), device=dev)
    B.e3_tp_scatter_fwd(plan, x, sh, w, snd, rcv, row_ptr, N, out=out)
    dx, dY, dw = B.e3_tp_scatter_bwd(plan, x, sh, w, snd, rcv, row_ptr, perm_s, col_ptr, N, G)
    dvec = B.e3_sh_bwd(plan, vec, dY)
    F = B.e3_force_reduce(dvec, row_ptr, perm_s, col_ptr, N)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all()) and bool(torch.isfinite(dx).all())

    # ---- properties at full size -------------------------------------------------------------
    s_out = float((G.double() * out.double()).sum())
    s_dx = float((dx.double() * x.double()).sum())
    s_dw = 0.0
    for a in range(0, E, 1 << 18):                                   # chunked fp64 reduction of 11 G elements
        s_dw += float((dw[a:a + (1 << 18)].double() * w[a:a + (1 << 18)].double()).sum())
    scale = float((G.double().abs() * out.double().abs()).sum())
    bar = 50 * (2e-3 if cfg.storage == "bf16" else 1e-6)
    assert abs(s_out - s_dx) <= bar * scale and abs(s_out - s_dw) <= bar * scale, (s_out, s_dx, s_dw, scale)
    assert float(F.double().sum(0).abs().max()) <= 1e-4 * float(F.abs().max()) * np.sqrt(N)

    # ---- oracle's own SH of the stored edge vectors, rounded once to the storage dtype --------
    srng = np.random.default_rng(1234 + k)
    vec64 = g.vec.astype(np.float64)

    def oracle_sh(eidx):
        Y = O.sh(cfg.sh_lmax, vec64[eidx])
        return W.round_to_storage(Y, cfg.storage).astype(np.float64) if cfg.storage == "bf16" else Y

    def rows(t, idx):
        return t[torch.from_numpy(np.asarray(idx)).to(dev)].float().cpu().numpy().astype(np.float64)

    # forward: sampled receivers
    rs = np.sort(srng.choice(N, size=48, replace=False))
    rp = np.concatenate([[0], np.cumsum(np.bincount(g.receivers, minlength=N))])
    eidx = np.concatenate([np.arange(rp[r], rp[r + 1]) for r in rs])
    us, s_loc = _compact(g.senders[eidx])
    _, r_loc = _compact(g.receivers[eidx])
    n_loc = max(len(us), len(rs))                      # one local index space for x rows and out rows
    xs_ = np.pad(x_h[us].astype(np.float64), ((0, n_loc - len(us)), (0, 0)))
    ref = O.tp_scatter_fwd(*pl, xs_, oracle_sh(eidx), rows(w, eidx), s_loc, r_loc, n_loc)
    e_out = relerr(rows(out, rs), ref[:len(rs)])
    # grad_feats: sampled senders with all their out-edges
    ss = np.sort(srng.choice(N, size=48, replace=False))
    cp = np.concatenate([[0], np.cumsum(np.bincount(g.senders, minlength=N))])
    eidx = np.sort(np.concatenate([perm_ref[cp[s]:cp[s + 1]] for s in ss]))
    s_loc = np.searchsorted(ss, g.senders[eidx]).astype(np.int32)
    ur, r_loc = _compact(g.receivers[eidx])
    n_loc = max(len(ss), len(ur))                      # one local index space for x rows and G rows
    xs_ = np.pad(x_h[ss].astype(np.float64), ((0, n_loc - len(ss)), (0, 0)))
    gs_ = np.pad(G_h[ur].astype(np.float64), ((0, n_loc - len(ur)), (0, 0)))
    rdx, _, _ = O.tp_scatter_bwd(*pl, xs_, oracle_sh(eidx), rows(w, eidx), s_loc, r_loc, n_loc, gs_)
    e_dx = relerr(rows(dx, ss), rdx[:len(ss)])
    # per-edge gradients: sampled edges
    es = np.sort(srng.choice(E, size=2048, replace=False))
    us, s_loc = _compact(g.senders[es])
    ur, r_loc = _compact(g.receivers[es])
    n_loc = max(len(us), len(ur))
    xs_ = np.pad(x_h[us].astype(np.float64), ((0, n_loc - len(us)), (0, 0)))
    gs_ = np.pad(G_h[ur].astype(np.float64), ((0, n_loc - len(ur)), (0, 0)))
    _, rdY, rdw = O.tp_scatter_bwd(*pl, xs_, oracle_sh(es), rows(w, es), s_loc, r_loc, n_loc, gs_)
    e_dY, e_dw = relerr(rows(dY, es), rdY), relerr(rows(dw, es), rdw)
    e_dv = relerr(rows(dvec, es), O.sh_bwd(cfg.sh_lmax, vec64[es], rdY))
    errs = dict(out=e_out, dx=e_dx, dY=e_dY, dw=e_dw, dvec=e_dv)
    # forces: every row of 48 sampled atoms, from the oracle's grad_vec of ALL their in- and out-edges
    if cfg.forces:
        fa = np.sort(srng.choice(N, size=48, replace=False))
        ein = np.concatenate([np.arange(rp[i], rp[i + 1]) for i in fa])
        eout = np.concatenate([perm_ref[cp[i]:cp[i + 1]] for i in fa])
        ef = np.unique(np.concatenate([ein, eout]))
        us, s_loc = _compact(g.senders[ef])
        ur, r_loc = _compact(g.receivers[ef])
        n_loc = max(len(us), len(ur))
        xs_ = np.pad(x_h[us].astype(np.float64), ((0, n_loc - len(us)), (0, 0)))
        gs_ = np.pad(G_h[ur].astype(np.float64), ((0, n_loc - len(ur)), (0, 0)))
        _, fdY, _ = O.tp_scatter_bwd(*pl, xs_, oracle_sh(ef), rows(w, ef), s_loc, r_loc, n_loc, gs_)
        fdv = O.sh_bwd(cfg.sh_lmax, vec64[ef], fdY)
        Fref = np.zeros((48, 3))
        for a_i, atom in enumerate(fa):                    # reading A10 / a7: F_i = -(sum over in-edges - sum over out-edges)
            Fref[a_i] = -(fdv[g.receivers[ef] == atom].sum(0) - fdv[g.senders[ef] == atom].sum(0))
        den = float(F.abs().max())
        errs["F"] = float(np.abs(rows(F, fa) - Fref).max() / den)
        assert errs["F"] <= tol_v, errs
    print(cfg.name, "E", E, {k_: f"{v:.2e}" for k_, v in errs.items()})
    assert e_out <= tol_f, errs
    assert e_dx <= tol_v and e_dY <= tol_v and e_dw <= tol_v and e_dv <= tol_v, errs


def test_full_size_radial_network_sampled_edges():
    """NEXT-1 at config 4's size (5.2 M edges x 2176 generated weights = 45.6 GB, the grid / tile split bench.py times): the generated
    weight rows and the radial force terms of 1024 sampled edges (plus the first and last tiles) against the oracle, row by row;
    every other row finite and, beyond the cutoff, exactly zero."""
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, total = torch.cuda.mem_get_info()
    if total < 160e9:
        pytest.skip("needs a 180 GB device (B200); this one is smaller")
    assert free >= 110e9, f"only {free / 1e9:.0f} GB free on a B200-class device"
    cfg = W.CONFIGS[4]
    g, _ = W.make_graph(cfg)
    E, n_out, K = g.n_edges, 34 * cfg.channels, 16
    rng = np.random.default_rng(41)
    f32 = lambda a: a.astype(np.float32)
    W1, W2, W3 = f32(rng.normal(size=(K, 64)) / 4.0), f32(rng.normal(size=(64, 64)) / 8.0), f32(rng.normal(size=(64, n_out)) / 8.0)
    net = B.Radial(K, 6, W.CUTOFF, W1, W2, W3)
    vec = torch.from_numpy(g.vec).cuda()
    w = torch.full((E, n_out), float("nan"), device="cuda")
    B.e3_radial_weights_fwd(net, vec, out=w)
    pick = np.unique(np.concatenate([np.arange(0, 130), np.arange(E - 130, E), rng.choice(E, 1024, replace=False)]))
    ref = O.radial_weights(g.vec[pick], K, 6, W.CUTOFF, W1, W2, W3)
    got = w[torch.from_numpy(pick).cuda()].cpu().numpy()
    assert relerr(got, ref) <= TOL_FWD, relerr(got, ref)
    assert bool(torch.isfinite(w).all())
    # VJP: a seeded cotangent drawn on the device; the oracle is fed the rows copied back
    gen = torch.Generator(device="cuda"); gen.manual_seed(7)
    dw = torch.randn((E, n_out), generator=gen, device="cuda")
    gv = B.e3_radial_weights_bwd(net, vec, dw)
    gref = O.radial_weights_bwd(g.vec[pick], K, 6, W.CUTOFF, W1, W2, W3, dw[torch.from_numpy(pick).cuda()].cpu().numpy())[0]
    assert relerr(gv[torch.from_numpy(pick).cuda()].cpu().numpy(), gref) <= TOL_VJP
    assert bool(torch.isfinite(gv).all())
    gv2 = B.e3_radial_weights_bwd(net, vec, dw)
    assert torch.equal(gv, gv2)                                   # run-to-run bit-identical
    net.destroy()
    del w, dw
    torch.cuda.empty_cache()
