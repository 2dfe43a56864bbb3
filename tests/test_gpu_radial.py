"""NEXT-1 on the GPU: the radial network generating the weights (e3_radial_*; tcgen05 3xTF32 GEMM for the last layer) against the
fp64 oracle (oracle/e3_oracle_next.c, readings R1-R4), alone and through the whole hot path (generated weights -> tensor product
-> VJP -> forces including the radial term)."""
import numpy as np
import pytest
import torch

import oracle as O
from helpers import TOL_FWD, TOL_VJP, gpu_plan, make_case, plan_inputs, relerr, to_dev
from paper_2605_22698_b200 import binding as B
from paper_2605_22698_b200 import workloads as W

pytestmark = pytest.mark.gpu
RC = 5.0


def _net(rng, K, n_out, H=64):
    f32 = lambda a: a.astype(np.float32)
    return f32(rng.normal(size=(K, H)) / np.sqrt(K)), f32(rng.normal(size=(H, H)) / np.sqrt(H)), f32(rng.normal(size=(H, n_out)) / np.sqrt(H))


@pytest.mark.parametrize("K,n_out,E", [(8, 64, 1), (8, 480, 2134), (16, 1664, 5000), (16, 2176, 777), (3, 8, 129), (16, 200, 1000)])
def test_radial_weights_and_vjp_against_oracle(K, n_out, E):
    rng = np.random.default_rng(K * 1000 + n_out)
    vec = (rng.normal(size=(E, 3)) * 2.2).astype(np.float32)
    vec[0] = [0.02, -0.01, 0.02]                       # a very short edge (reading A18)
    if E > 4:
        vec[1] = 0.0                                   # zero-length edge: finite weights, zero radial force
        vec[2] = [4.0, 3.0, 0.5]                       # beyond the cutoff: weights exactly zero
        vec[3] = [RC - 1e-4, 0.0, 0.0]                 # just inside
    W1, W2, W3 = _net(rng, K, n_out)
    net = B.Radial(K, 6, RC, W1, W2, W3)
    w = B.e3_radial_weights_fwd(net, to_dev(vec))
    ref = O.radial_weights(vec, K, 6, RC, W1, W2, W3)
    torch.cuda.synchronize()
    got = w.cpu().numpy()
    assert relerr(got, ref) <= TOL_FWD, relerr(got, ref)
    if E > 4:
        assert not got[2].any()
    # VJP with a random cotangent
    dw = rng.normal(size=(E, n_out)).astype(np.float32)
    gv = B.e3_radial_weights_bwd(net, to_dev(vec), to_dev(dw))
    gref = O.radial_weights_bwd(vec, K, 6, RC, W1, W2, W3, dw)[0]
    assert relerr(gv.cpu().numpy(), gref) <= TOL_VJP, relerr(gv.cpu().numpy(), gref)
    # accumulate: added to an existing grad_vec; and run-to-run bit-identical
    base = rng.normal(size=(E, 3)).astype(np.float32)
    acc = B.e3_radial_weights_bwd(net, to_dev(vec), to_dev(dw), grad_vec=to_dev(base), accumulate=True)
    assert np.array_equal(acc.cpu().numpy(), base + gv.cpu().numpy())
    assert np.array_equal(B.e3_radial_weights_fwd(net, to_dev(vec)).cpu().numpy(), got)
    net.destroy()


def test_radial_rejects_unsupported_shapes():
    rng = np.random.default_rng(0)
    W1, W2, W3 = _net(rng, 8, 64)
    with pytest.raises(B.E3Error) as ei:
        B.Radial(8, 6, RC, W1[:, :32], W2[:32, :32], W3[:32])
    assert ei.value.status == B.E3_ERR_UNSUPPORTED
    with pytest.raises(B.E3Error):
        B.Radial(8, 6, RC, W1, W2, W3[:, :60])


@pytest.mark.parametrize("k", [1, 2])
def test_whole_path_with_generated_weights(k):
    """positions -> SH and generated weights -> fused TP + scatter -> VJP -> forces = SH term + radial term, vs the oracle."""
    cfg = W.CONFIGS[k]
    pl, g, x, _, G = make_case(cfg)
    plan = gpu_plan(pl)
    P, C = len(pl[3]), cfg.channels
    rng = np.random.default_rng(50 + k)
    K = 8 if k == 1 else 16
    W1, W2, W3 = _net(rng, K, P * C)
    W3 *= W.w_sigma(cfg, P)
    net = B.Radial(K, 6, RC, W1, W2, W3)
    snd, rcv, vec = to_dev(g.senders), to_dev(g.receivers), to_dev(g.vec)
    xd, Gd = to_dev(x), to_dev(G)
    row_ptr, perm_s, col_ptr = B.e3_graph_prepare(snd, rcv, g.n_nodes, validate=True)
    sh = B.e3_sh_fwd(plan, vec)
    w = B.e3_radial_weights_fwd(net, vec)
    out = B.e3_tp_scatter_fwd(plan, xd, sh, w, snd, rcv, row_ptr, g.n_nodes)
    dx, dY, dw = B.e3_tp_scatter_bwd(plan, xd, sh, w, snd, rcv, row_ptr, perm_s, col_ptr, g.n_nodes, Gd)
    dvec = B.e3_sh_bwd(plan, vec, dY)
    B.e3_radial_weights_bwd(net, vec, dw, grad_vec=dvec, accumulate=True)
    F = B.e3_force_reduce(dvec, row_ptr, perm_s, col_ptr, g.n_nodes)
    torch.cuda.synchronize()
    v64 = g.vec.astype(np.float64)
    Y = O.sh(pl[1], v64)
    wr = O.radial_weights(v64, K, 6, RC, W1, W2, W3)
    outr = O.tp_scatter_fwd(*pl, x, Y, wr, g.senders, g.receivers, g.n_nodes)
    dxr, dYr, dwr = O.tp_scatter_bwd(*pl, x, Y, wr, g.senders, g.receivers, g.n_nodes, G)
    dvr = O.sh_bwd(pl[1], v64, dYr) + O.radial_weights_bwd(v64, K, 6, RC, W1, W2, W3, dwr)[0]
    Fr = O.force_reduce(dvr, g.senders, g.receivers, g.n_nodes)
    errs = dict(w=relerr(w.cpu().numpy(), wr), out=relerr(out.cpu().numpy(), outr), dx=relerr(dx.cpu().numpy(), dxr),
                dw=relerr(dw.cpu().numpy(), dwr), dvec=relerr(dvec.cpu().numpy(), dvr), F=relerr(F.cpu().numpy(), Fr))
    print(cfg.name, {a: f"{b:.2e}" for a, b in errs.items()})
    assert errs["w"] <= TOL_FWD and errs["out"] <= 2 * TOL_FWD, errs          # out: fp32 tensor product of fp32-rounded generated weights
    assert max(errs[a] for a in ("dx", "dw", "dvec", "F")) <= TOL_VJP, errs
    assert np.abs(F.cpu().numpy().astype(np.float64).sum(0)).max() <= 1e-3 * np.abs(Fr).max()
    net.destroy()


@pytest.mark.parametrize("pp", ["0", "16"])
def test_other_backward_gemm_kernels_still_match_the_oracle(pp):
    """E3_RADIAL_BWD_PP selects the lock-step backward GEMM (0) or the 512-row x K=16 shape of the warp-specialised one (16); the library
    reads it once per process, so the parity cases above are re-run in a child process with it set."""
    import os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(root, "tests", "test_gpu_radial.py"), "-q", "-x", "-m", "gpu",
                        "-k", "test_radial_weights_and_vjp_against_oracle", "-p", "no:cacheprovider"],
                       env={**os.environ, "E3_RADIAL_BWD_PP": pp}, cwd=root, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert "6 passed" in r.stdout, r.stdout[-500:]

