"""NEXT-3 on the GPU: symmetric contraction at correlation 2 (e3_symcon_*) against the fp64 oracle (orc_symcon2_*, reading S1)."""
import numpy as np
import pytest
import torch

import oracle as O
from helpers import TOL_FWD, TOL_VJP, relerr, to_dev
from paper_2605_22698_b200 import binding as B

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("C,lmax,out_lmax,N,S,natural", [(128, 3, 2, 1536, 4, True), (64, 2, 2, 700, 10, True), (33, 1, 1, 50, 1, False),
                                                          (8, 3, 3, 5, 3, False), (256, 2, 1, 64, 2, True),
                                                          (32, 3, 3, 300, 30, False),       # [species][path] accumulators too large for shared memory
                                                          (128, 3, 3, 20000, 4, True)])     # several waves of node chunks
@pytest.mark.parametrize("jit", [True, False])
def test_symmetric_contraction_against_oracle(C, lmax, out_lmax, N, S, natural, jit, monkeypatch):
    """Both kernel families: the run-time specialised ones (default) and the table-driven fallback (E3_SYMCON_JIT=0)."""
    if not jit:
        monkeypatch.setenv("E3_SYMCON_JIT", "0")
    rng = np.random.default_rng(C + 10 * lmax + N)
    irreps_in = [(l, (-1) ** l, C) for l in range(lmax + 1)]
    irreps_out, paths = O.symcon_paths(irreps_in, out_lmax, natural_parity_only=natural)
    in_dim = sum(2 * l + 1 for l, _, _ in irreps_in)
    A = rng.normal(size=(N, in_dim * C)).astype(np.float32)
    z = rng.integers(0, S, size=N).astype(np.int32)
    W = (rng.normal(size=(S, len(paths), C)) / np.sqrt(len(paths))).astype(np.float32)
    sc = B.SymCon(irreps_in, irreps_out, paths, S)
    assert sc.in_dim == in_dim and sc.n_paths == len(paths)
    Ad, zd, Wd = to_dev(A), to_dev(z), to_dev(W)
    out = sc.fwd(Ad, zd, Wd)
    ref = O.symcon2_fwd(irreps_in, irreps_out, paths, S, A, z, W)
    torch.cuda.synchronize()
    assert relerr(out.cpu().numpy(), ref) <= TOL_FWD, relerr(out.cpu().numpy(), ref)
    g = rng.normal(size=ref.shape).astype(np.float32)
    dA, dW = sc.bwd(Ad, zd, Wd, to_dev(g))
    rA, rW = O.symcon2_bwd(irreps_in, irreps_out, paths, S, A, z, W, g)
    errs = dict(dA=relerr(dA.cpu().numpy(), rA), dW=relerr(dW.cpu().numpy(), rW))
    print(C, lmax, N, {k: f"{v:.1e}" for k, v in errs.items()}, "terms", sc.n_terms)
    assert max(errs.values()) <= TOL_VJP, errs
    # partial outputs and determinism
    dA2, none = sc.bwd(Ad, zd, Wd, to_dev(g), want_weights=False)
    assert none is None and np.array_equal(dA2.cpu().numpy(), dA.cpu().numpy())
    _, dW2 = sc.bwd(Ad, zd, Wd, to_dev(g), want_feats=False)
    assert np.array_equal(dW2.cpu().numpy(), dW.cpu().numpy())
    assert np.array_equal(sc.fwd(Ad, zd, Wd).cpu().numpy(), out.cpu().numpy())
    sc.destroy()


def test_symmetric_contraction_rejects_bad_paths():
    C = 8
    with pytest.raises(B.E3Error) as ei:
        B.SymCon([(0, 1, C)], [(3, -1, C)], [(0, 0, 0)], 1)                 # 0 x 0 -> 3: triangle rule
    assert ei.value.status == B.E3_ERR_BAD_PATH
    with pytest.raises(B.E3Error):
        B.SymCon([(1, -1, C)], [(1, -1, C)], [(0, 0, 0)], 1)                # 1o x 1o -> 1o: parity rule
    with pytest.raises(B.E3Error):
        B.SymCon([(1, -1, C)], [(0, 1, C)], [(0, -1, 0)], 1)                # linear path must keep the irrep
