"""Pins for the oracle's TP+scatter forward, VJP, force reduction and graph preparation (CPU only).

The forward is pinned by a dense brute-force einsum, by special cases that reduce to textbook
operations (adjacency SpMV, dot product, cross product), by equivariance under rotations /
inversion and by linearity; the VJP by central finite differences, the Euler identity of the
trilinear map and the adjoint test; forces by finite differences of the energy with respect to
positions, momentum conservation and the zero-torque property; CSR by numpy's stable argsort.
"""
import math

import numpy as np
import pytest

import oracle as O
from test_oracle_cg_sh import random_rotation, unit, wigner_D_from_sh

SQ = math.sqrt


def tiny_graph(rng, n=7, e=30, sort=True):
    snd = rng.integers(0, n, size=e)
    rcv = rng.integers(0, n, size=e)
    if sort:
        o = np.lexsort((snd, rcv))
        snd, rcv = snd[o], rcv[o]
    return snd.astype(np.int32), rcv.astype(np.int32)


def plan(irreps_lp, C, sh_lmax, out_lmax, natural=False):
    irreps_in = [(l, p, C) for l, p in irreps_lp]
    irreps_out, paths = O.all_paths(irreps_in, sh_lmax, out_lmax, natural)
    return irreps_in, sh_lmax, irreps_out, paths


def offsets(irreps):
    off, o = [], 0
    for l, _, _ in irreps:
        off.append(o); o += 2 * l + 1
    return off, o


def brute_force(pl, x, Y, w, snd, rcv, n):
    """The definition as a dense einsum per edge (uses only oracle.cg_real)."""
    irreps_in, sh_lmax, irreps_out, paths = pl
    C = irreps_in[0][2]
    ioff, in_dim = offsets(irreps_in)
    ooff, out_dim = offsets(irreps_out)
    P = len(paths)
    xr = x.reshape(n, in_dim, C); wr = w.reshape(-1, P, C)
    out = np.zeros((n, out_dim, C))
    for e in range(len(snd)):
        for p, (i_in, l2, i_out) in enumerate(paths):
            l1, l3 = irreps_in[i_in][0], irreps_out[i_out][0]
            cg = O.cg_real(l1, l2, l3)
            xb = xr[snd[e], ioff[i_in]:ioff[i_in] + 2 * l1 + 1]
            yb = Y[e, l2 * l2:(l2 + 1) ** 2]
            out[rcv[e], ooff[i_out]:ooff[i_out] + 2 * l3 + 1] += np.einsum("abc,au,b,u->cu", cg, xb, yb, wr[e, p])
    return out.reshape(n, out_dim * C)


def rand_inputs(rng, pl, n, e):
    irreps_in, sh_lmax, irreps_out, paths = pl
    C = irreps_in[0][2]
    _, in_dim = offsets(irreps_in)
    _, out_dim = offsets(irreps_out)
    x = rng.normal(size=(n, in_dim * C))
    vec = rng.normal(size=(e, 3)) * 2
    w = rng.normal(size=(e, len(paths) * C))
    g = rng.normal(size=(n, out_dim * C))
    return x, vec, w, g


PLANS = [
    plan([(0, 1), (1, -1), (2, 1)], 3, 2, 2),
    plan([(0, 1), (1, -1)], 2, 3, 3),
    plan([(0, 1), (1, -1), (2, 1), (3, -1)], 2, 3, 3),
    plan([(1, 1), (2, -1)], 1, 2, 3, natural=False),
]


@pytest.mark.parametrize("pl", PLANS)
def test_fwd_matches_brute_force_einsum(pl):
    rng = np.random.default_rng(11)
    n, e = 6, 25
    snd, rcv = tiny_graph(rng, n, e)
    x, vec, w, _ = rand_inputs(rng, pl, n, e)
    Y = O.sh(pl[1], vec)
    got = O.tp_scatter_fwd(*pl, x, Y, w, snd, rcv, n)
    assert np.abs(got - brute_force(pl, x, Y, w, snd, rcv, n)).max() < 1e-12


def test_fwd_edge_order_isolated_nodes_and_empty_graph():
    rng = np.random.default_rng(12)
    pl = PLANS[0]
    n, e = 9, 20
    snd, rcv = tiny_graph(rng, n, e, sort=False)
    rcv[rcv == 4] = 5                                   # node 4 receives nothing
    x, vec, w, _ = rand_inputs(rng, pl, n, e)
    Y = O.sh(2, vec)
    a = O.tp_scatter_fwd(*pl, x, Y, w, snd, rcv, n)
    o = np.lexsort((snd, rcv))
    b = O.tp_scatter_fwd(*pl, x, Y[o], w[o], snd[o], rcv[o], n)
    assert np.abs(a - b).max() < 1e-13
    assert np.array_equal(a[4], np.zeros_like(a[4]))
    z = O.tp_scatter_fwd(*pl, x, Y[:0], w[:0], snd[:0], rcv[:0], n)
    assert z.shape == a.shape and not z.any()


def test_fwd_special_cases_reduce_to_textbook_ops():
    import scipy.sparse as sp
    rng = np.random.default_rng(13)
    n, e, C = 8, 40, 3
    snd, rcv = tiny_graph(rng, n, e)
    vec = rng.normal(size=(e, 3)); rhat = vec / np.linalg.norm(vec, axis=1, keepdims=True)
    Y = O.sh(1, vec)
    yzx = [1, 2, 0]
    # (0,0,0), w == 1  ->  adjacency SpMV
    x0 = rng.normal(size=(n, C))
    out = O.tp_scatter_fwd([(0, 1, C)], 1, [(0, 1, C)], [(0, 0, 0)], x0, Y, np.ones((e, C)), snd, rcv, n)
    A = sp.coo_matrix((np.ones(e), (rcv, snd)), shape=(n, n)).tocsr()
    assert np.abs(out - A @ x0).max() < 1e-13
    # (0,1,1)  ->  sum_e w x_s Y_1(e)
    w = rng.normal(size=(e, C))
    out = O.tp_scatter_fwd([(0, 1, C)], 1, [(1, -1, C)], [(0, 1, 0)], x0, Y, w, snd, rcv, n).reshape(n, 3, C)
    want = np.zeros((n, 3, C))
    for k in range(e):
        want[rcv[k]] += (SQ(3) * rhat[k][yzx])[:, None] * (w[k] * x0[snd[k]])[None, :]
    assert np.abs(out - want).max() < 1e-13
    # (1,1,0)  ->  - sum_e w (x_vec . rhat)      ;  (1,1,1)  ->  -sqrt(3/2) sum_e w (x_vec x rhat), (y,z,x) order
    xv = rng.normal(size=(n, 3, C))                      # Cartesian (x,y,z) vectors per channel
    x1 = xv[:, yzx, :].reshape(n, 3 * C)
    out0 = O.tp_scatter_fwd([(1, -1, C)], 1, [(0, 1, C)], [(0, 1, 0)], x1, Y, w, snd, rcv, n)
    out1 = O.tp_scatter_fwd([(1, -1, C)], 1, [(1, 1, C)], [(0, 1, 0)], x1, Y, w, snd, rcv, n).reshape(n, 3, C)
    want0 = np.zeros((n, C)); want1 = np.zeros((n, 3, C))
    for k in range(e):
        xs = xv[snd[k]]                                   # [3, C]
        want0[rcv[k]] += -w[k] * (xs * rhat[k][:, None]).sum(0)
        cr = np.cross(xs.T, rhat[k]).T                    # [3, C] Cartesian
        want1[rcv[k]] += -SQ(1.5) * w[k] * cr[yzx]
    assert np.abs(out0 - want0).max() < 1e-13
    assert np.abs(out1 - want1).max() < 1e-13


def test_fwd_shared_output_block_adds_and_linearity():
    rng = np.random.default_rng(14)
    C, n, e = 2, 5, 18
    irreps_in = [(0, 1, C), (1, -1, C)]
    # two paths land on the same 1o block (reading A6): 0e x Y1 -> 1o and 1o x Y0 -> 1o
    shared = (irreps_in, 1, [(1, -1, C)], [(0, 1, 0), (1, 0, 0)])
    sep = (irreps_in, 1, [(1, -1, C), (1, -1, C)], [(0, 1, 0), (1, 0, 1)])
    snd, rcv = tiny_graph(rng, n, e)
    x, vec, w, _ = rand_inputs(rng, shared, n, e)
    Y = O.sh(1, vec)
    a = O.tp_scatter_fwd(*shared, x, Y, w, snd, rcv, n).reshape(n, 3, C)
    b = O.tp_scatter_fwd(*sep, x, Y, w, snd, rcv, n).reshape(n, 6, C)
    assert np.abs(a - (b[:, :3] + b[:, 3:])).max() < 1e-13
    x2 = rng.normal(size=x.shape)
    lin = O.tp_scatter_fwd(*sep, 2 * x - 3 * x2, Y, w, snd, rcv, n)
    assert np.abs(lin - (2 * b.reshape(n, -1) - 3 * O.tp_scatter_fwd(*sep, x2, Y, w, snd, rcv, n))).max() < 1e-12


def block_diag_D(irreps, Ds, C):
    """Apply per-irrep D_l (times parity if improper) to rows laid out m*C + u."""
    def apply(x, improper=False):
        n = x.shape[0]
        off, dim = offsets(irreps)
        xr = x.reshape(n, dim, C).copy()
        for (l, p, _), o in zip(irreps, off):
            blk = np.einsum("ab,nbu->nau", Ds[l], xr[:, o:o + 2 * l + 1])
            xr[:, o:o + 2 * l + 1] = blk * (p if improper else 1)
        return xr.reshape(n, dim * C)
    return apply


@pytest.mark.parametrize("pl", PLANS[:3])
def test_fwd_equivariance_rotation_and_inversion(pl):
    rng = np.random.default_rng(15)
    irreps_in, lmax, irreps_out, paths = pl
    C = irreps_in[0][2]
    n, e = 6, 24
    snd, rcv = tiny_graph(rng, n, e)
    x, vec, w, _ = rand_inputs(rng, pl, n, e)
    R = random_rotation(rng)
    Ds = [wigner_D_from_sh(l, R, rng) for l in range(4)]
    Din, Dout = block_diag_D(irreps_in, Ds, C), block_diag_D(irreps_out, Ds, C)
    base = O.tp_scatter_fwd(*pl, x, O.sh(lmax, vec), w, snd, rcv, n)
    rot = O.tp_scatter_fwd(*pl, Din(x), O.sh(lmax, vec @ R.T), w, snd, rcv, n)
    assert np.abs(rot - Dout(base)).max() < 1e-11
    I = [np.eye(2 * l + 1) for l in range(4)]
    Pin, Pout = block_diag_D(irreps_in, I, C), block_diag_D(irreps_out, I, C)
    inv = O.tp_scatter_fwd(*pl, Pin(x, True), O.sh(lmax, -vec), w, snd, rcv, n)
    assert np.abs(inv - Pout(base, True)).max() < 1e-12


def test_fwd_node_relabelling_invariance():
    rng = np.random.default_rng(16)
    pl = PLANS[1]
    n, e = 7, 30
    snd, rcv = tiny_graph(rng, n, e)
    x, vec, w, _ = rand_inputs(rng, pl, n, e)
    Y = O.sh(3, vec)
    perm = rng.permutation(n)                              # new label of old node i is perm[i]
    xp = np.empty_like(x); xp[perm] = x
    a = O.tp_scatter_fwd(*pl, x, Y, w, snd, rcv, n)
    b = O.tp_scatter_fwd(*pl, xp, Y, w, perm[snd], perm[rcv], n)
    assert np.abs(b[perm] - a).max() < 1e-13


def test_invalid_plans_are_rejected():
    C = 2
    x = np.zeros((2, C)); Y = np.zeros((1, 4)); w = np.zeros((1, C))
    s = np.zeros(1, np.int32)
    with pytest.raises(ValueError):      # triangle: 0 x 1 -> 0
        O.tp_scatter_fwd([(0, 1, C)], 1, [(0, 1, C)], [(0, 1, 0)], x, Y, w, s, s, 2)
    with pytest.raises(ValueError):      # parity: 0e x Y1 -> 1e
        O.tp_scatter_fwd([(0, 1, C)], 1, [(1, 1, C)], [(0, 1, 0)], x, Y, w, s, s, 2)
    with pytest.raises(ValueError):      # l_sh > lmax
        O.tp_scatter_fwd([(0, 1, C)], 1, [(2, 1, C)], [(0, 2, 0)], x, Y, w, s, s, 2)


# ------------------------------------------------------------------ VJP
@pytest.mark.parametrize("pl", PLANS)
def test_vjp_finite_differences_euler_and_adjoint(pl):
    rng = np.random.default_rng(17)
    lmax = pl[1]
    n, e = 5, 16
    snd, rcv = tiny_graph(rng, n, e)
    x, vec, w, g = rand_inputs(rng, pl, n, e)
    Y = rng.normal(size=(e, (lmax + 1) ** 2))              # Y is an independent input of the trilinear map
    f = lambda x_, Y_, w_: O.tp_scatter_fwd(*pl, x_, Y_, w_, snd, rcv, n)
    dx, dY, dw = O.tp_scatter_bwd(*pl, x, Y, w, snd, rcv, n, g)
    out = f(x, Y, w)
    # Euler identity of a map linear in each argument
    s = (g * out).sum()
    for a, b in ((dx, x), (dY, Y), (dw, w)):
        assert abs((a * b).sum() - s) < 1e-11 * max(1.0, abs(s))
    # adjoint test <g, J v> = <J^T g, v> (exact, by linearity J_x v = f(v, Y, w))
    for grad, mk in ((dx, lambda v: f(v, Y, w)), (dY, lambda v: f(x, v, w)), (dw, lambda v: f(x, Y, v))):
        v = rng.normal(size=grad.shape)
        assert abs((g * mk(v)).sum() - (grad * v).sum()) < 1e-10
    # central finite differences on sampled entries of every input
    h = 1e-6
    for grad, arr, idx in ((dx, x, 0), (dY, Y, 1), (dw, w, 2)):
        flat = arr.reshape(-1)
        for j in rng.choice(flat.size, size=12, replace=False):
            args = [x.copy(), Y.copy(), w.copy()]
            args[idx].reshape(-1)[j] += h
            up = (g * f(*args)).sum()
            args[idx].reshape(-1)[j] -= 2 * h
            dn = (g * f(*args)).sum()
            assert abs((up - dn) / (2 * h) - grad.reshape(-1)[j]) < 1e-6


# ------------------------------------------------------------------ forces
def energy_from_positions(pl, pos, snd, rcv, x, w, G, quadratic=False):
    vec = pos[rcv] - pos[snd]
    out = O.tp_scatter_fwd(*pl, x, O.sh(pl[1], vec), w, snd, rcv, pos.shape[0])
    return (out ** 2).sum() if quadratic else (G * out).sum()


def forces_via_oracle(pl, pos, snd, rcv, x, w, G, quadratic=False):
    n = pos.shape[0]
    vec = pos[rcv] - pos[snd]
    Y = O.sh(pl[1], vec)
    g = 2 * O.tp_scatter_fwd(*pl, x, Y, w, snd, rcv, n) if quadratic else G
    _, dY, _ = O.tp_scatter_bwd(*pl, x, Y, w, snd, rcv, n, g)
    dvec = O.sh_bwd(pl[1], vec, dY)
    return O.force_reduce(dvec, snd, rcv, n), dvec, vec


def lattice_graph(rng, n=8, rc=2.2):
    pos = np.array([[i, j, k] for i in range(2) for j in range(2) for k in range(2)], float)[:n] * 1.5
    pos += rng.normal(scale=0.15, size=pos.shape)           # jittered lattice (reading A18)
    d = pos[:, None] - pos[None]
    r = np.linalg.norm(d, axis=-1)
    rcv, snd = np.nonzero((r < rc) & (r > 0))
    return pos, snd.astype(np.int32), rcv.astype(np.int32)


def test_forces_fd_momentum_orthogonality():
    rng = np.random.default_rng(18)
    pl = PLANS[0]
    pos, snd, rcv = lattice_graph(rng)
    n, e = pos.shape[0], len(snd)
    x, _, w, G = rand_inputs(rng, pl, n, e)
    F, dvec, vec = forces_via_oracle(pl, pos, snd, rcv, x, w, G)
    assert np.abs(F.sum(0)).max() < 1e-11                                  # translation invariance
    assert np.abs(np.einsum("ea,ea->e", dvec, vec)).max() < 1e-11          # dvec_e is orthogonal to r_e
    h = 1e-6
    for i in range(n):
        for a in range(3):
            p = pos.copy(); p[i, a] += h
            up = energy_from_positions(pl, p, snd, rcv, x, w, G)
            p[i, a] -= 2 * h
            dn = energy_from_positions(pl, p, snd, rcv, x, w, G)
            assert abs(-(up - dn) / (2 * h) - F[i, a]) < 2e-6


def test_forces_zero_torque_for_invariant_energy():
    # reading A13: x on 0e blocks only, E = sum |out|^2 is rotation invariant -> no net torque
    rng = np.random.default_rng(19)
    pl = plan([(0, 1)], 3, 2, 2)
    pos, snd, rcv = lattice_graph(rng)
    n, e = pos.shape[0], len(snd)
    x, _, w, _ = rand_inputs(rng, pl, n, e)
    F, _, _ = forces_via_oracle(pl, pos, snd, rcv, x, w, None, quadratic=True)
    assert np.abs(F.sum(0)).max() < 1e-10
    assert np.abs(np.cross(pos, F).sum(0)).max() < 1e-10
    assert np.abs(F).max() > 1e-3


def test_force_reduce_definition():
    rng = np.random.default_rng(20)
    n, e = 6, 20
    snd, rcv = tiny_graph(rng, n, e)
    dvec = rng.normal(size=(e, 3))
    F = O.force_reduce(dvec, snd, rcv, n)
    want = np.zeros((n, 3))
    np.add.at(want, rcv, -dvec); np.add.at(want, snd, dvec)
    assert np.abs(F - want).max() < 1e-14


# ------------------------------------------------------------------ graph preparation
@pytest.mark.parametrize("n,e", [(1, 0), (5, 1), (9, 60), (300, 5000)])
def test_graph_prepare_matches_numpy(n, e):
    rng = np.random.default_rng(21)
    snd, rcv = tiny_graph(rng, n, e)
    row_ptr, perm_s, col_ptr = O.graph_prepare(snd, rcv, n)
    assert np.array_equal(row_ptr, np.concatenate([[0], np.cumsum(np.bincount(rcv, minlength=n))]))
    assert np.array_equal(col_ptr, np.concatenate([[0], np.cumsum(np.bincount(snd, minlength=n))]))
    assert np.array_equal(perm_s, np.argsort(snd, kind="stable"))
    with pytest.raises(ValueError):
        O.graph_prepare(np.array([n], np.int32), np.array([0], np.int32), n)
