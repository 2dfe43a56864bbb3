"""Pins of the NEXT-2 / NEXT-4 oracle functions (oracle/e3_oracle_next.c) against things that are not themselves: the already
pinned equal-multiplicity oracle, brute-force einsum with sympy-free dense CG from the pinned orc_cg_real, finite differences of
the pinned first-order functions, symmetry of second derivatives, homogeneity identities.
PAPER.md L108-L126 (section 5.2, Eq. 3-4: Hessian rows as VJPs of force components), L484-L485 (NequIP irreps with unequal
multiplicities)."""
import numpy as np
import pytest

import oracle as O


def _graph(rng, n, e):
    snd = rng.integers(0, n, size=e); rcv = rng.integers(0, n, size=e)
    o = np.lexsort((snd, rcv))
    return snd[o].astype(np.int32), rcv[o].astype(np.int32)


# ------------------------------------------------------------------ NEXT-4: per-irrep multiplicities
def test_mul_oracle_equals_equal_multiplicity_oracle():
    rng = np.random.default_rng(1)
    C = 3
    irreps_in = [(0, 1, C), (1, -1, C), (2, 1, C)]
    irreps_out, paths = O.all_paths(irreps_in, 2, 2)
    n, e = 6, 25
    snd, rcv = _graph(rng, n, e)
    x = rng.normal(size=(n, 9 * C)); Y = rng.normal(size=(e, 9)); w = rng.normal(size=(e, len(paths) * C))
    G = rng.normal(size=(n, sum(2 * l + 1 for l, _, _ in irreps_out) * C))
    assert O.tp_mul_dims(irreps_in, 2, irreps_out, paths) == (9 * C, 9, G.shape[1], len(paths) * C)
    assert np.abs(O.tp_mul_fwd(irreps_in, 2, irreps_out, paths, x, Y, w, snd, rcv, n) -
                  O.tp_scatter_fwd(irreps_in, 2, irreps_out, paths, x, Y, w, snd, rcv, n)).max() < 1e-13
    a = O.tp_mul_bwd(irreps_in, 2, irreps_out, paths, x, Y, w, snd, rcv, n, G)
    b = O.tp_scatter_bwd(irreps_in, 2, irreps_out, paths, x, Y, w, snd, rcv, n, G)
    for p, q in zip(a, b):
        assert np.abs(p - q).max() < 1e-12


def _nequip_like():
    """PAPER.md L484-L485 pattern with small multiplicities: 4x0e + 4x0o + 2x1o + 2x1e + 2x2e + 2x2o."""
    irreps_in = [(0, 1, 4), (0, -1, 4), (1, -1, 2), (1, 1, 2), (2, 1, 2), (2, -1, 2)]
    irreps_out, paths = O.all_paths(irreps_in, 2, 2)
    return irreps_in, irreps_out, paths


def test_mul_oracle_brute_force_einsum_and_class_splitting():
    rng = np.random.default_rng(2)
    irreps_in, irreps_out, paths = _nequip_like()
    in_size, sh_dim, out_size, w_size = O.tp_mul_dims(irreps_in, 2, irreps_out, paths)
    assert in_size == 4 + 4 + 3 * 2 + 3 * 2 + 5 * 2 + 5 * 2 and sh_dim == 9
    assert w_size == sum(irreps_in[p[0]][2] for p in paths)
    n, e = 5, 17
    snd, rcv = _graph(rng, n, e)
    x = rng.normal(size=(n, in_size)); Y = rng.normal(size=(e, 9)); w = rng.normal(size=(e, w_size)); G = rng.normal(size=(n, out_size))
    out = O.tp_mul_fwd(irreps_in, 2, irreps_out, paths, x, Y, w, snd, rcv, n)
    # brute force: dense einsum per path with the pinned real CG tensors
    in_off = np.concatenate([[0], np.cumsum([(2 * l + 1) * m for l, _, m in irreps_in])])
    out_off = np.concatenate([[0], np.cumsum([(2 * l + 1) * m for l, _, m in irreps_out])])
    ref = np.zeros_like(out)
    wo = 0
    for (i_in, l2, i_out) in paths:
        l1, _, mu = irreps_in[i_in]
        l3 = irreps_out[i_out][0]
        Cg = O.cg_real(l1, l2, l3)
        xb = x[:, in_off[i_in]:in_off[i_in + 1]].reshape(n, 2 * l1 + 1, mu)
        msg = np.einsum("abc,eau,eb,eu->ecu", Cg, xb[snd], Y[:, l2 * l2:(l2 + 1) ** 2], w[:, wo:wo + mu])
        np.add.at(ref[:, out_off[i_out]:out_off[i_out + 1]].reshape(n, 2 * l3 + 1, mu), rcv, msg)
        wo += mu
    assert np.abs(out - ref).max() < 1e-12
    # splitting into multiplicity classes: the mul-4 irreps and the mul-2 irreps are two independent equal-multiplicity plans
    for mu in (4, 2):
        keep_in = [i for i, t in enumerate(irreps_in) if t[2] == mu]
        sub_in = [irreps_in[i] for i in keep_in]
        keep_p = [k for k, p in enumerate(paths) if p[0] in keep_in]
        sub_out = [irreps_out[paths[k][2]] for k in keep_p]
        sub_paths = [(keep_in.index(paths[k][0]), paths[k][1], j) for j, k in enumerate(keep_p)]
        xs = np.concatenate([x[:, in_off[i]:in_off[i + 1]] for i in keep_in], axis=1)
        w_off = np.concatenate([[0], np.cumsum([irreps_in[p[0]][2] for p in paths])])
        ws = np.concatenate([w[:, w_off[k]:w_off[k + 1]] for k in keep_p], axis=1)
        sub = O.tp_scatter_fwd(sub_in, 2, sub_out, sub_paths, xs, Y, ws, snd, rcv, n)
        full = np.concatenate([out[:, out_off[paths[k][2]]:out_off[paths[k][2] + 1]] for k in keep_p], axis=1)
        assert np.abs(sub - full).max() < 1e-12
    # VJP against central differences of <G, out> in a few entries of every input
    dx, dY, dw = O.tp_mul_bwd(irreps_in, 2, irreps_out, paths, x, Y, w, snd, rcv, n, G)
    L = lambda x_, Y_, w_: float((G * O.tp_mul_fwd(irreps_in, 2, irreps_out, paths, x_, Y_, w_, snd, rcv, n)).sum())
    h = 1e-6
    for arr, grad, k in ((x, dx, 0), (Y, dY, 1), (w, dw, 2)):
        for _ in range(10):
            idx = tuple(rng.integers(0, s) for s in arr.shape)
            ap, am = arr.copy(), arr.copy(); ap[idx] += h; am[idx] -= h
            args_p, args_m = [x, Y, w], [x, Y, w]
            args_p[k], args_m[k] = ap, am
            assert abs((L(*args_p) - L(*args_m)) / (2 * h) - grad[idx]) < 1e-7
    with pytest.raises(ValueError):                                         # a path joining irreps of different multiplicity is rejected
        O.tp_mul_dims([(0, 1, 4), (1, -1, 2)], 1, [(1, -1, 4)], [(0, 1, 0), (1, 0, 0)])


# ------------------------------------------------------------------ NEXT-2: VJP of the VJP
def test_vjp_vjp_against_finite_differences_of_the_first_order_oracle():
    rng = np.random.default_rng(3)
    C = 2
    irreps_in = [(0, 1, C), (1, -1, C), (2, 1, C)]
    irreps_out, paths = O.all_paths(irreps_in, 2, 2)
    pl = (irreps_in, 2, irreps_out, paths)
    n, e = 5, 14
    snd, rcv = _graph(rng, n, e)
    od = sum(2 * l + 1 for l, _, _ in irreps_out) * C
    x = rng.normal(size=(n, 9 * C)); Y = rng.normal(size=(e, 9)); w = rng.normal(size=(e, len(paths) * C)); g = rng.normal(size=(n, od))
    vx = rng.normal(size=x.shape); vY = rng.normal(size=Y.shape); vw = rng.normal(size=w.shape)
    gg, gx, gY, gw = O.tp_vjp_vjp(*pl, x, Y, w, snd, rcv, n, g, vx, vY, vw)

    def S(x_, Y_, w_, g_):
        dx, dY, dw = O.tp_scatter_bwd(*pl, x_, Y_, w_, snd, rcv, n, g_)
        return float((vx * dx).sum() + (vY * dY).sum() + (vw * dw).sum())
    h = 1e-6
    base = [x, Y, w, g]
    for k, grad in enumerate((gx, gY, gw, gg)):
        for _ in range(12):
            idx = tuple(rng.integers(0, s) for s in base[k].shape)
            ap, am = base[k].copy(), base[k].copy(); ap[idx] += h; am[idx] -= h
            a_p, a_m = list(base), list(base)
            a_p[k], a_m[k] = ap, am
            fd = (S(*a_p) - S(*a_m)) / (2 * h)
            assert abs(fd - grad[idx]) < 2e-7 * max(1.0, abs(fd)), (k, idx, fd, grad[idx])
    # gg is the tangent of the forward: T(vx,Y,w) + T(x,vY,w) + T(x,Y,vw)
    T = lambda a, b, c: O.tp_scatter_fwd(*pl, a, b, c, snd, rcv, n)
    assert np.abs(gg - (T(vx, Y, w) + T(x, vY, w) + T(x, Y, vw))).max() < 1e-12
    # the other three are first-order VJPs with one operand replaced by its cotangent (what the CUDA path composes)
    D = lambda a, b, c: O.tp_scatter_bwd(*pl, a, b, c, snd, rcv, n, g)
    assert np.abs(gx - (D(x, vY, w)[0] + D(x, Y, vw)[0])).max() < 1e-12
    assert np.abs(gY - (D(vx, Y, w)[1] + D(x, Y, vw)[1])).max() < 1e-12
    assert np.abs(gw - (D(vx, Y, w)[2] + D(x, vY, w)[2])).max() < 1e-12
    # symmetry of the second derivative of <g, T>: <vY, d/dY <vx, dx>> = <vx, d/dx <vY, dY>>
    z = np.zeros
    a = O.tp_vjp_vjp(*pl, x, Y, w, snd, rcv, n, g, vx, z(Y.shape), z(w.shape))[2]      # d<vx,dx>/dY
    b = O.tp_vjp_vjp(*pl, x, Y, w, snd, rcv, n, g, z(x.shape), vY, z(w.shape))[1]      # d<vY,dY>/dx
    assert abs((a * vY).sum() - (b * vx).sum()) < 1e-11


def test_vjp_vjp_with_unequal_multiplicities_is_the_composition_of_pinned_calls():
    """orc_tp_vjp_vjp on a plan with per-irrep multiplicities (NEXT-2 x NEXT-4) against the composition identities built from the pinned
    general-multiplicity first-order oracle (orc_tp_mul_*) and against central differences of it."""
    rng = np.random.default_rng(31)
    irreps_in, irreps_out, paths = _nequip_like()
    pl = (irreps_in, 2, irreps_out, paths)
    in_size, sh_dim, out_size, w_size = O.tp_mul_dims(*pl)
    n, e = 5, 13
    snd, rcv = _graph(rng, n, e)
    x = rng.normal(size=(n, in_size)); Y = rng.normal(size=(e, sh_dim)); w = rng.normal(size=(e, w_size)); g = rng.normal(size=(n, out_size))
    vx = rng.normal(size=x.shape); vY = rng.normal(size=Y.shape); vw = rng.normal(size=w.shape)
    gg, gx, gY, gw = O.tp_vjp_vjp(*pl, x, Y, w, snd, rcv, n, g, vx, vY, vw)
    T = lambda a, b, c: O.tp_mul_fwd(*pl, a, b, c, snd, rcv, n)
    D = lambda a, b, c: O.tp_mul_bwd(*pl, a, b, c, snd, rcv, n, g)
    assert np.abs(gg - (T(vx, Y, w) + T(x, vY, w) + T(x, Y, vw))).max() < 1e-12
    assert np.abs(gx - (D(x, vY, w)[0] + D(x, Y, vw)[0])).max() < 1e-12
    assert np.abs(gY - (D(vx, Y, w)[1] + D(x, Y, vw)[1])).max() < 1e-12
    assert np.abs(gw - (D(vx, Y, w)[2] + D(x, vY, w)[2])).max() < 1e-12

    def S(x_, Y_, w_):
        dx, dY, dw = O.tp_mul_bwd(*pl, x_, Y_, w_, snd, rcv, n, g)
        return float((vx * dx).sum() + (vY * dY).sum() + (vw * dw).sum())
    h = 1e-6
    for k, (arr, grad) in enumerate(((x, gx), (Y, gY), (w, gw))):
        for _ in range(8):
            idx = tuple(rng.integers(0, s_) for s_ in arr.shape)
            ap, am = arr.copy(), arr.copy(); ap[idx] += h; am[idx] -= h
            args_p, args_m = [x, Y, w], [x, Y, w]
            args_p[k], args_m[k] = ap, am
            fd = (S(*args_p) - S(*args_m)) / (2 * h)
            assert abs(fd - grad[idx]) < 2e-7 * max(1.0, abs(fd))


@pytest.mark.parametrize("lmax", [1, 2, 3])
def test_sh_second_derivative(lmax):
    rng = np.random.default_rng(10 + lmax)
    n, D = 9, (lmax + 1) ** 2
    vec = rng.normal(size=(n, 3)) * 1.7
    vec[3] = [0.0, 0.0, 2.0]                                               # on the polar axis
    dY = rng.normal(size=(n, D)); u = rng.normal(size=(n, 3))
    gv, gd = O.sh_bwd_bwd(lmax, vec, dY, u)
    assert np.abs(gd - np.einsum("nka,na->nk", O.sh_jac(lmax, vec), u)).max() < 1e-13      # J u, via the pinned Jacobian
    h = 1e-6
    fd = (O.sh_bwd(lmax, vec + h * u, dY) - O.sh_bwd(lmax, vec - h * u, dY)) / (2 * h)
    assert np.abs(gv - fd).max() < 1e-7 * max(1.0, np.abs(fd).max())
    # symmetry of sum_lm dY_lm Hess Y_lm:  u2 . (H u) = u . (H u2)
    u2 = rng.normal(size=(n, 3))
    gv2, _ = O.sh_bwd_bwd(lmax, vec, dY, u2)
    assert np.abs((gv * u2).sum(1) - (gv2 * u).sum(1)).max() < 1e-11
    # degree-0 homogeneity: Hess f . v = -grad f, so with u = vec the result is minus the first-order gradient
    gvv, gdv = O.sh_bwd_bwd(lmax, vec, dY, vec)
    assert np.abs(gvv + O.sh_bwd(lmax, vec, dY)).max() < 1e-11 and np.abs(gdv).max() < 1e-12
    # zero vector: zeros (reading A3)
    z1, z2 = O.sh_bwd_bwd(lmax, np.zeros((1, 3)), dY[:1], u[:1])
    assert not z1.any() and not z2.any()


def test_hessian_row_of_the_whole_path_against_finite_differences_of_forces():
    """PAPER.md Eq. 3-4: H_{rho j} = -dF_rho/dr_j for selected force components, by reverse mode through the force function:
    forces F = -dE/dpos of E = <G, out(x, Y(vec(pos)), w)> (x, w fixed), S = sum_i c_i . F_i, dS/dpos by the second-order functions."""
    rng = np.random.default_rng(5)
    C = 2
    irreps_in = [(0, 1, C), (1, -1, C)]
    irreps_out, paths = O.all_paths(irreps_in, 2, 2)
    pl = (irreps_in, 2, irreps_out, paths)
    n = 6
    pos = rng.normal(size=(n, 3)) * 1.5
    pairs = [(i, j) for i in range(n) for j in range(n) if i != j]
    snd = np.array([p[0] for p in pairs], np.int32); rcv = np.array([p[1] for p in pairs], np.int32)
    o = np.lexsort((snd, rcv)); snd, rcv = snd[o], rcv[o]
    e = snd.size
    od = sum(2 * l + 1 for l, _, _ in irreps_out) * C
    x = rng.normal(size=(n, 4 * C)); w = rng.normal(size=(e, len(paths) * C)); G = rng.normal(size=(n, od))
    c = np.zeros((n, 3)); c[2, 1] = 1.0                                     # the selected force component: F[2, y]

    def forces(p):
        vec = p[rcv] - p[snd]
        Y = O.sh(2, vec)
        _, dY, _ = O.tp_scatter_bwd(*pl, x, Y, w, snd, rcv, n, G)
        return O.force_reduce(O.sh_bwd(2, vec, dY), snd, rcv, n)
    vec = pos[rcv] - pos[snd]
    Y = O.sh(2, vec)
    _, dY, _ = O.tp_scatter_bwd(*pl, x, Y, w, snd, rcv, n, G)
    # S = <c, F> = -sum_e (c[rcv] - c[snd]) . dvec_e  ->  cotangent of dvec
    uvec = -(c[rcv] - c[snd])
    g_vec, g_dY = O.sh_bwd_bwd(2, vec, dY, uvec)                            # through dvec = J^T dY: w.r.t. vec (direct) and w.r.t. dY
    z = np.zeros
    _, _, gY, _ = O.tp_vjp_vjp(*pl, x, Y, w, snd, rcv, n, G, z(x.shape), g_dY, z(w.shape))   # dY depends on Y: d<g_dY, dY>/dY
    g_vec = g_vec + O.sh_bwd(2, vec, gY)                                    # and Y depends on vec
    dS_dpos = O.force_reduce(g_vec, snd, rcv, n) * -1.0                     # force_reduce returns -(in - out); dS/dpos = +(in - out)
    h = 1e-6
    for i in range(n):
        for a in range(3):
            pp, pm = pos.copy(), pos.copy(); pp[i, a] += h; pm[i, a] -= h
            fd = ((c * forces(pp)).sum() - (c * forces(pm)).sum()) / (2 * h)
            assert abs(fd - dS_dpos[i, a]) < 2e-6 * max(1.0, np.abs(dS_dpos).max()), (i, a, fd, dS_dpos[i, a])


# ------------------------------------------------------------------ NEXT-3: symmetric contraction, correlation 2
def _wigner_from_sh(l, R, rng):
    """Real Wigner-D of degree l obtained from the (pinned) SH alone: least squares of Y_l(R r) = D Y_l(r)."""
    v = rng.normal(size=(6 * (2 * l + 1), 3))
    Ya = O.sh(l, v)[:, l * l:(l + 1) ** 2]; Yb = O.sh(l, v @ R.T)[:, l * l:(l + 1) ** 2]
    return np.linalg.lstsq(Ya, Yb, rcond=None)[0].T


def test_symmetric_contraction_oracle():
    rng = np.random.default_rng(21)
    C, S = 3, 4
    irreps_in = [(0, 1, C), (1, -1, C), (2, 1, C)]
    irreps_out, paths = O.symcon_paths(irreps_in, 2)
    assert [p for p in paths if p[1] < 0] == [(0, -1, 0), (1, -1, 1), (2, -1, 2)]
    # quadratic, natural parity: (0,0,0) (0,1,1) (0,2,2) (1,1,0) (1,1,2) (1,2,1) (2,2,0) (2,2,2)   [(1,1,1), (1,2,2), (2,2,1) are pseudo-tensors]
    assert [(irreps_in[a][0], irreps_in[b][0], irreps_out[o][0]) for a, b, o in paths if b >= 0] == \
        [(0, 0, 0), (0, 1, 1), (0, 2, 2), (1, 1, 0), (1, 1, 2), (1, 2, 1), (2, 2, 0), (2, 2, 2)]
    N = 7
    A = rng.normal(size=(N, 9 * C)); z = rng.integers(0, S, size=N).astype(np.int32); W = rng.normal(size=(S, len(paths), C))
    B = O.symcon2_fwd(irreps_in, irreps_out, paths, S, A, z, W)
    # brute force with einsum
    in_off = np.concatenate([[0], np.cumsum([2 * l + 1 for l, _, _ in irreps_in])])
    out_off = np.concatenate([[0], np.cumsum([2 * l + 1 for l, _, _ in irreps_out])])
    blk = lambda i: A[:, in_off[i] * C:in_off[i + 1] * C].reshape(N, -1, C)
    ref = np.zeros_like(B)
    for k, (a, b, o) in enumerate(paths):
        dst = ref[:, out_off[o] * C:out_off[o + 1] * C].reshape(N, -1, C)
        if b < 0:
            dst += W[z, k][:, None, :] * blk(a)
        else:
            Cg = O.cg_real(irreps_in[a][0], irreps_in[b][0], irreps_out[o][0])
            dst += W[z, k][:, None, :] * np.einsum("abc,nau,nbu->ncu", Cg, blk(a), blk(b))
    assert np.abs(B - ref).max() < 1e-12
    # L = 0 closed form: C(l,l,0) = (-1)^l delta / sqrt(2l+1)  =>  W * (-1)^l |A_l|^2 / sqrt(2l+1)
    for k, (a, b, o) in enumerate(paths):
        if b == a and irreps_out[o][0] == 0:
            l = irreps_in[a][0]
            want = W[z, k] * ((-1) ** l / np.sqrt(2 * l + 1)) * (blk(a) ** 2).sum(1)
            only = np.zeros_like(W); only[:, k] = W[:, k]
            got = O.symcon2_fwd(irreps_in, irreps_out, paths, S, A, z, only)[:, out_off[o] * C:out_off[o + 1] * C]
            assert np.abs(got - want).max() < 1e-12
    # the antisymmetric self-product 1 x 1 -> 1 vanishes identically
    io2, p2 = O.symcon_paths([(1, -1, C)], 1, natural_parity_only=False)
    k11 = [k for k, (a, b, o) in enumerate(p2) if b == 0 and io2[o][0] == 1][0]
    W2 = np.zeros((S, len(p2), C)); W2[:, k11] = 1.0
    assert np.abs(O.symcon2_fwd([(1, -1, C)], io2, p2, S, A[:, C:4 * C], z, W2)).max() < 1e-13
    # equivariance: rotate every input block with its Wigner-D, outputs rotate with theirs; inversion flips odd blocks
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] *= -1
    D = {l: _wigner_from_sh(l, q, rng) for l in range(3)}
    rot = lambda X, irreps: np.concatenate([np.einsum("ab,nbu->nau", D[l], X[:, o * C:(o + 2 * l + 1) * C].reshape(N, 2 * l + 1, C)).reshape(N, -1)
                                           for (l, _, _), o in zip(irreps, np.concatenate([[0], np.cumsum([2 * t[0] + 1 for t in irreps])]))], axis=1)
    assert np.abs(O.symcon2_fwd(irreps_in, irreps_out, paths, S, rot(A, irreps_in), z, W) - rot(B, irreps_out)).max() < 1e-11
    par = lambda X, irreps: np.concatenate([p * X[:, o * C:(o + 2 * l + 1) * C] for (l, p, _), o in
                                            zip(irreps, np.concatenate([[0], np.cumsum([2 * t[0] + 1 for t in irreps])]))], axis=1)
    assert np.abs(O.symcon2_fwd(irreps_in, irreps_out, paths, S, par(A, irreps_in), z, W) - par(B, irreps_out)).max() < 1e-12
    # VJP: central differences in A and W; dW only touches the rows of species present
    g = rng.normal(size=B.shape)
    dA, dW = O.symcon2_bwd(irreps_in, irreps_out, paths, S, A, z, W, g)
    Lf = lambda A_, W_: float((g * O.symcon2_fwd(irreps_in, irreps_out, paths, S, A_, z, W_)).sum())
    h = 1e-6
    for arr, grad, k in ((A, dA, 0), (W, dW, 1)):
        for _ in range(15):
            idx = tuple(rng.integers(0, s) for s in arr.shape)
            ap, am = arr.copy(), arr.copy(); ap[idx] += h; am[idx] -= h
            args_p, args_m = [A, W], [A, W]
            args_p[k], args_m[k] = ap, am
            assert abs((Lf(*args_p) - Lf(*args_m)) / (2 * h) - grad[idx]) < 2e-7 * max(1.0, abs(grad[idx]))
    assert abs((dW * W).sum() - (g * B).sum()) < 1e-10                     # linear in W: Euler identity
    with pytest.raises(ValueError):
        O.symcon2_fwd(irreps_in, [(3, -1, C)], [(0, 0, 0)], S, A, z, np.zeros((S, 1, C)))       # 0 x 0 -> 3 violates the triangle rule
