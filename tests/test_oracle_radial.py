"""Pins of the NEXT-1 oracle (oracle/e3_oracle_next.c: radial basis, polynomial envelope, radial network, their VJP and the
radial force term) against things that are not the oracle: closed forms, a library spherical Bessel function, quadrature,
finite differences, a vectorised numpy / scipy restatement, a hand-typed scalar case, and conservation laws of the whole path.
Readings R1-R4."""
import numpy as np
import pytest
from scipy import special

import oracle as O

RC = 5.0


# ------------------------------------------------------------------ envelope (R2)
@pytest.mark.parametrize("p", [3, 5, 6])
def test_envelope_closed_forms(p):
    u, du = O.poly_envelope(p, [0.0, 1.0, 1.0 - 1e-12, 1.5])
    assert u[0] == 1.0 and du[0] == 0.0                      # u(0) = 1, flat at the origin
    assert abs(u[2]) < 1e-10 and abs(du[2]) < 1e-9           # u(1) = u'(1) = 0 (approached from inside)
    assert u[1] == 0.0 and u[3] == 0.0 and du[3] == 0.0      # identically zero outside
    h = 1e-4                                                 # u''(1) = 0: one-sided second difference of u' vanishes like h
    _, d = O.poly_envelope(p, [1.0 - h, 1.0 - 2 * h])
    assert abs((d[0] - 0.0) / h) < 10 * h * (p + 2) ** 3
    x = np.linspace(0.01, 0.99, 50)
    u, du = O.poly_envelope(p, x)
    fd = (O.poly_envelope(p, x + 1e-6)[0] - O.poly_envelope(p, x - 1e-6)[0]) / 2e-6
    assert np.abs(du - fd).max() < 1e-8
    assert np.all(np.diff(u) < 0)                            # monotone decreasing on (0, 1)


def test_envelope_p6_is_the_typed_polynomial():
    x = np.linspace(0, 0.999, 101)
    u, _ = O.poly_envelope(6, x)
    assert np.abs(u - (1 - 28 * x ** 6 + 48 * x ** 7 - 21 * x ** 8)).max() < 1e-14


# ------------------------------------------------------------------ Bessel basis (R1)
@pytest.mark.parametrize("K", [8, 16])
def test_bessel_basis_against_library_j0_zero_at_cutoff_and_orthonormality(K):
    r = np.linspace(0.0, RC, 301)
    f, _ = O.radial_basis(K, 6, RC, r)
    u, _ = O.poly_envelope(6, r / RC)
    k = np.arange(1, K + 1)
    ref = np.sqrt(2 / RC) * (k * np.pi / RC)[None, :] * special.spherical_jn(0, k[None, :] * np.pi * r[:, None] / RC) * u[:, None]
    assert np.abs(f - ref).max() < 1e-12
    assert np.abs(f[-1]).max() == 0.0                        # f(rc) = 0
    # textbook value: b_k(rc / (2k)) = sqrt(2/rc) * 2k / rc  (sin(pi/2) = 1)
    for kk in (1, 3, K):
        rr = RC / (2 * kk)
        fk, _ = O.radial_basis(K, 6, RC, [rr])
        uu, _ = O.poly_envelope(6, [rr / RC])
        assert abs(fk[0, kk - 1] / uu[0] - np.sqrt(2 / RC) * 2 * kk / RC) < 1e-12
    # orthonormality of the bare basis under int_0^rc . r^2 dr (Gauss-Legendre, envelope divided out)
    xg, wg = np.polynomial.legendre.leggauss(200)
    rq = 0.5 * RC * (xg + 1) * (1 - 1e-9) + 1e-12
    fq, _ = O.radial_basis(K, 6, RC, rq)
    uq, _ = O.poly_envelope(6, rq / RC)
    bq = fq / uq[:, None]
    gram = (bq * (0.5 * RC * wg * rq ** 2)[:, None]).T @ bq
    assert np.abs(gram - np.eye(K)).max() < 1e-6


def test_radial_basis_derivative_against_central_differences():
    r = np.array([0.035, 0.5, 1.7, 3.3, 4.9, 4.999])
    f, d = O.radial_basis(16, 6, RC, r)
    h = 1e-6
    fd = (O.radial_basis(16, 6, RC, r + h)[0] - O.radial_basis(16, 6, RC, r - h)[0]) / (2 * h)
    assert np.abs(d - fd).max() < 2e-7 * max(1.0, np.abs(d).max())
    f0, d0 = O.radial_basis(8, 6, RC, [0.0])                 # r = 0: finite value k pi / rc sqrt(2/rc), zero slope
    assert np.allclose(f0[0], np.sqrt(2 / RC) * np.arange(1, 9) * np.pi / RC) and not d0.any()
    fo, do = O.radial_basis(8, 6, RC, [5.0, 7.0])            # outside the cutoff: identically zero
    assert not fo.any() and not do.any()


# ------------------------------------------------------------------ network (R3)
def _net(rng, K=8, H=64, M=40):
    return (rng.normal(size=(K, H)) / np.sqrt(K), rng.normal(size=(H, H)) / np.sqrt(H), rng.normal(size=(H, M)) / np.sqrt(H))


def test_mlp_against_vectorised_library_restatement_and_scalar_case():
    rng = np.random.default_rng(1)
    W1, W2, W3 = _net(rng)
    f = rng.normal(size=(37, 8))
    sil = lambda a: a * special.expit(a)
    assert np.abs(O.radial_mlp_fwd(f, W1, W2, W3) - sil(sil(f @ W1) @ W2) @ W3).max() < 1e-13
    # K = H = M = 1, typed by hand: w = c * silu(b * silu(a * f))
    a, b, c, x = 0.7, -1.3, 2.0, 0.9
    s1 = a * x / (1 + np.exp(-a * x))
    s2 = b * s1 / (1 + np.exp(-b * s1))
    got = O.radial_mlp_fwd([[x]], [[a]], [[b]], [[c]])
    assert abs(got[0, 0] - c * s2) < 1e-15
    assert not O.radial_mlp_fwd(np.zeros((3, 8)), W1, W2, W3).any()      # silu(0) = 0, no biases: zero features give zero weights


def test_mlp_vjp_against_central_differences_and_adjoint_identity():
    rng = np.random.default_rng(2)
    K, H, M, n = 8, 16, 12, 9
    W1, W2, W3 = _net(rng, K, H, M)
    f = rng.normal(size=(n, K))
    g = rng.normal(size=(n, M))
    df, dW1, dW2, dW3 = O.radial_mlp_bwd(f, W1, W2, W3, g)
    L = lambda f_, a, b, c: float((O.radial_mlp_fwd(f_, a, b, c) * g).sum())
    h = 1e-6
    for name, arr, grad in (("f", f, df), ("W1", W1, dW1), ("W2", W2, dW2), ("W3", W3, dW3)):
        for _ in range(12):
            idx = tuple(rng.integers(0, s) for s in arr.shape)
            ap, am = arr.copy(), arr.copy()
            ap[idx] += h; am[idx] -= h
            vals = []
            for a_ in (ap, am):
                kw = dict(f_=f, a=W1, b=W2, c=W3)
                kw[{"f": "f_", "W1": "a", "W2": "b", "W3": "c"}[name]] = a_
                vals.append(L(**kw))
            fd = (vals[0] - vals[1]) / (2 * h)
            assert abs(fd - grad[idx]) < 1e-7 * max(1.0, abs(fd)), (name, idx, fd, grad[idx])
    # W3 is linear: <g, w> = <dW3, W3> (Euler identity of a linear map)
    assert abs((g * O.radial_mlp_fwd(f, W1, W2, W3)).sum() - (dW3 * W3).sum()) < 1e-11


# ------------------------------------------------------------------ whole path with generated weights (R4)
def _tiny_system(rng, n=7, C=2):
    pos = rng.normal(size=(n, 3)) * 1.6
    pairs = [(i, j) for i in range(n) for j in range(n) if i != j and np.linalg.norm(pos[i] - pos[j]) < RC]
    snd = np.array([p[0] for p in pairs], np.int32); rcv = np.array([p[1] for p in pairs], np.int32)
    o = np.lexsort((snd, rcv))
    return pos, snd[o], rcv[o]


def _energy(pos, snd, rcv, pl, x, G, net, K, quad=False):
    vec = pos[rcv] - pos[snd]
    Y = O.sh(pl[1], vec)
    w = O.radial_weights(vec, K, 6, RC, *net)
    out = O.tp_scatter_fwd(*pl, x, Y, w, snd, rcv, pos.shape[0])
    return float((out ** 2).sum()) if quad else float((G * out).sum())


def test_forces_with_radial_term_against_finite_differences_and_conservation():
    rng = np.random.default_rng(3)
    C, K = 2, 8
    irreps_in = [(0, 1, C), (1, -1, C)]
    irreps_out, paths = O.all_paths(irreps_in, 2, 2)
    pl = (irreps_in, 2, irreps_out, paths)
    out_dim = sum(2 * l + 1 for l, _, _ in irreps_out)
    pos, snd, rcv = _tiny_system(rng, 7, C)
    n = pos.shape[0]
    x = rng.normal(size=(n, 4 * C)); G = rng.normal(size=(n, out_dim * C))
    net = _net(rng, K, 16, len(paths) * C)
    vec = pos[rcv] - pos[snd]
    Y = O.sh(2, vec)
    w = O.radial_weights(vec, K, 6, RC, *net)
    # generated weights fed back as explicit weights: the same tensor product (R4)
    out = O.tp_scatter_fwd(*pl, x, Y, w, snd, rcv, n)
    dx, dY, dw = O.tp_scatter_bwd(*pl, x, Y, w, snd, rcv, n, G)
    dvec = O.sh_bwd(2, vec, dY) + O.radial_weights_bwd(vec, K, 6, RC, *net, dw)[0]
    F = O.force_reduce(dvec, snd, rcv, n)
    h = 1e-6
    for i in range(n):
        for a in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[i, a] += h; pm[i, a] -= h
            fd = -(_energy(pp, snd, rcv, pl, x, G, net, K) - _energy(pm, snd, rcv, pl, x, G, net, K)) / (2 * h)
            assert abs(fd - F[i, a]) < 2e-6 * max(1.0, np.abs(F).max()), (i, a, fd, F[i, a])
    assert np.abs(F.sum(0)).max() < 1e-10 * np.abs(F).max()                       # translation invariance
    # the radial term is parallel to the edge, the SH term perpendicular to it
    rad = O.radial_weights_bwd(vec, K, 6, RC, *net, dw)[0]
    assert np.abs(np.cross(rad, vec)).max() < 1e-10 * np.abs(rad).max() * np.abs(vec).max()
    # zero torque for a rotation-invariant scalar: x on 0e only, E = sum out^2 (reading A13)
    x0 = x.copy(); x0[:, C:] = 0.0
    out0 = O.tp_scatter_fwd(*pl, x0, Y, w, snd, rcv, n)
    _, dY0, dw0 = O.tp_scatter_bwd(*pl, x0, Y, w, snd, rcv, n, 2 * out0)
    dv0 = O.sh_bwd(2, vec, dY0) + O.radial_weights_bwd(vec, K, 6, RC, *net, dw0)[0]
    F0 = O.force_reduce(dv0, snd, rcv, n)
    assert np.abs(np.cross(pos, F0).sum(0)).max() < 1e-9 * np.abs(F0).max() * np.abs(pos).max()
    # and the weights really are a function of the distance only: rotating the system leaves them unchanged
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    assert np.abs(O.radial_weights(vec @ q.T, K, 6, RC, *net) - w).max() < 1e-12
