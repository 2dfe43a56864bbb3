"""Pins for the oracle's Clebsch-Gordan and spherical-harmonic functions (CPU only).

Each check compares the oracle with something that is not the oracle: library values
(sympy CG, scipy complex SH and Legendre), closed forms typed here from SURVEY.md 8(c)
readings A1/A2/A4, golden fixtures, or mathematical invariants.
"""
import itertools
import math

import numpy as np
import pytest

import oracle as O
from conftest import read_golden

SQ = math.sqrt
ALL_TRIPLES = [(a, b, c) for a in range(4) for b in range(4) for c in range(abs(a - b), min(a + b, 3) + 1)]


def unit(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


# ------------------------------------------------------------------ complex CG (Racah)
def test_cg_complex_matches_sympy_library():
    from sympy import S
    from sympy.physics.quantum.cg import CG
    for l1, l2 in itertools.product(range(3), range(3)):
        for l3 in range(abs(l1 - l2), l1 + l2 + 1):
            for m1 in range(-l1, l1 + 1):
                for m2 in range(-l2, l2 + 1):
                    m3 = m1 + m2
                    if abs(m3) > l3:
                        continue
                    ref = float(CG(S(l1), S(m1), S(l2), S(m2), S(l3), S(m3)).doit())
                    assert abs(O.cg_complex(l1, m1, l2, m2, l3, m3) - ref) < 1e-14, (l1, m1, l2, m2, l3, m3)


def test_cg_complex_textbook_values_and_selection_rules():
    assert abs(O.cg_complex(1, 0, 1, 0, 2, 0) - SQ(2 / 3)) < 1e-15
    assert abs(O.cg_complex(1, 0, 1, 0, 0, 0) + 1 / SQ(3)) < 1e-15
    assert abs(O.cg_complex(1, 1, 1, -1, 0, 0) - 1 / SQ(3)) < 1e-15
    assert abs(O.cg_complex(1, 1, 1, 0, 2, 1) - 1 / SQ(2)) < 1e-15
    assert abs(O.cg_complex(2, 0, 2, 0, 2, 0) + SQ(2 / 7)) < 1e-15
    assert abs(O.cg_complex(3, 2, 0, 0, 3, 2) - 1.0) < 1e-15
    assert O.cg_complex(1, 1, 1, 1, 2, 1) == 0.0        # m3 != m1 + m2
    assert O.cg_complex(1, 0, 1, 0, 3, 0) == 0.0        # triangle
    assert abs(O.cg_complex(1, 0, 1, 0, 1, 0)) < 1e-16  # odd sum, m = 0


def test_cg_complex_unitarity():
    for l1, l2 in itertools.product(range(4), range(4)):
        rows = []
        for l3 in range(abs(l1 - l2), l1 + l2 + 1):
            for m3 in range(-l3, l3 + 1):
                rows.append([O.cg_complex(l1, m1, l2, m2, l3, m3)
                             for m1 in range(-l1, l1 + 1) for m2 in range(-l2, l2 + 1)])
        M = np.array(rows)
        assert M.shape[0] == M.shape[1]
        assert np.abs(M @ M.T - np.eye(M.shape[0])).max() < 1e-14


# ------------------------------------------------------------------ real CG (reading A4)
@pytest.mark.parametrize("lll", ALL_TRIPLES + [(4, 2, 3), (4, 4, 4), (2, 4, 5)])
def test_cg_real_is_real_or_imaginary_and_orthogonal(lll):
    C, discarded = O.cg_real(*lll, return_discarded=True)
    assert discarded < 1e-14
    orth = np.einsum("abc,abd->cd", C, C)
    assert np.abs(orth - np.eye(2 * lll[2] + 1)).max() < 1e-14


def test_cg_real_closed_forms():
    for l in range(4):
        C = O.cg_real(0, l, l)
        assert np.abs(C[0] - np.eye(2 * l + 1)).max() < 1e-15
        C = O.cg_real(l, 0, l)
        assert np.abs(C[:, 0, :] - np.eye(2 * l + 1)).max() < 1e-15
        C = O.cg_real(l, l, 0)
        assert np.abs(C[:, :, 0] - (-1) ** l * np.eye(2 * l + 1) / SQ(2 * l + 1)).max() < 1e-15


def test_cg_111_is_minus_levi_civita_over_sqrt2():
    # component order of l=1 is (y, z, x) (reading A1); Cartesian label of index i:
    cart = {0: 1, 1: 2, 2: 0}  # index -> (x=0,y=1,z=2)
    eps = np.zeros((3, 3, 3))
    for i, j, k in itertools.permutations(range(3)):
        eps[i, j, k] = np.linalg.det(np.eye(3)[[i, j, k]])
    C = O.cg_real(1, 1, 1)
    for a, b, c in itertools.product(range(3), repeat=3):
        assert abs(C[a, b, c] + eps[cart[a], cart[b], cart[c]] / SQ(2)) < 1e-15
    # so the (1o x Y1 -> 1e) path is -(a x b)/sqrt2
    rng = np.random.default_rng(1)
    a, b = rng.normal(size=3), rng.normal(size=3)
    to_yzx = lambda v: v[[1, 2, 0]]
    got = np.einsum("abc,a,b->c", C, to_yzx(a), to_yzx(b))
    assert np.abs(got - to_yzx(-np.cross(a, b) / SQ(2))).max() < 1e-15


def test_cg_112_golden_nonzeros():
    C = O.cg_real(1, 1, 2)
    want = np.zeros_like(C)
    for m1, m2, m3, num, den in read_golden("cg_112.txt"):
        want[int(m1) + 1, int(m2) + 1, int(m3) + 2] = float(num) / SQ(float(den))
    assert np.count_nonzero(want) == 11
    assert np.abs(C - want).max() < 1e-15


def test_cg_swap_symmetry():
    for l1, l2, l3 in ALL_TRIPLES:
        A, B = O.cg_real(l1, l2, l3), O.cg_real(l2, l1, l3)
        sign = (-1) ** (l1 + l2 - l3)
        assert np.abs(A - sign * np.transpose(B, (1, 0, 2))).max() < 1e-14


def test_cg_nnz_structure_golden():
    rows = read_golden("cg_nnz.txt")
    assert len(rows) == 34
    tot_nnz = tot_nzm = 0
    for l1, l2, l3, nnz, nzm in (map(int, r) for r in rows):
        C = O.cg_real(l1, l2, l3)
        assert int((np.abs(C) > 1e-12).sum()) == nnz, (l1, l2, l3)
        assert int((np.abs(C).sum(axis=1) > 1e-12).sum()) == nzm, (l1, l2, l3)
        tot_nnz += nnz
        tot_nzm += nzm
    assert (tot_nnz, tot_nzm) == (611, 541)       # SURVEY 8(d) totals for lmax 3


# ------------------------------------------------------------------ SH values (A1, A2, A3)
def sh_polynomials(v):
    """Explicit component-normalised real SH up to l=3, typed from SURVEY.md 8(c) reading A2."""
    x, y, z = v
    return np.array([
        1.0,
        SQ(3) * y, SQ(3) * z, SQ(3) * x,
        SQ(15) * x * y, SQ(15) * y * z, SQ(5) / 2 * (3 * z * z - 1), SQ(15) * x * z, SQ(15) / 2 * (x * x - y * y),
        SQ(70) / 4 * y * (3 * x * x - y * y), SQ(105) * x * y * z, SQ(42) / 4 * y * (5 * z * z - 1),
        SQ(7) / 2 * z * (5 * z * z - 3), SQ(42) / 4 * x * (5 * z * z - 1), SQ(105) / 2 * z * (x * x - y * y),
        SQ(70) / 4 * x * (x * x - 3 * y * y),
    ])


def test_sh_matches_explicit_polynomials():
    rng = np.random.default_rng(2)
    u = unit(rng, 64)
    Y = O.sh(3, u)
    want = np.stack([sh_polynomials(v) for v in u])
    assert np.abs(Y - want).max() < 2e-15 * 10


def test_sh_normalises_its_input_and_handles_zero():
    rng = np.random.default_rng(3)
    u = unit(rng, 16)
    scale = rng.uniform(0.05, 7.0, size=(16, 1))
    assert np.abs(O.sh(3, u * scale) - O.sh(3, u)).max() < 1e-14
    Y0 = O.sh(3, np.zeros((2, 3)))
    assert np.array_equal(Y0[:, 0], np.ones(2)) and np.array_equal(Y0[:, 1:], np.zeros((2, 15)))   # reading A3


def test_sh_matches_scipy_complex_sh():
    from scipy.special import sph_harm_y
    rng = np.random.default_rng(4)
    u = unit(rng, 20)
    th, ph = np.arccos(u[:, 2]), np.arctan2(u[:, 1], u[:, 0])
    for lmax in (2, 4, 6):
        Y = O.sh(lmax, u)
        for l in range(lmax + 1):
            for m in range(-l, l + 1):
                yc = sph_harm_y(l, abs(m), th, ph)
                if m == 0:
                    ref = yc.real
                elif m > 0:
                    ref = SQ(2) * (-1) ** m * yc.real
                else:
                    ref = SQ(2) * (-1) ** m * yc.imag
                assert np.abs(Y[:, l * l + l + m] - SQ(4 * math.pi) * ref).max() < 1e-13, (l, m)


def test_sh_norm_addition_theorem_pole_parity():
    from scipy.special import eval_legendre
    rng = np.random.default_rng(5)
    a, b = unit(rng, 50), unit(rng, 50)
    lmax = 6
    Ya, Yb, Ym = O.sh(lmax, a), O.sh(lmax, b), O.sh(lmax, -a)
    Yz = O.sh(lmax, np.array([[0, 0, 1.0]]))[0]
    cosg = np.einsum("ij,ij->i", a, b)
    for l in range(lmax + 1):
        sl = slice(l * l, (l + 1) ** 2)
        assert np.abs((Ya[:, sl] ** 2).sum(1) - (2 * l + 1)).max() < 1e-12
        assert np.abs((Ya[:, sl] * Yb[:, sl]).sum(1) - (2 * l + 1) * eval_legendre(l, cosg)).max() < 1e-12
        want = np.zeros(2 * l + 1); want[l] = SQ(2 * l + 1)
        assert np.abs(Yz[sl] - want).max() < 1e-14
        assert np.abs(Ym[:, sl] - (-1) ** l * Ya[:, sl]).max() < 1e-14


def test_sh_orthonormal_on_sphere_quadrature():
    # Gauss-Legendre x uniform-phi quadrature: (1/4pi) int Y_a Y_b = delta_ab for component norm
    lmax = 4
    zs, wz = np.polynomial.legendre.leggauss(12)
    phis = np.arange(24) * 2 * math.pi / 24
    pts, wts = [], []
    for z, w in zip(zs, wz):
        for p in phis:
            s = SQ(1 - z * z)
            pts.append([s * math.cos(p), s * math.sin(p), z]); wts.append(w / 24 / 2)
    Y = O.sh(lmax, np.array(pts))
    G = np.einsum("ka,kb,k->ab", Y, Y, np.array(wts))
    assert np.abs(G - np.eye((lmax + 1) ** 2)).max() < 1e-12


# ------------------------------------------------------------------ SH gradient
def test_sh_jacobian_finite_differences_and_radial_nullspace():
    rng = np.random.default_rng(6)
    r = rng.normal(size=(12, 3)) * rng.uniform(0.3, 4.0, size=(12, 1))
    J = O.sh_jac(3, r)
    h = 1e-6
    for a in range(3):
        d = np.zeros(3); d[a] = h
        fd = (O.sh(3, r + d) - O.sh(3, r - d)) / (2 * h)
        assert np.abs(J[:, :, a] - fd).max() < 5e-9
    assert np.abs(np.einsum("eka,ea->ek", J, r)).max() < 1e-13          # degree-0 homogeneity
    assert np.abs(O.sh_jac(3, np.zeros((1, 3)))).max() == 0.0           # reading A3


def test_sh_jacobian_l1_closed_form():
    rng = np.random.default_rng(7)
    r = rng.normal(size=(5, 3)) * 2.0
    J = O.sh_jac(1, r)
    for e in range(5):
        n = np.linalg.norm(r[e]); u = r[e] / n
        Pm = SQ(3) * (np.eye(3) - np.outer(u, u)) / n                   # d(sqrt3 u)/dr, rows x,y,z
        assert np.abs(J[e, 1:4] - Pm[[1, 2, 0]]).max() < 1e-14          # rows permuted to (y,z,x)
        assert np.abs(J[e, 0]).max() == 0.0


def test_sh_bwd_is_jacobian_transpose():
    rng = np.random.default_rng(8)
    r = rng.normal(size=(9, 3)); dY = rng.normal(size=(9, 16))
    dv = O.sh_bwd(3, r, dY)
    h = 1e-6
    for a in range(3):
        d = np.zeros(3); d[a] = h
        fd = ((O.sh(3, r + d) - O.sh(3, r - d)) * dY).sum(1) / (2 * h)
        assert np.abs(dv[:, a] - fd).max() < 5e-8


# ------------------------------------------------------------------ SH <-> CG consistency, equivariance
def test_sh_cg_consistency_identity():
    from sympy import S
    from sympy.physics.quantum.cg import CG
    rng = np.random.default_rng(9)
    u = unit(rng, 10)
    Y = O.sh(3, u)
    gold = {(int(a), int(b), int(c)): float(k) for a, b, c, k in read_golden("gaunt_coeffs.txt")}
    for l1, l2, l3 in ALL_TRIPLES:
        C = O.cg_real(l1, l2, l3)
        lhs = np.einsum("abc,ea,eb->ec", C, Y[:, l1 * l1:(l1 + 1) ** 2], Y[:, l2 * l2:(l2 + 1) ** 2])
        if (l1 + l2 + l3) % 2:
            k = 0.0
        else:
            k = SQ((2 * l1 + 1) * (2 * l2 + 1) / (2 * l3 + 1)) * float(CG(S(l1), 0, S(l2), 0, S(l3), 0).doit())
        assert np.abs(lhs - k * Y[:, l3 * l3:(l3 + 1) ** 2]).max() < 1e-13, (l1, l2, l3)
        if (l1, l2, l3) in gold:
            assert abs(k - gold[(l1, l2, l3)]) < 1e-7


def random_rotation(rng):
    q, r = np.linalg.qr(rng.normal(size=(3, 3)))
    q = q @ np.diag(np.sign(np.diag(r)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def wigner_D_from_sh(l, R, rng):
    """Real Wigner-D from the SH alone: least-squares solution of Y_l(R r) = D Y_l(r)."""
    u = unit(rng, 6 * (2 * l + 1))
    A = O.sh(l, u)[:, l * l:]
    B = O.sh(l, u @ R.T)[:, l * l:]
    X, *_ = np.linalg.lstsq(A, B, rcond=None)
    return X.T


def test_wigner_d_and_cg_equivariance():
    rng = np.random.default_rng(10)
    R = random_rotation(rng)
    D = [wigner_D_from_sh(l, R, rng) for l in range(4)]
    for l in range(4):
        assert np.abs(D[l] @ D[l].T - np.eye(2 * l + 1)).max() < 1e-12
    assert np.abs(D[1] - R[np.ix_([1, 2, 0], [1, 2, 0])]).max() < 1e-12       # l=1 is (y,z,x)
    for l1, l2, l3 in ALL_TRIPLES:
        C = O.cg_real(l1, l2, l3)
        a, b = rng.normal(size=2 * l1 + 1), rng.normal(size=2 * l2 + 1)
        lhs = np.einsum("abc,a,b->c", C, D[l1] @ a, D[l2] @ b)
        rhs = D[l3] @ np.einsum("abc,a,b->c", C, a, b)
        assert np.abs(lhs - rhs).max() < 1e-12, (l1, l2, l3)
