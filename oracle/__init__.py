"""fp64 CPU oracle for the e3j hot path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes marshalling over ``oracle/e3_oracle.c`` (plain C, double precision, the
definitions of SURVEY.md section 8(c); see the header of that file for citations and pins).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It imports nothing from the CUDA
package ``paper_2605_22698_b200`` and the CUDA package never imports it.

Every array crossing this boundary is float64 / int32 numpy, C-contiguous.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "e3_oracle.c")
_SRC_NEXT = os.path.join(_HERE, "e3_oracle_next.c")      # SURVEY 8(f) NEXT rows (radial network, second order, ...)
_LIB = os.path.join(_HERE, "libe3_oracle.so")


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2, no fast-math).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_NEXT)):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", _SRC, _SRC_NEXT, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Irrep(C.Structure):
    _fields_ = [("l", C.c_int), ("parity", C.c_int), ("mul", C.c_int)]


class _Path(C.Structure):
    _fields_ = [("i_in", C.c_int), ("l_sh", C.c_int), ("i_out", C.c_int)]


_lib = None


def _L():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_cg_complex.restype = C.c_double
        _lib.orc_cg_complex.argtypes = [C.c_int] * 6
        _lib.orc_cg_real.restype = C.c_double
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _plan_args(irreps_in, sh_lmax, irreps_out, paths):
    """irreps_*: sequence of (l, parity(+1/-1), mul); paths: sequence of (i_in, l_sh, i_out)."""
    ii = (_Irrep * len(irreps_in))(*[_Irrep(*map(int, t)) for t in irreps_in])
    io = (_Irrep * len(irreps_out))(*[_Irrep(*map(int, t)) for t in irreps_out])
    pp = (_Path * len(paths))(*[_Path(*map(int, t)) for t in paths])
    return (ii, C.c_int(len(irreps_in)), C.c_int(int(sh_lmax)), io, C.c_int(len(irreps_out)), pp, C.c_int(len(paths)))


def num_threads() -> int:
    return int(_L().orc_num_threads())


def set_num_threads(n: int) -> None:
    _L().orc_set_num_threads(C.c_int(int(n)))


def cg_complex(l1, m1, l2, m2, l3, m3) -> float:
    """Condon-Shortley <l1 m1 l2 m2 | l3 m3> (Racah closed form)."""
    return float(_L().orc_cg_complex(l1, m1, l2, m2, l3, m3))


def cg_real(l1, l2, l3, return_discarded=False):
    """Dense real CG tensor [(2l1+1),(2l2+1),(2l3+1)] (reading A4)."""
    out = np.zeros((2 * l1 + 1, 2 * l2 + 1, 2 * l3 + 1), dtype=np.float64)
    d = _L().orc_cg_real(C.c_int(l1), C.c_int(l2), C.c_int(l3), _p(out))
    return (out, float(d)) if return_discarded else out


def sh(lmax, vec):
    """Y[n,(lmax+1)^2] of raw vectors vec[n,3] (component normalisation, readings A1-A3)."""
    vec = _f64(vec).reshape(-1, 3)
    Y = np.empty((vec.shape[0], (lmax + 1) ** 2), dtype=np.float64)
    _L().orc_sh(C.c_int(lmax), C.c_int64(vec.shape[0]), _p(vec), _p(Y))
    return Y


def sh_jac(lmax, vec):
    """J[n,(lmax+1)^2,3] = dY/dvec."""
    vec = _f64(vec).reshape(-1, 3)
    J = np.empty((vec.shape[0], (lmax + 1) ** 2, 3), dtype=np.float64)
    _L().orc_sh_jac(C.c_int(lmax), C.c_int64(vec.shape[0]), _p(vec), _p(J))
    return J


def sh_bwd(lmax, vec, dY):
    vec = _f64(vec).reshape(-1, 3)
    dY = _f64(dY)
    dvec = np.empty_like(vec)
    _L().orc_sh_bwd(C.c_int(lmax), C.c_int64(vec.shape[0]), _p(vec), _p(dY), _p(dvec))
    return dvec


def graph_prepare(senders, receivers, n_nodes):
    senders, receivers = _i32(senders), _i32(receivers)
    E = senders.shape[0]
    row_ptr = np.empty(n_nodes + 1, dtype=np.int32)
    col_ptr = np.empty(n_nodes + 1, dtype=np.int32)
    perm_s = np.empty(E, dtype=np.int32)
    rc = _L().orc_graph_prepare(_p(senders), _p(receivers), C.c_int64(E), C.c_int32(n_nodes),
                                _p(row_ptr), _p(perm_s), _p(col_ptr))
    if rc:
        raise ValueError("oracle graph_prepare: index out of range")
    return row_ptr, perm_s, col_ptr


def plan_dims(irreps_in, sh_lmax, irreps_out, paths):
    a = _plan_args(irreps_in, sh_lmax, irreps_out, paths)
    i, s, o = C.c_int(), C.c_int(), C.c_int()
    rc = _L().orc_plan_dims(*a, C.byref(i), C.byref(s), C.byref(o))
    if rc:
        raise ValueError(f"oracle plan invalid (code {rc})")
    return i.value, s.value, o.value


def tp_scatter_fwd(irreps_in, sh_lmax, irreps_out, paths, x, Y, w, senders, receivers, n_nodes):
    """out[N, out_dim*C] -- SURVEY 8(a) a4, dense definition."""
    a = _plan_args(irreps_in, sh_lmax, irreps_out, paths)
    in_dim, sh_dim, out_dim = plan_dims(irreps_in, sh_lmax, irreps_out, paths)
    Cm = int(irreps_in[0][2])
    x, Y, w = _f64(x), _f64(Y), _f64(w)
    senders, receivers = _i32(senders), _i32(receivers)
    E = senders.shape[0]
    assert x.size == n_nodes * in_dim * Cm and Y.size == E * sh_dim and w.size == E * len(paths) * Cm
    out = np.empty((n_nodes, out_dim * Cm), dtype=np.float64)
    rc = _L().orc_tp_scatter_fwd(*a, _p(x), _p(Y), _p(w), _p(senders), _p(receivers),
                                 C.c_int64(E), C.c_int32(n_nodes), _p(out))
    if rc:
        raise ValueError(f"oracle plan invalid (code {rc})")
    return out


def tp_scatter_bwd(irreps_in, sh_lmax, irreps_out, paths, x, Y, w, senders, receivers, n_nodes, g):
    """(dx[N,in_dim*C], dY[E,sh_dim], dw[E,P*C]) -- SURVEY 8(a) a5, dense definition."""
    a = _plan_args(irreps_in, sh_lmax, irreps_out, paths)
    in_dim, sh_dim, out_dim = plan_dims(irreps_in, sh_lmax, irreps_out, paths)
    Cm = int(irreps_in[0][2])
    x, Y, w, g = _f64(x), _f64(Y), _f64(w), _f64(g)
    senders, receivers = _i32(senders), _i32(receivers)
    E = senders.shape[0]
    assert g.size == n_nodes * out_dim * Cm
    dx = np.empty((n_nodes, in_dim * Cm), dtype=np.float64)
    dY = np.empty((E, sh_dim), dtype=np.float64)
    dw = np.empty((E, len(paths) * Cm), dtype=np.float64)
    rc = _L().orc_tp_scatter_bwd(*a, _p(x), _p(Y), _p(w), _p(senders), _p(receivers),
                                 C.c_int64(E), C.c_int32(n_nodes), _p(g), _p(dx), _p(dY), _p(dw))
    if rc:
        raise ValueError(f"oracle plan invalid (code {rc})")
    return dx, dY, dw


def force_reduce(dvec, senders, receivers, n_nodes):
    dvec = _f64(dvec).reshape(-1, 3)
    senders, receivers = _i32(senders), _i32(receivers)
    F = np.empty((n_nodes, 3), dtype=np.float64)
    _L().orc_force_reduce(_p(dvec), _p(senders), _p(receivers), C.c_int64(dvec.shape[0]), C.c_int32(n_nodes), _p(F))
    return F


def all_paths(irreps_in, sh_lmax, out_lmax, natural_parity_only=False):
    """Benchmark path table (reading A5/A6), the oracle's own enumerator.

    irreps_in: sequence of (l, parity, mul).  Every (i_in, l2 <= sh_lmax, l3) with
    |l1-l2| <= l3 <= min(l1+l2, out_lmax); output parity p1 * (-1)^l2 (pseudotensor outputs
    included unless natural_parity_only); order i_in, then l2, then l3 ascending; each path
    gets its own output block.  Returns (irreps_out, paths)."""
    irreps_out, paths = [], []
    for i_in, (l1, p1, mul) in enumerate(irreps_in):
        for l2 in range(sh_lmax + 1):
            for l3 in range(abs(l1 - l2), min(l1 + l2, out_lmax) + 1):
                p3 = p1 * (-1) ** l2
                if natural_parity_only and p3 != (-1) ** l3:
                    continue
                irreps_out.append((l3, p3, mul))
                paths.append((i_in, l2, len(irreps_out) - 1))
    return irreps_out, paths


# --------------------------------------------------------------------------------------------
# NEXT-1: radial network generating the weights (e3_oracle_next.c, readings R1-R4)
# --------------------------------------------------------------------------------------------
def poly_envelope(p, x):
    """(u(x), du/dx) of the polynomial envelope (reading R2)."""
    x = _f64(x).reshape(-1)
    u, du = np.empty_like(x), np.empty_like(x)
    _L().orc_poly_envelope(C.c_int(int(p)), C.c_int64(x.size), _p(x), _p(u), _p(du))
    return u, du


def radial_basis(K, p, rc, r):
    """(f[n,K], df/dr[n,K]): Bessel basis times polynomial envelope (readings R1, R2)."""
    r = _f64(r).reshape(-1)
    f, d = np.empty((r.size, K)), np.empty((r.size, K))
    _L().orc_radial_basis(C.c_int(int(K)), C.c_int(int(p)), C.c_double(float(rc)), C.c_int64(r.size), _p(r), _p(f), _p(d))
    return f, d


def radial_mlp_fwd(f, W1, W2, W3):
    """w[n,M] = silu(silu(f W1) W2) W3 (reading R3)."""
    f, W1, W2, W3 = _f64(f), _f64(W1), _f64(W2), _f64(W3)
    n, K = f.shape
    H, M = W3.shape
    assert W1.shape == (K, H) and W2.shape == (H, H)
    w = np.empty((n, M))
    _L().orc_radial_mlp_fwd(C.c_int(K), C.c_int(H), C.c_int(M), C.c_int64(n), _p(f), _p(W1), _p(W2), _p(W3), _p(w))
    return w


def radial_mlp_bwd(f, W1, W2, W3, dw):
    """(df, dW1, dW2, dW3) for a cotangent dw[n,M]."""
    f, W1, W2, W3, dw = _f64(f), _f64(W1), _f64(W2), _f64(W3), _f64(dw)
    n, K = f.shape
    H, M = W3.shape
    df, dW1, dW2, dW3 = np.empty((n, K)), np.empty((K, H)), np.empty((H, H)), np.empty((H, M))
    _L().orc_radial_mlp_bwd(C.c_int(K), C.c_int(H), C.c_int(M), C.c_int64(n), _p(f), _p(W1), _p(W2), _p(W3), _p(dw),
                            _p(df), _p(dW1), _p(dW2), _p(dW3))
    return df, dW1, dW2, dW3


def radial_weights(vec, K, p, rc, W1, W2, W3):
    """w[E, P*C] generated from the edge vectors (R1-R4)."""
    r = np.sqrt((_f64(vec).reshape(-1, 3) ** 2).sum(1))
    f, _ = radial_basis(K, p, rc, r)
    return radial_mlp_fwd(f, W1, W2, W3)


def radial_weights_bwd(vec, K, p, rc, W1, W2, W3, dw):
    """(grad_vec_radial[E,3], dW1, dW2, dW3): VJP of radial_weights; grad_vec = dE/dr * vec/|vec| (0 for a zero vector)."""
    vec = _f64(vec).reshape(-1, 3)
    r = np.sqrt((vec ** 2).sum(1))
    f, dfdr = radial_basis(K, p, rc, r)
    df, dW1, dW2, dW3 = radial_mlp_bwd(f, W1, W2, W3, dw)
    dr = (df * dfdr).sum(1)
    rhat = np.where(r[:, None] > 0, vec / np.where(r > 0, r, 1.0)[:, None], 0.0)
    return dr[:, None] * rhat, dW1, dW2, dW3


# --------------------------------------------------------------------------------------------
# NEXT-4 / NEXT-2: per-irrep multiplicities, second-order VJP, SH second derivative (e3_oracle_next.c)
# --------------------------------------------------------------------------------------------
def tp_mul_dims(irreps_in, sh_lmax, irreps_out, paths):
    a = _plan_args(irreps_in, sh_lmax, irreps_out, paths)
    v = [C.c_int() for _ in range(4)]
    rc = _L().orc_tp_mul_dims(*a, *[C.byref(t) for t in v])
    if rc:
        raise ValueError(f"oracle plan invalid (code {rc})")
    return tuple(t.value for t in v)          # in_size, sh_dim, out_size, w_size (elements per row)


def tp_mul_fwd(irreps_in, sh_lmax, irreps_out, paths, x, Y, w, senders, receivers, n_nodes):
    """Forward with per-irrep multiplicities (NEXT-4); rows are in_size / out_size / w_size elements wide."""
    a = _plan_args(irreps_in, sh_lmax, irreps_out, paths)
    in_size, sh_dim, out_size, w_size = tp_mul_dims(irreps_in, sh_lmax, irreps_out, paths)
    x, Y, w = _f64(x), _f64(Y), _f64(w)
    senders, receivers = _i32(senders), _i32(receivers)
    E = senders.shape[0]
    assert x.size == n_nodes * in_size and Y.size == E * sh_dim and w.size == E * w_size
    out = np.empty((n_nodes, out_size))
    rc = _L().orc_tp_mul_fwd(*a, _p(x), _p(Y), _p(w), _p(senders), _p(receivers), C.c_int64(E), C.c_int32(n_nodes), _p(out))
    if rc:
        raise ValueError(f"oracle plan invalid (code {rc})")
    return out


def tp_mul_bwd(irreps_in, sh_lmax, irreps_out, paths, x, Y, w, senders, receivers, n_nodes, g):
    a = _plan_args(irreps_in, sh_lmax, irreps_out, paths)
    in_size, sh_dim, out_size, w_size = tp_mul_dims(irreps_in, sh_lmax, irreps_out, paths)
    x, Y, w, g = _f64(x), _f64(Y), _f64(w), _f64(g)
    senders, receivers = _i32(senders), _i32(receivers)
    E = senders.shape[0]
    dx, dY, dw = np.empty((n_nodes, in_size)), np.empty((E, sh_dim)), np.empty((E, w_size))
    rc = _L().orc_tp_mul_bwd(*a, _p(x), _p(Y), _p(w), _p(senders), _p(receivers), C.c_int64(E), C.c_int32(n_nodes), _p(g),
                             _p(dx), _p(dY), _p(dw))
    if rc:
        raise ValueError(f"oracle plan invalid (code {rc})")
    return dx, dY, dw


def tp_vjp_vjp(irreps_in, sh_lmax, irreps_out, paths, x, Y, w, senders, receivers, n_nodes, g, vx, vY, vw):
    """(gg, gx, gY, gw): gradients of S = <vx,dx> + <vY,dY> + <vw,dw> (NEXT-2, section 5.2)."""
    a = _plan_args(irreps_in, sh_lmax, irreps_out, paths)
    in_size, sh_dim, out_size, w_size = tp_mul_dims(irreps_in, sh_lmax, irreps_out, paths)
    x, Y, w, g, vx, vY, vw = (_f64(t) for t in (x, Y, w, g, vx, vY, vw))
    senders, receivers = _i32(senders), _i32(receivers)
    E = senders.shape[0]
    gg, gx, gY, gw = np.empty((n_nodes, out_size)), np.empty((n_nodes, in_size)), np.empty((E, sh_dim)), np.empty((E, w_size))
    rc = _L().orc_tp_vjp_vjp(*a, _p(x), _p(Y), _p(w), _p(senders), _p(receivers), C.c_int64(E), C.c_int32(n_nodes), _p(g),
                             _p(vx), _p(vY), _p(vw), _p(gg), _p(gx), _p(gY), _p(gw))
    if rc:
        raise ValueError(f"oracle plan invalid (code {rc})")
    return gg, gx, gY, gw


def sh_bwd_bwd(lmax, vec, dY, u):
    """VJP of (vec, dY) -> J(vec)^T dY for a cotangent u[n,3]: (g_vec[n,3], g_dY[n,(lmax+1)^2])."""
    vec, dY, u = _f64(vec).reshape(-1, 3), _f64(dY), _f64(u).reshape(-1, 3)
    n = vec.shape[0]
    gv, gd = np.empty((n, 3)), np.empty((n, (lmax + 1) ** 2))
    rc = _L().orc_sh_bwd_bwd(C.c_int(lmax), C.c_int64(n), _p(vec), _p(dY), _p(u), _p(gv), _p(gd))
    if rc:
        raise ValueError("lmax out of range")
    return gv, gd


# --------------------------------------------------------------------------------------------
# NEXT-3: symmetric contraction at correlation 2 (e3_oracle_next.c, reading S1)
# --------------------------------------------------------------------------------------------
def symcon_paths(irreps_in, out_lmax, natural_parity_only=True):
    """Path table of the contraction: one linear path per input irrep with l <= out_lmax (its own output block) and one quadratic
    path per (i1 <= i2, L) allowed by the triangle rule, output parity p1*p2 (natural parity (-1)^L only, unless told otherwise);
    order: linear paths first (by i_in), then i1, i2, L ascending; each path gets its own output irrep.  Returns (irreps_out, paths)
    with paths as (i_in1, i_in2 or -1, i_out)."""
    irreps_out, paths = [], []
    for i, (l, p, mul) in enumerate(irreps_in):
        if l <= out_lmax:
            irreps_out.append((l, p, mul)); paths.append((i, -1, len(irreps_out) - 1))
    for i1, (l1, p1, mul) in enumerate(irreps_in):
        for i2 in range(i1, len(irreps_in)):
            l2, p2, _ = irreps_in[i2]
            for L in range(abs(l1 - l2), min(l1 + l2, out_lmax) + 1):
                if natural_parity_only and p1 * p2 != (-1) ** L:
                    continue
                irreps_out.append((L, p1 * p2, mul)); paths.append((i1, i2, len(irreps_out) - 1))
    return irreps_out, paths


class _ScPath(C.Structure):
    _fields_ = [("i_in1", C.c_int), ("i_in2", C.c_int), ("i_out", C.c_int)]


def _sc_args(irreps_in, irreps_out, paths, n_species):
    ii = (_Irrep * len(irreps_in))(*[_Irrep(*map(int, t)) for t in irreps_in])
    io = (_Irrep * len(irreps_out))(*[_Irrep(*map(int, t)) for t in irreps_out])
    pp = (_ScPath * len(paths))(*[_ScPath(*map(int, t)) for t in paths])
    return (ii, C.c_int(len(irreps_in)), io, C.c_int(len(irreps_out)), pp, C.c_int(len(paths)), C.c_int(int(n_species)))


def symcon2_fwd(irreps_in, irreps_out, paths, n_species, A, species, W):
    A, W, species = _f64(A), _f64(W), _i32(species)
    N = A.shape[0]
    Cm = int(irreps_in[0][2])
    out_dim = sum(2 * l + 1 for l, _, _ in irreps_out)
    assert W.shape == (n_species, len(paths), Cm)
    B = np.empty((N, out_dim * Cm))
    rc = _L().orc_symcon2_fwd(*_sc_args(irreps_in, irreps_out, paths, n_species), _p(A), _p(species), _p(W), C.c_int32(N), _p(B))
    if rc:
        raise ValueError(f"oracle symmetric contraction invalid (code {rc})")
    return B


def symcon2_bwd(irreps_in, irreps_out, paths, n_species, A, species, W, g):
    A, W, g, species = _f64(A), _f64(W), _f64(g), _i32(species)
    N = A.shape[0]
    dA, dW = np.empty_like(A), np.empty_like(W)
    rc = _L().orc_symcon2_bwd(*_sc_args(irreps_in, irreps_out, paths, n_species), _p(A), _p(species), _p(W), C.c_int32(N), _p(g), _p(dA), _p(dW))
    if rc:
        raise ValueError(f"oracle symmetric contraction invalid (code {rc})")
    return dA, dW


# ------------------------------------------------------------------------------------------------------------------
# NEXT-4 (the Graph class computes edge vectors from positions and connectivity; L82 "scale model
# deployment to larger systems"; L298 / L497 cutoff 5 A): neighbour list and receiver-range sharding.  Plain numpy, brute force.
# The paper prints neither, so both are readings (N1, N2).
# ------------------------------------------------------------------------------------------------------------------
def neighbor_build(pos, box, cutoff, only_receivers=None):
    """Reading N1.  All pairs, no cell list.  The inclusion test decides an integer (which edges exist), so it is taken in
    the kernel's precision, IEEE float32 with every operation rounded (no fused multiply-add):
        d_a = pos[r,a] - pos[s,a];  if box_a > 0:  d_a = d_a - box_a * rint(d_a / box_a)          (minimum image, reading A10)
        d2  = (d_x*d_x + d_y*d_y) + d_z*d_z;   edge s -> r  iff  s != r and d2 < cutoff*cutoff        (strict, reading A11)
    box_a = 0 means no periodicity along a; a periodic box_a must be >= 2*cutoff (one image at most).  Edges are ordered by
    receiver, ties by ascending sender (A11).  Returns senders, receivers (int32), vec [E,3] float32 (= d) and row_ptr.
    `only_receivers` (ascending atom ids) restricts the OUTPUT to the in-edges of those atoms (sampling for large systems; row_ptr
    is then None); the arithmetic is unchanged.
    Pins (tests/test_oracle_nb.py): scipy's cKDTree on the same positions, the simple cubic lattice's coordination numbers,
    pair symmetry, python-loop brute force on an open cluster, the harness graph of config 1."""
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    box = np.asarray(box, dtype=np.float32).reshape(3)
    rc = np.float32(cutoff)
    if any(b > 0 and b < 2 * rc for b in box):
        raise ValueError("a periodic box edge must be at least twice the cutoff")
    rc2 = rc * rc
    n = pos.shape[0]
    snd, rcv, vec = [], [], []
    rows = np.arange(n) if only_receivers is None else np.asarray(only_receivers, dtype=np.int64)
    for r0 in range(0, len(rows), 256):                           # receivers in slabs only to bound memory
        rid = rows[r0:r0 + 256]
        pr = pos[rid]
        d = pr[:, None, :] - pos[None, :, :]                       # [R, N, 3] float32
        for a in range(3):
            if box[a] > 0:
                d[:, :, a] = d[:, :, a] - box[a] * np.rint(d[:, :, a] / box[a])
        d2 = (d[:, :, 0] * d[:, :, 0] + d[:, :, 1] * d[:, :, 1]) + d[:, :, 2] * d[:, :, 2]
        keep = d2 < rc2
        keep[np.arange(pr.shape[0]), rid] = False
        rr, ss = np.nonzero(keep)                                  # row-major: receiver ascending, then sender ascending
        rcv.append(rid[rr]); snd.append(ss); vec.append(d[rr, ss])
    snd = np.concatenate(snd).astype(np.int32) if snd else np.zeros(0, np.int32)
    rcv = np.concatenate(rcv).astype(np.int32) if rcv else np.zeros(0, np.int32)
    vec = np.concatenate(vec).astype(np.float32) if vec else np.zeros((0, 3), np.float32)
    if only_receivers is not None:
        return snd, rcv, vec, None
    row_ptr = np.zeros(n + 1, np.int32)
    np.add.at(row_ptr, rcv + 1, 1)
    return snd, rcv, vec, np.cumsum(row_ptr).astype(np.int32)


def shard_ranges(receivers, n_nodes, world):
    """Reading N2: contiguous receiver ranges of about equal EDGE counts.  Boundary k (1 <= k < world) is the
    receiver of edge floor(k*E/world) (n_nodes when that index is E); boundaries are made non-decreasing; rank k owns the atoms
    [b_k, b_{k+1}) and all their in-edges."""
    receivers = np.asarray(receivers)
    E = receivers.shape[0]
    b = [0]
    for k in range(1, world):
        t = (k * E) // world
        b.append(max(b[-1], int(receivers[t]) if t < E else n_nodes))
    b.append(n_nodes)
    return b


def shard_local_graph(senders, receivers, n_nodes, world, rank):
    """Reading N2: the local problem of one rank.  Local node ids: the owned atoms b_k..b_{k+1}-1 first (in order), then the halo
    = the senders of the rank's edges that it does not own, ascending.  Returns dict(lo, hi, e_lo, e_hi, halo (global ids),
    senders_local, receivers_local)."""
    senders, receivers = np.asarray(senders), np.asarray(receivers)
    b = shard_ranges(receivers, n_nodes, world)
    lo, hi = b[rank], b[rank + 1]
    e_lo, e_hi = int(np.searchsorted(receivers, lo, "left")), int(np.searchsorted(receivers, hi, "left"))
    s, r = senders[e_lo:e_hi], receivers[e_lo:e_hi]
    halo = np.unique(s[(s < lo) | (s >= hi)])
    s_loc = np.where((s >= lo) & (s < hi), s - lo, (hi - lo) + np.searchsorted(halo, s))
    return dict(lo=lo, hi=hi, e_lo=e_lo, e_hi=e_hi, halo=halo.astype(np.int32), senders_local=s_loc.astype(np.int32),
                receivers_local=(r - lo).astype(np.int32))
