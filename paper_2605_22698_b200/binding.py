"""Thin Python binding of the C ABI in ``include/e3b200.h`` -- argument marshalling only.

Every function has the name of the C entry point it calls; tensors are torch tensors used purely
as device (or pinned host) memory handles, and the current torch CUDA stream is passed through.
No step of the hot path is computed here: if ``libe3b200.so`` is missing this module raises, it
never falls back to anything.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libe3b200.so")

E3_F32, E3_BF16 = 0, 1
E3_OK, E3_ERR_INVALID_ARG, E3_ERR_BAD_PATH, E3_ERR_UNSUPPORTED, E3_ERR_UNSORTED, E3_ERR_CUDA, E3_ERR_JIT, E3_ERR_WORKSPACE = range(8)

SYMBOLS = [
    "e3_status_string", "e3_last_error", "e3_all_paths", "e3_plan_create", "e3_plan_destroy", "e3_plan_dims",
    "e3_plan_sizes", "e3_plan_get_cg", "e3_plan_kernel_info", "e3_plan_work", "e3_jit_check", "e3_graph_workspace_bytes",
    "e3_graph_prepare", "e3_sh_fwd", "e3_sh_bwd", "e3_tp_scatter_fwd", "e3_bwd_workspace_bytes", "e3_tp_scatter_bwd",
    "e3_force_reduce", "e3_profile_set_mid_event", "e3_measure_fp32_peak", "e3_session_create", "e3_session_destroy", "e3_session_run_host",
    "e3_vjp_vjp_workspace_bytes", "e3_tp_scatter_vjp_vjp", "e3_sh_bwd_bwd",
    "e3_symcon_create", "e3_symcon_jit_check", "e3_symcon_destroy", "e3_symcon_dims", "e3_symcon_fwd", "e3_symcon_workspace_bytes", "e3_symcon_bwd",
    "e3_neighbor_workspace_bytes", "e3_neighbor_build", "e3_shard_ranges", "e3_shard_localize",
    "e3_radial_create", "e3_radial_destroy", "e3_radial_workspace_bytes", "e3_radial_weights_fwd", "e3_radial_weights_bwd",
    "e3_graph_noalloc_capacity_bytes", "e3_graph_prepare_noalloc",
]


class E3Error(RuntimeError):
    def __init__(self, status, where, detail):
        super().__init__(f"{where}: status {status} ({detail})")
        self.status = status


class _Irrep(C.Structure):
    _fields_ = [("l", C.c_int), ("parity", C.c_int), ("mul", C.c_int)]


class _Path(C.Structure):
    _fields_ = [("i_in", C.c_int), ("l_sh", C.c_int), ("i_out", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2605_22698_b200.build` "
                               "(there is no fallback path)")
        L = C.CDLL(LIB_PATH)
        L.e3_status_string.restype = C.c_char_p
        L.e3_last_error.restype = C.c_char_p
        L.e3_graph_workspace_bytes.restype = C.c_size_t
        L.e3_graph_workspace_bytes.argtypes = [C.c_int64, C.c_int32]
        L.e3_graph_noalloc_capacity_bytes.restype = C.c_size_t
        L.e3_graph_noalloc_capacity_bytes.argtypes = []
        L.e3_bwd_workspace_bytes.restype = C.c_size_t
        L.e3_bwd_workspace_bytes.argtypes = [C.c_void_p, C.c_int64, C.c_int32]
        L.e3_vjp_vjp_workspace_bytes.restype = C.c_size_t
        L.e3_vjp_vjp_workspace_bytes.argtypes = [C.c_void_p, C.c_int64, C.c_int32]
        L.e3_symcon_workspace_bytes.restype = C.c_size_t
        L.e3_symcon_workspace_bytes.argtypes = [C.c_void_p, C.c_int32]
        L.e3_neighbor_workspace_bytes.restype = C.c_size_t
        L.e3_neighbor_workspace_bytes.argtypes = [C.c_int32]
        L.e3_radial_workspace_bytes.restype = C.c_size_t
        L.e3_radial_workspace_bytes.argtypes = [C.c_void_p, C.c_int64]
        _lib = L
    return _lib


def _check(rc, where):
    if rc != E3_OK:
        L = lib()
        raise E3Error(rc, where, f"{L.e3_status_string(rc).decode()}: {L.e3_last_error().decode()}")


def _irreps(seq):
    return (_Irrep * len(seq))(*[_Irrep(*map(int, t)) for t in seq])


def _paths(seq):
    return (_Path * len(seq))(*[_Path(*map(int, t)) for t in seq])


def _ptr(t):
    return C.c_void_p(0) if t is None else C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _dev(t, dtype=None):
    assert t.is_cuda and t.is_contiguous(), "device-contiguous tensor required"
    if dtype is not None:
        assert t.dtype == dtype, f"expected {dtype}, got {t.dtype}"
    return t


# --------------------------------------------------------------------------------------------
def e3_all_paths(irreps_in, sh_lmax, out_lmax, natural_parity_only=False):
    ii = _irreps(irreps_in)
    n_out, n_paths = C.c_int(0), C.c_int(0)
    _check(lib().e3_all_paths(ii, len(irreps_in), int(sh_lmax), int(out_lmax), int(natural_parity_only),
                              None, C.byref(n_out), None, C.byref(n_paths)), "e3_all_paths")
    io = (_Irrep * n_out.value)()
    pp = (_Path * n_paths.value)()
    _check(lib().e3_all_paths(ii, len(irreps_in), int(sh_lmax), int(out_lmax), int(natural_parity_only),
                              io, C.byref(n_out), pp, C.byref(n_paths)), "e3_all_paths")
    return [(r.l, r.parity, r.mul) for r in io], [(p.i_in, p.l_sh, p.i_out) for p in pp]


class Plan:
    """Owns an ``e3_plan*``."""

    def __init__(self, handle, irreps_in, sh_lmax, irreps_out, paths, dtype):
        self.handle = handle
        self.irreps_in, self.sh_lmax, self.irreps_out, self.paths, self.dtype = irreps_in, sh_lmax, irreps_out, paths, dtype
        vals = [C.c_int() for _ in range(5)]
        _check(lib().e3_plan_dims(handle, *[C.byref(v) for v in vals]), "e3_plan_dims")
        self.in_dim, self.sh_dim, self.out_dim, self.weights_per_edge, self.nnz_total = [v.value for v in vals]
        self.channels = int(irreps_in[0][2])      # of the first irrep; rows are sized by the three fields below
        sz = [C.c_int64() for _ in range(3)]
        _check(lib().e3_plan_sizes(handle, *[C.byref(v) for v in sz]), "e3_plan_sizes")
        self.feats_per_node, self.out_per_node, self.weights_per_edge = [int(v.value) for v in sz]
        self.n_paths = len(paths)
        self.storage = torch.bfloat16 if dtype == E3_BF16 else torch.float32

    def kernel_info(self, which):
        vals = [C.c_int() for _ in range(6)]
        _check(lib().e3_plan_kernel_info(self.handle, which, *[C.byref(v) for v in vals]), "e3_plan_kernel_info")
        keys = ["regs", "spill_bytes", "smem_bytes", "threads_per_block", "n_roles", "channels_per_lane"]
        return dict(zip(keys, [v.value for v in vals]))

    def work(self):
        f, b = C.c_double(), C.c_double()
        _check(lib().e3_plan_work(self.handle, C.byref(f), C.byref(b)), "e3_plan_work")
        return f.value, b.value

    def get_cg(self, path):
        n = C.c_int()
        _check(lib().e3_plan_get_cg(self.handle, path, None, None, None, None, C.byref(n)), "e3_plan_get_cg")
        m1, m2, m3 = [(C.c_int * n.value)() for _ in range(3)]
        cf = (C.c_double * n.value)()
        _check(lib().e3_plan_get_cg(self.handle, path, m1, m2, m3, cf, C.byref(n)), "e3_plan_get_cg")
        return list(zip(m1, m2, m3, cf))

    def set_mid_event(self, event):
        """Profiling aid: `event` is a recorded-once torch.cuda.Event(enable_timing=True) or None."""
        h = C.c_void_p(event.cuda_event) if event is not None else C.c_void_p(0)
        _check(lib().e3_profile_set_mid_event(self.handle, h), "e3_profile_set_mid_event")

    def destroy(self):
        if self.handle:
            lib().e3_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def e3_plan_create(irreps_in, sh_lmax, irreps_out, paths, dtype=E3_F32) -> Plan:
    h = C.c_void_p()
    _check(lib().e3_plan_create(C.byref(h), _irreps(irreps_in), len(irreps_in), int(sh_lmax), _irreps(irreps_out),
                                len(irreps_out), _paths(paths), len(paths), int(dtype)), "e3_plan_create")
    return Plan(h, list(irreps_in), int(sh_lmax), list(irreps_out), list(paths), int(dtype))


def e3_jit_check(irreps_in, sh_lmax, irreps_out, paths, dtype=E3_F32, src_path=None):
    """Build-time compile check of the specialised kernels (no device needed)."""
    vals = [C.c_int() for _ in range(4)]
    sp = src_path.encode() if src_path else None
    _check(lib().e3_jit_check(_irreps(irreps_in), len(irreps_in), int(sh_lmax), _irreps(irreps_out), len(irreps_out),
                              _paths(paths), len(paths), int(dtype), sp, *[C.byref(v) for v in vals]), "e3_jit_check")
    return dict(zip(["fwd_regs", "fwd_spill", "bwd_regs", "bwd_spill"], [v.value for v in vals]))


def e3_graph_prepare(senders, receivers, n_nodes, validate=False, stream=None):
    _dev(senders, torch.int32); _dev(receivers, torch.int32)
    E = senders.numel()
    dev = senders.device
    row_ptr = torch.empty(n_nodes + 1, dtype=torch.int32, device=dev)
    col_ptr = torch.empty(n_nodes + 1, dtype=torch.int32, device=dev)
    perm_s = torch.empty(max(E, 1), dtype=torch.int32, device=dev)[:E]
    nbytes = lib().e3_graph_workspace_bytes(E, n_nodes)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    _check(lib().e3_graph_prepare(_ptr(senders), _ptr(receivers), C.c_int64(E), C.c_int32(n_nodes), _ptr(row_ptr),
                                  _ptr(perm_s), _ptr(col_ptr), _ptr(ws), C.c_size_t(nbytes), int(bool(validate)),
                                  _stream(stream)), "e3_graph_prepare")
    return row_ptr, perm_s, col_ptr


def e3_graph_noalloc_capacity_bytes():
    return int(lib().e3_graph_noalloc_capacity_bytes())


def e3_graph_prepare_noalloc(senders, receivers, n_nodes, row_ptr, perm_s, col_ptr, validate=False, stream=None):
    """e3_graph_prepare into caller-owned outputs with the library's static scratch: nothing is allocated, here or in the library."""
    _dev(senders, torch.int32); _dev(receivers, torch.int32)
    _dev(row_ptr, torch.int32); _dev(perm_s, torch.int32); _dev(col_ptr, torch.int32)
    E = senders.numel()
    if row_ptr.numel() < n_nodes + 1 or col_ptr.numel() < n_nodes + 1 or perm_s.numel() < E or receivers.numel() != E:
        raise ValueError("e3_graph_prepare_noalloc: output tensors too small")
    _check(lib().e3_graph_prepare_noalloc(_ptr(senders), _ptr(receivers), C.c_int64(E), C.c_int32(n_nodes), _ptr(row_ptr),
                                          _ptr(perm_s), _ptr(col_ptr), int(bool(validate)), _stream(stream)), "e3_graph_prepare_noalloc")


def e3_sh_fwd(plan: Plan, vec, out=None, stream=None):
    _dev(vec, torch.float32)
    E = vec.shape[0]
    sh = out if out is not None else torch.empty((E, plan.sh_dim), dtype=plan.storage, device=vec.device)
    _check(lib().e3_sh_fwd(plan.handle, _ptr(vec), C.c_int64(E), _ptr(_dev(sh, plan.storage)), _stream(stream)), "e3_sh_fwd")
    return sh


def e3_sh_bwd(plan: Plan, vec, grad_sh, out=None, stream=None):
    _dev(vec, torch.float32); _dev(grad_sh, torch.float32)
    E = vec.shape[0]
    gv = out if out is not None else torch.empty((E, 3), dtype=torch.float32, device=vec.device)
    _check(lib().e3_sh_bwd(plan.handle, _ptr(vec), _ptr(grad_sh), C.c_int64(E), _ptr(gv), _stream(stream)), "e3_sh_bwd")
    return gv


def e3_tp_scatter_fwd(plan: Plan, feats, sh, weights, senders, receivers, row_ptr, n_nodes, out=None, stream=None):
    _dev(feats, plan.storage); _dev(sh, plan.storage); _dev(weights, plan.storage)
    _dev(senders, torch.int32); _dev(row_ptr, torch.int32)
    E = senders.numel()
    if out is None:
        out = torch.empty((n_nodes, plan.out_per_node), dtype=torch.float32, device=feats.device)
    _check(lib().e3_tp_scatter_fwd(plan.handle, _ptr(feats), _ptr(sh), _ptr(weights), _ptr(senders), _ptr(receivers),
                                   _ptr(row_ptr), C.c_int64(E), C.c_int32(n_nodes), _ptr(_dev(out, torch.float32)),
                                   _stream(stream)), "e3_tp_scatter_fwd")
    return out


def e3_measure_fp32_peak(ms_target=200.0, stream=None):
    """Sustained packed-FMA rate of this board in TFLOP/s (measurement aid, see include/e3b200.h)."""
    t = C.c_double(0.0)
    _check(lib().e3_measure_fp32_peak(C.byref(t), C.c_double(ms_target), _stream(stream)), "e3_measure_fp32_peak")
    return float(t.value)


def e3_bwd_workspace_bytes(plan: Plan, n_edges, n_nodes):
    return int(lib().e3_bwd_workspace_bytes(plan.handle, C.c_int64(n_edges), C.c_int32(n_nodes)))


def e3_tp_scatter_bwd(plan: Plan, feats, sh, weights, senders, receivers, row_ptr, perm_s, col_ptr, n_nodes, grad_out,
                      want_grad_weights=True, grad_feats=None, grad_sh=None, grad_weights=None, workspace=None, stream=None):
    _dev(feats, plan.storage); _dev(sh, plan.storage); _dev(weights, plan.storage); _dev(grad_out, torch.float32)
    E = senders.numel()
    dev = feats.device
    if grad_feats is None:
        grad_feats = torch.empty((n_nodes, plan.feats_per_node), dtype=torch.float32, device=dev)
    if grad_sh is None:
        grad_sh = torch.empty((E, plan.sh_dim), dtype=torch.float32, device=dev)
    if grad_weights is None and want_grad_weights:
        grad_weights = torch.empty((E, plan.weights_per_edge), dtype=plan.storage, device=dev)
    nbytes = e3_bwd_workspace_bytes(plan, E, n_nodes)
    if workspace is None:
        workspace = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    _check(lib().e3_tp_scatter_bwd(plan.handle, _ptr(feats), _ptr(sh), _ptr(weights), _ptr(senders), _ptr(receivers),
                                   _ptr(row_ptr), _ptr(perm_s), _ptr(col_ptr), C.c_int64(E), C.c_int32(n_nodes),
                                   _ptr(grad_out), _ptr(grad_feats), _ptr(grad_sh),
                                   _ptr(grad_weights if want_grad_weights else None), _ptr(workspace),
                                   C.c_size_t(workspace.numel()), _stream(stream)), "e3_tp_scatter_bwd")
    return grad_feats, grad_sh, (grad_weights if want_grad_weights else None)


def e3_force_reduce(grad_vec, row_ptr, perm_s, col_ptr, n_nodes, out=None, stream=None):
    _dev(grad_vec, torch.float32)
    E = grad_vec.shape[0]
    F = out if out is not None else torch.empty((n_nodes, 3), dtype=torch.float32, device=grad_vec.device)
    _check(lib().e3_force_reduce(_ptr(grad_vec), _ptr(row_ptr), _ptr(perm_s), _ptr(col_ptr), C.c_int64(E),
                                 C.c_int32(n_nodes), _ptr(F), _stream(stream)), "e3_force_reduce")
    return F


class Session:
    """Owns an ``e3_session*`` (device buffers for the host-buffer entry point)."""

    def __init__(self, plan: Plan, max_edges, max_nodes):
        self.plan = plan
        self.handle = C.c_void_p()
        _check(lib().e3_session_create(C.byref(self.handle), plan.handle, C.c_int64(max_edges), C.c_int32(max_nodes)),
               "e3_session_create")

    def run_host(self, vec, feats, weights, senders, receivers, n_nodes, grad_out=None, out=None, grad_feats=None,
                 grad_weights=None, grad_vec=None, forces=None):
        """All arguments are HOST tensors (ideally pinned); outputs are written in place."""
        for t in (vec, feats, weights, senders, receivers, grad_out, out, grad_feats, grad_weights, grad_vec, forces):
            assert t is None or (not t.is_cuda and t.is_contiguous())
        up, down = C.c_int64(), C.c_int64()
        _check(lib().e3_session_run_host(self.handle, _ptr(vec), _ptr(feats), _ptr(weights), _ptr(senders), _ptr(receivers),
                                         C.c_int64(senders.numel()), C.c_int32(n_nodes), _ptr(grad_out), _ptr(out),
                                         _ptr(grad_feats), _ptr(grad_weights), _ptr(grad_vec), _ptr(forces),
                                         C.byref(up), C.byref(down)), "e3_session_run_host")
        return up.value, down.value

    def destroy(self):
        if self.handle:
            lib().e3_session_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Radial:
    """Owns an ``e3_radial*`` (NEXT-1: the radial network generating the weights).  W1/W2/W3 are host float32 arrays."""

    def __init__(self, num_rbf, envelope_p, cutoff, W1, W2, W3):
        import numpy as np
        W1, W2, W3 = (np.ascontiguousarray(a, dtype=np.float32) for a in (W1, W2, W3))
        self.num_rbf, self.n_hidden, self.n_out = int(num_rbf), int(W2.shape[0]), int(W3.shape[1])
        assert W1.shape == (num_rbf, self.n_hidden) and W3.shape[0] == self.n_hidden
        self.handle = C.c_void_p()
        _check(lib().e3_radial_create(C.byref(self.handle), int(num_rbf), int(envelope_p), C.c_double(float(cutoff)), self.n_hidden,
                                      self.n_out, W1.ctypes.data_as(C.c_void_p), W2.ctypes.data_as(C.c_void_p),
                                      W3.ctypes.data_as(C.c_void_p)), "e3_radial_create")

    def workspace(self, n_edges, device):
        return torch.empty(lib().e3_radial_workspace_bytes(self.handle, C.c_int64(n_edges)), dtype=torch.uint8, device=device)

    def destroy(self):
        if self.handle:
            lib().e3_radial_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def e3_radial_weights_fwd(net: Radial, vec, out=None, workspace=None, stream=None):
    _dev(vec, torch.float32)
    E = vec.shape[0]
    w = out if out is not None else torch.empty((E, net.n_out), dtype=torch.float32, device=vec.device)
    ws = workspace if workspace is not None else net.workspace(E, vec.device)
    _check(lib().e3_radial_weights_fwd(net.handle, _ptr(vec), C.c_int64(E), _ptr(_dev(w, torch.float32)), _ptr(ws),
                                       C.c_size_t(ws.numel()), _stream(stream)), "e3_radial_weights_fwd")
    return w


def e3_radial_weights_bwd(net: Radial, vec, grad_weights, grad_vec=None, accumulate=False, workspace=None, stream=None):
    _dev(vec, torch.float32); _dev(grad_weights, torch.float32)
    E = vec.shape[0]
    gv = grad_vec if grad_vec is not None else torch.empty((E, 3), dtype=torch.float32, device=vec.device)
    ws = workspace if workspace is not None else net.workspace(E, vec.device)
    _check(lib().e3_radial_weights_bwd(net.handle, _ptr(vec), C.c_int64(E), _ptr(grad_weights), _ptr(_dev(gv, torch.float32)),
                                       int(bool(accumulate)), _ptr(ws), C.c_size_t(ws.numel()), _stream(stream)), "e3_radial_weights_bwd")
    return gv


def e3_tp_scatter_vjp_vjp(plan: Plan, feats, sh, weights, senders, receivers, row_ptr, perm_s, col_ptr, n_nodes, grad_out,
                          v_feats=None, v_sh=None, v_weights=None, want=("gg", "gx", "gY", "gw"), stream=None):
    """Second-order VJP (NEXT-2).  Returns a dict with the requested outputs among gg, gx, gY, gw (float32 device tensors)."""
    E = senders.numel()
    dev = feats.device
    f32 = torch.float32
    outs = {"gg": (n_nodes, plan.out_per_node), "gx": (n_nodes, plan.feats_per_node),
            "gY": (E, plan.sh_dim), "gw": (E, plan.weights_per_edge)}
    bufs = {k: (torch.empty(shape, dtype=f32, device=dev) if k in want else None) for k, shape in outs.items()}
    nbytes = int(lib().e3_vjp_vjp_workspace_bytes(plan.handle, C.c_int64(E), C.c_int32(n_nodes)))
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    _check(lib().e3_tp_scatter_vjp_vjp(plan.handle, _ptr(feats), _ptr(sh), _ptr(weights), _ptr(senders), _ptr(receivers), _ptr(row_ptr),
                                       _ptr(perm_s), _ptr(col_ptr), C.c_int64(E), C.c_int32(n_nodes), _ptr(grad_out), _ptr(v_feats),
                                       _ptr(v_sh), _ptr(v_weights), _ptr(bufs["gg"]), _ptr(bufs["gx"]), _ptr(bufs["gY"]), _ptr(bufs["gw"]),
                                       _ptr(ws), C.c_size_t(nbytes), _stream(stream)), "e3_tp_scatter_vjp_vjp")
    return {k: v for k, v in bufs.items() if v is not None}


def e3_sh_bwd_bwd(plan: Plan, vec, grad_sh, u, want_vec=True, want_sh=True, stream=None):
    _dev(vec, torch.float32); _dev(u, torch.float32)
    E = vec.shape[0]
    gv = torch.empty((E, 3), dtype=torch.float32, device=vec.device) if want_vec else None
    gs = torch.empty((E, plan.sh_dim), dtype=torch.float32, device=vec.device) if want_sh else None
    _check(lib().e3_sh_bwd_bwd(plan.handle, _ptr(vec), _ptr(grad_sh), _ptr(u), C.c_int64(E), _ptr(gv), _ptr(gs), _stream(stream)),
           "e3_sh_bwd_bwd")
    return gv, gs


class _PairPath(C.Structure):
    _fields_ = [("i_in1", C.c_int), ("i_in2", C.c_int), ("i_out", C.c_int)]


class SymCon:
    """Owns an ``e3_symcon*`` (NEXT-3: symmetric contraction at correlation 2).  paths: (i_in1, i_in2 or -1, i_out)."""

    def __init__(self, irreps_in, irreps_out, paths, n_species):
        self.handle = C.c_void_p()
        pp = (_PairPath * len(paths))(*[_PairPath(*map(int, t)) for t in paths])
        _check(lib().e3_symcon_create(C.byref(self.handle), _irreps(irreps_in), len(irreps_in), _irreps(irreps_out), len(irreps_out),
                                      pp, len(paths), int(n_species)), "e3_symcon_create")
        v = [C.c_int() for _ in range(4)]
        _check(lib().e3_symcon_dims(self.handle, *[C.byref(t) for t in v]), "e3_symcon_dims")
        self.in_dim, self.out_dim, self.n_paths, self.n_terms = [t.value for t in v]
        self.channels, self.n_species = int(irreps_in[0][2]), int(n_species)

    def fwd(self, feats, species, weights, stream=None):
        _dev(feats, torch.float32); _dev(species, torch.int32); _dev(weights, torch.float32)
        N = feats.shape[0]
        out = torch.empty((N, self.out_dim * self.channels), dtype=torch.float32, device=feats.device)
        _check(lib().e3_symcon_fwd(self.handle, _ptr(feats), _ptr(species), _ptr(weights), C.c_int32(N), _ptr(out), _stream(stream)), "e3_symcon_fwd")
        return out

    def bwd(self, feats, species, weights, grad_out, want_feats=True, want_weights=True, stream=None):
        _dev(grad_out, torch.float32)
        N = feats.shape[0]
        dA = torch.empty_like(feats) if want_feats else None
        dW = torch.empty_like(weights) if want_weights else None
        nb = int(lib().e3_symcon_workspace_bytes(self.handle, C.c_int32(N)))
        ws = torch.empty(nb, dtype=torch.uint8, device=feats.device)
        _check(lib().e3_symcon_bwd(self.handle, _ptr(feats), _ptr(species), _ptr(weights), C.c_int32(N), _ptr(grad_out), _ptr(dA), _ptr(dW),
                                   _ptr(ws), C.c_size_t(nb), _stream(stream)), "e3_symcon_bwd")
        return dA, dW

    def destroy(self):
        if self.handle:
            lib().e3_symcon_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def e3_neighbor_build(pos, box, cutoff, max_edges=None, stream=None):
    """pos: [N,3] float32 device tensor; box: three host floats (0 = open axis).  Returns senders, receivers, vec, row_ptr.
    Without max_edges the call is made twice when the first capacity guess (64 edges per atom) is too small."""
    _dev(pos, torch.float32)
    N, dev = pos.shape[0], pos.device
    bx = (C.c_float * 3)(*[float(b) for b in box])
    nbytes = int(lib().e3_neighbor_workspace_bytes(C.c_int32(N)))
    ws = torch.empty(max(nbytes, 1), dtype=torch.uint8, device=dev)
    row_ptr = torch.empty(N + 1, dtype=torch.int32, device=dev)
    cap = int(max_edges) if max_edges is not None else 64 * N
    for attempt in range(2):
        snd = torch.empty(max(cap, 1), dtype=torch.int32, device=dev)
        rcv = torch.empty(max(cap, 1), dtype=torch.int32, device=dev)
        vec = torch.empty((max(cap, 1), 3), dtype=torch.float32, device=dev)
        n = C.c_int64(0)
        rc = lib().e3_neighbor_build(_ptr(pos), C.c_int32(N), bx, C.c_float(float(cutoff)), C.c_int64(cap), _ptr(snd), _ptr(rcv), _ptr(vec),
                                     _ptr(row_ptr), C.byref(n), _ptr(ws), C.c_size_t(ws.numel()), _stream(stream))
        if rc == E3_ERR_WORKSPACE and n.value > cap and max_edges is None and attempt == 0:
            cap = int(n.value)
            continue
        _check(rc, "e3_neighbor_build")
        E = int(n.value)
        return snd[:E], rcv[:E], vec[:E], row_ptr


def _hptr(a, dtype):
    assert isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous
    return a.ctypes.data_as(C.c_void_p)


def e3_shard_ranges(receivers_h, n_nodes, world):
    """HOST numpy int32 receivers (ascending) -> list of world+1 atom boundaries."""
    b = np.empty(world + 1, dtype=np.int32)
    _check(lib().e3_shard_ranges(_hptr(receivers_h, np.int32), C.c_int64(receivers_h.shape[0]), C.c_int32(n_nodes), C.c_int(world),
                                 _hptr(b, np.int32)), "e3_shard_ranges")
    return [int(v) for v in b]


def e3_shard_localize(senders_h, receivers_h, n_nodes, lo, hi):
    """HOST numpy int32 index arrays -> dict(lo, hi, e_lo, e_hi, halo, senders_local, receivers_local) of the owner of [lo, hi)."""
    e_lo, e_hi, nh = C.c_int64(), C.c_int64(), C.c_int32()
    E = receivers_h.shape[0]
    args = (_hptr(senders_h, np.int32), _hptr(receivers_h, np.int32), C.c_int64(E), C.c_int32(n_nodes), C.c_int32(lo), C.c_int32(hi))
    _check(lib().e3_shard_localize(*args, C.byref(e_lo), C.byref(e_hi), None, None, None, None), "e3_shard_localize")
    n = e_hi.value - e_lo.value
    halo, sl, rl = (np.empty(max(n, 1), dtype=np.int32) for _ in range(3))
    _check(lib().e3_shard_localize(*args, C.byref(e_lo), C.byref(e_hi), _hptr(halo, np.int32), C.byref(nh), _hptr(sl, np.int32),
                                   _hptr(rl, np.int32)), "e3_shard_localize")
    return dict(lo=lo, hi=hi, e_lo=e_lo.value, e_hi=e_hi.value, halo=halo[:nh.value].copy(), senders_local=sl[:n], receivers_local=rl[:n])


def e3_symcon_jit_check(irreps_in, irreps_out, paths):
    """Build-time compile check of the specialised symmetric-contraction kernels (no device needed)."""
    pp = (_PairPath * len(paths))(*[_PairPath(*map(int, t)) for t in paths])
    regs, spill = C.c_int(), C.c_int()
    _check(lib().e3_symcon_jit_check(_irreps(irreps_in), len(irreps_in), _irreps(irreps_out), len(irreps_out), pp, len(paths),
                                     C.byref(regs), C.byref(spill)), "e3_symcon_jit_check")
    return dict(fwd_regs=regs.value, fwd_spill=spill.value)
