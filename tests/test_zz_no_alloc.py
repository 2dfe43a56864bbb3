"""e3_graph_prepare_noalloc (include/e3b200.h): graph preparation with the library's static device scratch, for callers that cannot
call cudaMalloc.  Collected LAST on purpose (the suite runs with pytest -x).  Integer work: the bar is bit-exact equality with the
existing path, e3_graph_prepare with a caller-owned workspace (itself checked against the oracle in test_gpu_parity.py), and with
the oracle's graph_prepare."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import oracle as O
from helpers import to_dev
from paper_2605_22698_b200 import binding as B

pytestmark = pytest.mark.gpu


def _graph(seed, n, max_deg, hub=0):
    rng = np.random.default_rng(seed)
    rcv, snd = [], []
    for r in range(n):
        d = int(rng.integers(0, max_deg + 1)) if r % 5 else 0            # isolated receivers included
        rcv += [r] * d
        snd += list(rng.integers(0, n, size=d))                          # unsorted senders, repeats allowed
    if hub:                                                              # one sender with a long out-list (merge-sort branch)
        extra = np.sort(rng.integers(0, n, size=hub))
        rcv, snd = np.concatenate([rcv, extra]), np.concatenate([snd, np.full(hub, n // 2)])
        order = np.argsort(rcv, kind="stable")
        rcv, snd = rcv[order], snd[order]
    return np.asarray(snd, np.int32), np.asarray(rcv, np.int32)


def _outputs(n, e, fill):
    return (torch.full((n + 1,), fill, dtype=torch.int32, device="cuda"), torch.full((max(e, 1),), fill, dtype=torch.int32, device="cuda")[:e],
            torch.full((n + 1,), fill, dtype=torch.int32, device="cuda"))


def _check_one(snd, rcv, n, validate):
    sd, rd = to_dev(snd), to_dev(rcv)
    ref = B.e3_graph_prepare(sd, rd, n, validate=True)                   # the existing path (caller-owned workspace)
    got = _outputs(n, len(snd), -7)
    B.e3_graph_prepare_noalloc(sd, rd, n, *got, validate=validate)
    torch.cuda.synchronize()
    for name, a, b in zip(("row_ptr", "perm_s", "col_ptr"), got, ref):
        assert torch.equal(a, b), name
    row_ptr, perm_s, col_ptr = O.graph_prepare(snd, rcv, n)
    assert np.array_equal(got[0].cpu().numpy(), row_ptr) and np.array_equal(got[1].cpu().numpy(), perm_s)
    assert np.array_equal(got[2].cpu().numpy(), col_ptr)


def test_noalloc_graph_prepare_matches_the_existing_path_on_consecutive_calls():
    # calls in a row share the static array and it keeps the previous call's contents: a large graph, then smaller and
    # differently shaped ones (stale cursor / fill entries of the first call lie beyond what the later calls overwrite),
    # then the first again; with and without validation
    cases = [(_graph(1, 3001, 40, hub=700), 3001), (_graph(2, 257, 12), 257), (_graph(3, 1024, 33, hub=300), 1024),
             (_graph(1, 3001, 40, hub=700), 3001), ((np.zeros(0, np.int32), np.zeros(0, np.int32)), 5)]
    for k, ((snd, rcv), n) in enumerate(cases):
        _check_one(snd, rcv, n, validate=bool(k % 2))
    # the same call twice in a row on one stream, no host synchronisation in between
    (snd, rcv), n = cases[0]
    sd, rd = to_dev(snd), to_dev(rcv)
    a, b = _outputs(n, len(snd), -1), _outputs(n, len(snd), -2)
    B.e3_graph_prepare_noalloc(sd, rd, n, *a)
    B.e3_graph_prepare_noalloc(sd, rd, n, *b)
    torch.cuda.synchronize()
    ref = B.e3_graph_prepare(sd, rd, n)
    assert all(torch.equal(x, y) and torch.equal(x, z) for x, y, z in zip(a, b, ref))


def test_noalloc_graph_prepare_allocates_nothing_and_rejects_sizes_beyond_the_static_array():
    cap = B.e3_graph_noalloc_capacity_bytes()
    assert cap == 32 << 20
    (snd, rcv), n = _graph(4, 2000, 30), 2000
    sd, rd = to_dev(snd), to_dev(rcv)
    out = _outputs(n, len(snd), -3)
    B.e3_graph_prepare_noalloc(sd, rd, n, *out)                          # set-up (cudaGetSymbolAddress) done,
    B.e3_graph_prepare_noalloc(sd, rd, n, *out, validate=True)           # every kernel of the call loaded
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        B.e3_graph_prepare_noalloc(sd, rd, n, *out, validate=True)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                                # the driver handed out no device memory
    # validation errors are the existing path's
    with pytest.raises(B.E3Error) as ei:
        B.e3_graph_prepare_noalloc(sd, to_dev(rcv[::-1].copy()), n, *out, validate=True)
    assert ei.value.status == B.E3_ERR_UNSORTED
    # one entry beyond the limit: refused before anything is launched, outputs untouched
    n_big = cap // 4 - 8 + 1
    assert B.lib().e3_graph_workspace_bytes(0, n_big) > cap >= B.lib().e3_graph_workspace_bytes(0, n_big - 1)
    big = _outputs(n_big, 0, -5)
    empty = torch.zeros(0, dtype=torch.int32, device="cuda")
    with pytest.raises(B.E3Error) as ei:
        B.e3_graph_prepare_noalloc(empty, empty, n_big, *big)
    assert ei.value.status == B.E3_ERR_WORKSPACE and "static array" in str(ei.value)
    torch.cuda.synchronize()
    assert int(big[0].min()) == -5 and int(big[2].max()) == -5
    B.e3_graph_prepare_noalloc(empty, empty, n_big - 1, *big)            # exactly at the limit: accepted
    torch.cuda.synchronize()
    assert int(big[0][:n_big].abs().max()) == 0 and int(big[2][:n_big].abs().max()) == 0
