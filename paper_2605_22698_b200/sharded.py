"""NEXT-4 / SURVEY 8(e): one graph sharded over the GPUs of a node by receiver range (reading N2 in DESIGN.md).

One process per GPU.  Rank k owns the atoms [b_k, b_{k+1}) and all their in-edges, so the dominant streams (weights, SH rows,
`out` rows, grad_weights) never leave the rank.  A pass needs ONE exchange each way and nothing else:

  forward    the feature rows of the rank's halo atoms (senders it does not own) arrive from their owners;
  backward   the grad_feats rows the rank produced for its halo atoms return to their owners, which add them in RANK ORDER
             (fixed order, no atomics: results are run-to-run bit-identical).

The planning (ranges, halo, local relabelling) is the C library's (`e3_shard_ranges`, `e3_shard_localize`, host code); this module
is plumbing only: index bookkeeping and `torch.distributed` point-to-point calls (NCCL over NVLink on GPUs; the same code runs over
gloo on CPU tensors, which is how tests/test_multirank_cpu.py covers it).  The local problem is an ordinary
`e3_tp_scatter_fwd` / `e3_tp_scatter_bwd` call; `compute` lets a test substitute those two calls, the default is the CUDA library
and there is no CPU fallback.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist

from . import binding as B


class _CudaCompute:
    """The two local calls through the C ABI (device tensors)."""

    def __init__(self, plan):
        self.plan = plan

    def prepare(self, senders_local, receivers_local, n_local, device):
        self.snd = torch.from_numpy(senders_local).to(device)
        self.rcv = torch.from_numpy(receivers_local).to(device)
        self.n = n_local
        self.row_ptr, self.perm_s, self.col_ptr = B.e3_graph_prepare(self.snd, self.rcv, n_local)

    def fwd(self, x_local, sh, w):
        return B.e3_tp_scatter_fwd(self.plan, x_local, sh, w, self.snd, self.rcv, self.row_ptr, self.n)

    def bwd(self, x_local, sh, w, g_local):
        return B.e3_tp_scatter_bwd(self.plan, x_local, sh, w, self.snd, self.rcv, self.row_ptr, self.perm_s, self.col_ptr, self.n, g_local)


class ShardedTP:
    """Receiver-range shard of one graph on this rank.

    senders_h / receivers_h: HOST int32 numpy arrays of the WHOLE graph (receiver-sorted; index arrays are small and replicated).
    Edge-indexed tensors passed to fwd / bwd are the rank's slice [e_lo, e_hi); node-indexed ones are the rank's owned rows."""

    def __init__(self, plan, senders_h, receivers_h, n_nodes, device, group=None, compute=None):
        self.group = group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.device = torch.device(device)
        self.bounds = B.e3_shard_ranges(receivers_h, n_nodes, self.world)
        L = B.e3_shard_localize(senders_h, receivers_h, n_nodes, self.bounds[self.rank], self.bounds[self.rank + 1])
        self.lo, self.hi, self.e_lo, self.e_hi = L["lo"], L["hi"], L["e_lo"], L["e_hi"]
        self.n_own, self.halo = self.hi - self.lo, L["halo"]
        self.n_local = self.n_own + len(self.halo)
        # what I need from each owner (halo ids are ascending and the owners' ranges are ascending: contiguous runs of the halo)
        owner = np.searchsorted(np.asarray(self.bounds[1:]), self.halo, side="right")
        self.need = [self.halo[owner == j] for j in range(self.world)]
        # what every other rank needs from me: exchanged once (counts, then ids)
        counts = torch.tensor([len(a) for a in self.need], dtype=torch.int64)
        theirs = torch.zeros(self.world, dtype=torch.int64)
        self._p2p([(counts[j:j + 1], theirs[j:j + 1]) for j in range(self.world)])
        send_ids = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.int64)) for a in self.need]
        recv_ids = [torch.empty(int(theirs[j]), dtype=torch.int64) for j in range(self.world)]
        self._p2p(list(zip(send_ids, recv_ids)))
        self.give = [(ids - self.lo).to(self.device) for ids in recv_ids]      # my local rows each rank reads / returns gradients for
        for j, ids in enumerate(self.give):
            assert ids.numel() == 0 or (int(ids.min()) >= 0 and int(ids.max()) < self.n_own), f"rank {j} asked for rows this rank does not own"
        self.compute = compute if compute is not None else _CudaCompute(plan)
        self.compute.prepare(L["senders_local"], L["receivers_local"], self.n_local, self.device)

    # pairs[j] = (tensor to send to rank j, tensor to receive from rank j); the rank's own pair is a local copy
    def _p2p(self, pairs):
        ops = []
        for j, (snd, rcv) in enumerate(pairs):
            if j == self.rank:
                rcv.copy_(snd)
                continue
            peer = dist.get_global_rank(self.group, j) if self.group is not None else j
            if snd.numel():
                ops.append(dist.P2POp(dist.isend, snd, peer, self.group))
            if rcv.numel():
                ops.append(dist.P2POp(dist.irecv, rcv, peer, self.group))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()

    def gather_halo(self, x_own):
        """[n_own, row] owned rows -> [n_local, row]: owned rows, then the halo rows fetched from their owners."""
        row = x_own.shape[1]
        x_local = torch.empty((self.n_local, row), dtype=x_own.dtype, device=x_own.device)
        x_local[:self.n_own] = x_own
        send = [x_own.index_select(0, ids) for ids in self.give]
        off, recv = self.n_own, []
        for a in self.need:
            recv.append(x_local[off:off + len(a)])
            off += len(a)
        self._p2p(list(zip(send, recv)))
        return x_local

    def scatter_halo_grads(self, dx_local):
        """[n_local, row] local grad_feats -> [n_own, row]: own part plus what the other ranks computed for my atoms, in rank order."""
        dx_own = dx_local[:self.n_own].clone()
        off, send = self.n_own, []
        for a in self.need:
            send.append(dx_local[off:off + len(a)].contiguous())
            off += len(a)
        recv = [torch.empty((ids.numel(), dx_local.shape[1]), dtype=dx_local.dtype, device=dx_local.device) for ids in self.give]
        self._p2p(list(zip(send, recv)))
        for j in range(self.world):                      # fixed order; the ids of one rank are distinct, so each add is race-free
            if j != self.rank and self.give[j].numel():
                dx_own.index_add_(0, self.give[j], recv[j])
        return dx_own

    def fwd(self, x_own, sh, w):
        """out rows of the owned atoms."""
        self._x_local = self.gather_halo(x_own)
        return self.compute.fwd(self._x_local, sh, w)[:self.n_own]

    def bwd(self, x_own, sh, w, g_own, x_local=None):
        """(grad_feats of the owned atoms, grad_sh and grad_weights of the rank's edges)."""
        x_local = x_local if x_local is not None else self.gather_halo(x_own)
        g_local = torch.zeros((self.n_local, g_own.shape[1]), dtype=g_own.dtype, device=g_own.device)
        g_local[:self.n_own] = g_own
        dx_local, dY, dw = self.compute.bwd(x_local, sh, w, g_local)
        return self.scatter_halo_grads(dx_local), dY, dw
