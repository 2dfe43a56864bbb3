"""Multi-rank host logic on CPU (gloo, world_size 2): the path is "replicas only", so the N > 1 code is
bench.py's aggregation (max over ranks, whole-job edges/s) and the reference arm's rank gating."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    elapsed = [12.5, 20.0][rank]                      # rank 1 is the slow replica
    ms, value = bench.aggregate_replicas(elapsed, n_edges=1000, steps=4, world=world, device=torch.device("cpu"))
    dist.barrier()
    q.put((rank, ms, value))
    dist.destroy_process_group()


def test_replica_aggregation_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value in res:
        assert ms == 20.0                              # max over ranks, on every rank
        assert abs(value - 2 * 1000 * 4 / 20.0e-3) < 1e-6   # edges of BOTH replicas over the slowest rank's time


def test_single_rank_aggregation_is_identity():
    import bench
    ms, value = bench.aggregate_replicas(10.0, 500, 2, 1, torch.device("cpu"))
    assert ms == 10.0 and value == 500 * 2 / 10.0e-3


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "1", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "1", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0


# ------------------------------------------------------------------ NEXT-4 / SURVEY 8(e): receiver-range sharding with halo exchange
class _OracleCompute:
    """Test-side stand-in for the two local CUDA calls (there is no GPU here): the fp64 oracle on the rank's LOCAL graph.  What the
    test checks is everything around it: ranges, halo lists, relabelling and the two torch.distributed exchanges of ShardedTP."""

    def __init__(self, pl):
        self.pl = pl

    def prepare(self, senders_local, receivers_local, n_local, device):
        self.s, self.r, self.n = senders_local, receivers_local, n_local

    def fwd(self, x_local, sh, w):
        import oracle as O
        return torch.from_numpy(O.tp_scatter_fwd(*self.pl, x_local.numpy(), sh.numpy(), w.numpy(), self.s, self.r, self.n))

    def bwd(self, x_local, sh, w, g_local):
        import oracle as O
        return tuple(torch.from_numpy(a) for a in O.tp_scatter_bwd(*self.pl, x_local.numpy(), sh.numpy(), w.numpy(), self.s, self.r, self.n, g_local.numpy()))


def _shard_case():
    import numpy as np
    import oracle as O
    from paper_2605_22698_b200 import workloads as W
    cfg = W.small_config(n_atoms=70, channels=4, irreps_in=((0, 1), (1, -1)), sh_lmax=2, out_lmax=2, box=11.0, k=8)
    g, rng = W.make_graph(cfg)
    irreps_in = [(l, p, cfg.channels) for l, p in cfg.irreps_in]
    irreps_out, paths = O.all_paths(irreps_in, 2, 2)
    pl = (irreps_in, 2, irreps_out, paths)
    od = sum(2 * l + 1 for l, _, _ in irreps_out)
    x = rng.normal(size=(g.n_nodes, 4 * 4)); w = rng.normal(size=(g.n_edges, len(paths) * 4)); G = rng.normal(size=(g.n_nodes, od * 4))
    Y = O.sh(2, g.vec.astype(np.float64))
    return pl, g, x, w, G, Y


def _shard_worker(rank, world, port, q):
    import numpy as np
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2605_22698_b200.sharded import ShardedTP
    pl, g, x, w, G, Y = _shard_case()
    sh = ShardedTP(None, g.senders, g.receivers, g.n_nodes, "cpu", compute=_OracleCompute(pl))
    e = slice(sh.e_lo, sh.e_hi)
    T = lambda a: torch.from_numpy(np.ascontiguousarray(a))
    out = sh.fwd(T(x[sh.lo:sh.hi]), T(Y[e]), T(w[e]))
    dx, dY, dw = sh.bwd(T(x[sh.lo:sh.hi]), T(Y[e]), T(w[e]), T(G[sh.lo:sh.hi]))
    dist.barrier()
    q.put((rank, sh.lo, sh.hi, sh.e_lo, sh.e_hi, len(sh.halo), out.numpy(), dx.numpy(), dY.numpy(), dw.numpy()))
    dist.destroy_process_group()


def test_sharded_tp_halo_exchange_gloo_world2():
    import numpy as np
    import oracle as O
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    pl, g, x, w, G, Y = _shard_case()
    out = O.tp_scatter_fwd(*pl, x, Y, w, g.senders, g.receivers, g.n_nodes)
    dx, dY, dw = O.tp_scatter_bwd(*pl, x, Y, w, g.senders, g.receivers, g.n_nodes, G)
    assert res[0][1] == 0 and res[0][2] == res[1][1] and res[1][2] == g.n_nodes and res[0][4] == res[1][3] and res[1][4] == g.n_edges
    assert res[0][5] > 0 and res[1][5] > 0                                   # both ranks really have a halo (periodic box)
    for rank, lo, hi, e_lo, e_hi, _, o, a, b, c in res:
        assert np.abs(o - out[lo:hi]).max() < 1e-12 and np.abs(a - dx[lo:hi]).max() < 1e-12
        assert np.abs(b - dY[e_lo:e_hi]).max() < 1e-12 and np.abs(c - dw[e_lo:e_hi]).max() < 1e-12


def test_shard_planner_matches_the_oracle_reading():
    import numpy as np
    import oracle as O
    from paper_2605_22698_b200 import binding as B
    from paper_2605_22698_b200 import workloads as W
    g, _ = W.make_graph(W.CONFIGS[2])
    for world in (1, 2, 3, 8):
        b = B.e3_shard_ranges(g.receivers, g.n_nodes, world)
        assert b == O.shard_ranges(g.receivers, g.n_nodes, world)
        for k in range(world):
            L = B.e3_shard_localize(g.senders, g.receivers, g.n_nodes, b[k], b[k + 1])
            R = O.shard_local_graph(g.senders, g.receivers, g.n_nodes, world, k)
            assert all(L[key] == R[key] for key in ("lo", "hi", "e_lo", "e_hi"))
            assert all(np.array_equal(L[key], R[key]) for key in ("halo", "senders_local", "receivers_local"))
    assert B.e3_shard_ranges(np.zeros(0, np.int32), 5, 3) == [0, 5, 5, 5]
    import pytest
    with pytest.raises(B.E3Error) as e:
        B.e3_shard_ranges(np.array([3, 1], np.int32), 5, 2)
    assert e.value.status == B.E3_ERR_UNSORTED
