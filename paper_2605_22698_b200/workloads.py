"""Seeded synthetic workloads (BASELINE.json configs 1-5) -- input generation ONLY.

This module serves both the CUDA path and the fp64 oracle with identical stored inputs.
It holds none of the method's arithmetic: no spherical harmonics, no Clebsch-Gordan
coefficients, no path enumeration, no tensor product.  It draws positions, builds the
5 A cutoff neighbour list (host-side harness code, reading A11), and draws node
features, per-edge weights and the output cotangent G.

The paper's own workloads are molecular datasets that are not available here; these
configs stand in for them with the paper's shapes (PAPER.md L298 cutoff 5 A; L484-L486
and L533-L534 irreps / l_max / channels; L610 system sizes; L498 batches of small
molecules).  Recipe: numpy Generator(Philox(20260522 + k)),
draw order positions -> (cell sort) -> edges -> x -> w -> G, everything drawn in fp64 and
rounded once to the storage dtype.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

CUTOFF = 5.0
SEED0 = 20260522


@dataclass(frozen=True)
class Config:
    k: int
    name: str
    geometry: str              # "periodic" | "molecules"
    n_atoms: int
    box: float                 # periodic cube edge (A); 0 for molecules
    irreps_in: tuple           # ((l, parity), ...)
    channels: int
    sh_lmax: int
    out_lmax: int
    w_std: str = "1"           # "1" | "1/sqrt(P)"
    storage: str = "f32"       # "f32" | "bf16"
    n_graphs: int = 1
    forces: bool = True
    cell_sort: bool = True

    @property
    def seed(self) -> int:
        return SEED0 + self.k


def _box(n, rho=0.1):
    return (n / rho) ** (1.0 / 3.0)


CONFIGS = {
    1: Config(1, "cfg1_64atoms_32ch_l2", "periodic", 64, 10.0, ((0, 1), (1, -1), (2, 1)), 32, 2, 2),
    2: Config(2, "cfg2_mace_1536atoms_128ch_l3", "periodic", 1536, _box(1536), ((0, 1), (1, -1)), 128, 3, 3,
              w_std="1/sqrt(P)"),
    3: Config(3, "cfg3_256x30mol_64ch_l2", "molecules", 7680, 0.0, ((0, 1), (1, -1), (2, 1)), 64, 2, 2,
              n_graphs=256, forces=False, cell_sort=False),
    4: Config(4, "cfg4_100k_64ch_l3", "periodic", 100000, _box(100000), ((0, 1), (1, -1), (2, 1), (3, -1)), 64, 3, 3),
    5: Config(5, "cfg5_100k_128ch_l3_bf16", "periodic", 100000, _box(100000),
              ((0, 1), (1, -1), (2, 1), (3, -1)), 128, 3, 3, storage="bf16", forces=False),
}


def small_config(n_atoms=24, channels=4, irreps_in=((0, 1), (1, -1)), sh_lmax=2, out_lmax=2, box=8.0, k=100,
                 storage="f32", geometry="periodic", n_graphs=1):
    """Tiny ad-hoc config for parity/edge-case tests (seed 20260522 + k)."""
    return Config(k, f"tiny_{k}", geometry, n_atoms, box, tuple(irreps_in), channels, sh_lmax, out_lmax,
                  storage=storage, n_graphs=n_graphs, cell_sort=False)


# --------------------------------------------------------------------------------------
# geometry + neighbour list
# --------------------------------------------------------------------------------------
def _morton_order(pos, box, cell=CUTOFF):
    """Stable permutation sorting atoms by the Morton code of their `cell`-sized grid cell."""
    n = max(1, int(math.floor(box / cell)))
    c = np.minimum((pos / (box / n)).astype(np.int64), n - 1)
    code = np.zeros(pos.shape[0], dtype=np.int64)
    for bit in range(10):
        for a in range(3):
            code |= ((c[:, a] >> bit) & 1) << (3 * bit + a)
    return np.argsort(code, kind="stable")


def _pairs_periodic(pos, box, rc):
    from scipy.spatial import cKDTree
    t = cKDTree(pos, boxsize=box)
    pr = t.query_pairs(rc, output_type="ndarray")
    return pr[:, 0].astype(np.int64), pr[:, 1].astype(np.int64)


def _pairs_open(pos, rc):
    from scipy.spatial import cKDTree
    t = cKDTree(pos)
    pr = t.query_pairs(rc, output_type="ndarray")
    return pr[:, 0].astype(np.int64), pr[:, 1].astype(np.int64)


def _directed_edges(pos, i, j, box):
    """Both directions of every pair, strict d < CUTOFF, sorted by (receiver, sender).

    Edge vector (reading A10): r_e = pos[receiver] - pos[sender] + shift (minimum image)."""
    snd = np.concatenate([i, j])
    rcv = np.concatenate([j, i])
    d = pos[rcv] - pos[snd]
    if box > 0:
        d -= box * np.round(d / box)
    keep = np.einsum("ij,ij->i", d, d) < CUTOFF * CUTOFF
    snd, rcv, d = snd[keep], rcv[keep], d[keep]
    order = np.lexsort((snd, rcv))
    return snd[order].astype(np.int32), rcv[order].astype(np.int32), d[order]


@dataclass
class Graph:
    n_nodes: int
    pos: np.ndarray            # [N,3] f64
    senders: np.ndarray        # [E] i32
    receivers: np.ndarray      # [E] i32, ascending; ties in ascending sender
    vec: np.ndarray            # [E,3] f32  (stored edge vectors, sender -> receiver)
    box: float
    extra: dict = field(default_factory=dict)

    @property
    def n_edges(self) -> int:
        return int(self.senders.shape[0])


def make_graph(cfg: Config, rng: np.random.Generator | None = None) -> tuple[Graph, np.random.Generator]:
    rng = rng if rng is not None else np.random.Generator(np.random.Philox(cfg.seed))
    if cfg.geometry == "periodic":
        pos = rng.uniform(0.0, cfg.box, size=(cfg.n_atoms, 3))
        if cfg.cell_sort:
            pos = pos[_morton_order(pos, cfg.box)]
        i, j = _pairs_periodic(pos, cfg.box, CUTOFF)
        snd, rcv, d = _directed_edges(pos, i, j, cfg.box)
    elif cfg.geometry == "molecules":
        per = cfg.n_atoms // cfg.n_graphs
        pos = rng.normal(0.0, 1.5, size=(cfg.n_atoms, 3))
        ss, rr, dd = [], [], []
        for gidx in range(cfg.n_graphs):
            p = pos[gidx * per:(gidx + 1) * per]
            i, j = _pairs_open(p, CUTOFF)
            s_, r_, d_ = _directed_edges(p, i, j, 0.0)
            ss.append(s_ + gidx * per); rr.append(r_ + gidx * per); dd.append(d_)
        snd = np.concatenate(ss).astype(np.int32)
        rcv = np.concatenate(rr).astype(np.int32)
        d = np.concatenate(dd)
    else:
        raise ValueError(cfg.geometry)
    g = Graph(cfg.n_atoms, pos, snd, rcv, d.astype(np.float32), cfg.box)
    return g, rng


# --------------------------------------------------------------------------------------
# tensors
# --------------------------------------------------------------------------------------
def round_to_storage(a64: np.ndarray, storage: str) -> np.ndarray:
    """Round fp64 draws once to the storage dtype; returned as fp32 holding exactly the stored values."""
    a = a64.astype(np.float32)
    if storage == "bf16":
        b = a.view(np.uint32)
        b = ((b + 0x7FFF + ((b >> 16) & 1)) >> 16) << 16
        a = b.astype(np.uint32).view(np.float32)
    elif storage != "f32":
        raise ValueError(storage)
    return a


def in_dim(cfg: Config) -> int:
    return sum(2 * l + 1 for l, _ in cfg.irreps_in)


def w_sigma(cfg: Config, n_paths: int) -> float:
    return 1.0 / math.sqrt(n_paths) if cfg.w_std == "1/sqrt(P)" else 1.0


def draw_x(cfg: Config, rng) -> np.ndarray:
    """Node features x[N, in_dim*C] ~ N(0,1), layout m*C + u inside each irrep block (A7)."""
    return round_to_storage(rng.normal(size=(cfg.n_atoms, in_dim(cfg) * cfg.channels)), cfg.storage)


def draw_w(cfg: Config, rng, n_edges: int, n_paths: int) -> np.ndarray:
    """Per-edge, per-path, per-channel weights w[E, P*C] (host draw; small configs only)."""
    if n_edges * n_paths * cfg.channels > 2_000_000_000:
        raise MemoryError("host weight draw too large; use draw_w_device")
    w = rng.normal(size=(n_edges, n_paths * cfg.channels)) * w_sigma(cfg, n_paths)
    return round_to_storage(w, cfg.storage)


def draw_g(cfg: Config, rng, out_dim: int) -> np.ndarray:
    """Output cotangent G[N, out_dim*C] ~ N(0,1) fp32 (reading A13: E = sum G*out)."""
    return rng.normal(size=(cfg.n_atoms, out_dim * cfg.channels)).astype(np.float32)


def draw_w_device(cfg: Config, n_edges: int, n_paths: int, device):
    """Weights for configs whose w does not fit the host (cfg4/5: 45.6 GB): drawn on the device by
    torch's seeded Philox generator in row chunks, rounded once to the storage dtype.  The oracle is
    given rows copied back from this very tensor, so both sides still see identical stored values."""
    import torch
    dt = torch.bfloat16 if cfg.storage == "bf16" else torch.float32
    gen = torch.Generator(device=device)
    gen.manual_seed(cfg.seed)
    cols = n_paths * cfg.channels
    w = torch.empty((n_edges, cols), dtype=dt, device=device)
    chunk = max(1, (1 << 28) // cols)
    sig = w_sigma(cfg, n_paths)
    for a in range(0, n_edges, chunk):
        b = min(n_edges, a + chunk)
        t = torch.randn((b - a, cols), generator=gen, device=device, dtype=torch.float32)
        w[a:b] = (t * sig).to(dt)
    return w
