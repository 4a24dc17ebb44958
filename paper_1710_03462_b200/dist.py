"""NEXT-4: the path across several GPUs; one process per GPU, torch.distributed for the plumbing.

Steps, transposes and the energy shard by particle index with NO data-path collective (particles are independent;
the paper itself runs on one processor).  Two places need an exchange:

  * the energy: one 8-byte partial per rank, all-gathered and summed in RANK ORDER (deterministic, unlike a tree
    all-reduce whose order may change with the algorithm NCCL picks);
  * binning: after it, every GPU must own a contiguous range of cells.  `bin_exchange` does it in one exchange step,
    with the particles travelling as ARRAY-OF-STRUCTS records -- the use the paper names for the AoS view of an SoA:
    "MPI transfer of particle objects":
        1. local soax_bin_permute: this rank's particles sorted by cell (stable) + its per-cell counts;
        2. all-reduce of the counts (G^3 uint32 -> int64, 2 MB for G = 64); every rank derives the same split of the
           cell range into `world` contiguous pieces holding about N/world particles each (`split_cells`);
        3. because the local set is sorted by cell, what goes to rank r is ONE contiguous slice of every array:
           soax_soa_to_aos packs the sorted set into 40-byte records and a single all_to_all_single (NCCL over
           NVLink 5 / NVSwitch: every peer is one hop away, so the flat all-to-all is the right shape) moves them;
        4. the received records are `world` sorted runs in rank order: soax_aos_to_soa + one more local
           soax_bin_permute merges them.  Stability makes the result unique: within a cell, particles are ordered by
           (source rank, source index), i.e. exactly the stable sort of the rank-major concatenation of all inputs.

The exchange logic below touches no particle data itself: it works on counts and byte offsets, and calls an ENGINE for
the device work.  `SoaxEngine` is the product engine (the CUDA library through container.Soax); the CPU tests drive the
same logic under a world-size-2 gloo group with a stand-in engine.  Only one GPU is available to this repository's
tests, so the NCCL path is exercised at world size 1 on the GPU and at world size 2 on CPU (gloo).
"""
from __future__ import annotations

from typing import Protocol, Sequence

import torch
import torch.distributed as dist


# ---- pure host logic ---------------------------------------------------------------------------------------------------
def split_cells(global_counts: torch.Tensor, world: int) -> list[int]:
    """Boundaries b[0..world] of contiguous cell ranges [b[r], b[r+1]) balanced by particle count: b[r] is the smallest
    boundary with at least ceil(r*N/world) particles to its left.  Every rank computes the same list from the same
    all-reduced counts.  Ranges may be empty when a few cells hold most particles."""
    c = global_counts.to(torch.int64).cpu()
    ncell, total = c.numel(), int(c.sum())
    exc = torch.zeros(ncell + 1, dtype=torch.int64)
    exc[1:] = torch.cumsum(c, 0)
    targets = torch.tensor([(r * total + world - 1) // world for r in range(1, world)], dtype=torch.int64)
    inner = torch.searchsorted(exc, targets, right=False).tolist() if world > 1 else []
    return [0] + [int(b) for b in inner] + [ncell]


def send_counts(local_counts: torch.Tensor, bounds: Sequence[int]) -> list[int]:
    """Number of this rank's particles whose cell falls in each range (its sorted set is cut at these prefix sums)."""
    c = local_counts.to(torch.int64).cpu()
    exc = torch.zeros(c.numel() + 1, dtype=torch.int64)
    exc[1:] = torch.cumsum(c, 0)
    return [int(exc[bounds[r + 1]] - exc[bounds[r]]) for r in range(len(bounds) - 1)]


def shard_sizes(n: int, world: int) -> list[int]:
    """Contiguous index shards of n particles (the step / transpose / energy decomposition)."""
    return [(n * (r + 1)) // world - (n * r) // world for r in range(world)]


# ---- the engine: what the exchange needs from the device -------------------------------------------------------------------
class Engine(Protocol):
    stride: int      # bytes of one packed AoS record
    ncell: int

    def local_sort(self) -> tuple[torch.Tensor, torch.Tensor]:
        """-> (per-cell counts of this rank [ncell], the rank's particles sorted by cell as packed records [n*stride] uint8)"""

    def merge(self, records: torch.Tensor, n: int) -> object:
        """records: n packed records (sorted runs in rank order) -> the final local container, stably sorted by cell"""


class SoaxEngine:
    """The product engine: every step is a call into libsoax.so on this rank's GPU."""

    def __init__(self, src, grid_dim: int, drift_dt: float = 0.0):
        from . import binding as B, container as Cn
        self._B, self._Cn = B, Cn
        self.src, self.grid_dim, self.drift_dt = src, grid_dim, drift_dt
        self.ncell = grid_dim ** 3
        self.stride, _ = B.soax_layout_aos(src.layout, True)
        self.kinetic = None

    def local_sort(self):
        tmp = self._Cn.Soax(self.src.fields, 0, capacity=max(self.src.n, 1))
        r = self.src.bin_permute(tmp, self.grid_dim, drift_dt=self.drift_dt, want_kinetic=self.drift_dt != 0.0)
        self.kinetic = r["kinetic"]
        return r["counts"].to(torch.int64), tmp.to_aos()

    def merge(self, records: torch.Tensor, n: int):
        tmp = self._Cn.Soax(self.src.fields, 0, capacity=max(n, 1))
        tmp.from_aos(records, n)
        out = self._Cn.Soax(self.src.fields, 0, capacity=max(n, 1))
        r = tmp.bin_permute(out, self.grid_dim)
        return out, r["counts"], r["offsets"]


# ---- the exchange -------------------------------------------------------------------------------------------------------------
def bin_exchange(engine: Engine, group=None):
    """One binning step across the group (see the module docstring).  Returns (engine.merge(...) result, bounds, n_local):
    this rank then owns the cells [bounds[rank], bounds[rank+1])."""
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    counts, records = engine.local_sort()
    dev = records.device
    global_counts = counts.clone()
    dist.all_reduce(global_counts, op=dist.ReduceOp.SUM, group=group)
    bounds = split_cells(global_counts, world)
    n_send = send_counts(counts, bounds)
    t_send = torch.tensor(n_send, dtype=torch.int64, device=dev)
    t_recv = torch.empty(world, dtype=torch.int64, device=dev)
    dist.all_to_all_single(t_recv, t_send, group=group)
    n_recv = [int(x) for x in t_recv.cpu()]
    expect = int(global_counts.cpu()[bounds[rank]:bounds[rank + 1]].sum())
    assert sum(n_recv) == expect, "received particle count differs from the all-reduced cell counts"
    s = engine.stride
    recv = torch.empty(max(sum(n_recv) * s, 16), dtype=torch.uint8, device=dev)
    dist.all_to_all_single(recv[:sum(n_recv) * s], records[:sum(n_send) * s], output_split_sizes=[k * s for k in n_recv],
                           input_split_sizes=[k * s for k in n_send], group=group)
    return engine.merge(recv, sum(n_recv)), bounds, sum(n_recv)


def energy_sum(local_energy: torch.Tensor, group=None) -> float:
    """Total energy of the group: the 8-byte partials are gathered and added in rank order (deterministic)."""
    world = dist.get_world_size(group)
    parts = [torch.empty_like(local_energy) for _ in range(world)]
    dist.all_gather(parts, local_energy, group=group)
    total = 0.0
    for p in parts:
        total += float(p)
    return total
