"""NEXT-4: the path across several GPUs; one process per GPU, torch.distributed for the plumbing.

Steps, transposes and the energy shard by particle index with NO data-path collective (particles are independent;
the paper itself runs on one processor).  Three places need an exchange:

  * the energy: one 8-byte partial per rank, all-gathered and summed in RANK ORDER (deterministic, unlike a tree
    all-reduce whose order may change with the algorithm NCCL picks);
  * binning (`bin_exchange`): after it, every GPU must own a contiguous range of cells.  One exchange step, with the
    particles travelling as ARRAY-OF-STRUCTS records -- the use the paper names for the AoS view of an SoA: "MPI transfer
    of particle objects":
        1. local soax_bin_permute: this rank's particles sorted by cell (stable) + its per-cell counts;
        2. ONE all-gather of the per-cell counts (world x G^3 int64; 2 MB per rank for G = 64).  From it every rank derives,
           ON THE DEVICE, the same split of the cell range into `world` contiguous pieces holding about N/world particles
           each (`plan_exchange`: cumulative sum + searchsorted), what it sends to every rank and what it receives from
           every rank; one small tensor (3 world + 1 integers) crosses to the host -- the only host round trip;
        3. because the local set is sorted by cell, what goes to rank r is ONE contiguous slice of every array:
           soax_soa_to_aos packs the sorted set into 40-byte records and a single all_to_all_single (NCCL over
           NVLink 5 / NVSwitch: every peer is one hop away, so the flat all-to-all is the right shape) moves them;
        4. the received records are `world` sorted runs in rank order whose per-cell counts are already known (the
           all-gather): the merge is ONE segmented gather (soax_gather_segments_aos: 40 B read + 40 B written per particle)
           instead of a transpose plus a second full sort.  Stability makes the result unique: within a cell, particles are ordered by
           (source rank, source index), i.e. exactly the stable sort of the rank-major concatenation of all inputs.
  * per-step migration (`migrate`): after an integration step the particles whose cell left this rank's range
    [bounds[rank], bounds[rank+1]) are flagged ON THE DEVICE (a mask program, soax_expr_mask), copied out in order
    (soax_remove STABLE with the complementary mask), removed in place by the paper's overwrite-with-last (soax_remove
    SWAP_LAST: only as many rows move as particles leave), sorted by cell (soax_bin_permute on the few
    leavers, so that each destination's share is one contiguous slice), shipped as AoS records in ONE all_to_all and
    appended by the receiver (soax_push_back_aos).  The result is deterministic: the stayers in the
    overwrite-with-last arrangement, then the arrivals by source rank, each rank's in (cell, source order).

The exchange logic below touches no particle data itself: it works on counts and byte offsets, and calls an ENGINE for
the device work.  `SoaxEngine` is the product engine (the CUDA library through container.Soax).  The collectives go
through `_all_gather` / `_all_to_all`, which stage device tensors through host memory when the group's backend cannot
move them (gloo): that is how the tests run the PRODUCT engine in a real 2-rank exchange with both ranks on the one GPU
this repository's tests ever see (host-level collectives only: no kernel of one rank waits for another rank).
No multi-GPU timing exists: unmeasured on hardware.
"""
from __future__ import annotations

from typing import Protocol, Sequence

import torch
import torch.distributed as dist


# ---- collectives: NCCL moves device tensors; any other backend gets them staged through the host ---------------------------
def _all_gather(t: torch.Tensor, group=None) -> torch.Tensor:
    """-> tensor [world, *t.shape] on t's device"""
    world = dist.get_world_size(group)
    if dist.get_backend(group) == "nccl":
        out = torch.empty((world,) + tuple(t.shape), dtype=t.dtype, device=t.device)
        dist.all_gather_into_tensor(out, t.contiguous(), group=group)
        return out
    src = t.cpu().contiguous()
    parts = [torch.empty_like(src) for _ in range(world)]
    dist.all_gather(parts, src, group=group)
    return torch.stack(parts).to(t.device)


def _all_to_all(recv: torch.Tensor, send: torch.Tensor, recv_splits: Sequence[int], send_splits: Sequence[int], group=None) -> None:
    if dist.get_backend(group) == "nccl":
        dist.all_to_all_single(recv, send, output_split_sizes=list(recv_splits), input_split_sizes=list(send_splits), group=group)
        return
    r = torch.empty(recv.shape, dtype=recv.dtype)
    _all_to_all_by_gather(r, send.cpu(), recv_splits, send_splits, group)
    recv.copy_(r)


def _all_to_all_by_gather(recv: torch.Tensor, send: torch.Tensor, recv_splits, send_splits, group) -> None:
    """all-to-all out of all-gathers of padded buffers (CPU tensors, tests only): every rank publishes its whole send
    buffer and its split sizes; each rank picks its pieces."""
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    splits = torch.tensor(list(send_splits), dtype=torch.int64)
    all_splits = [torch.empty_like(splits) for _ in range(world)]
    dist.all_gather(all_splits, splits, group=group)
    most = max(int(s.sum()) for s in all_splits)
    padded = torch.zeros(max(most, 1), dtype=send.dtype)
    padded[:send.numel()] = send.reshape(-1)
    bufs = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(bufs, padded, group=group)
    at = 0
    for q in range(world):
        start = int(all_splits[q][:rank].sum())
        k = int(all_splits[q][rank])
        assert k == recv_splits[q]
        recv.reshape(-1)[at:at + k] = bufs[q][start:start + k]
        at += k


# ---- pure count logic (host or device tensors) ------------------------------------------------------------------------------
def split_cells(global_counts: torch.Tensor, world: int) -> list[int]:
    """Boundaries b[0..world] of contiguous cell ranges [b[r], b[r+1]) balanced by particle count: b[r] is the smallest
    boundary with at least ceil(r*N/world) particles to its left.  Every rank computes the same list from the same
    counts.  Ranges may be empty when a few cells hold most particles."""
    return [int(x) for x in _bounds(global_counts.to(torch.int64), world).cpu()]


def _bounds(global_counts: torch.Tensor, world: int) -> torch.Tensor:
    """split_cells on the device of `global_counts`: int64 tensor [world + 1]"""
    c = global_counts
    ncell = c.numel()
    exc = torch.zeros(ncell + 1, dtype=torch.int64, device=c.device)
    exc[1:] = torch.cumsum(c, 0)
    total = exc[-1]
    r = torch.arange(1, world, dtype=torch.int64, device=c.device)
    targets = (r * total + (world - 1)) // world
    inner = torch.searchsorted(exc, targets, right=False)
    return torch.cat([torch.zeros(1, dtype=torch.int64, device=c.device), inner, torch.full((1,), ncell, dtype=torch.int64, device=c.device)])


def send_counts(local_counts: torch.Tensor, bounds: Sequence[int]) -> list[int]:
    """Number of this rank's particles whose cell falls in each range (its sorted set is cut at these prefix sums)."""
    c = local_counts.to(torch.int64).cpu()
    exc = torch.zeros(c.numel() + 1, dtype=torch.int64)
    exc[1:] = torch.cumsum(c, 0)
    return [int(exc[bounds[r + 1]] - exc[bounds[r]]) for r in range(len(bounds) - 1)]


def plan_exchange(all_counts: torch.Tensor, rank: int, bounds: torch.Tensor | None = None):
    """all_counts: int64 [world, ncell] (every rank's per-cell counts, on any device).  Computes on that device and returns,
    after ONE transfer to the host, (bounds [world+1], n_send [world], n_recv [world]) as lists of ints: the cell ranges
    (or the given ones), how many of this rank's particles go to every rank, and how many it receives from every rank."""
    world, ncell = all_counts.shape
    b = _bounds(all_counts.sum(0), world) if bounds is None else bounds.to(all_counts.device)
    exc = torch.zeros((world, ncell + 1), dtype=torch.int64, device=all_counts.device)
    exc[:, 1:] = torch.cumsum(all_counts, 1)
    at = exc[:, b]                                             # [world, world + 1]: rank q's particles left of boundary r
    per = at[:, 1:] - at[:, :-1]                               # per[q, r] = particles of rank q in range r
    packed = torch.cat([b, per[rank], per[:, rank]]).cpu()     # the one host round trip
    vals = [int(x) for x in packed]
    return vals[:world + 1], vals[world + 1:2 * world + 1], vals[2 * world + 1:]


def shard_sizes(n: int, world: int) -> list[int]:
    """Contiguous index shards of n particles (the step / transpose / energy decomposition)."""
    return [(n * (r + 1)) // world - (n * r) // world for r in range(world)]


# ---- the engine: what the exchange needs from the device -------------------------------------------------------------------
class Engine(Protocol):
    stride: int      # bytes of one packed AoS record
    ncell: int

    def local_sort(self) -> tuple[torch.Tensor, torch.Tensor]:
        """-> (per-cell counts of this rank [ncell], the rank's particles sorted by cell as packed records [n*stride] uint8)"""

    def merge(self, records: torch.Tensor, n: int, run_counts: torch.Tensor, lo: int) -> object:
        """records: n packed records = `world` runs in rank order, each sorted by cell; run_counts [world, hi - lo]: the
        number of records of every cell of this rank's range [lo, hi) in every run -> the final local container, stably
        sorted by cell"""


class SoaxEngine:
    """The product engine: every step is a call into libsoax.so on this rank's GPU."""

    def __init__(self, src, grid_dim: int, drift_dt: float = 0.0):
        from . import binding as B, container as Cn
        self._B, self._Cn = B, Cn
        self.src, self.grid_dim, self.drift_dt = src, grid_dim, drift_dt
        self.ncell = grid_dim ** 3
        self.stride, _ = B.soax_layout_aos(src.layout, True)
        self.kinetic = None
        self._masks = {}

    def local_sort(self):
        """With drift_dt != 0 the drift happens on the way into the sorted copy: soax_bin_permute leaves `src` READ ONLY
        (Q22), so after this call self.src still holds the PRE-drift positions while the records handed to the
        exchange are the drifted ones.  self.src is stale from here on; the state of the step is what `merge` returns."""
        tmp = self._Cn.Soax(self.src.fields, 0, capacity=max(self.src.n, 1))
        r = self.src.bin_permute(tmp, self.grid_dim, drift_dt=self.drift_dt, want_kinetic=self.drift_dt != 0.0)
        self.kinetic = r["kinetic"]
        return r["counts"].to(torch.int64), tmp.to_aos()

    def merge(self, records: torch.Tensor, n: int, run_counts: torch.Tensor, lo: int):
        """The runs are sorted and their per-cell counts are known, so the merge is ONE segmented gather (80 B/particle):
        segment (cell c, run q) goes to [sum of the counts before it in (cell, run) order) and comes from run q's slice
        of cell c.  The two tables are built from counts with torch (plumbing); the records move in libsoax.so."""
        cnt = run_counts.to(records.device)                          # [world, m]
        run_start = torch.cumsum(cnt.sum(1), 0) - cnt.sum(1)
        src_start = run_start[:, None] + torch.cumsum(cnt, 1) - cnt
        flat = cnt.t().reshape(-1)
        seg_dst = (torch.cumsum(flat, 0) - flat).to(torch.int32)
        seg_src = src_start.t().reshape(-1).to(torch.int32)
        out = self._Cn.Soax(self.src.fields, 0, capacity=max(n, 1))
        out.from_aos_segments(records, seg_dst, seg_src, n)
        counts = torch.zeros(self.ncell, dtype=torch.int64, device=records.device)
        counts[lo:lo + cnt.shape[1]] = cnt.sum(0)
        offsets = torch.cumsum(counts, 0) - counts
        return out, counts.to(torch.int32), offsets.to(torch.int32)

    # ---- migration (every device step is a libsoax.so call) ----------------------------------------------------------------
    def _mask(self, cond: str):
        if cond not in self._masks:
            self._masks[cond] = self._Cn.MaskProgram(self.src.fields, cond, ["lo", "hi"])
        return self._masks[cond]

    def take_leavers(self, s, lo: int, hi: int):
        """Removes from `s` (in place, overwrite-with-last) the particles whose cell is outside [lo, hi); returns
        (per-cell counts of the leavers [ncell], the leavers sorted by cell as packed records, their number)."""
        G = self.grid_dim
        leave = self._mask(f"(double(cell({G})) < lo) | (double(cell({G})) >= hi)").mask(s, lo=lo, hi=hi)
        out = self._Cn.Soax(s.fields, 0, capacity=max(s.n, 1))
        s.remove_async(leave, stable=True, dst=out, keep_flagged=True)   # the leavers, in order (the flagged ones are KEPT)
        s.remove_async(leave)                                        # the holes are filled from the end
        m = out.n
        srt = self._Cn.Soax(s.fields, 0, capacity=max(m, 1))
        r = out.bin_permute(srt, G)                                  # few rows: each destination's share becomes one slice
        return r["counts"].to(torch.int64), srt.to_aos(), m

    def append(self, s, records: torch.Tensor, n: int) -> None:
        s.push_back_aos(records, n)


# ---- the exchanges ------------------------------------------------------------------------------------------------------------
def _ship(engine: Engine, counts: torch.Tensor, records: torch.Tensor, group, bounds: torch.Tensor | None):
    """the all-gather of the counts, the plan, and the one all-to-all of the records; returns (recv buffer, n_recv list,
    bounds list, all_counts)"""
    rank = dist.get_rank(group)
    all_counts = _all_gather(counts, group)
    b, n_send, n_recv = plan_exchange(all_counts, rank, bounds)
    s = engine.stride
    recv = torch.empty(max(sum(n_recv) * s, 16), dtype=torch.uint8, device=records.device)
    timed = records.is_cuda                                       # measurement aid (bench.py): events around the one all-to-all
    ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) if timed else None
    if timed:
        ev[0].record()
    _all_to_all(recv[:sum(n_recv) * s], records[:sum(n_send) * s], [k * s for k in n_recv], [k * s for k in n_send], group)
    if timed:
        ev[1].record()
    try:
        engine.last_ship = {"n_send": n_send, "n_recv": n_recv, "events": ev, "stride": s}
    except AttributeError:
        pass
    return recv, n_recv, b, all_counts


def bin_exchange(engine: Engine, group=None):
    """One binning step across the group (see the module docstring).  Returns (engine.merge(...) result, bounds, n_local):
    this rank then owns the cells [bounds[rank], bounds[rank+1]).  One host round trip (the split sizes)."""
    rank = dist.get_rank(group)
    counts, records = engine.local_sort()
    recv, n_recv, bounds, all_counts = _ship(engine, counts, records, group, None)
    lo, hi = bounds[rank], bounds[rank + 1]
    return engine.merge(recv, sum(n_recv), all_counts[:, lo:hi], lo), bounds, sum(n_recv)


def migrate(engine: SoaxEngine, s, bounds: Sequence[int], group=None) -> int:
    """Per-step migration: the particles of `s` whose cell left [bounds[rank], bounds[rank+1]) move to the rank that owns
    their cell; arrivals are appended.  Returns the new local particle count."""
    rank = dist.get_rank(group)
    counts, records, _ = engine.take_leavers(s, bounds[rank], bounds[rank + 1])
    recv, n_recv, _, _ = _ship(engine, counts, records, group, torch.tensor(list(bounds), dtype=torch.int64))
    if sum(n_recv):
        engine.append(s, recv, sum(n_recv))
    return s.n


def energy_sum(local_energy: torch.Tensor, group=None) -> float:
    """Total energy of the group: the 8-byte partials are gathered and added in rank order (deterministic)."""
    parts = _all_gather(local_energy.reshape(1), group)
    total = 0.0
    for p in parts.cpu():
        total += float(p)
    return total
