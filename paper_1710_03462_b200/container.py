"""Device plumbing around the C ABI: torch owns the device memory and the streams, the library does the work.

`Soax` holds one torch uint8 slab carved by soax_alloc into per-component arrays and forwards
every operation to the soax_* calls of binding.py.  Nothing here computes on particles.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B

# layouts as (name, soax_dtype, dim) lists, declaration order (BASELINE.json config 4)
R1 = (("id", B.SOAX_I32, 1), ("pos", B.SOAX_F64, 3), ("vel", B.SOAX_F32, 3))
R1R = (("pos", B.SOAX_F64, 3), ("vel", B.SOAX_F32, 3), ("id", B.SOAX_I32, 1))      # Q1 sensitivity row: naturally aligned AoS
R2 = (("id", B.SOAX_I64, 1), ("pos", B.SOAX_F64, 3), ("vel", B.SOAX_F64, 3), ("acc", B.SOAX_F64, 3),
      ("mass", B.SOAX_F32, 1), ("charge", B.SOAX_F32, 1), ("flags", B.SOAX_U8, 1))


def B6(size_extra: int):
    base = (("pos", B.SOAX_F32, 3), ("vel", B.SOAX_F32, 3))
    return base if size_extra == 0 else base + (("temp", B.SOAX_F32, size_extra),)


NP_DTYPE = {B.SOAX_I32: np.int32, B.SOAX_I64: np.int64, B.SOAX_U8: np.uint8, B.SOAX_F32: np.float32, B.SOAX_F64: np.float64}
TORCH_DTYPE = {B.SOAX_I32: torch.int32, B.SOAX_I64: torch.int64, B.SOAX_U8: torch.uint8, B.SOAX_F32: torch.float32,
               B.SOAX_F64: torch.float64}


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


class Soax:
    """An SoA particle container on the current CUDA device (the paper's `Soax<ArrayTypes> soax(n)`)."""

    def __init__(self, fields, n: int, capacity: int | None = None, device="cuda", dynamic: bool = False):
        self.fields = tuple(fields)
        self.layout = (B.soax_layout_define_dynamic if dynamic else B.soax_layout_define)(self.fields)
        self.capacity = n if capacity is None else capacity
        self.slab_bytes = B.soax_slab_bytes(self.layout, self.capacity)
        self.slab = torch.empty(self.slab_bytes, dtype=torch.uint8, device=device)
        self.handle = B.soax_alloc(self.layout, n, self.capacity, self.slab.data_ptr(), self.slab_bytes)
        self.ncomp = B.soax_layout_ncomp(self.layout)
        self.comp_dtype = [B.soax_layout_comp(self.layout, c)[2] for c in range(self.ncomp)]
        self._escratch = None

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h:
            try:
                B.soax_free(h)
            except Exception:
                pass

    @property
    def n(self) -> int:
        return B.soax_size(self.handle)

    # ---- views ---------------------------------------------------------------------------------------------
    def field_index(self, name: str) -> int:
        return [f[0] for f in self.fields].index(name)

    def comp_view(self, field: str | int, comp: int = 0) -> torch.Tensor:
        """torch view (no copy) of one component array: the paper's posArr(c)."""
        f = self.field_index(field) if isinstance(field, str) else field
        ptr = B.soax_field_ptr(self.handle, f, comp)
        dt = self.fields[f][1]
        off = ptr - self.slab.data_ptr()
        return self.slab[off:off + self.n * B.DTYPE_SIZE[dt]].view(TORCH_DTYPE[dt])

    # ---- host <-> device through the C ABI (end-to-end path) ---------------------------------------------------
    def _host_ptrs(self, host: dict, writable: bool):
        ptrs, keep = [], []
        for name, dt, dim in self.fields:
            a = host.get(name)
            for c in range(dim):
                if a is None:
                    ptrs.append(None)
                    continue
                row = a[c]
                if isinstance(row, torch.Tensor):
                    assert row.is_contiguous() and row.dtype == TORCH_DTYPE[dt]
                    ptrs.append(row.data_ptr())
                else:
                    assert row.flags["C_CONTIGUOUS"] and row.dtype == NP_DTYPE[dt] and (row.flags["WRITEABLE"] or not writable)
                    ptrs.append(row.ctypes.data)
                keep.append(row)
        return ptrs, keep

    def upload(self, host: dict, n: int | None = None) -> None:
        """host: name -> (dim, N) numpy array or (pinned) torch CPU tensor, component-major."""
        n = next(iter(host.values())).shape[1] if n is None else n
        ptrs, keep = self._host_ptrs(host, writable=False)
        B.soax_upload(self.handle, ptrs, n, _stream())
        torch.cuda.current_stream().synchronize()      # pageable sources must outlive the copy
        del keep

    def download(self, into: dict | None = None) -> dict:
        n = self.n
        out = into if into is not None else {name: np.empty((dim, n), NP_DTYPE[dt]) for name, dt, dim in self.fields}
        ptrs, keep = self._host_ptrs(out, writable=True)
        B.soax_download(self.handle, ptrs, n, _stream())
        torch.cuda.current_stream().synchronize()
        del keep
        return out

    # ---- hot path ---------------------------------------------------------------------------------------------------
    def step(self, kind: int, dt: float, nsteps: int = 1, k: float = 1.0, center: float = 0.5, flag_mask: int = 1) -> None:
        B.soax_step(self.handle, B.step_params(kind, dt, k, center, flag_mask), nsteps, _stream())

    def energy_async(self, kind: int, k: float = 1.0, center: float = 0.5, out: torch.Tensor | None = None) -> torch.Tensor:
        if self._escratch is None:
            self._escratch = torch.empty(B.soax_energy_scratch_bytes(), dtype=torch.uint8, device=self.slab.device)
        out = torch.empty(1, dtype=torch.float64, device=self.slab.device) if out is None else out
        B.soax_reduce_energy(self.handle, kind, k, center, self._escratch.data_ptr(), self._escratch.numel(),
                             out.data_ptr(), _stream())
        return out

    def energy(self, kind: int, k: float = 1.0, center: float = 0.5) -> float:
        return float(self.energy_async(kind, k, center).item())

    def from_aos(self, aos: torch.Tensor, n: int) -> None:
        B.soax_aos_to_soa(self.handle, aos.data_ptr(), n, _stream())

    def to_aos(self, aos: torch.Tensor | None = None) -> torch.Tensor:
        stride, _ = B.soax_layout_aos(self.layout, True)
        n = self.n
        aos = torch.empty(n * stride, dtype=torch.uint8, device=self.slab.device) if aos is None else aos
        B.soax_soa_to_aos(self.handle, aos.data_ptr(), n, _stream())
        return aos

    def bin_permute(self, dst: "Soax", grid_dim: int, drift_dt: float = 0.0, want_kinetic: bool = False,
                    scratch: torch.Tensor | None = None, inplace: bool = False) -> dict:
        """Returns device tensors: counts, offsets (uint32 as int32 views), perm, and kinetic (or None).
        inplace: the sorted set returns to self and `dst` is only a work container (soax_bin_permute_inplace)."""
        dev, n = self.slab.device, self.n
        ncell = grid_dim ** 3
        need = (B.soax_scratch_bytes_inplace if inplace else B.soax_scratch_bytes)(self.layout, n, grid_dim)
        if scratch is None:
            scratch = torch.empty(need, dtype=torch.uint8, device=dev)
        counts = torch.empty(ncell, dtype=torch.int32, device=dev)
        offsets = torch.empty(ncell, dtype=torch.int32, device=dev)
        perm = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
        kin = torch.empty(1, dtype=torch.float64, device=dev) if want_kinetic else None
        (B.soax_bin_permute_inplace if inplace else B.soax_bin_permute)(
            self.handle, dst.handle, grid_dim, drift_dt, counts.data_ptr(), offsets.data_ptr(), perm.data_ptr(),
            None if kin is None else kin.data_ptr(), scratch.data_ptr(), scratch.numel(), _stream())
        return {"counts": counts, "offsets": offsets, "perm": perm[:n], "kinetic": kin, "scratch": scratch}


    # ---- container operations (NEXT-3) --------------------------------------------------------
    def remove(self, kill: torch.Tensor, stable: bool = False, dst: "Soax | None" = None, scratch: torch.Tensor | None = None) -> int:
        """kill: uint8 device tensor, one byte per live particle, non-zero = remove.  Unstable (the paper's overwrite
        with the last element) works in place; stable compacts into `dst`.  Returns the survivor count."""
        assert kill.dtype == torch.uint8 and kill.is_contiguous() and kill.numel() >= self.n
        need = B.soax_remove_scratch_bytes(self.n)
        if scratch is None:
            scratch = torch.empty(max(need, 256), dtype=torch.uint8, device=self.slab.device)
        self.remove_async(kill, stable=stable, dst=dst, scratch=scratch)
        return (dst if stable else self).n                      # soax_size waits for the count, not for the rows

    def remove_async(self, kill: torch.Tensor, stable: bool = False, dst: "Soax | None" = None, scratch: torch.Tensor | None = None,
                     keep_flagged: bool = False) -> None:
        """soax_remove without touching the count: nothing waits, the handle learns its new size when it is next needed.
        keep_flagged: the mask marks the particles that STAY (SOAX_REMOVE_KEEP_FLAGGED)."""
        need = B.soax_remove_scratch_bytes(self.n)
        if scratch is None:
            scratch = torch.empty(max(need, 256), dtype=torch.uint8, device=self.slab.device)
        self._remove_scratch = scratch                          # keep it alive until the enqueued kernels have run
        B.soax_remove(self.handle, dst.handle if stable else None, kill.data_ptr(),
                      (B.SOAX_REMOVE_STABLE if stable else B.SOAX_REMOVE_SWAP_LAST) | (B.SOAX_REMOVE_KEEP_FLAGGED if keep_flagged else 0),
                      scratch.data_ptr(), scratch.numel(), _stream())

    def remove_stable_noalloc(self, kill: torch.Tensor, dst: "Soax", count: torch.Tensor, keep_flagged: bool = False) -> None:
        """soax_remove_stable_noalloc: the stable removal for callers that may not allocate -- no scratch is passed and the
        library allocates none (its work area is built into libsoax.so; at most B.SOAX_NOALLOC_MAX_N particles).  `count`:
        a one-element int64 device tensor of the caller that receives the survivor count; dst's live count is NOT updated
        (that needs the count on the host): after synchronising, call B.soax_resize(dst.handle, int(count))."""
        assert kill.dtype == torch.uint8 and kill.is_contiguous() and kill.numel() >= self.n
        assert count.dtype == torch.int64 and count.is_cuda and count.numel() >= 1
        B.soax_remove_stable_noalloc(self.handle, dst.handle, kill.data_ptr(), keep_flagged, count.data_ptr(), _stream())

    def reserve(self, capacity: int) -> None:
        """Regrow (the paper's resize / push_back grow every array).  The C ABI never allocates -- the
        caller owns device memory -- so growing is done here, on the caller's side: a new torch slab of at least
        max(capacity, 1.5 x the old capacity) particles, soax_alloc over it, ONE soax_copy of the live particles (a device
        copy of every component array, enqueued on the current stream), then the handle and the slab are swapped and the old
        handle is freed.  The old slab goes back to torch's allocator, which orders its reuse after the copy on this stream.
        Views from comp_view() and graphs captured for the old arrays do not follow (graph keys hold the array addresses and
        the allocation serial, so they invalidate themselves).  No-op if the capacity already suffices."""
        if capacity <= self.capacity:
            return
        new_cap = max(int(capacity), self.capacity + self.capacity // 2, 1)
        slab_bytes = B.soax_slab_bytes(self.layout, new_cap)
        slab = torch.empty(slab_bytes, dtype=torch.uint8, device=self.slab.device)
        h = B.soax_alloc(self.layout, 0, new_cap, slab.data_ptr(), slab_bytes)
        try:
            B.soax_copy(h, self.handle, _stream())                  # sets the new handle's live count to the old one's
        except Exception:
            B.soax_free(h)
            raise
        old, self.handle = self.handle, h
        self.slab, self.slab_bytes, self.capacity = slab, slab_bytes, new_cap
        B.soax_free(old)

    def resize(self, n: int) -> None:
        """`soax.resize(n)`: the live count becomes n, growing the arrays first if n exceeds the capacity.
        New rows are uninitialised, as with the paper's arrays."""
        self.reserve(n)
        B.soax_resize(self.handle, n)

    def push_back_aos(self, aos: torch.Tensor, m: int) -> None:
        """`soax.push_back(particle)`, bulk: m packed records are appended; the arrays grow geometrically
        through reserve() when they are full (soax_push_back_aos itself answers ALLOC past the capacity)."""
        self.reserve(self.n + m)
        B.soax_push_back_aos(self.handle, aos.data_ptr(), m, _stream())

    def get_elements(self, idx: torch.Tensor, aos: torch.Tensor | None = None) -> torch.Tensor:
        """idx: int32/uint32 device tensor of row numbers; returns the rows as packed AoS records (uint8 tensor)."""
        assert idx.dtype in (torch.int32, torch.uint32) and idx.is_contiguous()
        stride, _ = B.soax_layout_aos(self.layout, True)
        m = idx.numel()
        aos = torch.empty(max(m * stride, 16), dtype=torch.uint8, device=self.slab.device) if aos is None else aos
        B.soax_get_elements(self.handle, idx.data_ptr(), m, aos.data_ptr(), _stream())
        return aos[:m * stride]

    def from_aos_segments(self, aos: torch.Tensor, seg_dst: torch.Tensor, seg_src: torch.Tensor, n: int) -> None:
        """merge of sorted runs of AoS records as a segmented gather (soax_gather_segments_aos); tables: int32/uint32 device"""
        assert seg_dst.dtype in (torch.int32, torch.uint32) and seg_src.dtype == seg_dst.dtype and seg_dst.numel() == seg_src.numel()
        B.soax_gather_segments_aos(self.handle, aos.data_ptr(), seg_dst.data_ptr(), seg_src.data_ptr(), seg_dst.numel(), n, _stream())

    def copy_from(self, src: "Soax") -> None:
        B.soax_copy(self.handle, src.handle, _stream())


class Program:
    """A fused element-wise program compiled for one layout (soax_expr_compile): the paper's whole-array expressions
    `soax.posArr(0) = soax.velArr(1) - soax.velArr(2)` as ONE generated kernel per program."""

    def __init__(self, fields, source: str, scalar_names=(), dynamic: bool = False):
        self.fields, self.source, self.scalar_names = tuple(fields), source, tuple(scalar_names)
        self.layout = (B.soax_layout_define_dynamic if dynamic else B.soax_layout_define)(self.fields)
        self.handle = B.soax_expr_compile(self.layout, source, self.scalar_names)
        self.bytes_read, self.bytes_written = B.soax_expr_traffic(self.handle)

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h:
            try:
                B.soax_expr_free(h)
            except Exception:
                pass

    @property
    def cuda_source(self) -> str:
        return B.soax_expr_cuda_source(self.handle)

    def run(self, s: Soax, nsteps: int = 1, **scalars) -> None:
        vals = [scalars[k] for k in self.scalar_names]
        B.soax_expr_run(s.handle, self.handle, vals, nsteps, _stream())


class SumProgram:
    """A user-written reduction (soax_expr_compile_sum): the sum over the particles of one expression, in double, with
    the reduction tree of soax_reduce_energy."""

    def __init__(self, fields, expression: str, scalar_names=(), dynamic: bool = False):
        self.fields, self.expression, self.scalar_names = tuple(fields), expression, tuple(scalar_names)
        self.layout = (B.soax_layout_define_dynamic if dynamic else B.soax_layout_define)(self.fields)
        self.handle = B.soax_expr_compile_sum(self.layout, expression, self.scalar_names)
        self.bytes_read, _ = B.soax_expr_traffic(self.handle)
        self._scratch = None

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h:
            try:
                B.soax_expr_free(h)
            except Exception:
                pass

    def sum_async(self, s: Soax, out: torch.Tensor | None = None, **scalars) -> torch.Tensor:
        if self._scratch is None:
            self._scratch = torch.empty(B.soax_energy_scratch_bytes(), dtype=torch.uint8, device=s.slab.device)
        out = torch.empty(1, dtype=torch.float64, device=s.slab.device) if out is None else out
        B.soax_expr_sum(s.handle, self.handle, [scalars[k] for k in self.scalar_names], self._scratch.data_ptr(),
                        self._scratch.numel(), out.data_ptr(), _stream())
        return out

    def sum(self, s: Soax, **scalars) -> float:
        return float(self.sum_async(s, **scalars).item())


class MaskProgram:
    """A user-written condition compiled into a kernel that writes one byte per particle (soax_expr_compile_mask): the kill
    mask soax_remove consumes, produced on the device (e.g. "(flags & 1) != 0", or the particles that left a cell range)."""

    def __init__(self, fields, condition: str, scalar_names=(), dynamic: bool = False):
        self.fields, self.condition, self.scalar_names = tuple(fields), condition, tuple(scalar_names)
        self.layout = (B.soax_layout_define_dynamic if dynamic else B.soax_layout_define)(self.fields)
        self.handle = B.soax_expr_compile_mask(self.layout, condition, self.scalar_names)
        self.bytes_read, self.bytes_written = B.soax_expr_traffic(self.handle)

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h:
            try:
                B.soax_expr_free(h)
            except Exception:
                pass

    @property
    def cuda_source(self) -> str:
        return B.soax_expr_cuda_source(self.handle)

    def mask(self, s: Soax, out: torch.Tensor | None = None, **scalars) -> torch.Tensor:
        n = s.n
        out = torch.empty(max(n, 4), dtype=torch.uint8, device=s.slab.device) if out is None else out
        assert out.dtype == torch.uint8 and out.numel() >= n
        B.soax_expr_mask(s.handle, self.handle, [scalars[k] for k in self.scalar_names], out.data_ptr(), _stream())
        return out[:n]


def aos_step(fields, aos: torch.Tensor, n: int, kind: int, dt: float, nsteps: int = 1, variant: int = 0, k: float = 1.0,
             center: float = 0.5) -> None:
    layout = B.soax_layout_define(fields)
    B.soax_step_aos(layout, aos.data_ptr(), n, B.step_params(kind, dt, k, center), nsteps, variant, _stream())
