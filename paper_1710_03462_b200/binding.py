"""Thin ctypes binding of include/soax.h -- same names, argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind libsoax.so; this module converts Python values to C
arguments and turns negative status codes into SoaxError.  There is no CPU fallback: if the library cannot be
loaded the import fails.  Device pointers are plain ints (torch.Tensor.data_ptr()), streams are ints
(torch.cuda.Stream.cuda_stream), 0 = the legacy default stream.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Sequence

from . import build as _build

SOAX_OK, SOAX_ERR_INVALID_ARG, SOAX_ERR_UNKNOWN_LAYOUT, SOAX_ERR_UNSUPPORTED, SOAX_ERR_ALLOC, SOAX_ERR_CUDA = 0, -1, -2, -3, -4, -5
SOAX_ERR_TOO_LARGE = -6
SOAX_NOALLOC_MAX_N = 1 << 24
SOAX_I32, SOAX_I64, SOAX_U8, SOAX_F32, SOAX_F64 = 0, 1, 2, 3, 4
SOAX_STEP_DRIFT, SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED, SOAX_STEP_EULER_NOWRAP = 0, 1, 2, 3
SOAX_ENERGY_KINETIC, SOAX_ENERGY_KINETIC_PLUS_HARMONIC = 0, 1
SOAX_REMOVE_SWAP_LAST, SOAX_REMOVE_STABLE, SOAX_REMOVE_KEEP_FLAGGED = 0, 1, 4
DTYPE_SIZE = {SOAX_I32: 4, SOAX_I64: 8, SOAX_U8: 1, SOAX_F32: 4, SOAX_F64: 8}


class soax_field(C.Structure):
    _fields_ = [("name", C.c_char_p), ("dtype", C.c_int32), ("dim", C.c_int32)]


class soax_step_params(C.Structure):
    _fields_ = [("kind", C.c_int32), ("flag_mask", C.c_uint8), ("pad_", C.c_uint8 * 3), ("dt", C.c_double),
                ("k", C.c_double), ("center", C.c_double)]


class SoaxError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().soax_strerror(status).decode()
        if status == SOAX_ERR_CUDA:
            msg += f" [cudaError {lib().soax_last_cuda_error()}]"
        super().__init__(f"{where}: {msg} ({status})")


_lib = None

# name -> (restype, argtypes): every symbol include/soax.h declares
_vp, _i64, _i32, _f64, _sz = C.c_void_p, C.c_int64, C.c_int32, C.c_double, C.c_size_t
SIGNATURES = {
    "soax_layout_define": (C.c_int, [C.POINTER(soax_field), _i32, C.POINTER(_vp)]),
    "soax_layout_define_dynamic": (C.c_int, [C.POINTER(soax_field), _i32, C.POINTER(_vp)]),
    "soax_layout_nfields": (C.c_int, [_vp]),
    "soax_layout_ncomp": (C.c_int, [_vp]),
    "soax_layout_comp": (C.c_int, [_vp, _i32, C.POINTER(_i32), C.POINTER(_i32), C.POINTER(_i32)]),
    "soax_layout_aos": (C.c_int, [_vp, _i32, C.POINTER(_sz), C.POINTER(_sz)]),
    "soax_slab_bytes": (_sz, [_vp, _i64]),
    "soax_alloc": (C.c_int, [_vp, _i64, _i64, _vp, _sz, C.POINTER(_vp)]),
    "soax_free": (C.c_int, [_vp]),
    "soax_size": (_i64, [_vp]),
    "soax_resize": (C.c_int, [_vp, _i64]),
    "soax_field_ptr": (C.c_int, [_vp, _i32, _i32, C.POINTER(_vp)]),
    "soax_upload": (C.c_int, [_vp, C.POINTER(_vp), _i64, _vp]),
    "soax_download": (C.c_int, [_vp, C.POINTER(_vp), _i64, _vp]),
    "soax_step": (C.c_int, [_vp, C.POINTER(soax_step_params), _i32, _vp]),
    "soax_step_aos": (C.c_int, [_vp, _vp, _i64, C.POINTER(soax_step_params), _i32, _i32, _vp]),
    "soax_aos_to_soa": (C.c_int, [_vp, _vp, _i64, _vp]),
    "soax_soa_to_aos": (C.c_int, [_vp, _vp, _i64, _vp]),
    "soax_energy_scratch_bytes": (_sz, []),
    "soax_reduce_energy": (C.c_int, [_vp, _i32, _f64, _f64, _vp, _sz, _vp, _vp]),
    "soax_scratch_bytes": (_sz, [_vp, _i64, _i32]),
    "soax_bin_permute": (C.c_int, [_vp, _vp, _i32, _f64, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "soax_scratch_bytes_inplace": (_sz, [_vp, _i64, _i32]),
    "soax_bin_permute_inplace": (C.c_int, [_vp, _vp, _i32, _f64, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "soax_gather_segments_aos": (C.c_int, [_vp, _vp, _vp, _vp, _i64, _i64, _vp]),
    "soax_remove_scratch_bytes": (_sz, [_i64]),
    "soax_remove": (C.c_int, [_vp, _vp, _vp, _i32, _vp, _sz, C.POINTER(_i64), _vp]),
    "soax_remove_stable_noalloc": (C.c_int, [_vp, _vp, _vp, _i32, _vp, _vp]),
    "soax_push_back_aos": (C.c_int, [_vp, _vp, _i64, _vp]),
    "soax_get_elements": (C.c_int, [_vp, _vp, _i64, _vp, _vp]),
    "soax_copy": (C.c_int, [_vp, _vp, _vp]),
    "soax_expr_compile": (C.c_int, [_vp, C.c_char_p, C.POINTER(C.c_char_p), _i32, C.POINTER(_vp)]),
    "soax_expr_compile_sum": (C.c_int, [_vp, C.c_char_p, C.POINTER(C.c_char_p), _i32, C.POINTER(_vp)]),
    "soax_expr_sum": (C.c_int, [_vp, _vp, C.POINTER(_f64), _i32, _vp, _sz, _vp, _vp]),
    "soax_expr_compile_mask": (C.c_int, [_vp, C.c_char_p, C.POINTER(C.c_char_p), _i32, C.POINTER(_vp)]),
    "soax_expr_mask": (C.c_int, [_vp, _vp, C.POINTER(_f64), _i32, _vp, _vp]),
    "soax_expr_run": (C.c_int, [_vp, _vp, C.POINTER(_f64), _i32, _i32, _vp]),
    "soax_expr_free": (C.c_int, [_vp]),
    "soax_expr_error": (C.c_char_p, []),
    "soax_expr_cuda_source": (C.c_char_p, [_vp]),
    "soax_expr_traffic": (C.c_int, [_vp, C.POINTER(_i32), C.POINTER(_i32)]),
    "soax_strerror": (C.c_char_p, [C.c_int]),
    "soax_last_cuda_error": (C.c_int, []),
    "soax_launch_count": (_i64, []),
    "soax_reset_launch_count": (None, []),
    "soax_tune": (C.c_int, [C.c_char_p, _i64]),
}


def library_path() -> str:
    return _build.LIB


def lib() -> C.CDLL:
    """Load libsoax.so (building it first if it is missing or older than its sources).  No fallback."""
    global _lib
    if _lib is None:
        try:
            path = _build.build()
        except Exception as e:  # the built library still travels with the tree: use it if the rebuild cannot run
            if not os.path.exists(_build.LIB):
                raise ImportError(f"libsoax.so is missing and could not be built: {e}") from e
            path = _build.LIB
        L = C.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)      # AttributeError if the library does not export a declared symbol
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(status: int, where: str) -> None:
    if status != SOAX_OK:
        raise SoaxError(status, where)


# ---- layout registry ----------------------------------------------------------------------------------------
def soax_layout_define(fields: Sequence[tuple[str, int, int]]) -> int:
    """fields: (name, soax_dtype, dim) in declaration order.  Returns the registry's layout handle."""
    arr = (soax_field * len(fields))(*[soax_field(n.encode(), int(dt), int(dim)) for n, dt, dim in fields])
    out = _vp()
    _check(lib().soax_layout_define(arr, len(fields), C.byref(out)), "soax_layout_define")
    return out.value


def soax_layout_define_dynamic(fields: Sequence[tuple[str, int, int]]) -> int:
    """Any field list: a compiled layout if one matches, else a run-time layout (container + expression programs)."""
    arr = (soax_field * len(fields))(*[soax_field(n.encode(), int(dt), int(dim)) for n, dt, dim in fields])
    out = _vp()
    _check(lib().soax_layout_define_dynamic(arr, len(fields), C.byref(out)), "soax_layout_define_dynamic")
    return out.value


def soax_layout_nfields(layout: int) -> int:
    return lib().soax_layout_nfields(layout)


def soax_layout_ncomp(layout: int) -> int:
    return lib().soax_layout_ncomp(layout)


def soax_layout_comp(layout: int, c: int) -> tuple[int, int, int]:
    f, k, dt = _i32(), _i32(), _i32()
    _check(lib().soax_layout_comp(layout, c, C.byref(f), C.byref(k), C.byref(dt)), "soax_layout_comp")
    return f.value, k.value, dt.value


def soax_layout_aos(layout: int, packed: bool = True) -> tuple[int, list[int]]:
    nc = soax_layout_ncomp(layout)
    stride, offs = _sz(), (_sz * nc)()
    _check(lib().soax_layout_aos(layout, 1 if packed else 0, C.byref(stride), offs), "soax_layout_aos")
    return stride.value, list(offs)


def soax_slab_bytes(layout: int, capacity: int) -> int:
    return lib().soax_slab_bytes(layout, capacity)


# ---- container ------------------------------------------------------------------------------------------------
def soax_alloc(layout: int, n: int, capacity: int, dev_slab: int, slab_bytes: int) -> int:
    out = _vp()
    _check(lib().soax_alloc(layout, n, capacity, dev_slab, slab_bytes, C.byref(out)), "soax_alloc")
    return out.value


def soax_free(s: int) -> None:
    _check(lib().soax_free(s), "soax_free")


def soax_size(s: int) -> int:
    return lib().soax_size(s)


def soax_resize(s: int, n: int) -> None:
    _check(lib().soax_resize(s, n), "soax_resize")


def soax_field_ptr(s: int, field: int, comp: int) -> int:
    out = _vp()
    _check(lib().soax_field_ptr(s, field, comp, C.byref(out)), "soax_field_ptr")
    return out.value


def _ptr_array(ptrs: Sequence[int | None]):
    return (_vp * len(ptrs))(*[None if p is None else int(p) for p in ptrs])


def soax_upload(s: int, host_comps: Sequence[int | None], n: int, stream: int = 0) -> None:
    _check(lib().soax_upload(s, _ptr_array(host_comps), n, stream), "soax_upload")


def soax_download(s: int, host_comps: Sequence[int | None], n: int, stream: int = 0) -> None:
    _check(lib().soax_download(s, _ptr_array(host_comps), n, stream), "soax_download")


# ---- hot path -----------------------------------------------------------------------------------------------------
def step_params(kind: int, dt: float, k: float = 1.0, center: float = 0.5, flag_mask: int = 1) -> soax_step_params:
    p = soax_step_params()
    p.kind, p.flag_mask, p.dt, p.k, p.center = kind, flag_mask, dt, k, center
    return p


def soax_step(s: int, params: soax_step_params, nsteps: int, stream: int = 0) -> None:
    _check(lib().soax_step(s, C.byref(params), nsteps, stream), "soax_step")


def soax_step_aos(layout: int, dev_aos: int, n: int, params: soax_step_params, nsteps: int, variant: int = 0,
                  stream: int = 0) -> None:
    _check(lib().soax_step_aos(layout, dev_aos, n, C.byref(params), nsteps, variant, stream), "soax_step_aos")


def soax_aos_to_soa(dst: int, dev_aos: int, n: int, stream: int = 0) -> None:
    _check(lib().soax_aos_to_soa(dst, dev_aos, n, stream), "soax_aos_to_soa")


def soax_soa_to_aos(src: int, dev_aos: int, n: int, stream: int = 0) -> None:
    _check(lib().soax_soa_to_aos(src, dev_aos, n, stream), "soax_soa_to_aos")


def soax_energy_scratch_bytes() -> int:
    return lib().soax_energy_scratch_bytes()


def soax_reduce_energy(s: int, kind: int, k: float, center: float, dev_scratch: int, scratch_bytes: int, dev_out: int,
                       stream: int = 0) -> None:
    _check(lib().soax_reduce_energy(s, kind, k, center, dev_scratch, scratch_bytes, dev_out, stream), "soax_reduce_energy")


def soax_scratch_bytes(layout: int, n: int, grid_dim: int) -> int:
    return lib().soax_scratch_bytes(layout, n, grid_dim)


def soax_bin_permute(src: int, dst: int, grid_dim: int, drift_dt: float, dev_counts: int | None, dev_offsets: int | None,
                     dev_perm: int | None, dev_kinetic: int | None, dev_scratch: int, scratch_bytes: int,
                     stream: int = 0) -> None:
    _check(lib().soax_bin_permute(src, dst, grid_dim, drift_dt, dev_counts, dev_offsets, dev_perm, dev_kinetic,
                                  dev_scratch, scratch_bytes, stream), "soax_bin_permute")


def soax_scratch_bytes_inplace(layout: int, n: int, grid_dim: int) -> int:
    return lib().soax_scratch_bytes_inplace(layout, n, grid_dim)


def soax_bin_permute_inplace(s: int, work: int, grid_dim: int, drift_dt: float, dev_counts: int | None, dev_offsets: int | None,
                             dev_perm: int | None, dev_kinetic: int | None, dev_scratch: int, scratch_bytes: int,
                             stream: int = 0) -> None:
    _check(lib().soax_bin_permute_inplace(s, work, grid_dim, drift_dt, dev_counts, dev_offsets, dev_perm, dev_kinetic,
                                          dev_scratch, scratch_bytes, stream), "soax_bin_permute_inplace")


# ---- container operations (NEXT-3) ------------------------------------------------------------------------------------
def soax_remove_scratch_bytes(n: int) -> int:
    return lib().soax_remove_scratch_bytes(n)


def soax_remove(s: int, dst: int | None, dev_kill: int, mode: int, dev_scratch: int, scratch_bytes: int, stream: int = 0,
                host_new_n: int | None = None) -> None:
    """Asynchronous: everything is enqueued and the call returns.  The live count of the target handle (s for SWAP_LAST,
    dst for STABLE) is learnt lazily by the first later call that needs it (soax_size waits for the one event that marks
    the count ready).  host_new_n: optional address of a PINNED int64 that also receives the survivor count."""
    ptr = C.cast(host_new_n, C.POINTER(_i64)) if host_new_n else None
    _check(lib().soax_remove(s, dst, dev_kill, mode, dev_scratch, scratch_bytes, ptr, stream), "soax_remove")


def soax_remove_stable_noalloc(s: int, dst: int, dev_kill: int, keep_flagged: bool, dev_new_n: int, stream: int = 0) -> None:
    """The stable removal for callers that cannot allocate (see include/soax.h): no scratch argument, nothing allocated by
    the library either; at most SOAX_NOALLOC_MAX_N particles (SoaxError with status SOAX_ERR_TOO_LARGE beyond).  The
    survivor count lands in the int64 DEVICE word dev_new_n; dst's live count is left for the caller to set (soax_resize)."""
    _check(lib().soax_remove_stable_noalloc(s, dst, dev_kill, 1 if keep_flagged else 0, dev_new_n, stream), "soax_remove_stable_noalloc")


def soax_push_back_aos(s: int, dev_aos: int, m: int, stream: int = 0) -> None:
    _check(lib().soax_push_back_aos(s, dev_aos, m, stream), "soax_push_back_aos")


def soax_get_elements(s: int, dev_idx: int, m: int, dev_aos: int, stream: int = 0) -> None:
    _check(lib().soax_get_elements(s, dev_idx, m, dev_aos, stream), "soax_get_elements")


def soax_gather_segments_aos(dst: int, dev_aos: int, dev_seg_dst: int, dev_seg_src: int, nseg: int, n: int, stream: int = 0) -> None:
    _check(lib().soax_gather_segments_aos(dst, dev_aos, dev_seg_dst, dev_seg_src, nseg, n, stream), "soax_gather_segments_aos")


def soax_copy(dst: int, src: int, stream: int = 0) -> None:
    _check(lib().soax_copy(dst, src, stream), "soax_copy")


# ---- fused element-wise programs (NEXT-2) ---------------------------------------------------------------------------------
def soax_expr_compile(layout: int, source: str, scalar_names: Sequence[str] = ()) -> int:
    names = (C.c_char_p * max(len(scalar_names), 1))(*[n.encode() for n in scalar_names])
    out = _vp()
    status = lib().soax_expr_compile(layout, source.encode(), names, len(scalar_names), C.byref(out))
    if status != SOAX_OK:
        e = SoaxError(status, "soax_expr_compile")
        e.args = (f"{e.args[0]}: {lib().soax_expr_error().decode()}",)
        raise e
    return out.value


def soax_expr_compile_sum(layout: int, expression: str, scalar_names: Sequence[str] = ()) -> int:
    names = (C.c_char_p * max(len(scalar_names), 1))(*[n.encode() for n in scalar_names])
    out = _vp()
    status = lib().soax_expr_compile_sum(layout, expression.encode(), names, len(scalar_names), C.byref(out))
    if status != SOAX_OK:
        e = SoaxError(status, "soax_expr_compile_sum")
        e.args = (f"{e.args[0]}: {lib().soax_expr_error().decode()}",)
        raise e
    return out.value


def soax_expr_compile_mask(layout: int, condition: str, scalar_names: Sequence[str] = ()) -> int:
    names = (C.c_char_p * max(len(scalar_names), 1))(*[n.encode() for n in scalar_names])
    out = _vp()
    status = lib().soax_expr_compile_mask(layout, condition.encode(), names, len(scalar_names), C.byref(out))
    if status != SOAX_OK:
        e = SoaxError(status, "soax_expr_compile_mask")
        e.args = (f"{e.args[0]}: {lib().soax_expr_error().decode()}",)
        raise e
    return out.value


def soax_expr_mask(s: int, e: int, scalars: Sequence[float], dev_mask: int, stream: int = 0) -> None:
    arr = (_f64 * max(len(scalars), 1))(*[float(x) for x in scalars])
    _check(lib().soax_expr_mask(s, e, arr, len(scalars), dev_mask, stream), "soax_expr_mask")


def soax_expr_sum(s: int, e: int, scalars: Sequence[float], dev_scratch: int, scratch_bytes: int, dev_out: int, stream: int = 0) -> None:
    arr = (_f64 * max(len(scalars), 1))(*[float(x) for x in scalars])
    _check(lib().soax_expr_sum(s, e, arr, len(scalars), dev_scratch, scratch_bytes, dev_out, stream), "soax_expr_sum")


def soax_expr_run(s: int, e: int, scalars: Sequence[float] = (), nsteps: int = 1, stream: int = 0) -> None:
    arr = (_f64 * max(len(scalars), 1))(*[float(x) for x in scalars])
    _check(lib().soax_expr_run(s, e, arr, len(scalars), nsteps, stream), "soax_expr_run")


def soax_expr_free(e: int) -> None:
    _check(lib().soax_expr_free(e), "soax_expr_free")


def soax_expr_error() -> str:
    return lib().soax_expr_error().decode()


def soax_expr_cuda_source(e: int) -> str:
    return lib().soax_expr_cuda_source(e).decode()


def soax_expr_traffic(e: int) -> tuple[int, int]:
    r, w = _i32(), _i32()
    _check(lib().soax_expr_traffic(e, C.byref(r), C.byref(w)), "soax_expr_traffic")
    return r.value, w.value


# ---- diagnostics ------------------------------------------------------------------------------------------------------
def soax_strerror(status: int) -> str:
    return lib().soax_strerror(status).decode()


def soax_last_cuda_error() -> int:
    return lib().soax_last_cuda_error()


def soax_launch_count() -> int:
    return lib().soax_launch_count()


def soax_reset_launch_count() -> None:
    lib().soax_reset_launch_count()


def soax_tune(key: str, value: int) -> None:
    _check(lib().soax_tune(key.encode(), value), f"soax_tune({key})")
