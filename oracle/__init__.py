"""Python face of the ORACLE (oracle/soax_oracle.cpp) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It imports nothing from paper_1710_03462_b200 (the CUDA path) and that package imports nothing
from here.  Host particle sets are dicts name -> ndarray (dim, N) (component-major SoA, as produced by the
seeded generators); this wrapper packs them into the oracle's array of structs, calls the single-threaded
C++ routine, and unpacks.  The packing itself is plain numpy structured-array assignment.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

# Packed 40-byte record of BASELINE.json config 3 and the natural 96-byte wide record.
R1_DTYPE = np.dtype({"names": ["id", "pos", "vel"], "formats": ["<i4", ("<f8", 3), ("<f4", 3)],
                     "offsets": [0, 4, 28], "itemsize": 40})
R2_DTYPE = np.dtype({"names": ["id", "pos", "vel", "acc", "mass", "charge", "flags"],
                     "formats": ["<i8", ("<f8", 3), ("<f8", 3), ("<f8", 3), "<f4", "<f4", "u1"],
                     "offsets": [0, 8, 32, 56, 80, 84, 88], "itemsize": 96})

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        vp, i64, i32, f64, u8 = C.c_void_p, C.c_int64, C.c_int32, C.c_double, C.c_uint8
        L.soax_oracle_wrap.restype = f64
        L.soax_oracle_wrap.argtypes = [f64]
        L.soax_oracle_r1_stride.restype = i64
        L.soax_oracle_r2_stride.restype = i64
        L.soax_oracle_r1_offsets.argtypes = [vp]
        L.soax_oracle_r1_drift.argtypes = [vp, i64, f64, i32]
        L.soax_oracle_r1_symplectic_euler.argtypes = [vp, i64, f64, f64, f64, i32]
        L.soax_oracle_r2_rk2.argtypes = [vp, i64, f64, f64, f64, u8, i32]
        L.soax_oracle_r2_drift.argtypes = [vp, i64, f64, i32]
        L.soax_oracle_r1_energy.restype = f64
        L.soax_oracle_r1_energy.argtypes = [vp, i64, i32, f64, f64]
        L.soax_oracle_r2_energy.restype = f64
        L.soax_oracle_r2_energy.argtypes = [vp, i64, i32, f64, f64]
        L.soax_oracle_r1_aos_to_soa.argtypes = [vp, i64] + [vp] * 7
        L.soax_oracle_r1_soa_to_aos.argtypes = [vp, i64] + [vp] * 7
        L.soax_oracle_r1_bin.restype = i32
        L.soax_oracle_r1_bin.argtypes = [vp, i64, i32, vp, vp, vp, vp, vp]
        L.soax_oracle_r1_permute.argtypes = [vp, vp, i64, vp]
        L.soax_oracle_b6_euler.argtypes = [vp, i64, i32, C.c_float, i32]
        L.soax_oracle_fma_f64.argtypes = [vp, vp, vp, vp, i64]
        L.soax_oracle_remove_swap_last.restype = i64
        L.soax_oracle_remove_swap_last.argtypes = [vp, i64, i64, vp]
        L.soax_oracle_remove_stable.restype = i64
        L.soax_oracle_remove_stable.argtypes = [vp, i64, i64, vp]
        L.soax_oracle_get_elements.argtypes = [vp, i64, vp, i64, vp]
        L.soax_oracle_fma_f32.argtypes = [vp, vp, vp, vp, i64]
        L.soax_oracle_gather_segments.argtypes = [vp, i64, vp, vp, i64, i64, vp]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


# ---- packing between the generators' component-major dicts and the oracle's array of structs -----------
def pack(soa: dict, dtype: np.dtype) -> np.ndarray:
    n = next(iter(soa.values())).shape[1]
    aos = np.zeros(n, dtype)
    for name in dtype.names:
        v = soa[name]
        aos[name] = v[0] if v.shape[0] == 1 else v.T
    return aos


def unpack(aos: np.ndarray) -> dict:
    out = {}
    for name in aos.dtype.names:
        f = aos[name]
        out[name] = np.ascontiguousarray(f[None, :] if f.ndim == 1 else f.T)
    return out


def pack_r1(soa):
    return pack(soa, R1_DTYPE)


def pack_r2(soa):
    return pack(soa, R2_DTYPE)


def wrap(x: float) -> float:
    return lib().soax_oracle_wrap(float(x))


# ---- operations on host SoA dicts (return new dicts; inputs untouched) -------------------------------
def drift(soa: dict, dt: float, nsteps: int) -> dict:
    if soa["vel"].dtype == np.float32:
        aos = pack_r1(soa)
        lib().soax_oracle_r1_drift(_p(aos), aos.size, dt, nsteps)
    else:
        aos = pack_r2(soa)
        lib().soax_oracle_r2_drift(_p(aos), aos.size, dt, nsteps)
    return unpack(aos)


def symplectic_euler(soa: dict, dt: float, nsteps: int, k: float = 1.0, center: float = 0.5) -> dict:
    aos = pack_r1(soa)
    lib().soax_oracle_r1_symplectic_euler(_p(aos), aos.size, dt, k, center, nsteps)
    return unpack(aos)


def rk2_midpoint_masked(soa: dict, dt: float, nsteps: int, k: float = 1.0, center: float = 0.5,
                        mask: int = 1) -> dict:
    aos = pack_r2(soa)
    lib().soax_oracle_r2_rk2(_p(aos), aos.size, dt, k, center, mask, nsteps)
    return unpack(aos)


KINETIC, KINETIC_PLUS_HARMONIC = 0, 1


def energy(soa: dict, kind: int, k: float = 1.0, center: float = 0.5) -> float:
    if soa["vel"].dtype == np.float32:
        aos = pack_r1(soa)
        return lib().soax_oracle_r1_energy(_p(aos), aos.size, kind, k, center)
    aos = pack_r2(soa)
    return lib().soax_oracle_r2_energy(_p(aos), aos.size, kind, k, center)


def r1_aos_to_soa(aos_bytes: np.ndarray) -> dict:
    """aos_bytes: uint8 array of 40*n bytes (any content).  Returns the 7 component arrays as an R1 dict."""
    n = aos_bytes.size // 40
    out = {"id": np.empty((1, n), np.int32), "pos": np.empty((3, n), np.float64), "vel": np.empty((3, n), np.float32)}
    lib().soax_oracle_r1_aos_to_soa(_p(aos_bytes), n, _p(out["id"][0]), *[_p(out["pos"][c]) for c in range(3)],
                                    *[_p(out["vel"][c]) for c in range(3)])
    return out


def r1_soa_to_aos(soa: dict) -> np.ndarray:
    n = soa["id"].shape[1]
    aos = np.zeros(40 * n, np.uint8)
    s = {k: np.ascontiguousarray(v) for k, v in soa.items()}
    lib().soax_oracle_r1_soa_to_aos(_p(aos), n, _p(s["id"][0]), *[_p(s["pos"][c]) for c in range(3)],
                                    *[_p(s["vel"][c]) for c in range(3)])
    return aos


def bin_r1(soa: dict, grid_dim: int, want_perm: bool = True) -> dict:
    """Cell index, counts, exclusive scan, stable gather permutation and its inverse (a10..a13)."""
    aos = pack_r1(soa)
    n, ncell = aos.size, grid_dim ** 3
    out = {"cell": np.empty(n, np.uint32), "counts": np.empty(ncell, np.uint32), "offsets": np.empty(ncell, np.uint32)}
    if want_perm:
        out["perm"] = np.empty(n, np.uint32)
        out["dest"] = np.empty(n, np.uint32)
    rc = lib().soax_oracle_r1_bin(_p(aos), n, grid_dim, _p(out["cell"]), _p(out["counts"]), _p(out["offsets"]),
                                  _p(out.get("perm")), _p(out.get("dest")))
    if rc != 0:
        raise ValueError("oracle: cell index out of range (pos outside [0,1)?)")
    return out


def permute_r1(soa: dict, perm: np.ndarray) -> dict:
    """a14: new[j] = old[perm[j]] for every field."""
    old = pack_r1(soa)
    new = np.zeros_like(old)
    lib().soax_oracle_r1_permute(_p(old), _p(new), old.size, _p(np.ascontiguousarray(perm, np.uint32)))
    return unpack(new)


def b6_euler(pos: np.ndarray, vel: np.ndarray, size_extra: int, dt: float, nsteps: int):
    """PAPER.md:134-157 benchmark on Particle<SIZE>: returns the new (3, n) float positions."""
    n = pos.shape[1]
    aos = np.zeros((n, 6 + size_extra), np.float32)
    aos[:, 0:3] = pos.T
    aos[:, 3:6] = vel.T
    lib().soax_oracle_b6_euler(_p(aos), n, size_extra, dt, nsteps)
    return np.ascontiguousarray(aos[:, 0:3].T), np.ascontiguousarray(aos[:, 3:6].T)


def fma(a: np.ndarray, b: np.ndarray, c: np.ndarray) -> np.ndarray:
    """Element-wise correctly rounded a*b+c (std::fma / std::fmaf) on equal-length float64 or float32 arrays."""
    assert a.dtype == b.dtype == c.dtype and a.shape == b.shape == c.shape and a.ndim == 1
    a, b, c = (np.ascontiguousarray(x) for x in (a, b, c))
    out = np.empty_like(a)
    fn = lib().soax_oracle_fma_f64 if a.dtype == np.float64 else lib().soax_oracle_fma_f32
    assert a.dtype in (np.float64, np.float32)
    fn(_p(a), _p(b), _p(c), _p(out), a.size)
    return out


# ---- NEXT-3: container operations on packed records (uint8 array of n*stride bytes) ---------------------------------
def remove_swap_last(aos_bytes: np.ndarray, stride: int, kill: np.ndarray) -> np.ndarray:
    """PAPER.md:175 in a forward loop: a flagged record is overwritten by the last one and the slot is examined again
    (Q20).  Returns the new bytes."""
    a = np.array(aos_bytes, dtype=np.uint8)
    n = a.size // stride
    k = np.array(kill[:n], dtype=np.uint8)                          # consumed by the routine
    m = lib().soax_oracle_remove_swap_last(_p(a), n, stride, _p(k))
    return a[:m * stride].copy()


def remove_stable(aos_bytes: np.ndarray, stride: int, kill: np.ndarray) -> np.ndarray:
    a = np.array(aos_bytes, dtype=np.uint8)
    n = a.size // stride
    k = np.ascontiguousarray(kill[:n], np.uint8)
    m = lib().soax_oracle_remove_stable(_p(a), n, stride, _p(k))
    return a[:m * stride].copy()


def get_elements(aos_bytes: np.ndarray, stride: int, idx: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(aos_bytes, np.uint8)
    i = np.ascontiguousarray(idx, np.uint32)
    out = np.empty(i.size * stride, np.uint8)
    lib().soax_oracle_get_elements(_p(a), stride, _p(i), i.size, _p(out))
    return out


def gather_segments(aos_bytes: np.ndarray, stride: int, seg_dst: np.ndarray, seg_src: np.ndarray, n: int) -> np.ndarray:
    """NEXT-4, the merge of sorted runs written as a segmented gather of packed records (include/soax.h
    soax_gather_segments_aos): output row j comes from input row seg_src[i] + (j - seg_dst[i]) where i is the LAST
    segment with seg_dst[i] <= j.  Plain definition, one row at a time."""
    a = np.ascontiguousarray(aos_bytes, np.uint8).reshape(-1, stride)
    seg_dst = np.asarray(seg_dst, np.int64)
    seg_src = np.asarray(seg_src, np.int64)
    out = np.empty((n, stride), np.uint8)
    i = 0
    for j in range(n):
        while i + 1 < seg_dst.size and seg_dst[i + 1] <= j:
            i += 1
        out[j] = a[seg_src[i] + (j - seg_dst[i])]
    return out.reshape(-1)


def gather_segments_c(aos_bytes: np.ndarray, stride: int, seg_dst: np.ndarray, seg_src: np.ndarray, n: int) -> np.ndarray:
    """The same definition as gather_segments, the row loop written in C (soax_oracle_gather_segments) so that the sizes the
    product is timed at (2^24 rows, 2 M segments) finish in seconds.  Pinned against the Python loop above."""
    a = np.ascontiguousarray(aos_bytes, np.uint8)
    sd, ss = np.ascontiguousarray(seg_dst, np.int64), np.ascontiguousarray(seg_src, np.int64)
    out = np.empty(n * stride, np.uint8)
    lib().soax_oracle_gather_segments(_p(a), stride, _p(sd), _p(ss), sd.size, n, _p(out))
    return out
