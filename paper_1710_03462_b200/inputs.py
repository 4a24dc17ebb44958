"""Seeded synthetic particle sets (SURVEY.md §8(c) Q9/Q10, §8(d) "Synthetic inputs").

This module serves BOTH the oracle-side tests and the CUDA path.  It holds none of the
method's arithmetic (no drift, wrap, force, energy, cell index or sort): it only draws
the initial field values that BASELINE.json's configs describe, on the host, with numpy.

Generator (Q10): counter-based.  value = G(seed, field, component, draw, particle index),
so generation is order independent, chunkable and thread-safe.  G is two rounds of the
SplitMix64 finaliser over (index * golden + key).  Nothing pins the generator to a
published stream ("parity unpinned", harmless: both sides consume the same arrays).

Host representation of an SoA particle set: dict  name -> ndarray of shape (dim, N),
C-contiguous, i.e. component-major ("three heap-allocated arrays for x and
v"), dim = 1 or 3.
"""
from __future__ import annotations

import math
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_M64 = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15
_C1 = 0xBF58476D1CE4E5B9
_C2 = 0x94D049BB133111EB
_CHUNK = 1 << 22

# (name, numpy dtype, dim) in declaration order.  R1 = PAPER.md:41; R2 = BASELINE.json config 4;
# B6 = PAPER.md:144-155 (Listing 4 with SIZE=0: float x[3]; float v[3]).
R1_FIELDS = (("id", np.int32, 1), ("pos", np.float64, 3), ("vel", np.float32, 3))
R2_FIELDS = (("id", np.int64, 1), ("pos", np.float64, 3), ("vel", np.float64, 3),
             ("acc", np.float64, 3), ("mass", np.float32, 1), ("charge", np.float32, 1),
             ("flags", np.uint8, 1))

_STREAM = {"id": 1, "pos": 2, "vel": 3, "acc": 4, "mass": 5, "charge": 6, "flags": 7}


def _mix_int(z: int) -> int:
    z &= _M64
    z = ((z ^ (z >> 30)) * _C1) & _M64
    z = ((z ^ (z >> 27)) * _C2) & _M64
    return z ^ (z >> 31)


def _mix_arr(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * np.uint64(_C1)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(_C2)
    return z ^ (z >> np.uint64(31))


def _key(seed: int, field: str, comp: int, draw: int) -> int:
    s = _mix_int(seed * _GOLDEN + 0x1234567)
    return _mix_int(s ^ (((_STREAM[field] << 16) | (comp << 8) | draw) * _C2))


def raw_u64(seed: int, field: str, comp: int, draw: int, lo: int, hi: int) -> np.ndarray:
    """64 random bits for particle indices lo..hi-1 of one (seed, field, comp, draw) stream."""
    key = np.uint64(_key(seed, field, comp, draw))
    idx = np.arange(lo, hi, dtype=np.uint64)
    with np.errstate(over="ignore"):
        return _mix_arr(_mix_arr(idx * np.uint64(_GOLDEN) + key) ^ key)


def _uniform01(seed, field, comp, draw, lo, hi) -> np.ndarray:
    """Uniform in [0,1): top 53 bits * 2^-53."""
    return (raw_u64(seed, field, comp, draw, lo, hi) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def _normal(seed, field, comp, lo, hi) -> np.ndarray:
    """Standard normal in double: Box-Muller on two independent uniform streams."""
    u1 = 1.0 - _uniform01(seed, field, comp, 0, lo, hi)        # (0, 1]
    u2 = _uniform01(seed, field, comp, 1, lo, hi)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos((2.0 * math.pi) * u2)


def _chunked(n: int, fill, out: np.ndarray, threads: int) -> None:
    spans = [(lo, min(lo + _CHUNK, n)) for lo in range(0, n, _CHUNK)]
    if threads <= 1 or len(spans) <= 1:
        for lo, hi in spans:
            out[lo:hi] = fill(lo, hi)
        return

    def work(span):
        out[span[0]:span[1]] = fill(*span)

    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(work, spans))


def random_permutation(seed: int, n: int, dtype, lo: int = 0, hi: int | None = None) -> np.ndarray:
    """ids[i] = P_seed(i): a seeded bijection of 0..n-1 ("ids are a random permutation").

    Counter-based: four rounds of (odd multiply + add, xor-shift) on k = ceil(log2 n) bits, each
    round a bijection of Z/2^k, with cycle walking for n that is not a power of two.
    """
    hi = n if hi is None else hi
    k = max(1, (n - 1).bit_length())
    mask = np.uint64((1 << k) - 1)
    sh = np.uint64(max(1, (k + 1) // 2))
    rounds = []
    for r in range(4):
        mul = (_key(seed, "id", 0, 2 * r) | 1) & _M64
        add = _key(seed, "id", 0, 2 * r + 1)
        rounds.append((np.uint64(mul), np.uint64(add)))

    def f(x):
        with np.errstate(over="ignore"):
            for mul, add in rounds:
                x = (x * mul + add) & mask
                x = x ^ (x >> sh)
        return x

    x = f(np.arange(lo, hi, dtype=np.uint64))
    bad = x >= np.uint64(n)
    while bad.any():                         # cycle walking: stays a bijection on 0..n-1
        x[bad] = f(x[bad])
        bad = x >= np.uint64(n)
    return x.astype(dtype)


def make_r1(n: int, seed: int, threads: int = 8) -> dict:
    """Record R1 {int32 id; double pos[3]; float vel[3]} (BASELINE.json configs 1, 2, 3, 5).

    id = seeded permutation of 0..n-1; pos ~ U[0,1)^3 (53-bit); vel = (float) N(0,1).
    """
    out = {"id": np.empty((1, n), np.int32), "pos": np.empty((3, n), np.float64),
           "vel": np.empty((3, n), np.float32)}
    _chunked(n, lambda lo, hi: random_permutation(seed, n, np.int32, lo, hi), out["id"][0], threads)
    for c in range(3):
        _chunked(n, lambda lo, hi, c=c: _uniform01(seed, "pos", c, 0, lo, hi), out["pos"][c], threads)
        _chunked(n, lambda lo, hi, c=c: _normal(seed, "vel", c, lo, hi).astype(np.float32), out["vel"][c], threads)
    return out


def make_r2(n: int, seed: int, threads: int = 8) -> dict:
    """Record R2 (BASELINE.json config 4).

    id int64 permutation; pos U[0,1)^3; vel double N(0,1); acc = 0; mass = (float) U[0.5,2) with a
    result of exactly 2.0f clamped to the float below 2; charge = +-1 (p = 1/2); flags uniform uint8.
    """
    out = {"id": np.empty((1, n), np.int64), "pos": np.empty((3, n), np.float64),
           "vel": np.empty((3, n), np.float64), "acc": np.zeros((3, n), np.float64),
           "mass": np.empty((1, n), np.float32), "charge": np.empty((1, n), np.float32),
           "flags": np.empty((1, n), np.uint8)}
    _chunked(n, lambda lo, hi: random_permutation(seed, n, np.int64, lo, hi), out["id"][0], threads)
    for c in range(3):
        _chunked(n, lambda lo, hi, c=c: _uniform01(seed, "pos", c, 0, lo, hi), out["pos"][c], threads)
        _chunked(n, lambda lo, hi, c=c: _normal(seed, "vel", c, lo, hi), out["vel"][c], threads)
    _chunked(n, lambda lo, hi: mass_from_uniform(_uniform01(seed, "mass", 0, 0, lo, hi)), out["mass"][0], threads)
    _chunked(n, lambda lo, hi: np.where(raw_u64(seed, "charge", 0, 0, lo, hi) >> np.uint64(63), 1.0, -1.0)
             .astype(np.float32), out["charge"][0], threads)
    _chunked(n, lambda lo, hi: (raw_u64(seed, "flags", 0, 0, lo, hi) >> np.uint64(56)).astype(np.uint8),
             out["flags"][0], threads)
    return out


def mass_from_uniform(u: np.ndarray) -> np.ndarray:
    """(float)(0.5 + 1.5 u), u in [0,1); a rounding up to 2.0f is clamped (Q9: the clamp is live)."""
    m = (0.5 + 1.5 * u).astype(np.float32)
    below2 = np.nextafter(np.float32(2.0), np.float32(0.0))
    return np.where(m >= np.float32(2.0), below2, m).astype(np.float32)


def make_b6(n: int, seed: int, threads: int = 8) -> dict:
    """Paper-replica benchmark record: float x[3]; float v[3]; named pos/vel."""
    out = {"pos": np.empty((3, n), np.float32), "vel": np.empty((3, n), np.float32)}
    for c in range(3):
        _chunked(n, lambda lo, hi, c=c: _uniform01(seed, "pos", c, 0, lo, hi).astype(np.float32), out["pos"][c], threads)
        _chunked(n, lambda lo, hi, c=c: _normal(seed, "vel", c, lo, hi).astype(np.float32), out["vel"][c], threads)
    # (float) of a double in [0,1) can round to 1.0f; keep the record inside the box
    np.minimum(out["pos"], np.nextafter(np.float32(1.0), np.float32(0.0)), out=out["pos"])
    return out


def take(soa: dict, idx: np.ndarray) -> dict:
    """Sub-sample particles idx of a host SoA set (copy)."""
    return {k: np.ascontiguousarray(v[:, idx]) for k, v in soa.items()}


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous index range of rank `rank` when n particles are split over `world` ranks (§8(e))."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
