"""CPU-only tests of the host side: the C-ABI library loads and exports every symbol include/soax.h declares, the
layout registry / slab carving / argument checking behave as documented (no kernel is launched: device pointers are
fake, never dereferenced), and the N>1 sharding logic works under a world-size-2 gloo group."""
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
from paper_1710_03462_b200 import binding as B, container as Cn, inputs  # noqa: E402


def declared_functions():
    src = open(os.path.join(ROOT, "include", "soax.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(soax_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert len(names) >= 26 and "soax_bin_permute" in names and "soax_step" in names
    import ctypes
    L = ctypes.CDLL(B.library_path() if os.path.exists(B.library_path()) else B.lib()._name)
    for n in names:
        assert hasattr(L, n), f"libsoax.so does not export {n}"
    assert sorted(B.SIGNATURES) == names, "binding.py must bind exactly what the header declares"
    out = subprocess.run(["nm", "-D", "--defined-only", B.library_path()], capture_output=True, text=True).stdout
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l)
    assert exported == names, "only the header's functions are exported (built with -fvisibility=hidden)"


def test_library_is_sm100a_and_uses_wide_and_bulk_accesses():
    """the shipped cubin targets sm_100a and contains the Blackwell-only 256-bit accesses and the TMA bulk copies"""
    sass = subprocess.run(["cuobjdump", "-sass", B.library_path()], capture_output=True, text=True)
    if sass.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    text = sass.stdout
    assert "sm_100a" in text
    assert "LDG.E.NA.ENL2.256" in text or "LDG.E.ENL2.256" in text or ".256" in text
    assert "UBLKCP" in text
    assert "DFMA" in text and "UCGABAR_ARV" in text and "VOTE" in text   # explicit fma; cluster barrier + ballots of the scatter


def test_layout_registry_and_aos_image():
    L1 = B.soax_layout_define(Cn.R1)
    assert B.soax_layout_define(Cn.R1) == L1                       # registry-owned, stable handle
    assert B.soax_layout_nfields(L1) == 3 and B.soax_layout_ncomp(L1) == 7
    assert B.soax_layout_aos(L1, True) == (40, [0, 4, 12, 20, 28, 32, 36])          # Q1 / PAPER.md:41
    assert B.soax_layout_aos(L1, False) == (48, [0, 8, 16, 24, 32, 36, 40])         # natural C layout
    assert [B.soax_layout_comp(L1, c) for c in range(7)] == [(0, 0, B.SOAX_I32)] + [(1, k, B.SOAX_F64) for k in range(3)] + \
        [(2, k, B.SOAX_F32) for k in range(3)]
    L2 = B.soax_layout_define(Cn.R2)
    assert B.soax_layout_ncomp(L2) == 13 and B.soax_layout_aos(L2, True)[0] == 89 and B.soax_layout_aos(L2, False)[0] == 96
    for size, stride in ((0, 24), (8, 56), (16, 88), (32, 152)):   # 6*4 = 24 bytes at SIZE = 0
        assert B.soax_layout_aos(B.soax_layout_define(Cn.B6(size)), True)[0] == stride
    for bad in ([("id", B.SOAX_I32, 1), ("pos", B.SOAX_F64, 2)],    # no such instantiation
                [("pos", B.SOAX_F64, 3), ("id", B.SOAX_I32, 1), ("vel", B.SOAX_F32, 3)],   # order matters
                [("id", B.SOAX_I32, 1), ("pos", B.SOAX_F32, 3), ("vel", B.SOAX_F32, 3)]):
        with pytest.raises(B.SoaxError) as e:
            B.soax_layout_define(bad)
        assert e.value.status == B.SOAX_ERR_UNKNOWN_LAYOUT
    with pytest.raises(B.SoaxError) as e:
        B.soax_layout_define([("id", 99, 1)])
    assert e.value.status == B.SOAX_ERR_INVALID_ARG


def test_slab_carving_alignment_and_errors():
    L1 = B.soax_layout_define(Cn.R1)
    cap = 1001
    need = B.soax_slab_bytes(L1, cap)
    sizes = [4] + [8] * 3 + [4] * 3
    assert need == sum((cap * s + 255) // 256 * 256 for s in sizes)
    base = 0x7000000000                                             # fake device address, 256-byte aligned
    s = B.soax_alloc(L1, 1000, cap, base, need)
    try:
        assert B.soax_size(s) == 1000
        ptrs = [B.soax_field_ptr(s, 0, 0)] + [B.soax_field_ptr(s, 1, k) for k in range(3)] + [B.soax_field_ptr(s, 2, k) for k in range(3)]
        assert ptrs[0] == base and all(p % 256 == 0 for p in ptrs)
        for a, b, sz in zip(ptrs, ptrs[1:], sizes):
            assert b - a == (cap * sz + 255) // 256 * 256           # contiguous, non-overlapping component arrays
        assert ptrs[-1] + cap * 4 <= base + need
        with pytest.raises(B.SoaxError) as e:
            B.soax_field_ptr(s, 1, 3)                               # pos has 3 components
        assert e.value.status == B.SOAX_ERR_UNSUPPORTED
        with pytest.raises(B.SoaxError) as e:
            B.soax_field_ptr(s, 3, 0)
        assert e.value.status == B.SOAX_ERR_INVALID_ARG
        B.soax_resize(s, cap)
        assert B.soax_size(s) == cap
        with pytest.raises(B.SoaxError):
            B.soax_resize(s, cap + 1)
    finally:
        B.soax_free(s)
    for args, status in (((L1, 10, 5, base, need), B.SOAX_ERR_INVALID_ARG),        # n > capacity
                         ((L1, 10, cap, base + 8, need), B.SOAX_ERR_INVALID_ARG),   # misaligned slab
                         ((L1, 10, cap, base, need - 1), B.SOAX_ERR_ALLOC)):        # slab too small
        with pytest.raises(B.SoaxError) as e:
            B.soax_alloc(*args)
        assert e.value.status == status
    assert B.soax_slab_bytes(L1, -1) == 0


def test_argument_checks_without_launching():
    L1 = B.soax_layout_define(Cn.R1)
    base = 0x7000000000
    s = B.soax_alloc(L1, 0, 16, base, B.soax_slab_bytes(L1, 16))
    try:
        B.soax_step(s, B.step_params(B.SOAX_STEP_DRIFT, 1e-3), 5)                  # n = 0: nothing is launched
        before = B.soax_launch_count()
        with pytest.raises(B.SoaxError) as e:
            B.soax_step(s, B.step_params(7, 1e-3), 1)
        assert B.soax_launch_count() == before
        with pytest.raises(B.SoaxError) as e:
            B.soax_bin_permute(s, s, 64, 0.0, None, None, None, None, base, 1 << 20)   # src must not alias dst
        assert e.value.status == B.SOAX_ERR_INVALID_ARG
        assert B.soax_scratch_bytes(L1, 1000, 3) == 0                               # grid must be a power of two
        assert B.soax_scratch_bytes(L1, 1000, 64) > 52 * 1000
        assert B.soax_scratch_bytes(B.soax_layout_define(Cn.B6(0)), 1000, 64) == 0  # no double pos[3]: unsupported
        assert B.soax_energy_scratch_bytes() % 8 == 0
        assert "layout" in B.soax_strerror(B.SOAX_ERR_UNKNOWN_LAYOUT)
        with pytest.raises(B.SoaxError):
            B.soax_tune("no_such_knob", 1)
    finally:
        B.soax_free(s)


def test_step_params_struct_matches_header():
    import ctypes
    assert ctypes.sizeof(B.soax_step_params) == 32 and B.soax_step_params.dt.offset == 8
    assert ctypes.sizeof(B.soax_field) == 16


def test_shard_range_partitions():
    for n, w in ((10, 3), (1 << 24, 8), (7, 8), (0, 2)):
        spans = [inputs.shard_range(n, r, w) for r in range(w)]
        assert spans[0][0] == 0 and spans[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
        assert max(h - l for l, h in spans) - min(h - l for l, h in spans) <= 1


_GLOO_WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
import oracle
from paper_1710_03462_b200 import inputs
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + sys.argv[2], rank=int(sys.argv[3]), world_size=2)
rank, n = dist.get_rank(), 4001
# N>1 path of the library: particles are sharded by index, every rank works on its own contiguous range with no
# data-path exchange; only the energy needs one 8-byte reduction, summed in rank order for determinism (SURVEY 8(e)).
lo, hi = inputs.shard_range(n, rank, 2)
full = inputs.make_r1(n, seed=0)
mine = inputs.take(full, np.arange(lo, hi))
out = oracle.symplectic_euler(mine, 1e-3, 5)                       # stands in for the device step on this shard
e = torch.tensor([oracle.energy(out, oracle.KINETIC_PLUS_HARMONIC)], dtype=torch.float64)
parts = [torch.zeros(1, dtype=torch.float64) for _ in range(2)]
dist.all_gather(parts, e)
total = float(parts[0] + parts[1])
ref = oracle.symplectic_euler(full, 1e-3, 5)
assert np.array_equal(ref["pos"][:, lo:hi], out["pos"]) and np.array_equal(ref["vel"][:, lo:hi], out["vel"])
eref = oracle.energy(ref, oracle.KINETIC_PLUS_HARMONIC)
assert abs(total - eref) <= 1e-12 * eref, (total, eref)
t = torch.tensor([float(rank + 1)]); dist.all_reduce(t, op=dist.ReduceOp.MAX)      # the bench's max-over-ranks timing
assert t.item() == 2.0
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
"""


def test_two_rank_sharding_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER)
    port = str(29500 + os.getpid() % 2000)
    procs = [subprocess.Popen([sys.executable, str(script), ROOT, port, str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
    assert sorted(o.strip().splitlines()[-1] for o in outs) == ["ok 0", "ok 1"]


def test_maximum_sizes_are_refused_before_any_launch():
    """Permutations, counts and offsets are uint32 (include/soax.h): 2^32 particles or more are UNSUPPORTED for binning and
    removal.  Checked with fake device pointers: the calls must answer from their argument checks, without touching memory."""
    L = B.soax_layout_define(Cn.R1)
    n = 1 << 32
    bytes_ = B.soax_slab_bytes(L, n)
    assert bytes_ == 7 * 0 + (4 + 3 * 8 + 3 * 4) * n                  # every array of 2^32 elements is already 256-byte aligned
    fake = 1 << 40
    a = B.soax_alloc(L, n, n, fake, bytes_)
    b = B.soax_alloc(L, 0, n, fake + bytes_, bytes_)
    for call in (lambda: B.soax_bin_permute(a, b, 64, 0.0, None, None, None, None, 256, 1 << 62),
                 lambda: B.soax_remove(a, None, 256, B.SOAX_REMOVE_SWAP_LAST, 256, 1 << 62)):
        with pytest.raises(B.SoaxError) as e:
            call()
        assert e.value.status == B.SOAX_ERR_UNSUPPORTED
    assert B.soax_scratch_bytes(L, (1 << 32) - 1, 64) > 40 * ((1 << 32) - 1)     # the plan itself is computed in 64 bits
    B.soax_free(a), B.soax_free(b)


def test_committed_traffic_names_commits_that_exist():
    """profiles/kernel_traffic.json feeds roofline.traffic in bench.py: every captured_at_commit in it must resolve in this
    repository's history (checked here, where the history is; the GPU box gets the tree without .git), and bench.py withholds
    the number when one does not."""
    import json
    import subprocess
    import bench
    if not os.path.isdir(os.path.join(ROOT, ".git")):
        pytest.skip("no git history here")
    with open(os.path.join(ROOT, "profiles", "kernel_traffic.json")) as f:
        table = json.load(f)
    assert table
    for key, d in table.items():
        rev = d["captured_at_commit"].split()[0]
        r = subprocess.run(["git", "-C", ROOT, "cat-file", "-t", rev], capture_output=True, text=True)
        assert r.returncode == 0 and r.stdout.strip() == "commit", (key, rev)
        traffic, prov = bench.committed_traffic(key)
        assert traffic == d["dram_bytes_per_launch"] and "rejected" not in prov
    assert bench.commit_in_history("0123456789abcdef0123456789abcdef01234567") is False
