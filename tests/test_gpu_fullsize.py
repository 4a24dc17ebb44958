"""GPU parity at BASELINE.json's FULL sizes, on the inputs the configs name (inputs.make_r1 / make_r2 with the config's
seed), in the launch configuration bench.py times (default tuning).

The oracle cannot STEP 2^24..2^26 particles 20-100 times in seconds, but particles are independent, so the integrators are
checked on SAMPLED particles (oracle on the same seeded inputs, bit for bit) plus whole-array properties; the energy sums
and config 5 (one drift step + binning) are compared with the oracle over ALL particles."""
import os

import numpy as np
import pytest

import oracle
from paper_1710_03462_b200 import inputs

pytestmark = pytest.mark.gpu
DT = 1e-3


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available()
    from paper_1710_03462_b200 import binding as B, container as Cn
    B.lib()
    return torch, B, Cn


def bits(a):
    a = np.ascontiguousarray(a)
    return a.view({4: np.uint32, 8: np.uint64, 1: np.uint8}[a.dtype.itemsize])


def sample_indices(n, m=8192, seed=123):
    rng = np.random.default_rng(seed)
    idx = np.unique(np.concatenate([rng.integers(0, n, m), np.arange(0, 64), np.arange(n - 64, n)]))
    return idx.astype(np.int64)


def gather(torch, s, idx):
    """download the particles `idx` of a device container as a host SoA dict (torch indexing is plumbing)"""
    t = torch.from_numpy(idx).cuda()
    out = {}
    for name, dt, dim in s.fields:
        out[name] = np.stack([s.comp_view(name, c)[t].cpu().numpy() for c in range(dim)])
    return out



def test_config2_full_size_sampled(gpu):
    torch, B, Cn = gpu
    n = 1 << 24
    host = inputs.make_r1(n, seed=0)
    s = Cn.Soax(Cn.R1, n)
    s.upload(host)
    e0 = s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC)
    s.step(B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=100)
    e100 = s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC)
    idx = sample_indices(n)
    got = gather(torch, s, idx)
    exp = oracle.symplectic_euler(inputs.take(host, idx), DT, 100)
    for name in exp:
        assert np.array_equal(bits(got[name]), bits(exp[name])), name
    # energies: the oracle's compensated sum over ALL particles of the same states (step 0: inputs; step 100: download)
    o0 = oracle.energy(host, oracle.KINETIC_PLUS_HARMONIC)
    final = s.download()
    o100 = oracle.energy(final, oracle.KINETIC_PLUS_HARMONIC)
    assert abs(e0 - o0) <= 1e-10 * o0 and abs(e100 - o100) <= 1e-10 * o100
    assert abs(e0 / n - 1.625) < 1e-3                               # KE 1.5 + PE 3*(1/2)(1/12)  (SURVEY 8(c) pin 4)
    assert abs(e100 - e0) / e0 < 1e-3                               # symplectic Euler keeps the energy bounded
    assert (final["pos"] >= 0).all() and (final["pos"] < 1).all()
    assert np.array_equal(final["id"], host["id"])                  # ids untouched

    # config 3 at full size: AoS kernels and transposes against the SoA result (oracle-free) and the oracle's packing
    aos0 = torch.from_numpy(oracle.r1_soa_to_aos(host)).cuda()
    t = Cn.Soax(Cn.R1, n)
    t.from_aos(aos0, n)
    for name, dt, dim in Cn.R1:
        for c in range(dim):
            assert torch.equal(t.comp_view(name, c).cpu(), torch.from_numpy(host[name][c])), (name, c)
    assert torch.equal(t.to_aos(), aos0)                            # byte-exact round trip at 2^24
    want = s.to_aos()
    for variant in (0, 1):
        a = aos0.clone()
        Cn.aos_step(Cn.R1, a, n, B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=100, variant=variant)
        assert torch.equal(a, want), f"AoS variant {variant} differs from SoA kernel + soa_to_aos"


def test_config4_full_size_sampled(gpu):
    """BASELINE.json config 4 as written: N = 2^26, record R2, inputs.make_r2(seed 0), 20 masked RK2 steps."""
    torch, B, Cn = gpu
    n = 1 << 26
    host = inputs.make_r2(n, seed=0, threads=os.cpu_count() or 8)
    s = Cn.Soax(Cn.R2, n)
    s.upload(host)
    idx = sample_indices(n)
    before = inputs.take(host, idx)
    e_before = s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC)
    s.step(B.SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED, DT, nsteps=20, k=1.0, flag_mask=1)
    got = gather(torch, s, idx)
    exp = oracle.rk2_midpoint_masked(before, DT, 20, k=1.0, mask=1)
    for name in exp:
        assert np.array_equal(bits(got[name]), bits(exp[name])), name
    active = (before["flags"][0] & 1) != 0
    assert 0.4 < active.mean() < 0.6
    assert (got["acc"][:, ~active] == 0).all() and (got["acc"][:, active] != 0).any()
    pos = torch.stack([s.comp_view("pos", c) for c in range(3)])
    assert bool((pos >= 0).all()) and bool((pos < 1).all())
    del pos
    # fields the step must not touch, bitwise over ALL particles; inactive particles bitwise unchanged in every field
    for name in ("id", "mass", "charge", "flags"):
        assert torch.equal(s.comp_view(name).cpu(), torch.from_numpy(host[name][0])), name
    inactive = torch.from_numpy((host["flags"][0] & 1) == 0)
    for name in ("pos", "vel", "acc"):
        for c in range(3):
            assert torch.equal(s.comp_view(name, c).cpu()[inactive], torch.from_numpy(host[name][c])[inactive]), (name, c)
    # the energy reduction on the double-velocity record at full size (a8 on R2): oracle = compensated sum in index order
    o_before = oracle.energy(host, oracle.KINETIC_PLUS_HARMONIC)
    assert abs(e_before - o_before) <= 1e-10 * o_before


def test_config5_full_size_vs_oracle(gpu):
    """BASELINE.json config 5 as written: N = 2^27, inputs.make_r1(seed 7), one drift step, 64^3 cells, counts, exclusive
    scan, stable permutation applied to all arrays, kinetic energy -- ids, counts, offsets and the permutation compared
    with the ORACLE over all 2^27 particles, bit for bit; every permuted array against oracle-drifted values gathered by
    the oracle's permutation."""
    torch, B, Cn = gpu
    n, G = 1 << 27, 64
    host = inputs.make_r1(n, seed=7, threads=os.cpu_count() or 8)
    src, dst = Cn.Soax(Cn.R1, n), Cn.Soax(Cn.R1, n)
    src.upload(host)
    r = src.bin_permute(dst, G, drift_dt=DT, want_kinetic=True)
    torch.cuda.synchronize()
    del r["scratch"]
    torch.cuda.empty_cache()
    for name, dt, dim in Cn.R1:                                      # src is read only (the drift is applied on the way to dst)
        for c in range(dim):
            assert torch.equal(src.comp_view(name, c).cpu(), torch.from_numpy(host[name][c])), (name, c)
    # the oracle on the whole set: drift, then cell / counts / scan / stable permutation
    aos = oracle.pack_r1(host)
    L = oracle.lib()
    L.soax_oracle_r1_drift(aos.ctypes.data, n, DT, 1)
    exp = {k: np.empty(m, np.uint32) for k, m in (("cell", n), ("counts", G ** 3), ("offsets", G ** 3), ("perm", n))}
    assert L.soax_oracle_r1_bin(aos.ctypes.data, n, G, exp["cell"].ctypes.data, exp["counts"].ctypes.data, exp["offsets"].ctypes.data,
                                exp["perm"].ctypes.data, None) == 0
    as_i32 = lambda a: torch.from_numpy(a.view(np.int32)).cuda()     # noqa: E731
    assert torch.equal(r["counts"], as_i32(exp["counts"]))
    assert torch.equal(r["offsets"], as_i32(exp["offsets"]))
    perm = as_i32(exp["perm"])
    assert torch.equal(r["perm"], perm)                              # the unique stable permutation, all 2^27 entries
    assert int(exp["counts"].sum()) == n
    perm = perm.to(torch.int64)
    drifted = oracle.unpack(aos)
    del aos, exp
    for name, dt, dim in Cn.R1:                                      # dst.f[j] == drifted.f[perm[j]] bitwise, every array
        for c in range(dim):
            want = torch.from_numpy(drifted[name][c]).cuda()[perm]
            assert torch.equal(dst.comp_view(name, c), want), (name, c)
            del want
    ids = torch.sort(dst.comp_view("id"))[0]
    assert torch.equal(ids, torch.arange(n, dtype=torch.int32, device="cuda"))     # ids stay a permutation
    ke = float(r["kinetic"].item())
    oke = oracle.energy(host, oracle.KINETIC)                        # the drift does not change vel
    assert abs(ke - oke) <= 1e-10 * oke and abs(ke / n - 1.5) < 1e-3
    # the same call IN PLACE (soax_bin_permute_inplace: the set returns to src, dst is the work area) must reproduce what was
    # just checked against the oracle, bit for bit, with half the scratch
    del drifted, perm, ids
    checked = dst.slab.clone()
    assert B.soax_scratch_bytes_inplace(src.layout, n, G) < 0.51 * B.soax_scratch_bytes(src.layout, n, G)
    r2 = src.bin_permute(dst, G, drift_dt=DT, want_kinetic=True, inplace=True)
    torch.cuda.synchronize()
    for k in ("counts", "offsets", "perm"):
        assert torch.equal(r2[k], r[k]), k
    assert float(r2["kinetic"].item()) == ke
    assert src.n == n and torch.equal(src.slab, checked)             # same layout, same capacity: the slabs are images of each other


# ---- NEXT-3 / NEXT-4 at the sizes bench.py times them (2^24): every row against the oracle ------------------------------------
# n = 2^24 + 3 is ragged and has 4097 mask tiles, so the one-CTA scan of the tile counts (kill_scan_kernel) walks five chunks
# of 1024 with its carry; the gather's table has 2 M segments; the mask program and the bulk getElement run at 2^24.
N_BIG = (1 << 24) + 3


@pytest.fixture(scope="module")
def big(gpu):
    torch, B, Cn = gpu
    host = inputs.make_r1(N_BIG, seed=11, threads=os.cpu_count() or 8)
    base = oracle.r1_soa_to_aos(host)
    s = Cn.Soax(Cn.R1, N_BIG)
    s.upload(host)
    return host, base, s


def big_masks(n):
    rng = np.random.default_rng(24)
    yield "random 10 %", (rng.random(n) < 0.1).astype(np.uint8)
    k = np.zeros(n, np.uint8); k[: n // 2] = 1; yield "front half (every hole below m, every mover above)", k
    k = np.zeros(n, np.uint8); k[n // 2:] = 200; yield "back half (pure truncation)", k


def test_remove_full_size_vs_oracle(gpu, big):
    """soax_remove over 2^24 + 3 particles in SWAP_LAST, STABLE and STABLE | KEEP_FLAGGED against the oracle's forward loop
    and stable filter, every byte of every surviving record (Q20)."""
    torch, B, Cn = gpu
    host, base, s = big
    n = N_BIG
    work, d = Cn.Soax(Cn.R1, 0, capacity=n), Cn.Soax(Cn.R1, 0, capacity=n)
    for what, kill in big_masks(n):
        kd = torch.from_numpy(kill).cuda()
        m_exp = int((kill == 0).sum())
        work.copy_from(s)
        assert work.remove(kd) == m_exp
        assert np.array_equal(work.to_aos().cpu().numpy(), oracle.remove_swap_last(base, 40, kill)), what
        assert s.remove(kd, stable=True, dst=d) == m_exp
        assert np.array_equal(d.to_aos().cpu().numpy(), oracle.remove_stable(base, 40, kill)), what
        s.remove_async(kd, stable=True, dst=d, keep_flagged=True)    # the same mask read the other way: the flagged rows stay
        assert d.n == n - m_exp
        assert np.array_equal(d.to_aos().cpu().numpy(), oracle.remove_stable(base, 40, (kill == 0).astype(np.uint8))), what
    assert s.n == n and np.array_equal(s.to_aos().cpu().numpy(), base)  # the source of the stable removals is untouched


def test_mask_program_full_size_vs_oracle(gpu, big):
    """The cell-range condition of the migration step (soax_expr_mask) over 2^24 + 3 particles against oracle.expr.mask."""
    from oracle import expr as oexpr
    torch, B, Cn = gpu
    host, base, s = big
    cond, sc = "(double(cell(64)) < lo) | (double(cell(64)) >= hi)", {"lo": 70000, "hi": 190000}
    got = Cn.MaskProgram(Cn.R1, cond, ["lo", "hi"]).mask(s, **sc).cpu().numpy()
    exp = oexpr.mask(host, cond, sc)
    assert got.shape == exp.shape and np.array_equal(got, exp) and 0 < int(exp.sum()) < N_BIG


def test_get_elements_full_size_vs_oracle(gpu, big):
    """Bulk getElement of 2^20 random rows (repeats, first and last row included) of the 2^24 + 3 against the oracle."""
    torch, B, Cn = gpu
    host, base, s = big
    rng = np.random.default_rng(5)
    idx = rng.integers(0, N_BIG, 1 << 20).astype(np.uint32)
    idx[:4] = [0, N_BIG - 1, N_BIG - 1, 0]
    got = s.get_elements(torch.from_numpy(idx.view(np.int32)).cuda()).cpu().numpy()
    assert np.array_equal(got, oracle.get_elements(base, 40, idx))


def test_gather_segments_full_size_vs_oracle(gpu, big):
    """The exchange's merge at the size bench.py times it: 8 runs, 64^3 cells = 2 097 152 segments (many empty or one row
    long), 2^24 + 3 rows, against the oracle's row loop.  The tables are built from random per-run per-cell counts the way
    dist.SoaxEngine.merge builds them; the records are the big set's bytes (a gather looks at no field)."""
    torch, B, Cn = gpu
    host, base, s = big
    world, ncell, n = 8, 64 ** 3, N_BIG
    rng = np.random.default_rng(8)
    cnt = rng.multinomial(n, np.full(world * ncell, 1.0 / (world * ncell))).reshape(world, ncell).astype(np.int64)
    sizes = cnt.sum(1)
    src_start = (np.cumsum(sizes) - sizes)[:, None] + np.cumsum(cnt, 1) - cnt
    flat = cnt.T.reshape(-1)
    seg_dst, seg_src = (np.cumsum(flat) - flat), src_start.T.reshape(-1)
    want = oracle.gather_segments_c(base, 40, seg_dst, seg_src, n)
    d = Cn.Soax(Cn.R1, 0, capacity=n)
    recs = torch.empty(n * 40 + 16, dtype=torch.uint8, device="cuda")
    recs[:n * 40] = torch.from_numpy(base).cuda()
    d.from_aos_segments(recs, torch.from_numpy(seg_dst.astype(np.int32)).cuda(), torch.from_numpy(seg_src.astype(np.int32)).cuda(), n)
    assert d.n == n and np.array_equal(d.to_aos().cpu().numpy(), want)
