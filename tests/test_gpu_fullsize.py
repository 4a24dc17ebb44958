"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default tuning).

The oracle cannot step 2^24..2^27 particles in seconds, but particles are independent, so it is run on SAMPLED
particles (the same seeded inputs, gathered before the device steps) and compared bit for bit with the device's
result at those indices; whole-array statements use properties that hold at any size and library routines that are
independent of the CUDA path (torch.sort(stable=True) for the unique stable permutation, torch.bincount / cumsum for
counts and offsets, a gather for the permuted arrays)."""
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


def device_fill(torch, s, seed):
    from bench import device_fill as fill
    fill(torch, s, seed)


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
    torch, B, Cn = gpu
    n = 1 << 26
    s = Cn.Soax(Cn.R2, n)
    device_fill(torch, s, 0)
    idx = sample_indices(n)
    before = gather(torch, s, idx)
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


def test_config5_full_size_properties(gpu):
    torch, B, Cn = gpu
    n, G = 1 << 27, 64
    src, dst = Cn.Soax(Cn.R1, n), Cn.Soax(Cn.R1, n)
    device_fill(torch, src, 7)
    idx = sample_indices(n)
    before = gather(torch, src, idx)
    r = src.bin_permute(dst, G, drift_dt=DT, want_kinetic=True)
    torch.cuda.synchronize()
    del r["scratch"]
    torch.cuda.empty_cache()
    # fused drift, sampled against the oracle
    after = gather(torch, src, idx)
    exp = oracle.drift(before, DT, 1)
    for name in exp:
        assert np.array_equal(bits(after[name]), bits(exp[name])), name
    # cell keys recomputed with torch from the drifted positions (exact: x*64 then truncation)
    cell = torch.zeros(n, dtype=torch.int64, device="cuda")
    for c in range(3):
        cell = cell * G + (src.comp_view("pos", c) * float(G)).to(torch.int64)
    assert int(cell.min()) >= 0 and int(cell.max()) < G ** 3
    counts = torch.bincount(cell, minlength=G ** 3)
    assert torch.equal(r["counts"].to(torch.int64), counts)
    assert int(counts.sum()) == n
    offs = torch.cumsum(counts, 0) - counts
    assert torch.equal(r["offsets"].to(torch.int64), offs)
    del counts, offs
    # the stable permutation is unique: it must equal a stable argsort of the keys
    perm = r["perm"].to(torch.int64)
    _, order = torch.sort(cell.to(torch.int32), stable=True)
    assert torch.equal(perm, order)
    del order, cell
    torch.cuda.empty_cache()
    # every component array was permuted: new.f[j] == old.f[perm[j]] bitwise
    for name, dt, dim in Cn.R1:
        for c in range(dim):
            assert torch.equal(dst.comp_view(name, c), src.comp_view(name, c)[perm]), (name, c)
    ids = torch.sort(dst.comp_view("id"))[0]
    assert torch.equal(ids, torch.arange(n, dtype=torch.int32, device="cuda"))     # ids stay a permutation
    ke = float(r["kinetic"].item())
    ref = 0.5 * sum(float((src.comp_view("vel", c).double() ** 2).sum()) for c in range(3))
    assert abs(ke - ref) <= 1e-10 * ref and abs(ke / n - 1.5) < 1e-3
