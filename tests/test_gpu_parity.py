"""GPU parity: the CUDA path (through the C ABI, libsoax.so) against the oracle, element by element, on the same
seeded inputs.  Sizes span several tiles (4 particles/thread x 256 threads; 256-record transpose tiles; 4096-key
sort tiles) plus a ragged tail.  Bars (BASELINE.json north_star): ids / counts / offsets / perm bit-exact; double
positions within 1e-12 absolute (periodic distance); float velocities within 4 ulp; energy within 1e-10 relative.
Because both sides run the same IEEE operation sequence (explicit fma, no contraction) the EXPECTATION is
bit-equality, which the tests also assert where the arithmetic contract promises it.
"""
import numpy as np
import pytest

import oracle
from paper_1710_03462_b200 import inputs

pytestmark = pytest.mark.gpu

DT = 1e-3


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1710_03462_b200 import binding as B, container as Cn
    B.lib()                                     # fail loudly if libsoax.so is missing: there is no fallback
    return torch, B, Cn


def bits(a):
    a = np.ascontiguousarray(a)
    return a.view({4: np.uint32, 8: np.uint64, 1: np.uint8}[a.dtype.itemsize])


def pdist(a, b):
    d = np.abs(np.asarray(a, np.float64) - np.asarray(b, np.float64))
    return np.minimum(d, 1.0 - d)


def ulp_dist32(a, b):
    """distance in units in the last place between float32 arrays (sign-magnitude -> ordered integers)"""
    def ordered(x):
        i = np.ascontiguousarray(x).view(np.int32).astype(np.int64)
        return np.where(i < 0, -(i & 0x7FFFFFFF), i)
    return np.abs(ordered(a) - ordered(b))


def check_r1(got, exp, expect_bits=True):
    assert np.array_equal(got["id"], exp["id"])
    assert pdist(got["pos"], exp["pos"]).max() <= 1e-12
    assert ulp_dist32(got["vel"], exp["vel"]).max() <= 4
    assert (got["pos"] >= 0).all() and (got["pos"] < 1).all()
    if expect_bits:
        assert np.array_equal(bits(got["pos"]), bits(exp["pos"])), "positions differ in some bit"
        assert np.array_equal(bits(got["vel"]), bits(exp["vel"])), "velocities differ in some bit"


def to_device(Cn, fields, host):
    n = next(iter(host.values())).shape[1]
    s = Cn.Soax(fields, n)
    s.upload(host)
    return s


# ------------------------------------------------------------------------------------------ a2: drift (config 1)
@pytest.mark.parametrize("n", [65536, 4099, 3, 1, 0])
@pytest.mark.parametrize("ppt", [4, 2, 1])
def test_drift_config1(gpu, n, ppt):
    torch, B, Cn = gpu
    B.soax_tune("step_ppt", ppt)
    try:
        host = inputs.make_r1(n, seed=0)
        s = to_device(Cn, Cn.R1, host)
        s.step(B.SOAX_STEP_DRIFT, DT, nsteps=10)
        got = s.download()
    finally:
        B.soax_tune("step_ppt", 4)
    exp = oracle.drift(host, DT, 10) if n else host
    if n:
        check_r1(got, exp)
        assert np.array_equal(bits(got["vel"]), bits(host["vel"]))        # vel untouched


def test_drift_face_crossings_and_special_values(gpu):
    torch, B, Cn = gpu
    host = inputs.make_r1(1000, seed=5)
    host["vel"] *= np.float32(400.0)                                  # |dt v| up to ~2: wraps, incl. the slow floor path
    host["pos"][0, :8] = [0.0, 0.999, 0.001, 1.0 - 2.0 ** -53, 0.0, 0.5, 0.0, 2.0 ** -1074]
    host["vel"][0, :8] = [-1e-17, 2.0, -2.0, 1e-20, -0.0, 3000.0, -2500.0, -1e-30]
    s = to_device(Cn, Cn.R1, host)
    s.step(B.SOAX_STEP_DRIFT, DT, nsteps=3)
    check_r1(s.download(), oracle.drift(host, DT, 3))


# ------------------------------------------------------------------------- a4 + a8: symplectic Euler (config 2)
@pytest.mark.parametrize("n,nsteps", [(1 << 16, 100), (10007, 7)])
def test_symplectic_euler_and_energy(gpu, n, nsteps):
    torch, B, Cn = gpu
    host = inputs.make_r1(n, seed=0)
    s = to_device(Cn, Cn.R1, host)
    e0 = s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC)
    s.step(B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=nsteps)
    e1 = s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC)
    ke1 = s.energy(B.SOAX_ENERGY_KINETIC)
    got = s.download()
    exp = oracle.symplectic_euler(host, DT, nsteps)
    check_r1(got, exp)
    o0 = oracle.energy(host, oracle.KINETIC_PLUS_HARMONIC)
    o1 = oracle.energy(exp, oracle.KINETIC_PLUS_HARMONIC)
    assert abs(e0 - o0) <= 1e-10 * abs(o0) and abs(e1 - o1) <= 1e-10 * abs(o1)
    assert abs(ke1 - oracle.energy(exp, oracle.KINETIC)) <= 1e-10 * abs(ke1)
    assert s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC) == e1          # run-to-run deterministic


def test_symplectic_euler_general_k_and_center(gpu):
    torch, B, Cn = gpu
    host = inputs.make_r1(5000, seed=3)
    s = to_device(Cn, Cn.R1, host)
    s.step(B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=5, k=2.5, center=0.25)
    check_r1(s.download(), oracle.symplectic_euler(host, DT, 5, k=2.5, center=0.25))
    e = s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC, k=2.5, center=0.25)
    o = oracle.energy(s.download(), oracle.KINETIC_PLUS_HARMONIC, k=2.5, center=0.25)
    assert abs(e - o) <= 1e-10 * abs(o)


@pytest.mark.parametrize("n", [1, 3, 4099, 100003])
def test_energy_wide_record_r2(gpu, n):
    """a8 on the double-velocity record R2 (config 4's layout): both kinds, general k / centre, ragged tails."""
    torch, B, Cn = gpu
    host = inputs.make_r2(n, seed=11)
    host["acc"][:] = np.random.default_rng(1).normal(size=host["acc"].shape)       # must not enter the sum
    s = to_device(Cn, Cn.R2, host)
    for kind, okind, k, ctr in ((B.SOAX_ENERGY_KINETIC, oracle.KINETIC, 1.0, 0.5),
                                (B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC, oracle.KINETIC_PLUS_HARMONIC, 1.0, 0.5),
                                (B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC, oracle.KINETIC_PLUS_HARMONIC, 2.5, 0.25)):
        e = s.energy(kind, k=k, center=ctr)
        o = oracle.energy(host, okind, k=k, center=ctr)
        assert abs(e - o) <= 1e-10 * abs(o), (kind, k, ctr)
        assert s.energy(kind, k=k, center=ctr) == e                                  # run-to-run deterministic
    if n == 1:                                                                       # one particle: no summation, bit-equal terms
        assert s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC, k=2.5, center=0.25) == oracle.energy(host, oracle.KINETIC_PLUS_HARMONIC, 2.5, 0.25)


def test_energy_hand_fixture_r2_on_gpu(gpu):
    torch, B, Cn = gpu
    vel = np.array([[1, 2, 2], [0, 0, 0], [3, 4, 0], [-1, -1, -1]], np.float64)       # tests/golden/energy_4particles.txt
    pos = np.array([[.5, .5, .5], [0, .5, .5], [.25, .75, .5], [.5, .5, 0]], np.float64)
    host = {"id": np.arange(4, dtype=np.int64)[None, :].copy(), "pos": np.ascontiguousarray(pos.T), "vel": np.ascontiguousarray(vel.T),
            "acc": np.full((3, 4), 7.0), "mass": np.array([[3, 5, 9, 17]], np.float32), "charge": np.array([[-1, 1, -1, 1]], np.float32),
            "flags": np.array([[1, 2, 3, 4]], np.uint8)}
    s = to_device(Cn, Cn.R2, host)
    assert s.energy(B.SOAX_ENERGY_KINETIC) == 18.5
    assert s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC) == 18.8125
    assert s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC, k=4.0) == 18.5 + 4.0 * 0.3125


def test_energy_hand_fixture_on_gpu(gpu):
    torch, B, Cn = gpu
    vel = np.array([[1, 2, 2], [0, 0, 0], [3, 4, 0], [-1, -1, -1]], np.float32).T.copy()
    pos = np.array([[.5, .5, .5], [0, .5, .5], [.25, .75, .5], [.5, .5, 0]], np.float64).T.copy()
    s = to_device(Cn, Cn.R1, {"id": np.arange(4, dtype=np.int32)[None], "pos": pos, "vel": vel})
    assert s.energy(B.SOAX_ENERGY_KINETIC) == 18.5                      # tests/golden/energy_4particles.txt
    assert s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC) == 18.8125


# ------------------------------------------------------------------------------- a5, a6, a7: AoS (config 3)
# shape = (xpose_ring, xpose_r, xpose_ns, xpose_ctas): the default ring transposes, the one-tile-per-visit kernels they
# replaced, and ring shapes forced deep (two stages, one CTA per SM: every CTA walks many tiles) at a size with a tail
@pytest.mark.parametrize("n,shape", [(1 << 16, (1, 0, 0, 0)), (70001, (1, 0, 0, 0)), (255, (1, 0, 0, 0)), (1, (1, 0, 0, 0)),
                                     (70001, (0, 0, 0, 0)), (255, (0, 0, 0, 0)),
                                     (1024 * 700 + 13, (1, 1, 2, 1)), (1024 * 700 + 13, (1, 4, 2, 1)), (1024 * 700 + 13, (1, 2, 1, 1))])
def test_aos_soa_transposes_byte_exact(gpu, n, shape):
    torch, B, Cn = gpu
    rng = np.random.default_rng(n)
    raw = rng.integers(0, 256, 40 * n, dtype=np.uint8)                # arbitrary bytes: NaN payloads, denormals, ...
    aos = torch.from_numpy(raw).cuda()
    s = Cn.Soax(Cn.R1, n)
    try:
        for key, v in zip(("xpose_ring", "xpose_r", "xpose_ns", "xpose_ctas"), shape):
            B.soax_tune(key, v)
        s.from_aos(aos, n)
        got = s.download()
        back = s.to_aos()
    finally:
        for key, v in (("xpose_ring", 1), ("xpose_r", 0), ("xpose_ns", 0), ("xpose_ctas", 0)):
            B.soax_tune(key, v)
    exp = oracle.r1_aos_to_soa(raw)
    for name in exp:
        assert np.array_equal(bits(got[name]), bits(exp[name])), name
    assert np.array_equal(back.cpu().numpy(), raw)                    # round trip is byte exact
    assert np.array_equal(oracle.r1_soa_to_aos(exp), raw)


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("n", [1 << 16, 7001])
def test_aos_step_matches_oracle_and_soa_kernel(gpu, variant, n):
    torch, B, Cn = gpu
    host = inputs.make_r1(n, seed=0)
    raw = oracle.r1_soa_to_aos(host)
    aos = torch.from_numpy(raw).cuda()
    Cn.aos_step(Cn.R1, aos, n, B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=20, variant=variant)
    got = oracle.r1_aos_to_soa(aos.cpu().numpy())
    check_r1(got, oracle.symplectic_euler(host, DT, 20))
    # oracle-free cross-check: SoA kernel + SoA->AoS must reproduce the AoS kernel's bytes
    s = to_device(Cn, Cn.R1, host)
    s.step(B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=20)
    assert torch.equal(s.to_aos(), aos)
    aos2 = torch.from_numpy(raw).cuda()
    Cn.aos_step(Cn.R1, aos2, n, B.SOAX_STEP_DRIFT, DT, nsteps=3, variant=variant)
    check_r1(oracle.r1_aos_to_soa(aos2.cpu().numpy()), oracle.drift(host, DT, 3))


def test_transposes_wide_record(gpu):
    torch, B, Cn = gpu
    n = 5003
    host = inputs.make_r2(n, seed=2)
    s = to_device(Cn, Cn.R2, host)
    aos = s.to_aos()
    stride, offs = B.soax_layout_aos(s.layout, True)
    assert stride == 89
    raw = aos.cpu().numpy().reshape(n, stride)
    c = 0
    for name, dt, dim in Cn.R2:
        for k in range(dim):
            sz = B.DTYPE_SIZE[dt]
            col = np.ascontiguousarray(raw[:, offs[c]:offs[c] + sz]).view(Cn.NP_DTYPE[dt])[:, 0]
            assert np.array_equal(bits(col), bits(host[name][k])), (name, k)
            c += 1
    t = Cn.Soax(Cn.R2, n)
    t.from_aos(aos, n)
    back = t.download()
    for name in host:
        assert np.array_equal(bits(back[name]), bits(host[name])), name


# ----------------------------------------------------------------------------------------- a9: RK2 (config 4)
@pytest.mark.parametrize("n,nsteps,mask", [(1 << 15, 20, 1), (4099, 3, 0x10), (257, 2, 0xFF)])
def test_rk2_masked_wide_record(gpu, n, nsteps, mask):
    torch, B, Cn = gpu
    host = inputs.make_r2(n, seed=0)
    if n == 4099:
        host["vel"] *= 300.0                                          # wraps at the midpoint and at the end
    s = to_device(Cn, Cn.R2, host)
    s.step(B.SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED, DT, nsteps=nsteps, k=1.0, flag_mask=mask)
    got = s.download()
    exp = oracle.rk2_midpoint_masked(host, DT, nsteps, k=1.0, mask=mask)
    assert pdist(got["pos"], exp["pos"]).max() <= 1e-12
    assert np.abs(got["vel"] - exp["vel"]).max() <= 1e-12 and np.abs(got["acc"] - exp["acc"]).max() <= 1e-12
    for name in host:                                                 # the contract promises bit equality
        assert np.array_equal(bits(got[name]), bits(exp[name])), name
    inactive = (host["flags"][0] & mask) == 0
    for name in host:
        assert np.array_equal(bits(got[name])[:, inactive], bits(host[name])[:, inactive]), name


def test_rk2_acc_of_inactive_particles_is_preserved(gpu):
    torch, B, Cn = gpu
    host = inputs.make_r2(1001, seed=4)
    host["acc"][:] = np.random.default_rng(0).normal(size=host["acc"].shape)   # not zero: must survive bit for bit
    s = to_device(Cn, Cn.R2, host)
    s.step(B.SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED, DT, nsteps=1)
    got, exp = s.download(), oracle.rk2_midpoint_masked(host, DT, 1)
    for name in host:
        assert np.array_equal(bits(got[name]), bits(exp[name])), name


def test_drift_wide_record(gpu):
    torch, B, Cn = gpu
    host = inputs.make_r2(3001, seed=6)
    s = to_device(Cn, Cn.R2, host)
    s.step(B.SOAX_STEP_DRIFT, DT, nsteps=4)
    got, exp = s.download(), oracle.drift(host, DT, 4)
    for name in host:
        assert np.array_equal(bits(got[name]), bits(exp[name])), name


# ------------------------------------------------------------------------------ a10..a14: binning (config 5)
def run_bin(gpu, host, G, drift_dt=0.0, kinetic=False):
    torch, B, Cn = gpu
    n = host["id"].shape[1]
    src, dst = to_device(Cn, Cn.R1, host), Cn.Soax(Cn.R1, n)
    r = src.bin_permute(dst, G, drift_dt=drift_dt, want_kinetic=kinetic)
    torch.cuda.synchronize()
    out = {k: (v.cpu().numpy().view(np.uint32) if k in ("counts", "offsets", "perm") else v) for k, v in r.items()}
    return src.download(), (dst.download() if n else None), out


def check_bin(host_after_drift, sorted_soa, out, G):
    exp = oracle.bin_r1(host_after_drift, G)
    assert np.array_equal(out["counts"], exp["counts"])
    assert np.array_equal(out["offsets"], exp["offsets"])
    assert np.array_equal(out["perm"], exp["perm"])
    want = oracle.permute_r1(host_after_drift, exp["perm"])
    for name in want:
        assert np.array_equal(bits(sorted_soa[name]), bits(want[name])), name
    assert int(out["counts"].sum()) == host_after_drift["id"].shape[1]


@pytest.fixture(params=[(0, 0, 1), (9, 1, 1), (6, 0, 1), (4, 8, 1), (9, 16, 0), (7, 2, 1)],
                ids=["default-9bit-cluster4", "9bit-no-cluster", "6bit-3pass", "4bit-5pass-cluster8", "9bit-cluster16-nosync", "7bit-cluster2"])
def bin_stage(request, gpu):
    """every digit width (1..5 passes) and launch shape (cluster size, cluster barrier on/off) of the counting sort
    (soax_tune bin_bits / bin_cluster / bin_csync) must give the same unique result"""
    for key, v in zip(("bin_bits", "bin_cluster", "bin_csync"), request.param):
        gpu[1].soax_tune(key, v)
    yield request.param
    for key, v in (("bin_bits", 0), ("bin_cluster", 0), ("bin_csync", 1)):
        gpu[1].soax_tune(key, v)


@pytest.mark.parametrize("n,G", [(100003, 64), (4096, 64), (4097, 8), (50000, 2), (31, 64), (1, 64), (70000, 1), (8191, 64)])
def test_bin_permute_matches_oracle(gpu, bin_stage, n, G):
    host = inputs.make_r1(n, seed=7)
    src_after, sorted_soa, out = run_bin(gpu, host, G)
    for name in host:                                                 # no drift requested: src is read only
        assert np.array_equal(bits(src_after[name]), bits(host[name]))
    check_bin(host, sorted_soa, out, G)


@pytest.mark.parametrize("case", ["one_cell", "sorted", "reverse", "two_cells_far"])
def test_bin_permute_degenerate_distributions(gpu, bin_stage, case):
    n, G = 20011, 64
    host = inputs.make_r1(n, seed=9)
    if case == "one_cell":
        host["pos"][:] = 0.99 + 0.005 * host["pos"]                   # everything in the last cell
    elif case in ("sorted", "reverse"):
        order = np.argsort(oracle.bin_r1(host, G)["cell"], kind="stable")
        host = inputs.take(host, order if case == "sorted" else order[::-1].copy())
    else:
        host["pos"][:, ::2] = 0.001
        host["pos"][:, 1::2] = 0.999
    src_after, sorted_soa, out = run_bin(gpu, host, G)
    check_bin(host, sorted_soa, out, G)


def test_bin_permute_fused_drift_and_kinetic_config5_shape(gpu):
    torch, B, Cn = gpu
    n, G = 1 << 17, 64
    host = inputs.make_r1(n, seed=7)
    src_after, sorted_soa, out = run_bin(gpu, host, G, drift_dt=DT, kinetic=True)
    drifted = oracle.drift(host, DT, 1)
    for name in host:                                                 # src is read only: the drift is applied on the way to dst
        assert np.array_equal(bits(src_after[name]), bits(host[name])), name
    check_bin(drifted, sorted_soa, out, G)                            # dst = the DRIFTED particles in cell order, bit for bit
    ke = float(out["kinetic"].item())
    oke = oracle.energy(drifted, oracle.KINETIC)
    assert abs(ke - oke) <= 1e-10 * oke
    assert np.array_equal(np.sort(sorted_soa["id"][0]), np.arange(n, dtype=np.int32))   # ids stay a permutation


def test_bin_permute_wide_record_r2_with_drift(gpu):
    """binning of the 13-array record R2 (double vel): the drift fused into the first pass uses the double-velocity fma;
    every one of the 13 arrays is permuted.  Oracle: r2 drift, then the R1 binning oracle on the drifted positions."""
    torch, B, Cn = gpu
    n, G = 30011, 16
    host = inputs.make_r2(n, seed=3)
    host["acc"][:] = np.random.default_rng(2).normal(size=host["acc"].shape)
    src, dst = to_device(Cn, Cn.R2, host), Cn.Soax(Cn.R2, n)
    r = src.bin_permute(dst, G, drift_dt=DT, want_kinetic=True)
    torch.cuda.synchronize()
    drifted = oracle.drift(host, DT, 1)
    as_r1 = {"id": np.zeros((1, n), np.int32), "pos": drifted["pos"], "vel": np.zeros((3, n), np.float32)}
    exp = oracle.bin_r1(as_r1, G)
    for k in ("counts", "offsets", "perm"):
        assert np.array_equal(r[k].cpu().numpy().view(np.uint32), exp[k]), k
    got = dst.download()
    for name in host:
        assert np.array_equal(bits(got[name]), bits(drifted[name][:, exp["perm"]])), name
    assert np.array_equal(bits(src.download()["pos"]), bits(host["pos"]))             # src untouched
    oke = oracle.energy(host, oracle.KINETIC)
    assert abs(float(r["kinetic"].item()) - oke) <= 1e-10 * oke


@pytest.mark.parametrize("want", ["none", "perm_only", "counts_only", "offsets_kinetic"])
def test_bin_permute_optional_outputs(gpu, want):
    """dev_counts / dev_offsets / dev_perm / dev_kinetic may each be NULL: the arrays are still permuted, and the outputs
    that are asked for are the same as when all are asked for (the carried index / the sorted keys are skipped otherwise)."""
    torch, B, Cn = gpu
    n, G = 50021, 64
    host = inputs.make_r1(n, seed=5)
    src, dst = to_device(Cn, Cn.R1, host), Cn.Soax(Cn.R1, n)
    exp = oracle.bin_r1(host, G)
    want_sorted = oracle.permute_r1(host, exp["perm"])
    i32 = lambda m: torch.full((m,), -1, dtype=torch.int32, device="cuda")           # noqa: E731
    counts, offsets, perm, kin = i32(G ** 3), i32(G ** 3), i32(n), torch.zeros(1, dtype=torch.float64, device="cuda")
    scratch = torch.empty(B.soax_scratch_bytes(src.layout, n, G), dtype=torch.uint8, device="cuda")
    use = {"none": (), "perm_only": ("perm",), "counts_only": ("counts",), "offsets_kinetic": ("offsets", "kinetic")}[want]
    B.soax_bin_permute(src.handle, dst.handle, G, 0.0, counts.data_ptr() if "counts" in use else None,
                       offsets.data_ptr() if "offsets" in use else None, perm.data_ptr() if "perm" in use else None,
                       kin.data_ptr() if "kinetic" in use else None, scratch.data_ptr(), scratch.numel(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    got = dst.download()
    for name in want_sorted:
        assert np.array_equal(bits(got[name]), bits(want_sorted[name])), name
    for name, t in (("counts", counts), ("offsets", offsets), ("perm", perm)):
        if name in use:
            assert np.array_equal(t.cpu().numpy().view(np.uint32), exp[name]), name
        else:
            assert bool((t == -1).all()), name                                       # not asked for: not written
    if "kinetic" in use:
        oke = oracle.energy(host, oracle.KINETIC)
        assert abs(float(kin.item()) - oke) <= 1e-10 * oke


@pytest.mark.parametrize("n,G,drift", [(100003, 64, 0.0), (4097, 16, DT), (8191, 32, 0.0), (1, 64, DT), (0, 64, 0.0)])
def test_bin_permute_inplace_r1(gpu, n, G, drift):
    """soax_bin_permute_inplace: the sorted [drifted] set returns to the SAME container, the second one is a work area;
    counts / offsets / perm / every array equal the oracle's, as for the out-of-place call; the scratch is smaller."""
    torch, B, Cn = gpu
    host = inputs.make_r1(n, seed=11)
    s, work = to_device(Cn, Cn.R1, host), Cn.Soax(Cn.R1, max(n, 1))
    need_in, need_out = B.soax_scratch_bytes_inplace(s.layout, max(n, 1), G), B.soax_scratch_bytes(s.layout, max(n, 1), G)
    assert 0 < need_in <= need_out and (n < 4096 or need_out - need_in >= 23 * n)   # R1: 48 -> 24 bytes per particle (give or take the 256-byte alignment)
    r = s.bin_permute(work, G, drift_dt=drift, want_kinetic=True, inplace=True)
    torch.cuda.synchronize()
    assert s.n == n
    if n == 0:
        assert int(r["counts"].sum()) == 0
        return
    after = oracle.drift(host, drift, 1) if drift else host
    out = {k: r[k].cpu().numpy().view(np.uint32) for k in ("counts", "offsets", "perm")}
    check_bin(after, s.download(), out, G)
    oke = oracle.energy(host, oracle.KINETIC)
    assert abs(float(r["kinetic"].item()) - oke) <= 1e-10 * max(oke, 1e-300)


def test_bin_permute_inplace_r2_and_limits(gpu):
    """the 13-array record in place (its 8-byte arrays travel through the work container, mass/charge as a pair and the
    flags through scratch), without a carried index; grids that need one or three passes answer UNSUPPORTED."""
    torch, B, Cn = gpu
    n, G = 30011, 16
    host = inputs.make_r2(n, seed=5)
    host["acc"][:] = np.random.default_rng(3).normal(size=host["acc"].shape)
    s, work = to_device(Cn, Cn.R2, host), Cn.Soax(Cn.R2, n)
    scratch = torch.empty(B.soax_scratch_bytes_inplace(s.layout, n, G), dtype=torch.uint8, device="cuda")
    counts = torch.empty(G ** 3, dtype=torch.int32, device="cuda")
    B.soax_bin_permute_inplace(s.handle, work.handle, G, DT, counts.data_ptr(), None, None, None, scratch.data_ptr(), scratch.numel(),
                               torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    drifted = oracle.drift(host, DT, 1)
    as_r1 = {"id": np.zeros((1, n), np.int32), "pos": drifted["pos"], "vel": np.zeros((3, n), np.float32)}
    exp = oracle.bin_r1(as_r1, G)
    assert np.array_equal(counts.cpu().numpy().view(np.uint32), exp["counts"])
    got = s.download()
    for name in host:
        assert np.array_equal(bits(got[name]), bits(drifted[name][:, exp["perm"]])), name
    assert B.soax_scratch_bytes_inplace(s.layout, n, 8) == 0            # 9 key bits: one pass, the set would end in `work`
    with pytest.raises(Exception):
        B.soax_bin_permute_inplace(s.handle, work.handle, 8, 0.0, None, None, None, None, scratch.data_ptr(), scratch.numel(), 0)
    with pytest.raises(Exception):                                       # a container cannot be its own work area
        B.soax_bin_permute_inplace(s.handle, s.handle, G, 0.0, None, None, None, None, scratch.data_ptr(), scratch.numel(), 0)


def test_bin_empty(gpu):
    torch, B, Cn = gpu
    host = inputs.make_r1(0, seed=1)
    _, _, out = run_bin(gpu, host, 4)
    assert out["counts"].sum() == 0 and out["offsets"].sum() == 0


# ----------------------------------------------------------------------- NEXT-1: the paper's float benchmark
@pytest.mark.parametrize("size_extra", [0, 8, 32])
def test_paper_float_benchmark_euler(gpu, size_extra):
    torch, B, Cn = gpu
    n = 10001
    host = inputs.make_b6(n, seed=1)
    full = dict(host)
    if size_extra:
        full["temp"] = np.zeros((size_extra, n), np.float32)
    s = to_device(Cn, Cn.B6(size_extra), full)
    s.step(B.SOAX_STEP_EULER_NOWRAP, 1e-3, nsteps=5)
    got = s.download()
    epos, evel = oracle.b6_euler(host["pos"], host["vel"], size_extra, np.float32(1e-3), 5)
    assert np.array_equal(bits(got["pos"]), bits(epos)) and np.array_equal(bits(got["vel"]), bits(evel))


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("size_extra,n", [(0, 10001), (8, 4099), (32, 777)])
def test_paper_float_benchmark_aos_kernels(gpu, size_extra, n, variant):
    """K5 on the paper's own record Particle<SIZE> (Listing 4): both AoS kernels equal the oracle
    bitwise, leave v and temp[SIZE] untouched, and equal the SoA kernel (same operation sequence)."""
    torch, B, Cn = gpu
    host = inputs.make_b6(n, seed=2)
    rec = np.zeros((n, 6 + size_extra), np.float32)
    rec[:, 0:3], rec[:, 3:6] = host["pos"].T, host["vel"].T
    rec[:, 6:] = np.arange(n * size_extra, dtype=np.float32).reshape(n, size_extra)
    stride, offs = B.soax_layout_aos(B.soax_layout_define(Cn.B6(size_extra)), True)
    assert stride == 24 + 4 * size_extra and list(offs[:6]) == [0, 4, 8, 12, 16, 20]      # 24 bytes at SIZE=0
    aos = torch.from_numpy(rec.view(np.uint8).reshape(-1).copy()).cuda()
    Cn.aos_step(Cn.B6(size_extra), aos, n, B.SOAX_STEP_EULER_NOWRAP, 1e-3, 5, variant)
    got = aos.cpu().numpy().view(np.float32).reshape(n, 6 + size_extra)
    epos, evel = oracle.b6_euler(host["pos"], host["vel"], size_extra, np.float32(1e-3), 5)
    assert np.array_equal(bits(got[:, 0:3].T), bits(epos))
    assert np.array_equal(bits(got[:, 3:6].T), bits(evel))
    assert np.array_equal(got[:, 6:], rec[:, 6:])
    full = dict(host)
    if size_extra:
        full["temp"] = np.ascontiguousarray(rec[:, 6:].T)
    s = to_device(Cn, Cn.B6(size_extra), full)
    s.step(B.SOAX_STEP_EULER_NOWRAP, 1e-3, nsteps=5)
    assert np.array_equal(s.to_aos().cpu().numpy(), got.view(np.uint8).reshape(-1))


# ------------------------------------------------------------------------------- graph replay of the step loop
def test_step_graph_replay_on_side_stream(gpu):
    """soax_step(nsteps >= 2) on a capturable stream replays a captured graph: same bits as the oracle, also when the
    call is repeated (replay), when its parameters change (re-capture) and after a resize."""
    torch, B, Cn = gpu
    n = 30011
    host = inputs.make_r1(n, seed=5)
    with torch.cuda.stream(torch.cuda.Stream()):
        s = to_device(Cn, Cn.R1, host)
        l0 = B.soax_launch_count()
        s.step(B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=7)      # capture + launch
        s.step(B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=7)      # replay
        s.step(B.SOAX_STEP_DRIFT, DT, nsteps=3)                          # other parameters: re-capture
        s.step(B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, 2 * DT, nsteps=7)
        assert B.soax_launch_count() - l0 == 7 + 7 + 3 + 7
        torch.cuda.current_stream().synchronize()
        exp = oracle.symplectic_euler(oracle.drift(oracle.symplectic_euler(host, DT, 14), DT, 3), 2 * DT, 7)
        check_r1(s.download(), exp)
        B.soax_resize(s.handle, 1000)                                    # fewer live particles: the old graph must not run
        s.step(B.SOAX_STEP_DRIFT, DT, nsteps=3)
        torch.cuda.current_stream().synchronize()
        B.soax_resize(s.handle, n)
        got = s.download()
        exp2 = oracle.drift(inputs.take(exp, np.arange(1000)), DT, 3)
        for name in exp2:
            assert np.array_equal(bits(got[name][:, :1000]), bits(exp2[name])), name
            assert np.array_equal(bits(got[name][:, 1000:]), bits(exp[name][:, 1000:])), name


# ------------------------------------------------------------------------------------------- error behaviour
def test_error_codes(gpu):
    torch, B, Cn = gpu
    s = Cn.Soax(Cn.R1, 100)
    with pytest.raises(B.SoaxError) as e:
        B.soax_field_ptr(s.handle, 1, 3)                              # pos(42) on a 3-vector
    assert e.value.status == B.SOAX_ERR_UNSUPPORTED
    with pytest.raises(B.SoaxError) as e:
        s.step(B.SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED, DT)          # R1 has no acc/mass/flags
    assert e.value.status == B.SOAX_ERR_UNSUPPORTED
    with pytest.raises(B.SoaxError) as e:
        B.soax_resize(s.handle, 101)
    assert e.value.status == B.SOAX_ERR_INVALID_ARG
    b6 = Cn.Soax(Cn.B6(0), 10)
    with pytest.raises(B.SoaxError) as e:
        b6.bin_permute(Cn.Soax(Cn.B6(0), 10), 4, scratch=torch.empty(1 << 20, dtype=torch.uint8, device="cuda"))
    assert e.value.status == B.SOAX_ERR_UNSUPPORTED


@pytest.mark.parametrize("variant", [0, 1])
def test_reordered_record_aos_kernels(gpu, variant):
    """Q1 sensitivity row: the record declared {pos; vel; id} (packed offsets 0/24/36, naturally aligned).  Same fields,
    same arithmetic: the SoA kernel must match the oracle, and SoA kernel + SoA->AoS must reproduce the AoS kernel's bytes."""
    torch, B, Cn = gpu
    n = 70001
    host = inputs.make_r1(n, seed=9)
    stride, offs = B.soax_layout_aos(B.soax_layout_define(Cn.R1R), True)
    assert stride == 40 and offs == [0, 8, 16, 24, 28, 32, 36]
    s = to_device(Cn, Cn.R1R, host)
    aos = s.to_aos()
    packed = np.zeros(n, np.dtype({"names": ["pos", "vel", "id"], "formats": [("<f8", 3), ("<f4", 3), "<i4"], "offsets": [0, 24, 36], "itemsize": 40}))
    packed["pos"], packed["vel"], packed["id"] = host["pos"].T, host["vel"].T, host["id"][0]
    assert np.array_equal(aos.cpu().numpy(), packed.view(np.uint8).reshape(-1))       # the packed image is the numpy struct
    s.step(B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=7)
    check_r1(s.download(), oracle.symplectic_euler(host, DT, 7))
    Cn.aos_step(Cn.R1R, aos, n, B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC, DT, nsteps=7, variant=variant)
    assert torch.equal(s.to_aos(), aos)
    t = Cn.Soax(Cn.R1R, n)
    t.from_aos(aos, n)
    check_r1(t.download(), oracle.symplectic_euler(host, DT, 7))
