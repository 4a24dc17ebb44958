"""GPU parity of NEXT-3 (container operations): removal by kill mask (the paper's
overwrite-with-last, and a stable compaction), push_back of AoS records, bulk getElement and copy -- byte-exact
against the oracle on the packed AoS image of the container (every component of every row is compared)."""
import numpy as np
import pytest

import oracle
from paper_1710_03462_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1710_03462_b200 import binding as B, container as Cn
    B.lib()
    return torch, B, Cn


def device(Cn, fields, host, capacity=None):
    n = next(iter(host.values())).shape[1]
    s = Cn.Soax(fields, n, capacity)
    s.upload(host)
    return s


def image(s):
    return s.to_aos().cpu().numpy()


def masks(n, seed):
    rng = np.random.default_rng(seed)
    yield (rng.random(n) < 0.5).astype(np.uint8)
    yield (rng.random(n) < 0.03).astype(np.uint8) * 255              # any non-zero byte counts
    yield (rng.random(n) < 0.97).astype(np.uint8)
    yield np.zeros(n, np.uint8)
    yield np.ones(n, np.uint8)
    k = np.zeros(n, np.uint8); k[: n // 2] = 1; yield k               # every hole below m, every mover above
    k = np.zeros(n, np.uint8); k[n // 2:] = 1; yield k                # pure truncation: nothing moves


@pytest.mark.parametrize("n", [1 << 15, 70001, 4097, 31, 1])
def test_remove_matches_oracle(gpu, n):
    torch, B, Cn = gpu
    host = inputs.make_r1(n, seed=n)
    base = oracle.r1_soa_to_aos(host)
    for kill in masks(n, n):
        kd = torch.from_numpy(kill).cuda()
        s = device(Cn, Cn.R1, host)
        m = s.remove(kd)                                             # the paper's default: overwrite with the last element
        exp = oracle.remove_swap_last(base, 40, kill)
        assert m == exp.size // 40 == s.n == n - int((kill != 0).sum())
        assert np.array_equal(image(s), exp)
        s = device(Cn, Cn.R1, host)
        d = Cn.Soax(Cn.R1, 0, capacity=n)
        m2 = s.remove(kd, stable=True, dst=d)
        assert m2 == m == d.n and s.n == n
        assert np.array_equal(image(d), oracle.remove_stable(base, 40, kill))
        assert np.array_equal(image(s), base)                        # the source of a stable removal is untouched


@pytest.mark.parametrize("n", [70001, 4097, 31])
def test_remove_keep_flagged(gpu, n):
    """SOAX_REMOVE_KEEP_FLAGGED: the mask marks the particles that STAY -- both modes equal the oracle run on the complemented
    mask (any non-zero byte is a flag), and together with the plain call one mask splits a set into stayers and leavers."""
    torch, B, Cn = gpu
    host = inputs.make_r1(n, seed=n + 1)
    base = oracle.r1_soa_to_aos(host)
    for keep in masks(n, n + 7):
        comp = (keep == 0).astype(np.uint8)                           # what the oracle is told to remove
        kd = torch.from_numpy(keep).cuda()
        s = device(Cn, Cn.R1, host)
        s.remove_async(kd, keep_flagged=True)
        assert s.n == int((keep != 0).sum())
        assert np.array_equal(image(s), oracle.remove_swap_last(base, 40, comp))
        s = device(Cn, Cn.R1, host)
        kept, dropped = Cn.Soax(Cn.R1, 0, capacity=n), Cn.Soax(Cn.R1, 0, capacity=n)
        s.remove_async(kd, stable=True, dst=kept, keep_flagged=True)
        s.remove_async(kd, stable=True, dst=dropped)
        assert kept.n + dropped.n == n
        assert np.array_equal(image(kept), oracle.remove_stable(base, 40, comp))
        assert np.array_equal(image(dropped), oracle.remove_stable(base, 40, keep))


def test_remove_wide_record_and_errors(gpu):
    torch, B, Cn = gpu
    n = 20011
    host = inputs.make_r2(n, seed=3)
    s = device(Cn, Cn.R2, host)
    base = image(s)
    kill = (np.random.default_rng(9).random(n) < 0.4).astype(np.uint8)
    kd = torch.from_numpy(kill).cuda()
    d = Cn.Soax(Cn.R2, 0, capacity=n)
    s.remove(kd, stable=True, dst=d)
    assert np.array_equal(image(d), oracle.remove_stable(base, 89, kill))
    s.remove(kd)
    assert np.array_equal(image(s), oracle.remove_swap_last(base, 89, kill))
    small = Cn.Soax(Cn.R2, 0, capacity=10)
    s2 = device(Cn, Cn.R2, host)
    # too small a destination: it receives the survivors that fit, its live count is its capacity, and the pinned host
    # word still reports the true survivor count (soax_remove never synchronises, so it cannot answer ALLOC itself)
    true_m = torch.zeros(1, dtype=torch.int64).pin_memory()
    scratch = torch.empty(B.soax_remove_scratch_bytes(n), dtype=torch.uint8, device="cuda")
    B.soax_remove(s2.handle, small.handle, kd.data_ptr(), B.SOAX_REMOVE_STABLE, scratch.data_ptr(), scratch.numel(),
                  torch.cuda.current_stream().cuda_stream, host_new_n=true_m.data_ptr())
    assert small.n == 10
    torch.cuda.synchronize()
    assert int(true_m[0]) == int((kill == 0).sum()) > 10
    assert np.array_equal(image(small), oracle.remove_stable(base, 89, kill)[:10 * 89])
    with pytest.raises(B.SoaxError):
        B.soax_remove(s2.handle, s2.handle, kd.data_ptr(), B.SOAX_REMOVE_STABLE, kd.data_ptr(), 1 << 20)   # dst aliases s
    e = Cn.Soax(Cn.R2, 0, capacity=4)
    assert e.remove(kd) == 0


def test_push_back_get_elements_copy(gpu):
    torch, B, Cn = gpu
    n, m = 5000, 3001
    a, b = inputs.make_r1(n, seed=1), inputs.make_r1(m, seed=2)
    s = device(Cn, Cn.R1, a, capacity=n + m)
    extra = torch.from_numpy(oracle.r1_soa_to_aos(b)).cuda()
    s.push_back_aos(extra, m)                                        # PAPER.md:304-307 push_back(particle), bulk
    assert s.n == n + m
    whole = np.concatenate([oracle.r1_soa_to_aos(a), oracle.r1_soa_to_aos(b)])
    assert np.array_equal(image(s), whole)
    with pytest.raises(B.SoaxError) as ei:
        B.soax_push_back_aos(s.handle, extra.data_ptr(), 1)
    assert ei.value.status == B.SOAX_ERR_ALLOC                       # the C call never allocates: the caller owns the memory
    idx = np.random.default_rng(4).integers(0, n + m, 1234).astype(np.uint32)
    idx[:3] = [0, n + m - 1, 0]
    got = s.get_elements(torch.from_numpy(idx.view(np.int32)).cuda()).cpu().numpy()
    assert np.array_equal(got, oracle.get_elements(whole, 40, idx))   # PAPER.md:304 getElement(i), bulk
    idx = np.arange(512, dtype=np.uint32)[::-1].copy()                # exactly two full 256-record tiles
    got = s.get_elements(torch.from_numpy(idx.view(np.int32)).cuda()).cpu().numpy()
    assert np.array_equal(got, oracle.get_elements(whole, 40, idx))
    big = Cn.Soax(Cn.R1, 0, capacity=2 * (n + m))                     # the paper's resize: larger slab + copy
    big.copy_from(s)
    assert big.n == n + m and np.array_equal(image(big), whole)


def test_every_call_accepts_an_empty_container(gpu):
    """n = 0 is a legal particle count for every entry point: nothing is launched, sizes stay 0, the energy is 0."""
    torch, B, Cn = gpu
    for fields in (Cn.R1, Cn.R2):
        s = Cn.Soax(fields, 0, capacity=64)
        for kind in (B.SOAX_STEP_DRIFT, B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC):
            s.step(kind, 1e-3, nsteps=3)
        assert s.energy(B.SOAX_ENERGY_KINETIC) == 0.0 and s.energy(B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC) == 0.0
        aos = torch.zeros(64, dtype=torch.uint8, device="cuda")
        s.to_aos(aos)
        s.from_aos(aos, 0)
        s.push_back_aos(aos, 0)
        assert s.n == 0 and s.get_elements(torch.zeros(0, dtype=torch.int32, device="cuda")).numel() == 0
        d = Cn.Soax(fields, 0, capacity=64)
        assert s.remove(torch.zeros(1, dtype=torch.uint8, device="cuda")) == 0
        assert s.remove(torch.zeros(1, dtype=torch.uint8, device="cuda"), stable=True, dst=d) == 0 and d.n == 0
        d.copy_from(s)
        Cn.Program(fields, "pos = pos + 1").run(s)
        if fields is Cn.R1:
            r = s.bin_permute(d, 8, drift_dt=1e-3, want_kinetic=True)
            assert int(r["counts"].sum()) == 0 and float(r["kinetic"]) == 0.0
        else:
            s.step(B.SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED, 1e-3, nsteps=2)
        torch.cuda.synchronize()
        assert all(len(v[0]) == 0 for v in s.download().values())


def test_remove_is_asynchronous_and_the_count_is_learnt_lazily(gpu):
    """soax_remove enqueues and returns (no call synchronises).  Several removals are queued back to back on a
    side stream without reading any count; every later call that needs a live count picks it up by itself, and the chain
    equals the oracle's chain."""
    torch, B, Cn = gpu
    n = 70001
    host = inputs.make_r1(n, seed=8)
    rng = np.random.default_rng(4)
    k1 = (rng.random(n) < 0.3).astype(np.uint8)
    base = oracle.r1_soa_to_aos(host)
    after1 = oracle.remove_swap_last(base, 40, k1)
    n1 = after1.size // 40
    k2 = (rng.random(n) < 0.5).astype(np.uint8)                      # only its first n1 bytes are read by the second removal
    after2 = oracle.remove_stable(after1, 40, k2[:n1])
    with torch.cuda.stream(torch.cuda.Stream()):
        s = device(Cn, Cn.R1, host)
        d = Cn.Soax(Cn.R1, 0, capacity=n)
        kd1, kd2 = torch.from_numpy(k1).cuda(), torch.from_numpy(k2).cuda()
        s.remove_async(kd1)                                          # in place; s.n now pending
        s.step(B.SOAX_STEP_DRIFT, 0.0, nsteps=1)                     # needs the count: resolves it by itself (dt = 0: no change)
        s.remove_async(kd2, stable=True, dst=d)                      # d.n pending
        e = d.energy(B.SOAX_ENERGY_KINETIC)                          # needs d's count
        assert s.n == n1 and d.n == after2.size // 40
        assert np.array_equal(image(s), after1) and np.array_equal(image(d), after2)
        oke = oracle.energy(oracle.r1_aos_to_soa(after2), oracle.KINETIC)
        assert abs(e - oke) <= 1e-10 * oke


def test_get_elements_out_of_range_rows_are_zero_records(gpu):
    torch, B, Cn = gpu
    n = 1000
    host = inputs.make_r1(n, seed=1)
    s = device(Cn, Cn.R1, host)
    idx = np.array([0, 999, 1000, 5, 2 ** 31 - 1, 17], np.uint32)
    got = s.get_elements(torch.from_numpy(idx.view(np.int32)).cuda()).cpu().numpy().reshape(-1, 40)
    base = oracle.r1_soa_to_aos(host).reshape(-1, 40)
    for j, i in enumerate(idx):
        assert np.array_equal(got[j], base[i] if i < n else np.zeros(40, np.uint8)), (j, i)


@pytest.mark.parametrize("world,n_each", [(3, 4001), (8, 700), (1, 5000), (2, 0), (8, 100), (5, 1)])
def test_gather_segments_merges_sorted_runs(gpu, world, n_each):
    """soax_gather_segments_aos against oracle.gather_segments, on the tables of a `world`-run merge by cell (G = 8).
    (8, 100) and (5, 1): more segments per 1024-row tile than the kernel stages in shared memory (mostly empty ones), so the
    whole-table search runs; the others take the staged path, with ragged last tiles."""
    torch, B, Cn = gpu
    G = 8
    rng = np.random.default_rng(world)
    runs, cnts = [], []
    for q in range(world):
        h = inputs.make_r1(n_each + 13 * q if n_each else 0, seed=20 + q)
        b = oracle.bin_r1(h, G)
        runs.append(oracle.r1_soa_to_aos(oracle.permute_r1(h, b["perm"])))
        cnts.append(b["counts"].astype(np.int64))
    recs = np.concatenate(runs) if runs else np.zeros(0, np.uint8)
    n = recs.size // 40
    cnt = np.stack(cnts)
    sizes = cnt.sum(1)
    src_start = (np.cumsum(sizes) - sizes)[:, None] + np.cumsum(cnt, 1) - cnt
    flat = cnt.T.reshape(-1)
    seg_dst, seg_src = (np.cumsum(flat) - flat).astype(np.int32), src_start.T.reshape(-1).astype(np.int32)
    want = oracle.gather_segments(recs, 40, seg_dst, seg_src, n)
    d = Cn.Soax(Cn.R1, 0, capacity=max(n, 1))
    d.from_aos_segments(torch.from_numpy(np.concatenate([recs, np.zeros(16, np.uint8)])).cuda(), torch.from_numpy(seg_dst).cuda(),
                        torch.from_numpy(seg_src).cuda(), n)
    assert d.n == n and np.array_equal(image(d), want)
    if n:                                                             # and it IS the stable sort by cell of the concatenation
        whole = oracle.r1_aos_to_soa(recs)
        assert np.array_equal(want, oracle.r1_soa_to_aos(oracle.permute_r1(whole, oracle.bin_r1(whole, G)["perm"])))


def test_push_back_regrows_like_the_papers_container(gpu):
    """push_back past the capacity and resize(n) grow every array.  Repeated push_back into a
    container that starts with room for 3 particles equals the oracle-side concatenation byte for byte after every step, and
    the capacity grows geometrically (few regrows, not one per call); R2 as well, and resize() beyond the capacity keeps the
    live rows."""
    torch, B, Cn = gpu
    for fields, make, to_aos in ((Cn.R1, inputs.make_r1, oracle.r1_soa_to_aos),):
        s = Cn.Soax(fields, 0, capacity=3)
        whole, caps = np.zeros(0, np.uint8), []
        for step, m in enumerate([1, 2, 1, 700, 4097, 0, 33, 20000]):
            rec = to_aos(make(m, seed=100 + step)) if m else np.zeros(0, np.uint8)
            s.push_back_aos(torch.from_numpy(np.concatenate([rec, np.zeros(16, np.uint8)])).cuda(), m)
            whole = np.concatenate([whole, rec])
            caps.append(s.capacity)
            assert s.n == whole.size // 40 <= s.capacity
            assert np.array_equal(image(s), whole), step
        assert caps[0] == 3 and caps[2] >= 4 and len(set(caps)) <= 6 and caps[-1] >= 24834
        live = s.n
        s.resize(2 * s.capacity + 5)                                  # the paper's resize: the live rows survive a regrow
        assert s.n == 2 * caps[-1] + 5 and s.capacity >= s.n
        B.soax_resize(s.handle, live)
        assert np.array_equal(image(s), whole)
        s.step(B.SOAX_STEP_DRIFT, 1e-3, nsteps=3)                     # the regrown container is a full citizen (graph replay included)
        exp = oracle.drift(oracle.r1_aos_to_soa(whole), 1e-3, 3)
        assert np.array_equal(image(s), oracle.r1_soa_to_aos(exp))
    h = inputs.make_r2(501, seed=4)
    s2 = device(Cn, Cn.R2, h)
    before = image(s2)
    s2.reserve(502)
    assert s2.capacity == 751 and s2.n == 501 and np.array_equal(image(s2), before)


def test_advice_hardening_of_remove_and_gather(gpu):
    """(a) soax_remove answers UNSUPPORTED while its stream is being captured (the count event would never fire and the handle
    would read a stale word); (b) soax_gather_segments_aos with a table that does not start at row 0 is served from segment 0
    with offset 0 instead of reading index -1; (c) a call that sets a handle's count while a removal count is pending waits
    for it, and the handle reports the new count."""
    torch, B, Cn = gpu
    n = 5000
    host = inputs.make_r1(n, seed=77)
    base = oracle.r1_soa_to_aos(host)
    s = device(Cn, Cn.R1, host)
    kd = torch.from_numpy((np.arange(n) % 3 == 0).astype(np.uint8)).cuda()
    scratch = torch.empty(B.soax_remove_scratch_bytes(n), dtype=torch.uint8, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        with pytest.raises(B.SoaxError) as ei:
            B.soax_remove(s.handle, None, kd.data_ptr(), B.SOAX_REMOVE_SWAP_LAST, scratch.data_ptr(), scratch.numel(), side.cuda_stream)
    assert ei.value.status == B.SOAX_ERR_UNSUPPORTED
    torch.cuda.synchronize()
    assert s.n == n and np.array_equal(image(s), base)                # nothing was enqueued
    # (b)
    d = Cn.Soax(Cn.R1, 0, capacity=8)
    recs = torch.from_numpy(np.concatenate([base[:40 * 16], np.zeros(16, np.uint8)])).cuda()
    d.from_aos_segments(recs, torch.tensor([2, 4], dtype=torch.int32).cuda(), torch.tensor([0, 5], dtype=torch.int32).cuda(), 6)
    rows = base.reshape(-1, 40)
    assert np.array_equal(image(d).reshape(-1, 40), rows[[0, 0, 0, 1, 5, 6]])
    # (c)
    s.remove_async(kd)                                                # count pending on s
    B.soax_resize(s.handle, 10)                                       # waits for the pending count, then sets its own
    assert s.n == 10
    assert np.array_equal(image(s), oracle.remove_swap_last(base, 40, kd.cpu().numpy())[:400])
