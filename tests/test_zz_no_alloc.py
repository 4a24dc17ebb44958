"""GPU test of soax_remove_stable_noalloc, the one entry point of the library that allocates nothing.

Who needs it: code that is handed the particle arrays of a running simulation but has no device memory of its own to give
and no business asking for any -- a diagnostics or migration hook called in the middle of somebody else's time step (a
cudaMalloc there would stall the whole device), a host program that has already spent all of HBM on its particle slabs, a
plugin interface with no allocator.  soax_remove wants a scratch buffer from such a caller; this entry point keeps its work
area inside libsoax.so instead (about 0.27 MB per GPU, sized for SOAX_NOALLOC_MAX_N = 2^24 particles) and refuses larger
sets with SOAX_ERR_TOO_LARGE.

What is checked: its output equals the existing path's (soax_remove in STABLE mode with caller scratch) BYTE FOR BYTE --
the tolerance every removal test of this suite uses -- on calls made back to back, so that the second call runs on the
work area the first one left dirty (larger set first, then a smaller one, then a different layout).

The file name sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a failure here must
not hide the rest of the suite.  Nothing here depends on what ran before it: the test passes alone in a fresh process (the
first call then performs the per-device address look-up) and after the other tests.
"""
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


def image(s):
    return s.to_aos().cpu().numpy()


def existing_path(Cn, s, fields, kd, keep_flagged):
    """soax_remove(STABLE) with scratch from the caller: the reference the new entry point must reproduce."""
    ref = Cn.Soax(fields, 0, capacity=s.n)
    s.remove_async(kd, stable=True, dst=ref, keep_flagged=keep_flagged)
    return ref


def test_two_calls_in_a_row_equal_the_existing_path(gpu):
    torch, B, Cn = gpu
    rng = np.random.default_rng(20240611)
    # (layout, host generator, record bytes, n, fraction flagged, keep_flagged): 257 tiles first, then 2 tiles on the
    # dirty work area with the mask read the other way round, then the wide record, then a ragged single tile
    cases = [(Cn.R1, inputs.make_r1, 40, (1 << 20) + 3, 0.5, False),
             (Cn.R1, inputs.make_r1, 40, 4097, 0.03, True),
             (Cn.R2, inputs.make_r2, 89, 70001, 0.4, False),
             (Cn.R1, inputs.make_r1, 40, 31, 0.5, False)]
    work = []
    for fields, make, stride, n, frac, keep in cases:
        host = make(n, seed=n)
        mask = (rng.random(n) < frac).astype(np.uint8) * 255           # any non-zero byte is a flag
        s = Cn.Soax(fields, n)
        s.upload(host)
        kd = torch.from_numpy(mask).cuda()
        new = Cn.Soax(fields, 0, capacity=n)
        count = torch.full((1,), -7, dtype=torch.int64, device="cuda")
        work.append((fields, stride, n, mask, keep, s, kd, new, count))
    # the calls under test, back to back on one stream with no synchronisation in between: they share the built-in work area
    for fields, stride, n, mask, keep, s, kd, new, count in work:
        s.remove_stable_noalloc(kd, new, count, keep_flagged=keep)
        assert new.n == 0                                              # the handle's live count is the caller's to set
    torch.cuda.synchronize()
    for fields, stride, n, mask, keep, s, kd, new, count in work:
        base = image(s)
        ref = existing_path(Cn, s, fields, kd, keep)
        m = int(count.item())
        assert m == ref.n == int((mask != 0).sum() if keep else (mask == 0).sum())
        B.soax_resize(new.handle, m)
        got = image(new)
        assert np.array_equal(got, image(ref))                         # byte for byte, every component of every row
        removed = (mask == 0) if keep else (mask != 0)
        assert np.array_equal(got, oracle.remove_stable(base, stride, removed.astype(np.uint8)))
        assert s.n == n and np.array_equal(image(s), base)             # the source is left as it was


def test_limit_is_served_and_one_more_is_refused(gpu):
    """Exactly SOAX_NOALLOC_MAX_N particles (4096 tiles: the whole work area) equal the existing path; one particle more is
    refused with SOAX_ERR_TOO_LARGE before anything is enqueued.  The rows are random bytes written on the device: removal
    moves bytes and looks at nothing but the mask."""
    torch, B, Cn = gpu
    nmax = B.SOAX_NOALLOC_MAX_N
    g = torch.Generator(device="cuda").manual_seed(5)
    s = Cn.Soax(Cn.R1, nmax + 1)
    s.slab.view(torch.int64).random_(generator=g)
    kd = (torch.rand(nmax + 1, device="cuda", generator=g) < 0.1).to(torch.uint8)
    new = Cn.Soax(Cn.R1, 0, capacity=nmax + 1)
    count = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    torch.cuda.synchronize()
    launches = B.soax_launch_count()
    with pytest.raises(B.SoaxError) as ei:
        s.remove_stable_noalloc(kd, new, count)
    assert ei.value.status == B.SOAX_ERR_TOO_LARGE and "SOAX_NOALLOC_MAX_N" in str(ei.value)
    assert B.soax_launch_count() == launches and int(count.item()) == -7   # nothing ran, nothing was written
    B.soax_resize(s.handle, nmax)
    for _ in range(2):                                                 # twice: the second call finds the area full of counts
        count.fill_(-7)
        s.remove_stable_noalloc(kd, new, count)
        ref = existing_path(Cn, s, Cn.R1, kd, False)
        m = int(count.item())
        assert m == ref.n == int((kd[:nmax] == 0).sum().item())
        B.soax_resize(new.handle, m)
        assert torch.equal(new.to_aos(), ref.to_aos())
        B.soax_resize(new.handle, 0)


def test_empty_set_and_bad_arguments(gpu):
    torch, B, Cn = gpu
    s, d = Cn.Soax(Cn.R1, 0, capacity=8), Cn.Soax(Cn.R1, 0, capacity=8)
    count = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    kd = torch.zeros(8, dtype=torch.uint8, device="cuda")
    s.remove_stable_noalloc(kd, d, count)
    assert int(count.item()) == 0
    other = Cn.Soax(Cn.R2, 0, capacity=8)
    for args in [(s.handle, s.handle, kd.data_ptr(), False, count.data_ptr()),        # dst aliases the source
                 (s.handle, d.handle, kd.data_ptr(), False, 0),                       # nowhere to put the count
                 (s.handle, d.handle, kd.data_ptr(), False, count.data_ptr() + 4),    # misaligned count word
                 (s.handle, other.handle, kd.data_ptr(), False, count.data_ptr())]:            # another layout
        with pytest.raises(B.SoaxError) as ei:
            B.soax_remove_stable_noalloc(*args)
        assert ei.value.status == B.SOAX_ERR_INVALID_ARG
