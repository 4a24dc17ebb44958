"""Guard-band tests: no call writes a byte outside what include/soax.h says it writes.

compute-sanitizer is not available on the machines these tests run on (see profiles/r3_sanitizers.md), so out-of-bounds
WRITES are looked for directly: every output -- the component arrays of a container beyond its live rows (the tail of each
array up to the next array's start, in a container with spare capacity), flat buffers, scratch areas -- is painted with a
canary byte before the call, given exactly the size the header asks for inside a larger allocation, and checked afterwards.
Sizes are ragged on purpose (not multiples of the tile, the vector width or the 4-particles-per-thread grouping).  The
results themselves are compared with the oracle elsewhere (test_gpu_parity.py, test_gpu_container.py)."""
import numpy as np
import pytest

from paper_1710_03462_b200 import inputs

pytestmark = pytest.mark.gpu
CANARY, PAD = 0xA5, 4096
SIZES = [70001, 4097, 4095, 257, 5, 1]


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1710_03462_b200 import binding as B, container as Cn
    B.lib()
    return torch, B, Cn


class Guarded:
    """`nbytes` usable bytes (256-byte aligned) with PAD canary bytes on either side."""

    def __init__(self, torch, nbytes, paint_inside=True):
        self.n = nbytes
        self.buf = torch.full((nbytes + 2 * PAD,), CANARY, dtype=torch.uint8, device="cuda")
        self.view = self.buf[PAD:PAD + nbytes]
        if not paint_inside:
            self.view.zero_()

    def ptr(self):
        return self.buf.data_ptr() + PAD

    def intact(self):
        return bool((self.buf[:PAD] == CANARY).all()) and bool((self.buf[PAD + self.n:] == CANARY).all())


def painted(Cn, fields, n, room=None, spare=777):
    """a container with n live rows and room for `room` (default n) rows plus some spare, every byte of it the canary"""
    s = Cn.Soax(fields, n, capacity=(n if room is None else room) + spare)
    s.slab.fill_(CANARY)
    return s


def tails_intact(B, s, n):
    """every byte of the slab that is not one of the first n rows of a component array still holds the canary"""
    base, starts = s.slab.data_ptr(), []
    for f, (name, dt, dim) in enumerate(s.fields):
        for c in range(dim):
            starts.append((B.soax_field_ptr(s.handle, f, c) - base, B.DTYPE_SIZE[dt]))
    ends = [st for st, _ in starts[1:]] + [s.slab.numel()]
    return all(bool((s.slab[st + n * sz:en] == CANARY).all()) for (st, sz), en in zip(starts, ends))


def stream(torch):
    return torch.cuda.current_stream().cuda_stream


@pytest.mark.parametrize("n", SIZES)
def test_steps_transposes_and_container_calls_stay_inside(gpu, n):
    torch, B, Cn = gpu
    for fields, make, stride in ((Cn.R1, inputs.make_r1, 40), (Cn.R2, inputs.make_r2, 89)):
        host = make(n, seed=n)
        s = painted(Cn, fields, n)
        s.upload(host)
        assert tails_intact(B, s, n)
        for kind in (B.SOAX_STEP_DRIFT, B.SOAX_STEP_SYMPLECTIC_EULER_HARMONIC) + ((B.SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED,) if fields is Cn.R2 else ()):
            s.step(kind, 1e-3, nsteps=2)
        assert tails_intact(B, s, n), "step"
        aos = Guarded(torch, n * stride + (-n * stride) % 16)
        B.soax_soa_to_aos(s.handle, aos.ptr(), n, stream(torch))
        assert aos.intact() and bool((aos.view[n * stride:] == CANARY).all()), "soa_to_aos"
        d = painted(Cn, fields, 0, room=n)
        B.soax_aos_to_soa(d.handle, aos.ptr(), n, stream(torch))
        assert tails_intact(B, d, n), "aos_to_soa"
        m = n // 3 + 1                                                # push_back of m records behind the n live ones
        d2 = painted(Cn, fields, 0, room=n + m)
        d2.copy_from(s)
        assert tails_intact(B, d2, n), "copy"
        B.soax_push_back_aos(d2.handle, aos.ptr(), m, stream(torch))
        assert d2.n == n + m and tails_intact(B, d2, n + m), "push_back"
        idx = torch.randint(0, n, (m,), device="cuda", dtype=torch.int32)
        rows = Guarded(torch, m * stride + (-m * stride) % 16)
        B.soax_get_elements(s.handle, idx.data_ptr(), m, rows.ptr(), stream(torch))
        assert rows.intact() and bool((rows.view[m * stride:] == CANARY).all()), "get_elements"
        seg_dst = torch.tensor([0, n // 2], dtype=torch.int32, device="cuda")
        seg_src = torch.tensor([n - n // 2, 0], dtype=torch.int32, device="cuda")
        d3 = painted(Cn, fields, 0, room=n)
        B.soax_gather_segments_aos(d3.handle, aos.ptr(), seg_dst.data_ptr(), seg_src.data_ptr(), 2, n, stream(torch))
        assert tails_intact(B, d3, n), "gather_segments"
        esc = Guarded(torch, B.soax_energy_scratch_bytes())
        out = Guarded(torch, 8)
        B.soax_reduce_energy(s.handle, B.SOAX_ENERGY_KINETIC_PLUS_HARMONIC, 1.0, 0.5, esc.ptr(), esc.n, out.ptr(), stream(torch))
        assert esc.intact() and out.intact(), "energy"


@pytest.mark.parametrize("n", SIZES)
def test_removal_and_mask_stay_inside(gpu, n):
    torch, B, Cn = gpu
    host = inputs.make_r1(n, seed=n + 1)
    s = painted(Cn, Cn.R1, n)
    s.upload(host)
    mask = Guarded(torch, n)                                          # soax.h: n bytes, one per live particle
    prog = Cn.MaskProgram(Cn.R1, "(pos[0] < a) | (vel[1] > 0.0)", ["a"])
    B.soax_expr_mask(s.handle, prog.handle, [0.3], mask.ptr(), stream(torch))
    assert mask.intact(), "expr_mask"
    survivors = int((mask.view == 0).sum().item())
    scratch = Guarded(torch, B.soax_remove_scratch_bytes(n))
    d = painted(Cn, Cn.R1, 0, room=n)
    B.soax_remove(s.handle, d.handle, mask.ptr(), B.SOAX_REMOVE_STABLE, scratch.ptr(), scratch.n, stream(torch))
    assert d.n == survivors and tails_intact(B, d, survivors) and scratch.intact() and mask.intact(), "stable removal"
    d = painted(Cn, Cn.R1, 0, room=n)
    count = Guarded(torch, 8)
    B.soax_remove_stable_noalloc(s.handle, d.handle, mask.ptr(), True, count.ptr(), stream(torch))
    torch.cuda.synchronize()
    kept = int(count.view.view(torch.int64).item())
    assert kept == n - survivors and tails_intact(B, d, kept) and count.intact(), "stable removal, no-allocation entry"
    B.soax_remove(s.handle, None, mask.ptr(), B.SOAX_REMOVE_SWAP_LAST, scratch.ptr(), scratch.n, stream(torch))
    assert s.n == survivors and tails_intact(B, s, n) and scratch.intact(), "swap-last removal"   # rows [survivors, n) may hold anything


@pytest.mark.parametrize("n,G", [(70001, 64), (4097, 16), (257, 64), (5, 32), (1, 64)])
def test_binning_stays_inside(gpu, n, G):
    torch, B, Cn = gpu
    for fields, make in ((Cn.R1, inputs.make_r1), (Cn.R2, inputs.make_r2)):
        host = make(n, seed=n + 2)
        s = painted(Cn, fields, n)
        s.upload(host)
        for inplace in (False, True):
            need = (B.soax_scratch_bytes_inplace if inplace else B.soax_scratch_bytes)(s.layout, n, G)
            scratch = Guarded(torch, need)
            counts, offsets, perm, kin = Guarded(torch, 4 * G ** 3), Guarded(torch, 4 * G ** 3), Guarded(torch, 4 * n), Guarded(torch, 8)
            d = painted(Cn, fields, 0, room=n)
            (B.soax_bin_permute_inplace if inplace else B.soax_bin_permute)(
                s.handle, d.handle, G, 1e-3, counts.ptr(), offsets.ptr(), perm.ptr(), kin.ptr(), scratch.ptr(), scratch.n, stream(torch))
            torch.cuda.synchronize()
            what = f"bin_permute inplace={inplace}"
            assert scratch.intact() and counts.intact() and offsets.intact() and perm.intact() and kin.intact(), what
            assert tails_intact(B, s, n) and tails_intact(B, d, n), what   # in place: d is the work area, also only n rows of it
            assert int(counts.view.view(torch.int32).sum().item()) == n
