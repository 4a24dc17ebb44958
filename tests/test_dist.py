"""NEXT-4: the cross-GPU binning exchange.  Host logic (cell-range split, send counts) on CPU; the whole
exchange under a world-size-2 gloo group with the oracle standing in for the device engine; and, on the GPU, the product
engine (libsoax.so) through an NCCL group of world size 1 (one GPU is all this repository's tests ever see)."""
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
from paper_1710_03462_b200 import dist as D  # noqa: E402


def test_split_cells_balances_and_covers():
    rng = np.random.default_rng(0)
    for world in (1, 2, 3, 8):
        for counts in (rng.integers(0, 50, 512), np.r_[np.zeros(100, int), 1000, np.zeros(100, int)], np.zeros(64, int), np.ones(7, int)):
            c = torch.from_numpy(np.asarray(counts, np.int64))
            b = D.split_cells(c, world)
            assert b[0] == 0 and b[-1] == c.numel() and len(b) == world + 1 and all(x <= y for x, y in zip(b, b[1:]))
            sent = D.send_counts(c, b)
            assert sum(sent) == int(c.sum())
            total, left = int(c.sum()), 0
            for r in range(1, world):                                # smallest boundary with >= ceil(r N / world) to its left
                left = int(c[:b[r]].sum())
                target = -(-r * total // world)
                assert left >= target and (b[r] == 0 or int(c[:b[r] - 1].sum()) < target)
    assert D.split_cells(torch.tensor([5, 0, 3, 2, 0, 0, 10, 1]), 3) == [0, 3, 7, 8]     # worked by hand: targets 7 and 14
    assert D.shard_sizes(10, 3) == [3, 3, 4] and sum(D.shard_sizes(1 << 24, 7)) == 1 << 24


_WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
import oracle
from paper_1710_03462_b200 import inputs, dist as D
rank, world, G = int(sys.argv[3]), 2, 4
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + sys.argv[2], rank=rank, world_size=world)
sizes = [3001, 1777]                                               # unequal shards
hosts = [inputs.make_r1(sizes[r], seed=10 + r) for r in range(world)]
for r in range(world):
    hosts[r]["id"][0] = np.arange(sizes[r]) + 100000 * r           # globally unique ids
    hosts[r]["pos"][0] = hosts[r]["pos"][0] ** 2                     # non-uniform: unequal cell ranges


class OracleEngine:                                                # stands in for SoaxEngine: same interface, CPU oracle inside
    stride, ncell = 40, G ** 3

    def __init__(self, host):
        self.host = host

    def _sort(self, soa):
        b = oracle.bin_r1(soa, G)
        return b, oracle.permute_r1(soa, b["perm"])

    def local_sort(self):
        b, srt = self._sort(self.host)
        return torch.from_numpy(b["counts"].astype(np.int64)), torch.from_numpy(oracle.r1_soa_to_aos(srt))

    def merge(self, records, n):
        soa = oracle.r1_aos_to_soa(records[:n * 40].numpy())
        b, srt = self._sort(soa)
        return srt, b["counts"]


(mine, counts), bounds, n_local = D.bin_exchange(OracleEngine(hosts[rank]))
# expectation: the stable sort of the rank-major concatenation of ALL inputs, cut at this rank's cell range
whole = {k: np.concatenate([h[k] for h in hosts], axis=1) for k in hosts[0]}
gb = oracle.bin_r1(whole, G)
gs = oracle.permute_r1(whole, gb["perm"])
lo, hi = int(gb["offsets"][bounds[rank]]), (int(gb["offsets"][bounds[rank + 1]]) if bounds[rank + 1] < G ** 3 else sum(sizes))
assert n_local == hi - lo and 0 < n_local < sum(sizes)
for k in gs:
    assert np.array_equal(gs[k][:, lo:hi].view(np.uint8), mine[k].view(np.uint8)), k
assert np.array_equal(counts[bounds[rank]:bounds[rank + 1]], gb["counts"][bounds[rank]:bounds[rank + 1]]) and counts.sum() == n_local
assert abs(n_local - sum(sizes) / world) < 0.2 * sum(sizes)        # balanced to within the size of one cell
e = D.energy_sum(torch.tensor([oracle.energy(hosts[rank], oracle.KINETIC)], dtype=torch.float64))
eref = oracle.energy(whole, oracle.KINETIC)
assert abs(e - eref) <= 1e-12 * eref
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
"""


def test_bin_exchange_two_ranks_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    port = str(31500 + os.getpid() % 2000)
    procs = [subprocess.Popen([sys.executable, str(script), ROOT, port, str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=300)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
    assert sorted(o.strip().splitlines()[-1] for o in outs) == ["ok 0", "ok 1"]


@pytest.mark.gpu
def test_bin_exchange_product_engine_nccl_world1():
    """The real engine end to end on one GPU: NCCL group of size 1, libsoax.so for every device step, against the oracle."""
    import torch.distributed as dist
    import oracle
    from paper_1710_03462_b200 import container as Cn, inputs
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{32500 + os.getpid() % 2000}", rank=0, world_size=1,
                            device_id=torch.device("cuda", 0))
    try:
        n, G, dt = 50021, 16, 1e-3
        host = inputs.make_r1(n, seed=5)
        s = Cn.Soax(Cn.R1, n)
        s.upload(host)
        eng = D.SoaxEngine(s, G, drift_dt=dt)
        (out, counts, offsets), bounds, n_local = D.bin_exchange(eng)
        torch.cuda.synchronize()
        assert bounds == [0, G ** 3] and n_local == n
        drifted = oracle.drift(host, dt, 1)
        b = oracle.bin_r1(drifted, G)
        exp = oracle.permute_r1(drifted, b["perm"])
        got = out.download()
        for k in exp:
            assert np.array_equal(got[k].view(np.uint8), exp[k].view(np.uint8)), k
        assert np.array_equal(counts.cpu().numpy().view(np.uint32), b["counts"])
        ke = D.energy_sum(eng.kinetic)
        ref = oracle.energy(host, oracle.KINETIC)
        assert abs(ke - ref) <= 1e-10 * ref
    finally:
        dist.destroy_process_group()
