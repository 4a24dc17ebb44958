"""NEXT-4: the cross-GPU binning exchange and the per-step migration.  Host logic (cell-range split, the
exchange plan) on CPU; the whole exchange + migration under a world-size-2 gloo group, once with the oracle standing in for
the device engine (CPU) and once with the PRODUCT engine (libsoax.so), both ranks on the one GPU these tests see, device
tensors staged through the host for the collectives; and the product engine through an NCCL group of world size 1."""
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


def test_plan_exchange_is_consistent_across_ranks():
    """every rank derives the same bounds; what q sends to r is what r receives from q; sums match the counts"""
    rng = np.random.default_rng(1)
    world, ncell = 4, 64
    allc = torch.from_numpy(rng.integers(0, 30, (world, ncell)).astype(np.int64))
    plans = [D.plan_exchange(allc, r) for r in range(world)]
    assert all(p[0] == plans[0][0] for p in plans) and plans[0][0] == D.split_cells(allc.sum(0), world)
    for q in range(world):
        assert sum(plans[q][1]) == int(allc[q].sum())
        assert plans[q][1] == D.send_counts(allc[q], plans[0][0])
        for r in range(world):
            assert plans[q][1][r] == plans[r][2][q]
    given = torch.tensor([0, 10, 10, 50, 64])                        # fixed bounds (migration): one empty range
    p = D.plan_exchange(allc, 2, given)
    assert p[0] == [0, 10, 10, 50, 64] and p[1] == D.send_counts(allc[2], p[0]) and p[2] == [int(allc[q, 10:50].sum()) for q in range(world)]


_WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
import oracle
from oracle import expr as oexpr
from paper_1710_03462_b200 import inputs, dist as D
rank, world, G, kind = int(sys.argv[3]), 2, 4, sys.argv[4]
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + sys.argv[2], rank=rank, world_size=world)
sizes = [3001, 1777]                                               # unequal shards
hosts = [inputs.make_r1(sizes[r], seed=10 + r) for r in range(world)]
for r in range(world):
    hosts[r]["id"][0] = np.arange(sizes[r]) + 100000 * r           # globally unique ids
    hosts[r]["pos"][0] = hosts[r]["pos"][0] ** 2                     # non-uniform: unequal cell ranges
DT = 0.05                                                          # a long drift: many particles change cell


def sort_by_cell(soa):
    b = oracle.bin_r1(soa, G)
    return b, oracle.permute_r1(soa, b["perm"])


class HostSet:                                                     # the oracle engine's "container": packed records on the host
    def __init__(self, soa):
        self.aos = oracle.r1_soa_to_aos(soa)

    @property
    def n(self):
        return self.aos.size // 40


class OracleEngine:                                                # stands in for SoaxEngine: same interface, CPU oracle inside
    stride, ncell = 40, G ** 3

    def __init__(self, host):
        self.host = host

    def local_sort(self):
        b, srt = sort_by_cell(self.host)
        return torch.from_numpy(b["counts"].astype(np.int64)), torch.from_numpy(oracle.r1_soa_to_aos(srt))

    def merge(self, records, n, run_counts, lo):
        b, srt = sort_by_cell(oracle.r1_aos_to_soa(records[:n * 40].numpy()))
        assert np.array_equal(run_counts.sum(0).numpy(), b["counts"][lo:lo + run_counts.shape[1]])
        return srt, b["counts"]

    def take_leavers(self, s, lo, hi):
        soa = oracle.r1_aos_to_soa(s.aos)
        cond = f"(double(cell({G})) < lo) | (double(cell({G})) >= hi)"
        leave = oexpr.mask(soa, cond, {"lo": lo, "hi": hi})
        gone = oracle.r1_aos_to_soa(oracle.remove_stable(s.aos, 40, 1 - leave))
        s.aos = oracle.remove_swap_last(s.aos, 40, leave)
        b, srt = sort_by_cell(gone)
        return torch.from_numpy(b["counts"].astype(np.int64)), torch.from_numpy(oracle.r1_soa_to_aos(srt)), gone["id"].shape[1]

    def append(self, s, records, n):
        s.aos = np.concatenate([s.aos, records[:n * 40].numpy()])


if kind == "oracle":
    engine = OracleEngine(hosts[rank])
    (mine, counts), bounds, n_local = D.bin_exchange(engine)
    local = HostSet(oracle.drift(mine, DT, 1))                     # the integration step between binning and migration
    n_after = D.migrate(engine, local, bounds)
    after = local.aos
    counts = np.asarray(counts)
    ke_local = torch.tensor([oracle.energy(hosts[rank], oracle.KINETIC)], dtype=torch.float64)
else:
    from paper_1710_03462_b200 import binding as B, container as Cn
    torch.cuda.set_device(0)                                       # BOTH ranks on the one GPU; collectives are host-level (gloo)
    src = Cn.Soax(Cn.R1, sizes[rank])
    src.upload(hosts[rank])
    engine = D.SoaxEngine(src, G)
    (out, c32, _), bounds, n_local = D.bin_exchange(engine)
    mine = out.download()
    counts = c32.cpu().numpy().view(np.uint32)
    big = out                                                      # sized to the LOCAL count: arrivals beyond it regrow it (Soax.reserve)
    big.step(B.SOAX_STEP_DRIFT, DT, nsteps=1)
    n_after = D.migrate(engine, big, bounds)
    after = big.to_aos().cpu().numpy()
    ke_local = src.energy_async(B.SOAX_ENERGY_KINETIC)
    torch.cuda.synchronize()

# ---- expectation 1: the stable sort of the rank-major concatenation of ALL inputs, cut at this rank's cell range
whole = {k: np.concatenate([h[k] for h in hosts], axis=1) for k in hosts[0]}
gb, gs = sort_by_cell(whole)
cut = lambda r: (int(gb["offsets"][bounds[r]]), int(gb["offsets"][bounds[r + 1]]) if bounds[r + 1] < G ** 3 else sum(sizes))   # noqa: E731
lo, hi = cut(rank)
assert n_local == hi - lo and 0 < n_local < sum(sizes)
for k in gs:
    assert np.array_equal(gs[k][:, lo:hi].view(np.uint8), mine[k].view(np.uint8)), k
assert np.array_equal(counts[bounds[rank]:bounds[rank + 1]], gb["counts"][bounds[rank]:bounds[rank + 1]]) and counts.sum() == n_local
assert abs(n_local - sum(sizes) / world) < 0.2 * sum(sizes)        # balanced to within the size of one cell

# ---- expectation 2 (migration): stayers in the overwrite-with-last arrangement, then the arrivals by source rank, each
# rank's leavers in (cell, source order) -- all from the oracle, for every rank, from the global sort
cond = f"(double(cell({G})) < lo) | (double(cell({G})) >= hi)"
parts, moved = [], 0
for q in range(world):
    a, b = cut(q)
    loc = oracle.drift({k: np.ascontiguousarray(v[:, a:b]) for k, v in gs.items()}, DT, 1)
    leave = oexpr.mask(loc, cond, {"lo": bounds[q], "hi": bounds[q + 1]})
    aos = oracle.r1_soa_to_aos(loc)
    if q == rank:
        stay = oracle.remove_swap_last(aos, 40, leave)
    gone = oracle.r1_aos_to_soa(oracle.remove_stable(aos, 40, 1 - leave))
    gcell, gsorted = sort_by_cell(gone)
    c = gcell["cell"][gcell["perm"]] if gone["id"].shape[1] else np.zeros(0, np.uint32)
    sel = (c >= bounds[rank]) & (c < bounds[rank + 1])
    parts.append(oracle.r1_soa_to_aos({k: np.ascontiguousarray(v[:, sel]) for k, v in gsorted.items()}))
    moved += int(leave.sum())
want = np.concatenate([stay] + parts)
assert moved > 50, "the test must move particles"
assert n_after == want.size // 40 and np.array_equal(after, want)
final = oracle.r1_aos_to_soa(after)                                # every particle now sits on the rank that owns its cell
fc = oracle.bin_r1(final, G)["cell"]
assert ((fc >= bounds[rank]) & (fc < bounds[rank + 1])).all()
tot = torch.tensor([n_after], dtype=torch.int64)
dist.all_reduce(tot)
assert int(tot) == sum(sizes)                                      # nobody lost, nobody duplicated

e = D.energy_sum(ke_local)
eref = oracle.energy(whole, oracle.KINETIC)
assert abs(e - eref) <= 1e-10 * eref
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
"""


def _run_two_ranks(tmp_path, kind):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    port = str(31500 + os.getpid() % 2000 + (7 if kind == "soax" else 0))
    procs = [subprocess.Popen([sys.executable, str(script), ROOT, port, str(r), kind], stdout=subprocess.PIPE, stderr=subprocess.STDOUT,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=600)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
    assert sorted(o.strip().splitlines()[-1] for o in outs) == ["ok 0", "ok 1"]


def test_bin_exchange_and_migration_two_ranks_gloo_oracle_engine(tmp_path):
    _run_two_ranks(tmp_path, "oracle")


@pytest.mark.gpu
def test_bin_exchange_and_migration_two_ranks_product_engine(tmp_path):
    """The PRODUCT engine (libsoax.so: soax_bin_permute, soax_soa_to_aos, soax_aos_to_soa, soax_expr_mask, soax_remove in both
    modes, soax_push_back_aos, soax_step) in a real 2-rank exchange and migration: two processes, both on cuda:0, a gloo
    group, the all-to-all payload staged through host memory."""
    _run_two_ranks(tmp_path, "soax")


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
        assert D.migrate(eng, out, bounds) == n                       # one rank owns every cell: nobody leaves
        ke = D.energy_sum(eng.kinetic)
        ref = oracle.energy(host, oracle.KINETIC)
        assert abs(ke - ref) <= 1e-10 * ref
    finally:
        dist.destroy_process_group()


def test_bench_gpus_n_spawns_n_ranks():
    """`python bench.py --gpus 2` without a launcher starts 2 ranks itself (torch.distributed.run on 127.0.0.1) and prints ONE
    line with n_gpus = 2 -- the launch path alone, over gloo, no GPU (the driver invokes exactly this form)."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--spawn-check"], capture_output=True, text=True,
                       timeout=300, env=env)
    assert r.returncode == 0, r.stdout + r.stderr
    lines = [json.loads(x) for x in r.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1 and lines[0]["n_gpus"] == 2 and lines[0]["sum_of_rank_plus_1"] == 3
    # --impl reference under N ranks: rank 0 alone prints, the others exit 0 (checked through the same spawn path)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, r.stdout + r.stderr
    lines = [json.loads(x) for x in r.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1 and lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2


@pytest.mark.gpu
def test_exchange_leg_world2_over_nccl():
    """The exchange and the per-step migration with the product engine over the NCCL branch at world size 2 -- device tensors
    through all_gather_into_tensor and all_to_all_single, one rank per GPU -- as `bench.py --gpus 2` runs it: the global
    particle count and the rank-ordered kinetic energy survive, records do cross between the ranks, and the split is balanced.
    Needs two GPUs; skipped on a one-GPU box (where the same engine runs over gloo in the test above, and over an NCCL group of
    one rank in test_bin_exchange_product_engine_nccl_world1)."""
    import json
    if torch.cuda.device_count() < 2:
        pytest.skip("needs 2 GPUs")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "2", "--warmup", "3", "--no-extras"],
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout + r.stderr
    line = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
    ex = line["extras"]["exchange"]
    assert line["n_gpus"] == 2 and ex["world"] == 2 and ex["backend"] == "nccl"
    assert ex["verified"] and ex["conserved_count"] and ex["kinetic_rel_err"] <= 1e-10
    assert ex["all_to_all_bytes_all_ranks"] > 0 and ex["migration_particles_moved_per_step_all_ranks"] > 0
    assert ex["imbalance_max_over_mean"] < 1.05
