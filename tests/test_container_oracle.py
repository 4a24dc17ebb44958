"""CPU pins of the NEXT-3 oracle (container operations): the C++ routines against plain Python
list surgery written out here (pop / overwrite-with-last, one element at a time), numpy boolean masking (a library
routine for the stable case), invariants, and hand cases."""
import numpy as np
import pytest

import oracle


def records(n, stride, seed=0):
    rng = np.random.default_rng(seed)
    a = rng.integers(0, 256, (n, stride), dtype=np.uint8)
    a[:, :4] = np.arange(n, dtype=np.uint32).view(np.uint8).reshape(n, 4)        # first word = row number, for reading results
    return a


def ids(aos_bytes, stride):
    return aos_bytes.reshape(-1, stride)[:, :4].copy().view(np.uint32)[:, 0].tolist()


def test_swap_last_hand_cases():
    """Worked by hand from PAPER.md:175's rule in a forward loop that re-examines the slot it just filled (Q20)."""
    a = records(8, 12)
    for kill, want in (([0, 0, 1, 0, 0, 1, 0, 1], [0, 1, 6, 3, 4]),            # 2 <- 7 (flagged: again) <- 6; then 5 is the last: dropped
                       ([0, 1, 1, 0, 0, 0, 0, 0], [0, 7, 6, 3, 4, 5]),         # 1 <- 7, 2 <- 6
                       ([0, 1, 1, 0, 0, 0, 1, 0], [0, 7, 5, 3, 4]),            # 1 <- 7; 2 <- 6 (flagged: again) <- 5
                       ([1] * 8, []), ([0] * 8, list(range(8))), ([1, 0, 0, 0, 0, 0, 0, 0], [7, 1, 2, 3, 4, 5, 6])):
        got = oracle.remove_swap_last(a.reshape(-1), 12, np.array(kill, np.uint8))
        assert ids(got, 12) == want


@pytest.mark.parametrize("n,p,seed", [(1, 0.5, 0), (2, 0.5, 1), (17, 0.3, 2), (64, 0.5, 3), (64, 0.9, 4), (64, 0.05, 5), (1000, 0.5, 6)])
def test_removals_equal_python_list_surgery(n, p, seed):
    stride = 40
    a = records(n, stride, seed)
    kill = (np.random.default_rng(100 + seed).random(n) < p).astype(np.uint8)
    rows = [bytes(r) for r in a]
    lst, flg, i = list(rows), kill.tolist(), 0
    while i < len(lst):                                                          # one removal at a time, as the paper states it
        if flg[i]:
            lst[i], flg[i] = lst[-1], flg[-1]
            lst.pop(), flg.pop()
        else:
            i += 1
    got = oracle.remove_swap_last(a.reshape(-1), stride, kill)
    assert got.tobytes() == b"".join(lst)
    stable = oracle.remove_stable(a.reshape(-1), stride, kill)
    assert np.array_equal(stable.reshape(-1, stride), a[kill == 0])              # numpy masking keeps order
    # closed form: with m survivors, the k-th flagged slot below m (ascending) holds the k-th survivor from the END
    m = n - int(kill.sum())
    holes = [i for i in range(m) if kill[i]]
    movers = [j for j in range(n - 1, m - 1, -1) if not kill[j]]
    assert len(holes) == len(movers)
    for hole, mv in zip(holes, movers):
        assert got.reshape(-1, stride)[hole].tobytes() == rows[mv]
    # invariants: same multiset of survivors; rows that were below the new length and not flagged never move
    assert sorted(ids(got, stride)) == ids(stable, stride)
    for i in range(m):
        if not kill[i]:
            assert got.reshape(-1, stride)[i].tobytes() == rows[i]


def test_get_elements_is_row_indexing():
    a = records(50, 24, 7)
    idx = np.array([3, 3, 49, 0, 17], np.uint32)
    assert np.array_equal(oracle.get_elements(a.reshape(-1), 24, idx).reshape(-1, 24), a[idx])
    assert oracle.get_elements(a.reshape(-1), 24, np.zeros(0, np.uint32)).size == 0


def test_gather_segments_is_the_merge_of_sorted_runs():
    """oracle.gather_segments pinned by hand and by what it is for: with the tables built from per-run per-cell counts it
    reproduces the stable sort (by cell) of the concatenation of runs that are each sorted by cell."""
    rows = np.arange(10 * 3, dtype=np.uint8).reshape(10, 3)          # 10 records of 3 bytes: record r = (3r, 3r+1, 3r+2)
    out = oracle.gather_segments(rows.reshape(-1), 3, [0, 2, 2, 5], [7, 0, 4, 1], 6).reshape(-1, 3)
    assert out[:, 0].tolist() == [21, 24, 12, 15, 18, 3]             # rows 7,8 | (empty) | 4,5,6 | 1
    rng = np.random.default_rng(0)
    world, ncell = 3, 17
    runs = [np.sort(rng.integers(0, ncell, rng.integers(0, 60))) for _ in range(world)]       # each run sorted by cell
    cells = np.concatenate(runs)
    recs = np.stack([cells.astype(np.uint8), np.arange(cells.size, dtype=np.uint8)], axis=1)   # (cell, position in the concatenation)
    cnt = np.stack([np.bincount(r, minlength=ncell) for r in runs])                          # [world, ncell]
    run_start = np.concatenate([[0], np.cumsum([r.size for r in runs])[:-1]])
    src_start = run_start[:, None] + np.cumsum(cnt, axis=1) - cnt                             # first record of (run q, cell c)
    flat = cnt.T.reshape(-1)                                                                 # (cell, run) order = destination order
    seg_dst = np.cumsum(flat) - flat
    got = oracle.gather_segments(recs.reshape(-1), 2, seg_dst, src_start.T.reshape(-1), cells.size).reshape(-1, 2)
    order = np.argsort(cells, kind="stable")
    assert np.array_equal(got, recs[order])


def test_gather_segments_c_is_the_python_row_loop():
    """The C row loop (used at 2^24 rows by the full-size GPU test) returns what the plain Python definition returns: random
    tables with empty segments, repeated sources, single-row segments and a ragged end."""
    rng = np.random.default_rng(11)
    for trial in range(20):
        stride = int(rng.choice([1, 3, 40, 89]))
        nsrc, nseg = int(rng.integers(1, 300)), int(rng.integers(1, 40))
        lens = rng.integers(0, 12, nseg)
        seg_dst = np.cumsum(lens) - lens                              # starts at 0, non-decreasing, empty segments repeat
        n = int(lens.sum())
        seg_src = np.array([rng.integers(0, max(nsrc - l, 0) + 1) for l in lens])
        a = rng.integers(0, 256, (nsrc + 12) * stride, dtype=np.uint8)
        assert np.array_equal(oracle.gather_segments_c(a, stride, seg_dst, seg_src, n), oracle.gather_segments(a, stride, seg_dst, seg_src, n))
    rows = np.arange(10 * 3, dtype=np.uint8)
    assert oracle.gather_segments_c(rows, 3, [0, 2, 2, 5], [7, 0, 4, 1], 6).reshape(-1, 3)[:, 0].tolist() == [21, 24, 12, 15, 18, 3]
