"""Pins for oracle_stats (brute-force counting, sum rules) and oracle_wrap (BFS on the unwrapped cover)."""
from collections import Counter

import numpy as np
import pytest

import graphs
from oracle import oracle


def test_stats_against_counter():
    rng = np.random.default_rng(5)
    for trial in range(50):
        n = int(rng.integers(1, 400))
        m = int(rng.integers(0, 2 * n))
        src, dst = graphs.random_graph(rng, n, m)
        labels = graphs.bfs_min_labels(n, src, dst)
        st, hd, hl = oracle.stats(labels, n_dense=16)
        sizes = Counter(labels.tolist())
        assert st["n_clusters"] == len(sizes)
        big = max(sizes.values())
        assert st["largest"] == big
        assert st["largest_label"] == min(l for l, s in sizes.items() if s == big)
        assert st["sum_s2"] == sum(s * s for s in sizes.values())
        for s in range(1, 17):
            assert hd[s] == sum(1 for v in sizes.values() if v == s)
        for k in range(32):
            assert hl[k] == sum(1 for v in sizes.values() if (1 << k) <= v < (1 << (k + 1)))
        assert hl.sum() == len(sizes)


def test_stats_sum_rule_and_extremes():
    n = 1000
    st, hd, hl = oracle.stats(np.arange(n, dtype=np.int32), n_dense=4)
    assert st == dict(n_clusters=n, largest=1, largest_label=0, sum_s2=n) and hd[1] == n and hl[0] == n
    st, hd, hl = oracle.stats(np.zeros(n, dtype=np.int32), n_dense=n)
    assert st == dict(n_clusters=1, largest=n, largest_label=0, sum_s2=n * n) and hd[n] == 1 and hl[9] == 1
    L = 64
    src, dst = oracle.gen_honeycomb(L)
    mask, _ = oracle.gen_occupancy(src.size, 0.6, seed=1)
    labels = oracle.label(2 * L * L, src, dst, mask)
    st, hd, hl = oracle.stats(labels, n_dense=2 * L * L)
    assert (np.arange(hd.size) * hd).sum() == 2 * L * L          # sum_s s * hist[s] = N when n_dense >= largest
    assert hd.sum() == st["n_clusters"] == hl.sum()


def test_stats_empty():
    st, hd, hl = oracle.stats(np.zeros(0, dtype=np.int32), n_dense=3)
    assert st["n_clusters"] == 0 and st["largest"] == 0 and st["sum_s2"] == 0


# ------------------------------------------------------------------ wrapping
@pytest.mark.parametrize("gen,spc", [(oracle.gen_triangular, 1), (oracle.gen_honeycomb, 2)])
def test_wrap_vs_bfs_cover(gen, spc):
    rng = np.random.default_rng(17)
    pc = 0.3473 if spc == 1 else 0.6527
    n_wrapping = 0
    for trial in range(400):
        L = int(rng.integers(2, 8))
        src, dst, dx, dy = gen(L, with_disp=True)
        p = pc + rng.uniform(-0.15, 0.15)
        mask, _ = oracle.gen_occupancy(src.size, p, seed=1000 + trial)
        got = oracle.wrap(spc * L * L, src, dst, dx, dy, mask)
        assert got == graphs.bfs_winding(spc * L * L, src, dst, dx, dy, mask), trial
        n_wrapping += got[0] or got[1]
    assert 50 < n_wrapping < 350


def test_wrap_closed_forms():
    L = 6
    src, dst, dx, dy = oracle.gen_triangular(L, with_disp=True)
    n = L * L
    assert oracle.wrap(n, src, dst, dx, dy, np.zeros(src.size, np.uint8)) == (False, False)     # p = 0
    assert oracle.wrap(n, src, dst, dx, dy, np.ones(src.size, np.uint8)) == (True, True)        # p = 1
    row = np.zeros(src.size, np.uint8)
    row[[3 * (2 * L + x) + 0 for x in range(L)]] = 1           # the L horizontal bonds of row y = 2
    assert oracle.wrap(n, src, dst, dx, dy, row) == (True, False)
    row[3 * (2 * L + 3)] = 0                                    # cut it once: no wrapping
    assert oracle.wrap(n, src, dst, dx, dy, row) == (False, False)
    col = np.zeros(src.size, np.uint8)
    col[[3 * (y * L + 4) + 1 for y in range(L)]] = 1           # a vertical line
    assert oracle.wrap(n, src, dst, dx, dy, col) == (False, True)
    diag = np.zeros(src.size, np.uint8)
    diag[[3 * (i * L + i) + 2 for i in range(L)]] = 1          # the main diagonal winds once in x and once in y
    assert oracle.wrap(n, src, dst, dx, dy, diag) == (True, True)

    src, dst, dx, dy = oracle.gen_honeycomb(L, with_disp=True)
    n = 2 * L * L
    assert oracle.wrap(n, src, dst, dx, dy, np.ones(src.size, np.uint8)) == (True, True)
    zig = np.zeros(src.size, np.uint8)
    for x in range(L):                                          # zig-zag A-B-A-B along row y = 1
        zig[3 * (1 * L + x) + 0] = 1
        zig[3 * (1 * L + x) + 1] = 1
    assert oracle.wrap(n, src, dst, dx, dy, zig) == (True, False)


def test_relabel_sequential_against_numpy_unique_and_brute_force():
    """PAPER.md:115.  Pins: np.unique's inverse (sorted distinct labels = clusters in ascending order of smallest site)
    and a brute-force count on tiny inputs."""
    rng = np.random.default_rng(115)
    for trial in range(50):
        n = int(rng.integers(1, 400))
        m = int(rng.integers(0, 2 * n))
        src, dst = graphs.random_graph(rng, n, m, self_loops=True)
        labels = oracle.label(n, src, dst) if m else np.arange(n, dtype=np.int32)
        seq, c = oracle.relabel_sequential(labels)
        uniq, inv = np.unique(labels, return_inverse=True)
        assert c == uniq.size and np.array_equal(seq, inv)
        if n <= 60:
            roots = [i for i in range(n) if labels[i] == i]
            assert [sum(1 for r in roots if r < labels[i]) for i in range(n)] == seq.tolist()
    seq, c = oracle.relabel_sequential(np.zeros(0, dtype=np.int32))
    assert c == 0 and seq.size == 0
