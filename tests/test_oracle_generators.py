"""Pins for the CPU generators of oracle/ccl_oracle.c (Philox4x32-10, lattices, random z-regular, occupancy)."""
from fractions import Fraction

import numpy as np
import pytest

import graphs
from oracle import oracle


def test_philox_known_answers():
    for ctr, key, want in graphs.read_philox_kat():
        got = oracle.philox4x32_10(ctr, key)
        assert [int(x) for x in got] == want


def test_philox_is_a_bijection_on_a_counter_slice_and_key_sensitive():
    outs = {tuple(int(x) for x in oracle.philox4x32_10([c, 0, 0, 0], [1, 2])) for c in range(2000)}
    assert len(outs) == 2000
    a = oracle.philox4x32_10([5, 0, 0, 0], [1, 2])
    b = oracle.philox4x32_10([5, 0, 0, 0], [1, 3])
    assert (a != b).all()


def test_occupancy_thresholds_file(golden_dir):
    import os
    with open(os.path.join(golden_dir, "occupancy_thresholds.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            ptxt, ttxt = line.split()
            p = 1.0 / 3.0 if ptxt == "1/3" else float(ptxt)
            exact = int(Fraction(p) * (1 << 32))       # floor of the exact binary value of the double p times 2^32
            assert exact == int(ttxt), ptxt


@pytest.mark.parametrize("p,seed,r", [(0.3473, 1, 0), (0.6527, 2, 3), (1.0 / 3.0, 3, 1)])
def test_occupancy_matches_threshold_definition(p, seed, r):
    m = 1003                                            # ragged: not a multiple of 4 or 32
    mask, bits = oracle.gen_occupancy(m, p, seed, r)
    T = int(Fraction(p) * (1 << 32))
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for b in (0, 1, 2, 3, 4, 31, 32, 33, 500, 1000, 1001, 1002):
        w = oracle.philox4x32_10([b >> 2, 0, r, 0], key)
        assert mask[b] == (int(w[b & 3]) < T)
    assert np.array_equal(bits, graphs.pack_bits(mask))
    assert set(np.unique(mask).tolist()) <= {0, 1}


def test_occupancy_edges_rate_and_nesting():
    m = 1 << 20
    assert not oracle.gen_occupancy(m, 0.0, 9)[0].any()
    assert oracle.gen_occupancy(m, 1.0, 9)[0].all()
    assert oracle.gen_occupancy(33, 1.0, 9)[1].tolist() == [0xFFFFFFFF, 1]
    prev = None
    for p in (0.25, 1.0 / 3.0, 0.45, 0.6527):
        mask, _ = oracle.gen_occupancy(m, p, seed=42)
        assert abs(mask.mean() - p) < 5 * np.sqrt(p * (1 - p) / m)
        if prev is not None:
            assert (mask >= prev).all()
        prev = mask
    a, _ = oracle.gen_occupancy(m, 0.5, seed=42, realization=0)
    b, _ = oracle.gen_occupancy(m, 0.5, seed=42, realization=1)
    c, _ = oracle.gen_occupancy(m, 0.5, seed=43, realization=0)
    assert abs((a == b).mean() - 0.5) < 0.01 and abs((a == c).mean() - 0.5) < 0.01
    assert np.array_equal(a, oracle.gen_occupancy(m, 0.5, seed=42, realization=0)[0])


@pytest.mark.parametrize("L", [1, 2, 3, 8, 33])
def test_triangular_geometry(L):
    src, dst, dx, dy = oracle.gen_triangular(L, with_disp=True)
    n = L * L
    assert src.size == 3 * n
    deg = np.bincount(np.concatenate([src, dst]), minlength=n)
    assert (deg == 6).all()
    x, y = src % L, src // L
    assert np.array_equal(dst, ((y + dy) % L) * L + (x + dx) % L)
    assert np.array_equal(src, np.repeat(np.arange(n), 3))
    if L >= 3:
        keys = np.minimum(src, dst).astype(np.int64) * n + np.maximum(src, dst)
        assert np.unique(keys).size == 3 * n and (src != dst).all()


@pytest.mark.parametrize("L", [1, 2, 3, 8, 33])
def test_honeycomb_geometry(L):
    src, dst, dx, dy = oracle.gen_honeycomb(L, with_disp=True)
    n = 2 * L * L
    assert src.size == 3 * L * L
    deg = np.bincount(np.concatenate([src, dst]), minlength=n)
    assert (deg == 3).all()
    # bipartite: every bond joins an A site (even) to a B site (odd)
    assert ((src + dst) % 2 == 1).all()
    cs, cd = src // 2, dst // 2
    assert np.array_equal(cd, ((cs // L + dy) % L) * L + (cs % L + dx) % L)
    if L >= 2:
        keys = np.minimum(src, dst).astype(np.int64) * n + np.maximum(src, dst)
        assert np.unique(keys).size == 3 * L * L


def test_baseline_config_counts():
    """BASELINE.json configs: honeycomb L=64 -> 8,192 sites / 12,288 bonds; L=4096 -> 33,554,432 / 50,331,648;
    triangular L=4096 -> 16,777,216 / 50,331,648; 3-regular 2^24 -> 25,165,824; 4-regular 2^26 -> 134,217,728."""
    src, dst = oracle.gen_honeycomb(64)
    assert src.size == 12288 and int(max(src.max(), dst.max())) == 8191
    assert 2 * 4096 * 4096 == 33554432 and 3 * 4096 * 4096 == 50331648
    assert (1 << 24) * 3 // 2 == 25165824 and (1 << 26) * 4 // 2 == 134217728


@pytest.mark.parametrize("n,z,seed", [(64, 3, 1), (1000, 3, 2), (4096, 4, 3), (50000, 4, 4), (10, 4, 5), (6, 3, 6)])
def test_regular_graph_is_simple_and_regular(n, z, seed):
    src, dst, nrep = oracle.gen_regular(n, z, seed)
    assert src.size == n * z // 2
    assert (np.bincount(np.concatenate([src, dst]), minlength=n) == z).all()
    assert (src != dst).all()
    keys = np.minimum(src, dst).astype(np.int64) * n + np.maximum(src, dst)
    assert np.unique(keys).size == src.size
    s2, d2, nrep2 = oracle.gen_regular(n, z, seed)
    assert np.array_equal(src, s2) and np.array_equal(dst, d2) and nrep == nrep2


def test_regular_graph_defect_rate_matches_configuration_model():
    """Before repair the configuration model has on average (z-1)/2 self-loops and (z-1)^2/4 duplicate pairs whatever
    N is, so the number of repaired defects per graph is O(1): mean ~ 2 for z=3, ~3.75 for z=4."""
    for z, expect in ((3, 1.0 + 1.0), (4, 1.5 + 2.25)):
        reps = [oracle.gen_regular(2000, z, seed)[2] for seed in range(100, 160)]
        assert 0.6 * expect < np.mean(reps) < 1.4 * expect, (z, np.mean(reps))


def test_regular_graph_endpoints_are_uncorrelated_in_memory():
    """'bonds shuffled so endpoints are uncorrelated in memory' (BASELINE.json config 5)."""
    n = 1 << 16
    src, dst, _ = oracle.gen_regular(n, 4, seed=8)
    for a in (src, dst):
        a = a.astype(np.float64)
        assert abs(np.corrcoef(a[:-1], a[1:])[0, 1]) < 0.02
    assert abs(np.corrcoef(src.astype(np.float64), dst.astype(np.float64))[0, 1]) < 0.02
    assert abs(np.mean(src < dst) - 0.5) < 0.01
