"""Pins for the labeling oracle (oracle/ccl_oracle.c: oracle_label, oracle_label_bits; oracle/komura_steps.py).

Sources of truth used here, none of which is the oracle itself:
  * the paper's worked example, Fig. 1 -> Figs. 2, 3, 4 (tests/golden/);
  * a breadth-first search written in tests/graphs.py, exhaustively on tiny graphs and on random ones;
  * closed forms: p = 0, p = 1, path graphs, forests (cluster count = N - occupied bonds), the empty residual
    lists of the centre-numbered Cayley tree;
  * invariants of the canonical labeling.
"""
import itertools

import numpy as np
import pytest

import graphs
from oracle import komura_steps, oracle


# ------------------------------------------------------------------ the paper's worked example (E0)
def test_fig1_nn_list_is_symmetric_with_26_bonds():
    nn = graphs.read_fig1_nn_list()
    assert len(nn) == 22
    for i, row in enumerate(nn):
        for j in row:
            assert i in nn[j], (i, j)
    src, dst = graphs.bonds_from_nn_list(nn)
    assert src.size == 26


def test_fig1_final_labels_match_fig4():
    nn = graphs.read_fig1_nn_list()
    want, _ = graphs.read_e0_labels()
    src, dst = graphs.bonds_from_nn_list(nn)
    got = oracle.label(22, src, dst)
    assert got.tolist() == want["fig4_right"]
    ones = np.ones(src.size, dtype=np.uint8)
    assert oracle.label(22, src, dst, ones).tolist() == want["fig4_right"]
    assert oracle.label_bits(22, src, dst, graphs.pack_bits(ones)).tolist() == want["fig4_right"]
    # orientation and order of the bonds do not matter
    assert oracle.label(22, dst[::-1].copy(), src[::-1].copy()).tolist() == want["fig4_right"]
    # three components
    assert sorted(set(got.tolist())) == [0, 1, 2]


def test_four_steps_reproduce_figs_2_3_4():
    nn = graphs.read_fig1_nn_list()
    want, residual_want = graphs.read_e0_labels()
    label, residual = komura_steps.initialization(nn)
    assert label == want["fig2_right"]                                   # Fig. 2 right: labels
    for i in range(22):
        assert residual[i] == residual_want.get(i, []), i                 # Fig. 2 right: residual lists
    after_i, after_ii, after_iii, after_iv = komura_steps.four_steps(nn)
    assert after_i == want["fig2_right"]
    assert after_ii == want["fig3_left"]
    assert after_iv == want["fig4_right"]
    # analysis of the state the paper prints after (iii) gives Fig. 4 right
    assert komura_steps.analysis(want["fig3_right"]) == want["fig4_right"]


def test_fig3_right_is_a_reachable_state_and_every_schedule_ends_in_fig4():
    """Fig. 3 right is 'the actual output' of one run; intermediate states depend on thread order
    (reading R5), the final state does not."""
    nn = graphs.read_fig1_nn_list()
    want, _ = graphs.read_e0_labels()
    seen = set()
    for seed in range(300):
        _, _, after_iii, after_iv = komura_steps.four_steps(nn, schedule_seed=seed)
        assert after_iv == want["fig4_right"], seed
        seen.add(tuple(after_iii))
    assert tuple(want["fig3_right"]) in seen
    assert len(seen) <= 4          # SURVEY: two states are reachable (site 14 holds 0 or 12)


# ------------------------------------------------------------------ brute force
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
def test_exhaustive_all_graphs_up_to_5_sites(n):
    pairs = list(itertools.combinations(range(n), 2))
    src = np.array([p[0] for p in pairs], dtype=np.int32)
    dst = np.array([p[1] for p in pairs], dtype=np.int32)
    for code in range(1 << len(pairs)):
        occ = np.array([(code >> b) & 1 for b in range(len(pairs))], dtype=np.uint8)
        want = graphs.bfs_min_labels(n, src, dst, occ)
        assert np.array_equal(oracle.label(n, src, dst, occ), want), (n, code)
        assert np.array_equal(oracle.label_bits(n, src, dst, graphs.pack_bits(occ)), want), (n, code)


def test_exhaustive_6_sites_sampled():
    pairs = list(itertools.combinations(range(6), 2))
    src = np.array([p[0] for p in pairs], dtype=np.int32)
    dst = np.array([p[1] for p in pairs], dtype=np.int32)
    for code in range(0, 1 << 15, 7):
        occ = np.array([(code >> b) & 1 for b in range(15)], dtype=np.uint8)
        assert np.array_equal(oracle.label(6, src, dst, occ), graphs.bfs_min_labels(6, src, dst, occ)), code


def test_random_graphs_vs_bfs():
    rng = np.random.default_rng(20160328)
    for trial in range(400):
        n = int(rng.integers(1, 65))
        m = int(rng.integers(0, 3 * n + 1))
        src, dst = graphs.random_graph(rng, n, m, self_loops=True)
        occ = (rng.random(m) < rng.random()).astype(np.uint8)
        want = graphs.bfs_min_labels(n, src, dst, occ)
        assert np.array_equal(oracle.label(n, src, dst, occ), want), trial
        assert np.array_equal(oracle.label_bits(n, src, dst, graphs.pack_bits(occ)), want), trial


def test_four_steps_vs_bfs_under_random_schedules():
    """Reading R3 of Algorithm 1's garbled last lines is correct under arbitrary interleavings; the alternative
    (trailing `label_2 <- label_3` unconditional) is not."""
    rng = np.random.default_rng(1603)
    bad_alt = 0
    for trial in range(300):
        n = int(rng.integers(2, 25))
        m = int(rng.integers(1, 3 * n))
        src, dst = graphs.random_graph(rng, n, m)
        want = graphs.bfs_min_labels(n, src, dst).tolist()
        nn = komura_steps.nn_list_from_bonds(n, zip(src.tolist(), dst.tolist()))
        for s in range(3):
            got = komura_steps.four_steps(nn, schedule_seed=1000 * trial + s)[3]
            assert got == want, (trial, s)
        try:
            alt = komura_steps.four_steps(nn, schedule_seed=trial, alt_reading=True)[3]
            bad_alt += alt != want
        except RuntimeError:
            bad_alt += 1
    assert bad_alt > 0


# ------------------------------------------------------------------ closed forms and special cases
def test_empty_and_degenerate_inputs():
    e = np.zeros(0, dtype=np.int32)
    assert oracle.label(0, e, e).size == 0
    assert oracle.label(5, e, e).tolist() == [0, 1, 2, 3, 4]
    src = np.array([2, 2, 3, 3], dtype=np.int32)
    dst = np.array([2, 4, 3, 3], dtype=np.int32)          # self-loops and a duplicate self-loop
    assert oracle.label(5, src, dst).tolist() == [0, 1, 2, 3, 2]
    assert oracle.label(5, src, dst, np.zeros(4, np.uint8)).tolist() == [0, 1, 2, 3, 4]   # p = 0
    src = np.array([0, 0, 0], dtype=np.int32)
    dst = np.array([1, 1, 1], dtype=np.int32)             # repeated bond
    assert oracle.label(3, src, dst).tolist() == [0, 0, 2]


@pytest.mark.parametrize("order", ["ascending", "descending", "shuffled"])
def test_path_graph_is_one_cluster(order):
    rng = np.random.default_rng(7)
    n = 1 << 16
    src, dst = graphs.path_graph(n, order, rng)
    assert not oracle.label(n, src, dst).any()


@pytest.mark.parametrize("gen,sites_per_cell", [(oracle.gen_triangular, 1), (oracle.gen_honeycomb, 2)])
def test_p1_lattice_is_one_cluster_and_p0_is_identity(gen, sites_per_cell):
    L = 17
    src, dst = gen(L)
    n = sites_per_cell * L * L
    assert not oracle.label(n, src, dst).any()
    assert np.array_equal(oracle.label(n, src, dst, np.zeros(src.size, np.uint8)), np.arange(n))


def test_cayley_tree_standard_numbering_has_empty_residual_lists():
    """with numbering from the centre 'the remaining sites in the residual list for all sites become
    zero at all probabilities'."""
    n, src, dst = oracle.gen_cayley3(6)
    assert n == 3 * 2 ** 6 - 2 and src.size == n - 1
    deg = np.bincount(np.concatenate([src, dst]), minlength=n)
    assert set(deg.tolist()) == {1, 3} and (deg == 1).sum() == 3 * 2 ** 5
    for p in (0.25, 0.5, 0.75, 1.0):
        mask, _ = oracle.gen_occupancy(src.size, p, seed=5)
        nn = komura_steps.nn_list_from_bonds(n, [(int(u), int(v)) for u, v, o in zip(src, dst, mask) if o])
        _, residual = komura_steps.initialization(nn)
        assert all(len(r) == 0 for r in residual)
        labels = oracle.label(n, src, dst, mask)
        assert (labels == np.arange(n)).sum() == n - int(mask.sum())        # forest: clusters = N - occupied bonds
        assert komura_steps.four_steps(nn)[3] == labels.tolist()


def test_cayley_tree_random_numbering_same_partition():
    rng = np.random.default_rng(3)
    n, src, dst = oracle.gen_cayley3(8)
    perm = rng.permutation(n).astype(np.int32)
    n2, psrc, pdst = oracle.gen_cayley3(8, perm)
    mask, _ = oracle.gen_occupancy(src.size, 0.75, seed=9)
    a = oracle.label(n, src, dst, mask)
    b = oracle.label(n, psrc, pdst, mask)
    assert graphs.same_partition(a, b[perm])
    assert (b == np.arange(n)).sum() == n - int(mask.sum())


# ------------------------------------------------------------------ invariants (PAPER.md:115 canonical form)
def _check_invariants(n, src, dst, occ, labels):
    idx = np.arange(n)
    assert (labels <= idx).all()
    assert np.array_equal(labels[labels], labels)
    on = occ.astype(bool)
    assert np.array_equal(labels[src[on]], labels[dst[on]])
    sizes = np.bincount(labels, minlength=n)
    assert sizes.sum() == n
    n_clusters = int((labels == idx).sum())
    assert n_clusters >= n - int(on.sum())
    # idempotence: relabeling the star graph (i, labels[i]) gives the same array
    assert np.array_equal(oracle.label(n, idx.astype(np.int32), labels), labels)


@pytest.mark.parametrize("case", ["triangular", "honeycomb", "regular3", "regular4"])
def test_invariants_and_symmetries(case):
    rng = np.random.default_rng(11)
    if case == "triangular":
        L = 48; src, dst = oracle.gen_triangular(L); n = L * L; p = 0.3473
    elif case == "honeycomb":
        L = 40; src, dst = oracle.gen_honeycomb(L); n = 2 * L * L; p = 0.6527
    elif case == "regular3":
        n = 4096; src, dst, _ = oracle.gen_regular(n, 3, seed=1); p = 0.5
    else:
        n = 4096; src, dst, _ = oracle.gen_regular(n, 4, seed=2); p = 0.45
    occ, bits = oracle.gen_occupancy(src.size, p, seed=77)
    labels = oracle.label(n, src, dst, occ)
    assert np.array_equal(labels, oracle.label_bits(n, src, dst, bits))
    _check_invariants(n, src, dst, occ, labels)
    assert np.array_equal(labels, graphs.bfs_min_labels(n, src, dst, occ))
    # bond permutation and endpoint swap
    perm = rng.permutation(src.size)
    flip = rng.random(src.size) < 0.5
    s2 = np.where(flip, dst, src)[perm].astype(np.int32)
    d2 = np.where(flip, src, dst)[perm].astype(np.int32)
    assert np.array_equal(oracle.label(n, s2, d2, occ[perm]), labels)
    # site permutation: same partition
    sp = rng.permutation(n).astype(np.int32)
    lp = oracle.label(n, sp[src], sp[dst], occ)
    assert graphs.same_partition(labels, lp[sp])


def test_monotone_coupling():
    """Same seed, p1 < p2 => occupied sets nested => the partition at p2 coarsens the one at p1."""
    L = 64
    src, dst = oracle.gen_triangular(L)
    n = L * L
    prev_mask, prev_labels, prev_largest = None, None, 0
    for p in (0.1, 0.3, 0.3473, 0.4, 0.6):
        mask, _ = oracle.gen_occupancy(src.size, p, seed=123)
        labels = oracle.label(n, src, dst, mask)
        largest = int(np.bincount(labels).max())
        if prev_mask is not None:
            assert (mask >= prev_mask).all()
            # every old cluster lies inside one new cluster
            assert np.array_equal(labels[prev_labels], labels)
            assert largest >= prev_largest
        prev_mask, prev_labels, prev_largest = mask, labels, largest
