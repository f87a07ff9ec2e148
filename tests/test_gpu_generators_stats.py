"""Device generators and the statistics reducer against the oracle's CPU versions: bit-exact integers."""
import numpy as np
import pytest
import torch

import graphs
from oracle import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ccl():
    import paper_1603_08357_b200 as pkg
    assert torch.cuda.is_available()
    return pkg


@pytest.mark.parametrize("L", [1, 2, 3, 7, 64, 257])
def test_lattice_generators(ccl, L):
    for dev_gen, cpu_gen in ((ccl.gen_triangular, oracle.gen_triangular), (ccl.gen_honeycomb, oracle.gen_honeycomb)):
        s, d = dev_gen(L)
        ws, wd = cpu_gen(L)
        assert np.array_equal(s.cpu().numpy(), ws) and np.array_equal(d.cpu().numpy(), wd)


@pytest.mark.parametrize("m,p,r", [(1, 0.5, 0), (31, 0.5, 1), (32, 0.3473, 0), (33, 0.6527, 2), (1003, 1 / 3, 0),
                                   (12288, 0.6527, 0), (1 << 20, 0.45, 7), (77, 0.0, 0), (77, 1.0, 0), (77, 1.5, 0)])
def test_occupancy_generator(ccl, m, p, r):
    seed = oracle.seed_for(1)
    mask, bits = ccl.gen_occupancy(m, p, seed, r)
    wm, wb = oracle.gen_occupancy(m, p, seed, r)
    assert np.array_equal(mask.cpu().numpy(), wm)
    assert np.array_equal(bits.cpu().numpy().view(np.uint32), wb)
    only_bits = ccl.gen_occupancy(m, p, seed, r, want_mask=False)[1]
    assert torch.equal(only_bits, bits)


@pytest.mark.parametrize("n,z,seed", [(6, 3, 6), (10, 4, 5), (64, 3, 1), (1000, 3, 2), (4096, 4, 3), (50000, 4, 4),
                                      ((1 << 18) + 2, 3, 11), (1 << 20, 4, 12)])
def test_regular_generator(ccl, n, z, seed):
    s, d = ccl.gen_regular(n, z, seed)
    ws, wd, nrep = oracle.gen_regular(n, z, seed)
    assert np.array_equal(s.cpu().numpy(), ws) and np.array_equal(d.cpu().numpy(), wd)


def test_regular_generator_repairs_defects(ccl):
    """Make sure the comparison above exercises the repair path: among these seeds several graphs need repairs."""
    total = 0
    for seed in range(100, 110):
        s, d = ccl.gen_regular(2000, 4, seed)
        ws, wd, nrep = oracle.gen_regular(2000, 4, seed)
        total += nrep
        assert np.array_equal(s.cpu().numpy(), ws) and np.array_equal(d.cpu().numpy(), wd)
    assert total >= 10


@pytest.mark.parametrize("case", ["identity", "one", "honeycomb", "regular4_giant", "tiny"])
def test_cluster_stats(ccl, case):
    if case == "identity":
        labels = np.arange(1000, dtype=np.int32)
    elif case == "one":
        labels = np.zeros(100000, dtype=np.int32)
    elif case == "tiny":
        labels = np.array([0, 0, 2, 2, 4], dtype=np.int32)       # tie between clusters 0 and 2 -> label 0
    elif case == "honeycomb":
        L = 200
        src, dst = oracle.gen_honeycomb(L)
        mask, _ = oracle.gen_occupancy(src.size, 0.6527, oracle.seed_for(3))
        labels = oracle.label(2 * L * L, src, dst, mask)
    else:
        n = 1 << 19
        src, dst, _ = oracle.gen_regular(n, 4, oracle.seed_for(5))
        mask, _ = oracle.gen_occupancy(src.size, 0.45, oracle.seed_for(5))
        labels = oracle.label(n, src, dst, mask)
    n_dense = 64
    want, whd, whl = oracle.stats(labels, n_dense)
    got, hd, hl = ccl.cluster_stats(torch.from_numpy(labels).cuda(), n_dense)
    assert got == want
    assert np.array_equal(hd.numpy(), whd) and np.array_equal(hl.numpy(), whl)
    # derived floats come from exact integers on both sides -> identical (north_star: 1e-12 relative)
    n = labels.size
    for f in (lambda s: s["largest"] / n, lambda s: (s["sum_s2"] - s["largest"] ** 2) / n):
        a, b = f(got), f(want)
        assert abs(a - b) <= 1e-12 * max(abs(b), 1e-300)


def test_cluster_stats_empty(ccl):
    got, hd, hl = ccl.cluster_stats(torch.zeros(0, dtype=torch.int32, device="cuda"), 4)
    assert got == dict(n_clusters=0, largest=0, largest_label=-1, sum_s2=0)


def test_pipeline_on_device_matches_oracle_pipeline(ccl):
    """Device generators -> ccl_label_bits -> ccl_cluster_stats, against the oracle doing the same on the CPU."""
    L = 128
    s, d = ccl.gen_triangular(L)
    _, bits = ccl.gen_occupancy(3 * L * L, 0.3473, oracle.seed_for(2), 3, want_mask=False)
    lab = ccl.label_bits(L * L, s, d, bits)
    ws, wd = oracle.gen_triangular(L)
    wm, _ = oracle.gen_occupancy(3 * L * L, 0.3473, oracle.seed_for(2), 3)
    wl = oracle.label(L * L, ws, wd, wm)
    assert np.array_equal(lab.cpu().numpy(), wl)
    assert ccl.cluster_stats(lab)[0] == oracle.stats(wl)[0]


@pytest.mark.parametrize("g", [1, 2, 5, 16])
def test_cayley_generator(ccl, g):
    """PAPER.md:189-193 workload: device generator == oracle generator, standard and random numbering."""
    n, src, dst = ccl.gen_cayley3(g)
    wn, wsrc, wdst = oracle.gen_cayley3(g)
    assert n == wn == 3 * (1 << g) - 2
    assert np.array_equal(src.cpu().numpy(), wsrc) and np.array_equal(dst.cpu().numpy(), wdst)
    perm = np.random.default_rng(g).permutation(n).astype(np.int32)
    _, src, dst = ccl.gen_cayley3(g, torch.from_numpy(perm).cuda())
    _, wsrc, wdst = oracle.gen_cayley3(g, perm)
    assert np.array_equal(src.cpu().numpy(), wsrc) and np.array_equal(dst.cpu().numpy(), wdst)
    # a forest at every p: clusters = N - occupied bonds
    mask, bits = oracle.gen_occupancy(n - 1, 0.5, oracle.seed_for(6))
    lab = ccl.label(n, src, dst, torch.from_numpy(mask).cuda())
    stats, _, _ = ccl.cluster_stats(lab, 0)
    assert stats["n_clusters"] == n - int(mask.sum())


def _wrap_vectors_from_oracle(family, L):
    """Wrap vectors derived on the test side from the oracle generator's displacements: the bond leaves cell (x, y) by
    (dx, dy) cells; it crosses the seam iff the target cell lies outside [0, L)."""
    src, dst, dx, dy = (oracle.gen_triangular if family == "triangular" else oracle.gen_honeycomb)(L, with_disp=True)
    cell = src.astype(np.int64) // (2 if family == "honeycomb" else 1)
    wx = ((cell % L + dx) // L).astype(np.int8)
    wy = ((cell // L + dy) // L).astype(np.int8)
    return src, dst, dx, dy, wx, wy


@pytest.mark.parametrize("family", ["triangular", "honeycomb"])
def test_wrapping_detection_small_lattices(ccl, family):
    """GPU: open-lattice labels + lock-free weighted union-find over the seam bonds.  Oracle: displacement union-find
    over all bonds (pinned by BFS on the unwrapped cover).  Different formulations, same answer, 1200 realizations."""
    pc = 0.3473 if family == "triangular" else 0.6527
    seen = set()
    for L in (1, 2, 3, 4, 5, 7, 9, 16, 33):
        src, dst, dx, dy, wx, wy = _wrap_vectors_from_oracle(family, L)
        gx, gy = ccl.gen_wrap_vectors(family, L)
        assert np.array_equal(gx.cpu().numpy(), wx) and np.array_equal(gy.cpu().numpy(), wy)
        n = (2 if family == "honeycomb" else 1) * L * L
        s, d = torch.from_numpy(src).cuda(), torch.from_numpy(dst).cuda()
        for r in range(70):
            p = [0.0, 1.0, pc, pc - 0.1, pc + 0.1, pc + 0.03, pc - 0.03][r % 7]
            mask, bits = oracle.gen_occupancy(src.size, p, oracle.seed_for(3), realization=r)
            want = oracle.wrap(n, src, dst, dx, dy, mask)
            got_x, got_y, lab_open = ccl.wrap(n, s, d, torch.from_numpy(bits.view(np.int32)).cuda(), gx, gy)
            assert (got_x, got_y) == want, (L, p, r)
            open_mask = mask & ((wx == 0) & (wy == 0)).astype(np.uint8)
            assert np.array_equal(lab_open.cpu().numpy(), oracle.label(n, src, dst, open_mask))
            seen.add(want)
    assert len(seen) == 4                                   # none, x only, y only, both all occurred


@pytest.mark.parametrize("family,L", [("triangular", 257), ("honeycomb", 301)])
def test_wrapping_detection_larger_lattices(ccl, family, L):
    pc = 0.3473 if family == "triangular" else 0.6527
    src, dst, dx, dy, wx, wy = _wrap_vectors_from_oracle(family, L)
    n = (2 if family == "honeycomb" else 1) * L * L
    s, d = torch.from_numpy(src).cuda(), torch.from_numpy(dst).cuda()
    gx, gy = torch.from_numpy(wx).cuda(), torch.from_numpy(wy).cuda()
    for r, p in enumerate([pc - 0.02, pc - 0.005, pc, pc, pc, pc + 0.005, pc + 0.02, 1.0]):
        mask, bits = oracle.gen_occupancy(src.size, p, oracle.seed_for(3), realization=r)
        got = ccl.wrap(n, s, d, torch.from_numpy(bits.view(np.int32)).cuda(), gx, gy)[:2]
        assert got == oracle.wrap(n, src, dst, dx, dy, mask), (p, r)
    # all bonds occupied without a mask; a single occupied row wraps in x only
    assert ccl.wrap(n, s, d, None, gx, gy)[:2] == (True, True)
    if family == "triangular":
        row = np.zeros(src.size, dtype=np.uint8)
        row[3 * np.arange(5 * L, 6 * L)] = 1                # bonds k = 0 of row y = 5
        got = ccl.wrap(n, s, d, torch.from_numpy(graphs.pack_bits(row).view(np.int32)).cuda(), gx, gy)[:2]
        assert got == (True, False) == oracle.wrap(n, src, dst, dx, dy, row)


@pytest.mark.parametrize("family", ["triangular", "honeycomb"])
def test_wrapping_detection_with_reversed_bonds(ccl, family):
    """A bond listed the other way round carries the negated wrap vector (-1 entries); the answer must not change."""
    pc = 0.3473 if family == "triangular" else 0.6527
    rng = np.random.default_rng(17)
    for L in (4, 9, 33, 64):
        src, dst, dx, dy, wx, wy = _wrap_vectors_from_oracle(family, L)
        n = (2 if family == "honeycomb" else 1) * L * L
        flip = rng.random(src.size) < 0.5
        s2 = np.where(flip, dst, src).astype(np.int32)
        d2 = np.where(flip, src, dst).astype(np.int32)
        wx2 = np.where(flip, -wx, wx).astype(np.int8)
        wy2 = np.where(flip, -wy, wy).astype(np.int8)
        perm = rng.permutation(src.size)                    # and in any bond order
        for r in range(30):
            mask, _ = oracle.gen_occupancy(src.size, pc + 0.04 * (r % 5 - 2), oracle.seed_for(3), realization=200 + r)
            want = oracle.wrap(n, src, dst, dx, dy, mask)
            bits = graphs.pack_bits(mask[perm])
            got = ccl.wrap(n, torch.from_numpy(s2[perm]).cuda(), torch.from_numpy(d2[perm]).cuda(),
                           torch.from_numpy(bits.view(np.int32)).cuda(), torch.from_numpy(wx2[perm]).cuda(),
                           torch.from_numpy(wy2[perm]).cuda())[:2]
            assert got == want, (L, r)


@pytest.mark.parametrize("family,pc", [("triangular", 0.34729635533386066), ("honeycomb", 0.6527036446661394)])
def test_wrapping_probability_curves_cross_at_the_exact_threshold(ccl, family, pc):
    """The paper's own correctness evidence (Figs. 5-6): the spanning-probability curves of different
    sizes cross at p_c.  Here through the CUDA path alone (device generators, ccl_wrap), 400 realizations per point:
    below p_c the larger lattice wraps less often, above p_c more often, and at p_c the two agree."""
    reals = 400
    R = {}
    for L in (24, 72):
        src, dst = (ccl.gen_triangular if family == "triangular" else ccl.gen_honeycomb)(L)
        wx, wy = ccl.gen_wrap_vectors(family, L)
        n = (2 if family == "honeycomb" else 1) * L * L
        lab = torch.empty(n, dtype=torch.int32, device="cuda")
        for p in (pc - 0.02, pc, pc + 0.02):
            hits = 0
            for r in range(reals):
                _, bits = ccl.gen_occupancy(3 * L * L, p, oracle.seed_for(3) + L, r, want_mask=False)
                x, y, _ = ccl.wrap(n, src, dst, bits, wx, wy, labels_open=lab)
                hits += x or y
            R[(L, p)] = hits / reals
    lo, hi = pc - 0.02, pc + 0.02
    assert R[(72, lo)] < R[(24, lo)] - 0.08, R             # curves fan out on both sides ...
    assert R[(72, hi)] > R[(24, hi)] + 0.03, R
    assert abs(R[(72, pc)] - R[(24, pc)]) < 0.12, R        # ... and meet at the exact threshold (4 sigma of 400 draws)
    assert 0.5 < R[(24, pc)] < 0.85 and 0.5 < R[(72, pc)] < 0.85, R      # R_either ~ 0.68-0.69 at p_c
