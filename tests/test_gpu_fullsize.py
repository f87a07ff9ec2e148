"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default options, device-resident
inputs, ccl_label_bits): every label of configs 2-5 is compared with the oracle's, the device generators are compared
with the oracle's generators at full size, and the statistics reducer is checked on the result.  The oracle needs a
few minutes of host time for the 2^26-site graph (its stub sort is a plain single-threaded radix sort)."""
import numpy as np
import pytest
import torch

from oracle import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ccl():
    import paper_1603_08357_b200 as pkg
    assert torch.cuda.is_available()
    pkg.set_option("reset")
    return pkg


def _check(ccl, n, src, dst, d_src, d_dst, ps, cfg, n_dense=32):
    assert np.array_equal(d_src.cpu().numpy(), src) and np.array_equal(d_dst.cpu().numpy(), dst)
    labels = torch.empty(n, dtype=torch.int32, device="cuda")
    for p in ps:
        mask, bits = oracle.gen_occupancy(src.size, p, oracle.seed_for(cfg), 0)
        _, d_bits = ccl.gen_occupancy(src.size, p, oracle.seed_for(cfg), 0, want_mask=False)
        assert np.array_equal(d_bits.cpu().numpy().view(np.uint32), bits)
        want = oracle.label_bits(n, src, dst, bits)
        ccl.label_bits(n, d_src, d_dst, d_bits, labels=labels)
        got = labels.cpu().numpy()
        assert np.array_equal(got, want), (cfg, p, int((got != want).sum()))
        st, hd, hl = ccl.cluster_stats(labels, n_dense)
        wst, whd, whl = oracle.stats(want, n_dense)
        assert st == wst and np.array_equal(hd.numpy(), whd) and np.array_equal(hl.numpy(), whl)
        del mask, bits, want, got


def test_cfg2_triangular_L4096(ccl):
    L = 4096
    src, dst = oracle.gen_triangular(L)
    d_src, d_dst = ccl.gen_triangular(L)
    _check(ccl, L * L, src, dst, d_src, d_dst, [0.3473], 2)


def test_cfg3_honeycomb_L4096(ccl):
    L = 4096
    src, dst = oracle.gen_honeycomb(L)
    d_src, d_dst = ccl.gen_honeycomb(L)
    _check(ccl, 2 * L * L, src, dst, d_src, d_dst, [0.60, 0.6527, 0.70], 3)


def test_cfg3_wrapping_statistics_L4096(ccl):
    """Config 3 asks for wrapping statistics per p, and the crossing of the wrapping probability at p_c is the paper's own
    correctness evidence.  ccl_wrap (open-lattice labels, a 128 MiB label array, + seam-graph union-find)
    against the oracle's displacement union-find at the full size, for the three configured p and three realizations at
    the threshold itself, where the answer is not a foregone conclusion."""
    L = 4096
    n = 2 * L * L
    src, dst, dx, dy = oracle.gen_honeycomb(L, with_disp=True)
    cell = src.astype(np.int64) // 2
    wx = ((cell % L + dx) // L).astype(np.int8)
    wy = ((cell // L + dy) // L).astype(np.int8)
    d_src, d_dst = ccl.gen_honeycomb(L)
    gx, gy = ccl.gen_wrap_vectors("honeycomb", L)
    assert np.array_equal(gx.cpu().numpy(), wx) and np.array_equal(gy.cpu().numpy(), wy)
    seen = set()
    for p, r in [(0.60, 0), (0.6527, 0), (0.70, 0), (0.6527, 1), (0.6527, 2), (0.6527, 3)]:
        mask, bits = oracle.gen_occupancy(src.size, p, oracle.seed_for(3), r)
        want = oracle.wrap(n, src, dst, dx, dy, mask)
        got_x, got_y, lab_open = ccl.wrap(n, d_src, d_dst, torch.from_numpy(bits.view(np.int32)).cuda(), gx, gy)
        assert (got_x, got_y) == want, (p, r)
        seen.add(want)
        if r == 0:
            open_mask = mask & ((wx == 0) & (wy == 0)).astype(np.uint8)
            assert np.array_equal(lab_open.cpu().numpy(), oracle.label(n, src, dst, open_mask)), p
        del mask, bits, lab_open
    assert (False, False) in seen and (True, True) in seen


def test_cfg4_regular3_2p24(ccl):
    n = 1 << 24
    src, dst, _ = oracle.gen_regular(n, 3, oracle.seed_for(4))
    d_src, d_dst = ccl.gen_regular(n, 3, oracle.seed_for(4))
    _check(ccl, n, src, dst, d_src, d_dst, [0.5], 4)


def test_cfg5_regular4_2p26(ccl):
    n = 1 << 26
    src, dst, _ = oracle.gen_regular(n, 4, oracle.seed_for(5))
    d_src, d_dst = ccl.gen_regular(n, 4, oracle.seed_for(5))
    torch.cuda.empty_cache()
    _check(ccl, n, src, dst, d_src, d_dst, [0.25, 1.0 / 3.0, 0.45], 5)


def test_maximum_site_count(ccl):
    """n_sites = 2^31 - 1 (the largest the int32 labels allow): 4 M random bonds over the whole range plus a few placed at
    the very ends.  Expected labels of the touched sites come from the oracle on the order-preserving compaction of the
    touched sites (the smallest site of a component stays the smallest); every other site must be its own label."""
    n = (1 << 31) - 1
    rng = np.random.default_rng(2031)
    m = 1 << 22
    src = rng.integers(0, n, size=m, dtype=np.int64)
    dst = rng.integers(0, n, size=m, dtype=np.int64)
    src[:6] = [0, n - 2, 5, n - 1, 1 << 30, (1 << 30) + 1]
    dst[:6] = [n - 1, n - 1, 7, 12345, (1 << 30) - 1, n - 3]
    mask = (rng.random(m) < 0.8).astype(np.uint8)
    mask[:6] = 1
    touched, inv = np.unique(np.concatenate([src, dst]), return_inverse=True)
    csrc, cdst = inv[:m].astype(np.int32), inv[m:].astype(np.int32)
    want_compact = oracle.label(touched.size, csrc, cdst, mask)
    want = touched[want_compact]                                        # expected label of site touched[k]
    s = torch.from_numpy(src.astype(np.int32)).cuda()
    d = torch.from_numpy(dst.astype(np.int32)).cuda()
    for form in ("u8", "bits"):
        if form == "u8":
            lab = ccl.label(n, s, d, torch.from_numpy(mask).cuda())
        else:
            import graphs
            lab = ccl.label_bits(n, s, d, torch.from_numpy(graphs.pack_bits(mask).view(np.int32)).cuda())
        got = lab[torch.from_numpy(touched).cuda()].cpu().numpy().astype(np.int64)
        assert np.array_equal(got, want)
        moved = 0                                                      # sites whose label is not their own index
        step = 1 << 28
        for lo in range(0, n, step):
            hi = min(n, lo + step)
            moved += int((lab[lo:hi] != torch.arange(lo, hi, dtype=torch.int32, device="cuda")).sum().item())
        assert moved == int((want != touched).sum())
        del lab
        torch.cuda.empty_cache()
