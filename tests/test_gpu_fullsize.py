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
