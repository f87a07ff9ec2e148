"""ccl_label_batch (many realizations, one launch) and ccl_relabel_sequential against the oracle,
bit-exact.  Inputs come from the oracle-side generators only."""
import numpy as np
import pytest
import torch

import graphs
from oracle import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ccl():
    import paper_1603_08357_b200 as pkg
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; there is no CPU fallback"
    return pkg


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("family,L", [("honeycomb", 64), ("honeycomb", 7), ("triangular", 128), ("triangular", 181)])
def test_batch_of_lattice_realizations(ccl, family, L):
    src, dst = (oracle.gen_honeycomb if family == "honeycomb" else oracle.gen_triangular)(L)
    n = (2 if family == "honeycomb" else 1) * L * L
    ps = [0.0, 0.3473, 0.5, 0.6527, 0.70, 1.0]
    n_batch = 24
    words = (src.size + 31) // 32 + 3                       # a stride larger than the mask itself
    bits = np.zeros((n_batch, words), dtype=np.uint32)
    want = []
    for r in range(n_batch):
        mask, b = oracle.gen_occupancy(src.size, ps[r % len(ps)], oracle.seed_for(1), realization=r)
        bits[r, :b.size] = b
        bits[r, b.size:] = 0xFFFFFFFF                        # padding words are never read as bonds
        want.append(oracle.label(n, src, dst, mask))
    got = ccl.label_batch(n, dev(src), dev(dst), dev(bits.view(np.int32)), n_batch).cpu().numpy()
    assert got.shape == (n_batch, n)
    for r in range(n_batch):
        assert np.array_equal(got[r], want[r]), "realization %d" % r
    # no mask: every bond occupied in every realization
    full = ccl.label_batch(n, dev(src), dev(dst), None, 3).cpu().numpy()
    assert not full.any()


def test_batch_random_graphs_and_edge_cases(ccl):
    rng = np.random.default_rng(2024)
    for trial in range(25):
        n = int(rng.integers(1, 3000)) if trial else 1 << 15
        m = int(rng.integers(1, 3 * n + 1))
        src, dst = graphs.random_graph(rng, n, m, self_loops=True)
        n_batch = int(rng.integers(1, 6))
        masks = (rng.random((n_batch, m)) < rng.random()).astype(np.uint8)
        bits = np.stack([graphs.pack_bits(masks[r]) for r in range(n_batch)])
        got = ccl.label_batch(n, dev(src), dev(dst), dev(bits.view(np.int32)), n_batch).cpu().numpy()
        for r in range(n_batch):
            assert np.array_equal(got[r], oracle.label(n, src, dst, masks[r]))
    e = torch.zeros(0, dtype=torch.int32, device="cuda")
    assert ccl.label_batch(5, e, e, None, 2).cpu().tolist() == [[0, 1, 2, 3, 4]] * 2
    assert ccl.label_batch(5, e, e, None, 0).numel() == 0
    with pytest.raises(ccl.CclError):                        # does not fit one CTA's shared memory
        ccl.label_batch((1 << 15) + 1, e, e, None, 1)
    path = np.arange(1 << 15, dtype=np.int32)                # worst-case depth inside one CTA
    assert not ccl.label_batch(1 << 15, dev(path[:-1]), dev(path[1:]), None, 2).any().item()


@pytest.mark.parametrize("n", [1, 2, 255, 256, 257, 100003, (1 << 20) + 5])
def test_relabel_sequential(ccl, n):
    rng = np.random.default_rng(n)
    m = int(0.6 * n)
    src, dst = graphs.random_graph(rng, n, m) if m else (np.zeros(0, np.int32), np.zeros(0, np.int32))
    labels = oracle.label(n, src, dst) if m else np.arange(n, dtype=np.int32)
    want, c = oracle.relabel_sequential(labels)
    lab = dev(labels)
    got, count = ccl.relabel_sequential(lab)
    assert count == c and np.array_equal(got.cpu().numpy(), want)
    got2, count2 = ccl.relabel_sequential(lab, out=lab)      # in place
    assert count2 == c and np.array_equal(lab.cpu().numpy(), want)


def test_relabel_after_labeling_a_lattice(ccl):
    L = 300
    src, dst = oracle.gen_triangular(L)
    mask, bits = oracle.gen_occupancy(src.size, 0.3473, oracle.seed_for(2))
    lab = ccl.label_bits(L * L, dev(src), dev(dst), dev(bits.view(np.int32)))
    seq, c = ccl.relabel_sequential(lab)
    want, wc = oracle.relabel_sequential(oracle.label(L * L, src, dst, mask))
    assert c == wc and np.array_equal(seq.cpu().numpy(), want)
    stats, _, _ = ccl.cluster_stats(lab, 0)
    assert stats["n_clusters"] == c
