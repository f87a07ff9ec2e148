"""ccl_label_nn -- the paper's own interface (nearest-neighbour list, four steps in the paper's form)
against the oracle, bit-exact."""
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


def test_fig1_nn_list_gives_fig4_labels(ccl):
    nn = graphs.read_fig1_nn_list()                         # PAPER.md:41-55, as printed (every bond at both ends)
    want, _ = graphs.read_e0_labels()
    z = max(len(r) for r in nn)
    arr = np.full((z, len(nn)), -1, dtype=np.int32)
    for i, r in enumerate(nn):
        arr[:len(r), i] = r
    assert ccl.label_nn(dev(arr)).cpu().tolist() == want["fig4_right"]


@pytest.mark.parametrize("both_sides", [True, False, "lower", "random"])
def test_random_graphs(ccl, both_sides):
    """include/ccl.h: every entry is a connection, listed from one side or from both -- whichever side."""
    rng = np.random.default_rng(111 + [True, False, "lower", "random"].index(both_sides))
    for trial in range(40):
        n = int(rng.integers(1, 30000))
        m = int(rng.integers(0, 3 * n + 1))
        src, dst = graphs.random_graph(rng, n, m, self_loops=True)
        mask = (rng.random(m) < rng.random()).astype(np.uint8)
        nn = graphs.nn_list_from_bonds(n, src, dst, mask, both_sides, rng)
        got = ccl.label_nn(dev(nn).reshape(nn.shape[0], n)).cpu().numpy()
        want = oracle.label(n, src, dst, mask) if m else np.arange(n, dtype=np.int32)
        assert np.array_equal(got, want)


@pytest.mark.parametrize("family,L,p", [("triangular", 257, 0.3473), ("triangular", 257, 0.52), ("honeycomb", 301, 0.6527),
                                        ("honeycomb", 301, 0.98)])
def test_lattices(ccl, family, L, p):
    src, dst = (oracle.gen_triangular if family == "triangular" else oracle.gen_honeycomb)(L)
    n = (2 if family == "honeycomb" else 1) * L * L
    mask, _ = oracle.gen_occupancy(src.size, p, oracle.seed_for(2))
    nn = graphs.nn_list_from_bonds(n, src, dst, mask)
    assert nn.shape[0] <= (6 if family == "triangular" else 3)
    assert np.array_equal(ccl.label_nn(dev(nn)).cpu().numpy(), oracle.label(n, src, dst, mask))


def test_cayley_tree_and_paths(ccl):
    n, src, dst = oracle.gen_cayley3(15)
    perm = np.random.default_rng(3).permutation(n).astype(np.int32)
    for s, d in [(src, dst), oracle.gen_cayley3(15, perm)[1:]]:
        mask, _ = oracle.gen_occupancy(s.size, 0.75, oracle.seed_for(6))
        nn = graphs.nn_list_from_bonds(n, s, d, mask)
        assert np.array_equal(ccl.label_nn(dev(nn)).cpu().numpy(), oracle.label(n, s, d, mask))
    rng = np.random.default_rng(8)
    for order in ("ascending", "descending", "shuffled"):
        s, d = graphs.path_graph(1 << 18, order, rng)
        for sides in (True, "lower"):
            got = ccl.label_nn(dev(graphs.nn_list_from_bonds(1 << 18, s, d, None, sides)))
            assert int(got.max().item()) == 0 and int(got.min().item()) == 0
    empty = torch.zeros((0, 9), dtype=torch.int32, device="cuda")
    assert ccl.label_nn(empty).cpu().tolist() == list(range(9))
