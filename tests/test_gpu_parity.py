"""Parity of the CUDA path (through the C ABI of libccl.so) with the CPU oracle, element by element, on the same
seeded inputs.  Integer work: the bar is bit-exact.  Inputs always come from the oracle-side generators or from
tests/graphs.py (never from the CUDA path); the device generators are compared against the oracle's separately."""
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


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.view(dtype)
    return t.cuda()


def all_zero(t):
    """Every label is 0: the maximum alone would miss a negative label."""
    return int(t.max().item()) == 0 and int(t.min().item()) == 0


def bits_dev(bits):
    return dev(bits.view(np.int32))


def run_all_forms(ccl, n, src, dst, mask):
    """labels through ccl_label (uint8 mask) and ccl_label_bits (packed); both must equal the oracle's."""
    want = oracle.label(n, src, dst, mask)
    s, d = dev(src), dev(dst)
    got8 = ccl.label(n, s, d, None if mask is None else dev(mask)).cpu().numpy()
    assert np.array_equal(got8, want)
    if mask is not None:
        gotb = ccl.label_bits(n, s, d, bits_dev(graphs.pack_bits(mask))).cpu().numpy()
        assert np.array_equal(gotb, want)
    return want


# ------------------------------------------------------------------ the paper's example and tiny graphs
def test_fig1_example(ccl):
    nn = graphs.read_fig1_nn_list()
    want, _ = graphs.read_e0_labels()
    src, dst = graphs.bonds_from_nn_list(nn)
    got = ccl.label(22, dev(src), dev(dst)).cpu().tolist()
    assert got == want["fig4_right"]                       # PAPER.md:95-107, Fig. 4 right


def test_random_small_graphs(ccl):
    rng = np.random.default_rng(8357)
    for trial in range(120):
        n = int(rng.integers(1, 200))
        m = int(rng.integers(0, 4 * n + 1))
        src, dst = graphs.random_graph(rng, n, m, self_loops=True)
        mask = (rng.random(m) < rng.random()).astype(np.uint8)
        if m == 0:
            got = ccl.label(n, dev(src), dev(dst)).cpu().numpy()
            assert np.array_equal(got, np.arange(n))
            continue
        want = run_all_forms(ccl, n, src, dst, mask)
        assert np.array_equal(want, graphs.bfs_min_labels(n, src, dst, mask))


def test_edge_cases(ccl):
    e = torch.zeros(0, dtype=torch.int32, device="cuda")
    assert ccl.label(0, e, e).numel() == 0
    assert ccl.label(1, e, e).cpu().tolist() == [0]
    assert ccl.label(7, e, e).cpu().tolist() == list(range(7))
    assert ccl.label_bits(7, e, e, None).cpu().tolist() == list(range(7))
    src = dev(np.array([2, 2, 3, 3, 0, 0, 0], dtype=np.int32))
    dst = dev(np.array([2, 4, 3, 3, 1, 1, 1], dtype=np.int32))          # self-loops, duplicates
    assert ccl.label(5, src, dst).cpu().tolist() == [0, 0, 2, 3, 2]
    assert ccl.label(5, src, dst, torch.zeros(7, dtype=torch.uint8, device="cuda")).cpu().tolist() == [0, 1, 2, 3, 4]
    assert ccl.validate_bonds(5, src, dst) == 0 and ccl.validate_bonds(4, src, dst) == 1
    # labels need no initial content
    lab = torch.full((5,), -12345, dtype=torch.int32, device="cuda")
    ccl.label(5, src, dst, labels=lab)
    assert lab.cpu().tolist() == [0, 0, 2, 3, 2]


@pytest.mark.parametrize("m", [1, 2, 3, 4, 5, 31, 32, 33, 127, 1023, 1025, 4099])
def test_ragged_tails_and_unaligned_pointers(ccl, m):
    rng = np.random.default_rng(m)
    n = max(2, m // 2)
    src, dst = graphs.random_graph(rng, n, m)
    mask = (rng.random(m) < 0.7).astype(np.uint8)
    want = run_all_forms(ccl, n, src, dst, mask)
    # unaligned views: element offset 1 breaks the 16-byte alignment of src/dst and the 4-byte alignment of the mask
    s = dev(np.concatenate([[0], src]).astype(np.int32))[1:]
    d = dev(np.concatenate([[0], dst]).astype(np.int32))[1:]
    o = dev(np.concatenate([[1], mask]).astype(np.uint8))[1:]
    assert np.array_equal(ccl.label(n, s, d, o).cpu().numpy(), want)
    assert np.array_equal(ccl.label_bits(n, s, d, bits_dev(graphs.pack_bits(mask))).cpu().numpy(), want)
    # garbage in the unused high bits of the last mask word must be ignored
    bits = graphs.pack_bits(mask).copy()
    if m % 32:
        bits[-1] |= np.uint32(0xFFFFFFFF) << np.uint32(m % 32)
    assert np.array_equal(ccl.label_bits(n, dev(src), dev(dst), bits_dev(bits)).cpu().numpy(), want)


@pytest.mark.parametrize("order", ["ascending", "descending", "shuffled"])
def test_path_graph_worst_case_depth(ccl, order):
    rng = np.random.default_rng(5)
    n = 1 << 20
    src, dst = graphs.path_graph(n, order, rng)
    got = ccl.label(n, dev(src), dev(dst))
    assert int(got.max().item()) == 0 and int(got.min().item()) == 0
    perm = rng.permutation(src.size)
    got = ccl.label(n, dev(src[perm]), dev(dst[perm]))
    assert int(got.max().item()) == 0 and int(got.min().item()) == 0


def test_star_and_clique_contention(ccl):
    n = 1 << 16
    hub = np.full(n - 1, n - 1, dtype=np.int32)              # every bond hits the highest-numbered site
    leaves = np.arange(n - 1, dtype=np.int32)
    assert all_zero(ccl.label(n, dev(hub), dev(leaves)))
    k = 300
    iu = np.triu_indices(k, 1)
    src, dst = iu[1].astype(np.int32) + 5, iu[0].astype(np.int32) + 5
    got = ccl.label(k + 10, dev(src), dev(dst)).cpu().numpy()
    assert np.array_equal(got, oracle.label(k + 10, src, dst))


# ------------------------------------------------------------------ the benchmark workloads, several tiles + tails
def _case(name):
    if name == "cfg1_honeycomb_L64":
        L = 64; src, dst = oracle.gen_honeycomb(L); return 2 * L * L, src, dst, [0.6527], 1
    if name == "honeycomb_L301":
        L = 301; src, dst = oracle.gen_honeycomb(L); return 2 * L * L, src, dst, [0.60, 0.6527, 0.70], 3
    if name == "triangular_L257":
        L = 257; src, dst = oracle.gen_triangular(L); return L * L, src, dst, [0.3473 / 2, 0.3473, 0.52], 2
    if name == "regular3":
        n = (1 << 18) + 2; src, dst, _ = oracle.gen_regular(n, 3, oracle.seed_for(4)); return n, src, dst, [0.25, 0.5, 0.75], 4
    if name == "regular4":
        n = (1 << 19) + 1; src, dst, _ = oracle.gen_regular(n, 4, oracle.seed_for(5)); return n, src, dst, [0.25, 1 / 3, 0.45], 5
    if name == "cayley_standard":
        n, src, dst = oracle.gen_cayley3(16); return n, src, dst, [0.25, 0.5, 0.75], 6
    if name == "cayley_random":
        n, _, _ = oracle.gen_cayley3(16)
        perm = np.random.default_rng(16).permutation(n).astype(np.int32)
        n, src, dst = oracle.gen_cayley3(16, perm); return n, src, dst, [0.25, 0.5, 0.75], 7
    raise KeyError(name)


@pytest.mark.parametrize("name", ["cfg1_honeycomb_L64", "honeycomb_L301", "triangular_L257", "regular3", "regular4",
                                  "cayley_standard", "cayley_random"])
def test_workloads_bit_exact(ccl, name):
    n, src, dst, ps, cfg = _case(name)
    for p in ps + [0.0, 1.0]:
        for r in range(2):
            mask, bits = oracle.gen_occupancy(src.size, p, oracle.seed_for(cfg), realization=r)
            want = run_all_forms(ccl, n, src, dst, mask)
            if p == 0.0:
                assert np.array_equal(want, np.arange(n))
    # repeated calls on the same buffers give the same answer (the call leaves no state behind)
    mask, bits = oracle.gen_occupancy(src.size, ps[-1], oracle.seed_for(cfg))
    s, d, b = dev(src), dev(dst), bits_dev(bits)
    lab = torch.empty(n, dtype=torch.int32, device="cuda")
    first = ccl.label_bits(n, s, d, b, labels=lab).clone()
    for _ in range(3):
        assert torch.equal(ccl.label_bits(n, s, d, b, labels=lab), first)


def test_bond_order_and_orientation_do_not_matter(ccl):
    n, src, dst, ps, cfg = _case("regular4")
    rng = np.random.default_rng(1)
    mask, _ = oracle.gen_occupancy(src.size, 0.45, oracle.seed_for(cfg))
    want = oracle.label(n, src, dst, mask)
    perm = rng.permutation(src.size)
    flip = rng.random(src.size) < 0.5
    s2 = np.where(flip, dst, src)[perm].astype(np.int32)
    d2 = np.where(flip, src, dst)[perm].astype(np.int32)
    assert np.array_equal(ccl.label(n, dev(s2), dev(d2), dev(mask[perm])).cpu().numpy(), want)
    order = np.argsort(np.maximum(src, dst), kind="stable")         # adversarial: all bonds of a site together
    assert np.array_equal(ccl.label(n, dev(src[order]), dev(dst[order]), dev(mask[order])).cpu().numpy(), want)


def test_on_a_side_stream(ccl):
    n, src, dst, ps, cfg = _case("triangular_L257")
    mask, bits = oracle.gen_occupancy(src.size, 0.3473, oracle.seed_for(cfg))
    want = oracle.label(n, src, dst, mask)
    s, d, b = dev(src), dev(dst), bits_dev(bits)
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        got = ccl.label_bits(n, s, d, b)
    st.synchronize()
    assert np.array_equal(got.cpu().numpy(), want)


def test_host_buffer_entry_point(ccl):
    n, src, dst, ps, cfg = _case("regular3")
    mask, bits = oracle.gen_occupancy(src.size, 0.5, oracle.seed_for(cfg))
    want = oracle.label(n, src, dst, mask)
    hs = torch.from_numpy(src).pin_memory()
    hd = torch.from_numpy(dst).pin_memory()
    hb = torch.from_numpy(bits.view(np.int32)).pin_memory()
    out = torch.empty(n, dtype=torch.int32).pin_memory()
    ccl.label_bits_host(n, hs, hd, hb, out)
    assert np.array_equal(out.numpy(), want)
    out2 = torch.empty(n, dtype=torch.int32)                         # pageable memory works too
    ccl.label_bits_host(n, torch.from_numpy(src), torch.from_numpy(dst), torch.from_numpy(bits.view(np.int32)), out2)
    assert np.array_equal(out2.numpy(), want)


def test_host_buffer_sweep_entry_point(ccl):
    n, src, dst, ps, cfg = _case("regular4")
    hs, hd = torch.from_numpy(src).pin_memory(), torch.from_numpy(dst).pin_memory()
    masks, wants = [], []
    for r, p in enumerate([0.25, 1 / 3, 0.45, 0.0, 1.0]):
        mask, bits = oracle.gen_occupancy(src.size, p, oracle.seed_for(cfg), realization=r)
        masks.append(torch.from_numpy(bits.view(np.int32)).pin_memory())
        wants.append(oracle.label(n, src, dst, mask))
    masks.append(None)                                               # no mask: every bond occupied
    wants.append(oracle.label(n, src, dst))
    outs = [torch.empty(n, dtype=torch.int32).pin_memory() for _ in masks]
    ccl.label_sweep_host(n, hs, hd, masks, outs)
    for got, want in zip(outs, wants):
        assert np.array_equal(got.numpy(), want)
    one = [torch.empty(n, dtype=torch.int32)]                        # a single mask, pageable memory
    ccl.label_sweep_host(n, torch.from_numpy(src), torch.from_numpy(dst), [torch.from_numpy(masks[2].numpy().copy())], one)
    assert np.array_equal(one[0].numpy(), wants[2])
    ccl.label_sweep_host(n, hs, hd, [], [])


# ------------------------------------------------------------------ region-bucketed form of step (iii)
@pytest.fixture
def bucketed(ccl):
    """Force the bucketed form on small inputs: every call eligible, 2^10..2^14-site regions."""
    yield ccl
    ccl.set_tuning()                                   # restore defaults


@pytest.mark.parametrize("shift,cap", [(10, 0), (12, 0), (14, 0), (12, 64), (16, 1000), (11, 20000)])
def test_bucketed_form_random_small_graphs(bucketed, shift, cap):
    ccl = bucketed
    ccl.set_tuning(0, shift, 1, cap)                   # cap > 0: a pool of one to three chunks; when it runs dry the pairs are
                                                       # dropped and the direct kernel redoes the bond list behind the descent
    rng = np.random.default_rng(shift * 131 + cap)
    for trial in range(40):
        n = int(rng.integers(2, 60000))
        m = int(rng.integers(1, 3 * n + 1))
        src, dst = graphs.random_graph(rng, n, m, self_loops=True)
        mask = (rng.random(m) < rng.random()).astype(np.uint8)
        run_all_forms(ccl, n, src, dst, mask)
        assert np.array_equal(ccl.label(n, dev(src), dev(dst)).cpu().numpy(), oracle.label(n, src, dst))


@pytest.mark.parametrize("name", ["cfg1_honeycomb_L64", "honeycomb_L301", "triangular_L257", "regular3", "regular4",
                                  "cayley_standard", "cayley_random"])
@pytest.mark.parametrize("mode", [1, -1])
def test_bucketed_form_workloads_bit_exact(bucketed, name, mode):
    ccl = bucketed
    n, src, dst, ps, cfg = _case(name)
    ccl.set_tuning(0, 15, mode, 0)                     # 2^15-site regions; mode -1 lets the device probe choose
    for p in ps + [1.0]:
        mask, bits = oracle.gen_occupancy(src.size, p, oracle.seed_for(cfg), realization=5)
        run_all_forms(ccl, n, src, dst, mask)


@pytest.mark.parametrize("m", [2047, 2048, 2049, 4096, 6143, 6144 + 7, 10 * 2048 + 2047])
def test_bucketed_scatter_tile_boundaries(bucketed, m):
    """The bulk-copy scatter kernel takes whole 2048-bond tiles of 16-byte aligned input, the register kernel the tail,
    unaligned input and everything when the tiles are switched off: bond counts around the tile size, every mask kind
    (none, uint8, packed), aligned and unaligned views, both kernels."""
    ccl = bucketed
    rng = np.random.default_rng(m)
    n = 5000
    src, dst = graphs.random_graph(rng, n, m, self_loops=True)
    mask = (rng.random(m) < 0.6).astype(np.uint8)
    want = oracle.label(n, src, dst, mask)
    want_all = oracle.label(n, src, dst)
    bits = graphs.pack_bits(mask)
    for tiles in (1, 0):
        ccl.set_tuning(0, 9, 1, 0)                     # 2^9-site regions: ten of them
        ccl.set_option("scatter_tiles", tiles)
        s, d = dev(src), dev(dst)
        assert np.array_equal(ccl.label(n, s, d, dev(mask)).cpu().numpy(), want)
        assert np.array_equal(ccl.label_bits(n, s, d, bits_dev(bits)).cpu().numpy(), want)
        assert np.array_equal(ccl.label(n, s, d).cpu().numpy(), want_all)
        # element offset 1: src/dst lose their 16-byte alignment, the masks theirs
        s1 = dev(np.concatenate([[0], src]).astype(np.int32))[1:]
        d1 = dev(np.concatenate([[0], dst]).astype(np.int32))[1:]
        o1 = dev(np.concatenate([[1], mask]).astype(np.uint8))[1:]
        assert np.array_equal(ccl.label(n, s1, d1, o1).cpu().numpy(), want)
        assert np.array_equal(ccl.label_bits(n, s1, d1, bits_dev(bits)).cpu().numpy(), want)
        b1 = dev(np.concatenate([[0], bits.view(np.int32)]).astype(np.int32))[1:]      # packed mask 4-, not 16-byte aligned
        assert np.array_equal(ccl.label_bits(n, s, d, b1).cpu().numpy(), want)


def test_bucketed_form_adversarial(bucketed):
    ccl = bucketed
    ccl.set_tuning(0, 12, 1, 0)
    rng = np.random.default_rng(99)
    n = 1 << 17
    for order in ("ascending", "descending", "shuffled"):
        src, dst = graphs.path_graph(n, order, rng)
        assert all_zero(ccl.label(n, dev(src), dev(dst)))
    hub = np.full(n - 1, n - 1, dtype=np.int32)        # star on the highest site: every pair lands in one bucket
    leaves = np.arange(n - 1, dtype=np.int32)
    assert all_zero(ccl.label(n, dev(hub), dev(leaves)))
    # interleaved path 0, n/2, 1, n/2+1, ...: every bond crosses regions and the lower half becomes one long chain
    half = n // 2
    i = np.arange(half - 1, dtype=np.int32)
    src = np.concatenate([i, i + half]).astype(np.int32)
    dst = np.concatenate([i + half, i + 1]).astype(np.int32)
    got = ccl.label(n, dev(src), dev(dst)).cpu().numpy()
    assert np.array_equal(got, oracle.label(n, src, dst))


@pytest.fixture
def options(ccl):
    yield ccl
    ccl.set_option("reset")


# ------------------------------------------------------------------ two-pass direct form (hook, flatten, join)
@pytest.mark.parametrize("two_pass", [0, 1])
def test_two_pass_form(options, two_pass):
    ccl = options
    ccl.set_option("reset")
    ccl.set_option("two_pass", two_pass)
    rng = np.random.default_rng(31 + two_pass)
    for trial in range(40):
        n = int(rng.integers(2, 50000))
        m = int(rng.integers(1, 4 * n + 1))
        src, dst = graphs.random_graph(rng, n, m, self_loops=True)
        mask = (rng.random(m) < rng.random()).astype(np.uint8)
        run_all_forms(ccl, n, src, dst, mask)
    for name in ["honeycomb_L301", "triangular_L257", "regular4", "cayley_random"]:
        n, src, dst, ps, cfg = _case(name)
        for p in ps + [1.0]:
            mask, bits = oracle.gen_occupancy(src.size, p, oracle.seed_for(cfg), realization=9)
            run_all_forms(ccl, n, src, dst, mask)
    n = 1 << 18
    for order in ("ascending", "descending", "shuffled"):
        src, dst = graphs.path_graph(n, order, rng)
        assert all_zero(ccl.label(n, dev(src), dev(dst)))


def test_options_belong_to_the_calling_thread(ccl):
    """ccl_set_option on another host thread cannot change a call on this one (and vice versa): the knobs are
    thread-local like the error string and the launch counter, and a call reads them once on entry."""
    import threading
    rng = np.random.default_rng(77)
    n, m = 50000, 120000
    src, dst = graphs.random_graph(rng, n, m)
    s, d = dev(src), dev(dst)
    want = oracle.label(n, src, dst)
    ccl.set_option("reset")
    base = ccl.launch_count()
    ccl.label(n, s, d)
    plain = ccl.launch_count() - base                      # direct form: k_init, k_reduce, k_flatten
    seen = {}

    def other():
        torch.cuda.set_device(0)
        ccl.set_option("bucket_min_label_bytes", 0)        # on THIS thread every call takes the bucketed form
        ccl.set_option("region_shift", 12)
        ccl.set_option("force_mode", 1)
        before = ccl.launch_count()
        got = ccl.label(n, s, d)
        seen["launches"] = ccl.launch_count() - before
        seen["ok"] = bool(np.array_equal(got.cpu().numpy(), want))
    t = threading.Thread(target=other)
    t.start()
    t.join()
    assert seen["ok"] and seen["launches"] > plain         # the other thread really ran another path
    base = ccl.launch_count()
    got = ccl.label(n, s, d)
    assert ccl.launch_count() - base == plain              # ... and this thread's options are untouched
    assert np.array_equal(got.cpu().numpy(), want)


def test_scratch_is_reported_and_can_be_trimmed(ccl):
    """include/ccl.h: scratch stays in the library's pool for the next call until ccl_trim_scratch hands it back."""
    torch.cuda.synchronize()
    ccl.trim_scratch(0)                                    # whatever earlier tests left in the pool
    ccl.set_tuning(0, 16, 1, 0)                            # bucketed form: draws a workspace
    rng = np.random.default_rng(5)
    n, m = 1 << 20, 1 << 22                                # cfg4-like shape, scaled
    src, dst = graphs.random_graph(rng, n, m)
    got = ccl.label(n, dev(src), dev(dst))
    torch.cuda.synchronize()
    reserved, in_use = ccl.scratch_bytes()
    assert reserved >= 8 * m and in_use == 0               # pair chunks for >= m pairs were drawn and returned to the pool
    assert reserved <= 16 * m + (64 << 20)                 # ... and the pool is sized by the pairs that can exist (1.25 M), not 4 M
    ccl.trim_scratch(0)
    assert ccl.scratch_bytes()[0] == 0
    assert np.array_equal(got.cpu().numpy(), oracle.label(n, src, dst))
    assert np.array_equal(ccl.label(n, dev(src), dev(dst)).cpu().numpy(), got.cpu().numpy())     # works again after a trim
    ccl.set_tuning()
    ccl.trim_scratch(0)


def test_chunk_pool_grows_after_running_dry(ccl):
    """The pair pool of the bucketed form holds 1.25 pairs per bond.  A densely occupied random graph files about 2.5: the
    first call runs dry and is finished by the direct kernel behind the bucketed kernels, which also tells the host; the
    next calls on the same bond list draw a pool twice (four, eight times) as large.  Labels are right every time."""
    torch.cuda.synchronize()
    ccl.trim_scratch(0)
    ccl.set_tuning(0, 16, 1, 0)                            # bucketed form, 2^16-site regions, default pool size
    rng = np.random.default_rng(808)
    n, m = 1 << 20, 1 << 22                                # (large enough for the pool's 32 MiB granules to show)
    src, dst = graphs.random_graph(rng, n, m)
    s, d = dev(src), dev(dst)
    want = oracle.label(n, src, dst)
    reserved = []
    for rep in range(5):
        got = ccl.label(n, s, d)                           # every bond occupied
        torch.cuda.synchronize()
        assert np.array_equal(got.cpu().numpy(), want), rep
        reserved.append(ccl.scratch_bytes()[0])
    assert reserved[1] > reserved[0]                       # the second call drew a larger pool
    assert reserved[-1] == reserved[-2]                    # ... and it stops growing once nothing is dropped
    assert reserved[-1] <= 8 * reserved[0]
    ccl.set_tuning()
    ccl.trim_scratch(0)


def test_remembered_direct_answer_draws_no_workspace(ccl):
    """The bucketed form is an optimisation.  Once the probe's answer for a bond list is "direct" and the host remembers
    it, later calls on that bond list reserve nothing from the pool (include/ccl.h, "What a call draws")."""
    rng = np.random.default_rng(31)
    n, m = 300000, 900000
    src = rng.integers(0, n, size=m).astype(np.int32)
    dst = np.clip(src + rng.integers(-3, 4, size=m), 0, n - 1).astype(np.int32)      # local in the site numbering
    s, d = dev(src), dev(dst)
    want = oracle.label(n, src, dst)
    ccl.set_option("reset")
    ccl.set_option("bucket_min_label_bytes", 0)
    ccl.set_option("region_shift", 13)
    assert np.array_equal(ccl.label(n, s, d).cpu().numpy(), want)         # first call: both forms behind the probe
    torch.cuda.synchronize()
    ccl.trim_scratch(0)
    assert np.array_equal(ccl.label(n, s, d).cpu().numpy(), want)         # remembered: direct kernels only
    torch.cuda.synchronize()
    assert ccl.scratch_bytes() == (0, 0)
    ccl.set_option("reset")


def test_workspace_that_cannot_be_allocated_falls_back_to_the_direct_kernels(ccl):
    """A pool request the device cannot satisfy (here: room for 2^40 pairs) must not fail the call -- the direct kernels
    need no workspace -- and must not poison later calls on the same bond list."""
    rng = np.random.default_rng(32)
    n, m = 200000, 600000
    src, dst = graphs.random_graph(rng, n, m)
    s, d = dev(src), dev(dst)
    mask = (rng.random(m) < 0.5).astype(np.uint8)
    want = oracle.label(n, src, dst, mask)
    for force in (1, -1):
        ccl.set_tuning(0, 13, force, 1 << 40)
        for rep in range(2):
            assert np.array_equal(ccl.label(n, s, d, dev(mask)).cpu().numpy(), want), (force, rep)
        torch.cuda.synchronize()
    ccl.set_tuning(0, 13, 1, 0)                                          # an ordinary pool again: the bucketed form runs
    before = ccl.launch_count()
    assert np.array_equal(ccl.label(n, s, d, dev(mask)).cpu().numpy(), want)
    assert ccl.launch_count() - before > 6                                # scatter + one descend per region + ...
    ccl.set_tuning()
    ccl.trim_scratch(0)


def test_l2_persist_option_changes_no_label(ccl):
    """ccl_set_option("l2_persist", 1) attaches an access-policy window to the k_descend / windowed k_flatten launches:
    a cache hint, so the labels are the oracle's either way (bucketed form forced on small graphs, several regions and
    several flatten windows)."""
    rng = np.random.default_rng(77)
    n, m = 150000, 400000
    src, dst = graphs.random_graph(rng, n, m, self_loops=True)
    mask = (rng.random(m) < 0.55).astype(np.uint8)
    want = oracle.label(n, src, dst, mask)
    s, d, mk = dev(src), dev(dst), dev(mask)
    for on in (1, 0):
        ccl.set_tuning(0, 14, 1, 0)
        ccl.set_option("flatten_window_min_bytes", 0)
        ccl.set_option("flatten_window_bytes", 1 << 17)
        ccl.set_option("l2_persist", on)
        for rep in range(2):
            assert np.array_equal(ccl.label(n, s, d, mk).cpu().numpy(), want), (on, rep)
    ccl.set_tuning()
    ccl.trim_scratch(0)


def test_probe_cache_on_and_off(ccl):
    """The host-side memory of the device probe's answer changes which kernels are enqueued, never the labels: repeated
    calls on one bond list (first call: probe undecided, later calls: decided) and the same with the cache off."""
    rng = np.random.default_rng(21)
    n, m = 200000, 500000
    for local in (False, True):
        src, dst = graphs.random_graph(rng, n, m)
        if local:
            dst = np.clip(src + rng.integers(-3, 4, size=m), 0, n - 1).astype(np.int32)
        s, d = dev(src), dev(dst)
        for cache in (1, 0):
            ccl.set_option("reset")
            ccl.set_option("bucket_min_label_bytes", 0)
            ccl.set_option("region_shift", 13)
            ccl.set_option("probe_cache", cache)
            counts = []
            for rep in range(4):
                mask = (rng.random(m) < 0.6).astype(np.uint8)
                before = ccl.launch_count()
                got = ccl.label(n, s, d, dev(mask))
                torch.cuda.synchronize()                   # lets the probe's answer reach the host
                counts.append(ccl.launch_count() - before)
                assert np.array_equal(got.cpu().numpy(), oracle.label(n, src, dst, mask)), (local, cache, rep)
            if cache and local:
                assert counts[-1] < counts[0]              # once decided, only the chosen (direct) form is enqueued
                ccl.set_option("probe_cache", 1)           # setting the option forgets the remembered bond lists
                before = ccl.launch_count()
                got = ccl.label(n, s, d, dev(mask))
                torch.cuda.synchronize()
                assert ccl.launch_count() - before == counts[0]        # ... so this is a first call again
                assert np.array_equal(got.cpu().numpy(), oracle.label(n, src, dst, mask))
            elif not cache:
                assert counts[-1] == counts[0]
    ccl.set_option("reset")


def test_tuning_argument_checks(ccl):
    with pytest.raises(ccl.CclError):
        ccl.set_tuning(0, 2, 0)
    with pytest.raises(ccl.CclError):
        ccl.set_tuning(0, 12, 5)
    ccl.set_tuning()


def test_no_write_outside_the_label_buffer(ccl):
    """Guard bands around every output buffer stay untouched (compute-sanitizer is not available on the GPU pool)."""
    rng = np.random.default_rng(404)
    GUARD, MAGIC = 64, -77
    for n in (1, 5, 1023, 1024, 1025, 32768, 32769, 100001):
        m = 3 * n
        src, dst = graphs.random_graph(rng, n, m, self_loops=True)
        mask = (rng.random(m) < 0.5).astype(np.uint8)
        want = oracle.label(n, src, dst, mask)
        s, d, b = dev(src), dev(dst), bits_dev(graphs.pack_bits(mask))

        def guarded():
            buf = torch.full((n + 2 * GUARD,), MAGIC, dtype=torch.int32, device="cuda")
            return buf, buf[GUARD:GUARD + n]

        def intact(buf):
            return bool((buf[:GUARD] == MAGIC).all().item()) and bool((buf[GUARD + n:] == MAGIC).all().item())

        for opts in ({}, {"two_pass": 1}, {"flatten_window_min_bytes": 0, "flatten_window_bytes": 4096},
                     {"bucket_min_label_bytes": 0, "region_shift": 10, "force_mode": 1},
                     {"bucket_min_label_bytes": 0, "region_shift": 10, "scatter_tiles": 0},
                     {"bucket_min_label_bytes": 0, "region_shift": 10, "bucket_capacity": 100, "flatten_window_bytes": 8192}):
            ccl.set_option("reset")
            for k, v in opts.items():
                ccl.set_option(k, v)
            buf, lab = guarded()
            if GUARD % 4 == 0:                                  # labels must be 16-byte aligned
                ccl.label_bits(n, s, d, b, labels=lab)
                assert intact(buf) and np.array_equal(lab.cpu().numpy(), want), (n, opts)
        ccl.set_option("reset")
        buf, lab = guarded()
        seq, c = ccl.relabel_sequential(dev(want), out=lab)
        assert intact(buf) and c == int((want == np.arange(n)).sum())
        if n <= 32768:
            buf = torch.full((3 * n + 2 * GUARD,), MAGIC, dtype=torch.int32, device="cuda")
            out = buf[GUARD:GUARD + 3 * n].view(3, n)
            ccl.label_batch(n, s, d, torch.stack([b, b, b]), 3, labels=out)
            assert bool((buf[:GUARD] == MAGIC).all().item()) and bool((buf[GUARD + 3 * n:] == MAGIC).all().item())
            assert np.array_equal(out[2].cpu().numpy(), want)
        buf, lab = guarded()
        ccl.label_nn(dev(graphs.nn_list_from_bonds(n, src, dst, mask)), labels=lab)
        assert intact(buf) and np.array_equal(lab.cpu().numpy(), want)
