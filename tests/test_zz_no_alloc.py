"""ccl_cluster_stats_static -- the statistics reducer for callers that cannot allocate device memory.

Who that is: a program that reserved the whole GPU for its own arena at start-up (any further cudaMalloc fails), or
code on a path where cudaMalloc / cudaFree are off limits because they synchronise the device.  Such a caller cannot
hand ccl_cluster_stats the int32-per-site scratch it asks for, so this entry point keeps that table in a fixed 16 MiB
array inside libccl.so (at most CCL_STATS_STATIC_MAX_SITES = 2^22 sites) and allocates nothing.

What is checked: the same exact integers as the existing ccl_cluster_stats on the same labels, on calls in a row
that share the array (a larger input, then a smaller one, then the larger one again: counters left behind by one call
must not reach the next), that the calls reserve no device memory, and that sizes past the limit are refused.

The file name sorts last on purpose: the array is shared by every call in the process, and `pytest -x` would hide
every test behind a failure here.
"""
import ctypes as C

import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ccl():
    import paper_1603_08357_b200 as pkg
    assert torch.cuda.is_available()
    return pkg


def _labels(ccl, family, L, p, seed):
    """Canonical labels from the library's own generators and ccl_label_bits (no oracle needed here)."""
    src, dst = (ccl.gen_triangular if family == "triangular" else ccl.gen_honeycomb)(L)
    n_sites = L * L if family == "triangular" else 2 * L * L
    _, bits = ccl.gen_occupancy(src.numel(), p, seed, 0, want_mask=False)
    return ccl.label_bits(n_sites, src, dst, bits)


def _same(a, b):
    (sa, hda, hla), (sb, hdb, hlb) = a, b
    assert sa == sb                                             # exact integers: n_clusters, largest, its label, sum s^2
    assert torch.equal(hda, hdb) and torch.equal(hla, hlb)


def test_two_calls_in_a_row_match_the_allocating_path(ccl):
    big = _labels(ccl, "triangular", 700, 0.3473, 11)           # 490000 sites, at the threshold: clusters of all sizes
    small = _labels(ccl, "honeycomb", 100, 0.70, 12)            # 20000 sites, one giant cluster
    n_dense = 64
    want_big = ccl.cluster_stats(big, n_dense)
    want_small = ccl.cluster_stats(small, n_dense)
    assert want_big[0]["n_clusters"] > 1000 and want_small[0]["largest"] > 10000
    _same(ccl.cluster_stats_static(big, n_dense), want_big)     # first call on this device: looks the array up
    _same(ccl.cluster_stats_static(small, n_dense), want_small) # reuses the array: big's counters must be gone
    _same(ccl.cluster_stats_static(big, n_dense), want_big)     # and the other way round
    _same(ccl.cluster_stats_static(big, n_dense), want_big)     # same input twice


def test_the_calls_reserve_no_device_memory(ccl):
    from paper_1603_08357_b200 import binding
    labels = _labels(ccl, "triangular", 512, 0.40, 13)
    want = ccl.cluster_stats(labels, 8)
    out = torch.empty(4, dtype=torch.int64, device="cuda")
    hd = torch.empty(9, dtype=torch.int64, device="cuda")
    hl = torch.empty(32, dtype=torch.int64, device="cuda")
    ccl.cluster_stats_static(labels, 8, out=out, hist_dense=hd, hist_log2=hl)      # set-up call (kernels get loaded)
    torch.cuda.synchronize()
    pool_before = ccl.scratch_bytes()
    free_before = torch.cuda.mem_get_info()[0]
    stream = torch.cuda.current_stream().cuda_stream
    for _ in range(2):                                          # straight through the C ABI: no tensor is created
        rc = binding.lib.ccl_cluster_stats_static(labels.numel(), labels.data_ptr(), out.data_ptr(), hd.data_ptr(), 8,
                                                  hl.data_ptr(), stream)
        assert rc == 0, binding.last_error()
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before          # the driver handed out nothing
    assert ccl.scratch_bytes() == pool_before                   # and neither did the library's pool
    o = out.cpu().tolist()
    assert dict(n_clusters=o[0], largest=o[1], largest_label=o[2], sum_s2=o[3]) == want[0]
    assert torch.equal(hd.cpu(), want[1]) and torch.equal(hl.cpu(), want[2])


def test_largest_size_and_one_beyond(ccl):
    from paper_1603_08357_b200 import binding
    n_max = binding.STATS_STATIC_MAX_SITES
    ident = torch.arange(n_max + 1, dtype=torch.int32, device="cuda")      # every site its own cluster
    got, _, hl = ccl.cluster_stats_static(ident[:n_max], 0)
    assert got == dict(n_clusters=n_max, largest=1, largest_label=0, sum_s2=n_max) and int(hl[0]) == n_max
    with pytest.raises(binding.CclError) as e:
        ccl.cluster_stats_static(ident, 0)
    assert e.value.code == 1 and "CCL_STATS_STATIC_MAX_SITES" in str(e.value)
    # the refusal left the array usable
    assert ccl.cluster_stats_static(ident[:1000], 0)[0]["n_clusters"] == 1000


def test_empty_input(ccl):
    got, _, _ = ccl.cluster_stats_static(torch.zeros(0, dtype=torch.int32, device="cuda"), 4)
    assert got == dict(n_clusters=0, largest=0, largest_label=-1, sum_s2=0)
