"""The C-ABI library loads and exports every symbol include/ccl.h declares; host-side argument checking works
without a GPU; without a device the compute path fails loudly instead of falling back to anything."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    with open(os.path.join(ROOT, "include", "ccl.h")) as f:
        text = f.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ccl_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported():
    from paper_1603_08357_b200 import binding
    names = _declared()
    assert "ccl_label" in names and "ccl_label_bits" in names and len(names) >= 12
    for n in names:
        assert hasattr(binding.lib, n), n
    assert sorted(binding.EXPORTS) == names
    assert binding.version() >= 100
    assert os.path.dirname(binding._LIB_PATH) == os.path.join(ROOT, "paper_1603_08357_b200")      # in-tree


def test_argument_checking_is_host_side():
    from paper_1603_08357_b200 import binding
    lib = binding.lib
    buf = (C.c_int32 * 64)()
    p = C.addressof(buf)
    assert lib.ccl_label(-1, 0, None, None, None, p, None) == 1
    assert "n_sites" in binding.last_error()
    assert lib.ccl_label(1 << 31, 0, None, None, None, p, None) == 1
    assert lib.ccl_label(4, -1, None, None, None, p, None) == 1
    assert lib.ccl_label(4, 3, None, p, None, p, None) == 1
    assert lib.ccl_label(4, 3, p, p, None, None, None) == 1
    assert lib.ccl_label_bits(4, 3, p, None, None, p, None) == 1
    assert lib.ccl_label(0, 0, None, None, None, None, None) == 0            # empty graph: no-op
    assert lib.ccl_label(4, 0, None, None, None, ((p + 15) & ~15) + 4, None) == 1    # labels must be 16-byte aligned
    assert "16-byte" in binding.last_error()
    assert lib.ccl_set_option(b"no_such_option", 1) == 1
    assert lib.ccl_set_option(b"scatter_tiles", 0) == 0 and lib.ccl_set_option(b"reset", 0) == 0
    assert lib.ccl_gen_triangular(0, p, p, None) == 1
    assert lib.ccl_gen_honeycomb(40000, p, p, None) == 1                      # 2 L^2 > 2^31-1
    assert lib.ccl_gen_occupancy(8, -0.5, 1, 0, p, None, None) == 1
    assert lib.ccl_gen_occupancy(8, 0.5, 1, 0, None, None, None) == 1
    need = C.c_size_t(0)
    assert lib.ccl_gen_regular(5, 3, 1, None, None, None, C.byref(need), None) == 1     # odd stub count
    assert lib.ccl_cluster_stats(-1, None, None, p, None, 0, None, None) == 1
    # the no-allocation variant refuses label arrays beyond its fixed table before it touches the device
    assert lib.ccl_cluster_stats_static(binding.STATS_STATIC_MAX_SITES + 1, p, p, None, 0, None, None) == 1
    assert "CCL_STATS_STATIC_MAX_SITES" in binding.last_error()
    assert lib.ccl_cluster_stats_static(-1, p, p, None, 0, None, None) == 1


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback_without_a_device():
    from paper_1603_08357_b200 import binding
    buf = (C.c_int32 * 64)()
    p = (C.addressof(buf) + 15) & ~15
    rc = binding.lib.ccl_label(4, 0, None, None, None, p, None)
    assert rc == 2 and binding.last_error()                                    # CCL_CUDA_ERROR, not a silent CPU result
    with pytest.raises(TypeError):
        binding.label(4, torch.zeros(2, dtype=torch.int32), torch.zeros(2, dtype=torch.int32))


def test_every_option_is_documented_in_the_header():
    """Every name ccl_set_option accepts is described in include/ccl.h, and the header names no option that is gone."""
    with open(os.path.join(ROOT, "paper_1603_08357_b200", "csrc", "ccl_api.cu")) as f:
        accepted = set(re.findall(r'strcmp\(name, "([a-z0-9_]+)"\)', f.read()))
    with open(os.path.join(ROOT, "include", "ccl.h")) as f:
        text = f.read()
    block = text[text.index("ccl_set_option(name, value)"):text.index("int ccl_set_option(")]
    documented = set(re.findall(r'^ \*   "([a-z0-9_]+)"', block, flags=re.M))
    assert accepted and accepted == documented, (sorted(accepted - documented), sorted(documented - accepted))
    from paper_1603_08357_b200 import binding
    for name in sorted(accepted):
        assert binding.lib.ccl_set_option(name.encode(), -1 if name != "region_shift" else 20) == 0, name
    assert binding.lib.ccl_set_option(b"reset", 0) == 0


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1603_08357_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, f)) as fh:
                    text = fh.read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "liboracle" not in text and "ccl_oracle" not in text, f
    with open(os.path.join(ROOT, "oracle", "ccl_oracle.c")) as fh:
        text = fh.read()
    assert "#include \"" not in text and "cuda" not in text.lower().replace("the cuda library", "")
