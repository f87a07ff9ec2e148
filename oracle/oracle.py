"""ctypes front end of oracle/ccl_oracle.c (numpy in, numpy out).  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Every function is a thin marshalling wrapper; the arithmetic lives in ccl_oracle.c, where each function cites the
passage of PAPER.md (arXiv 1603.08357) or the DESIGN.md reading it follows.
"""
import ctypes as C
import numpy as np

from .build import build

_lib = C.CDLL(build())

_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
_i64p = np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS")


class Stats(C.Structure):
    _fields_ = [("n_clusters", C.c_int64), ("largest", C.c_int64), ("largest_label", C.c_int64), ("sum_s2", C.c_uint64)]


def _ptr(a, ctype):
    return None if a is None else a.ctypes.data_as(C.POINTER(ctype))


_lib.oracle_label.restype = C.c_int
_lib.oracle_label.argtypes = [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.oracle_label_bits.restype = C.c_int
_lib.oracle_label_bits.argtypes = [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.oracle_stats.restype = C.c_int
_lib.oracle_stats.argtypes = [C.c_int64, C.c_void_p, C.POINTER(Stats), C.c_void_p, C.c_int32, C.c_void_p]
_lib.oracle_wrap.restype = C.c_int
_lib.oracle_wrap.argtypes = [C.c_int64, C.c_int64] + [C.c_void_p] * 6
_lib.oracle_philox4x32_10.restype = None
_lib.oracle_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.oracle_gen_triangular.restype = C.c_int
_lib.oracle_gen_triangular.argtypes = [C.c_int32] + [C.c_void_p] * 4
_lib.oracle_gen_honeycomb.restype = C.c_int
_lib.oracle_gen_honeycomb.argtypes = [C.c_int32] + [C.c_void_p] * 4
_lib.oracle_gen_occupancy.restype = C.c_int
_lib.oracle_gen_occupancy.argtypes = [C.c_int64, C.c_double, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p]
_lib.oracle_gen_regular.restype = C.c_int
_lib.oracle_gen_regular.argtypes = [C.c_int64, C.c_int32, C.c_uint64, C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)]
_lib.oracle_gen_cayley3.restype = C.c_int
_lib.oracle_gen_cayley3.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]


def _addr(a):
    return None if a is None else a.ctypes.data


def _check(rc, what):
    if rc != 0:
        raise RuntimeError("%s failed with code %d" % (what, rc))


def _bonds(src, dst):
    src = np.ascontiguousarray(src, dtype=np.int32)
    dst = np.ascontiguousarray(dst, dtype=np.int32)
    assert src.shape == dst.shape and src.ndim == 1
    return src, dst


def label(n_sites, src, dst, occupied=None):
    """labels[i] = smallest site index in i's component; occupied: uint8 per bond or None (= all)."""
    src, dst = _bonds(src, dst)
    occ = None if occupied is None else np.ascontiguousarray(occupied, dtype=np.uint8)
    assert occ is None or occ.shape == src.shape
    labels = np.empty(n_sites, dtype=np.int32)
    _check(_lib.oracle_label(n_sites, src.size, _addr(src), _addr(dst), _addr(occ), _addr(labels)), "oracle_label")
    return labels


def label_bits(n_sites, src, dst, occupied_bits):
    """Same with a packed mask: bond b is bit (b & 31) of uint32 word (b >> 5)."""
    src, dst = _bonds(src, dst)
    bits = None if occupied_bits is None else np.ascontiguousarray(occupied_bits, dtype=np.uint32)
    assert bits is None or bits.size >= (src.size + 31) // 32
    labels = np.empty(n_sites, dtype=np.int32)
    _check(_lib.oracle_label_bits(n_sites, src.size, _addr(src), _addr(dst), _addr(bits), _addr(labels)),
           "oracle_label_bits")
    return labels


def stats(labels, n_dense=0):
    """(dict, hist_dense[n_dense+1] with [0] unused, hist_log2[32]) from canonical labels."""
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    st = Stats()
    hd = np.zeros(n_dense + 1, dtype=np.int64)
    hl = np.zeros(32, dtype=np.int64)
    _check(_lib.oracle_stats(labels.size, _addr(labels), C.byref(st), _addr(hd), n_dense, _addr(hl)), "oracle_stats")
    d = dict(n_clusters=int(st.n_clusters), largest=int(st.largest), largest_label=int(st.largest_label),
             sum_s2=int(st.sum_s2))
    return d, hd, hl


def relabel_sequential(labels):
    """the min-site labels renumbered sequentially.  Cluster k (k = 0..C-1) is the one with the k-th
    smallest label; returns (seq, C).  Written out from the definition: a site is a root iff labels[i] == i, and
    seq[i] = number of roots below labels[i]."""
    labels = np.asarray(labels, dtype=np.int64)
    is_root = labels == np.arange(labels.size)
    below = np.cumsum(is_root) - is_root          # roots strictly below each index
    return below[labels].astype(np.int32), int(is_root.sum())


def wrap(n_sites, src, dst, dx, dy, occupied=None):
    """(wrap_x, wrap_y): does some cluster hold a cycle with non-zero x / y winding (reading R7)."""
    src, dst = _bonds(src, dst)
    dx = np.ascontiguousarray(dx, dtype=np.int8)
    dy = np.ascontiguousarray(dy, dtype=np.int8)
    occ = None if occupied is None else np.ascontiguousarray(occupied, dtype=np.uint8)
    out = np.zeros(2, dtype=np.int32)
    _check(_lib.oracle_wrap(n_sites, src.size, _addr(src), _addr(dst), _addr(dx), _addr(dy), _addr(occ), _addr(out)),
           "oracle_wrap")
    return bool(out[0]), bool(out[1])


def philox4x32_10(ctr, key):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    assert ctr.size == 4 and key.size == 2
    out = np.empty(4, dtype=np.uint32)
    _lib.oracle_philox4x32_10(_addr(ctr), _addr(key), _addr(out))
    return out


def _lattice(fn, L, n_bonds, with_disp):
    src = np.empty(n_bonds, dtype=np.int32)
    dst = np.empty(n_bonds, dtype=np.int32)
    dx = np.empty(n_bonds, dtype=np.int8) if with_disp else None
    dy = np.empty(n_bonds, dtype=np.int8) if with_disp else None
    _check(fn(L, _addr(src), _addr(dst), _addr(dx), _addr(dy)), "lattice generator")
    return (src, dst, dx, dy) if with_disp else (src, dst)


def gen_triangular(L, with_disp=False):
    """L*L sites, 3*L*L bonds (DESIGN.md input recipe)."""
    return _lattice(_lib.oracle_gen_triangular, L, 3 * L * L, with_disp)


def gen_honeycomb(L, with_disp=False):
    """2*L*L sites, 3*L*L bonds."""
    return _lattice(_lib.oracle_gen_honeycomb, L, 3 * L * L, with_disp)


def gen_occupancy(n_bonds, p, seed, realization=0):
    """(uint8 mask[n_bonds], uint32 bits[ceil(n_bonds/32)])."""
    mask = np.empty(n_bonds, dtype=np.uint8)
    bits = np.empty((n_bonds + 31) // 32, dtype=np.uint32)
    _check(_lib.oracle_gen_occupancy(n_bonds, float(p), seed, realization, _addr(mask), _addr(bits)),
           "oracle_gen_occupancy")
    return mask, bits


def gen_regular(n_sites, z, seed):
    """(src, dst, n_repaired) of a simple random z-regular graph, n_sites*z/2 bonds in random order."""
    m = n_sites * z // 2
    src = np.empty(m, dtype=np.int32)
    dst = np.empty(m, dtype=np.int32)
    nrep = C.c_int64(0)
    _check(_lib.oracle_gen_regular(n_sites, z, seed, _addr(src), _addr(dst), C.byref(nrep)), "oracle_gen_regular")
    return src, dst, int(nrep.value)


def gen_cayley3(g, perm=None):
    """Cayley tree z=3 with g generations: N = 3*2^g - 2 sites, N-1 bonds."""
    n = 3 * (1 << g) - 2
    src = np.empty(n - 1, dtype=np.int32)
    dst = np.empty(n - 1, dtype=np.int32)
    p = None if perm is None else np.ascontiguousarray(perm, dtype=np.int32)
    assert p is None or p.size == n
    _check(_lib.oracle_gen_cayley3(g, _addr(p), _addr(src), _addr(dst)), "oracle_gen_cayley3")
    return n, src, dst


def seed_for(cfg):
    """Seed convention of DESIGN.md's input recipe: 0x1603_0835_7000_0000 + cfg."""
    return 0x1603083570000000 + cfg
