"""ctypes binding of libccl.so.  Same names as include/ccl.h without the `ccl_` prefix; marshalling only.

Every compute call takes torch CUDA tensors (device memory owned by the caller) and enqueues on torch's current
stream.  Nothing here computes: every step of the path runs in the CUDA kernels of csrc/.
"""
import ctypes as C

import torch

from .build import build

_LIB_PATH = build()            # raises if nvcc fails: no fallback
lib = C.CDLL(_LIB_PATH)

EXPORTS = ["ccl_label", "ccl_label_bits", "ccl_validate_bonds", "ccl_gen_triangular", "ccl_gen_honeycomb",
           "ccl_gen_regular", "ccl_gen_occupancy", "ccl_cluster_stats", "ccl_label_bits_host",
           "ccl_set_profile_events", "ccl_set_option", "ccl_label_batch", "ccl_relabel_sequential", "ccl_gen_cayley3",
           "ccl_gen_wrap_vectors", "ccl_wrap", "ccl_label_nn", "ccl_label_sweep_host", "ccl_trim_scratch",
           "ccl_scratch_bytes", "ccl_cluster_stats_static", "ccl_last_error", "ccl_version", "ccl_launch_count"]

_vp, _i64, _i32, _u64, _u32 = C.c_void_p, C.c_int64, C.c_int32, C.c_uint64, C.c_uint32
lib.ccl_label.argtypes = [_i64, _i64, _vp, _vp, _vp, _vp, _vp]
lib.ccl_label_bits.argtypes = [_i64, _i64, _vp, _vp, _vp, _vp, _vp]
lib.ccl_label_bits_host.argtypes = [_i64, _i64, _vp, _vp, _vp, _vp, _vp]
lib.ccl_validate_bonds.argtypes = [_i64, _i64, _vp, _vp, _vp, _vp]
lib.ccl_gen_triangular.argtypes = [_i32, _vp, _vp, _vp]
lib.ccl_gen_honeycomb.argtypes = [_i32, _vp, _vp, _vp]
lib.ccl_gen_regular.argtypes = [_i64, _i32, _u64, _vp, _vp, _vp, C.POINTER(C.c_size_t), _vp]
lib.ccl_gen_occupancy.argtypes = [_i64, C.c_double, _u64, _u32, _vp, _vp, _vp]
lib.ccl_cluster_stats.argtypes = [_i64, _vp, _vp, _vp, _vp, _i32, _vp, _vp]
lib.ccl_cluster_stats_static.argtypes = [_i64, _vp, _vp, _vp, _i32, _vp, _vp]
lib.ccl_last_error.restype = C.c_char_p
lib.ccl_last_error.argtypes = []
lib.ccl_version.argtypes = []
lib.ccl_launch_count.restype = _i64
lib.ccl_launch_count.argtypes = []
lib.ccl_set_profile_events.argtypes = [_vp, _vp, _vp]
lib.ccl_set_option.argtypes = [C.c_char_p, _i64]
lib.ccl_label_batch.argtypes = [_i64, _i64, _vp, _vp, _vp, _i64, _i32, _vp, _vp]
lib.ccl_relabel_sequential.argtypes = [_i64, _vp, _vp, _vp, _vp, C.POINTER(C.c_size_t), _vp]
lib.ccl_gen_cayley3.argtypes = [_i32, _vp, _vp, _vp, _vp]
lib.ccl_gen_wrap_vectors.argtypes = [_i32, _i32, _vp, _vp, _vp]
lib.ccl_wrap.argtypes = [_i64, _i64, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.POINTER(C.c_size_t), _vp]
lib.ccl_label_nn.argtypes = [_i64, _i32, _vp, _vp, _vp]
lib.ccl_label_sweep_host.argtypes = [_i64, _i64, _vp, _vp, _i32, _vp, _vp, _vp]
lib.ccl_trim_scratch.argtypes = [C.c_size_t, _vp]
lib.ccl_scratch_bytes.argtypes = [C.POINTER(_i64), C.POINTER(_i64)]
for _n in EXPORTS[:21]:
    getattr(lib, _n).restype = C.c_int


class CclError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        super().__init__("%s failed with status %d: %s" % (what, code, last_error()))


def last_error():
    return lib.ccl_last_error().decode()


def version():
    return lib.ccl_version()


def launch_count():
    return int(lib.ccl_launch_count())


def _check(rc, what):
    if rc != 0:
        raise CclError(rc, what)


def _stream():
    return torch.cuda.current_stream().cuda_stream


def _dev(t, dtype, what):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CUDA tensor of dtype %s" % (what, dtype))
    return t.data_ptr()


def _sizes(n_sites, n_bonds, labels, mask, mask_len, what):
    """The C ABI takes bare pointers: refuse tensors that are shorter than the counts say."""
    if labels.numel() < n_sites:
        raise ValueError("%s: labels has %d elements, n_sites = %d" % (what, labels.numel(), n_sites))
    if mask is not None and mask.numel() < mask_len:
        raise ValueError("%s: the occupancy tensor has %d elements, %d are needed" % (what, mask.numel(), mask_len))


def label(n_sites, src, dst, occupied=None, labels=None):
    """ccl_label: uint8 mask (or None = all bonds occupied).  Returns the int32 label tensor."""
    if labels is None:
        labels = torch.empty(n_sites, dtype=torch.int32, device=src.device)
    if dst.numel() < src.numel():
        raise ValueError("ccl_label: dst is shorter than src")
    _sizes(n_sites, src.numel(), labels, occupied, src.numel(), "ccl_label")
    _check(lib.ccl_label(n_sites, src.numel(), _dev(src, torch.int32, "src"), _dev(dst, torch.int32, "dst"),
                         _dev(occupied, torch.uint8, "occupied"), _dev(labels, torch.int32, "labels"), _stream()),
           "ccl_label")
    return labels


def label_bits(n_sites, src, dst, occupied_bits, labels=None, n_bonds=None):
    """ccl_label_bits: packed mask as an int32 tensor of ceil(n_bonds/32) words (bit b&31 of word b>>5)."""
    if labels is None:
        labels = torch.empty(n_sites, dtype=torch.int32, device=src.device)
    m = src.numel() if n_bonds is None else n_bonds
    if src.numel() < m or dst.numel() < m:
        raise ValueError("ccl_label_bits: src/dst are shorter than n_bonds")
    _sizes(n_sites, m, labels, occupied_bits, (m + 31) // 32, "ccl_label_bits")
    _check(lib.ccl_label_bits(n_sites, m, _dev(src, torch.int32, "src"), _dev(dst, torch.int32, "dst"),
                              _dev(occupied_bits, torch.int32, "occupied_bits"),
                              _dev(labels, torch.int32, "labels"), _stream()), "ccl_label_bits")
    return labels


def label_nn(nn_list, labels=None):
    """ccl_label_nn: nn_list is an int32 CUDA tensor [z_max, n_sites] (negative = padding)."""
    z_max, n_sites = nn_list.shape
    if labels is None:
        labels = torch.empty(n_sites, dtype=torch.int32, device=nn_list.device)
    _check(lib.ccl_label_nn(n_sites, z_max, _dev(nn_list, torch.int32, "nn_list"), _dev(labels, torch.int32, "labels"),
                            _stream()), "ccl_label_nn")
    return labels


def label_batch(n_sites, src, dst, occupied_bits, n_batch, labels=None):
    """ccl_label_batch: occupied_bits is an int32 tensor [n_batch, words >= ceil(n_bonds/32)] (or None); returns int32
    labels [n_batch, n_sites].  One launch, one CTA per realization; n_sites <= 32768."""
    if labels is None:
        labels = torch.empty((n_batch, n_sites), dtype=torch.int32, device=src.device)
    stride = 0 if occupied_bits is None else (occupied_bits.shape[1] if occupied_bits.dim() == 2 else occupied_bits.numel() // max(n_batch, 1))
    _check(lib.ccl_label_batch(n_sites, src.numel(), _dev(src, torch.int32, "src"), _dev(dst, torch.int32, "dst"),
                               _dev(occupied_bits, torch.int32, "occupied_bits"), stride, n_batch,
                               _dev(labels, torch.int32, "labels"), _stream()), "ccl_label_batch")
    return labels


def relabel_sequential(labels, out=None):
    """ccl_relabel_sequential: canonical labels -> (sequential labels 0..C-1, C)."""
    n = labels.numel()
    if out is None:
        out = torch.empty_like(labels)
    need = C.c_size_t(0)
    _check(lib.ccl_relabel_sequential(n, None, None, None, None, C.byref(need), _stream()), "ccl_relabel_sequential")
    ws = torch.empty(max(need.value, 1), dtype=torch.uint8, device=labels.device)
    count = torch.zeros(1, dtype=torch.int64, device=labels.device)
    _check(lib.ccl_relabel_sequential(n, _dev(labels, torch.int32, "labels"), _dev(out, torch.int32, "out"),
                                      count.data_ptr(), ws.data_ptr(), C.byref(need), _stream()), "ccl_relabel_sequential")
    return out, int(count.item())


def _host(t, what):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CPU int32 tensor" % what)
    return t.data_ptr()


def label_bits_host(n_sites, src, dst, occupied_bits, labels):
    """ccl_label_bits_host: HOST tensors in (pinned for full speed), host labels out; synchronises."""
    _check(lib.ccl_label_bits_host(n_sites, src.numel(), _host(src, "src"), _host(dst, "dst"),
                                   _host(occupied_bits, "occupied_bits"), _host(labels, "labels"), _stream()),
           "ccl_label_bits_host")
    return labels


def label_sweep_host(n_sites, src, dst, masks, labels):
    """ccl_label_sweep_host: HOST tensors; masks / labels are lists of CPU int32 tensors (a mask may be None)."""
    n = len(masks)
    assert len(labels) == n
    mp = (C.c_void_p * n)(*[_host(m, "mask") for m in masks])
    lp = (C.c_void_p * n)(*[_host(t, "labels") for t in labels])
    _check(lib.ccl_label_sweep_host(n_sites, src.numel(), _host(src, "src"), _host(dst, "dst"), n, mp, lp, _stream()),
           "ccl_label_sweep_host")
    return labels


def set_profile_events(after_init=None, after_reduce=None, after_flatten=None):
    """ccl_set_profile_events with torch.cuda.Event objects (created with enable_timing=True) or None."""
    def h(e):
        if e is None:
            return None
        e.record()                      # torch creates the underlying cudaEvent_t lazily: force it into existence
        return e.cuda_event
    _check(lib.ccl_set_profile_events(h(after_init), h(after_reduce), h(after_flatten)), "ccl_set_profile_events")


def set_option(name, value=0):
    """ccl_set_option(name, value); see include/ccl.h for the names."""
    _check(lib.ccl_set_option(name.encode(), int(value)), "ccl_set_option")


def trim_scratch(keep_bytes=0):
    """ccl_trim_scratch on torch's current stream (synchronises it)."""
    _check(lib.ccl_trim_scratch(int(keep_bytes), _stream()), "ccl_trim_scratch")


def scratch_bytes():
    """ccl_scratch_bytes: (reserved, in_use) of the library's memory pool on the current device."""
    r, u = _i64(0), _i64(0)
    _check(lib.ccl_scratch_bytes(C.byref(r), C.byref(u)), "ccl_scratch_bytes")
    return int(r.value), int(u.value)


def set_tuning(bucket_min_label_bytes=-1, region_shift=-1, force_mode=-1, bucket_capacity=0):
    """Convenience for the tests: reset, then set the four knobs of the bucketed form."""
    set_option("reset")
    set_option("bucket_min_label_bytes", bucket_min_label_bytes)
    set_option("region_shift", region_shift)
    set_option("force_mode", force_mode)
    set_option("bucket_capacity", bucket_capacity)


def validate_bonds(n_sites, src, dst):
    """Number of bonds with an endpoint outside [0, n_sites) (synchronises to return a Python int)."""
    out = torch.zeros(1, dtype=torch.int64, device=src.device)
    _check(lib.ccl_validate_bonds(n_sites, src.numel(), _dev(src, torch.int32, "src"), _dev(dst, torch.int32, "dst"),
                                  out.data_ptr(), _stream()), "ccl_validate_bonds")
    return int(out.item())


def _lattice(fn, name, L, device):
    m = 3 * L * L
    src = torch.empty(m, dtype=torch.int32, device=device)
    dst = torch.empty(m, dtype=torch.int32, device=device)
    _check(fn(L, src.data_ptr(), dst.data_ptr(), _stream()), name)
    return src, dst


def gen_triangular(L, device="cuda"):
    return _lattice(lib.ccl_gen_triangular, "ccl_gen_triangular", L, device)


def gen_honeycomb(L, device="cuda"):
    return _lattice(lib.ccl_gen_honeycomb, "ccl_gen_honeycomb", L, device)


def gen_wrap_vectors(family, L, device="cuda"):
    """ccl_gen_wrap_vectors: (wx, wy) int8 tensors for the bonds of gen_triangular ("triangular") / gen_honeycomb."""
    fam = {"triangular": 0, "honeycomb": 1}[family]
    wx = torch.empty(3 * L * L, dtype=torch.int8, device=device)
    wy = torch.empty(3 * L * L, dtype=torch.int8, device=device)
    _check(lib.ccl_gen_wrap_vectors(fam, L, wx.data_ptr(), wy.data_ptr(), _stream()), "ccl_gen_wrap_vectors")
    return wx, wy


def wrap(n_sites, src, dst, occupied_bits, wx, wy, labels_open=None):
    """ccl_wrap: (wrap_x, wrap_y, labels_open).  Reads the flags back (synchronises)."""
    if labels_open is None:
        labels_open = torch.empty(n_sites, dtype=torch.int32, device=src.device)
    need = C.c_size_t(0)
    _check(lib.ccl_wrap(n_sites, src.numel(), None, None, None, None, None, None, None, None, C.byref(need), _stream()), "ccl_wrap")
    ws = torch.empty(need.value, dtype=torch.uint8, device=src.device)
    out = torch.zeros(4, dtype=torch.int32, device=src.device)
    _check(lib.ccl_wrap(n_sites, src.numel(), _dev(src, torch.int32, "src"), _dev(dst, torch.int32, "dst"),
                        _dev(occupied_bits, torch.int32, "occupied_bits"), _dev(wx, torch.int8, "wx"), _dev(wy, torch.int8, "wy"),
                        _dev(labels_open, torch.int32, "labels_open"), out.data_ptr(), ws.data_ptr(), C.byref(need), _stream()),
           "ccl_wrap")
    flags = out.cpu().tolist()
    if flags[2]:
        raise CclError(3, "ccl_wrap (sheet offset overflow)")
    return bool(flags[0]), bool(flags[1]), labels_open


def gen_cayley3(g, perm=None, device="cuda"):
    """ccl_gen_cayley3: (n_sites, src, dst) of the z = 3 Cayley tree with g generations; perm = int32 CUDA permutation."""
    n = 3 * (1 << g) - 2
    src = torch.empty(n - 1, dtype=torch.int32, device=device)
    dst = torch.empty(n - 1, dtype=torch.int32, device=device)
    _check(lib.ccl_gen_cayley3(g, _dev(perm, torch.int32, "perm"), src.data_ptr(), dst.data_ptr(), _stream()),
           "ccl_gen_cayley3")
    return n, src, dst


def gen_regular(n_sites, z, seed, device="cuda"):
    m = n_sites * z // 2
    need = C.c_size_t(0)
    _check(lib.ccl_gen_regular(n_sites, z, seed, None, None, None, C.byref(need), _stream()), "ccl_gen_regular(size)")
    ws = torch.empty(need.value, dtype=torch.uint8, device=device)
    src = torch.empty(m, dtype=torch.int32, device=device)
    dst = torch.empty(m, dtype=torch.int32, device=device)
    _check(lib.ccl_gen_regular(n_sites, z, seed, src.data_ptr(), dst.data_ptr(), ws.data_ptr(), C.byref(need),
                               _stream()), "ccl_gen_regular")
    del ws
    return src, dst


def gen_occupancy(n_bonds, p, seed, realization=0, want_mask=True, want_bits=True, device="cuda"):
    """(uint8 mask or None, int32-typed packed bits or None)."""
    mask = torch.empty(n_bonds, dtype=torch.uint8, device=device) if want_mask else None
    bits = torch.empty((n_bonds + 31) // 32, dtype=torch.int32, device=device) if want_bits else None
    _check(lib.ccl_gen_occupancy(n_bonds, float(p), seed, realization, None if mask is None else mask.data_ptr(),
                                 None if bits is None else bits.data_ptr(), _stream()), "ccl_gen_occupancy")
    return mask, bits


class Stats(C.Structure):
    _fields_ = [("n_clusters", C.c_int64), ("largest", C.c_int64), ("largest_label", C.c_int64), ("sum_s2", C.c_uint64)]


def cluster_stats(labels, n_dense=0):
    """(dict of exact integers, hist_dense[n_dense+1] int64 CPU tensor, hist_log2[32]); synchronises to read back."""
    n = labels.numel()
    dev = labels.device
    scratch = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
    out = torch.empty(4, dtype=torch.int64, device=dev)
    hd = torch.empty(n_dense + 1, dtype=torch.int64, device=dev)
    hl = torch.empty(32, dtype=torch.int64, device=dev)
    _check(lib.ccl_cluster_stats(n, _dev(labels, torch.int32, "labels"), scratch.data_ptr(), out.data_ptr(),
                                 hd.data_ptr(), n_dense, hl.data_ptr(), _stream()), "ccl_cluster_stats")
    o = out.cpu().tolist()
    d = dict(n_clusters=o[0], largest=o[1], largest_label=o[2], sum_s2=o[3] & 0xFFFFFFFFFFFFFFFF)
    return d, hd.cpu(), hl.cpu()


STATS_STATIC_MAX_SITES = 1 << 22       # CCL_STATS_STATIC_MAX_SITES of include/ccl.h


def cluster_stats_static(labels, n_dense=0, out=None, hist_dense=None, hist_log2=None):
    """ccl_cluster_stats_static: cluster_stats for callers that cannot allocate device memory (all of it belongs to
    their own arena, or a cudaMalloc's device-wide synchronisation is not acceptable where they call from).  The size
    table sits in a fixed 16 MiB array inside libccl.so, so at most STATS_STATIC_MAX_SITES labels; the library call
    allocates nothing.  Pass `out` (int64[4]), `hist_dense` (int64[n_dense+1]) and `hist_log2` (int64[32]) CUDA
    tensors to keep this wrapper from allocating the outputs as well.  Calls on one device share the array: do not
    let two of them overlap on the GPU.  Returns like cluster_stats (synchronises to read back)."""
    n = labels.numel()
    dev = labels.device
    out = torch.empty(4, dtype=torch.int64, device=dev) if out is None else out
    hd = torch.empty(n_dense + 1, dtype=torch.int64, device=dev) if hist_dense is None else hist_dense
    hl = torch.empty(32, dtype=torch.int64, device=dev) if hist_log2 is None else hist_log2
    if out.numel() < 4 or hd.numel() < n_dense + 1 or hl.numel() < 32:
        raise ValueError("ccl_cluster_stats_static: an output tensor is too short")
    _check(lib.ccl_cluster_stats_static(n, _dev(labels, torch.int32, "labels"), _dev(out, torch.int64, "out"),
                                        _dev(hd, torch.int64, "hist_dense"), n_dense,
                                        _dev(hl, torch.int64, "hist_log2"), _stream()), "ccl_cluster_stats_static")
    o = out.cpu().tolist()
    d = dict(n_clusters=o[0], largest=o[1], largest_label=o[2], sum_s2=o[3] & 0xFFFFFFFFFFFFFFFF)
    return d, hd.cpu(), hl.cpu()
