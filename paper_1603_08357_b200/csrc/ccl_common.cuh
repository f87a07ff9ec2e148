// ccl_common.cuh -- host-side plumbing shared by the translation units of libccl.so (error string, launch
// counter, stream cast) and the small device helpers (cache-hinted loads/stores).  Product code: nothing under
// oracle/ is included from here or includes this.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/ccl.h"

namespace ccl {

// Number of SMs of the current device (queried once per device and cached; grids are capped at a multiple of it).
// 148 on B200 (2 dies x 74 SMs), which is also what is assumed should the query fail.
int sm_count();

// ---- host plumbing ---------------------------------------------------------------------------------------
void set_error(const char* fmt, ...);
void count_launch(int n = 1);

inline cudaStream_t as_stream(void* s) { return reinterpret_cast<cudaStream_t>(s); }

#define CCL_CUDA_TRY(expr)                                                                         \
    do {                                                                                           \
        cudaError_t err__ = (expr);                                                                \
        if (err__ != cudaSuccess) {                                                                \
            ::ccl::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(err__), __FILE__,   \
                             __LINE__);                                                            \
            return CCL_CUDA_ERROR;                                                                 \
        }                                                                                          \
    } while (0)

#define CCL_CHECK_LAUNCH(name)                                                                     \
    do {                                                                                           \
        cudaError_t err__ = cudaGetLastError();                                                    \
        if (err__ != cudaSuccess) {                                                                \
            ::ccl::set_error("launch of %s failed: %s", name, cudaGetErrorString(err__));          \
            return CCL_CUDA_ERROR;                                                                 \
        }                                                                                          \
        ::ccl::count_launch();                                                                     \
    } while (0)

#define CCL_REQUIRE(cond, msg)                                                                     \
    do {                                                                                           \
        if (!(cond)) {                                                                             \
            ::ccl::set_error("invalid argument: %s", msg);                                         \
            return CCL_INVALID_ARG;                                                                \
        }                                                                                          \
    } while (0)

// ---- programmatic dependent launch -----------------------------------------------------------------------
// A kernel launched with launch_pdl may be scheduled while its predecessor on the stream is still draining; it calls
// pdl_wait() before it touches anything the predecessor wrote (the wait returns when the predecessor has completed and
// its writes are visible), and pdl_go() early, to let its own successor be scheduled the same way.  This hides the
// launch latency between the kernels of one call (a dozen short launches on config 5).  Both calls are no-ops in a
// kernel that was launched the ordinary way.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_go() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... Params, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(Params...), unsigned grid, unsigned block, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<Params>(args)...);
}

template <typename... Params, typename... Args>
inline cudaError_t launch_pdl_smem(void (*kernel)(Params...), unsigned grid, unsigned block, size_t smem, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<Params>(args)...);
}

// ---- L2 residency: a per-launch access-policy window ---------------------------------------------------------
// The bucketed form works on one slice of label[] at a time (a region in k_descend, a gather window in k_flatten).
// With ccl_set_option("l2_persist", 1) those launches carry cudaLaunchAttributeAccessPolicyWindow over their slice
// (hitProp = persisting), so that the streams passing through L2 in the same launch (pair chunks, the sites above
// the window) do not push the slice out.  l2_persist_bytes() sets the device-wide limit
// cudaLimitPersistingL2CacheSize to the device's maximum on first use (a side effect on the whole device, documented
// in include/ccl.h) and returns it; 0 = not available.
struct L2Window {
    const void* base = nullptr;
    size_t bytes = 0;                              // 0: no window
};
size_t l2_persist_bytes();
size_t l2_max_window_bytes();

template <typename... Params, typename... Args>
inline cudaError_t launch_pdl_window(void (*kernel)(Params...), unsigned grid, unsigned block, size_t smem, cudaStream_t st,
                                     L2Window win, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const size_t persist = win.bytes ? l2_persist_bytes() : 0;
    if (persist > 0) {
        size_t bytes = win.bytes;
        const size_t max_window = l2_max_window_bytes();
        if (max_window > 0 && bytes > max_window) bytes = max_window;
        attr[1].id = cudaLaunchAttributeAccessPolicyWindow;
        attr[1].val.accessPolicyWindow.base_ptr = const_cast<void*>(win.base);
        attr[1].val.accessPolicyWindow.num_bytes = bytes;
        attr[1].val.accessPolicyWindow.hitRatio = bytes <= persist ? 1.0f : (float)((double)persist / (double)bytes);
        attr[1].val.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
        attr[1].val.accessPolicyWindow.missProp = cudaAccessPropertyNormal;
        cfg.numAttrs = 2;
    }
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<Params>(args)...);
}

// ---- region-bucketed label reduction (ccl_bucket.cu) -----------------------------------------------------
constexpr int kMaxRegions = 32;
constexpr int kMinChunkShift = 11, kMaxChunkShift = 21;   // a bucket is a sequence of chunks of 2^11 .. 2^21 pairs

struct BucketHeader {                              // lives in device memory at the head of the call's workspace
    int32_t mode;                                  // written by probe_regions: 0 = direct kernels, 1 = bucketed kernels
    int32_t overflow;                              // != 0: the chunk pool ran dry and pairs were dropped; the direct kernel
                                                   // then runs over the whole bond list behind the bucketed kernels
    unsigned int next_chunk;                       // chunks handed out so far
    unsigned int pad;
    unsigned long long count[kMaxRegions];         // pairs filed under each region (logical length of its bucket)
};

struct Tuning {                                    // ccl_set_option(); one set of knobs per host thread
    int64_t bucket_min_label_bytes = 96ll << 20;   // label[] beyond this cannot stay resident in the 126 MB L2
    int64_t bucket_min_bonds = 1 << 20;
    int32_t region_shift = 23;                     // 2^23 sites = 32 MiB of labels per region
    int32_t force_mode = -1;                       // -1: device-side probe decides; 0: direct; 1: bucketed
    int64_t bucket_capacity = 0;                   // pairs the chunk pool can hold; 0 = 5 M / 4 + slack
    int32_t two_pass = -1;                         // direct form of step (iii): 0 one pass (k_reduce), 1 hook + flatten +
                                                   // join (the paper's order), -1 by bonds per site (>= 2.5: two passes)
    int32_t scatter_tiles = 1;                     // 1: k_scatter_tiles (bulk copies into shared memory) for aligned input
    int32_t probe_cache = 1;                       // remember the probe's answer per bond list (host side, hint only)
    int64_t flatten_window_bytes = 64ll << 20;     // step (iv) gathers from one L2-resident window of label[] at a time
    int64_t flatten_window_min_bytes = 96ll << 20; // ... for label arrays of at least this size (0: always; < 0: never)
    int32_t l2_persist = 0;                        // 1: k_descend / windowed k_flatten launches carry an access-policy window
};
Tuning& tuning();

void forget_probe_hints();                         // ccl_label.cu: drops this host thread's per-bond-list memory (R15)

// The library's own stream-ordered memory pool on the current device (created on first use; ccl_trim_scratch returns
// what it holds to the driver), so scratch freed by one call is reused by the next.
int scratch_alloc(void** ptr, size_t bytes, cudaStream_t st);

struct ProbeJob {                                  // the region probe rides in block 0 of k_init (ccl_label.cu)
    BucketHeader* hdr = nullptr;                   // NULL: no probe
    int64_t n_bonds = 0;
    const int32_t* src = nullptr;
    const int32_t* dst = nullptr;
    int shift = 0;
};
struct BucketPlan {
    BucketHeader* hdr = nullptr;
    unsigned int* table = nullptr;                 // table[r * stride + k] = 1 + pool index of the k-th chunk of bucket r
    int2* pool = nullptr;
    unsigned int n_chunks = 0, stride = 0;
    int shift = 0, n_regions = 0;
    int cshift = kMinChunkShift;                   // chunk = 2^cshift pairs
    int scatter_tiles = 1;
    int l2_persist = 0;
    int lazy_init = 0;                             // 1: label[] of region r is written by the kernel that runs before k_descend(r)
    int gated = 0;                                 // 1: the kernels return at once unless hdr->mode == 1 (probe undecided on the host)
};
// bucketed_begin allocates and clears the workspace (*ws_out: the caller frees it with cudaFreeAsync after the last
// kernel that reads it has been enqueued); bucketed_launch enqueues k_scatter and one k_descend per region.
int bucket_region_shift(int64_t n_sites, const Tuning& t);
int bucketed_begin(int64_t n_sites, int64_t n_bonds, const Tuning& t, int pool_doublings, cudaStream_t st, BucketPlan* plan,
                   void** ws_out);
int bucketed_launch(const BucketPlan& plan, int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                    const void* occ, int mask_kind, int32_t* labels, cudaStream_t st);

// ---- device helpers --------------------------------------------------------------------------------------
// Streaming (read-once) loads: bypass L1 allocation and mark the L2 line evict-first, so that the bond stream
// does not push label[] sectors out of L2.
__device__ __forceinline__ uint64_t evict_first_policy()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ int4 ld_stream_v4(const int32_t* p, uint64_t pol)
{
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.s32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ int32_t ld_stream_s32(const int32_t* p, uint64_t pol)
{
    int32_t r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.s32 %0, [%1], %2;" : "=r"(r) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ uint32_t ld_stream_u32(const uint32_t* p, uint64_t pol)
{
    uint32_t r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.u32 %0, [%1], %2;" : "=r"(r) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ uint32_t ld_stream_u8(const uint8_t* p, uint64_t pol)
{
    uint32_t r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.u8 %0, [%1], %2;" : "=r"(r) : "l"(p), "l"(pol));
    return r;
}

__device__ __forceinline__ void st_stream_pair(int2* p, int2 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.s32 [%0], {%1, %2}, %3;" ::"l"(p), "r"(v.x), "r"(v.y), "l"(pol)
                 : "memory");
}

// Samples up to 8192 bonds at a fixed stride and looks at how many join two different regions (random numbering: 1 - 1/R of
// them; raster-ordered lattice: only those on region borders): mode 1 = region-bucketed form, 0 = direct kernels.  Called
// by all threads of ONE block.
__device__ __forceinline__ void probe_regions(const ProbeJob& job)
{
    __shared__ int s_cross;
    if (threadIdx.x == 0) s_cross = 0;
    __syncthreads();
    const int64_t samples = job.n_bonds < 8192 ? job.n_bonds : 8192;
    const int64_t stride = job.n_bonds / samples;
    int cross = 0;
#pragma unroll 8
    for (int64_t i = threadIdx.x; i < samples; i += blockDim.x) {
        const int32_t u = job.src[i * stride], v = job.dst[i * stride];
        cross += (u >> job.shift) != (v >> job.shift);
    }
    for (int o = 16; o > 0; o >>= 1) cross += __shfl_xor_sync(0xffffffffu, cross, o);
    if ((threadIdx.x & 31) == 0 && cross) atomicAdd(&s_cross, cross);
    __syncthreads();
    if (threadIdx.x == 0) job.hdr->mode = (4 * (int64_t)s_cross >= samples) ? 1 : 0;
}

// Label reads during root finding and flattening go through L1 (ld.global.ca).  L1 is not coherent, so a read may
// return an older value of label[x] -- which is still an ancestor of x, so every walk stays correct and only gets a
// little longer; every decision that matters is re-validated by the value an atomicMin
// returns.  What L1 buys: the top of a big cluster's tree is read by every walk through that cluster, and with
// L2-only loads (ld.relaxed.gpu, the first version) those reads all queue up at the one L2 slice that owns the
// sector (k_flatten on honeycomb p = 0.70: 1.29 ms with L2-only loads, 0.14 ms through L1; round 1).
__device__ __forceinline__ int32_t ld_label(const int32_t* p)
{
    int32_t r;
    asm volatile("ld.global.ca.s32 %0, [%1];" : "=r"(r) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st_label(int32_t* p, int32_t v)
{
    asm volatile("st.relaxed.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// read-once load of data this thread may write afterwards (no .nc): skips L1 allocation, evict-first in L2
__device__ __forceinline__ int4 ld_once_v4(const int32_t* p, uint64_t pol)
{
    int4 r;
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v4.s32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p), "l"(pol)
                 : "memory");
    return r;
}
__device__ __forceinline__ void st_stream_v4(int32_t* p, int4 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v4.s32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
                 "r"(v.w), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p)
{
    unsigned int r;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(r) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st_release_u32(unsigned int* p, unsigned int v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// label[i] = i for i in [lo, hi), lo a multiple of 4, 16-byte stores; called by `nthreads` threads with ranks `rank`.
__device__ __forceinline__ void init_range(int32_t* __restrict__ label, int64_t lo, int64_t hi, int64_t rank, int64_t nthreads)
{
    for (int64_t i = lo + rank * 4; i < hi; i += nthreads * 4) {
        if (i + 4 <= hi) {
            const int32_t b = (int32_t)i;
            *reinterpret_cast<int4*>(label + i) = make_int4(b, b + 1, b + 2, b + 3);   // label is 16 B aligned
        } else {
            for (int64_t j = i; j < hi; ++j) label[j] = (int32_t)j;
        }
    }
}

}  // namespace ccl
