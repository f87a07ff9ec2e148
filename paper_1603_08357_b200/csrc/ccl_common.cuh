// ccl_common.cuh -- host-side plumbing shared by the translation units of libccl.so (error string, launch
// counter, stream cast) and the small device helpers (cache-hinted loads/stores).  Product code: nothing under
// oracle/ is included from here or includes this.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/ccl.h"

namespace ccl {

constexpr int kSMs = 148;                 // B200: 2 dies x 74 SMs

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

// ---- region-bucketed label reduction (ccl_bucket.cu) -----------------------------------------------------
constexpr int kMaxRegions = 32;

struct BucketHeader {                              // lives in device memory at the head of the call's workspace
    int32_t mode;                                  // written by probe_regions: 0 = direct kernel, 1 = bucketed, 2 = nothing
    int32_t pad;
    unsigned long long count[kMaxRegions];         // pairs filed under each region (may exceed the capacity: the
                                                   // excess was joined on the spot by the general algorithm)
};

// Header of the tiled form's workspace (ccl_tile.cu).  Starts with a BucketHeader so that k_descend and cta_emit work
// on the region buckets unchanged.
constexpr int kMaxSubRegions = 2048;               // sub-regions (tiles of label[] held in shared memory) per call
constexpr int kFineStride = 8;                     // one fine counter per 32-byte sector (no false sharing in L2)
struct TileHeader {
    BucketHeader bh;
    unsigned long long overflow;                   // pairs in the overflow list
    unsigned long long pad;
    unsigned int fine[kMaxSubRegions * kFineStride];   // pairs filed under sub-region s: fine[s * kFineStride]
};

struct Tuning {                                    // ccl_set_option(); process-wide
    int64_t bucket_min_label_bytes = 96ll << 20;   // label[] beyond this cannot stay resident in the 126 MB L2
    int64_t bucket_min_bonds = 1 << 20;
    int32_t region_shift = 23;                     // 2^23 sites = 32 MiB of labels per region
    int32_t force_mode = -1;                       // -1: device-side probe decides; 0: direct; 1: bucketed
    int64_t bucket_capacity = 0;                   // pairs per region bucket; 0 = 4 M / regions + 4096
    int32_t two_pass = -1;                         // direct form of step (iii): 0 one pass (k_reduce), 1 hook + flatten +
                                                   // join (the paper's order), -1 by bonds per site (>= 2.5: two passes)
    int32_t tile_mode = 0;                         // tiled form (ccl_tile.cu): 0 off (default: measured slower, see
                                                   // profiles/r1_notes.md), -1 a device-side probe decides, 1 always
    int32_t sub_shift = -1;                        // 2^sub_shift sites per sub-region; -1 = from n_sites
    int64_t fine_capacity = 0;                     // pairs per sub-region bucket; 0 = 2 M / S + 8192
    int64_t tile_min_bonds = 1 << 18;
    int64_t small_max_sites = 1 << 15;             // one-CTA kernel for label arrays up to this many sites              // auto: calls with fewer bonds keep the direct kernel
};
Tuning& tuning();

// The library's own stream-ordered memory pool on the current device (created on first use, release threshold
// unlimited, so scratch freed by one call is reused by the next instead of going back to the driver).
int scratch_alloc(void** ptr, size_t bytes, cudaStream_t st);

// Enqueues probe + scatter + one descend launch per region.  *ws_out is a cudaMallocAsync allocation the caller
// frees (cudaFreeAsync) after the kernels that read *hdr_out have been enqueued.
// The region-bucketed form in two halves, so that its probe can ride in k_init (one block of k_init samples the bond
// list while the others write label[i] = i; as a kernel of its own the probe was 12 us of pure latency on the critical
// path of every call).  bucketed_begin allocates and clears the workspace and fills in the probe job;
// bucketed_launch enqueues the scatter and one descend launch per region.  *ws_out is a cudaMallocAsync allocation the
// caller frees (cudaFreeAsync) after the kernels that read the header have been enqueued.
struct ProbeJob {
    BucketHeader* hdr = nullptr;                   // NULL: no probe
    int64_t n_bonds = 0;
    const int32_t* src = nullptr;
    const int32_t* dst = nullptr;
    int shift = 0;
    int force_mode = -1;
};
struct BucketPlan {
    BucketHeader* hdr = nullptr;
    void* buckets = nullptr;
    unsigned long long cap = 0;
    int shift = 0, n_regions = 0;
};
int bucketed_begin(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst, cudaStream_t st,
                   BucketPlan* plan, ProbeJob* job, void** ws_out);
int bucketed_launch(const BucketPlan& plan, int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ,
                    int mask_kind, int32_t* labels, cudaStream_t st);

// Tiled form of steps (i)-(iii) for bond lists that are local in the site numbering (ccl_tile.cu).  *done says what
// was enqueued: kTiledNo nothing (call outside its range); kTiledFinal labels are final (one-CTA kernel); kTiledIfLocal
// a device-side probe decides -- *not_local points at a device flag that is 0 if the tiled kernels did steps (i)-(iii)
// and non-zero if they returned at once, so the caller enqueues the other forms gated on it; kTiledForced the tiled
// kernels ran unconditionally.  *ws_out (if set) is freed by the caller with cudaFreeAsync after the last kernel that
// reads the flag has been enqueued.
enum { kTiledNo = 0, kTiledFinal = 1, kTiledIfLocal = 2, kTiledForced = 3 };
int tiled_reduce(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ,
                 int mask_kind, int32_t* labels, cudaStream_t st, int* done, const int32_t** not_local, void** ws_out);

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
// them; raster-ordered lattice: only those on region borders): mode 1 = region-bucketed form, 0 = direct kernel.  Called
// by all threads of ONE block; gated = another form has done the work (mode 2: nothing to do).
__device__ __forceinline__ void probe_regions(const ProbeJob& job, bool gated)
{
    __shared__ int s_cross;
    if (gated) { if (threadIdx.x == 0) job.hdr->mode = 2; return; }
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
    if (threadIdx.x == 0)
        job.hdr->mode = job.force_mode >= 0 ? job.force_mode : ((4 * (int64_t)s_cross >= samples) ? 1 : 0);
}

// Label reads during root finding and flattening go through L1 (ld.global.ca).  L1 is not coherent, so a read may
// return an older value of label[x] -- which is still an ancestor of x, so every walk stays correct and only gets a
// little longer; every decision that matters is re-validated by the value an atomicMin
// returns.  What L1 buys: the top of a big cluster's tree is read by every walk through that cluster, and with
// L2-only loads (ld.relaxed.gpu, the first version) those reads all queue up at the one L2 slice that owns the
// sector (profiles/r1_notes.md).
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

}  // namespace ccl
