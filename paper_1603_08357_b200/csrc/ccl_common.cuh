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

// ---- region-bucketed label reduction (ccl_bucket.cu) -----------------------------------------------------
constexpr int kMaxRegions = 32;

struct BucketHeader {                              // lives in device memory at the head of the call's workspace
    int32_t mode;                                  // written by k_probe: 0 = direct one-pass kernel, 1 = bucketed
    int32_t pad;
    unsigned long long count[kMaxRegions];         // pairs filed under each region (may exceed the capacity: the
                                                   // excess was joined on the spot by the general algorithm)
};

struct Tuning {                                    // ccl_set_option(); process-wide
    int64_t bucket_min_label_bytes = 96ll << 20;   // label[] beyond this cannot stay resident in the 126 MB L2
    int64_t bucket_min_bonds = 1 << 20;
    int32_t region_shift = 23;                     // 2^23 sites = 32 MiB of labels per region
    int32_t force_mode = -1;                       // -1: device-side probe decides; 0: direct; 1: bucketed
    int64_t bucket_capacity = 0;                   // pairs per region bucket; 0 = 4 M / regions + 4096
};
Tuning& tuning();

// The library's own stream-ordered memory pool on the current device (created on first use, release threshold
// unlimited, so scratch freed by one call is reused by the next instead of going back to the driver).
int scratch_alloc(void** ptr, size_t bytes, cudaStream_t st);

// Enqueues probe + scatter + one descend launch per region.  *ws_out is a cudaMallocAsync allocation the caller
// frees (cudaFreeAsync) after the kernels that read *hdr_out have been enqueued.
int bucketed_reduce(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ,
                    int mask_kind, int32_t* labels, cudaStream_t st, BucketHeader** hdr_out, void** ws_out);

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
