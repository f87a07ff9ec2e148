// ccl_emit.cuh -- CTA-wide append of (lo, hi) pairs to per-region buckets in global memory, shared by the
// region-bucketed form (ccl_bucket.cu) and the tiled form (ccl_tile.cu) of step (iii).  Product code.
#pragma once

#include "ccl_common.cuh"
#include "ccl_unionfind.cuh"

namespace ccl {

// Shared-memory scratch of the CTA-wide append: pairs are counted per target region, one global atomicAdd per
// region reserves the CTA's range in that bucket, and the pairs leave through a staging array so that consecutive
// threads write consecutive addresses.
template <int THREADS, int P>
struct EmitSmem {
    int cnt[kMaxRegions];
    int pref[kMaxRegions + 1];
    int lim[kMaxRegions];                 // staging indices below lim[r] fit into bucket r
    int2* gptr[kMaxRegions];              // bucket r's slot of staging index j is gptr[r] + j
    int2 stage[THREADS * P];
};

// What happens to a pair whose bucket is full.  JoinNow: Algorithm 1 on the spot (label[] must be valid everywhere).
struct JoinNow {
    int32_t* label;
    __device__ __forceinline__ void operator()(int2 pr) const { algorithm1(label, pr.x, pr.y); }
};
// Every thread hands in up to P pairs (lo[k] < 0 = none).  Must be called by all THREADS threads of the CTA.
template <int THREADS, int P, typename Overflow>
__device__ __forceinline__ void cta_emit(EmitSmem<THREADS, P>& sm, const int32_t (&lo)[P], const int32_t (&hi)[P],
                                         int shift, BucketHeader* hdr, int2* buckets, unsigned long long cap,
                                         const Overflow& overflow, uint64_t pol)
{
    const int tid = threadIdx.x;
    if (tid < kMaxRegions) sm.cnt[tid] = 0;
    __syncthreads();
    int rank[P];
#pragma unroll
    for (int k = 0; k < P; ++k) rank[k] = (lo[k] >= 0) ? atomicAdd(&sm.cnt[hi[k] >> shift], 1) : 0;
    __syncthreads();
    if (tid < 32) {
        const int c = sm.cnt[tid];
        int incl = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (tid >= o) incl += t;
        }
        const int pref = incl - c;
        sm.pref[tid] = pref;
        if (tid == 31) sm.pref[32] = incl;
        const unsigned long long base = c ? atomicAdd(&hdr->count[tid], (unsigned long long)c) : 0ull;
        const unsigned long long room = base < cap ? cap - base : 0ull;          // free slots left in bucket tid
        sm.lim[tid] = pref + (int)(room < (unsigned long long)c ? room : (unsigned long long)c);
        sm.gptr[tid] = buckets + (size_t)tid * cap + base - pref;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < P; ++k)
        if (lo[k] >= 0) sm.stage[sm.pref[hi[k] >> shift] + rank[k]] = make_int2(lo[k], hi[k]);
    __syncthreads();
    const int total = sm.pref[32];
    for (int j = tid; j < total; j += THREADS) {
        const int2 pr = sm.stage[j];
        const int r = pr.y >> shift;
        if (j < sm.lim[r]) st_stream_pair(sm.gptr[r] + j, pr, pol);
        else overflow(pr);                            // bucket full
    }
    __syncthreads();
}

}  // namespace ccl
