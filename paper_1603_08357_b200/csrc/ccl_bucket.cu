// ccl_bucket.cu -- step (iii) of PAPER.md:113 for label arrays that do not fit in L2: region-bucketed label reduction.
//
// Why: on B200 a random atomicMin into a 256 MiB label[] runs at ~31 G/s (every access is an HBM sector fetch plus a
// write-back), into an L2-resident 32-64 MiB slice at ~130 G/s (profiles/r1_ubench.txt).  So the site range is cut
// into regions whose labels fit in L2, every occupied bond is filed under the region of its HIGHER endpoint, and the
// regions are reduced one after the other from the highest down.  Within region r each pair (a, b), a < b, runs
// Algorithm 1's atomic loop directly on its own endpoints:
//
//       old = atomicMin(&label[b], a)      -- b lies in region r: L2 hit
//       old == b : b was a root, now hangs under a          -> done   (label_3 = label_1 in the paper's notation)
//       old == a : already linked                           -> done   (label_3 = label_2)
//       else     : the pair still to be joined is {a, old}  -> its higher site is < b
//
// The higher site of a pending pair only ever decreases, so a pair either stays in region r (the loop goes on in
// the same thread) or is re-filed under a LOWER region, which has not been reduced yet.  No root finding and no
// access outside the region are needed; after region 0 label[] is a forest with label[x] <= x, and step (iv)
// flattens it.  Measured chain lengths: 1.3-2.2 atomics per occupied bond on random regular graphs.
//
// A device-side probe decides whether to take this form at all: graphs whose bonds are local in the site numbering
// (raster-ordered lattices) keep the direct one-pass kernel of ccl_label.cu, whose gathers hit L2 anyway.
#include "ccl_common.cuh"
#include "ccl_unionfind.cuh"
#include "ccl_emit.cuh"

namespace ccl {

constexpr int kBThreads = 256;

// -------------------------------------------------------------------------------------------------- scatter
// One pass over the bond stream: occupied, non-loop bonds become (lo, hi) pairs filed under region(hi).
template <int MASK>
__global__ void __launch_bounds__(kBThreads)
k_scatter(int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
          const void* __restrict__ occ, int vec, int shift, BucketHeader* hdr, int2* buckets,
          unsigned long long cap, int32_t* label)
{
    constexpr int P = 8;
    __shared__ EmitSmem<kBThreads, P> sm;
    pdl_wait();
    if (hdr->mode != 1) return;
    const uint64_t pol = evict_first_policy();
    const int64_t tiles = (n_bonds + kBThreads * P - 1) / (kBThreads * P);
    for (int64_t tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
        const int64_t b0 = (tile * kBThreads + threadIdx.x) * P;
        int32_t lo[P], hi[P];
        int cnt = 0;
        if (b0 < n_bonds) cnt = (n_bonds - b0 >= P) ? P : (int)(n_bonds - b0);
        uint32_t m = (1u << cnt) - 1u;
        if (cnt > 0) {
            if (MASK == 2) {
                m &= ld_stream_u32(static_cast<const uint32_t*>(occ) + (b0 >> 5), pol) >> (b0 & 31);   // b0 % 8 == 0
            } else if (MASK == 1) {
                const uint8_t* o = static_cast<const uint8_t*>(occ) + b0;
                uint32_t mm = 0;
                for (int k = 0; k < cnt; ++k) mm |= (uint32_t)(ld_stream_u8(o + k, pol) != 0) << k;
                m &= mm;
            }
        }
        int32_t u[P], v[P];
        if (vec && cnt == P) {
            const int4 s0 = ld_stream_v4(src + b0, pol), s1 = ld_stream_v4(src + b0 + 4, pol);
            const int4 d0 = ld_stream_v4(dst + b0, pol), d1 = ld_stream_v4(dst + b0 + 4, pol);
            u[0] = s0.x; u[1] = s0.y; u[2] = s0.z; u[3] = s0.w; u[4] = s1.x; u[5] = s1.y; u[6] = s1.z; u[7] = s1.w;
            v[0] = d0.x; v[1] = d0.y; v[2] = d0.z; v[3] = d0.w; v[4] = d1.x; v[5] = d1.y; v[6] = d1.z; v[7] = d1.w;
        } else {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                u[k] = (k < cnt) ? ld_stream_s32(src + b0 + k, pol) : 0;
                v[k] = (k < cnt) ? ld_stream_s32(dst + b0 + k, pol) : 0;
            }
        }
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const bool on = ((m >> k) & 1u) && u[k] != v[k];
            lo[k] = on ? min(u[k], v[k]) : -1;
            hi[k] = max(u[k], v[k]);
        }
        cta_emit<kBThreads, P>(sm, lo, hi, shift, hdr, buckets, cap, JoinNow{label}, pol);
    }
}

// -------------------------------------------------------------------------------------------------- descend
// Reduce region r: all label[] traffic of this launch falls into [r << shift, (r+1) << shift).
template <int P>
__global__ void __launch_bounds__(kBThreads)
k_descend(int r, int shift, BucketHeader* hdr, int2* buckets, unsigned long long cap, int32_t* label)
{
    __shared__ EmitSmem<kBThreads, P> sm;
    pdl_wait();
    if (hdr->mode != 1) return;
    const uint64_t pol = evict_first_policy();
    unsigned long long n = hdr->count[r];
    if (n > cap) n = cap;
    const int2* bucket = buckets + (size_t)r * cap;
    const long long tiles = (long long)((n + kBThreads * P - 1) / (kBThreads * P));
    for (long long tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
        const unsigned long long i0 = ((unsigned long long)tile * kBThreads + threadIdx.x) * P;
        int32_t a[P], b[P], old[P];
        if (i0 + P <= n) {
#pragma unroll
            for (int q = 0; q < P / 2; ++q) {
                const int4 v = ld_stream_v4(reinterpret_cast<const int32_t*>(bucket + i0 + 2 * q), pol);
                a[2 * q] = v.x; b[2 * q] = v.y; a[2 * q + 1] = v.z; b[2 * q + 1] = v.w;
            }
        } else {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                a[k] = -1; b[k] = 0;
                if (i0 + k < n) {
                    a[k] = ld_stream_s32(reinterpret_cast<const int32_t*>(bucket + i0 + k), pol);
                    b[k] = ld_stream_s32(reinterpret_cast<const int32_t*>(bucket + i0 + k) + 1, pol);
                }
            }
        }
        // first atomics of the four pairs in flight together
#pragma unroll
        for (int k = 0; k < P; ++k) old[k] = (a[k] >= 0) ? atomicMin(label + b[k], a[k]) : a[k];
        // Continuation: the pairs whose first atomic found b linked already.  The P chains of a thread advance together,
        // one link per round with their loads (and then their atomics) in flight at the same time; walked one after the
        // other they made the last region, where every chain of the giant cluster ends, pure memory latency (0.42 ms
        // at p = 0.45 on config 5).
        bool act[P], pend[P];
#pragma unroll
        for (int k = 0; k < P; ++k) { act[k] = a[k] >= 0 && old[k] != b[k] && old[k] != a[k]; pend[k] = false; }
        for (;;) {
            int32_t v[P];
            bool any = false;
#pragma unroll
            for (int k = 0; k < P; ++k) {
                v[k] = 0;
                if (act[k]) {
                    const int32_t na = min(a[k], old[k]), nb = max(a[k], old[k]);      // the pair left is {a, old}
                    a[k] = na; b[k] = nb;
                    if ((nb >> shift) != r) { pend[k] = true; act[k] = false; }         // leaves the region: re-file it lower down
                    // Continuation steps mostly land on sites that are linked already, and the lowest sites of a big
                    // cluster are hit by millions of them: look before writing.  A (possibly stale, L1-cached) value
                    // v <= a means the atomic would not write, and {v, a} is the pair that is left (or nothing, if
                    // v == a): whoever replaced v later took over the duty of joining v to its successor.
                    else v[k] = label[nb];
                }
            }
#pragma unroll
            for (int k = 0; k < P; ++k)
                if (act[k]) old[k] = (v[k] > a[k]) ? atomicMin(label + b[k], a[k]) : v[k];
#pragma unroll
            for (int k = 0; k < P; ++k)
                if (act[k]) { act[k] = old[k] != b[k] && old[k] != a[k]; any |= act[k]; }
            if (!any) break;
        }
#pragma unroll
        for (int k = 0; k < P; ++k) if (!pend[k]) a[k] = -1;
        cta_emit<kBThreads, P>(sm, a, b, shift, hdr, buckets, cap, JoinNow{label}, pol);
    }
    pdl_go();                                              // this CTA is done: the next launch may take its place
}

// ------------------------------------------------------------------------------------------------- host side
int bucketed_begin(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst, cudaStream_t st,
                   BucketPlan* plan, ProbeJob* job, void** ws_out)
{
    // region size: 2^23 sites (32 MiB of labels) unless that would need more than kMaxRegions regions
    int shift = tuning().region_shift;
    while (((n_sites - 1) >> shift) + 1 > kMaxRegions) ++shift;
    const int n_regions = (int)(((n_sites - 1) >> shift) + 1);
    unsigned long long cap = (unsigned long long)((4 * n_bonds) / n_regions + 4096);
    if (tuning().bucket_capacity > 0) cap = (unsigned long long)tuning().bucket_capacity;
    cap = (cap + 7ull) & ~7ull;                                   // keeps every bucket 64-byte aligned
    const size_t hdr_bytes = (sizeof(BucketHeader) + 255) & ~(size_t)255;
    const size_t bytes = hdr_bytes + (size_t)n_regions * cap * sizeof(int2);
    void* ws = nullptr;
    { const int rc = scratch_alloc(&ws, bytes, st); if (rc != CCL_OK) return rc; }
    *ws_out = ws;
    plan->hdr = static_cast<BucketHeader*>(ws);
    plan->buckets = static_cast<char*>(ws) + hdr_bytes;
    plan->cap = cap;
    plan->shift = shift;
    plan->n_regions = n_regions;
    job->hdr = plan->hdr;
    job->n_bonds = n_bonds;
    job->src = src;
    job->dst = dst;
    job->shift = shift;
    job->force_mode = tuning().force_mode;
    CCL_CUDA_TRY(cudaMemsetAsync(plan->hdr, 0, sizeof(BucketHeader), st));
    return CCL_OK;
}

int bucketed_launch(const BucketPlan& plan, int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ,
                    int mask_kind, int32_t* labels, cudaStream_t st)
{
    BucketHeader* hdr = plan.hdr;
    int2* buckets = static_cast<int2*>(plan.buckets);
    const unsigned long long cap = plan.cap;
    const int shift = plan.shift;
    const uintptr_t al = reinterpret_cast<uintptr_t>(src) | reinterpret_cast<uintptr_t>(dst);
    const int vec = (al & 15) == 0;
    const int grid = kSMs * 6;
    if (occ == nullptr)
        CCL_CUDA_TRY(launch_pdl(k_scatter<0>, (unsigned)grid, (unsigned)kBThreads, st, n_bonds, src, dst, (const void*)nullptr, vec, shift, hdr, buckets, cap, labels));
    else if (mask_kind == 1)
        CCL_CUDA_TRY(launch_pdl(k_scatter<1>, (unsigned)grid, (unsigned)kBThreads, st, n_bonds, src, dst, occ, vec, shift, hdr, buckets, cap, labels));
    else
        CCL_CUDA_TRY(launch_pdl(k_scatter<2>, (unsigned)grid, (unsigned)kBThreads, st, n_bonds, src, dst, occ, vec, shift, hdr, buckets, cap, labels));
    count_launch();
    for (int r = plan.n_regions - 1; r >= 0; --r) {
        CCL_CUDA_TRY(launch_pdl(k_descend<4>, (unsigned)grid, (unsigned)kBThreads, st, r, shift, hdr, buckets, cap, labels));
        count_launch();
    }
    return CCL_OK;
}

}  // namespace ccl
