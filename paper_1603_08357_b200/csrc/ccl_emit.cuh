// ccl_emit.cuh -- CTA-wide append of (lo, hi) pairs to the per-region buckets of the region-bucketed form of step (iii)
// (ccl_bucket.cu).  Product code.
//
// A bucket is a dense logical array of pairs, cut into chunks of 2^cshift pairs that are drawn on demand from one pool
// shared by all regions (table[r * stride + k] = 1 + pool index of the k-th chunk of bucket r), so the workspace is
// sized by the number of pairs that exist, not by the worst case per region.  A CTA reserves its range of a bucket
// with one atomicAdd, as it would in a flat array.  The CTA whose range covers the first slot of a chunk draws that
// chunk from the pool and publishes it; CTAs that reserved later slots of the same chunk wait for the table entry
// (the publisher is past its reservation, i.e. running, and only ever waits for chunks reserved before its own, so the
// wait ends).  Chunks are large (the pool holds a few dozen), so a CTA almost always finds the entry it needs in the
// copy it keeps in shared memory and the table is read only when a bucket moves on to its next chunk.  When the pool
// is dry the entry becomes kChunkInvalid, the pairs are dropped and hdr->overflow is set: the direct kernel then
// processes the whole bond list behind the bucketed kernels (ccl_label.cu), which is correct on top of any partial
// forest.
#pragma once

#include "ccl_common.cuh"

namespace ccl {

struct BucketRef {                         // what the kernels need of a BucketPlan
    BucketHeader* hdr;
    unsigned int* table;
    int2* pool;
    unsigned int n_chunks, stride;
    int shift;                             // region = site >> shift
    int cshift;                            // chunk = 2^cshift pairs
};

constexpr unsigned int kChunkInvalid = 0xFFFFFFFFu;    // table entry of a chunk the pool could not supply

// Shared-memory scratch of the CTA-wide append: pairs are counted per target region, one global atomicAdd per region
// reserves the CTA's range in that bucket, and the pairs leave through a staging array so that consecutive threads
// write consecutive addresses.  known_ci / known_e persist over the tiles a CTA works through.
struct EmitSmem {
    int cnt[kMaxRegions];
    int pref[kMaxRegions + 1];
    int first[kMaxRegions];               // the first `first[r]` pairs of this round go to ptr0[r], the rest to ptr1[r]
    int2* ptr0[kMaxRegions];              // NULL: dropped (pool dry)
    int2* ptr1[kMaxRegions];
    unsigned long long known_ci[kMaxRegions];
    unsigned int known_e[kMaxRegions];
};

__device__ __forceinline__ void emit_begin(EmitSmem& sm)
{
    if (threadIdx.x < kMaxRegions) { sm.known_ci[threadIdx.x] = ~0ull; sm.cnt[threadIdx.x] = 0; }
    __syncthreads();
}

__device__ __forceinline__ unsigned int chunk_entry(const BucketRef& bk, int r, unsigned long long ci, bool owner)
{
    if (ci >= bk.stride) {                                 // beyond anything the pool could ever supply
        if (owner) bk.hdr->overflow = 1;
        return kChunkInvalid;
    }
    unsigned int* slot = bk.table + (size_t)r * bk.stride + ci;
    if (owner) {
        const unsigned int phys = atomicAdd(&bk.hdr->next_chunk, 1u);
        const unsigned int e = phys < bk.n_chunks ? phys + 1u : kChunkInvalid;
        if (e == kChunkInvalid) bk.hdr->overflow = 1;
        st_release_u32(slot, e);
        return e;
    }
    unsigned int e;
    while ((e = ld_acquire_u32(slot)) == 0u) { }
    return e;
}

__device__ __forceinline__ int2* chunk_ptr(const BucketRef& bk, unsigned int e)
{
    return e == kChunkInvalid ? nullptr : bk.pool + ((size_t)(e - 1) << bk.cshift);
}

// A round of the append, after the caller has ranked its pairs per region with atomicAdd(&sm.cnt[r], 1) and a
// __syncthreads() (sm.cnt must be zero before the ranking starts; emit_scan leaves it zero again):
//   emit_scan      warp 0: prefix over the regions (sm.pref); returns the lane's own count
//   emit_reserve   warp 0, lane r: one global atomicAdd on bucket r -- the value comes back ~1 us later
//   (caller)       __syncthreads(); stage[sm.pref[r] + rank] = pair    -- needs sm.pref only
//   emit_place     warp 0, lane r: where the reserved range lives (chunk bookkeeping) -> sm.first / ptr0 / ptr1
//   (caller)       __syncthreads()
//   emit_copy_out  consecutive threads write consecutive addresses of each bucket
__device__ __forceinline__ int emit_scan(EmitSmem& sm)
{
    const int tid = threadIdx.x;                           // < 32
    const int c = sm.cnt[tid];
    int incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (tid >= o) incl += t;
    }
    sm.pref[tid] = incl - c;
    if (tid == 31) sm.pref[32] = incl;
    sm.cnt[tid] = 0;
    return c;
}

__device__ __forceinline__ unsigned long long emit_reserve(const BucketRef& bk, int c)
{
    return c ? atomicAdd(&bk.hdr->count[threadIdx.x], (unsigned long long)c) : 0ull;
}

__device__ __forceinline__ void emit_place(EmitSmem& sm, const BucketRef& bk, int c, unsigned long long base)
{
    const int tid = threadIdx.x;                           // < 32
    if (c == 0) return;
    const unsigned long long c0 = base >> bk.cshift, c1 = (base + c - 1) >> bk.cshift;
    const unsigned long long off = base & ((1ull << bk.cshift) - 1);
    const unsigned int e0 = (c0 == sm.known_ci[tid]) ? sm.known_e[tid] : chunk_entry(bk, tid, c0, off == 0);
    unsigned int e1 = e0;
    int first = c;
    if (c1 != c0) {                                        // the run crosses into a chunk whose first slot it holds
        e1 = chunk_entry(bk, tid, c1, true);
        first = (int)((1ull << bk.cshift) - off);
    }
    sm.known_ci[tid] = c1; sm.known_e[tid] = e1;
    int2* p0 = chunk_ptr(bk, e0);
    sm.first[tid] = first;
    sm.ptr0[tid] = p0 ? p0 + off : nullptr;
    sm.ptr1[tid] = chunk_ptr(bk, e1);
}

template <int THREADS>
__device__ __forceinline__ void emit_copy_out(EmitSmem& sm, const int2* stage, const BucketRef& bk, uint64_t pol)
{
    const int total = sm.pref[32];
    for (int j = threadIdx.x; j < total; j += THREADS) {
        const int2 pr = stage[j];
        const int r = pr.y >> bk.shift;
        const int k = j - sm.pref[r], f = sm.first[r];
        int2* dst = (k < f) ? sm.ptr0[r] : sm.ptr1[r];
        if (dst != nullptr) st_stream_pair(dst + (k < f ? k : k - f), pr, pol);      // NULL: pool dry, hdr->overflow is set
    }
}

// Every thread hands in up to P pairs (lo[k] < 0 = none); stage holds THREADS * P pairs (<= 2^cshift).  Must be called
// by all THREADS threads of the CTA.
template <int THREADS, int P>
__device__ __forceinline__ void cta_emit(EmitSmem& sm, int2* stage, const int32_t (&lo)[P], const int32_t (&hi)[P],
                                         const BucketRef& bk, uint64_t pol)
{
    int rank[P];
#pragma unroll
    for (int k = 0; k < P; ++k) rank[k] = (lo[k] >= 0) ? atomicAdd(&sm.cnt[hi[k] >> bk.shift], 1) : 0;
    __syncthreads();
    int c = 0;
    unsigned long long base = 0;
    if (threadIdx.x < 32) { c = emit_scan(sm); base = emit_reserve(bk, c); }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < P; ++k)
        if (lo[k] >= 0) stage[sm.pref[hi[k] >> bk.shift] + rank[k]] = make_int2(lo[k], hi[k]);
    if (threadIdx.x < 32) emit_place(sm, bk, c, base);
    __syncthreads();
    emit_copy_out<THREADS>(sm, stage, bk, pol);
    __syncthreads();
}

// Address of the tile of pairs that starts at logical index i0 of bucket r (tiles never straddle a chunk), or NULL if
// that part of the bucket was dropped.
__device__ __forceinline__ const int2* bucket_tile(const BucketRef& bk, int r, unsigned long long i0)
{
    const unsigned long long ci = i0 >> bk.cshift;
    if (ci >= bk.stride) return nullptr;
    const unsigned int e = bk.table[(size_t)r * bk.stride + ci];
    if (e == 0u || e == kChunkInvalid) return nullptr;
    return bk.pool + ((size_t)(e - 1) << bk.cshift) + (size_t)(i0 & ((1ull << bk.cshift) - 1));
}

}  // namespace ccl
