// ccl_bucket.cu -- step (iii) of PAPER.md:113 for label arrays that do not fit in L2: region-bucketed label reduction.
//
// Why: on B200 a random atomicMin into a 256 MiB label[] runs at ~31 G/s (every access is an HBM sector fetch plus a
// write-back), into an L2-resident 32-64 MiB slice at ~130 G/s (profiles/r1_ubench.md).  So the site range is cut
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
// flattens it.  This orders the WORK by region; no region is labeled on its own and nothing is merged across region
// borders afterwards (reading R14).
//
// Step (i) rides along: label[] of region r is written (label[i] = i) by the kernel that runs just before
// k_descend(r), so the lines are still in L2 when the first atomic arrives, and the write to HBM and the fetch back
// that a separate initialization pass costs disappear.
#include <mutex>

#include "ccl_common.cuh"
#include "ccl_unionfind.cuh"
#include "ccl_emit.cuh"

namespace ccl {

constexpr int kBThreads = 256;
constexpr int kScatterP = 8;                               // bonds per thread and tile in k_scatter
constexpr int kDescendP = 4;                               // pairs per thread and tile in k_descend

// label[i] = i for the regions that are touched before any k_descend has run: [lo, n_sites).
__global__ void __launch_bounds__(kBThreads)
k_init_top(int64_t lo, int64_t n_sites, int32_t* __restrict__ label)
{
    init_range(label, lo, n_sites, (int64_t)blockIdx.x * kBThreads + threadIdx.x, (int64_t)gridDim.x * kBThreads);
}

// -------------------------------------------------------------------------------------------------- scatter
// One pass over the bond stream: occupied, non-loop bonds become (lo, hi) pairs filed under region(hi).
//
// k_scatter: the general kernel (any alignment, any length), 8 bonds per thread in registers.
template <int MASK>
__global__ void __launch_bounds__(kBThreads)
k_scatter(int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
          const void* __restrict__ occ, int vec, BucketRef bk, int gated)
{
    constexpr int P = kScatterP;
    __shared__ EmitSmem sm;
    __shared__ int2 stage[kBThreads * P];
    pdl_wait();
    if (gated && bk.hdr->mode != 1) return;
    const uint64_t pol = evict_first_policy();
    emit_begin(sm);
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
        cta_emit<kBThreads, P>(sm, stage, lo, hi, bk, pol);
    }
    pdl_go();
}

// k_scatter_tiles: whole tiles of 2048 bonds of 16-byte aligned input.  The kernel above issues ~70 instructions per
// bond slot and most of them are predicated off (three quarters of the slots hold unoccupied bonds at p = 0.25).  Here a
// tile -- src, dst and their mask bits -- is copied to shared memory by the bulk-copy engine (cp.async.bulk, completion
// on an mbarrier; two tiles in flight per CTA, so the HBM stream never waits for the arithmetic); every warp compacts
// the occupied bonds of its 256 with ballots into an index list and only then forms pairs, with all lanes busy; the
// pairs are ranked per region, sorted through the staging array (which reuses the tile's own input buffer) and
// appended to the buckets as in cta_emit.
constexpr int kTileBonds = 2048;
template <int MASK>
struct ScatterTile {
    int32_t src[kTileBonds];
    int32_t dst[kTileBonds];               // src + dst are reused as the staging array int2[kTileBonds] of the append
    uint32_t mask[MASK == 1 ? kTileBonds / 4 : kTileBonds / 32];      // MASK 1: 2048 bytes; MASK 2: 64 words
};
template <int MASK>
struct ScatterSmem {
    ScatterTile<MASK> in[2];
    int2 pairs[kTileBonds];                // warp w's compacted pairs at [256 w, 256 w + n_w)
    uint16_t slot[kTileBonds];             // rank of the pair within its region; the upper half of warp w's 512 bytes
                                           // first holds the warp's index list (one byte per occupied bond)
    EmitSmem emit;
    unsigned long long mbar[2];
};

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void bulk_load(void* dst_smem, const void* src_gmem, uint32_t bytes, unsigned long long* mbar,
                                          uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(smem_addr(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_addr(mbar)), "l"(pol)
                 : "memory");
}

template <int MASK>
__device__ __forceinline__ void tile_fetch(ScatterTile<MASK>& t, unsigned long long* mbar, int64_t tile,
                                           const int32_t* src, const int32_t* dst, const void* occ, uint64_t pol)
{
    constexpr uint32_t kMaskBytes = MASK == 2 ? kTileBonds / 8 : MASK == 1 ? kTileBonds : 0;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(mbar)),
                 "r"((uint32_t)(2 * kTileBonds * sizeof(int32_t)) + kMaskBytes)
                 : "memory");
    bulk_load(t.src, src + tile * kTileBonds, kTileBonds * sizeof(int32_t), mbar, pol);
    bulk_load(t.dst, dst + tile * kTileBonds, kTileBonds * sizeof(int32_t), mbar, pol);
    if (MASK != 0) bulk_load(t.mask, static_cast<const char*>(occ) + tile * kMaskBytes, kMaskBytes, mbar, pol);
}

__device__ __forceinline__ void mbar_wait(unsigned long long* mbar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        ::"r"(smem_addr(mbar)), "r"(parity)
        : "memory");
}

template <int MASK>
__global__ void __launch_bounds__(kBThreads, 4)
k_scatter_tiles(int64_t n_tiles, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
                const void* __restrict__ occ, BucketRef bk, int gated)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    ScatterSmem<MASK>& sm = *reinterpret_cast<ScatterSmem<MASK>*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_addr(&sm.mbar[0])));
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_addr(&sm.mbar[1])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    pdl_wait();
    if (gated && bk.hdr->mode != 1) return;
    const uint64_t pol = evict_first_policy();
    emit_begin(sm.emit);                                   // (barrier: the mbarriers are initialised for everybody)
    const int64_t stride = gridDim.x;
    if (tid == 0) {
        if ((int64_t)blockIdx.x < n_tiles) tile_fetch<MASK>(sm.in[0], &sm.mbar[0], blockIdx.x, src, dst, occ, pol);
        if ((int64_t)blockIdx.x + stride < n_tiles) tile_fetch<MASK>(sm.in[1], &sm.mbar[1], blockIdx.x + stride, src, dst, occ, pol);
    }
    int2* my_pairs = sm.pairs + warp * 256;
    uint16_t* my_slot = sm.slot + warp * 256;
    uint8_t* my_idx = reinterpret_cast<uint8_t*>(my_slot) + 256;       // entry j is read before slot j' >= 128 overwrites it
    int it = 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += stride, ++it) {
        const int cur = it & 1;
        ScatterTile<MASK>& in = sm.in[cur];
        mbar_wait(&sm.mbar[cur], (it >> 1) & 1);
        // ---- the warp's occupied bonds, compacted
        int n = 0;
#pragma unroll
        for (int row = 0; row < 8; ++row) {
            bool on = true;
            if (MASK == 2) on = (in.mask[warp * 8 + row] >> lane) & 1u;
            else if (MASK == 1) on = reinterpret_cast<const uint8_t*>(in.mask)[warp * 256 + row * 32 + lane] != 0;
            const unsigned bal = __ballot_sync(0xffffffffu, on);
            if (on) my_idx[n + __popc(bal & ((1u << lane) - 1u))] = (uint8_t)(row * 32 + lane);
            n += __popc(bal);
        }
        __syncwarp();
        // ---- pairs: (lo, hi) and their rank within the target region
        for (int j0 = 0; j0 < n; j0 += 32) {
            const int j = j0 + lane;
            int32_t lo = -1, hi = 0;
            if (j < n) {
                const int b = warp * 256 + my_idx[j];
                const int32_t u = in.src[b], v = in.dst[b];
                hi = max(u, v);
                if (u != v) lo = min(u, v);
            }
            __syncwarp();                                  // every lane has read its index byte
            if (j < n) {
                my_pairs[j] = make_int2(lo, hi);
                if (lo >= 0) my_slot[j] = (uint16_t)atomicAdd(&sm.emit.cnt[hi >> bk.shift], 1);
            }
        }
        __syncthreads();                                   // all pairs ranked; nobody reads in.src / in.dst any more
        int c = 0;
        unsigned long long base = 0;
        if (tid < 32) { c = emit_scan(sm.emit); base = emit_reserve(bk, c); }
        __syncthreads();
        int2* stage = reinterpret_cast<int2*>(in.src);
        for (int j = lane; j < n; j += 32) {
            const int2 pr = my_pairs[j];
            if (pr.x >= 0) stage[sm.emit.pref[pr.y >> bk.shift] + my_slot[j]] = pr;
        }
        if (tid < 32) emit_place(sm.emit, bk, c, base);
        __syncthreads();
        emit_copy_out<kBThreads>(sm.emit, stage, bk, pol);
        __syncthreads();                                   // the buffer is free again
        if (tid == 0 && tile + 2 * stride < n_tiles) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic-proxy writes (staging) before the bulk copy
            tile_fetch<MASK>(in, &sm.mbar[cur], tile + 2 * stride, src, dst, occ, pol);
        }
    }
    pdl_go();
}

// -------------------------------------------------------------------------------------------------- descend
// Reduce region r: all label[] traffic of this launch falls into [r << shift, (r+1) << shift).  init_lo < init_hi: the
// labels of the region that comes next are written on the way out (step (i) for that region).
__global__ void __launch_bounds__(kBThreads, 8)
k_descend(int r, BucketRef bk, int gated, int64_t init_lo, int64_t init_hi, int32_t* label)
{
    constexpr int P = kDescendP;
    __shared__ EmitSmem sm;
    __shared__ int2 stage[kBThreads * P];
    pdl_wait();
    if (gated && bk.hdr->mode != 1) return;
    const uint64_t pol = evict_first_policy();
    const int shift = bk.shift;
    emit_begin(sm);
    const unsigned long long n = bk.hdr->count[r];
    const long long tiles = (long long)((n + kBThreads * P - 1) / (kBThreads * P));
    for (long long tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
        const unsigned long long t0 = (unsigned long long)tile * kBThreads * P;
        const int2* base = bucket_tile(bk, r, t0);
        if (base == nullptr) continue;                                 // dropped (pool dry): CTA-uniform
        const unsigned long long i0 = t0 + (unsigned long long)threadIdx.x * P;
        const int2* mine = base + threadIdx.x * P;
        int32_t a[P], b[P], old[P];
        if (i0 + P <= n) {
#pragma unroll
            for (int q = 0; q < P / 2; ++q) {
                const int4 v = ld_stream_v4(reinterpret_cast<const int32_t*>(mine + 2 * q), pol);
                a[2 * q] = v.x; b[2 * q] = v.y; a[2 * q + 1] = v.z; b[2 * q + 1] = v.w;
            }
        } else {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                a[k] = -1; b[k] = 0;
                if (i0 + k < n) {
                    a[k] = ld_stream_s32(reinterpret_cast<const int32_t*>(mine + k), pol);
                    b[k] = ld_stream_s32(reinterpret_cast<const int32_t*>(mine + k) + 1, pol);
                }
            }
        }
        // first atomics of the P pairs in flight together
#pragma unroll
        for (int k = 0; k < P; ++k) old[k] = (a[k] >= 0) ? atomicMin(label + b[k], a[k]) : a[k];
        // Continuation: the pairs whose first atomic found b linked already.  The P chains of a thread advance together,
        // one link per round with their loads (and then their atomics) in flight at the same time; walked one after the
        // other they made the last region, where every chain of the giant cluster ends, pure memory latency.
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
        bool pending = false;
#pragma unroll
        for (int k = 0; k < P; ++k) { if (!pend[k]) a[k] = -1; pending |= pend[k]; }
        if (__syncthreads_or(pending)) cta_emit<kBThreads, P>(sm, stage, a, b, bk, pol);
    }
    if (init_lo < init_hi)
        init_range(label, init_lo, init_hi, (int64_t)blockIdx.x * kBThreads + threadIdx.x, (int64_t)gridDim.x * kBThreads);
    pdl_go();                                              // this CTA is done: the next launch may take its place
}

// ------------------------------------------------------------------------------------------------- host side
// Persistent grids: as many CTAs as are resident at once (every CTA works through the same number of tiles, so a CTA
// that had to wait for a free slot would finish alone).
template <typename K>
static int resident_grid(K kernel, size_t smem)
{
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kBThreads, smem) != cudaSuccess) per_sm = 0;
    cudaGetLastError();
    if (per_sm < 1) per_sm = 1;
    return per_sm * sm_count();
}

// The grids -- and the opt-in to more than 48 KB of dynamic shared memory that k_scatter_tiles needs -- belong to a
// device, not to the process: one entry per device, filled under a lock by the first eligible call on that device.
struct BucketGrids { bool ready = false; int scatter = 0, tiles[3] = {0, 0, 0}, descend = 0; };
static std::mutex g_grids_mutex;
static BucketGrids g_grids[64];

template <int MASK>
static int tiles_grid()
{
    // 0 = the opt-in failed on this device: the register kernel (k_scatter) takes the whole bond list instead
    if (cudaFuncSetAttribute(k_scatter_tiles<MASK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ScatterSmem<MASK>)) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return resident_grid(k_scatter_tiles<MASK>, sizeof(ScatterSmem<MASK>));
}

static int bucket_grids(BucketGrids* out)
{
    int dev = 0;
    CCL_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) { set_error("device index %d out of range", dev); return CCL_UNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_grids_mutex);
    BucketGrids& g = g_grids[dev];
    if (!g.ready) {
        g.scatter = resident_grid(k_scatter<2>, 0);
        g.tiles[0] = tiles_grid<0>();
        g.tiles[1] = tiles_grid<1>();
        g.tiles[2] = tiles_grid<2>();
        g.descend = resident_grid(k_descend, 0);
        g.ready = true;
    }
    *out = g;
    return CCL_OK;
}

// region size: 2^23 sites (32 MiB of labels) unless that would need more than kMaxRegions regions
int bucket_region_shift(int64_t n_sites, const Tuning& t)
{
    int shift = t.region_shift;
    while (((n_sites - 1) >> shift) + 1 > kMaxRegions) ++shift;
    return shift;
}

int bucketed_begin(int64_t n_sites, int64_t n_bonds, const Tuning& t, int pool_doublings, cudaStream_t st, BucketPlan* plan,
                   void** ws_out)
{
    const int shift = bucket_region_shift(n_sites, t);
    const int n_regions = (int)(((n_sites - 1) >> shift) + 1);
    // Pool: room for 1.25 pairs per bond (every occupied bond, and what the descent re-files) in chunks of about 1/64 of
    // that, plus the chunk every region leaves partly filled.
    int cshift = kMinChunkShift;
    while (cshift < kMaxChunkShift && (n_bonds >> (cshift + 6)) > 0) ++cshift;
    unsigned long long n_chunks;
    if (t.bucket_capacity > 0) n_chunks = (((unsigned long long)t.bucket_capacity - 1) >> cshift) + 1;
    else n_chunks = ((((unsigned long long)n_bonds * 5 / 4) << (pool_doublings < 0 ? 0 : pool_doublings > 3 ? 3 : pool_doublings)) >> cshift) +
                    (unsigned long long)n_regions + 2;
    if (n_chunks > 0x7FFFFFF0ull) n_chunks = 0x7FFFFFF0ull;
    const size_t hdr_bytes = (sizeof(BucketHeader) + 255) & ~(size_t)255;
    const size_t table_bytes = (((size_t)n_regions * n_chunks * sizeof(unsigned int)) + 255) & ~(size_t)255;
    const size_t bytes = hdr_bytes + table_bytes + ((size_t)n_chunks << cshift) * sizeof(int2);
    void* ws = nullptr;
    { const int rc = scratch_alloc(&ws, bytes, st); if (rc != CCL_OK) return rc; }
    *ws_out = ws;
    plan->hdr = static_cast<BucketHeader*>(ws);
    plan->table = reinterpret_cast<unsigned int*>(static_cast<char*>(ws) + hdr_bytes);
    plan->pool = reinterpret_cast<int2*>(static_cast<char*>(ws) + hdr_bytes + table_bytes);
    plan->n_chunks = (unsigned int)n_chunks;
    plan->stride = (unsigned int)n_chunks;
    plan->shift = shift;
    plan->cshift = cshift;
    plan->n_regions = n_regions;
    plan->scatter_tiles = t.scatter_tiles;
    plan->l2_persist = t.l2_persist;
    CCL_CUDA_TRY(cudaMemsetAsync(ws, 0, hdr_bytes + table_bytes, st));
    return CCL_OK;
}

int bucketed_launch(const BucketPlan& plan, int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                    const void* occ, int mask_kind, int32_t* labels, cudaStream_t st)
{
    BucketRef bk;
    bk.hdr = plan.hdr; bk.table = plan.table; bk.pool = plan.pool;
    bk.n_chunks = plan.n_chunks; bk.stride = plan.stride; bk.shift = plan.shift; bk.cshift = plan.cshift;
    const int R = plan.n_regions, shift = plan.shift;
    const uintptr_t al = reinterpret_cast<uintptr_t>(src) | reinterpret_cast<uintptr_t>(dst);
    const int vec = (al & 15) == 0;
    BucketGrids grids;
    { const int rc = bucket_grids(&grids); if (rc != CCL_OK) return rc; }
    const int mk = occ == nullptr ? 0 : mask_kind;
    // the top region must hold label[i] = i before the first k_descend touches it; every k_descend writes the labels
    // of the region that comes next
    if (plan.lazy_init) {
        const int64_t lo = (int64_t)(R - 1) << shift;
        int64_t blocks = ((n_sites - lo + 3) / 4 + kBThreads - 1) / kBThreads;
        if (blocks > (int64_t)sm_count() * 16) blocks = (int64_t)sm_count() * 16;
        k_init_top<<<(unsigned)blocks, kBThreads, 0, st>>>(lo, n_sites, labels);
        CCL_CHECK_LAUNCH("k_init_top");
    }
    const int gated = plan.gated;
    // whole tiles of 16-byte aligned input go through the bulk-copy kernel, the rest (a tail, or everything) through
    // the register kernel
    int64_t done = 0;
    const bool mask_ok = occ == nullptr || (reinterpret_cast<uintptr_t>(occ) & 15) == 0;
    if (vec && mask_ok && plan.scatter_tiles && n_bonds >= kTileBonds && grids.tiles[mk] > 0) {
        const int64_t n_tiles = n_bonds / kTileBonds;
        int tg = grids.tiles[mk];
        if (tg > n_tiles) tg = (int)n_tiles;
        if (mk == 0) CCL_CUDA_TRY(launch_pdl_smem(k_scatter_tiles<0>, (unsigned)tg, (unsigned)kBThreads, sizeof(ScatterSmem<0>), st, n_tiles, src, dst, (const void*)nullptr, bk, gated));
        else if (mk == 1) CCL_CUDA_TRY(launch_pdl_smem(k_scatter_tiles<1>, (unsigned)tg, (unsigned)kBThreads, sizeof(ScatterSmem<1>), st, n_tiles, src, dst, occ, bk, gated));
        else CCL_CUDA_TRY(launch_pdl_smem(k_scatter_tiles<2>, (unsigned)tg, (unsigned)kBThreads, sizeof(ScatterSmem<2>), st, n_tiles, src, dst, occ, bk, gated));
        count_launch();
        done = n_tiles * kTileBonds;
    }
    if (done < n_bonds) {
        const int64_t rest = n_bonds - done;
        const int32_t *s2 = src + done, *d2 = dst + done;
        const int vec2 = ((reinterpret_cast<uintptr_t>(s2) | reinterpret_cast<uintptr_t>(d2)) & 15) == 0;
        const unsigned sg = (unsigned)grids.scatter;
        if (mk == 0) CCL_CUDA_TRY(launch_pdl(k_scatter<0>, sg, (unsigned)kBThreads, st, rest, s2, d2, (const void*)nullptr, vec2, bk, gated));
        else if (mk == 1) CCL_CUDA_TRY(launch_pdl(k_scatter<1>, sg, (unsigned)kBThreads, st, rest, s2, d2, (const void*)(static_cast<const uint8_t*>(occ) + done), vec2, bk, gated));
        else CCL_CUDA_TRY(launch_pdl(k_scatter<2>, sg, (unsigned)kBThreads, st, rest, s2, d2, (const void*)(static_cast<const uint32_t*>(occ) + done / 32), vec2, bk, gated));
        count_launch();
    }
    for (int r = R - 1; r >= 0; --r) {
        // the kernel before k_descend(r - 1) writes that region's labels, unless they were written up front
        int64_t init_lo = 0, init_hi = 0;
        if (plan.lazy_init && r >= 1) {
            init_lo = (int64_t)(r - 1) << shift;
            init_hi = (int64_t)r << shift;
            if (init_hi > n_sites) init_hi = n_sites;
        }
        L2Window win;                                                  // region r's labels: every atomic of this launch lands there
        if (plan.l2_persist) {
            const int64_t lo = (int64_t)r << shift, hi = ((int64_t)(r + 1) << shift) < n_sites ? ((int64_t)(r + 1) << shift) : n_sites;
            win.base = labels + lo;
            win.bytes = (size_t)(hi - lo) * sizeof(int32_t);
        }
        CCL_CUDA_TRY(launch_pdl_window(k_descend, (unsigned)grids.descend, (unsigned)kBThreads, 0, st, win, r, bk, gated, init_lo, init_hi, labels));
        count_launch();
    }
    return CCL_OK;
}

}  // namespace ccl
