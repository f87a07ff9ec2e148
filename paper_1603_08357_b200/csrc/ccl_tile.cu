// ccl_tile.cu -- tiled form of steps (i)-(iii) of PAPER.md:113 for bond lists that are LOCAL in the site numbering
// (raster-ordered lattices): label reduction in shared memory.
//
// Why: Algorithm 1 is a stream of atomicMin's and root walks on label[].  In L2 that costs one
// transaction per access (131 G atomics/s for the whole GPU, profiles/r1_ubench.txt); one SM does the same on shared
// memory an order of magnitude faster, and where bonds join nearby site numbers almost every bond of a window of
// 2^15 sites (128 KiB of labels, one CTA's shared memory) has both ends inside it:
//
//   k_probe_local   samples the bond list: local (few bonds leave their window) or not.  Not local -> every kernel
//                   below returns at once and the other forms (ccl_label.cu, ccl_bucket.cu) do the call.
//   k_scatter_fine  one pass over the bond stream: every occupied bond becomes a pair (lo, hi) filed under the
//                   window of hi.  A warp's pairs nearly always share a window: one atomicAdd, consecutive stores.
//   k_local         one CTA per window.  Step (i) label[i] = i is written in shared memory and never touches HBM.
//                   Then, as in the paper: hook every site to its smallest lower neighbour (one atomicMin per pair,
//                   the first wave of step (iii)); flatten the window (step (ii)); run Algorithm 1 on every pair
//                   with root walks that stay inside the window.  A pair whose two representatives both lie below
//                   the window cannot be finished here and goes to the residue list.  The window's labels leave
//                   once, flattened locally.
//   k_residual      Algorithm 1 with full root walks on the global label array over the residue (about the bonds
//                   that cross a window border).
//
// The result is the same forest invariant as the direct form (label[x] <= x, one tree per component); step (iv)
// (k_flatten, ccl_label.cu) follows.  Correctness of deferring: a pair is an obligation "a and b end in one tree";
// Algorithm 1 may discharge it, or replace it by the pair its atomicMin returns (R3), in any order.
//
// Measured and dropped (profiles/r1_notes.md): the same pipeline for bonds that are NOT local (random regular
// graphs).  Filing 60 M pairs under 2048 windows costs one L2 transaction per pair whatever the mechanism (direct
// atomicAdd + 8-byte store: 0.86-1.4 ms on config 5; a lock-free write-combining ring in shared memory: the same),
// against 0.34-0.40 ms for the 32-way CTA-sorted scatter of ccl_bucket.cu.
#include "ccl_common.cuh"
#include "ccl_unionfind.cuh"
#include "ccl_bonds.cuh"

namespace ccl {

constexpr int kTThreads = 1024;                    // k_local, k_small: one CTA per SM
constexpr int kSThreads = 256;                     // k_scatter_fine


// ------------------------------------------------------------------------------------------ local Algorithm 1
// Shared-memory window L[0 .. W) holds label[base .. base + W).  Walk x up while its parent stays in the window;
// returns the last site inside (a local root, L[x] == x, or an "exit" whose parent lies below the window).
__device__ __forceinline__ int32_t local_rep(volatile int32_t* L, int32_t base, int32_t x)
{
    for (;;) {
        const int32_t p = L[x - base];
        if (p == x || p < base) return x;
        const int32_t gp = L[p - base];
        if (gp == p || gp < base) return p;
        L[x - base] = gp;                  // path halving; only ever writes an ancestor inside the window
        x = gp;
    }
}

// Algorithm 1 on the pair (a, b) with all label traffic in the window.  Returns true and the pair (a < b < base)
// that is left when both representatives lie below the window.
__device__ __forceinline__ bool local_join(int32_t* L, int32_t base, int32_t& a, int32_t& b)
{
    for (;;) {
        if (b >= base) b = local_rep(L, base, b);
        if (a >= base) a = local_rep(L, base, a);
        if (a == b) return false;
        if (a > b) { const int32_t t = a; a = b; b = t; }
        if (b < base) return true;
        const int32_t old = atomicMin(L + (b - base), a);
        if (old == b || old == a) return false;            // linked now / was linked already (R4)
        // b was not a root: the pair left to join is {a, old} (reading R3)
        b = max(a, old);
        a = min(a, old);
    }
}

// ------------------------------------------------------------------------------------------- k_scatter_fine
// Where a flushed pair goes: slot gpos of sub-region s if it exists, else the overflow list.
__device__ __forceinline__ void put_fine(int s, unsigned gpos, int2 pr, TileHeader* hdr, int2* fine, unsigned cap_f,
                                         int2* ovf, unsigned long long cap_o, uint64_t pol)
{
    if (gpos < cap_f) {
        st_stream_pair(fine + (size_t)s * cap_f + gpos, pr, pol);
    } else {
        const unsigned long long o = atomicAdd(&hdr->overflow, 1ull);
        if (o < cap_o) ovf[o] = pr;
    }
}

// Persistent CTAs.  A warp whose pairs all go to one window (the normal case here) files them with a single global
// atomicAdd and consecutive stores.  Otherwise every pair reserves its own slot: one atomicAdd on the window's counter
// (one counter per 32-byte sector), the four of a lane in flight together.
template <int MASK>
__global__ void __launch_bounds__(kSThreads)
k_scatter_fine(int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
               const void* __restrict__ occ, int vec, int sub_shift, TileHeader* hdr, int2* fine,
               unsigned cap_f, int2* ovf, unsigned long long cap_o)
{
    if (hdr->bh.mode != 0) return;                 // bonds not local: the other forms take the call
    const int tid = threadIdx.x, lane = tid & 31;
    const uint64_t pol = evict_first_policy();
    // Every CTA takes a contiguous range of tiles: with bonds that are local in the numbering the CTAs then work on
    // different sub-regions, instead of all of them hammering the same few bucket counters at the same time.
    const int64_t tiles = (n_bonds + kSThreads * 4 - 1) / (kSThreads * 4);
    const int64_t per = (tiles + gridDim.x - 1) / gridDim.x;
    int64_t tile = (int64_t)blockIdx.x * per;
    const int64_t tile_end = (tile + per < tiles) ? tile + per : tiles;
    Bonds4 nx = load_bonds4<MASK>(n_bonds, tile < tile_end ? (tile * kSThreads + tid) * 4 : n_bonds, src, dst, occ, vec, pol);
    for (; tile < tile_end; ++tile) {
        const Bonds4 cur = nx;
        const int64_t tn = tile + 1;
        nx = load_bonds4<MASK>(n_bonds, tn < tile_end ? (tn * kSThreads + tid) * 4 : n_bonds, src, dst, occ, vec, pol);
        int32_t lo[4], hi[4];
        uint32_t pm = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            lo[k] = min(cur.u[k], cur.v[k]);
            hi[k] = max(cur.u[k], cur.v[k]);
            if (((cur.m >> k) & 1u) && lo[k] != hi[k]) pm |= 1u << k;
        }
        const unsigned any = __ballot_sync(0xffffffffu, pm != 0);
        if (any == 0) continue;
        const int first = __ffs(any) - 1;
        const int my_s = ((pm & 1u) ? hi[0] : (pm & 2u) ? hi[1] : (pm & 4u) ? hi[2] : hi[3]) >> sub_shift;
        const int s0 = __shfl_sync(0xffffffffu, my_s, first);
        bool mine_same = true;
#pragma unroll
        for (int k = 0; k < 4; ++k) if (((pm >> k) & 1u) && (hi[k] >> sub_shift) != s0) mine_same = false;
        if (__all_sync(0xffffffffu, mine_same)) {
            const int cnt = __popc(pm);
            int incl = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            unsigned gpos = 0;
            if (lane == 31) gpos = atomicAdd(&hdr->fine[s0 * kFineStride], (unsigned)incl);
            gpos = __shfl_sync(0xffffffffu, gpos, 31) + (unsigned)(incl - cnt);
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if ((pm >> k) & 1u) put_fine(s0, gpos++, make_int2(lo[k], hi[k]), hdr, fine, cap_f, ovf, cap_o, pol);
            continue;
        }
        unsigned gp[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            gp[k] = 0;
            if ((pm >> k) & 1u) gp[k] = atomicAdd(&hdr->fine[(hi[k] >> sub_shift) * kFineStride], 1u);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if ((pm >> k) & 1u) put_fine(hi[k] >> sub_shift, gp[k], make_int2(lo[k], hi[k]), hdr, fine, cap_f, ovf, cap_o, pol);
    }
}

// -------------------------------------------------------------------------------------------------- k_local
// One CTA per sub-region s = blockIdx.x: sites [base, base + W).  Shared memory: L[W].
__device__ __forceinline__ void local_writeback(const int32_t* L, int32_t base, int32_t W, int64_t n_sites,
                                                int32_t* __restrict__ label)
{
    // Local step (iv): every site leaves with the top of its chain inside the window -- a local root, or the
    // parent (below the window) of the exit its chain ends in.  Read-only walks, so no ordering is needed.
    for (int32_t i0 = threadIdx.x * 4; i0 < W; i0 += blockDim.x * 4) {
        int32_t out[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            int32_t x = L[i0 + k];
            for (;;) {
                if (x < base) break;
                const int32_t p = L[x - base];
                if (p == x) break;
                x = p;
            }
            out[k] = x;
        }
        const int64_t g = (int64_t)base + i0;
        if (g + 4 <= n_sites) {
            *reinterpret_cast<int4*>(label + g) = make_int4(out[0], out[1], out[2], out[3]);
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k) if (g + k < n_sites) label[g + k] = out[k];
        }
    }
}

// The paper's steps (i)-(ii) inside the window: L[] holds label[i] = i; every pair hooks its higher
// site to the lower one with one atomicMin (no return value needed), then every site is re-pointed at the top of its
// chain inside the window.  Joining pair by pair from scratch instead means long root walks under heavy contention on
// lattice clusters; after this the join pass starts from flat trees and finds most pairs connected already.
template <typename LoadPair>
__device__ __forceinline__ void local_hook_and_flatten(int32_t* L, int32_t base, int32_t W, unsigned n, LoadPair load)
{
    // batches of 8 loads in flight per thread: with one CTA per SM a one-load-one-atomic loop is all memory latency
    for (unsigned i0 = 0; i0 < n; i0 += blockDim.x * 8) {
        int2 pr[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const unsigned i = i0 + k * blockDim.x + threadIdx.x;
            pr[k] = i < n ? load(i) : make_int2(-1, -1);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k)
            if (pr[k].x >= 0 && pr[k].x != pr[k].y) atomicMin(L + (max(pr[k].x, pr[k].y) - base), min(pr[k].x, pr[k].y));
    }
    __syncthreads();
    for (int32_t i = threadIdx.x; i < W; i += blockDim.x) {
        int32_t x = base + i;
        for (;;) {
            const int32_t p = reinterpret_cast<volatile int32_t*>(L)[x - base];
            if (p == x || p < base) break;
            x = p;
        }
        if (x != base + i) L[i] = x;                        // the local representative (a local root or an exit)
    }
    __syncthreads();
}

constexpr int kListCap = 8192;                     // residue pairs one CTA stages in shared memory (64 KiB)

__global__ void __launch_bounds__(kTThreads, 1)
k_local(int64_t n_sites, int sub_shift, int S, TileHeader* hdr, const int2* __restrict__ fine, unsigned cap_f, int2* ovf,
        unsigned long long cap_o, int32_t* __restrict__ label)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (hdr->bh.mode != 0) return;
    int32_t* L = reinterpret_cast<int32_t*>(smem_raw);
    const int tid = threadIdx.x;
    const int32_t W = 1 << sub_shift;
    int2* list = reinterpret_cast<int2*>(smem_raw + (size_t)W * sizeof(int32_t));
    __shared__ unsigned s_cnt;
    __shared__ unsigned long long s_base;
    const uint64_t pol = evict_first_policy();
    constexpr int P = 4;
    for (int s = blockIdx.x; s < S; s += gridDim.x) {        // persistent: a gated-off launch costs one wave of CTAs
        const int32_t base = s << sub_shift;
        if (tid == 0) s_cnt = 0;
        for (int32_t i = tid * 4; i < W; i += kTThreads * 4)
            *reinterpret_cast<int4*>(L + i) = make_int4(base + i, base + i + 1, base + i + 2, base + i + 3);    // step (i)
        unsigned n = hdr->fine[s * kFineStride];
        if (n > cap_f) n = cap_f;
        const int2* bucket = fine + (size_t)s * cap_f;
        __syncthreads();
        local_hook_and_flatten(L, base, W, n, [&](unsigned i) { return __ldg(bucket + i); });   // read again below: L2 hit
        // Algorithm 1 on every pair; no barrier inside, so uneven walk lengths average out over a thread's pairs.
        auto load_round = [&](unsigned i0, int2 (&pr)[P]) {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                const unsigned i = i0 + k * kTThreads + tid;
                pr[k] = make_int2(-1, -1);
                if (i < n) {
                    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.s32 {%0,%1}, [%2], %3;"
                                 : "=r"(pr[k].x), "=r"(pr[k].y) : "l"(bucket + i), "l"(pol));
                }
            }
        };
        int2 nxt[P];
        load_round(0, nxt);
        for (unsigned i0 = 0; i0 < n; i0 += kTThreads * P) {
            int2 pr[P];
#pragma unroll
            for (int k = 0; k < P; ++k) pr[k] = nxt[k];
            load_round(i0 + kTThreads * P, nxt);             // next round's pairs travel while this round is joined
#pragma unroll
            for (int k = 0; k < P; ++k) {
                int32_t a = pr[k].x, b = pr[k].y;
                if (a >= 0 && local_join(L, base, a, b)) {
                    const unsigned j = atomicAdd(&s_cnt, 1u);
                    if (j < (unsigned)kListCap) {
                        list[j] = make_int2(a, b);
                    } else {                                 // staging full: file it directly
                        const unsigned long long o = atomicAdd(&hdr->overflow, 1ull);
                        if (o < cap_o) ovf[o] = make_int2(a, b);
                    }
                }
            }
        }
        __syncthreads();
        const unsigned m = s_cnt < (unsigned)kListCap ? s_cnt : (unsigned)kListCap;
        if (tid == 0 && m) s_base = atomicAdd(&hdr->overflow, (unsigned long long)m);
        __syncthreads();
        for (unsigned j = tid; j < m; j += kTThreads) {
            const unsigned long long o = s_base + j;
            if (o < cap_o) ovf[o] = list[j];
        }
        local_writeback(L, base, W, n_sites, label);
        __syncthreads();                                     // L[] and the list are reused by the next window
    }
}

// ------------------------------------------------------------------------------------------------- k_small
// n_sites <= 2^15: the whole label array is one window; one CTA does steps (i)-(iv) in one launch.
template <int MASK>
__global__ void __launch_bounds__(kTThreads, 1)
k_small(int64_t n_sites, int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
        const void* __restrict__ occ, int32_t* __restrict__ label)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int32_t* L = reinterpret_cast<int32_t*>(smem_raw);
    const int tid = threadIdx.x;
    const int32_t W = (int32_t)((n_sites + 3) & ~3ll);
    for (int32_t i = tid * 4; i < W; i += kTThreads * 4) *reinterpret_cast<int4*>(L + i) = make_int4(i, i + 1, i + 2, i + 3);
    __syncthreads();
    auto load = [&](unsigned b) {
        bool on = true;
        if (MASK == 1) on = static_cast<const uint8_t*>(occ)[b] != 0;
        if (MASK == 2) on = (static_cast<const uint32_t*>(occ)[b >> 5] >> (b & 31)) & 1u;
        return on ? make_int2(src[b], dst[b]) : make_int2(-1, -1);
    };
    local_hook_and_flatten(L, 0, W, (unsigned)n_bonds, load);
    for (unsigned b = tid; b < (unsigned)n_bonds; b += kTThreads) {
        const int2 pr = load(b);
        int32_t u = pr.x, v = pr.y;
        if (u >= 0) local_join(L, 0, u, v);                  // base 0: nothing lies below the window
    }
    __syncthreads();
    local_writeback(L, 0, W, n_sites, label);
}

// ----------------------------------------------------------------------------------------------- k_residual
// Algorithm 1 with full root walks on the global label array, over the residue list.
__global__ void __launch_bounds__(256)
k_residual(TileHeader* hdr, const int2* __restrict__ ovf, unsigned long long cap_o, int32_t* label)
{
    if (hdr->bh.mode != 0) return;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    unsigned long long n = hdr->overflow;
    if (n > cap_o) n = cap_o;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int2 pr = ovf[i];
        algorithm1(label, pr.x, pr.y);
    }
}

// -------------------------------------------------------------------------------------------- k_probe_local
// Samples up to 8192 bonds at a fixed stride: local = fewer than a quarter of them leave their window.  mode 0 = local
// (the tiled form runs), 1 = not local.  force: -1 decide, 0/1 fixed.
__global__ void __launch_bounds__(1024)
k_probe_local(int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst, int sub_shift, int force,
              TileHeader* hdr)
{
    __shared__ int s_cross;
    if (threadIdx.x == 0) s_cross = 0;
    __syncthreads();
    const int64_t samples = n_bonds < 8192 ? n_bonds : 8192;
    const int64_t stride = n_bonds / samples;
    int cross = 0;
    for (int64_t i = threadIdx.x; i < samples; i += 1024) {
        const int32_t u = src[i * stride], v = dst[i * stride];
        cross += (u >> sub_shift) != (v >> sub_shift);
    }
    for (int o = 16; o > 0; o >>= 1) cross += __shfl_xor_sync(0xffffffffu, cross, o);
    if ((threadIdx.x & 31) == 0 && cross) atomicAdd(&s_cross, cross);
    __syncthreads();
    if (threadIdx.x == 0) hdr->bh.mode = force >= 0 ? force : ((4 * (int64_t)s_cross >= samples) ? 1 : 0);
}

// ------------------------------------------------------------------------------------------------- host side
static int ceil_log2_i64(int64_t x)
{
    int k = 0;
    while (((int64_t)1 << k) < x) ++k;
    return k;
}

template <typename K>
static int allow_smem(K kernel, size_t bytes)
{
    CCL_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return CCL_OK;
}

template <int MASK>
static int launch_small(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ,
                        int32_t* labels, cudaStream_t st)
{
    const size_t smem = (size_t)((n_sites + 3) & ~3ll) * sizeof(int32_t);
    { const int rc = allow_smem(k_small<MASK>, smem); if (rc != CCL_OK) return rc; }
    k_small<MASK><<<1, kTThreads, smem, st>>>(n_sites, n_bonds, src, dst, occ, labels);
    CCL_CHECK_LAUNCH("k_small");
    return CCL_OK;
}

template <int MASK>
static int launch_scatter_fine(int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ, int vec,
                               int sub_shift, TileHeader* hdr, int2* fine, unsigned cap_f, int2* ovf,
                               unsigned long long cap_o, cudaStream_t st)
{
    const int64_t tiles = (n_bonds + kSThreads * 4 - 1) / (kSThreads * 4);
    const int grid = (int)(tiles < kSMs * 8 ? tiles : kSMs * 8);
    k_scatter_fine<MASK><<<grid, kSThreads, 0, st>>>(n_bonds, src, dst, occ, vec, sub_shift, hdr, fine, cap_f, ovf, cap_o);
    CCL_CHECK_LAUNCH("k_scatter_fine");
    return CCL_OK;
}

int tiled_reduce(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ,
                 int mask_kind, int32_t* labels, cudaStream_t st, int* done, const int32_t** not_local, void** ws_out)
{
    *done = kTiledNo;
    *not_local = nullptr;
    *ws_out = nullptr;
    const Tuning& t = tuning();
    if (t.tile_mode == 0 || n_bonds <= 0) return CCL_OK;
    const uintptr_t al = reinterpret_cast<uintptr_t>(src) | reinterpret_cast<uintptr_t>(dst);
    int vec = (al & 15) == 0;
    if (occ != nullptr && mask_kind == 1) vec = vec && (reinterpret_cast<uintptr_t>(occ) & 3) == 0;
    if (occ != nullptr && mask_kind == 2 && (reinterpret_cast<uintptr_t>(occ) & 3) != 0) {
        set_error("invalid argument: occupied_bits is not 4-byte aligned");
        return CCL_INVALID_ARG;
    }
    const int mk = occ == nullptr ? 0 : mask_kind;
    int rc = CCL_OK;

    // the whole label array fits one CTA's shared memory: one launch does steps (i)-(iv)
    if (n_sites <= t.small_max_sites && n_sites <= (1 << 15) && t.sub_shift < 0 && n_bonds <= (1 << 20)) {
        if (mk == 0) rc = launch_small<0>(n_sites, n_bonds, src, dst, occ, labels, st);
        else if (mk == 1) rc = launch_small<1>(n_sites, n_bonds, src, dst, occ, labels, st);
        else rc = launch_small<2>(n_sites, n_bonds, src, dst, occ, labels, st);
        if (rc == CCL_OK) *done = kTiledFinal;
        return rc;
    }
    if (t.tile_mode < 0 && n_bonds < t.tile_min_bonds) return CCL_OK;

    // as large a window as shared memory holds (2^15 sites), smaller only to keep at least ~128 CTAs in k_local
    int sub_shift = t.sub_shift >= 0 ? t.sub_shift : ceil_log2_i64(n_sites) - 7;
    if (sub_shift < 10 && t.sub_shift < 0) sub_shift = 10;
    if (sub_shift > 15) sub_shift = 15;
    if (sub_shift < 2) sub_shift = 2;
    const int64_t S64 = ((n_sites - 1) >> sub_shift) + 1;
    if (S64 > kMaxSubRegions) return CCL_OK;         // beyond 2^26 sites: the other forms take the call
    const int S = (int)S64;

    unsigned long long cap_f = (unsigned long long)(2 * n_bonds / S + 8192);
    if (t.fine_capacity > 0) cap_f = (unsigned long long)t.fine_capacity;
    cap_f = (cap_f + 7ull) & ~7ull;
    const unsigned long long cap_o = ((unsigned long long)n_bonds + 7ull) & ~7ull;
    const size_t hdr_bytes = (sizeof(TileHeader) + 255) & ~(size_t)255;
    const size_t bytes = hdr_bytes + ((size_t)S * cap_f + cap_o) * sizeof(int2);
    void* ws = nullptr;
    if ((rc = scratch_alloc(&ws, bytes, st)) != CCL_OK) return rc;
    TileHeader* hdr = static_cast<TileHeader*>(ws);
    int2* fine = reinterpret_cast<int2*>(static_cast<char*>(ws) + hdr_bytes);
    int2* ovf = fine + (size_t)S * cap_f;

    auto fail = [&](int code) { cudaFreeAsync(ws, st); return code; };
    auto launched = [&](const char* name) {
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) { set_error("launch of %s failed: %s", name, cudaGetErrorString(e)); return false; }
        count_launch();
        return true;
    };
    if (cudaMemsetAsync(hdr, 0, sizeof(TileHeader), st) != cudaSuccess) { set_error("cudaMemsetAsync failed"); return fail(CCL_CUDA_ERROR); }
    k_probe_local<<<1, 1024, 0, st>>>(n_bonds, src, dst, sub_shift, t.tile_mode == 1 ? 0 : -1, hdr);
    if (!launched("k_probe_local")) return fail(CCL_CUDA_ERROR);
    if (mk == 0) rc = launch_scatter_fine<0>(n_bonds, src, dst, occ, vec, sub_shift, hdr, fine, (unsigned)cap_f, ovf, cap_o, st);
    else if (mk == 1) rc = launch_scatter_fine<1>(n_bonds, src, dst, occ, vec, sub_shift, hdr, fine, (unsigned)cap_f, ovf, cap_o, st);
    else rc = launch_scatter_fine<2>(n_bonds, src, dst, occ, vec, sub_shift, hdr, fine, (unsigned)cap_f, ovf, cap_o, st);
    if (rc != CCL_OK) return fail(rc);

    const size_t lsmem = (sizeof(int32_t) << sub_shift) + (size_t)kListCap * sizeof(int2);
    if ((rc = allow_smem(k_local, lsmem)) != CCL_OK) return fail(rc);
    k_local<<<S < kSMs ? S : kSMs, kTThreads, lsmem, st>>>(n_sites, sub_shift, S, hdr, fine, (unsigned)cap_f, ovf, cap_o, labels);
    if (!launched("k_local")) return fail(CCL_CUDA_ERROR);
    k_residual<<<kSMs * 8, 256, 0, st>>>(hdr, ovf, cap_o, labels);
    if (!launched("k_residual")) return fail(CCL_CUDA_ERROR);
    *ws_out = ws;                                    // the caller frees it once every kernel that reads the flag is enqueued
    *not_local = &hdr->bh.mode;
    *done = t.tile_mode == 1 ? kTiledForced : kTiledIfLocal;
    return CCL_OK;
}

}  // namespace ccl
