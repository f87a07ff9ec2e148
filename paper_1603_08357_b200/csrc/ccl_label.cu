// ccl_label.cu -- steps (i)-(iv) of Komura's generalized CCL on a bond list, for sm_100a.
//
//   k_init     step (i)   label[i] = i                       (BASELINE.json north_star form; with it step (ii),
//                         the first analysis, has nothing to do: every site is its own root -- DESIGN.md R1)
//   k_reduce   step (iii) one pass over the bond stream; every occupied bond runs Algorithm 1
//                         (PAPER.md:118-149): atomicMin(&label[larger], smaller), following the returned value
//   k_flatten  step (iv)  label[i] <- root(i)                ("analysis", Fig. 4)
//
// Everything is integer work on int32 labels; the bound is HBM / L2 gather traffic, so there are no tensor cores
// here.
#include "ccl_common.cuh"
#include "ccl_unionfind.cuh"
#include "ccl_bonds.cuh"

namespace ccl {

constexpr int kThreads = 256;

// ------------------------------------------------------------------------------------------------ step (i)
__global__ void __launch_bounds__(kThreads)
k_init(int64_t n_sites, int32_t* __restrict__ label, ProbeJob job)
{
    // the probe of the region-bucketed form rides along in block 0, which starts first (ccl_common.cuh)
    if (job.hdr != nullptr && blockIdx.x == 0) probe_regions(job);
    init_range(label, 0, n_sites, (int64_t)blockIdx.x * kThreads + threadIdx.x, (int64_t)gridDim.x * kThreads);
}

// Which of the enqueued forms of step (iii) runs is decided on the device when the host does not know yet whether the
// bond list is local in the site numbering (BucketHeader::mode, written by the probe) -- no host round trip.
enum { kGateNone = 0, kGateDirect = 1, kGateDirectOrOverflow = 2, kGateOverflow = 3 };
__device__ __forceinline__ bool gate_open(const BucketHeader* hdr, int kind)
{
    if (kind == kGateNone) return true;
    if (kind == kGateDirect) return hdr->mode == 0;
    if (kind == kGateDirectOrOverflow) return hdr->mode == 0 || hdr->overflow != 0;
    return hdr->overflow != 0;
}

// ---------------------------------------------------------------------------------------------- step (iii)
// MASK: 0 = every bond occupied, 1 = uint8 per bond, 2 = packed bits.  VEC: src/dst 16-byte aligned (and the
// uint8 mask 4-byte aligned), so a thread fetches its 4 bonds with two 128-bit loads.
//
// First touch of a thread's (up to) 4 bonds: Algorithm 1's atomicMin applied straight to the bond's own endpoints, all
// four in flight at once.  If the higher site was still a root this IS the link (the paper's step (i) hook,
// PAPER.md:113, done as the first wave of step (iii)); otherwise the returned value tells which pair is left to join.
// Returns how many pairs are left; they are stored in pa[]/pb[] front-packed.
__device__ __forceinline__ int first_touch4(const Bonds4& c, int32_t* label, int32_t (&pa)[4], int32_t (&pb)[4])
{
    if (c.m == 0) return 0;
    int32_t lo[4], old[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        lo[k] = min(c.u[k], c.v[k]);
        const int32_t hi = max(c.u[k], c.v[k]);
        old[k] = lo[k];                                    // "nothing left to do"
        const bool need = ((c.m >> k) & 1u) && hi != lo[k];
        if (need) {
            const int32_t o = atomicMin(label + hi, lo[k]);
            old[k] = (o == hi) ? lo[k] : o;
        }
    }
    int n = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (old[k] != lo[k]) {
#pragma unroll
            for (int q = 0; q < 4; ++q) if (q == n) { pa[q] = old[k]; pb[q] = lo[k]; }    // keeps pa/pb in registers
            ++n;
        }
    return n;
}

// One pass over the bond stream.  About a quarter of the occupied bonds survive the first touch and need root
// walks, which are long chains of dependent L2 loads; left where they arise they would keep a quarter of the lanes
// busy for four rounds.  So every warp packs its survivors into a shared-memory queue and works through the queue
// 32 pairs at a time, every lane busy; fewer than 32 pairs stay queued for the next iteration (the order in which
// bonds are joined is free), at most 31 + 128 of them.
constexpr int kQueueSlots = 160;
template <int MASK, bool VEC>
__global__ void __launch_bounds__(kThreads)
k_reduce(int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
         const void* __restrict__ occ, int32_t* label, const BucketHeader* hdr, int gate,
         int32_t* notify, int32_t notify_value)
{
    __shared__ int2 queue[kThreads / 32][kQueueSlots];
    pdl_wait();
    if (!gate_open(hdr, gate)) return;                     // the bucketed form (ccl_bucket.cu) did step (iii)
    // Running as the safety net of the bucketed form (its chunk pool ran dry): tell the host, through mapped pinned
    // memory, that the next call on this bond list should draw a larger pool (label_impl).
    if (notify != nullptr && hdr != nullptr && hdr->overflow != 0 && blockIdx.x == 0 && threadIdx.x == 0) {
        *reinterpret_cast<volatile int32_t*>(notify) = notify_value;
        __threadfence_system();
    }
    const uint64_t pol = evict_first_policy();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t stride = (int64_t)gridDim.x * kThreads * 4;
    const int64_t n_round = ((n_bonds + 127) / 128) * 128;                 // whole warps take part in every round
    int qn = 0;                                            // pairs waiting in this warp's queue (the same in every lane)
    int64_t b0 = ((int64_t)blockIdx.x * kThreads + threadIdx.x) * 4;
    uint32_t m_next = load_mask4<MASK>(n_bonds, b0, occ, VEC, pol);
    for (; b0 < n_round; b0 += stride) {
        // this iteration's endpoints and the next iteration's occupancy bits travel together
        const Bonds4 c = load_ends4(n_bonds, b0, m_next, src, dst, VEC, pol);
        m_next = load_mask4<MASK>(n_bonds, b0 + stride, occ, VEC, pol);
        int32_t pa[4], pb[4];
        const int n = first_touch4(c, label, pa, pb);
        int incl = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        if (total == 0) continue;
        const int off = qn + incl - n;
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (q < n) queue[warp][off + q] = make_int2(pa[q], pb[q]);
        qn += total;
        __syncwarp();
        while (qn >= 32) {                                 // whole rounds only: every lane has a pair to walk
            qn -= 32;
            const int2 pr = queue[warp][qn + lane];
            algorithm1(label, pr.x, pr.y);
        }
        __syncwarp();
    }
    if (lane < qn) {                                       // what is left at the end of the warp's share of the bonds
        const int2 pr = queue[warp][lane];
        algorithm1(label, pr.x, pr.y);
    }
}

// ------------------------------------------------------------------------------- two-pass form of step (iii)
// The paper's own order of work: (i) every site takes its smallest lower-numbered neighbour as initial
// label -- here one atomicMin per occupied bond whose result nobody waits for (k_hook) -- (ii) analysis (k_flatten),
// (iii) Algorithm 1 over the bonds (k_join), (iv) analysis.  After (ii) the trees are flat, so k_join reads two labels
// per bond, finds most bonds joined already, and only the rest walk and link.  Costs a second pass over the bond stream
// and a second flatten; pays where root walks dominate the one-pass kernel (clusters much larger than a warp's bonds).
template <int MASK>
__global__ void __launch_bounds__(kThreads)
k_hook(int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst, const void* __restrict__ occ,
       int vec, int32_t* label, const BucketHeader* hdr, int gate)
{
    pdl_wait();
    if (!gate_open(hdr, gate)) return;                     // another form did step (iii)
    const uint64_t pol = evict_first_policy();
    const int64_t stride = (int64_t)gridDim.x * kThreads * 4;
    const int64_t n_round = ((n_bonds + 127) / 128) * 128;                 // whole warps take part in every round
    int64_t b0 = ((int64_t)blockIdx.x * kThreads + threadIdx.x) * 4;
    uint32_t m_next = load_mask4<MASK>(n_bonds, b0, occ, vec, pol);
    for (; b0 < n_round; b0 += stride) {
        const Bonds4 c = load_ends4(n_bonds, b0, m_next, src, dst, vec, pol);
        m_next = load_mask4<MASK>(n_bonds, b0 + stride, occ, vec, pol);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const bool need = ((c.m >> k) & 1u) && c.u[k] != c.v[k];
            const int32_t lo = min(c.u[k], c.v[k]), hi = max(c.u[k], c.v[k]);
            if (need) atomicMin(label + hi, lo);
        }
    }
}

template <int MASK>
__global__ void __launch_bounds__(kThreads)
k_join(int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst, const void* __restrict__ occ,
       int vec, int32_t* label, const BucketHeader* hdr, int gate)
{
    __shared__ int2 queue[kThreads / 32][kQueueSlots];
    pdl_wait();
    if (!gate_open(hdr, gate)) return;
    const uint64_t pol = evict_first_policy();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t stride = (int64_t)gridDim.x * kThreads * 4;
    const int64_t n_round = ((n_bonds + 127) / 128) * 128;                 // whole warps take part in every round
    int qn = 0;                                            // as in k_reduce: whole rounds of 32 pairs, the rest waits
    int64_t b0 = ((int64_t)blockIdx.x * kThreads + threadIdx.x) * 4;
    uint32_t m_next = load_mask4<MASK>(n_bonds, b0, occ, vec, pol);
    for (; b0 < n_round; b0 += stride) {
        const Bonds4 c = load_ends4(n_bonds, b0, m_next, src, dst, vec, pol);
        m_next = load_mask4<MASK>(n_bonds, b0 + stride, occ, vec, pol);
        // labels of both ends, all eight loads in flight; after the flatten they are roots unless k_join moved them
        int32_t la[4], lb[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const bool on = (c.m >> k) & 1u;
            la[k] = on ? ld_label(label + c.u[k]) : 0;
            lb[k] = on ? ld_label(label + c.v[k]) : 0;
        }
        int n = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) n += la[k] != lb[k];
        int incl = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        if (total == 0) continue;
        int off = qn + incl - n;
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (la[k] != lb[k]) queue[warp][off++] = make_int2(la[k], lb[k]);     // joining the two labels joins the two sites
        qn += total;
        __syncwarp();
        while (qn >= 32) {
            qn -= 32;
            const int2 pr = queue[warp][qn + lane];
            algorithm1(label, pr.x, pr.y);
        }
        __syncwarp();
    }
    if (lane < qn) {
        const int2 pr = queue[warp][lane];
        algorithm1(label, pr.x, pr.y);
    }
}

// ----------------------------------------------------------------------------------------------- step (iv)
// Every site follows its chain to the root and stores it (reading R2: per-site chase).  Concurrent
// writers only ever replace a chain pointer by the root of the same chain, so a reader sees either and still
// arrives at the root.  Roots and already-flat sites are not rewritten.
//
// One launch covers the sites [lo, n_sites) and resolves those whose label lies in the window [lo, hi).  With
// (lo, hi) = (0, n_sites) that is the whole analysis step.  For label arrays beyond L2 the windows are taken in
// ascending order, one launch each: label[x] <= x always, so when the window [lo, hi) runs every label below lo is
// final (a root) -- a chase that starts in the window either ends at a root inside it or leaves it downwards and is
// then finished.  All gathers of one launch fall into the window, which stays L2-resident, while the sites above it
// stream past once (evict-first).  A random gather into 256 MiB costs an HBM sector fetch each; into 64 MiB it is an
// L2 hit.
__global__ void __launch_bounds__(kThreads)
k_flatten(int64_t n_sites, int32_t* label, int64_t lo, int64_t hi, const BucketHeader* hdr, int gate)
{
    pdl_wait();
    if (!gate_open(hdr, gate)) return;                     // only for the mid-call flatten of the two-pass form
    constexpr int S = 4, G = 1;                            // four sites (one 16-byte group) per thread
    // the groups of a thread lie kThreads groups apart, so that a warp's loads stay contiguous
    const int64_t g0 = lo + ((int64_t)blockIdx.x * kThreads * G + threadIdx.x) * 4;
    const int32_t wlo = (int32_t)lo, whi = (int32_t)(hi - 1);          // window = [wlo, whi]
    const uint64_t pol = evict_first_policy();
    int32_t cur[S], c[S], par[S];
    bool w[S], full[G], above[G], any = false;
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const int64_t i0 = g0 + (int64_t)g * kThreads * 4;
        full[g] = i0 + 4 <= n_sites;
        above[g] = i0 >= hi;                                           // streams past: read once, written at most once
        int4 l = make_int4(0, 0, 0, 0);
        if (full[g]) l = above[g] ? ld_once_v4(label + i0, pol) : *reinterpret_cast<const int4*>(label + i0);
        cur[4 * g] = l.x; cur[4 * g + 1] = l.y; cur[4 * g + 2] = l.z; cur[4 * g + 3] = l.w;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int q = 4 * g + k;
            c[q] = cur[q];
            w[q] = full[g] && cur[q] != (int32_t)(i0 + k) && cur[q] >= wlo && cur[q] <= whi;
            any |= w[q];
        }
    }
    if (any) {
        // the chases advance together: one round = up to S independent loads in flight
#pragma unroll
        for (int q = 0; q < S; ++q) par[q] = w[q] ? ld_label(label + c[q]) : c[q];
        for (;;) {
            any = false;
#pragma unroll
            for (int q = 0; q < S; ++q) {
                if (w[q]) {
                    if (par[q] == c[q]) w[q] = false;                               // c is a root
                    else if (par[q] < wlo) { c[q] = par[q]; w[q] = false; }          // left the window: final
                    else c[q] = par[q];
                }
                any |= w[q];
            }
            if (!any) break;
#pragma unroll
            for (int q = 0; q < S; ++q) if (w[q]) par[q] = ld_label(label + c[q]);
        }
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const int64_t i0 = g0 + (int64_t)g * kThreads * 4;
            const bool changed = (c[4 * g] != cur[4 * g]) | (c[4 * g + 1] != cur[4 * g + 1]) | (c[4 * g + 2] != cur[4 * g + 2]) |
                                 (c[4 * g + 3] != cur[4 * g + 3]);
            if (changed) {
                const int4 out = make_int4(c[4 * g], c[4 * g + 1], c[4 * g + 2], c[4 * g + 3]);
                if (above[g]) st_stream_v4(label + i0, out, pol);
                else *reinterpret_cast<int4*>(label + i0) = out;
            }
        }
    }
    // the ragged end of the array (fewer than four sites), by the thread whose group it would have been
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const int64_t i0 = g0 + (int64_t)g * kThreads * 4;
        if (!full[g] && i0 < n_sites) {
            for (int64_t i = i0; i < n_sites; ++i) {
                int32_t x = label[i];
                if (x == (int32_t)i || x < wlo || x > whi) continue;
                int32_t p = ld_label(label + x);
                while (p != x && p >= wlo) { x = p; p = ld_label(label + x); }
                label[i] = (p == x) ? x : p;
            }
        }
    }
    pdl_go();
}

__global__ void __launch_bounds__(kThreads)
k_validate(int64_t n_sites, int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
           unsigned long long* out_bad)
{
    unsigned long long bad = 0;
    const int64_t stride = (int64_t)gridDim.x * kThreads;
    for (int64_t b = (int64_t)blockIdx.x * kThreads + threadIdx.x; b < n_bonds; b += stride) {
        const int64_t u = src[b], v = dst[b];
        bad += (u < 0 || u >= n_sites || v < 0 || v >= n_sites);
    }
    for (int o = 16; o > 0; o >>= 1) bad += __shfl_xor_sync(0xffffffffu, bad, o);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(out_bad, bad);
}

// ------------------------------------------------------------------------------------------------- host side
static int check_args(int64_t n_sites, int64_t n_bonds, const void* src, const void* dst, const void* labels)
{
    CCL_REQUIRE(n_sites >= 0, "n_sites < 0");
    CCL_REQUIRE(n_sites <= 2147483647LL, "n_sites > 2^31-1 (labels are int32)");
    CCL_REQUIRE(n_bonds >= 0, "n_bonds < 0");
    CCL_REQUIRE(n_sites == 0 || labels != nullptr, "labels is NULL");
    CCL_REQUIRE(n_bonds == 0 || (src != nullptr && dst != nullptr), "src/dst is NULL with n_bonds > 0");
    CCL_REQUIRE(n_bonds == 0 || n_sites > 0, "bonds given but n_sites == 0");
    CCL_REQUIRE((reinterpret_cast<uintptr_t>(labels) & 3) == 0, "labels is not 4-byte aligned");
    return CCL_OK;
}

template <int MASK>
static int launch_reduce(int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ,
                         int32_t* labels, const BucketHeader* hdr, int gate, cudaStream_t st, int32_t* notify = nullptr,
                         int32_t notify_value = 0)
{
    const int64_t groups = (n_bonds + 3) / 4;
    int64_t blocks = (groups + kThreads - 1) / kThreads;
    if (blocks > (int64_t)sm_count() * 8 * 4) blocks = (int64_t)sm_count() * 8 * 4;       // grid-stride beyond 4 waves of 8 CTAs/SM
    uintptr_t a = reinterpret_cast<uintptr_t>(src) | reinterpret_cast<uintptr_t>(dst);
    bool vec = (a & 15) == 0;
    if (MASK == 1) vec = vec && (reinterpret_cast<uintptr_t>(occ) & 3) == 0;
    if (vec) CCL_CUDA_TRY(launch_pdl(k_reduce<MASK, true>, (unsigned)blocks, (unsigned)kThreads, st, n_bonds, src, dst, occ, labels, hdr, gate, notify, notify_value));
    else     CCL_CUDA_TRY(launch_pdl(k_reduce<MASK, false>, (unsigned)blocks, (unsigned)kThreads, st, n_bonds, src, dst, occ, labels, hdr, gate, notify, notify_value));
    count_launch();
    return CCL_OK;
}

static int launch_flatten(int64_t n_sites, int32_t* labels, int64_t lo, int64_t hi, const BucketHeader* hdr, int gate,
                          cudaStream_t st, bool persist_window = false)
{
    const int64_t blocks = (((n_sites - lo + 3) / 4) + kThreads - 1) / kThreads;
    L2Window win;                                          // the gather window [lo, hi) of a windowed step (iv)
    if (persist_window) { win.base = labels + lo; win.bytes = (size_t)(hi - lo) * sizeof(int32_t); }
    const cudaError_t e = launch_pdl_window(k_flatten, (unsigned)blocks, (unsigned)kThreads, 0, st, win, n_sites, labels, lo, hi, hdr, gate);
    if (e != cudaSuccess) { set_error("launch of k_flatten failed: %s", cudaGetErrorString(e)); return CCL_CUDA_ERROR; }
    count_launch();
    return CCL_OK;
}

template <int MASK>
static int launch_two_pass(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ,
                           int32_t* labels, const BucketHeader* hdr, int gate, cudaStream_t st)
{
    const int64_t groups = (n_bonds + 3) / 4;
    int64_t blocks = (groups + kThreads - 1) / kThreads;
    // one resident wave, grid-stride (measured on cfg2: 1 / 4 / 8 / 16 waves 0.458 / 0.467 / 0.474 / 0.496 ms; the one-pass
    // kernel above is the other way round on the honeycomb lattice: 0.777 / 0.683 / 0.683 / 0.704 ms)
    if (blocks > (int64_t)sm_count() * 8) blocks = (int64_t)sm_count() * 8;
    uintptr_t a = reinterpret_cast<uintptr_t>(src) | reinterpret_cast<uintptr_t>(dst);
    int vec = (a & 15) == 0;
    if (MASK == 1) vec = vec && (reinterpret_cast<uintptr_t>(occ) & 3) == 0;
    // hook and the mid-call flatten are this form's own steps (i)/(ii); the join pass also serves as the safety net of
    // the bucketed form (it joins whatever the ends of an occupied bond still differ in)
    const int own = gate == kGateNone ? kGateNone : kGateDirect;
    CCL_CUDA_TRY(launch_pdl(k_hook<MASK>, (unsigned)blocks, (unsigned)kThreads, st, n_bonds, src, dst, occ, vec, labels, hdr, own));   // step (i), paper form
    count_launch();
    { const int rc = launch_flatten(n_sites, labels, 0, n_sites, hdr, own, st); if (rc != CCL_OK) return rc; }                      // step (ii)
    CCL_CUDA_TRY(launch_pdl(k_join<MASK>, (unsigned)blocks, (unsigned)kThreads, st, n_bonds, src, dst, occ, vec, labels, hdr, gate));   // step (iii)
    count_launch();
    return CCL_OK;
}

// Step (ii)/(iv) over the whole array.  windowed: gather from one L2-resident window at a time (see k_flatten).
static int flatten_all(int64_t n_sites, int32_t* labels, bool windowed, const Tuning& t, cudaStream_t st)
{
    int64_t w = n_sites;
    if (windowed && t.flatten_window_min_bytes >= 0 && n_sites * (int64_t)sizeof(int32_t) >= t.flatten_window_min_bytes) {
        w = t.flatten_window_bytes / (int64_t)sizeof(int32_t);
        if (w < 1024) w = 1024;
        w &= ~(int64_t)3;
    }
    for (int64_t lo = 0; lo < n_sites; lo += w) {
        const int rc = launch_flatten(n_sites, labels, lo, lo + w < n_sites ? lo + w : n_sites, nullptr, kGateNone, st,
                                      t.l2_persist && w < n_sites);
        if (rc != CCL_OK) return rc;
    }
    return CCL_OK;
}

// step (ii)/(iv) for the other translation units (ccl_nn.cu)
int flatten_labels(int64_t n_sites, int32_t* labels, cudaStream_t st)
{
    return flatten_all(n_sites, labels, false, tuning(), st);
}

// Optional per-step CUDA events (ccl_set_profile_events): recorded on the call's stream between the kernels so
// that a benchmark can read each step's device time from inside its own timed region.
static thread_local cudaEvent_t g_ev[3] = {nullptr, nullptr, nullptr};

static inline void mark(int k, cudaStream_t st)
{
    if (g_ev[k]) cudaEventRecord(g_ev[k], st);
}

// ---- what the region probe said about a bond list, remembered on the host ----------------------------------------
// Both forms of step (iii) are correct for every graph; the probe only picks the faster one.  The first call on a
// bond list enqueues both behind the device-side probe and copies the probe's answer to pinned host memory; later
// calls on the same (src, dst, n_bonds, n_sites) -- an occupancy sweep, the paper's use -- enqueue only the chosen form
// and can then fold step (i) into the bucketed kernels.  A stale entry (the caller rewrote the arrays) costs speed only.
struct ProbeHint {
    const void* src = nullptr;
    const void* dst = nullptr;
    int64_t n_bonds = -1, n_sites = 0;
    int shift = 0;
    int32_t* answer = nullptr;                     // two words of the thread's pinned block: [0] the probe's answer, -1 until
                                                   // the copy has landed; [1] how often the chunk pool ran dry on this bond
                                                   // list (written by the device: the pool of the next call is doubled that
                                                   // many times)
};
// Per host thread: four remembered bond lists, and ONE pinned block of kHintPairs answer pairs handed out round robin,
// so that a copy or a device-side store still in flight for a forgotten entry lands in a pair that is not handed out
// again until kHintPairs - 4 further bond lists have been seen (it could only cost speed, never a result).  The block
// is released when the thread exits.
constexpr int kHintPairs = 64;
struct HintStore {
    ProbeHint slot[4];
    int next_slot = 0, next_pair = 0;
    int32_t* pinned = nullptr;
    ~HintStore() { if (pinned) { cudaFreeHost(pinned); pinned = nullptr; } }    // (fails harmlessly once the runtime is gone)
};
static thread_local HintStore g_hints;

static ProbeHint* hint_find(const void* src, const void* dst, int64_t n_bonds, int64_t n_sites, int shift)
{
    for (ProbeHint& h : g_hints.slot)
        if (h.answer && h.src == src && h.dst == dst && h.n_bonds == n_bonds && h.n_sites == n_sites && h.shift == shift) return &h;
    return nullptr;
}

// ccl_set_option("probe_cache" | "reset"): what this host thread remembers about bond lists is forgotten (the pinned
// block is kept for reuse)
void forget_probe_hints()
{
    for (ProbeHint& h : g_hints.slot) { h.src = nullptr; h.dst = nullptr; h.n_bonds = -1; h.answer = nullptr; }
}

static ProbeHint* hint_new(const void* src, const void* dst, int64_t n_bonds, int64_t n_sites, int shift)
{
    HintStore& hs = g_hints;
    if (hs.pinned == nullptr && cudaHostAlloc(reinterpret_cast<void**>(&hs.pinned), kHintPairs * 2 * sizeof(int32_t), cudaHostAllocDefault) != cudaSuccess) {
        hs.pinned = nullptr;
        cudaGetLastError();
        return nullptr;
    }
    ProbeHint& h = hs.slot[hs.next_slot];
    hs.next_slot = (hs.next_slot + 1) % 4;
    h.answer = hs.pinned + 2 * hs.next_pair;
    hs.next_pair = (hs.next_pair + 1) % kHintPairs;
    reinterpret_cast<volatile int32_t*>(h.answer)[0] = -1;
    reinterpret_cast<volatile int32_t*>(h.answer)[1] = 0;
    h.src = src; h.dst = dst; h.n_bonds = n_bonds; h.n_sites = n_sites; h.shift = shift;
    return &h;
}

static int label_impl(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst, const void* occ,
                      int mask_kind, int32_t* labels, cudaStream_t st)
{
    int rc = check_args(n_sites, n_bonds, src, dst, labels);
    if (rc != CCL_OK) return rc;
    if (n_sites == 0) return CCL_OK;
    CCL_REQUIRE((reinterpret_cast<uintptr_t>(labels) & 15) == 0, "labels must be 16-byte aligned");
    CCL_REQUIRE(mask_kind != 2 || (reinterpret_cast<uintptr_t>(occ) & 3) == 0, "occupied_bits is not 4-byte aligned");
    const Tuning t = tuning();                             // one snapshot per call

    // Which form of step (iii)?  0 = direct kernels, 1 = region-bucketed, -1 = a device-side probe decides.
    int mode = 0;
    BucketPlan plan;
    void* bucket_ws = nullptr;
    ProbeHint* hint = nullptr;
    bool report_probe = false;
    const bool eligible = n_bonds > 0 && t.force_mode != 0 && n_sites * (int64_t)sizeof(int32_t) >= t.bucket_min_label_bytes &&
                          n_bonds >= t.bucket_min_bonds;
    int pool_doublings = 0;
    if (eligible) {
        mode = t.force_mode == 1 ? 1 : -1;
        if (t.probe_cache) {
            const int shift = bucket_region_shift(n_sites, t);
            hint = hint_find(src, dst, n_bonds, n_sites, shift);
            if (hint == nullptr) hint = hint_new(src, dst, n_bonds, n_sites, shift);
            if (hint) {
                const int32_t ans = reinterpret_cast<volatile int32_t*>(hint->answer)[0];
                if (mode < 0 && (ans == 0 || ans == 1)) mode = ans;
                pool_doublings = reinterpret_cast<volatile int32_t*>(hint->answer)[1];
                // no answer yet (first call, or earlier calls were forced or failed before the copy): ask for it again
                report_probe = mode < 0;
            }
        }
        // The bucketed form is an optimisation: the direct kernels need no workspace.  Nothing is drawn when the remembered
        // answer is "direct", and when the pool cannot supply the workspace the call goes on with the direct kernels (and
        // the next call on this bond list asks for a pool half as large again).
        if (mode != 0) {
            rc = bucketed_begin(n_sites, n_bonds, t, pool_doublings, st, &plan, &bucket_ws);
            if (rc != CCL_OK) {
                cudaGetLastError();
                if (bucket_ws) { cudaFreeAsync(bucket_ws, st); bucket_ws = nullptr; }
                if (hint && pool_doublings > 0) reinterpret_cast<volatile int32_t*>(hint->answer)[1] = pool_doublings - 1;
                plan = BucketPlan();
                mode = 0;
                report_probe = false;
            }
        }
    }
    auto done = [&](int code) { if (bucket_ws) cudaFreeAsync(bucket_ws, st); return code; };
    const int gate = mode < 0 ? kGateDirectOrOverflow : kGateOverflow;

    // ---- step (i); step (ii) has nothing to do after label[i] = i (every site is a root)
    if (mode != 1) {
        ProbeJob job;
        if (mode < 0) { job.hdr = plan.hdr; job.n_bonds = n_bonds; job.src = src; job.dst = dst; job.shift = plan.shift; }
        const int64_t site_blocks = (((n_sites + 3) / 4) + kThreads - 1) / kThreads;
        const int64_t init_blocks = site_blocks < (int64_t)sm_count() * 32 ? site_blocks : (int64_t)sm_count() * 32;
        k_init<<<(unsigned)init_blocks, kThreads, 0, st>>>(n_sites, labels, job);                // (+ the probe)
        { cudaError_t e = cudaGetLastError(); if (e != cudaSuccess) { set_error("launch of k_init failed: %s", cudaGetErrorString(e)); return done(CCL_CUDA_ERROR); } count_launch(); }
        mark(0, st);
    }
    if (n_bonds > 0) {
        // ---- step (iii)
        if (mode != 0) {
            plan.lazy_init = mode == 1;                    // step (i) region by region inside the bucketed kernels
            plan.gated = mode < 0;
            if (mode == 1) mark(0, st);                    // no separate initialization pass to time
            rc = bucketed_launch(plan, n_sites, n_bonds, src, dst, occ, mask_kind, labels, st);
            if (rc != CCL_OK) return done(rc);
        }
        // The direct kernels: the whole of step (iii) in direct mode; behind the bucketed kernels they return at once
        // unless the probe chose them (mode < 0) or the chunk pool ran dry.  Two passes pay where most bonds close
        // cycles (many bonds per site: triangular lattice); with 1.5-2 bonds per site they are neutral or slower.
        const BucketHeader* hdr = mode != 0 ? plan.hdr : nullptr;
        const int g = mode != 0 ? gate : kGateNone;
        const bool two_pass = mode != 1 && (t.two_pass > 0 || (t.two_pass < 0 && n_bonds >= (1 << 20) && 2 * n_bonds >= 5 * n_sites));
        if (two_pass) {
            if (occ == nullptr) rc = launch_two_pass<0>(n_sites, n_bonds, src, dst, nullptr, labels, hdr, g, st);
            else if (mask_kind == 1) rc = launch_two_pass<1>(n_sites, n_bonds, src, dst, occ, labels, hdr, g, st);
            else rc = launch_two_pass<2>(n_sites, n_bonds, src, dst, occ, labels, hdr, g, st);
        } else {
            // (the safety net reports a dry pool to the host: the next call on this bond list doubles it, up to 8 x)
            int32_t* notify = (hint != nullptr && mode != 0 && t.bucket_capacity <= 0 && pool_doublings < 3) ? hint->answer + 1 : nullptr;
            if (occ == nullptr) rc = launch_reduce<0>(n_bonds, src, dst, nullptr, labels, hdr, g, st, notify, pool_doublings + 1);
            else if (mask_kind == 1) rc = launch_reduce<1>(n_bonds, src, dst, occ, labels, hdr, g, st, notify, pool_doublings + 1);
            else rc = launch_reduce<2>(n_bonds, src, dst, occ, labels, hdr, g, st, notify, pool_doublings + 1);
        }
        if (rc != CCL_OK) return done(rc);
        mark(1, st);
        // ---- step (iv)
        rc = flatten_all(n_sites, labels, mode != 0, t, st);
        if (rc != CCL_OK) return done(rc);
        mark(2, st);
        if (report_probe && cudaMemcpyAsync(hint->answer, &plan.hdr->mode, sizeof(int32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess)
            cudaGetLastError();                            // a hint only
    } else {
        mark(1, st); mark(2, st);
    }
    return done(CCL_OK);
}

}  // namespace ccl

extern "C" int ccl_label(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                         const uint8_t* occupied, int32_t* labels, void* stream)
{
    return ccl::label_impl(n_sites, n_bonds, src, dst, occupied, 1, labels, ccl::as_stream(stream));
}

extern "C" int ccl_label_bits(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                              const uint32_t* occupied_bits, int32_t* labels, void* stream)
{
    return ccl::label_impl(n_sites, n_bonds, src, dst, occupied_bits, 2, labels, ccl::as_stream(stream));
}

extern "C" int ccl_set_profile_events(void* after_init, void* after_reduce, void* after_flatten)
{
    ccl::g_ev[0] = static_cast<cudaEvent_t>(after_init);
    ccl::g_ev[1] = static_cast<cudaEvent_t>(after_reduce);
    ccl::g_ev[2] = static_cast<cudaEvent_t>(after_flatten);
    return CCL_OK;
}

extern "C" int ccl_validate_bonds(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                                  int64_t* out_bad, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_sites >= 0 && n_bonds >= 0, "negative count");
    CCL_REQUIRE(out_bad != nullptr, "out_bad is NULL");
    CCL_REQUIRE(n_bonds == 0 || (src && dst), "src/dst is NULL with n_bonds > 0");
    cudaStream_t st = as_stream(stream);
    CCL_CUDA_TRY(cudaMemsetAsync(out_bad, 0, sizeof(int64_t), st));
    if (n_bonds == 0) return CCL_OK;
    int64_t blocks = (n_bonds + kThreads - 1) / kThreads;
    if (blocks > (int64_t)sm_count() * 16) blocks = (int64_t)sm_count() * 16;
    k_validate<<<(unsigned)blocks, kThreads, 0, st>>>(n_sites, n_bonds, src, dst,
                                                      reinterpret_cast<unsigned long long*>(out_bad));
    CCL_CHECK_LAUNCH("k_validate");
    return CCL_OK;
}

extern "C" int ccl_label_bits_host(int64_t n_sites, int64_t n_bonds, const int32_t* host_src,
                                   const int32_t* host_dst, const uint32_t* host_occupied_bits,
                                   int32_t* host_labels, void* stream)
{
    using namespace ccl;
    int rc = check_args(n_sites, n_bonds, host_src, host_dst, host_labels);
    if (rc != CCL_OK) return rc;
    if (n_sites == 0) return CCL_OK;
    cudaStream_t st = as_stream(stream);
    const size_t bond_bytes = (size_t)n_bonds * sizeof(int32_t);
    const size_t mask_bytes = host_occupied_bits ? (size_t)((n_bonds + 31) / 32) * sizeof(uint32_t) : 0;
    const size_t label_bytes = (size_t)n_sites * sizeof(int32_t);
    int32_t *d_src = nullptr, *d_dst = nullptr, *d_labels = nullptr;
    uint32_t* d_bits = nullptr;
    auto run = [&]() -> int {                              // every exit goes through the one cleanup below
        int r;
        if ((r = scratch_alloc((void**)&d_labels, label_bytes, st)) != CCL_OK) return r;
        if (n_bonds > 0) {
            if ((r = scratch_alloc((void**)&d_src, bond_bytes, st)) != CCL_OK) return r;
            if ((r = scratch_alloc((void**)&d_dst, bond_bytes, st)) != CCL_OK) return r;
            CCL_CUDA_TRY(cudaMemcpyAsync(d_src, host_src, bond_bytes, cudaMemcpyHostToDevice, st));
            CCL_CUDA_TRY(cudaMemcpyAsync(d_dst, host_dst, bond_bytes, cudaMemcpyHostToDevice, st));
            if (mask_bytes) {
                if ((r = scratch_alloc((void**)&d_bits, mask_bytes, st)) != CCL_OK) return r;
                CCL_CUDA_TRY(cudaMemcpyAsync(d_bits, host_occupied_bits, mask_bytes, cudaMemcpyHostToDevice, st));
            }
        }
        if ((r = label_impl(n_sites, n_bonds, d_src, d_dst, d_bits, 2, d_labels, st)) != CCL_OK) return r;
        CCL_CUDA_TRY(cudaMemcpyAsync(host_labels, d_labels, label_bytes, cudaMemcpyDeviceToHost, st));
        return CCL_OK;
    };
    rc = run();
    if (d_bits) cudaFreeAsync(d_bits, st);
    if (d_dst) cudaFreeAsync(d_dst, st);
    if (d_src) cudaFreeAsync(d_src, st);
    if (d_labels) cudaFreeAsync(d_labels, st);
    const cudaError_t e = cudaStreamSynchronize(st);
    if (rc == CCL_OK && e != cudaSuccess) { set_error("cudaStreamSynchronize failed: %s", cudaGetErrorString(e)); rc = CCL_CUDA_ERROR; }
    return rc;
}

// An occupancy sweep over one bond list with HOST buffers: the bond list crosses PCIe once, and the labels of mask k
// travel back on a second stream while mask k+1 is being labeled (two label buffers on the device).
extern "C" int ccl_label_sweep_host(int64_t n_sites, int64_t n_bonds, const int32_t* host_src, const int32_t* host_dst,
                                    int32_t n_masks, const uint32_t* const* host_occupied_bits, int32_t* const* host_labels,
                                    void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_masks >= 0, "n_masks < 0");
    CCL_REQUIRE(n_masks == 0 || (host_occupied_bits != nullptr && host_labels != nullptr), "mask / label pointer array is NULL");
    if (n_masks == 0) return CCL_OK;
    int rc = check_args(n_sites, n_bonds, host_src, host_dst, host_labels[0]);
    if (rc != CCL_OK) return rc;
    for (int k = 0; k < n_masks; ++k) CCL_REQUIRE(n_sites == 0 || host_labels[k] != nullptr, "a host_labels entry is NULL");
    if (n_sites == 0) return CCL_OK;
    cudaStream_t st = as_stream(stream);
    const size_t bond_bytes = (size_t)n_bonds * sizeof(int32_t);
    const size_t mask_bytes = (size_t)((n_bonds + 31) / 32) * sizeof(uint32_t);
    const size_t label_bytes = (size_t)n_sites * sizeof(int32_t);
    int32_t *d_src = nullptr, *d_dst = nullptr, *d_labels[2] = {nullptr, nullptr};
    uint32_t* d_bits[2] = {nullptr, nullptr};
    cudaStream_t side = nullptr;
    cudaEvent_t labeled[2] = {nullptr, nullptr}, copied[2] = {nullptr, nullptr};
    auto cleanup = [&]() {
        if (side) cudaStreamSynchronize(side);            // a copy may still be reading a label buffer
        for (int j = 0; j < 2; ++j) {
            if (d_bits[j]) cudaFreeAsync(d_bits[j], st);
            if (d_labels[j]) cudaFreeAsync(d_labels[j], st);
        }
        if (d_dst) cudaFreeAsync(d_dst, st);
        if (d_src) cudaFreeAsync(d_src, st);
        cudaStreamSynchronize(st);
        for (int j = 0; j < 2; ++j) { if (labeled[j]) cudaEventDestroy(labeled[j]); if (copied[j]) cudaEventDestroy(copied[j]); }
        if (side) cudaStreamDestroy(side);
    };
#define SWEEP_TRY(expr)                                                                             \
    do {                                                                                            \
        cudaError_t e__ = (expr);                                                                   \
        if (e__ != cudaSuccess) { set_error("%s failed: %s", #expr, cudaGetErrorString(e__)); cleanup(); return CCL_CUDA_ERROR; } \
    } while (0)
    SWEEP_TRY(cudaStreamCreateWithFlags(&side, cudaStreamNonBlocking));
    for (int j = 0; j < 2; ++j) {
        SWEEP_TRY(cudaEventCreateWithFlags(&labeled[j], cudaEventDisableTiming));
        SWEEP_TRY(cudaEventCreateWithFlags(&copied[j], cudaEventDisableTiming));
        if ((rc = scratch_alloc((void**)&d_labels[j], label_bytes, st)) != CCL_OK) { cleanup(); return rc; }
        if (n_bonds > 0 && (rc = scratch_alloc((void**)&d_bits[j], mask_bytes, st)) != CCL_OK) { cleanup(); return rc; }
    }
    if (n_bonds > 0) {
        if ((rc = scratch_alloc((void**)&d_src, bond_bytes, st)) != CCL_OK) { cleanup(); return rc; }
        if ((rc = scratch_alloc((void**)&d_dst, bond_bytes, st)) != CCL_OK) { cleanup(); return rc; }
        SWEEP_TRY(cudaMemcpyAsync(d_src, host_src, bond_bytes, cudaMemcpyHostToDevice, st));
        SWEEP_TRY(cudaMemcpyAsync(d_dst, host_dst, bond_bytes, cudaMemcpyHostToDevice, st));
    }
    for (int k = 0; k < n_masks; ++k) {
        const int j = k & 1;
        const uint32_t* bits = nullptr;
        if (n_bonds > 0 && host_occupied_bits[k] != nullptr) {
            SWEEP_TRY(cudaMemcpyAsync(d_bits[j], host_occupied_bits[k], mask_bytes, cudaMemcpyHostToDevice, st));
            bits = d_bits[j];
        }
        if (k >= 2) SWEEP_TRY(cudaStreamWaitEvent(st, copied[j], 0));        // label buffer j is free again
        rc = label_impl(n_sites, n_bonds, d_src, d_dst, bits, 2, d_labels[j], st);
        if (rc != CCL_OK) { cleanup(); return rc; }
        SWEEP_TRY(cudaEventRecord(labeled[j], st));
        SWEEP_TRY(cudaStreamWaitEvent(side, labeled[j], 0));
        SWEEP_TRY(cudaMemcpyAsync(host_labels[k], d_labels[j], label_bytes, cudaMemcpyDeviceToHost, side));
        SWEEP_TRY(cudaEventRecord(copied[j], side));
    }
    for (int j = 0; j < 2 && j < n_masks; ++j) SWEEP_TRY(cudaStreamWaitEvent(st, copied[j], 0));
#undef SWEEP_TRY
    cleanup();                                            // frees in stream order, synchronises, destroys the side stream
    return CCL_OK;
}

