// ccl_gen.cu -- seeded device generators of the benchmark workloads (include/ccl.h: ccl_gen_*; DESIGN.md "Input
// recipe").  Outside the timed metric.  The paper prepares its NN list "in advance" and draws bonds
// with probability p; lattice geometry, numbering and the RNG are this project's (readings R9, R10).
#include <cub/cub.cuh>

#include "ccl_common.cuh"

namespace ccl {

constexpr int kGenThreads = 256;

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): ten rounds of two 32x32->64 multiplies, key bumped by the
// Weyl constants between rounds.
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

// ---------------------------------------------------------------------------------------------- lattices
__global__ void __launch_bounds__(kGenThreads)
k_gen_triangular(int32_t L, int32_t* __restrict__ src, int32_t* __restrict__ dst)
{
    const int64_t n_bonds = 3ll * L * L;
    const int64_t stride = (int64_t)gridDim.x * kGenThreads;
    for (int64_t b = (int64_t)blockIdx.x * kGenThreads + threadIdx.x; b < n_bonds; b += stride) {
        const int64_t s = b / 3;
        const int k = (int)(b - 3 * s);
        const int32_t y = (int32_t)(s / L), x = (int32_t)(s - (int64_t)y * L);
        const int32_t xx = (k != 1) ? (x + 1 == L ? 0 : x + 1) : x;       // k = 0: (x+1,y); 1: (x,y+1); 2: (x+1,y+1)
        const int32_t yy = (k != 0) ? (y + 1 == L ? 0 : y + 1) : y;
        src[b] = (int32_t)s;
        dst[b] = (int32_t)((int64_t)yy * L + xx);
    }
}

__global__ void __launch_bounds__(kGenThreads)
k_gen_honeycomb(int32_t L, int32_t* __restrict__ src, int32_t* __restrict__ dst)
{
    const int64_t n_bonds = 3ll * L * L;
    const int64_t stride = (int64_t)gridDim.x * kGenThreads;
    for (int64_t b = (int64_t)blockIdx.x * kGenThreads + threadIdx.x; b < n_bonds; b += stride) {
        const int64_t c = b / 3;
        const int k = (int)(b - 3 * c);
        const int32_t y = (int32_t)(c / L), x = (int32_t)(c - (int64_t)y * L);
        int64_t other = c;                                                 // k = 0: A(c) - B(c)
        if (k == 1) other = (int64_t)y * L + (x + 1 == L ? 0 : x + 1);     // B(c) - A(x+1, y)
        if (k == 2) other = (int64_t)(y + 1 == L ? 0 : y + 1) * L + x;     // B(c) - A(x, y+1)
        src[b] = (int32_t)(k == 0 ? 2 * c : 2 * c + 1);
        dst[b] = (int32_t)(k == 0 ? 2 * c + 1 : 2 * other);
    }
}

// --------------------------------------------------------------------------------------------- occupancy
// One thread per 32 bonds = one word of the packed mask = 8 Philox calls.
__global__ void __launch_bounds__(kGenThreads)
k_gen_occupancy(int64_t n_bonds, uint32_t threshold, int all, uint2 key, uint32_t realization,
                uint8_t* __restrict__ mask, uint32_t* __restrict__ bits)
{
    const int64_t n_words = (n_bonds + 31) / 32;
    const int64_t stride = (int64_t)gridDim.x * kGenThreads;
    for (int64_t w = (int64_t)blockIdx.x * kGenThreads + threadIdx.x; w < n_words; w += stride) {
        uint32_t word = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const uint64_t ctr = (uint64_t)w * 8 + q;                      // = b >> 2
            const uint4 r = philox4x32_10(make_uint4((uint32_t)ctr, (uint32_t)(ctr >> 32), realization, 0u), key);
            const uint32_t nib = (uint32_t)(all || r.x < threshold) | ((uint32_t)(all || r.y < threshold) << 1) |
                                 ((uint32_t)(all || r.z < threshold) << 2) | ((uint32_t)(all || r.w < threshold) << 3);
            word |= nib << (4 * q);
        }
        const int64_t b0 = w * 32;
        if (n_bonds - b0 < 32) word &= (1u << (int)(n_bonds - b0)) - 1u;    // bits past n_bonds stay zero
        if (bits) bits[w] = word;
        if (mask) {
            const int cnt = (n_bonds - b0 < 32) ? (int)(n_bonds - b0) : 32;
            for (int j = 0; j < cnt; ++j) mask[b0 + j] = (uint8_t)((word >> j) & 1u);
        }
    }
}

// ------------------------------------------------------------------------------------- random z-regular
__global__ void __launch_bounds__(kGenThreads)
k_stub_keys(int64_t n_stubs, uint2 key, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const int64_t stride = (int64_t)gridDim.x * kGenThreads;
    for (int64_t t = (int64_t)blockIdx.x * kGenThreads + threadIdx.x; t < n_stubs; t += stride) {
        const uint4 r = philox4x32_10(make_uint4((uint32_t)t, (uint32_t)((uint64_t)t >> 32), 0u, 1u), key);
        keys[t] = ((uint64_t)r.x << 32) | r.y;
        vals[t] = (uint32_t)t;
    }
}

__device__ __forceinline__ uint64_t pair_key(int32_t u, int32_t v)
{
    const uint32_t lo = (uint32_t)min(u, v), hi = (uint32_t)max(u, v);
    return ((uint64_t)lo << 32) | hi;
}

// bond k joins the sites of sorted stubs 2k and 2k+1; also emit its unordered-pair key for the duplicate search
__global__ void __launch_bounds__(kGenThreads)
k_pair_stubs(int64_t n_bonds, uint32_t z, const uint32_t* __restrict__ sorted_stub, int32_t* __restrict__ src,
             int32_t* __restrict__ dst, uint64_t* __restrict__ pkeys, uint32_t* __restrict__ pidx)
{
    const int64_t stride = (int64_t)gridDim.x * kGenThreads;
    for (int64_t k = (int64_t)blockIdx.x * kGenThreads + threadIdx.x; k < n_bonds; k += stride) {
        const int32_t u = (int32_t)(sorted_stub[2 * k] / z), v = (int32_t)(sorted_stub[2 * k + 1] / z);
        src[k] = u;
        dst[k] = v;
        pkeys[k] = pair_key(u, v);
        pidx[k] = (uint32_t)k;
    }
}

// defect[k] = 1 for self-loops and for every repeat of an unordered pair after its first occurrence in bond order
// (the sort is stable, so within a run of equal keys the bond indices ascend)
__global__ void __launch_bounds__(kGenThreads)
k_flag_defects(int64_t n_bonds, const uint64_t* __restrict__ sorted_pkeys, const uint32_t* __restrict__ sorted_pidx,
               uint8_t* __restrict__ defect)
{
    const int64_t stride = (int64_t)gridDim.x * kGenThreads;
    for (int64_t i = (int64_t)blockIdx.x * kGenThreads + threadIdx.x; i < n_bonds; i += stride) {
        const uint64_t pk = sorted_pkeys[i];
        const bool loop = (uint32_t)(pk >> 32) == (uint32_t)pk;
        const bool repeat = i > 0 && sorted_pkeys[i - 1] == pk;
        defect[sorted_pidx[i]] = (uint8_t)(loop || repeat);
    }
}

struct RepairState {
    int32_t n_defects;        // written by cub::DeviceSelect
    int32_t n_repaired;
    int32_t overflow;         // overlay capacity exceeded
    int32_t pad;
};

__device__ int64_t count_sorted(const uint64_t* sorted, int64_t n, uint64_t pk)
{
    int64_t lo = 0, hi = n;
    while (lo < hi) { const int64_t mid = (lo + hi) / 2; if (sorted[mid] < pk) lo = mid + 1; else hi = mid; }
    int64_t c = 0;
    while (lo + c < n && sorted[lo + c] == pk) ++c;
    return c;
}

__device__ int64_t multiplicity(const uint64_t* sorted, int64_t n, const uint64_t* removed, const uint64_t* added,
                                int n_overlay, uint64_t pk)
{
    int64_t c = count_sorted(sorted, n, pk);
    for (int i = 0; i < n_overlay; ++i) { c -= (removed[i] == pk); c += (added[i] == pk); }
    return c;
}

// Sequential repair, one thread: defects in ascending bond index, partner bond from Philox(counter = (k lo, k hi,
// attempt, 2)); swap (u_k,v_k),(u_m,v_m) -> (u_k,u_m),(v_k,v_m) when both new bonds are non-loops, distinct and absent.
__global__ void k_repair(int64_t n_bonds, uint2 key, int32_t* src, int32_t* dst, const uint64_t* sorted_pkeys,
                         const int32_t* defect_list, RepairState* state, uint64_t* removed, uint64_t* added,
                         int overlay_cap)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int n_overlay = 0, repaired = 0;
    const int n_defects = state->n_defects;
    for (int d = 0; d < n_defects; ++d) {
        const int64_t k = defect_list[d];
        const uint64_t cur = pair_key(src[k], dst[k]);
        if (src[k] != dst[k] && multiplicity(sorted_pkeys, n_bonds, removed, added, n_overlay, cur) <= 1) continue;
        for (uint32_t attempt = 0;; ++attempt) {
            const uint4 r = philox4x32_10(make_uint4((uint32_t)k, (uint32_t)((uint64_t)k >> 32), attempt, 2u), key);
            const int64_t m = (int64_t)((((uint64_t)r.x << 32) | r.y) % (uint64_t)n_bonds);
            if (m == k) continue;
            const int32_t uk = src[k], vk = dst[k], um = src[m], vm = dst[m];
            if (uk == um || vk == vm) continue;
            const uint64_t a = pair_key(uk, um), b = pair_key(vk, vm);
            if (a == b) continue;
            if (multiplicity(sorted_pkeys, n_bonds, removed, added, n_overlay, a) != 0) continue;
            if (multiplicity(sorted_pkeys, n_bonds, removed, added, n_overlay, b) != 0) continue;
            if (n_overlay + 2 > overlay_cap) { state->overflow = 1; state->n_repaired = repaired; return; }
            removed[n_overlay] = pair_key(uk, vk); added[n_overlay] = a; ++n_overlay;
            removed[n_overlay] = pair_key(um, vm); added[n_overlay] = b; ++n_overlay;
            src[k] = uk; dst[k] = um;
            src[m] = vk; dst[m] = vm;
            ++repaired;
            break;
        }
    }
    state->n_repaired = repaired;
}

static inline size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }
static inline int64_t grid_for(int64_t n) {
    int64_t b = (n + kGenThreads - 1) / kGenThreads;
    const int64_t cap = (int64_t)sm_count() * 16;
    return b < 1 ? 1 : (b > cap ? cap : b);
}

}  // namespace ccl

extern "C" int ccl_gen_triangular(int32_t L, int32_t* src, int32_t* dst, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(L >= 1 && (int64_t)L * L <= 2147483647LL, "L out of range");
    CCL_REQUIRE(src && dst, "src/dst is NULL");
    k_gen_triangular<<<(unsigned)grid_for(3ll * L * L), kGenThreads, 0, as_stream(stream)>>>(L, src, dst);
    CCL_CHECK_LAUNCH("k_gen_triangular");
    return CCL_OK;
}

extern "C" int ccl_gen_honeycomb(int32_t L, int32_t* src, int32_t* dst, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(L >= 1 && 2ll * L * L <= 2147483647LL, "L out of range");
    CCL_REQUIRE(src && dst, "src/dst is NULL");
    k_gen_honeycomb<<<(unsigned)grid_for(3ll * L * L), kGenThreads, 0, as_stream(stream)>>>(L, src, dst);
    CCL_CHECK_LAUNCH("k_gen_honeycomb");
    return CCL_OK;
}

// Wrap vectors of the lattice bonds (how often bond b crosses the periodic seam from src to dst, per axis), in the bond
// order of k_gen_triangular / k_gen_honeycomb.  Input of ccl_wrap.
namespace ccl {
__global__ void __launch_bounds__(kGenThreads)
k_gen_wrap_vectors(int family, int32_t L, int8_t* __restrict__ wx, int8_t* __restrict__ wy)
{
    const int64_t n_bonds = 3ll * L * L;
    const int64_t stride = (int64_t)gridDim.x * kGenThreads;
    for (int64_t b = (int64_t)blockIdx.x * kGenThreads + threadIdx.x; b < n_bonds; b += stride) {
        const int64_t cell = b / 3;
        const int k = (int)(b - 3 * cell);
        const int32_t x = (int32_t)(cell % L), y = (int32_t)(cell / L);
        int sx, sy;                                    // the bond's step in cells
        if (family == 0) { sx = (k != 1); sy = (k != 0); }          // triangular: (1,0), (0,1), (1,1)
        else { sx = (k == 1); sy = (k == 2); }                      // honeycomb: A-B in the cell, B-A(x+1,y), B-A(x,y+1)
        wx[b] = (int8_t)(x + sx >= L);
        wy[b] = (int8_t)(y + sy >= L);
    }
}
}  // namespace ccl

extern "C" int ccl_gen_wrap_vectors(int32_t family, int32_t L, int8_t* wx, int8_t* wy, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(family == 0 || family == 1, "family must be 0 (triangular) or 1 (honeycomb)");
    CCL_REQUIRE(L >= 1 && 2ll * L * L <= 2147483647LL, "L out of range");
    CCL_REQUIRE(wx && wy, "wx/wy is NULL");
    k_gen_wrap_vectors<<<(unsigned)grid_for(3ll * L * L), kGenThreads, 0, as_stream(stream)>>>(family, L, wx, wy);
    CCL_CHECK_LAUNCH("k_gen_wrap_vectors");
    return CCL_OK;
}

// Cayley tree with coordination number 3 (the paper's "Bethe lattice", R11): site 0 has
// children 1, 2, 3; site i >= 1 has children 2i+2, 2i+3.  Bond k joins site k+1 to its parent.
namespace ccl {
__global__ void __launch_bounds__(kGenThreads)
k_gen_cayley3(int64_t n_bonds, const int32_t* __restrict__ perm, int32_t* __restrict__ src, int32_t* __restrict__ dst)
{
    const int64_t stride = (int64_t)gridDim.x * kGenThreads;
    for (int64_t k = (int64_t)blockIdx.x * kGenThreads + threadIdx.x; k < n_bonds; k += stride) {
        const int64_t child = k + 1, parent = child <= 3 ? 0 : (child - 2) / 2;
        src[k] = perm ? perm[parent] : (int32_t)parent;
        dst[k] = perm ? perm[child] : (int32_t)child;
    }
}
}  // namespace ccl

extern "C" int ccl_gen_cayley3(int32_t g, const int32_t* perm_or_null, int32_t* src, int32_t* dst, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(g >= 1 && g <= 28, "g out of range [1, 28]");
    CCL_REQUIRE(src && dst, "src/dst is NULL");
    const int64_t n_bonds = 3 * ((int64_t)1 << g) - 3;
    k_gen_cayley3<<<(unsigned)grid_for(n_bonds), kGenThreads, 0, as_stream(stream)>>>(n_bonds, perm_or_null, src, dst);
    CCL_CHECK_LAUNCH("k_gen_cayley3");
    return CCL_OK;
}

extern "C" int ccl_gen_occupancy(int64_t n_bonds, double p, uint64_t seed, uint32_t realization,
                                 uint8_t* mask_or_null, uint32_t* bits_or_null, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_bonds >= 0, "n_bonds < 0");
    CCL_REQUIRE(p >= 0.0, "p < 0 or NaN");
    CCL_REQUIRE(mask_or_null || bits_or_null, "both outputs are NULL");
    if (n_bonds == 0) return CCL_OK;
    const int all = p >= 1.0;
    const uint32_t threshold = all ? 0u : (uint32_t)(p * 4294967296.0);     // floor(p * 2^32), exact in double
    const uint2 key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
    k_gen_occupancy<<<(unsigned)grid_for((n_bonds + 31) / 32), kGenThreads, 0, as_stream(stream)>>>(
        n_bonds, threshold, all, key, realization, mask_or_null, bits_or_null);
    CCL_CHECK_LAUNCH("k_gen_occupancy");
    return CCL_OK;
}

extern "C" int ccl_gen_regular(int64_t n_sites, int32_t z, uint64_t seed, int32_t* src, int32_t* dst,
                               void* workspace, size_t* workspace_bytes, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_sites >= 1 && z >= 1 && z <= 16, "n_sites < 1 or z outside [1, 16]");
    CCL_REQUIRE(n_sites * z <= 2147483647LL, "n_sites * z > 2^31-1");
    CCL_REQUIRE(((n_sites * z) & 1) == 0, "n_sites * z is odd");
    CCL_REQUIRE(workspace_bytes != nullptr, "workspace_bytes is NULL");
    const int64_t S = n_sites * z, M = S / 2;
    constexpr int kOverlayCap = 4096;
    cudaStream_t st = as_stream(stream);

    // temp storage needed by the three CUB calls (size queries only: no work is enqueued with a NULL temp pointer)
    size_t t_sort_s = 0, t_sort_m = 0, t_sel = 0;
    {
        cub::DoubleBuffer<uint64_t> k(nullptr, nullptr);
        cub::DoubleBuffer<uint32_t> v(nullptr, nullptr);
        CCL_CUDA_TRY(cub::DeviceRadixSort::SortPairs(nullptr, t_sort_s, k, v, S, 0, 64, st));
        CCL_CUDA_TRY(cub::DeviceRadixSort::SortPairs(nullptr, t_sort_m, k, v, M, 0, 64, st));
        CCL_CUDA_TRY(cub::DeviceSelect::Flagged(nullptr, t_sel, cub::CountingInputIterator<int32_t>(0),
                                                (const uint8_t*)nullptr, (int32_t*)nullptr, (int32_t*)nullptr,
                                                (int)M, st));
    }
    size_t t_bytes = t_sort_s > t_sort_m ? t_sort_s : t_sort_m;
    t_bytes = t_bytes > t_sel ? t_bytes : t_sel;

    size_t off = 0;
    const size_t o_keys0 = off; off += align_up(sizeof(uint64_t) * (size_t)S);
    const size_t o_keys1 = off; off += align_up(sizeof(uint64_t) * (size_t)S);
    const size_t o_vals0 = off; off += align_up(sizeof(uint32_t) * (size_t)S);
    const size_t o_vals1 = off; off += align_up(sizeof(uint32_t) * (size_t)S);
    const size_t o_temp = off;  off += align_up(t_bytes);
    const size_t o_flag = off;  off += align_up((size_t)M);
    const size_t o_state = off; off += align_up(sizeof(RepairState));
    const size_t o_rem = off;   off += align_up(sizeof(uint64_t) * kOverlayCap);
    const size_t o_add = off;   off += align_up(sizeof(uint64_t) * kOverlayCap);
    const size_t need = off;

    if (workspace == nullptr) { *workspace_bytes = need; return CCL_OK; }
    if (*workspace_bytes < need) {
        set_error("workspace too small: %zu bytes given, %zu needed", *workspace_bytes, need);
        return CCL_WORKSPACE_TOO_SMALL;
    }
    CCL_REQUIRE(src && dst, "src/dst is NULL");
    CCL_REQUIRE((reinterpret_cast<uintptr_t>(workspace) & 255) == 0, "workspace is not 256-byte aligned");

    char* ws = static_cast<char*>(workspace);
    uint64_t* keys0 = reinterpret_cast<uint64_t*>(ws + o_keys0);
    uint64_t* keys1 = reinterpret_cast<uint64_t*>(ws + o_keys1);
    uint32_t* vals0 = reinterpret_cast<uint32_t*>(ws + o_vals0);
    uint32_t* vals1 = reinterpret_cast<uint32_t*>(ws + o_vals1);
    void* temp = ws + o_temp;
    uint8_t* defect = reinterpret_cast<uint8_t*>(ws + o_flag);
    RepairState* state = reinterpret_cast<RepairState*>(ws + o_state);
    uint64_t* removed = reinterpret_cast<uint64_t*>(ws + o_rem);
    uint64_t* added = reinterpret_cast<uint64_t*>(ws + o_add);
    const uint2 key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));

    CCL_CUDA_TRY(cudaMemsetAsync(state, 0, sizeof(RepairState), st));
    k_stub_keys<<<(unsigned)grid_for(S), kGenThreads, 0, st>>>(S, key, keys0, vals0);
    CCL_CHECK_LAUNCH("k_stub_keys");

    cub::DoubleBuffer<uint64_t> kbuf(keys0, keys1);
    cub::DoubleBuffer<uint32_t> vbuf(vals0, vals1);
    size_t tb = t_bytes;
    CCL_CUDA_TRY(cub::DeviceRadixSort::SortPairs(temp, tb, kbuf, vbuf, S, 0, 64, st));      // stable
    count_launch();

    // pair keys go to the buffers the sort left as scratch; the sorted stub keys are dead from here on
    cub::DoubleBuffer<uint64_t> pk(kbuf.Alternate(), kbuf.Current());
    cub::DoubleBuffer<uint32_t> pi(vbuf.Alternate(), vbuf.Current());
    k_pair_stubs<<<(unsigned)grid_for(M), kGenThreads, 0, st>>>(M, (uint32_t)z, vbuf.Current(), src, dst,
                                                                pk.Current(), pi.Current());
    CCL_CHECK_LAUNCH("k_pair_stubs");
    tb = t_bytes;
    CCL_CUDA_TRY(cub::DeviceRadixSort::SortPairs(temp, tb, pk, pi, M, 0, 64, st));
    count_launch();
    k_flag_defects<<<(unsigned)grid_for(M), kGenThreads, 0, st>>>(M, pk.Current(), pi.Current(), defect);
    CCL_CHECK_LAUNCH("k_flag_defects");
    int32_t* defect_list = reinterpret_cast<int32_t*>(pi.Alternate());
    tb = t_bytes;
    CCL_CUDA_TRY(cub::DeviceSelect::Flagged(temp, tb, cub::CountingInputIterator<int32_t>(0), defect, defect_list,
                                            &state->n_defects, (int)M, st));
    count_launch();
    k_repair<<<1, 32, 0, st>>>(M, key, src, dst, pk.Current(), defect_list, state, removed, added, kOverlayCap);
    CCL_CHECK_LAUNCH("k_repair");

    // The repair is sequential and its overlay is bounded: check it before handing the graph out.  This entry
    // point therefore synchronises the stream (it is a setup call, not part of the timed path).
    RepairState h;
    CCL_CUDA_TRY(cudaMemcpyAsync(&h, state, sizeof(h), cudaMemcpyDeviceToHost, st));
    CCL_CUDA_TRY(cudaStreamSynchronize(st));
    if (h.overflow) {
        set_error("ccl_gen_regular: more than %d endpoint swaps needed (%d defects)", kOverlayCap / 2, h.n_defects);
        return CCL_UNSUPPORTED;
    }
    return CCL_OK;
}
