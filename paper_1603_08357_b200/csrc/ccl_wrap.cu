// ccl_wrap.cu -- wrapping detection on periodic lattices (reading R7 of the paper's "spanning probability",
// PAPER.md:157,171): does some cluster hold a closed path with non-zero winding number?
//
// Every bond carries its wrap vector (wx, wy) in {-1,0,1}^2: how many times it crosses the periodic seam going from
// src to dst.  Method (SURVEY.md 8(c) point 7):
//   1. label the OPEN lattice -- occupied bonds with a zero wrap vector only -- with the ordinary hot path
//      (ccl_label_bits).  Inside an open cluster every site has a well-defined sheet, so no cycle winds.
//   2. the occupied seam bonds (O(L) of them) form a small graph on the open clusters, edge weight = wrap vector.
//      A weighted union-find over it keeps, for every open cluster, its sheet offset to its root; a seam bond whose two
//      clusters already share a root closes a cycle, whose winding is the mismatch of the offsets.
// Step 2 is lock-free: node[c] = parent (32 bits) | offset x (16) | offset y (16) in one 64-bit word, linked with
// atomicCAS from the self-pointing state; a node's word is written once (when it stops being a root) and never
// again, so offsets summed along a path are consistent whenever they are read.
//
// Checking only "a seam bond joins two sites of one open cluster" is not enough (a winding cycle may need several
// crossings; it misses 22-24 % of the wrapping realizations at p_c).  Product code: no oracle code here.
#include "ccl_common.cuh"

namespace ccl {

constexpr int kWrapThreads = 256;

__device__ __forceinline__ unsigned long long pack_node(int32_t parent, int ox, int oy)
{
    return ((unsigned long long)(uint32_t)parent << 32) | ((unsigned long long)(uint16_t)(int16_t)ox << 16) |
           (unsigned long long)(uint16_t)(int16_t)oy;
}

// bits_open = occupied & (wrap vector == 0); seam bonds are counted (for the caller's information)
__global__ void __launch_bounds__(kWrapThreads)
k_open_mask(int64_t n_bonds, const uint32_t* __restrict__ bits, const int8_t* __restrict__ wx,
            const int8_t* __restrict__ wy, uint32_t* __restrict__ bits_open)
{
    const int64_t words = (n_bonds + 31) / 32;
    const int64_t stride = (int64_t)gridDim.x * kWrapThreads;
    for (int64_t w = (int64_t)blockIdx.x * kWrapThreads + threadIdx.x; w < words; w += stride) {
        uint32_t occ = bits ? bits[w] : 0xFFFFFFFFu;
        uint32_t seam = 0;
        const int64_t b0 = w * 32;
        if (b0 + 32 <= n_bonds) {
            const int4* px = reinterpret_cast<const int4*>(wx + b0);      // wx, wy are 16-byte aligned (checked on the host)
            const int4* py = reinterpret_cast<const int4*>(wy + b0);
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const int4 a = px[q], c = py[q];
                const uint32_t v[4] = {(uint32_t)(a.x | c.x), (uint32_t)(a.y | c.y), (uint32_t)(a.z | c.z), (uint32_t)(a.w | c.w)};
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        if ((v[j] >> (8 * k)) & 0xFFu) seam |= 1u << (q * 16 + j * 4 + k);
            }
        } else {
            for (int k = 0; k < 32 && b0 + k < n_bonds; ++k)
                if (wx[b0 + k] | wy[b0 + k]) seam |= 1u << k;
            occ &= (n_bonds - b0 >= 32) ? 0xFFFFFFFFu : ((1u << (n_bonds - b0)) - 1u);
        }
        bits_open[w] = occ & ~seam;
    }
}

// Calls f(b, wx, wy) for every occupied bond with a non-zero wrap vector.  The wrap vectors are read 16 bonds at a time
// (two 128-bit loads, the arrays are 16-byte aligned); on a lattice all but O(L) of the groups are zero and end there.
template <typename F>
__device__ __forceinline__ void for_each_occupied_seam_bond(int64_t n_bonds, const uint32_t* __restrict__ bits,
                                                            const int8_t* __restrict__ wx, const int8_t* __restrict__ wy, F f)
{
    const int64_t groups = (n_bonds + 15) / 16;
    const int64_t stride = (int64_t)gridDim.x * kWrapThreads;
    for (int64_t g = (int64_t)blockIdx.x * kWrapThreads + threadIdx.x; g < groups; g += stride) {
        const int64_t b0 = g * 16;
        if (b0 + 16 <= n_bonds) {
            const int4 a = *reinterpret_cast<const int4*>(wx + b0), c = *reinterpret_cast<const int4*>(wy + b0);
            if ((a.x | a.y | a.z | a.w | c.x | c.y | c.z | c.w) == 0) continue;
        }
        const int64_t b1 = b0 + 16 < n_bonds ? b0 + 16 : n_bonds;
        for (int64_t b = b0; b < b1; ++b) {
            const int x = wx[b], y = wy[b];
            if ((x | y) == 0) continue;
            if (bits && !((bits[b >> 5] >> (b & 31)) & 1u)) continue;
            f(b, x, y);
        }
    }
}

__global__ void __launch_bounds__(kWrapThreads)
k_wrap_init(int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
            const uint32_t* __restrict__ bits, const int8_t* __restrict__ wx, const int8_t* __restrict__ wy,
            const int32_t* __restrict__ label, unsigned long long* node)
{
    for_each_occupied_seam_bond(n_bonds, bits, wx, wy, [&](int64_t b, int, int) {
        const int32_t cu = label[src[b]], cv = label[dst[b]];
        node[cu] = pack_node(cu, 0, 0);                      // every writer writes the same value
        node[cv] = pack_node(cv, 0, 0);
    });
}

// root of c and (ox, oy) = sheet(c) - sheet(root)
__device__ __forceinline__ int32_t wrap_find(const unsigned long long* node, int32_t c, int& ox, int& oy)
{
    ox = 0; oy = 0;
    for (;;) {
        const unsigned long long w = *reinterpret_cast<const volatile unsigned long long*>(node + c);
        const int32_t p = (int32_t)(w >> 32);
        if (p == c) return c;
        ox += (int16_t)(uint16_t)(w >> 16);
        oy += (int16_t)(uint16_t)w;
        c = p;
    }
}

__global__ void __launch_bounds__(kWrapThreads)
k_wrap_union(int64_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
             const uint32_t* __restrict__ bits, const int8_t* __restrict__ wx, const int8_t* __restrict__ wy,
             const int32_t* __restrict__ label, unsigned long long* node, int32_t* out)
{
    for_each_occupied_seam_bond(n_bonds, bits, wx, wy, [&](int64_t b, int dx, int dy) {
        const int32_t cu = label[src[b]], cv = label[dst[b]];
        for (;;) {
            int ux, uy, vx, vy;
            const int32_t ru = wrap_find(node, cu, ux, uy);
            const int32_t rv = wrap_find(node, cv, vx, vy);
            // the bond says sheet(cv) = sheet(cu) + (dx, dy)
            const int mx = ux + dx - vx, my = uy + dy - vy;   // = sheet(rv) - sheet(ru) if the two roots get joined
            if (ru == rv) {
                if (mx) atomicOr(out + 0, 1);                 // the cycle this bond closes winds mx times in x
                if (my) atomicOr(out + 1, 1);
                return;
            }
            if (mx > 32000 || mx < -32000 || my > 32000 || my < -32000) { atomicOr(out + 2, 1); return; }   // 16-bit offsets
            // hang the higher root under the lower one (the CAS succeeds only if it is still a root)
            const int32_t hi = ru > rv ? ru : rv, lo = ru > rv ? rv : ru;
            const unsigned long long want = ru > rv ? pack_node(lo, -mx, -my) : pack_node(lo, mx, my);
            if (atomicCAS(node + hi, pack_node(hi, 0, 0), want) == pack_node(hi, 0, 0)) return;
        }
    });
}

}  // namespace ccl

extern "C" int ccl_wrap(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                        const uint32_t* occupied_bits, const int8_t* wx, const int8_t* wy, int32_t* labels_open,
                        int32_t* out, void* workspace, size_t* workspace_bytes, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_sites >= 0 && n_sites <= 2147483647LL && n_bonds >= 0, "count out of range");
    CCL_REQUIRE(workspace_bytes != nullptr, "workspace_bytes is NULL");
    const size_t mask_bytes = (((size_t)((n_bonds + 31) / 32) * 4) + 255) & ~(size_t)255;
    const size_t need = mask_bytes + (size_t)n_sites * sizeof(unsigned long long) + 256;
    if (workspace == nullptr) { *workspace_bytes = need; return CCL_OK; }
    if (*workspace_bytes < need) { set_error("workspace too small: %zu < %zu", *workspace_bytes, need); return CCL_WORKSPACE_TOO_SMALL; }
    CCL_REQUIRE(out != nullptr, "out is NULL");
    CCL_REQUIRE(n_sites == 0 || labels_open != nullptr, "labels_open is NULL");
    CCL_REQUIRE(n_bonds == 0 || (src && dst && wx && wy), "src/dst/wx/wy is NULL with n_bonds > 0");
    CCL_REQUIRE(((reinterpret_cast<uintptr_t>(wx) | reinterpret_cast<uintptr_t>(wy)) & 15) == 0, "wx/wy must be 16-byte aligned");
    CCL_REQUIRE((reinterpret_cast<uintptr_t>(workspace) & 255) == 0, "workspace must be 256-byte aligned");
    cudaStream_t st = as_stream(stream);
    CCL_CUDA_TRY(cudaMemsetAsync(out, 0, 4 * sizeof(int32_t), st));
    uint32_t* bits_open = static_cast<uint32_t*>(workspace);
    unsigned long long* node = reinterpret_cast<unsigned long long*>(static_cast<char*>(workspace) + mask_bytes);
    int64_t blocks = ((n_bonds + 31) / 32 + kWrapThreads - 1) / kWrapThreads;
    if (blocks > (int64_t)sm_count() * 16) blocks = (int64_t)sm_count() * 16;
    if (n_bonds > 0) {
        k_open_mask<<<(unsigned)blocks, kWrapThreads, 0, st>>>(n_bonds, occupied_bits, wx, wy, bits_open);
        CCL_CHECK_LAUNCH("k_open_mask");
    }
    const int rc = ccl_label_bits(n_sites, n_bonds, src, dst, bits_open, labels_open, stream);
    if (rc != CCL_OK || n_bonds == 0) return rc;
    blocks = ((n_bonds + 15) / 16 + kWrapThreads - 1) / kWrapThreads;
    if (blocks > (int64_t)sm_count() * 16) blocks = (int64_t)sm_count() * 16;
    k_wrap_init<<<(unsigned)blocks, kWrapThreads, 0, st>>>(n_bonds, src, dst, occupied_bits, wx, wy, labels_open, node);
    CCL_CHECK_LAUNCH("k_wrap_init");
    k_wrap_union<<<(unsigned)blocks, kWrapThreads, 0, st>>>(n_bonds, src, dst, occupied_bits, wx, wy, labels_open, node, out);
    CCL_CHECK_LAUNCH("k_wrap_union");
    return CCL_OK;
}
