// ccl_bonds.cuh -- streaming load of four consecutive bonds and their occupancy bits, shared by the kernels that read
// the bond list (ccl_label.cu).  Product code.
#pragma once

#include "ccl_common.cuh"

namespace ccl {

// Bonds of one thread and tile: 4 consecutive bonds, mask in the low 4 bits of m.
struct Bonds4 {
    int32_t u[4], v[4];
    uint32_t m;
};

// Loaded in two halves, so that a kernel can fetch the occupancy bits of its NEXT four bonds while it works on the
// current ones: the mask word and the endpoints are two dependent trips to HBM otherwise (the endpoints of a group
// without an occupied bond are never fetched).
template <int MASK>
__device__ __forceinline__ uint32_t load_mask4(int64_t n_bonds, int64_t b0, const void* __restrict__ occ, int vec, uint64_t pol)
{
    if (b0 >= n_bonds) return 0;
    const int cnt = (n_bonds - b0 >= 4) ? 4 : (int)(n_bonds - b0);
    uint32_t m = 0xFu;
    if (MASK == 2) {
        m = (ld_stream_u32(static_cast<const uint32_t*>(occ) + (b0 >> 5), pol) >> (b0 & 31)) & 0xFu;
    } else if (MASK == 1) {
        const uint8_t* o = static_cast<const uint8_t*>(occ) + b0;
        if (vec && cnt == 4) {
            const uint32_t w = ld_stream_u32(reinterpret_cast<const uint32_t*>(o), pol);
            m = ((w & 0xFFu) != 0) | (((w & 0xFF00u) != 0) << 1) | (((w & 0xFF0000u) != 0) << 2) |
                (((w & 0xFF000000u) != 0) << 3);
        } else {
            m = 0;
            for (int k = 0; k < cnt; ++k) m |= (uint32_t)(ld_stream_u8(o + k, pol) != 0) << k;
        }
    }
    return m & ((1u << cnt) - 1u);
}

__device__ __forceinline__ Bonds4 load_ends4(int64_t n_bonds, int64_t b0, uint32_t m, const int32_t* __restrict__ src,
                                             const int32_t* __restrict__ dst, int vec, uint64_t pol)
{
    Bonds4 r;
    r.m = m;
#pragma unroll
    for (int k = 0; k < 4; ++k) { r.u[k] = 0; r.v[k] = 0; }
    if (m == 0) return r;                                  // (also: b0 >= n_bonds)
    const int cnt = (n_bonds - b0 >= 4) ? 4 : (int)(n_bonds - b0);
    if (vec && cnt == 4) {
        const int4 s = ld_stream_v4(src + b0, pol), d = ld_stream_v4(dst + b0, pol);
        r.u[0] = s.x; r.u[1] = s.y; r.u[2] = s.z; r.u[3] = s.w;
        r.v[0] = d.x; r.v[1] = d.y; r.v[2] = d.z; r.v[3] = d.w;
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (k < cnt) { r.u[k] = ld_stream_s32(src + b0 + k, pol); r.v[k] = ld_stream_s32(dst + b0 + k, pol); }
    }
    return r;
}

}  // namespace ccl
