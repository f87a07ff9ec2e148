// ccl_batch.cu -- the two follow-ups of PAPER.md:115 and SURVEY.md 8(f) NEXT-4:
//
//   ccl_label_batch          many occupancy realizations of one small bond list in ONE launch, one CTA per realization
//                            with the whole label array in shared memory (BASELINE.json config 1 is launch-bound as a
//                            single call; percolation studies average thousands of such realizations).
//   ccl_relabel_sequential   min-site labels -> sequential cluster numbers 0..C-1 ("the method shown in Fig. 4 of
//                            [14]"): flag the roots, exclusive prefix sum, gather.
//
// Product code: nothing under oracle/ is included here or includes this.
#include <cub/cub.cuh>

#include "ccl_common.cuh"
#include "ccl_unionfind.cuh"

namespace ccl {

constexpr int kBatchThreads = 512;
constexpr int kBatchMaxSites = 1 << 15;            // 128 KiB of labels: one CTA's shared memory

// Root of x in the shared-memory forest L (label[x] <= x), halving the path.
__device__ __forceinline__ int32_t smem_root(volatile int32_t* L, int32_t x)
{
    for (;;) {
        const int32_t p = L[x];
        if (p == x) return x;
        const int32_t gp = L[p];
        if (gp == p) return p;
        L[x] = gp;
        x = gp;
    }
}

// Analysis (PAPER.md:113 steps (ii)/(iv)) of the forest in shared memory by pointer jumping: every site is re-pointed at
// its grandparent until nothing changes, about log2(depth) sweeps.  (Walking every chain to its root instead costs the
// sum of all depths, and hooking raster-ordered lattice sites to their smallest lower neighbour builds long chains.)
// Must be called by all threads; ends with a barrier.
__device__ __forceinline__ void smem_flatten(int32_t* L, int32_t n_sites)
{
    volatile int32_t* V = L;
    for (;;) {
        bool changed = false;
        for (int32_t i = threadIdx.x; i < n_sites; i += kBatchThreads) {
            const int32_t p = V[i];
            const int32_t gp = V[p];
            if (gp != p) { V[i] = gp; changed = true; }
        }
        if (!__syncthreads_or(changed)) return;
    }
}

// Steps (i)-(iv) of PAPER.md:113 for realization r = blockIdx.x, all in shared memory:
//   (i)   L[i] = i, then every occupied bond hooks its higher site to the lower one (one atomicMin, no return value):
//         each site ends up pointing at its smallest lower-numbered neighbour, the paper's initial label (Fig. 2)
//   (ii)  analysis: every site re-pointed at the top of its chain (Fig. 3 left)
//   (iii) Algorithm 1 on every occupied bond (most bonds find their ends joined already)
//   (iv)  analysis, and the labels leave for global memory once
__global__ void __launch_bounds__(kBatchThreads)
k_label_batch(int32_t n_sites, int32_t n_bonds, const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
              const uint32_t* __restrict__ bits, int64_t mask_stride_words, int32_t* __restrict__ labels)
{
    extern __shared__ __align__(16) int32_t L[];
    const int tid = threadIdx.x;
    const uint32_t* occ = bits ? bits + (size_t)blockIdx.x * mask_stride_words : nullptr;
    int32_t* out = labels + (size_t)blockIdx.x * n_sites;
    for (int32_t i = tid; i < n_sites; i += kBatchThreads) L[i] = i;
    __syncthreads();
    for (int32_t b = tid; b < n_bonds; b += kBatchThreads) {
        if (occ && !((occ[b >> 5] >> (b & 31)) & 1u)) continue;
        const int32_t u = src[b], v = dst[b];
        if (u != v) atomicMin(L + max(u, v), min(u, v));
    }
    __syncthreads();
    smem_flatten(L, n_sites);
    for (int32_t b = tid; b < n_bonds; b += kBatchThreads) {
        if (occ && !((occ[b >> 5] >> (b & 31)) & 1u)) continue;
        int32_t l1 = src[b], l2 = dst[b];
        for (;;) {
            l1 = smem_root(L, l1);
            l2 = smem_root(L, l2);
            if (l1 == l2) break;
            if (l1 < l2) { const int32_t t = l1; l1 = l2; l2 = t; }
            const int32_t l3 = atomicMin(L + l1, l2);
            if (l3 == l1 || l3 == l2) break;
            l1 = l3;
        }
    }
    __syncthreads();
    smem_flatten(L, n_sites);
    for (int32_t i = tid; i < n_sites; i += kBatchThreads) out[i] = L[i];
}

// ---------------------------------------------------------------------------------------- sequential relabel
__global__ void __launch_bounds__(256) k_flag_roots(int64_t n_sites, const int32_t* __restrict__ labels, int32_t* flag)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_sites; i += stride)
        flag[i] = labels[i] == (int32_t)i;
}

__global__ void __launch_bounds__(256)
k_gather_rank(int64_t n_sites, const int32_t* __restrict__ labels, const int32_t* __restrict__ rank, int32_t* seq,
              int64_t* n_clusters)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_sites; i += stride) seq[i] = rank[labels[i]];
    if (n_clusters && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t last = n_sites - 1;
        *n_clusters = (int64_t)rank[last] + (labels[last] == (int32_t)last);
    }
}

}  // namespace ccl

extern "C" int ccl_label_batch(int64_t n_sites, int64_t n_bonds, const int32_t* src, const int32_t* dst,
                               const uint32_t* occupied_bits, int64_t mask_stride_words, int32_t n_batch,
                               int32_t* labels, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_sites >= 0 && n_bonds >= 0 && n_batch >= 0, "negative count");
    CCL_REQUIRE(n_bonds == 0 || (src && dst), "src/dst is NULL with n_bonds > 0");
    CCL_REQUIRE(n_bonds == 0 || n_sites > 0, "bonds given but n_sites == 0");
    CCL_REQUIRE(n_sites == 0 || n_batch == 0 || labels != nullptr, "labels is NULL");
    CCL_REQUIRE(occupied_bits == nullptr || mask_stride_words >= (n_bonds + 31) / 32, "mask_stride_words < ceil(n_bonds/32)");
    CCL_REQUIRE((reinterpret_cast<uintptr_t>(occupied_bits) & 3) == 0, "occupied_bits is not 4-byte aligned");
    if (n_sites > kBatchMaxSites || n_bonds > 2147483647LL) {
        set_error("ccl_label_batch: n_sites > 32768 does not fit one CTA's shared memory; call ccl_label_bits per realization");
        return CCL_UNSUPPORTED;
    }
    if (n_sites == 0 || n_batch == 0) return CCL_OK;
    cudaStream_t st = as_stream(stream);
    const size_t smem = (size_t)n_sites * sizeof(int32_t);
    CCL_CUDA_TRY(cudaFuncSetAttribute(k_label_batch, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_label_batch<<<(unsigned)n_batch, kBatchThreads, smem, st>>>((int32_t)n_sites, (int32_t)n_bonds, src, dst,
                                                                 occupied_bits, mask_stride_words, labels);
    CCL_CHECK_LAUNCH("k_label_batch");
    return CCL_OK;
}

extern "C" int ccl_relabel_sequential(int64_t n_sites, const int32_t* labels, int32_t* seq_labels, int64_t* n_clusters,
                                      void* workspace, size_t* workspace_bytes, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_sites >= 0 && n_sites <= 2147483647LL, "n_sites out of range");
    CCL_REQUIRE(workspace_bytes != nullptr, "workspace_bytes is NULL");
    cudaStream_t st = as_stream(stream);
    size_t temp = 0;
    CCL_CUDA_TRY(cub::DeviceScan::ExclusiveSum(nullptr, temp, (const int32_t*)nullptr, (int32_t*)nullptr,
                                               (int)(n_sites > 0 ? n_sites : 1), st));
    const size_t arr = (((size_t)n_sites * sizeof(int32_t)) + 255) & ~(size_t)255;
    const size_t need = 2 * arr + temp;
    if (workspace == nullptr) { *workspace_bytes = need; return CCL_OK; }
    if (*workspace_bytes < need) { set_error("workspace too small: %zu < %zu", *workspace_bytes, need); return CCL_WORKSPACE_TOO_SMALL; }
    CCL_REQUIRE(n_sites == 0 || (labels && seq_labels), "labels/seq_labels is NULL");
    if (n_sites == 0) {
        if (n_clusters) CCL_CUDA_TRY(cudaMemsetAsync(n_clusters, 0, sizeof(int64_t), st));
        return CCL_OK;
    }
    int32_t* flag = static_cast<int32_t*>(workspace);
    int32_t* rank = reinterpret_cast<int32_t*>(static_cast<char*>(workspace) + arr);
    void* tmp = static_cast<char*>(workspace) + 2 * arr;
    int64_t blocks = (n_sites + 255) / 256;
    if (blocks > (int64_t)sm_count() * 16) blocks = (int64_t)sm_count() * 16;
    k_flag_roots<<<(unsigned)blocks, 256, 0, st>>>(n_sites, labels, flag);
    CCL_CHECK_LAUNCH("k_flag_roots");
    CCL_CUDA_TRY(cub::DeviceScan::ExclusiveSum(tmp, temp, flag, rank, (int)n_sites, st));
    count_launch();
    k_gather_rank<<<(unsigned)blocks, 256, 0, st>>>(n_sites, labels, rank, seq_labels, n_clusters);
    CCL_CHECK_LAUNCH("k_gather_rank");
    return CCL_OK;
}
