// ccl_stats.cu -- cluster statistics from canonical labels (include/ccl.h: ccl_cluster_stats; reading R8;
// the paper itself measures only the spanning probability).  Outside the timed metric.
#include <mutex>

#include "ccl_common.cuh"

namespace ccl {

constexpr int kStatThreads = 256;

// size[l] = #{ i : labels[i] == l }.  Lanes of a warp that hold the same label are merged first
// (__match_any_sync), so the giant cluster costs one atomic per warp instead of one per site.
__global__ void __launch_bounds__(kStatThreads)
k_count_sizes(int64_t n_sites, const int32_t* __restrict__ labels, int32_t* size)
{
    const int64_t stride = (int64_t)gridDim.x * kStatThreads;
    const int lane = threadIdx.x & 31;
    for (int64_t base = (int64_t)blockIdx.x * kStatThreads; base < n_sites; base += stride) {
        const int64_t i = base + threadIdx.x;
        const bool on = i < n_sites;
        const int32_t l = on ? labels[i] : -1 - lane;              // distinct dummies for idle lanes
        const unsigned peers = __match_any_sync(0xffffffffu, l);
        if (on && lane == __ffs(peers) - 1) atomicAdd(size + l, __popc(peers));
    }
}

__global__ void __launch_bounds__(kStatThreads)
k_reduce_sizes(int64_t n_sites, const int32_t* __restrict__ size, ccl_stats* out, unsigned long long* hist_dense,
               int32_t n_dense, unsigned long long* hist_log2, unsigned long long* best_key)
{
    __shared__ unsigned long long s_log2[32];
    __shared__ unsigned long long s_ncl, s_sum2, s_best;
    if (threadIdx.x < 32) s_log2[threadIdx.x] = 0;
    if (threadIdx.x == 0) { s_ncl = 0; s_sum2 = 0; s_best = 0; }
    __syncthreads();

    unsigned long long ncl = 0, sum2 = 0, best = 0;
    const int64_t stride = (int64_t)gridDim.x * kStatThreads;
    for (int64_t l = (int64_t)blockIdx.x * kStatThreads + threadIdx.x; l < n_sites; l += stride) {
        const unsigned long long s = (unsigned long long)size[l];
        if (s == 0) continue;
        ncl += 1;
        sum2 += s * s;
        // larger size wins; equal sizes -> smaller label wins
        const unsigned long long key = (s << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)l);
        best = key > best ? key : best;
        if (hist_dense && s <= (unsigned long long)n_dense) atomicAdd(hist_dense + s, 1ull);
        if (hist_log2) atomicAdd(&s_log2[63 - __clzll((long long)s)], 1ull);
    }
    for (int o = 16; o > 0; o >>= 1) {
        ncl += __shfl_xor_sync(0xffffffffu, ncl, o);
        sum2 += __shfl_xor_sync(0xffffffffu, sum2, o);
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
        best = other > best ? other : best;
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&s_ncl, ncl);
        atomicAdd(&s_sum2, sum2);
        atomicMax(&s_best, best);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_ncl) atomicAdd(reinterpret_cast<unsigned long long*>(&out->n_clusters), s_ncl);
        if (s_sum2) atomicAdd(reinterpret_cast<unsigned long long*>(&out->sum_s2), s_sum2);
        if (s_best) atomicMax(best_key, s_best);
    }
    if (hist_log2 && threadIdx.x < 32 && s_log2[threadIdx.x]) atomicAdd(hist_log2 + threadIdx.x, s_log2[threadIdx.x]);
}

__global__ void k_finish_stats(ccl_stats* out, const unsigned long long* best_key)
{
    const unsigned long long key = *best_key;
    out->largest = (int64_t)(key >> 32);
    out->largest_label = key ? (int64_t)(0xFFFFFFFFu - (uint32_t)(key & 0xFFFFFFFFull)) : -1;
}

}  // namespace ccl

extern "C" int ccl_cluster_stats(int64_t n_sites, const int32_t* labels, int32_t* size_scratch, ccl_stats* out,
                                 int64_t* hist_dense, int32_t n_dense, int64_t* hist_log2, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_sites >= 0 && n_sites <= 2147483647LL, "n_sites out of range");
    CCL_REQUIRE(out != nullptr, "out is NULL");
    CCL_REQUIRE(n_sites == 0 || (labels && size_scratch), "labels/size_scratch is NULL");
    CCL_REQUIRE(n_dense >= 0, "n_dense < 0");
    cudaStream_t st = as_stream(stream);
    CCL_CUDA_TRY(cudaMemsetAsync(out, 0, sizeof(ccl_stats), st));
    if (hist_dense) CCL_CUDA_TRY(cudaMemsetAsync(hist_dense, 0, sizeof(int64_t) * ((size_t)n_dense + 1), st));
    if (hist_log2) CCL_CUDA_TRY(cudaMemsetAsync(hist_log2, 0, sizeof(int64_t) * 32, st));
    if (n_sites == 0) {
        // largest = 0, largest_label = -1 for the empty graph
        const int64_t minus1 = -1;
        CCL_CUDA_TRY(cudaMemcpyAsync(&out->largest_label, &minus1, sizeof(int64_t), cudaMemcpyHostToDevice, st));
        return CCL_OK;
    }
    CCL_CUDA_TRY(cudaMemsetAsync(size_scratch, 0, sizeof(int32_t) * (size_t)n_sites, st));
    int64_t blocks = (n_sites + kStatThreads - 1) / kStatThreads;
    if (blocks > (int64_t)sm_count() * 16) blocks = (int64_t)sm_count() * 16;
    k_count_sizes<<<(unsigned)blocks, kStatThreads, 0, st>>>(n_sites, labels, size_scratch);
    CCL_CHECK_LAUNCH("k_count_sizes");
    // best_key lives in out->largest until k_finish_stats unpacks it
    unsigned long long* best_key = reinterpret_cast<unsigned long long*>(&out->largest);
    k_reduce_sizes<<<(unsigned)blocks, kStatThreads, 0, st>>>(
        n_sites, size_scratch, out, reinterpret_cast<unsigned long long*>(hist_dense), n_dense,
        reinterpret_cast<unsigned long long*>(hist_log2), best_key);
    CCL_CHECK_LAUNCH("k_reduce_sizes");
    k_finish_stats<<<1, 1, 0, st>>>(out, best_key);
    CCL_CHECK_LAUNCH("k_finish_stats");
    return CCL_OK;
}

// ---- ccl_cluster_stats_static: the same statistics for callers that cannot allocate device memory ---------------
//
// ccl_cluster_stats needs one int32 per site of working memory (cluster sizes indexed by label) and asks the caller
// for it.  Some callers have no way to provide it: a simulation that has handed all device memory to its own arena
// at start-up (a cudaMalloc would fail, and the arena has no block to spare), or a measurement loop that must not
// issue cudaMalloc / cudaFree because those synchronise the whole device and would stall the other streams of the
// program.  For them the size table below is part of the library image: it is reserved when the module is loaded on
// a GPU and stays until the process exits, so this entry point calls no cudaMalloc, cudaFree, memory pool or
// allocating library routine -- only cudaMemsetAsync and kernel launches on the caller's stream.
namespace ccl {

// CCL_STATS_STATIC_MAX_SITES int32 counters = 16 MiB on every GPU that loads libccl.so.
static __device__ __align__(256) int32_t g_static_sizes[CCL_STATS_STATIC_MAX_SITES];

// In host code `g_static_sizes` is only the handle the runtime knows the array by, not its device address: the
// address is looked up once per device with that device current, and cached.
static std::mutex g_static_mutex;
static int32_t* g_static_ptr[64] = {};

static int static_sizes_on_current_device(int32_t** out)
{
    int dev = 0;
    CCL_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) { set_error("device index %d out of range", dev); return CCL_UNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (g_static_ptr[dev] == nullptr) {
        int32_t* p = nullptr;
        CCL_CUDA_TRY(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_sizes));
        if (p == nullptr) { set_error("cudaGetSymbolAddress returned a NULL address for the static size table"); return CCL_CUDA_ERROR; }
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return CCL_OK;
}

}  // namespace ccl

extern "C" int ccl_cluster_stats_static(int64_t n_sites, const int32_t* labels, ccl_stats* out, int64_t* hist_dense,
                                        int32_t n_dense, int64_t* hist_log2, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_sites >= 0, "n_sites out of range");
    if (n_sites > (int64_t)CCL_STATS_STATIC_MAX_SITES) {
        set_error("invalid argument: ccl_cluster_stats_static handles at most CCL_STATS_STATIC_MAX_SITES = %lld sites "
                  "(n_sites = %lld); use ccl_cluster_stats with a caller-provided size_scratch",
                  (long long)CCL_STATS_STATIC_MAX_SITES, (long long)n_sites);
        return CCL_INVALID_ARG;
    }
    CCL_REQUIRE(out != nullptr, "out is NULL");
    CCL_REQUIRE(n_sites == 0 || labels, "labels is NULL");
    CCL_REQUIRE(n_dense >= 0, "n_dense < 0");
    int32_t* sizes = nullptr;                       // device address of g_static_sizes on the current device
    const int rc = static_sizes_on_current_device(&sizes);
    if (rc != CCL_OK) return rc;
    cudaStream_t st = as_stream(stream);
    CCL_CUDA_TRY(cudaMemsetAsync(out, 0, sizeof(ccl_stats), st));
    if (hist_dense) CCL_CUDA_TRY(cudaMemsetAsync(hist_dense, 0, sizeof(int64_t) * ((size_t)n_dense + 1), st));
    if (hist_log2) CCL_CUDA_TRY(cudaMemsetAsync(hist_log2, 0, sizeof(int64_t) * 32, st));
    if (n_sites == 0) {
        const int64_t minus1 = -1;
        CCL_CUDA_TRY(cudaMemcpyAsync(&out->largest_label, &minus1, sizeof(int64_t), cudaMemcpyHostToDevice, st));
        return CCL_OK;
    }
    // the table still holds the sizes of the previous call: the first n_sites counters must start at zero
    CCL_CUDA_TRY(cudaMemsetAsync(sizes, 0, sizeof(int32_t) * (size_t)n_sites, st));
    int64_t blocks = (n_sites + kStatThreads - 1) / kStatThreads;
    if (blocks > (int64_t)sm_count() * 16) blocks = (int64_t)sm_count() * 16;
    k_count_sizes<<<(unsigned)blocks, kStatThreads, 0, st>>>(n_sites, labels, sizes);
    CCL_CHECK_LAUNCH("k_count_sizes");
    unsigned long long* best_key = reinterpret_cast<unsigned long long*>(&out->largest);
    k_reduce_sizes<<<(unsigned)blocks, kStatThreads, 0, st>>>(
        n_sites, sizes, out, reinterpret_cast<unsigned long long*>(hist_dense), n_dense,
        reinterpret_cast<unsigned long long*>(hist_log2), best_key);
    CCL_CHECK_LAUNCH("k_reduce_sizes");
    k_finish_stats<<<1, 1, 0, st>>>(out, best_key);
    CCL_CHECK_LAUNCH("k_finish_stats");
    return CCL_OK;
}
