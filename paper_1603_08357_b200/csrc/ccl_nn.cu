// ccl_nn.cu -- the paper's own interface: labeling from a nearest-neighbour
// list instead of a bond list, with the four steps in the paper's form.
//
//   NN list: dense z_max x N array, structure of arrays -- site i reads nn[i], nn[i + N], nn[i + 2N], ... (PAPER.md:111,
//   Fig. 1); entries < 0 are padding.  Every entry is a connection of the network to be labeled.
//
//   k_nn_init    step (i):  label[i] = smallest lower-numbered neighbour, else i.  The residual list of the paper (the
//                other lower-numbered neighbours) is not stored: it is re-read from the NN list in step (iii).  No
//                atomics: every site writes its own label.
//   k_flatten    step (ii): analysis (ccl_label.cu).
//   k_nn_reduce  step (iii): for every site i and every listed neighbour j != i: Algorithm 1 on
//                (i, j).  The labels are flat after (ii), so most pairs are seen to be joined by two reads.  (A bond
//                may be listed at its lower end only; step (i) does not see it there, step (iii) joins it.)
//   k_flatten    step (iv).
//
// Product code: nothing under oracle/ is included here or includes this.
#include "ccl_common.cuh"
#include "ccl_unionfind.cuh"

namespace ccl {

constexpr int kNnThreads = 256;

__global__ void __launch_bounds__(kNnThreads)
k_nn_init(int64_t n_sites, int z_max, const int32_t* __restrict__ nn, int32_t* __restrict__ label)
{
    const int64_t stride = (int64_t)gridDim.x * kNnThreads;
    for (int64_t i = (int64_t)blockIdx.x * kNnThreads + threadIdx.x; i < n_sites; i += stride) {
        int32_t m = (int32_t)i;
        for (int k = 0; k < z_max; ++k) {
            const int32_t j = nn[(int64_t)k * n_sites + i];
            if (j >= 0 && j < m) m = j;
        }
        label[i] = m;
    }
}

__global__ void __launch_bounds__(kNnThreads)
k_nn_reduce(int64_t n_sites, int z_max, const int32_t* __restrict__ nn, int32_t* label)
{
    __shared__ int2 queue[kNnThreads / 32][64];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t stride = (int64_t)gridDim.x * kNnThreads;
    const int64_t n_round = ((n_sites + 31) / 32) * 32;                    // whole warps take part in every round
    int qn = 0;                                                            // pairs waiting in the warp's queue (< 32 between looks)
    for (int64_t i = (int64_t)blockIdx.x * kNnThreads + threadIdx.x; i < n_round; i += stride) {
        const bool live = i < n_sites;
        for (int k = 0; k < z_max; ++k) {
            const int32_t j = live ? nn[(int64_t)k * n_sites + i] : -1;
            bool need = false;
            int32_t la = 0, lb = 0;
            // Every entry is a bond, whichever end lists it (include/ccl.h).  Lower-numbered neighbours are the paper's
            // residual list; an entry j > i joins the same way (Algorithm 1 is symmetric) -- if the list also names the
            // bond at site j, the second look finds the two labels equal and costs two reads.
            if (j >= 0 && j != (int32_t)i) {
                la = ld_label(label + i);
                lb = ld_label(label + j);
                need = la != lb;
            }
            // the pairs that are not visibly joined are packed and worked off 32 at a time, every lane busy (walks diverge
            // badly otherwise); fewer than 32 wait for the next look -- the order of the joins is free
            const unsigned m = __ballot_sync(0xffffffffu, need);
            if (m == 0) continue;
            if (need) queue[warp][qn + __popc(m & ((1u << lane) - 1u))] = make_int2(la, lb);
            qn += __popc(m);
            __syncwarp();
            if (qn >= 32) {
                qn -= 32;
                const int2 pr = queue[warp][qn + lane];
                algorithm1(label, pr.x, pr.y);
            }
            __syncwarp();
        }
    }
    if (lane < qn) {
        const int2 pr = queue[warp][lane];
        algorithm1(label, pr.x, pr.y);
    }
}

// defined in ccl_label.cu
int flatten_labels(int64_t n_sites, int32_t* labels, cudaStream_t st);

}  // namespace ccl

extern "C" int ccl_label_nn(int64_t n_sites, int32_t z_max, const int32_t* nn_list, int32_t* labels, void* stream)
{
    using namespace ccl;
    CCL_REQUIRE(n_sites >= 0 && n_sites <= 2147483647LL, "n_sites out of range");
    CCL_REQUIRE(z_max >= 0 && z_max <= 1024, "z_max out of range [0, 1024]");
    CCL_REQUIRE(n_sites == 0 || labels != nullptr, "labels is NULL");
    CCL_REQUIRE(n_sites == 0 || z_max == 0 || nn_list != nullptr, "nn_list is NULL");
    CCL_REQUIRE((reinterpret_cast<uintptr_t>(labels) & 15) == 0, "labels must be 16-byte aligned");
    if (n_sites == 0) return CCL_OK;
    cudaStream_t st = as_stream(stream);
    int64_t blocks = (n_sites + kNnThreads - 1) / kNnThreads;
    if (blocks > (int64_t)sm_count() * 32) blocks = (int64_t)sm_count() * 32;
    k_nn_init<<<(unsigned)blocks, kNnThreads, 0, st>>>(n_sites, z_max, nn_list, labels);          // step (i)
    CCL_CHECK_LAUNCH("k_nn_init");
    if (z_max == 0) return CCL_OK;
    int rc = flatten_labels(n_sites, labels, st);                                                  // step (ii)
    if (rc != CCL_OK) return rc;
    k_nn_reduce<<<(unsigned)blocks, kNnThreads, 0, st>>>(n_sites, z_max, nn_list, labels);        // step (iii)
    CCL_CHECK_LAUNCH("k_nn_reduce");
    return flatten_labels(n_sites, labels, st);                                                    // step (iv)
}
