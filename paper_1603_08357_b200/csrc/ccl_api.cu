// ccl_api.cu -- diagnostics of the C ABI (include/ccl.h): thread-local error string, version, launch counter.
#include <stdarg.h>
#include <string.h>

#include "ccl_common.cuh"

namespace ccl {

static thread_local char g_error[512] = "";
static thread_local int64_t g_launches = 0;

void set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_error, sizeof(g_error), fmt, ap);
    va_end(ap);
}

void count_launch(int n) { g_launches += n; }

Tuning& tuning()
{
    static Tuning t;
    return t;
}

int scratch_alloc(void** ptr, size_t bytes, cudaStream_t st)
{
    static cudaMemPool_t pools[64] = {};
    int dev = 0;
    CCL_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) { set_error("device index %d out of range", dev); return CCL_UNSUPPORTED; }
    if (pools[dev] == nullptr) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        CCL_CUDA_TRY(cudaMemPoolCreate(&pool, &props));
        unsigned long long keep = ~0ull;
        CCL_CUDA_TRY(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
        pools[dev] = pool;
    }
    CCL_CUDA_TRY(cudaMallocFromPoolAsync(ptr, bytes, pools[dev], st));
    return CCL_OK;
}

}  // namespace ccl

extern "C" const char* ccl_last_error(void) { return ccl::g_error; }
extern "C" int ccl_version(void) { return 200; }      // 0.2.0: + label_nn, label_batch, label_sweep_host, relabel, wrap
extern "C" int64_t ccl_launch_count(void) { return ccl::g_launches; }

extern "C" int ccl_set_option(const char* name, int64_t value)
{
    ccl::Tuning def;
    ccl::Tuning& t = ccl::tuning();
    if (name == nullptr) { ccl::set_error("invalid argument: option name is NULL"); return CCL_INVALID_ARG; }
    if (!strcmp(name, "reset")) { t = def; return CCL_OK; }
    if (!strcmp(name, "bucket_min_label_bytes")) {
        t.bucket_min_label_bytes = value >= 0 ? value : def.bucket_min_label_bytes;
        t.bucket_min_bonds = value >= 0 ? 0 : def.bucket_min_bonds;
        return CCL_OK;
    }
    if (!strcmp(name, "region_shift")) {
        if (value >= 0 && (value < 4 || value > 30)) {
            ccl::set_error("invalid argument: region_shift must lie in [4, 30]");
            return CCL_INVALID_ARG;
        }
        t.region_shift = value >= 0 ? (int32_t)value : def.region_shift;
        return CCL_OK;
    }
    if (!strcmp(name, "force_mode")) {
        if (value < -1 || value > 1) {
            ccl::set_error("invalid argument: force_mode must be -1, 0 or 1");
            return CCL_INVALID_ARG;
        }
        t.force_mode = (int32_t)value;
        return CCL_OK;
    }
    if (!strcmp(name, "bucket_capacity")) { t.bucket_capacity = value > 0 ? value : 0; return CCL_OK; }
    if (!strcmp(name, "two_pass")) { t.two_pass = value > 0 ? 1 : value < 0 ? -1 : 0; return CCL_OK; }
    if (!strcmp(name, "tile_mode")) {
        if (value < -1 || value > 1) {
            ccl::set_error("invalid argument: tile_mode must be -1, 0 or 1");
            return CCL_INVALID_ARG;
        }
        t.tile_mode = (int32_t)value;
        return CCL_OK;
    }
    if (!strcmp(name, "sub_shift")) {
        if (value > 15) {
            ccl::set_error("invalid argument: sub_shift must be at most 15 (128 KiB of labels in shared memory)");
            return CCL_INVALID_ARG;
        }
        t.sub_shift = value >= 2 ? (int32_t)value : -1;
        return CCL_OK;
    }
    if (!strcmp(name, "fine_capacity")) { t.fine_capacity = value > 0 ? value : 0; return CCL_OK; }
    if (!strcmp(name, "small_max_sites")) { t.small_max_sites = value >= 0 ? value : def.small_max_sites; return CCL_OK; }
    if (!strcmp(name, "tile_min_bonds")) { t.tile_min_bonds = value >= 0 ? value : def.tile_min_bonds; return CCL_OK; }
    ccl::set_error("invalid argument: unknown option '%s'", name);
    return CCL_INVALID_ARG;
}
