// ccl_api.cu -- diagnostics of the C ABI (include/ccl.h): thread-local error string, version, launch counter.
#include <stdarg.h>
#include <string.h>

#include <atomic>
#include <mutex>

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
    static thread_local Tuning t;                  // per host thread, like the error string and the launch counter
    return t;
}

int sm_count()
{
    static std::atomic<int> cached[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return 148; }
    int n = cached[dev].load(std::memory_order_relaxed);
    if (n <= 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) { cudaGetLastError(); return 148; }
        cached[dev].store(n, std::memory_order_relaxed);
    }
    return n;
}

// Persisting-L2 set-up, once per device: the limit is raised to the device's maximum the first time a launch asks
// for an access-policy window (ccl_set_option "l2_persist").
struct L2Persist { bool ready = false; size_t persist = 0, max_window = 0; };
static std::mutex g_l2_mutex;
static L2Persist g_l2[64];

static L2Persist l2_state()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return L2Persist(); }
    std::lock_guard<std::mutex> lock(g_l2_mutex);
    L2Persist& s = g_l2[dev];
    if (!s.ready) {
        int max_persist = 0, max_window = 0;
        cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, dev);
        cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, dev);
        if (max_persist > 0 && cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, (size_t)max_persist) == cudaSuccess) {
            size_t got = 0;
            if (cudaDeviceGetLimit(&got, cudaLimitPersistingL2CacheSize) == cudaSuccess) s.persist = got;
        }
        cudaGetLastError();
        s.max_window = max_window > 0 ? (size_t)max_window : 0;
        s.ready = true;
    }
    return s;
}
size_t l2_persist_bytes() { return l2_state().persist; }
size_t l2_max_window_bytes() { return l2_state().max_window; }

static std::mutex g_pool_mutex;
static cudaMemPool_t g_pools[64] = {};

static int pool_for_current_device(cudaMemPool_t* out, bool create)
{
    int dev = 0;
    CCL_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) { set_error("device index %d out of range", dev); return CCL_UNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (g_pools[dev] == nullptr && create) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        CCL_CUDA_TRY(cudaMemPoolCreate(&pool, &props));
        unsigned long long keep = ~0ull;           // freed scratch stays in the pool until ccl_trim_scratch
        CCL_CUDA_TRY(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
        g_pools[dev] = pool;
    }
    *out = g_pools[dev];
    return CCL_OK;
}

int scratch_alloc(void** ptr, size_t bytes, cudaStream_t st)
{
    cudaMemPool_t pool = nullptr;
    const int rc = pool_for_current_device(&pool, true);
    if (rc != CCL_OK) return rc;
    CCL_CUDA_TRY(cudaMallocFromPoolAsync(ptr, bytes, pool, st));
    return CCL_OK;
}

}  // namespace ccl

extern "C" const char* ccl_last_error(void) { return ccl::g_error; }
extern "C" int ccl_version(void) { return 400; }      // 0.4.0: ccl_cluster_stats_static, whole-round survivor walks, per-device set-up, l2_persist option
extern "C" int64_t ccl_launch_count(void) { return ccl::g_launches; }

extern "C" int ccl_set_option(const char* name, int64_t value)
{
    ccl::Tuning def;
    ccl::Tuning& t = ccl::tuning();
    if (name == nullptr) { ccl::set_error("invalid argument: option name is NULL"); return CCL_INVALID_ARG; }
    if (!strcmp(name, "reset")) { t = def; ccl::forget_probe_hints(); return CCL_OK; }
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
    if (!strcmp(name, "scatter_tiles")) { t.scatter_tiles = value != 0; return CCL_OK; }
    if (!strcmp(name, "probe_cache")) { t.probe_cache = value != 0; ccl::forget_probe_hints(); return CCL_OK; }
    if (!strcmp(name, "flatten_window_bytes")) {
        t.flatten_window_bytes = value > 0 ? value : def.flatten_window_bytes;
        return CCL_OK;
    }
    if (!strcmp(name, "flatten_window_min_bytes")) { t.flatten_window_min_bytes = value; return CCL_OK; }
    if (!strcmp(name, "l2_persist")) { t.l2_persist = value != 0; return CCL_OK; }
    ccl::set_error("invalid argument: unknown option '%s'", name);
    return CCL_INVALID_ARG;
}

extern "C" int ccl_trim_scratch(size_t keep_bytes, void* stream)
{
    using namespace ccl;
    cudaMemPool_t pool = nullptr;
    const int rc = pool_for_current_device(&pool, false);
    if (rc != CCL_OK) return rc;
    if (pool == nullptr) return CCL_OK;                    // nothing was ever allocated on this device
    CCL_CUDA_TRY(cudaStreamSynchronize(as_stream(stream)));   // scratch freed on the stream must have been released
    CCL_CUDA_TRY(cudaMemPoolTrimTo(pool, keep_bytes));
    return CCL_OK;
}

extern "C" int ccl_scratch_bytes(int64_t* reserved, int64_t* in_use)
{
    using namespace ccl;
    cudaMemPool_t pool = nullptr;
    const int rc = pool_for_current_device(&pool, false);
    if (rc != CCL_OK) return rc;
    unsigned long long r = 0, u = 0;
    if (pool != nullptr) {
        CCL_CUDA_TRY(cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReservedMemCurrent, &r));
        CCL_CUDA_TRY(cudaMemPoolGetAttribute(pool, cudaMemPoolAttrUsedMemCurrent, &u));
    }
    if (reserved) *reserved = (int64_t)r;
    if (in_use) *in_use = (int64_t)u;
    return CCL_OK;
}
