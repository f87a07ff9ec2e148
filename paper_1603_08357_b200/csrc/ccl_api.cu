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

}  // namespace ccl

extern "C" const char* ccl_last_error(void) { return ccl::g_error; }
extern "C" int ccl_version(void) { return 100; }      // 0.1.0
extern "C" int64_t ccl_launch_count(void) { return ccl::g_launches; }
