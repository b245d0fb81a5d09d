// Process-wide state of libbs: thread-local error text, handle ids, launch counter.
#include <cstdarg>

#include "bs_internal.cuh"

std::atomic<int64_t> g_bs_launches{0};
static thread_local char t_err[512] = "";
static std::atomic<u64> g_next_id{1};

void bs_set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
}

u64 bs_next_id() { return g_next_id.fetch_add(1); }

extern "C" const char* bs_last_error(void) { return t_err; }
extern "C" const char* bs_version(void) { return "libbs 0.1 (sm_100a)"; }
extern "C" int64_t bs_launch_count(void) { return g_bs_launches.load(); }
