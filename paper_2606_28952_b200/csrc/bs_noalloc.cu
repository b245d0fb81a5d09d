// bs_vdot_noalloc: <a|b> = sum conj(a_i) b_i (Eq. 5 with b = H psi) for callers that cannot allocate:
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// Variant of k_vdot (bs_apply.cu), whose per-block partial sums live in scratch the library cudaMalloc's per sector.
// Here the scratch is a file-scope __device__ array of a fixed, modest size: kNoAllocMaxTiles partials of 16 bytes =
// 128 KiB, held by every GPU that loads the library until the process exits.  One thread block reduces one TILE of
// kNoAllocTile consecutive amplitudes into one partial, so the array bounds the vector length:
//   n <= kNoAllocMaxTiles * kNoAllocTile = 8192 * 65536 = 536,870,912 amplitudes
// (BASELINE.json configs[4] has 419,225,625); longer vectors are rejected with BS_ERR_ARG.
//
// The entry point calls no cudaMalloc / cudaFree and no allocating library routine, copies nothing to the host and does
// not synchronise: inputs, the 16-byte result and the stream are the caller's.  In host code the array's NAME is a
// host-side stand-in, not a device address; its device address is taken once per device with cudaGetSymbolAddress
// (bs_noalloc_setup, with that device current) and that pointer is what the kernels receive.
//
// Shared state: every call on a device uses the same array, and the array keeps the last call's contents.  Nothing has
// to start at zero: the reduction kernel reads only the partials [0, n_tiles) that the first kernel of the SAME call
// wrote, each block writing its slot unconditionally (an empty tail contributes an explicit zero).  Calls that overlap on
// the GPU (different streams, or graphs replayed concurrently) race on the array: issue them on one stream at a time.
#include <mutex>

#include "bs_epilogue.cuh"

namespace {

constexpr int kNoAllocTile = 65536;      // amplitudes per thread block
constexpr int kNoAllocMaxTiles = 8192;   // partials in the static scratch
constexpr int kMaxDevices = 64;

static __device__ __align__(256) double2 g_noalloc_partials[kNoAllocMaxTiles];

std::mutex g_noalloc_mu;
double2* g_noalloc_ptr[kMaxDevices] = {};   // device address of the array on each device (nullptr: not set up)

// one block per tile of kNoAllocTile amplitudes, 128-bit loads, deterministic block reduction
__global__ void __launch_bounds__(256) k_vdot_tiles(const double2* __restrict__ a, const double2* __restrict__ b, i64 n,
                                                    double2* __restrict__ partials) {
    __shared__ double2 sh_red[32];
    const i64 lo = (i64)blockIdx.x * kNoAllocTile, hi = min(n, lo + (i64)kNoAllocTile);
    double2 v = make_double2(0.0, 0.0);
    for (i64 i = lo + threadIdx.x; i < hi; i += blockDim.x) {
        const double2 x = a[i], y = b[i];
        v.x += x.x * y.x + x.y * y.y;
        v.y += x.x * y.y - x.y * y.x;
    }
    v = block_sum(v, sh_red);
    if (threadIdx.x == 0) partials[blockIdx.x] = v;   // unconditional: no slot of [0, gridDim.x) keeps stale contents
}

// fixed-order sum of the partials [0, n_tiles) -> result (2 doubles on the device)
__global__ void __launch_bounds__(1024) k_vdot_tiles_finish(const double2* __restrict__ partials, int n_tiles,
                                                           double2* __restrict__ result) {
    __shared__ double2 sh_red[32];
    double2 v = make_double2(0.0, 0.0);
    for (int i = threadIdx.x; i < n_tiles; i += blockDim.x) {
        v.x += partials[i].x;
        v.y += partials[i].y;
    }
    v = block_sum(v, sh_red);
    if (threadIdx.x == 0) *result = v;
}

}  // namespace

// Takes the device address of the static scratch for the CURRENT device (once per device; later calls return at once).
// Call it before graph capture starts: cudaGetSymbolAddress may load the module, which capture does not allow.
extern "C" int bs_noalloc_setup(void) {
    int dev = 0;
    BS_CUDA(cudaGetDevice(&dev));
    BS_REQUIRE(dev >= 0 && dev < kMaxDevices, BS_ERR_ARG, "bs_noalloc_setup: device ordinal %d out of range", dev);
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (g_noalloc_ptr[dev]) return BS_OK;
    double2* p = nullptr;
    BS_CUDA(cudaGetSymbolAddress((void**)&p, g_noalloc_partials));   // the name is a host stand-in: never pass it to a kernel
    BS_REQUIRE(p, BS_ERR_CUDA, "bs_noalloc_setup: cudaGetSymbolAddress returned a null address");
    g_noalloc_ptr[dev] = p;
    return BS_OK;
}

extern "C" int64_t bs_noalloc_max_dim(void) { return (int64_t)kNoAllocMaxTiles * kNoAllocTile; }

extern "C" int bs_vdot_noalloc(const void* a, const void* b, int64_t n, void* result_dev, void* cuda_stream) {
    BS_REQUIRE(a && b && result_dev, BS_ERR_ARG, "bs_vdot_noalloc: NULL argument");
    BS_REQUIRE(((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(result_dev)) &
                15u) == 0,
               BS_ERR_ARG, "bs_vdot_noalloc: pointers must be 16-byte aligned");
    BS_REQUIRE(n >= 0, BS_ERR_ARG, "bs_vdot_noalloc: negative length");
    BS_REQUIRE(n <= bs_noalloc_max_dim(), BS_ERR_ARG,
               "bs_vdot_noalloc: %lld amplitudes exceed the static scratch (%d partials x %d amplitudes = %lld); use bs_vdot",
               (long long)n, kNoAllocMaxTiles, kNoAllocTile, (long long)bs_noalloc_max_dim());
    int dev = 0;
    BS_CUDA(cudaGetDevice(&dev));
    BS_REQUIRE(dev >= 0 && dev < kMaxDevices, BS_ERR_ARG, "bs_vdot_noalloc: device ordinal %d out of range", dev);
    if (!g_noalloc_ptr[dev]) {   // first use on this device outside a capture; under capture call bs_noalloc_setup first
        int rc = bs_noalloc_setup();
        if (rc != BS_OK) return rc;
    }
    double2* scratch = g_noalloc_ptr[dev];
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int n_tiles = (int)((n + kNoAllocTile - 1) / kNoAllocTile);
    if (n_tiles > 0)
        k_vdot_tiles<<<n_tiles, 256, 0, st>>>((const double2*)a, (const double2*)b, n, scratch);
    k_vdot_tiles_finish<<<1, 1024, 0, st>>>(scratch, n_tiles, (double2*)result_dev);   // n = 0: writes (0, 0)
    BS_COUNT_LAUNCH(n_tiles > 0 ? 2 : 1);
    BS_CUDA(cudaGetLastError());
    return BS_OK;
}
