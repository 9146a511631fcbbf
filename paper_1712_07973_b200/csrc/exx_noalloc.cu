// exx_noalloc.cu -- the one entry point of libexx_b200 that allocates NOTHING (include/exx.h exx_exchange_energy_noalloc).
//
// Some callers cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.  For them
// the exchange energy is offered through the operator identity
//     E_x = 1/2 dV sum_i f_i <psi_i | K psi_i>          (Eq. 5 with Eq. 3 inserted; pinned for the oracle as P8)
// i.e. a variant of the library's two-stage deterministic energy reduction (exx_api.cu: complex_combine_kernel /
// complex_energy_kernel, which keep their per-block partial sums in the plan's cudaMalloc'ed workspace) whose scratch -- the
// per-block partial sums and the device copy of the occupations -- lives in ONE file-scope `static __device__` array of a
// fixed, modest size.  Every GPU that loads the library holds that array (kScratchDoubles * 8 = 40 KB) until the process
// exits.  The caller passes the inputs (psi, K psi, occupations) and the output (E_x, device memory).
//
// The array's name is a host-side stand-in in host code, NOT a device address: the host obtains the device address once per
// device, with that device current, through cudaGetSymbolAddress and passes it to the kernels.
//
// All calls share the array, which keeps the last call's contents.  Nothing in it needs to start at zero: the occupations are
// uploaded and every partial-sum slot that the final reduction reads is overwritten by the first kernel of the same call.
// Calls that OVERLAP on the GPU (different streams, or different host threads without an ordering between their streams) race
// on the array; calls on one stream are ordered and safe.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/exx.h"

namespace {

constexpr int kMaxOrbitals = EXX_NOALLOC_MAX_ORBITALS;      // occupations held in the scratch
constexpr int kMaxBlocks = 1024;                            // per-block partial sums held in the scratch
constexpr int kScratchDoubles = kMaxBlocks + kMaxOrbitals;  // 5120 doubles = 40 KB per GPU
constexpr int kThreads = 256;
constexpr int kDevices = 64;

static __device__ __align__(256) double g_noalloc_scratch[kScratchDoubles];   // [0, kMaxBlocks): partials; then occupations

thread_local char g_noalloc_error[256] = "";

exx_status fail(exx_status st, const char* msg) {
    std::snprintf(g_noalloc_error, sizeof(g_noalloc_error), "%s", msg);
    return st;
}
exx_status cuda_fail(cudaError_t e, const char* what) {
    std::snprintf(g_noalloc_error, sizeof(g_noalloc_error), "%s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
    cudaGetLastError();
    return EXX_ERR_CUDA;
}

// device address of the scratch array, resolved once per device ordinal with that device current
std::mutex g_addr_mutex;
double* g_scratch_addr[kDevices] = {};

cudaError_t scratch_address(double** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_addr_mutex);
    if (!g_scratch_addr[dev]) {
        double* ptr = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

// partial[b] = sum over this block's share of  f_i psi_i(r) Kpsi_i(r)  (fixed order: grid-stride per thread, then a tree)
__global__ void __launch_bounds__(kThreads) noalloc_partial_kernel(const double* psi, const double* kpsi, long long n_points, long long total,
                                                                    double* scratch) {
    __shared__ double sh[kThreads];
    const double* occ = scratch + kMaxBlocks;
    double s = 0.0;
    for (long long k = blockIdx.x * static_cast<long long>(kThreads) + threadIdx.x; k < total; k += static_cast<long long>(gridDim.x) * kThreads)
        s += occ[k / n_points] * (psi[k] * kpsi[k]);
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = kThreads / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) scratch[blockIdx.x] = sh[0];
}

// *ex = scale * sum_b partial[b], b < n_blocks (exactly the slots the kernel above wrote in this call)
__global__ void __launch_bounds__(kThreads) noalloc_final_kernel(const double* scratch, int n_blocks, double scale, double* ex) {
    __shared__ double sh[kThreads];
    double s = 0.0;
    for (int k = threadIdx.x; k < n_blocks; k += kThreads) s += scratch[k];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = kThreads / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *ex = scale * sh[0];
}

bool device_pointer(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" {

const char* exx_noalloc_last_error(void) { return g_noalloc_error; }

exx_status exx_exchange_energy_noalloc(int n_orb, long long n_points, double dV, const double* psi_dev, const double* kpsi_dev,
                                       const double* occ_host, double* ex_dev, void* cuda_stream) {
    g_noalloc_error[0] = '\0';
    if (!psi_dev || !kpsi_dev || !occ_host || !ex_dev) return fail(EXX_ERR_INVALID_ARG, "NULL argument");
    if (n_orb < 1 || n_points < 1) return fail(EXX_ERR_INVALID_ARG, "n_orb and n_points must be positive");
    if (n_orb > kMaxOrbitals) {
        std::snprintf(g_noalloc_error, sizeof(g_noalloc_error),
                      "exx_exchange_energy_noalloc: n_orb = %d exceeds EXX_NOALLOC_MAX_ORBITALS = %d (the static device scratch is fixed-size)", n_orb,
                      kMaxOrbitals);
        return EXX_ERR_UNSUPPORTED_SIZE;
    }
    if (!(dV > 0.0) || !std::isfinite(dV)) return fail(EXX_ERR_INVALID_ARG, "dV must be > 0");
    if (!device_pointer(psi_dev) || !device_pointer(kpsi_dev) || !device_pointer(ex_dev))
        return fail(EXX_ERR_BAD_POINTER, "psi_dev, kpsi_dev and ex_dev must be device pointers");
    if (device_pointer(occ_host)) return fail(EXX_ERR_BAD_POINTER, "occ_host must be a host pointer");
    double* scratch = nullptr;
    cudaError_t e = scratch_address(&scratch);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(static scratch)");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    // occupations into the scratch (a copy out of pageable host memory returns once the source has been read)
    e = cudaMemcpyAsync(scratch + kMaxBlocks, occ_host, sizeof(double) * static_cast<size_t>(n_orb), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(e, "upload of the occupations");
    const long long total = static_cast<long long>(n_orb) * n_points;
    const long long want = (total + kThreads - 1) / kThreads;
    const int n_blocks = static_cast<int>(want < kMaxBlocks ? want : kMaxBlocks);
    noalloc_partial_kernel<<<n_blocks, kThreads, 0, s>>>(psi_dev, kpsi_dev, n_points, total, scratch);
    noalloc_final_kernel<<<1, kThreads, 0, s>>>(scratch, n_blocks, 0.5 * dV, ex_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launch of the energy reduction");
    return EXX_OK;
}

}  // extern "C"
