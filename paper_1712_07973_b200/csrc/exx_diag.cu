// exx_diag.cu -- device microbenchmarks behind exx_diag_fp64 (include/exx.h): the measured denominators of the FP64 leg
// of the roofline (north_star: "the slower of FFT+fusion bytes over 8 TB/s HBM and FP64 flops at peak").
// MEASURED_PEAKS.json holds HBM and bf16 tensor peaks only; the exact-exchange path runs on the plain FP64 pipe and
// moves its butterflies through shared memory, so bench.py measures those two pipes itself, on the device it times:
//   mode 0  DFMA   dependent chains, ILP 8, 16 warps per SM          -> FP64 FMA rate  (2 flops per instruction)
//   mode 1  DADD   same chains with additions only                    -> FP64 issue rate (FFT butterflies are add-heavy)
//   mode 2  LDS.128 conflict-free 16-byte shared-memory loads         -> shared-memory bandwidth per SM
//   mode 3  even warps DFMA, odd warps LDS.128                        -> do the two pipes overlap inside one SM?
//   mode 4 / 5  the two halves of mode 3 alone (even warps DFMA, odd idle / odd warps LDS, even idle)
//   mode 6  SHFL.BFLY 32-bit warp shuffles                             -> shuffle bandwidth per SM (4 bytes per lane each)
//   mode 7  even warps SHFL, odd warps LDS.128; modes 8 / 5 its halves  -> would a shuffle exchange ADD bandwidth beside
//           the shared-memory pipe, or do the two share one datapath?  (north_star names warp-shuffle butterflies; the
//           passes exchange through shared memory -- this is the measurement behind that choice, exx_diag_shfl)
// Not part of the hot path; nothing here is called by exx_apply*.
#include <cuda_runtime.h>

#include "../../include/exx.h"

namespace {

template <int MODE>
__global__ void __launch_bounds__(512, 1) diag_kernel(double* out, int iters) {
    extern __shared__ double2 sm[];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int i = tid; i < 4096; i += blockDim.x) sm[i] = make_double2(1.0 + i * 1e-9, 1.0 - i * 1e-9);
    __syncthreads();
    double a[8] = {1.0, 1.1, 1.2, 1.3, 1.4, 1.5, 1.6, 1.7};
    double2 acc = make_double2(0, 0);
    const double c = 0.999999, d = 1e-7;
    const bool do_f = MODE == 0 || MODE == 1 || ((MODE == 3 || MODE == 4) && (wid & 1) == 0);
    const bool do_l = MODE == 2 || ((MODE == 3 || MODE == 5 || MODE == 7) && (wid & 1) == 1);
    const bool do_s = MODE == 6 || ((MODE == 7 || MODE == 8) && (wid & 1) == 0);
    unsigned sv[8] = {1u + tid, 2u + tid, 3u + tid, 4u + tid, 5u + tid, 6u + tid, 7u + tid, 8u + tid};
    for (int it = 0; it < iters; ++it) {
        if (do_l) {
#pragma unroll
            for (int u = 0; u < 16; ++u) {                     // 16 LDS.128, conflict-free, 4 wavefronts each
                double2 v = sm[(u * 32 + lane + it * 7) & 4095];
                acc.x += v.x; acc.y += v.y;
            }
        }
        if (do_s) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {                      // 64 SHFL.BFLY, 8 independent chains
#pragma unroll
                for (int q = 0; q < 8; ++q) sv[q] = __shfl_xor_sync(0xffffffffu, sv[q], 1 + ((u + q) & 15)) + 1u;
            }
        }
        if (do_f) {
#pragma unroll
            for (int u = 0; u < 32; ++u) {                     // 256 FP64 instructions, ILP 8
#pragma unroll
                for (int q = 0; q < 8; ++q) a[q] = (MODE == 1) ? a[q] + d : a[q] * c + d;
            }
        }
    }
    double s = acc.x + acc.y;
    for (int q = 0; q < 8; ++q) s += a[q] + sv[q];
    if (s == 123.456) out[0] = s;                              // keeps the work alive
}

template <int MODE>
cudaError_t time_mode(double* out, int sms, int iters, cudaStream_t s, float* ms) {
    cudaEvent_t e0, e1;
    cudaError_t e = cudaFuncSetAttribute(diag_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
    if (e != cudaSuccess) return e;
    if ((e = cudaEventCreate(&e0)) != cudaSuccess) return e;
    if ((e = cudaEventCreate(&e1)) != cudaSuccess) { cudaEventDestroy(e0); return e; }
    diag_kernel<MODE><<<sms, 512, 65536, s>>>(out, 16);        // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0, s);
        diag_kernel<MODE><<<sms, 512, 65536, s>>>(out, iters);
        cudaEventRecord(e1, s);
        e = cudaEventSynchronize(e1);
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
        if (t < best) best = t;
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *ms = best;
    return e;
}

}  // namespace

extern "C" exx_status exx_diag_fp64(void* cuda_stream, double* dfma_tflops, double* dadd_tops, double* lds_gbs, double* overlap_ratio) {
    if (!dfma_tflops || !dadd_tops || !lds_gbs || !overlap_ratio) return EXX_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        cudaGetLastError();
        return EXX_ERR_CUDA;
    }
    double* out = nullptr;
    if (cudaMalloc(&out, sizeof(double)) != cudaSuccess) { cudaGetLastError(); return EXX_ERR_ALLOC; }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const int iters = 2000;
    float t_fma = 0, t_add = 0, t_lds = 0, t_both = 0, t_half_f = 0, t_half_l = 0;
    cudaError_t e = time_mode<0>(out, sms, iters, s, &t_fma);
    if (e == cudaSuccess) e = time_mode<1>(out, sms, iters, s, &t_add);
    if (e == cudaSuccess) e = time_mode<2>(out, sms, iters, s, &t_lds);
    if (e == cudaSuccess) e = time_mode<3>(out, sms, iters, s, &t_both);
    if (e == cudaSuccess) e = time_mode<4>(out, sms, iters, s, &t_half_f);
    if (e == cudaSuccess) e = time_mode<5>(out, sms, iters, s, &t_half_l);
    cudaFree(out);
    if (e != cudaSuccess) { cudaGetLastError(); return EXX_ERR_CUDA; }
    const double inst = static_cast<double>(sms) * 512.0 * 256.0 * iters;          // FP64 instructions (thread level)
    *dfma_tflops = 2.0 * inst / (t_fma * 1e-3) / 1e12;
    *dadd_tops = inst / (t_add * 1e-3) / 1e12;
    *lds_gbs = static_cast<double>(sms) * 512.0 * 16.0 * 16.0 * iters / (t_lds * 1e-3) / 1e9;
    // mode 3 = the 8 DFMA warps of mode 4 and the 8 LDS warps of mode 5 together: perfect overlap -> max(t4, t5),
    // no overlap -> t4 + t5
    const double ideal = t_half_f > t_half_l ? t_half_f : t_half_l, serial = static_cast<double>(t_half_f) + t_half_l;
    *overlap_ratio = serial > ideal ? (serial - t_both) / (serial - ideal) : 1.0;   // 1: full overlap, 0: serialised
    return EXX_OK;
}

extern "C" exx_status exx_diag_shfl(void* cuda_stream, double* shfl_gbs, double* shfl_lds_overlap) {
    if (!shfl_gbs || !shfl_lds_overlap) return EXX_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        cudaGetLastError();
        return EXX_ERR_CUDA;
    }
    double* out = nullptr;
    if (cudaMalloc(&out, sizeof(double)) != cudaSuccess) { cudaGetLastError(); return EXX_ERR_ALLOC; }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const int iters = 2000;
    float t_shfl = 0, t_both = 0, t_half_s = 0, t_half_l = 0;
    cudaError_t e = time_mode<6>(out, sms, iters, s, &t_shfl);
    if (e == cudaSuccess) e = time_mode<7>(out, sms, iters, s, &t_both);
    if (e == cudaSuccess) e = time_mode<8>(out, sms, iters, s, &t_half_s);
    if (e == cudaSuccess) e = time_mode<5>(out, sms, iters, s, &t_half_l);
    cudaFree(out);
    if (e != cudaSuccess) { cudaGetLastError(); return EXX_ERR_CUDA; }
    *shfl_gbs = static_cast<double>(sms) * 512.0 * 64.0 * 4.0 * iters / (t_shfl * 1e-3) / 1e9;
    const double ideal = t_half_s > t_half_l ? t_half_s : t_half_l, serial = static_cast<double>(t_half_s) + t_half_l;
    *shfl_lds_overlap = serial > ideal ? (serial - t_both) / (serial - ideal) : 1.0;
    return EXX_OK;
}
