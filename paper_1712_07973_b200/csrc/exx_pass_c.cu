// exx_pass_c.cu -- instantiation + dispatch of pass C (inverse b stage, inverse c-axis FFT, K psi / energy epilogue).
#include "exx_inst.cuh"
#include "exx_launch.h"

namespace exx {

template <int TC, int TB, bool FREE>
static cudaError_t run_c(const ArgsAC& args, cudaStream_t s, KernelInfo* info) {
    using T = TuneAC<TC, TB, FREE>;
    using C = typename T::Cfg;
    constexpr int NSTG = T::NSTG_C;                          // operand stages (psi_j, psi_l lines in flight)
    constexpr int smem = T::SMEM_C;
    static_assert(smem == (2 * C::SMEM_C * 16 + NSTG * C::OP_DOUBLES * 8) && smem <= kMaxSmemC, "pass C shared memory");
    auto kern = pass_c_kernel<C, T::NT_C, NSTG>;
    if (info) { info->threads = T::NT_C; info->smem_bytes = smem; info->tiles = args.na * C::TILES_PER_A; }
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    kern<<<args.na * C::TILES_PER_A, T::NT_C, smem, s>>>(args);
    return cudaGetLastError();
}

cudaError_t launch_pass_c(const Geometry& g, const ArgsAC& args, cudaStream_t s, KernelInfo* info) {
#define X(TC_, TB_)                                                                \
    if (g.tc == TC_ && g.tb == TB_)                                                \
        return g.free_bc ? run_c<TC_, TB_, true>(args, s, info) : run_c<TC_, TB_, false>(args, s, info);
    EXX_FOR_EACH_PAIR(X)
#undef X
    return cudaErrorInvalidValue;
}

}  // namespace exx
