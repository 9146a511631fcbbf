// exx_pass_a.cu -- instantiation + dispatch of pass A (co-density, padding, c-axis FFT, first b-axis stage).
#include "exx_inst.cuh"
#include "exx_launch.h"

namespace exx {

template <int TC, int TB, bool FREE>
static cudaError_t run_a(const ArgsAC& args, int count, cudaStream_t s, KernelInfo* info, bool launch) {
    using T = TuneAC<TC, TB, FREE>;
    using C = typename T::Cfg;
    constexpr int smem = C::SMEM_ELEMS * static_cast<int>(sizeof(double2));
    auto kern = pass_a_kernel<C, T::NT>;
    if (info) { info->threads = T::NT; info->smem_bytes = smem; info->tiles = args.na * C::TILES_PER_A; }
    if (!launch) return cudaSuccess;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    dim3 grid(args.na * C::TILES_PER_A, count);
    kern<<<grid, T::NT, smem, s>>>(args);
    return cudaGetLastError();
}

static cudaError_t dispatch_a(const Geometry& g, const ArgsAC& args, int count, cudaStream_t s, KernelInfo* info, bool launch) {
#define X(TC_, TB_)                                                                                  \
    if (g.tc == TC_ && g.tb == TB_)                                                                  \
        return g.free_bc ? run_a<TC_, TB_, true>(args, count, s, info, launch)                        \
                         : run_a<TC_, TB_, false>(args, count, s, info, launch);
    EXX_FOR_EACH_PAIR(X)
#undef X
    return cudaErrorInvalidValue;
}

cudaError_t launch_pass_a(const Geometry& g, const ArgsAC& args, int count, cudaStream_t s, KernelInfo* info) {
    return dispatch_a(g, args, count, s, info, true);
}

cudaError_t query_pass_ac(const Geometry& g, KernelInfo* info) {
    ArgsAC args{};
    args.na = g.free_bc ? g.ta / 2 : g.ta;
    return dispatch_a(g, args, 0, nullptr, info, false);
}

}  // namespace exx
