// exx_pass_a.cu -- instantiation + dispatch of pass A (co-density, padding, c-axis FFT, first b-axis stage).
#include "exx_inst.cuh"
#include "exx_launch.h"

namespace exx {

template <int TC, int TB, bool FREE>
static cudaError_t run_a(const ArgsAC& args, cudaStream_t s, KernelInfo* info, bool launch) {
    using T = TuneAC<TC, TB, FREE>;
    using C = typename T::CfgA;
    static_assert(T::SMEM_A == C::SMEM_A * 16 + T::NSTG_A * C::OP_DOUBLES * 8, "pass A shared memory");
    constexpr bool ws = T::WS_A;
    constexpr int smem = ws ? T::SMEM_A_WS : T::SMEM_A;
    constexpr int nt = ws ? 32 * (T::NAW + T::NBW) : T::NT_A;
    auto kern = ws ? pass_a_ws_kernel<C, T::NAW, T::NBW, T::NSTG_A_WS, T::MINB_A_WS> : pass_a_kernel<C, T::NT_A, T::NSTG_A, T::MINB_A>;
    static LaunchCache cache;
    int occ = 0;
    if (info) { info->threads = nt; info->smem_bytes = smem; info->tiles = args.na * C::TILES_PER_A; info->ctas_per_sm = 0; info->name = ws ? "pass_a_ws_kernel" : "pass_a_kernel"; }
    if (!launch) return cudaSuccess;
    cudaError_t e = prepare_launch(kern, smem, nt, cache, &occ);
    if (e != cudaSuccess) return e;
    if (info) info->ctas_per_sm = occ;
    kern<<<args.na * C::TILES_PER_A, nt, smem, s>>>(args);
    return cudaGetLastError();
}

static cudaError_t dispatch_a(const Geometry& g, const ArgsAC& args, cudaStream_t s, KernelInfo* info, bool launch) {
#define X(TC_, TB_)                                                                                  \
    if (g.tc == TC_ && g.tb == TB_)                                                                  \
        return g.free_bc ? run_a<TC_, TB_, true>(args, s, info, launch) : run_a<TC_, TB_, false>(args, s, info, launch);
    EXX_FOR_EACH_PAIR(X)
#undef X
    return cudaErrorInvalidValue;
}

cudaError_t launch_pass_a(const Geometry& g, const ArgsAC& args, cudaStream_t s, KernelInfo* info) {
    return dispatch_a(g, args, s, info, true);
}

cudaError_t query_pass_a(const Geometry& g, KernelInfo* info) {
    ArgsAC args{};
    args.na = g.free_bc ? g.ta / 2 : g.ta;
    return dispatch_a(g, args, nullptr, info, false);
}

}  // namespace exx
