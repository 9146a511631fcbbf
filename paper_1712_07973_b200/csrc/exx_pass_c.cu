// exx_pass_c.cu -- instantiation + dispatch of pass C (inverse b stage, inverse c-axis FFT, K psi / energy epilogue).
#include "exx_inst.cuh"
#include "exx_launch.h"

namespace exx {

template <int TC, int TB, bool FREE>
static cudaError_t run_c(const ArgsAC& args, cudaStream_t s, KernelInfo* info, bool launch) {
    using T = TuneAC<TC, TB, FREE>;
    using C = typename T::CfgC;
    constexpr int smem = T::SMEM_C;
    static_assert(smem == T::NBUF_C * C::SMEM_C * 16 + (T::NSTG_C * C::OP_DOUBLES + C::RES_DOUBLES) * 8, "pass C shared memory");
    static_assert(!T::WS_C || (T::NBUF_C == 2 && T::NSTG_C == 2), "warp-specialised pass C needs two buffers and two stages");
    constexpr bool ws = T::WS_C;
    constexpr int nt = ws ? 32 * (T::NAW_C + T::NBW_C) : T::NT_C;
    auto kern = ws ? pass_c_ws_kernel<C, T::NAW_C, T::NBW_C, 2, T::MINB_C_WS> : pass_c_kernel<C, T::NT_C, T::NSTG_C, T::NBUF_C, T::MINB_C>;
    static LaunchCache cache;
    int occ = 0;
    if (info) { info->threads = nt; info->smem_bytes = smem; info->tiles = args.na * C::TILES_PER_A; info->ctas_per_sm = 0; info->name = ws ? "pass_c_ws_kernel" : "pass_c_kernel"; }
    if (!launch) return cudaSuccess;
    cudaError_t e = prepare_launch(kern, smem, nt, cache, &occ);
    if (e != cudaSuccess) return e;
    if (info) info->ctas_per_sm = occ;
    kern<<<args.na * C::TILES_PER_A, nt, smem, s>>>(args);
    return cudaGetLastError();
}

static cudaError_t dispatch_c(const Geometry& g, const ArgsAC& args, cudaStream_t s, KernelInfo* info, bool launch) {
#define X(TC_, TB_)                                                                                  \
    if (g.tc == TC_ && g.tb == TB_)                                                                  \
        return g.free_bc ? run_c<TC_, TB_, true>(args, s, info, launch) : run_c<TC_, TB_, false>(args, s, info, launch);
    EXX_FOR_EACH_PAIR(X)
#undef X
    return cudaErrorInvalidValue;
}

cudaError_t launch_pass_c(const Geometry& g, const ArgsAC& args, cudaStream_t s, KernelInfo* info) {
    return dispatch_c(g, args, s, info, true);
}

cudaError_t query_pass_c(const Geometry& g, KernelInfo* info) {
    ArgsAC args{};
    args.na = g.free_bc ? g.ta / 2 : g.ta;
    return dispatch_c(g, args, nullptr, info, false);
}

}  // namespace exx
