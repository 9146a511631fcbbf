// exx_pass_b.cu -- instantiation + dispatch of pass B (second b stage, a-axis FFT, K^ multiply, inverse) for ONE
// middle-axis length: compiled once per length with -DEXX_TB=<length> (see exx_inst.cuh).
#include "exx_inst.cuh"
#include "exx_launch.h"

#ifndef EXX_TB
#error "compile with -DEXX_TB=<middle-axis transform length>"
#endif

namespace exx {

template <int TA, int TB, bool FREE>
static cudaError_t run_b(const ArgsB& args_in, int count, cudaStream_t s, KernelInfo* info, bool launch) {
    constexpr int CHUNK = ChunkOf<TA, TB, FREE>::value;
    using T = TuneB<TA, TB, FREE, CHUNK>;
    using C = typename T::Cfg;
    if constexpr (!T::FITS) {
        return cudaErrorInvalidValue;
    } else {
        auto kern = T::WS ? pass_b_ws_kernel<C, T::NY, T::NX, T::MINB, false>
                  : T::WSF ? pass_b_ws_kernel<C, T::NY, T::NX, T::MINB, true> : pass_b_kernel<C, T::NT, T::MINB>;
        static LaunchCache cache;
        int occ = 0, sms = 148;
        if (info) { info->threads = T::NT; info->smem_bytes = T::SMEM; info->tiles = C::R1 * args_in.npch; info->ctas_per_sm = 0; info->name = (T::WS || T::WSF) ? "pass_b_ws_kernel" : "pass_b_kernel"; }
        if (!launch) return cudaSuccess;
        cudaError_t e = prepare_launch(kern, T::SMEM, T::NT, cache, &occ, &sms);
        if (e != cudaSuccess) return e;
        if (info) info->ctas_per_sm = occ;
        ArgsB args = args_in;
        args.count = count;
        args.ntiles = count * C::R1 * args.npch;
        const int slots = sms * (occ > 0 ? occ : 1);
        const int grid = args.ntiles < slots ? args.ntiles : slots;
        kern<<<grid, T::NT, T::SMEM, s>>>(args);
        return cudaGetLastError();
    }
}

bool EXX_CAT(try_pass_b_, EXX_TB)(const Geometry& g, const ArgsB& args, int count, cudaStream_t s, KernelInfo* info, bool launch, cudaError_t* err) {
    if (g.tb != EXX_TB) return false;
#define X(TA_)                                                                                                       \
    if (g.ta == TA_) {                                                                                               \
        *err = g.free_bc ? run_b<TA_, EXX_TB, true>(args, count, s, info, launch) : run_b<TA_, EXX_TB, false>(args, count, s, info, launch); \
        return true;                                                                                                 \
    }
    if constexpr (is_main_length(EXX_TB)) {
        EXX_MAIN_LENGTHS(X)
    } else {
        X(EXX_TB)
    }
#undef X
    return false;
}

}  // namespace exx
