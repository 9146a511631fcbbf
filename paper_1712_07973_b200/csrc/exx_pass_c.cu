// exx_pass_c.cu -- instantiation + dispatch of pass C (inverse b stage, inverse c-axis FFT, K psi / energy epilogue) for
// ONE middle-axis length: compiled once per length with -DEXX_TB=<length> (see exx_inst.cuh).
#include "exx_inst.cuh"
#include "exx_launch.h"

#ifndef EXX_TB
#error "compile with -DEXX_TB=<middle-axis transform length>"
#endif

namespace exx {

template <int TC, int TB, bool FREE, int CHUNK>
static cudaError_t run_c_chunk(const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info, bool launch) {
    using T = TuneAC<TC, TB, FREE, CHUNK>;
    using C = typename T::CfgC;
    constexpr int smem = T::SMEM_C;
    static_assert(smem == T::NBUF_C * C::SMEM_C * 16 + (T::NSTG_C * C::OP_DOUBLES + C::RES_DOUBLES) * 8, "pass C shared memory");
    static_assert(!T::WS_C || (T::NBUF_C == 2 && T::NSTG_C == 2), "warp-specialised pass C needs two buffers and two stages");
    constexpr bool ws = T::WS_C;
    constexpr int nt = ws ? 32 * (T::NAW_C + T::NBW_C) : T::NT_C;
    static LaunchCache cache;
    int occ = 0;
    if (info) {
        info->threads = nt; info->smem_bytes = smem; info->tiles = args.na * C::TILES_PER_A; info->ctas_per_sm = 0;
        info->name = ws ? "pass_c_ws_kernel" : "pass_c_kernel";
        info->needs_w1_map = (!ws && pass_c_tma_gather<C, T::NBUF_C>()) ? 1 : 0;
    }
    if (!launch) return cudaSuccess;
    cudaError_t e;
    if constexpr (ws) {
        auto kern = pass_c_ws_kernel<C, T::NAW_C, T::NBW_C, 2, T::MINB_C_WS>;
        e = prepare_launch(kern, smem, nt, cache, &occ);
        if (e != cudaSuccess) return e;
        kern<<<args.na * C::TILES_PER_A, nt, smem, s>>>(args);
    } else {
        auto kern = pass_c_kernel<C, T::NT_C, T::NSTG_C, T::NBUF_C, T::MINB_C, T::EARLY_C>;
        e = prepare_launch(kern, smem, nt, cache, &occ);
        if (e != cudaSuccess) return e;
        kern<<<args.na * C::TILES_PER_A, nt, smem, s>>>(args, extra);
    }
    if (info) info->ctas_per_sm = occ;
    return cudaGetLastError();
}

template <int TC, int TB, bool FREE>
static cudaError_t run_c(int chunk, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info, bool launch) {
    if constexpr (chunk_possible<TB, FREE, 4>()) { if (chunk == 4) return run_c_chunk<TC, TB, FREE, 4>(args, extra, s, info, launch); }
    if constexpr (chunk_possible<TB, FREE, 2>()) { if (chunk == 2) return run_c_chunk<TC, TB, FREE, 2>(args, extra, s, info, launch); }
    if constexpr (chunk_possible<TB, FREE, 1>()) { if (chunk == 1) return run_c_chunk<TC, TB, FREE, 1>(args, extra, s, info, launch); }
    return cudaErrorInvalidValue;
}

bool EXX_CAT(try_pass_c_, EXX_TB)(const Geometry& g, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info, bool launch, cudaError_t* err) {
    if (g.tb != EXX_TB) return false;
#define X(TC_)                                                                                                       \
    if (g.tc == TC_) {                                                                                               \
        *err = g.free_bc ? run_c<TC_, EXX_TB, true>(g.chunk, args, extra, s, info, launch) : run_c<TC_, EXX_TB, false>(g.chunk, args, extra, s, info, launch); \
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
