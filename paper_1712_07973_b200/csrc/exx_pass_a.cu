// exx_pass_a.cu -- instantiation + dispatch of pass A (co-density, padding, c-axis FFT, first b-axis stage) for ONE
// middle-axis length: compiled once per length with -DEXX_TB=<length> (see exx_inst.cuh).
#include "exx_inst.cuh"
#include "exx_launch.h"

#ifndef EXX_TB
#error "compile with -DEXX_TB=<middle-axis transform length>"
#endif

namespace exx {

template <int TC, int TB, bool FREE, int CHUNK>
static cudaError_t run_a_chunk(const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info, bool launch) {
    using T = TuneAC<TC, TB, FREE, CHUNK>;
    using C = typename T::CfgA;
    static_assert(T::SMEM_A == C::SMEM_A * 16 + T::NSTG_A * C::OP_DOUBLES * 8, "pass A shared memory");
    constexpr bool ws = T::WS_A, ts = T::TS_A;
    constexpr int smem = ts ? T::SMEM_A_TS : ws ? T::SMEM_A_WS : T::SMEM_A;
    constexpr int nt = ws ? 32 * (T::NAW + T::NBW) : T::NT_A;
    static LaunchCache cache;
    int occ = 0;
    if (info) {
        info->threads = nt; info->smem_bytes = smem; info->tiles = args.na * C::TILES_PER_A; info->ctas_per_sm = 0;
        info->name = ts ? "pass_a_ts_kernel" : ws ? "pass_a_ws_kernel" : "pass_a_kernel";
        info->needs_w1_map = ts ? 1 : 0;
    }
    if (!launch) return cudaSuccess;
    cudaError_t e;
    if constexpr (ts) {
        auto kern = pass_a_ts_kernel<C, T::NAW, T::NBW, T::NSTG_A_TS, T::MINB_A_TS>;
        e = prepare_launch(kern, smem, nt, cache, &occ);
        if (e != cudaSuccess) return e;
        kern<<<args.na * C::TILES_PER_A, nt, smem, s>>>(args, extra);
    } else {
        auto kern = ws ? pass_a_ws_kernel<C, T::NAW, T::NBW, T::NSTG_A_WS, T::MINB_A_WS> : pass_a_kernel<C, T::NT_A, T::NSTG_A, T::MINB_A>;
        e = prepare_launch(kern, smem, nt, cache, &occ);
        if (e != cudaSuccess) return e;
        kern<<<args.na * C::TILES_PER_A, nt, smem, s>>>(args);
    }
    if (info) info->ctas_per_sm = occ;
    return cudaGetLastError();
}

template <int TC, int TB, bool FREE>
static cudaError_t run_a(int chunk, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info, bool launch) {
    if constexpr (chunk_possible<TB, FREE, 4>()) { if (chunk == 4) return run_a_chunk<TC, TB, FREE, 4>(args, extra, s, info, launch); }
    if constexpr (chunk_possible<TB, FREE, 2>()) { if (chunk == 2) return run_a_chunk<TC, TB, FREE, 2>(args, extra, s, info, launch); }
    if constexpr (chunk_possible<TB, FREE, 1>()) { if (chunk == 1) return run_a_chunk<TC, TB, FREE, 1>(args, extra, s, info, launch); }
    return cudaErrorInvalidValue;
}

// true if this translation unit owns the geometry (g.tb == EXX_TB and a compiled g.tc); *err then holds the outcome
bool EXX_CAT(try_pass_a_, EXX_TB)(const Geometry& g, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info, bool launch, cudaError_t* err) {
    if (g.tb != EXX_TB) return false;
#define X(TC_)                                                                                                       \
    if (g.tc == TC_) {                                                                                               \
        *err = g.free_bc ? run_a<TC_, EXX_TB, true>(g.chunk, args, extra, s, info, launch) : run_a<TC_, EXX_TB, false>(g.chunk, args, extra, s, info, launch); \
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
