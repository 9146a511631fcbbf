// exx_pass_b.cu -- instantiation + dispatch of pass B (second b stage, a-axis FFT, K^ multiply, inverse).
#include "exx_inst.cuh"
#include "exx_launch.h"

namespace exx {

template <int TA, int TB, bool FREE, int CHUNK>
static cudaError_t run_b(const ArgsB& args_in, int count, cudaStream_t s, KernelInfo* info, bool launch) {
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

static cudaError_t dispatch_b(const Geometry& g, const ArgsB& args, int count, cudaStream_t s, KernelInfo* info, bool launch) {
#define X(TA_, TB_)                                                                                              \
    if (g.ta == TA_ && g.tb == TB_) {                                                                            \
        if (g.free_bc) return run_b<TA_, TB_, true, chunk_for(TA_, TB_, true)>(args, count, s, info, launch);     \
        return run_b<TA_, TB_, false, chunk_for(TA_, TB_, false)>(args, count, s, info, launch);                  \
    }
    EXX_FOR_EACH_PAIR(X)
#undef X
    return cudaErrorInvalidValue;
}

cudaError_t launch_pass_b(const Geometry& g, const ArgsB& args, int count, cudaStream_t s, KernelInfo* info) {
    return dispatch_b(g, args, count, s, info, true);
}

cudaError_t query_pass_b(const Geometry& g, KernelInfo* info) {
    ArgsB args{};
    args.npch = g.tc / g.chunk;
    return dispatch_b(g, args, 0, nullptr, info, false);
}

bool length_supported(int t) {
    return t == 16 || t == 32 || t == 64 || t == 96 || t == 128 || t == 192 || t == 256;
}

int chunk_of(const Geometry& g) { return chunk_for(g.ta, g.tb, g.free_bc != 0); }

const char* unsupported_geometry_text() {
    return "transform lengths must be in {16,32,64,96,128,192,256}; non-cubic grids only with lengths <= 64";
}

bool geometry_supported(const Geometry& g) {
    if (!length_supported(g.ta) || !length_supported(g.tb) || !length_supported(g.tc)) return false;
    if (g.ta == g.tb && g.tb == g.tc) return true;
    return g.ta <= 64 && g.tb <= 64 && g.tc <= 64;
}

}  // namespace exx
