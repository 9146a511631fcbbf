// exx_pass_b.cu -- instantiation + dispatch of pass B (second b stage, a-axis FFT, K^ multiply, inverse).
#include "exx_inst.cuh"
#include "exx_launch.h"

namespace exx {

constexpr int kMaxSmemB = 200 * 1024;

template <int TA, int TB, bool FREE, int CHUNK>
static cudaError_t run_b(const ArgsB& args, int count, cudaStream_t s, KernelInfo* info, bool launch) {
    using T = TuneB<TA, TB, FREE, CHUNK>;
    using C = typename T::Cfg;
    constexpr int smem = C::SMEM_ELEMS * static_cast<int>(sizeof(double2));
    if constexpr (smem > kMaxSmemB) {
        return cudaErrorInvalidValue;                      // this CHUNK does not fit; the plan picks the other one
    } else {
        auto kern = pass_b_kernel<C, T::NT>;
        if (info) { info->threads = T::NT; info->smem_bytes = smem; info->tiles = C::R1 * args.npch; }
        if (!launch) return cudaSuccess;
        static bool attr_done = false;
        if (!attr_done) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e != cudaSuccess) return e;
            attr_done = true;
        }
        dim3 grid(C::R1 * args.npch, count);
        kern<<<grid, T::NT, smem, s>>>(args);
        return cudaGetLastError();
    }
}

static cudaError_t dispatch_b(const Geometry& g, const ArgsB& args, int count, cudaStream_t s, KernelInfo* info, bool launch) {
#define X(TA_, TB_)                                                                                              \
    if (g.ta == TA_ && g.tb == TB_) {                                                                            \
        if (g.chunk_log2 == 2)                                                                                   \
            return g.free_bc ? run_b<TA_, TB_, true, 4>(args, count, s, info, launch)                             \
                             : run_b<TA_, TB_, false, 4>(args, count, s, info, launch);                           \
        return g.free_bc ? run_b<TA_, TB_, true, 2>(args, count, s, info, launch)                                 \
                         : run_b<TA_, TB_, false, 2>(args, count, s, info, launch);                               \
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
    args.npch = g.tc >> g.chunk_log2;
    return dispatch_b(g, args, 0, nullptr, info, false);
}

int default_chunk_log2(int ta, int tb) {
    Geometry g{ta, tb, 16, 0, 2};
    KernelInfo info{};
    if (query_pass_b(g, &info) == cudaSuccess && info.smem_bytes <= 100 * 1024) return 2;
    return 1;
}

bool length_supported(int t) {
    return t == 16 || t == 32 || t == 64 || t == 96 || t == 128 || t == 192 || t == 256;
}

bool geometry_supported(const Geometry& g) {
    if (!length_supported(g.ta) || !length_supported(g.tb) || !length_supported(g.tc)) return false;
    if (g.ta == g.tb && g.tb == g.tc) return true;
    return g.ta <= 64 && g.tb <= 64 && g.tc <= 64;
}

}  // namespace exx
