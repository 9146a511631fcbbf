// exx_dispatch.cu -- routes a plan's geometry to the translation unit that holds its kernel instantiations (one unit per
// pass and middle-axis length, see exx_inst.cuh) and answers which geometries exist.
#include "exx_inst.cuh"
#include "exx_launch.h"

namespace exx {

#define X(T)                                                                                                                           \
    bool try_pass_a_##T(const Geometry&, const ArgsAC&, const ArgsCX&, cudaStream_t, KernelInfo*, bool, cudaError_t*);                                \
    bool try_pass_b_##T(const Geometry&, const ArgsB&, int, cudaStream_t, KernelInfo*, bool, cudaError_t*);                            \
    bool try_pass_c_##T(const Geometry&, const ArgsAC&, const ArgsCX&, cudaStream_t, KernelInfo*, bool, cudaError_t*);
EXX_ALL_LENGTHS(X)
#undef X

static cudaError_t dispatch_a(const Geometry& g, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info, bool launch) {
    cudaError_t err = cudaErrorInvalidValue;
#define X(T) if (try_pass_a_##T(g, args, extra, s, info, launch, &err)) return err;
    EXX_ALL_LENGTHS(X)
#undef X
    return cudaErrorInvalidValue;
}
static cudaError_t dispatch_b(const Geometry& g, const ArgsB& args, int count, cudaStream_t s, KernelInfo* info, bool launch) {
    cudaError_t err = cudaErrorInvalidValue;
#define X(T) if (try_pass_b_##T(g, args, count, s, info, launch, &err)) return err;
    EXX_ALL_LENGTHS(X)
#undef X
    return cudaErrorInvalidValue;
}
static cudaError_t dispatch_c(const Geometry& g, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info, bool launch) {
    cudaError_t err = cudaErrorInvalidValue;
#define X(T) if (try_pass_c_##T(g, args, extra, s, info, launch, &err)) return err;
    EXX_ALL_LENGTHS(X)
#undef X
    return cudaErrorInvalidValue;
}

cudaError_t launch_pass_a(const Geometry& g, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info) { return dispatch_a(g, args, extra, s, info, true); }
cudaError_t launch_pass_b(const Geometry& g, const ArgsB& args, int count, cudaStream_t s, KernelInfo* info) { return dispatch_b(g, args, count, s, info, true); }
cudaError_t launch_pass_c(const Geometry& g, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info) { return dispatch_c(g, args, extra, s, info, true); }

cudaError_t query_pass_a(const Geometry& g, KernelInfo* info) {
    ArgsAC args{};
    args.na = g.free_bc ? g.ta / 2 : g.ta;
    ArgsCX extra{};
    return dispatch_a(g, args, extra, nullptr, info, false);
}
cudaError_t query_pass_b(const Geometry& g, KernelInfo* info) {
    ArgsB args{};
    args.npch = g.tc / g.chunk;
    return dispatch_b(g, args, 0, nullptr, info, false);
}
cudaError_t query_pass_c(const Geometry& g, KernelInfo* info) {
    ArgsAC args{};
    args.na = g.free_bc ? g.ta / 2 : g.ta;
    ArgsCX extra{};
    return dispatch_c(g, args, extra, nullptr, info, false);
}

bool length_supported(int t) { return is_length(t); }

int chunk_of(const Geometry& g) { return chunk_for(g.ta, g.tb, g.free_bc != 0); }

const char* unsupported_geometry_text() {
    return "transform lengths (n periodic, 2n free) must be in {16,32,48,64,96,128,144,192,256} (any mix over the axes) or a cubic "
           "transform grid of 24 or 72";
}

bool geometry_supported(const Geometry& g) {
    if (!is_length(g.ta) || !is_length(g.tb) || !is_length(g.tc)) return false;
    const bool cubic = g.ta == g.tb && g.tb == g.tc;
    if (!(cubic || (is_main_length(g.ta) && is_main_length(g.tb) && is_main_length(g.tc)))) return false;
    Geometry q = g;
    q.chunk = chunk_of(g);
    KernelInfo info{};
    return query_pass_a(q, &info) == cudaSuccess && query_pass_b(q, &info) == cudaSuccess && query_pass_c(q, &info) == cudaSuccess;
}

}  // namespace exx
