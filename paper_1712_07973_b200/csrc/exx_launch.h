// exx_launch.h -- internal launch interface between the plan (exx_api.cu) and the instantiated pass kernels.
#pragma once

#include <cuda_runtime.h>

#include "exx_passes.cuh"

namespace exx {

// Geometry of a plan as seen by the kernels.
struct Geometry {
    int ta, tb, tc;      // transform lengths (n periodic, 2n free)
    int free_bc;         // 0 periodic, 1 free
    int chunk_log2;      // W1 layout parameter (CHUNK = 2 or 4)
};

struct KernelInfo {     // what a launcher reports about the instantiation it dispatches to
    int threads;
    int smem_bytes;
    int tiles;           // pass A/C: CTAs per transform (na * R2 / G);  pass B: CTAs per transform (R1 * TC / CHUNK)
};

// Transform lengths the FFT covers.
bool length_supported(int t);
// True if kernels for this (ta,tb,tc,bc) combination are compiled in (cubic grids of every supported length;
// any mix of lengths <= 64).
bool geometry_supported(const Geometry& g);

// Each returns cudaSuccess or the launch/attribute error.  count = transforms in the batch.
cudaError_t launch_pass_a(const Geometry& g, const ArgsAC& args, int count, cudaStream_t s, KernelInfo* info);
cudaError_t launch_pass_b(const Geometry& g, const ArgsB& args, int count, cudaStream_t s, KernelInfo* info);
cudaError_t launch_pass_c(const Geometry& g, const ArgsAC& args, cudaStream_t s, KernelInfo* info);
// Query only (no launch): fills info for the geometry.
cudaError_t query_pass_ac(const Geometry& g, KernelInfo* info);
cudaError_t query_pass_b(const Geometry& g, KernelInfo* info);

// Default CHUNK (log2) for a geometry: the largest of {4,2} whose pass-B tile fits shared memory comfortably.
int default_chunk_log2(int ta, int tb);

// Compile-time tuning shared by the instantiation files -------------------------------------------------------
constexpr int kMaxSmemC = 220 * 1024;                      // pass C: two work buffers + operand stages
constexpr int round_up32(int x) { return (x + 31) / 32 * 32; }

// bytes of pass-C shared memory for a tile of G b2-values with `nstg` operand stages (mirrors CfgAC)
template <int TC, int TB, bool FREE>
constexpr int smem_c_bytes(int g, int nstg) {
    constexpr int PC = Split<TC>::P, QC = Split<TC>::Q, R1 = BSplit<TB>::R1;
    constexpr int NB1 = FREE ? R1 / 2 : R1, NC = FREE ? TC / 2 : TC;
    constexpr int ROW = PC * (QC | 1);
    constexpr int LS = NC + (((QC - NC % 16) % 16) + 16) % 16;
    return 2 * g * (R1 * ROW + (g > 1 ? 4 : 0)) * 16 + nstg * 2 * g * NB1 * LS * 8;
}

// largest G dividing R2 with at most 256 epilogue items per tile whose pass-C tile fits shared memory
template <int TC, int TB, bool FREE>
constexpr int pick_g() {
    constexpr int R2 = BSplit<TB>::R2;
    constexpr int items = (FREE ? BSplit<TB>::R1 / 2 : BSplit<TB>::R1) * Split<TC>::Q;
    int g = 1;
    for (int c = 1; c <= R2; ++c)
        if (R2 % c == 0 && c * items <= 256 && smem_c_bytes<TC, TB, FREE>(c, 1) <= kMaxSmemC) g = c;
    return g;
}

template <int TC, int TB, bool FREE>
struct TuneAC {
    static constexpr int G = pick_g<TC, TB, FREE>();
    using Cfg = CfgAC<TC, TB, FREE, G>;
    static constexpr int NT = round_up32(Cfg::ITEMS_LINE_Q) < 32 ? 32 : round_up32(Cfg::ITEMS_LINE_Q);
    // pass C: more threads than epilogue items when the b-stage (ITEMS_POS items) is wider (free BC)
    static constexpr int NT_C = NT >= 256 ? NT : (Cfg::ITEMS_POS >= 256 ? 256 : (round_up32(Cfg::ITEMS_POS) > NT ? round_up32(Cfg::ITEMS_POS) : NT));
    static constexpr int NSTG_C = smem_c_bytes<TC, TB, FREE>(G, 2) <= kMaxSmemC ? 2 : 1;
    static constexpr int SMEM_C = smem_c_bytes<TC, TB, FREE>(G, NSTG_C);
};

template <int TA, int TB, bool FREE, int CHUNK>
struct TuneB {
    using Cfg = CfgB<TA, TB, FREE, CHUNK>;
    static constexpr int half = round_up32(Cfg::ITEMS_Q / 2);
    static constexpr int NT = half < 64 ? 64 : (half > 512 ? 512 : half);
};

}  // namespace exx
