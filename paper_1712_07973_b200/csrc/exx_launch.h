// exx_launch.h -- internal launch interface between the plan (exx_api.cu) and the instantiated pass kernels.
#pragma once

#include <cuda_runtime.h>

#include <mutex>

#include "exx_passes.cuh"

namespace exx {

// Geometry of a plan as seen by the kernels.
struct Geometry {
    int ta, tb, tc;      // transform lengths (n periodic, 2n free)
    int free_bc;         // 0 periodic, 1 free
    int chunk;           // W1 layout parameter (CHUNK = 2 or 4), = chunk_for(ta, tb, free_bc)
};

struct KernelInfo {     // what a launcher reports about the instantiation it dispatches to
    int threads;
    int smem_bytes;
    int tiles;           // pass A / C: CTAs per launch (na * R2 / G);  pass B: blocks per transform (R1 * TC / CHUNK)
    int ctas_per_sm;     // occupancy the launcher sized its grid for (pass B: persistent grid = SMs * this)
    const char* name;    // kernel the launcher dispatches to for this geometry
    int needs_w1_map;    // passes A / C: the kernel moves its W1 tile through ArgsCX::w1_map (TMA tensor-box store / copy)
};

// Transform lengths the FFT covers.
bool length_supported(int t);
// True if kernels for this (ta,tb,tc,bc) combination are compiled in: every mix of the main lengths
// {16,32,48,64,96,128,144,192,256}, cubic transform grids of the extra lengths {24,72}.
bool geometry_supported(const Geometry& g);
// W1 layout parameter CHUNK of a supported geometry, and the text of the EXX_ERR_UNSUPPORTED_SIZE message.
int chunk_of(const Geometry& g);
const char* unsupported_geometry_text();

// Each returns cudaSuccess or the launch/attribute error.  count = transforms in the batch.
cudaError_t launch_pass_a(const Geometry& g, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info);
cudaError_t launch_pass_b(const Geometry& g, const ArgsB& args, int count, cudaStream_t s, KernelInfo* info);
cudaError_t launch_pass_c(const Geometry& g, const ArgsAC& args, const ArgsCX& extra, cudaStream_t s, KernelInfo* info);
// Query only (no launch): fills info for the geometry.
cudaError_t query_pass_a(const Geometry& g, KernelInfo* info);
cudaError_t query_pass_b(const Geometry& g, KernelInfo* info);
cudaError_t query_pass_c(const Geometry& g, KernelInfo* info);

// Per-kernel, per-device launch state.  cudaFuncSetAttribute(MaxDynamicSharedMemorySize) applies to the CURRENT device
// only, so the opt-in and the occupancy it yields are cached per device ordinal (plans on different GPUs of one process
// are independent); the mutex makes the first launches of two host threads safe.
constexpr int kMaxDevices = 64;
struct LaunchCache {
    std::mutex m;
    int occ[kMaxDevices];
    int sms[kMaxDevices];
    LaunchCache() { for (int d = 0; d < kMaxDevices; ++d) { occ[d] = -1; sms[d] = 0; } }
};
// Makes `kern` launchable with `smem` bytes of dynamic shared memory on the current device; reports the resident CTAs
// per SM for `nt` threads and the device's SM count.
template <class K>
inline cudaError_t prepare_launch(K kern, int smem, int nt, LaunchCache& c, int* ctas_per_sm, int* sm_count = nullptr) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(c.m);
    if (c.occ[dev] < 0) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        int occ = 0, sms = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, nt, smem);
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        c.sms[dev] = sms > 0 ? sms : 148;
        c.occ[dev] = occ;
    }
    *ctas_per_sm = c.occ[dev];
    if (sm_count) *sm_count = c.sms[dev];
    return cudaSuccess;
}

// Compile-time tuning shared by the instantiation files -------------------------------------------------------
constexpr int kSmemPerSM = 227 * 1024;                     // usable shared memory per SM (and per CTA, opt-in)
constexpr int kMaxSmemAC = 216 * 1024;                     // passes A / C: work buffer(s) + operand stages
constexpr int round_up32(int x) { return (x + 31) / 32 * 32; }
constexpr int imin(int a, int b) { return a < b ? a : b; }
constexpr int imax(int a, int b) { return a > b ? a : b; }

// bytes of dynamic shared memory of pass A (one work buffer) / pass C (two work buffers, R1 lines per b2) for a tile of
// g b2-values with `nstg` operand stages (mirrors CfgAC)
template <int TC, int TB, bool FREE>
constexpr int smem_ac_bytes(int g, int nstg, bool pass_c, int nbuf = 2) {
    constexpr int PC = Split<TC>::P, QC = Split<TC>::Q, R1 = BSplit<TB>::R1;
    constexpr int NB1 = FREE ? R1 / 2 : R1, NC = FREE ? TC / 2 : TC;
    constexpr int ROW = PC * (QC | 1);
    constexpr int LS = NC + (((QC - NC % 16) % 16) + 16) % 16;
    const int work = g * ((pass_c ? R1 : NB1) * ROW + (g > 1 ? 4 : 0)) * 16;
    const int lines = g * NB1 * LS * 8;                    // one orbital's lines of the tile
    return (pass_c ? nbuf : 1) * work + nstg * lines + (pass_c ? 2 * lines : 0);
}

// largest G dividing R2 with at most 256 (line, n2) items per tile whose tile fits shared memory
template <int TC, int TB, bool FREE>
constexpr int pick_g(bool pass_c, int max_bytes) {
    constexpr int R2 = BSplit<TB>::R2;
    constexpr int items = (FREE ? BSplit<TB>::R1 / 2 : BSplit<TB>::R1) * Split<TC>::Q;
    int g = 1;
    for (int c = 1; c <= R2; ++c)
        if (R2 % c == 0 && c * items <= 256 && smem_ac_bytes<TC, TB, FREE>(c, 1, pass_c) <= max_bytes) g = c;
    return g;
}

// resident CTAs per SM to compile for: limited by shared memory, by a register floor per thread, and by `cap`; among
// the admissible counts the one that wastes the fewest CTA slots in the last wave of a cubic grid's `tiles` CTAs on 148
// SMs wins (a tile is a long loop over the batch, so a ragged last wave costs a whole loop), ties -> more CTAs
constexpr int pick_minb(int smem, int nt, int reg_floor, int cap, int tiles) {       // smem: dynamic + static bytes
    const int maxb = imax(1, imin(imin((kSmemPerSM + 1024) / (smem + 1024), 65536 / (nt * reg_floor)), cap));
    int best = 1, best_eff = -1;
    for (int b = 1; b <= maxb; ++b) {
        const int slots = 148 * b, waves = (tiles + slots - 1) / slots;
        const int eff = tiles * 1000 / (waves * slots) + (b > 1 ? 100 : 0);    // co-residency itself is worth 10 %
        if (eff >= best_eff) { best_eff = eff; best = b; }
    }
    return best;
}

// warps (<= cap) for `items` equal work items: the count that wastes the fewest lane-rounds, ties -> more warps
constexpr int pick_line_warps(int items, int cap) {
    int best = 1, best_waste = 1 << 30;
    for (int w = 1; w <= cap; ++w) {
        const int rounds = (items + 32 * w - 1) / (32 * w);
        const int waste = rounds * 32 * w - items;
        if (waste <= best_waste) { best_waste = waste; best = w; }
    }
    return best;
}

template <int TC, int TB, bool FREE, int CHUNK_>
struct TuneAC {
    static constexpr int CHUNK = CHUNK_;
    // ---- pass C
    static constexpr int G_C = pick_g<TC, TB, FREE>(true, kMaxSmemAC / 2);
    using CfgC = CfgAC<TC, TB, FREE, G_C, CHUNK>;
    // threads: one per (line, n2) item of C2 and, where that is fewer than the columns of C0 (free BC: the tile has twice as
    // many columns as C2 items), still only that many once they are >= 128 -- the warps that would idle through C1 / C2
    // are dropped, each thread takes two columns in C0, and the larger register budget admits the early gather
    // (256^3 free: pass C -6 %)
    static constexpr int NT_C_WIDE = imax(32, round_up32(imax(CfgC::ITEMS_LINE_Q, imin(CfgC::ITEMS_POS, 256))));
    static constexpr int NT_C = (CfgC::ITEMS_LINE_Q >= 128 && round_up32(CfgC::ITEMS_LINE_Q) < NT_C_WIDE) ? round_up32(CfgC::ITEMS_LINE_Q) : NT_C_WIDE;
    // double-buffered W1 tile where it fits next to one operand stage and the resident lines, else single-buffered
    // W1 tile buffers (NBUF) and operand stages (NSTG): the deepest pipeline with which two CTAs share an SM (the other
    // CTA then covers what a shallower pipeline exposes), else the deepest one that fits at all
    static constexpr int kStaticC = (TC + TB) * 16 + 1280;
    static constexpr bool two_fit(int nbuf, int nstg) {
        return (smem_ac_bytes<TC, TB, FREE>(G_C, nstg, true, nbuf) + kStaticC) * 2 <= kSmemPerSM + 1024;
    }
    static constexpr bool one_fits(int nbuf, int nstg) { return smem_ac_bytes<TC, TB, FREE>(G_C, nstg, true, nbuf) <= kMaxSmemAC; }
    static constexpr int NBUF_C = two_fit(2, 2) ? 2 : two_fit(1, 2) ? 1 : two_fit(1, 1) ? 1 : (one_fits(2, 2) || one_fits(2, 1)) ? 2 : 1;
    static constexpr int NSTG_C = two_fit(2, 2) ? 2 : two_fit(1, 2) ? 2 : two_fit(1, 1) ? 1 : one_fits(NBUF_C, 2) ? 2 : 1;
    static constexpr int SMEM_C = smem_ac_bytes<TC, TB, FREE>(G_C, NSTG_C, true, NBUF_C);
    static constexpr int MINB_C = pick_minb(SMEM_C + (TC + TB) * 16 + 256, NT_C, 128, 4, CfgC::NC * CfgC::TILES_PER_A);
    // single-buffered pass C: gather the next W1 tile from inside C2 (pass_c_kernel EARLY) where the register file leaves
    // room for the PC complex inputs of every C2 item next to the accumulators without spilling them
#if defined(EXX_EARLY_C_ALL)
    static constexpr bool EARLY_C = NBUF_C == 1;
#elif defined(EXX_EARLY_C_NONE)
    static constexpr bool EARLY_C = false;
#else
    static constexpr bool EARLY_C = NBUF_C == 1 && 65536 / (NT_C * MINB_C) >= 160;
#endif
    // ---- pass A
    static constexpr int G_A = pick_g<TC, TB, FREE>(false, kMaxSmemAC / 3);
    using CfgA = CfgAC<TC, TB, FREE, G_A, CHUNK>;
    static constexpr int NT_A = imax(32, round_up32(imax(CfgA::ITEMS_LINE_Q, imin(CfgA::ITEMS_POS, 256))));
    static constexpr int NSTG_A = 2;
    static constexpr int SMEM_A = smem_ac_bytes<TC, TB, FREE>(G_A, NSTG_A, false);
    static constexpr int MINB_A = pick_minb(SMEM_A + (TC + TB) * 16 + 64, NT_A, 96, 4, CfgA::NC * CfgA::TILES_PER_A);
    // ---- pass C, warp-specialised: only where two tile buffers + two operand stages still let two CTAs share an SM
    static constexpr bool WS_C = TC >= 96 && two_fit(2, 2);
    // gather + C0 warps: one keeps up with six line warps for periodic grids (measured); the pruned 2n-point stage of
    // free BC carries a larger share of the work
    static constexpr int NAW_C = FREE ? 2 : 1;
    static constexpr int NBW_C = pick_line_warps(CfgC::ITEMS_LINE_Q, 6);
    static constexpr int MINB_C_WS = pick_minb(SMEM_C + kStaticC, 32 * (NAW_C + NBW_C), 96, 2, CfgC::NC * CfgC::TILES_PER_A);
    // ---- pass A, warp-specialised (lengths >= 96): line warps for A0/A1, column warps for A2, two work buffers
    static constexpr bool WS_A = TC >= 96;
    static constexpr int NAW = pick_line_warps(imax(CfgA::ITEMS_LINE_Q, CfgA::ITEMS_LINE_P), 6);
    static constexpr int NBW = imax(2, 8 - NAW);
    static constexpr int kStaticA = (TC + TB) * 16 + 128;
    static constexpr int NSTG_A_WS =                       // one operand stage if that is what lets two CTAs share an SM
        (2 * CfgA::SMEM_A * 16 + 2 * CfgA::OP_DOUBLES * 8 + kStaticA) * 2 <= kSmemPerSM + 1024 ? 2 :
        (2 * CfgA::SMEM_A * 16 + 1 * CfgA::OP_DOUBLES * 8 + kStaticA) * 2 <= kSmemPerSM + 1024 ? 1 : 2;
    static constexpr int SMEM_A_WS = 2 * CfgA::SMEM_A * 16 + NSTG_A_WS * CfgA::OP_DOUBLES * 8;
    static constexpr int MINB_A_WS = pick_minb(SMEM_A_WS + kStaticA, 32 * (NAW + NBW), 96, 2, CfgA::NC * CfgA::TILES_PER_A);
    // ---- pass A with the TMA tile store (pass_a_ts_kernel): two dense R1 x TC work buffers
    static constexpr int kBufTS = BSplit<TB>::R1 * TC * 16;
    static constexpr int NSTG_A_TS =
        (2 * kBufTS + 2 * CfgA::OP_DOUBLES * 8 + kStaticA) * 2 <= kSmemPerSM + 1024 ? 2 :
        (2 * kBufTS + 1 * CfgA::OP_DOUBLES * 8 + kStaticA) * 2 <= kSmemPerSM + 1024 ? 1 : 2;
    static constexpr int SMEM_A_TS = 2 * kBufTS + NSTG_A_TS * CfgA::OP_DOUBLES * 8;
    static constexpr int MINB_A_TS = pick_minb(SMEM_A_TS + kStaticA, 32 * (NAW + NBW), 96, 2, CfgA::NC * CfgA::TILES_PER_A);
    static constexpr bool TS_A = WS_A && pass_a_tma_store<CfgA>() && SMEM_A_TS <= kMaxSmemAC;
    static_assert(SMEM_C <= kMaxSmemAC && SMEM_A <= kMaxSmemAC && SMEM_A_WS <= kMaxSmemAC, "tile does not fit shared memory");
};

template <int TA, int TB, bool FREE, int CHUNK>
struct TuneB {
    using Cfg = CfgB<TA, TB, FREE, CHUNK>;
    // warp-specialised variant (column warps + row warps, two block buffers) where it fits and the block is big enough
    // to feed both kinds of warps: WS with two full work buffers, else (free BC) WSF with NA-row buffers and per-warp
    // expansion scratch; else work + landing buffer with CTA barriers
    static constexpr int NY = Cfg::NGRP <= 12 ? Cfg::NGRP : Cfg::NGRP / 2;       // column warps
    // row warps: 4 (2, 3, 5, 6 measured slower at 96^3 and 256^3 free); 6 where eight column warps leave the registers for
    // them and the (a, pin) items of a block split evenly over 192 threads (192^3: pass B -5.5 %, measured after B4 had
    // become an in-place stage + TMA row stores)
    static constexpr int NX = (!FREE && NY == 8 && Cfg::ITEMS_IO % 192 == 0) ? 6 : 4;
    static constexpr bool kBig = Cfg::NGRP >= 6 && (Cfg::NGRP <= 12 || Cfg::NGRP % 2 == 0);
    static constexpr int SMEM_WS = (2 * Cfg::WORK_ELEMS + 2 * TA) * 16;
    static constexpr int SMEM_WSF = (2 * Cfg::P_ELEMS + NY * Cfg::E_ELEMS + 2 * TA) * 16;
    static constexpr bool WS = kBig && SMEM_WS <= kMaxSmemB;
    static constexpr bool WSF = kBig && !WS && FREE && SMEM_WSF <= kMaxSmemB;
    static constexpr int SMEM = WS ? SMEM_WS : WSF ? SMEM_WSF : Cfg::SMEM_BYTES;
    // one warp per column group, at most 16 warps; small blocks share an SM (persistent grid = SMs * MINB)
    static constexpr int NT = (WS || WSF) ? 32 * (NY + NX) : 32 * imin(Cfg::NGRP, 16);
    static constexpr int MINB = imax(1, imin(imin(kSmemPerSM / (SMEM + 1024), imax(1, 512 / NT)), 8));
    static constexpr bool FITS = SMEM <= kMaxSmemB;
};

}  // namespace exx
