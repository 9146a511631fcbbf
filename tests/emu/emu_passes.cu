// Host emulation of the pass kernels: runs the SAME per-work-item phase functions as the CUDA kernels
// (paper_1712_07973_b200/csrc/exx_passes.cuh), sequentially on the CPU, one CTA at a time.
// Test harness only (tests/test_host_emulation.py): validates index algebra, twiddles, pruning and the
// epilogue against the oracle without a GPU.  Not part of the product library.
#include <cstdio>
#include <cstring>
#include <vector>

#include "exx_passes.cuh"

using namespace exx;

template <int TA, int TB, int TC, bool FREE, int G, int CHUNK>
static int emu_batch(const double* psi, double* kpsi, int i, double fi, int count, const XformDesc* desc,
                     const double2* twa, const double2* twc, const double2* rootsb, const double* ks,
                     double* e_out /*[count][2]*/) {
    using AC = CfgAC<TC, TB, FREE, G>;
    static_assert(CHUNK == 2 || CHUNK == 4, "chunk");
    using B = CfgB<TA, TB, FREE, CHUNK>;
    const int na = B::NA;
    const long long m_points = static_cast<long long>(na) * AC::NB * AC::NC;
    std::vector<double2> w1(static_cast<size_t>(count) * na * TB * TC);
    const int ntiles = na * AC::TILES_PER_A;
    std::vector<double> epart(static_cast<size_t>(count) * ntiles * 2, 0.0);
    ArgsAC g{};
    g.psi = psi; g.kpsi = kpsi; g.w1 = w1.data(); g.desc = desc; g.twc = twc; g.rootsb = rootsb;
    g.epart = epart.data(); g.m_points = m_points; g.na = na; g.chunk_log2 = CHUNK == 4 ? 2 : 1; g.i = i; g.fi = fi; g.count = count;
    std::vector<double2> S(AC::SMEM_ELEMS > B::SMEM_ELEMS ? AC::SMEM_ELEMS : B::SMEM_ELEMS);
    // pass A
    for (int t = 0; t < count; ++t)
        for (int tile = 0; tile < ntiles; ++tile) {
            const int a = tile / AC::TILES_PER_A, b2base = (tile % AC::TILES_PER_A) * G;
            for (int w = 0; w < AC::ITEMS_LINE_Q; ++w) a0_item<AC>(w, S.data(), g, desc[t], a, b2base);
            for (int w = 0; w < AC::ITEMS_LINE_P; ++w) a1_item<AC>(w, S.data());
            for (int w = 0; w < AC::ITEMS_POS; ++w) a2_item<AC>(w, S.data(), g, t, a, b2base);
        }
    // pass B
    ArgsB gb{};
    gb.w1 = w1.data(); gb.twa = twa; gb.ks = ks; gb.tc = TC; gb.pc = Split<TC>::P; gb.qc = Split<TC>::Q;
    gb.npch = TC / CHUNK;
    for (int t = 0; t < count; ++t)
        for (int blk = 0; blk < B::R1 * gb.npch; ++blk) {
            const int q = blk % B::R1, pch = blk / B::R1;
            for (int w = 0; w < B::ITEMS_IO; ++w) b0_item<B>(w, S.data(), gb, t, q, pch);
            for (int w = 0; w < B::ITEMS_Q; ++w) b1_item<B>(w, S.data(), gb);
            for (int w = 0; w < B::ITEMS_P; ++w) b2_item<B>(w, S.data(), gb, q, pch);
            for (int w = 0; w < B::ITEMS_Q; ++w) b3_item<B>(w, S.data());
            for (int w = 0; w < B::ITEMS_IO; ++w) b4_item<B>(w, S.data(), gb, t, q, pch);
        }
    // pass C (v2): W1 tile landed in place in the work buffer (c_land_map = the kernel's cp.async gather), psi_j / psi_l
    // lines staged in an operand buffer that c2 overwrites with the K psi_j / K psi_l increments (the kernel's TMA
    // bulk loads and bulk reduce-adds are plain copies / adds here).
    std::vector<double2> SC(AC::SMEM_C);
    std::vector<double> op(AC::OP_DOUBLES);
    std::vector<double> acc(static_cast<size_t>(AC::ITEMS_LINE_Q) * AC::PCN), vi(acc.size());
    auto line_gmem = [&](int orb, int l, int a, int b2base) {
        const int gi = l / AC::NB1, b1 = l % AC::NB1;
        const int b = AC::R2 * b1 + b2base + gi;
        return static_cast<size_t>(orb) * m_points + (static_cast<size_t>(a) * AC::NB + b) * AC::NC;
    };
    for (int tile = 0; tile < ntiles; ++tile) {
        const int a = tile / AC::TILES_PER_A, b2base = (tile % AC::TILES_PER_A) * G;
        std::fill(acc.begin(), acc.end(), 0.0);
        for (int w = 0; w < AC::ITEMS_LINE_Q; ++w)
            for (int n1 = 0; n1 < AC::PCN; ++n1)
                vi[static_cast<size_t>(w) * AC::PCN + n1] = psi[line_gmem(i, w / AC::QC, a, b2base) + w % AC::QC + AC::QC * n1];
        for (int t = 0; t < count; ++t) {
            for (int e = 0; e < AC::TILE_ELEMS; ++e) {
                size_t src; int dst;
                c_land_map<AC>(e, g, t, a, b2base, &src, &dst);
                SC[dst] = w1[src];
            }
            for (int w = 0; w < AC::ITEMS_POS; ++w) c0_item<AC>(w, SC.data(), g, b2base);
            for (int w = 0; w < AC::ITEMS_LINE_P; ++w) c1_item<AC>(w, SC.data(), g);
            const XformDesc d = desc[t];
            for (int slot = 0; slot < (d.l >= 0 ? 2 : 1); ++slot)
                for (int l = 0; l < AC::LINES; ++l)
                    std::memcpy(&op[(slot * AC::LINES + l) * AC::LS], psi + line_gmem(slot ? d.l : d.j, l, a, b2base), AC::NC * sizeof(double));
            double e1 = 0.0, e2 = 0.0;
            for (int w = 0; w < AC::ITEMS_LINE_Q; ++w) {
                double* oj = &op[(w / AC::QC) * AC::LS + w % AC::QC];
                c2_item<AC>(w, SC.data(), d, fi, &vi[static_cast<size_t>(w) * AC::PCN], oj, oj + AC::LINES * AC::LS,
                            &acc[static_cast<size_t>(w) * AC::PCN], e1, e2);
            }
            e_out[2 * t] += e1;
            e_out[2 * t + 1] += e2;
            for (int slot = 0; slot < 2; ++slot) {
                const int orb = slot ? d.l : d.j;
                if (orb < 0 || orb == i) continue;
                for (int l = 0; l < AC::LINES; ++l)
                    for (int c = 0; c < AC::NC; ++c) kpsi[line_gmem(orb, l, a, b2base) + c] += op[(slot * AC::LINES + l) * AC::LS + c];
            }
        }
        for (int w = 0; w < AC::ITEMS_LINE_Q; ++w)
            c_flush_item<AC>(w, g, a, b2base, acc.data() + static_cast<size_t>(w) * AC::PCN);
    }
    return 0;
}

#define EMU_CASE(TA_, TB_, TC_, FREE_, G_, CH_)                                                              \
    if (ta == TA_ && tb == TB_ && tc == TC_ && free_bc == FREE_ && g == G_ && chunk == CH_)                    \
        return emu_batch<TA_, TB_, TC_, FREE_ != 0, G_, CH_>(psi, kpsi, i, fi, count, desc, twa, twc, rootsb, ks, e_out);

extern "C" int exx_emu_batch(int ta, int tb, int tc, int free_bc, int g, int chunk, const double* psi, double* kpsi,
                             int i, double fi, int count, const int* jl /*[count][2]*/, const double* fjl /*[count][2]*/,
                             const double* twa_, const double* twc_, const double* rootsb_, const double* ks,
                             double* e_out) {
    std::vector<XformDesc> dv(count);
    for (int t = 0; t < count; ++t) { dv[t].j = jl[2 * t]; dv[t].l = jl[2 * t + 1]; dv[t].fj = fjl[2 * t]; dv[t].fl = fjl[2 * t + 1]; }
    const XformDesc* desc = dv.data();
    const double2* twa = reinterpret_cast<const double2*>(twa_);
    const double2* twc = reinterpret_cast<const double2*>(twc_);
    const double2* rootsb = reinterpret_cast<const double2*>(rootsb_);
    for (int t = 0; t < 2 * count; ++t) e_out[t] = 0.0;
    EMU_CASE(16, 16, 16, 0, 1, 4)
    EMU_CASE(16, 16, 16, 0, 2, 2)
    EMU_CASE(16, 16, 16, 1, 2, 4)
    EMU_CASE(32, 32, 32, 0, 4, 4)
    EMU_CASE(32, 32, 32, 1, 1, 2)
    EMU_CASE(16, 32, 64, 0, 2, 4)
    EMU_CASE(64, 16, 32, 1, 4, 4)
    EMU_CASE(96, 96, 96, 0, 2, 4)
    EMU_CASE(16, 96, 16, 1, 3, 2)
    EMU_CASE(16, 16, 128, 0, 1, 4)
    EMU_CASE(128, 16, 16, 1, 1, 4)
    EMU_CASE(16, 192, 16, 0, 1, 4)
    EMU_CASE(192, 16, 16, 0, 1, 4)
    EMU_CASE(16, 16, 192, 1, 1, 4)
    EMU_CASE(16, 256, 16, 1, 1, 2)
    EMU_CASE(256, 16, 16, 0, 1, 2)
    EMU_CASE(16, 16, 256, 1, 1, 2)
    return -1;
}
