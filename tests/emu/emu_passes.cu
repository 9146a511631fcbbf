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
static int emu_batch(bool scratch, const double* psi, double* kpsi, int j, int l, double fj, double fl, int count, const XformDesc* desc,
                     const double2* twa, const double2* twc, const double2* rootsb, const double* ks_sym,
                     double* e_out /*[count][2]*/) {
    using AC = CfgAC<TC, TB, FREE, G, CHUNK>;
    static_assert(CHUNK == 1 || CHUNK == 2 || CHUNK == 4, "chunk");
    using B = CfgB<TA, TB, FREE, CHUNK>;
    const int na = B::NA;
    const long long m_points = static_cast<long long>(na) * AC::NB * AC::NC;
    std::vector<double2> w1(static_cast<size_t>(count) * na * TB * TC);
    const int ntiles = na * AC::TILES_PER_A;
    // tables the plan builds: twb[b2*R1+q] = W_TB^{b2 q};  K^ with the c index in scrambled order
    std::vector<double2> twb(static_cast<size_t>(AC::R1) * AC::R2);
    for (int b2 = 0; b2 < AC::R2; ++b2)
        for (int q = 0; q < AC::R1; ++q) twb[b2 * AC::R1 + q] = rootsb[(b2 * q) % TB];
    const int nah = TA / 2 + 1, nbh = TB / 2 + 1, nch = TC / 2 + 1;
    std::vector<double> ks(static_cast<size_t>(nbh) * TC * nah);      // [sb][p][sa], p = scrambled c position
    for (int sa = 0; sa < nah; ++sa)
        for (int sb = 0; sb < nbh; ++sb)
            for (int p = 0; p < TC; ++p) {
                const int kc = (p / AC::QC) + AC::PC * (p % AC::QC);
                ks[(static_cast<size_t>(sb) * TC + p) * nah + sa] = ks_sym[(static_cast<size_t>(sa) * nbh + sb) * nch + (kc <= TC - kc ? kc : TC - kc)];
            }
    std::vector<double2> twa2(TA);                                     // [n2*PA + k1]: the kernel's second smem copy
    for (int x = 0; x < TA; ++x) twa2[(x % B::QA) * B::PA + x / B::QA] = twa[x];
    ArgsAC g{};
    g.psi = psi; g.kpsi = kpsi; g.w1 = w1.data(); g.desc = desc; g.twc = twc; g.twb = twb.data();
    g.m_points = m_points; g.na = na; g.j = j; g.l = l; g.fj = fj; g.fl = fl; g.count = count;
    const size_t qstride = AC::w1_q(na), tstride = AC::w1_t(na);
    std::vector<double2> S(AC::SMEM_A), SC(AC::SMEM_C), W(B::WORK_ELEMS), L(B::LAND_ELEMS), E(B::E_ELEMS);
    std::vector<double> op(AC::OP_DOUBLES), res(AC::RES_DOUBLES);
    std::vector<double> vj(static_cast<size_t>(AC::ITEMS_LINE_Q) * AC::PCN), vl(vj.size()), accj(vj.size()), accl(vj.size());
    auto stage_lines = [&](int orb, double* dst, int a, int b2base) {       // the kernels' TMA bulk line loads
        for (int ln = 0; ln < AC::LINES; ++ln)
            std::memcpy(dst + ln * AC::LS, psi + static_cast<size_t>(orb) * m_points + line_offset<AC>(ln, a, b2base), AC::NC * sizeof(double));
    };
    const int lsafe = l >= 0 ? l : j;
    // pass A
    for (int tile = 0; tile < ntiles; ++tile) {
        const int a = tile / AC::TILES_PER_A, b2base = (tile % AC::TILES_PER_A) * G;
        for (int w = 0; w < AC::ITEMS_LINE_Q; ++w) {
            const LineQIdx x = lineq_index<AC, false>(w, a, b2base);
            for (int n1 = 0; n1 < AC::PCN; ++n1) {
                vj[static_cast<size_t>(w) * AC::PCN + n1] = psi[static_cast<size_t>(j) * m_points + x.gofs + AC::QC * n1];
                vl[static_cast<size_t>(w) * AC::PCN + n1] = psi[static_cast<size_t>(lsafe) * m_points + x.gofs + AC::QC * n1];
            }
        }
        for (int t = 0; t < count; ++t) {
            const XformDesc d = desc[t];
            stage_lines(d.i, op.data(), a, b2base);
            for (int w = 0; w < AC::ITEMS_LINE_Q; ++w) {
                const LineQIdx x = lineq_index<AC, false>(w, a, b2base);
                a0_compute<AC>(&vj[static_cast<size_t>(w) * AC::PCN], &vl[static_cast<size_t>(w) * AC::PCN], &op[x.op], d.flags, S.data() + x.row, twc + x.n2);
            }
            for (int w = 0; w < AC::ITEMS_LINE_P; ++w) a1_compute<AC>(S.data() + linep_index<AC, false>(w).seg);
            for (int w = 0; w < AC::ITEMS_POS; ++w) {
                const ColIdx x = col_index<AC, false>(w, a, b2base, na);
                a2_compute<AC>(S.data() + x.col, twb.data() + x.b2 * AC::R1, w1.data() + t * tstride + x.w1, qstride);
            }
        }
    }
    // pass B (block order and item -> thread mapping differ from the kernel; the index functions are the same)
    const int npch = TC / CHUNK;
    for (int id = 0; id < count * B::R1 * npch; ++id) {
        const int q = id % B::R1, pch = (id / B::R1) % npch, t = id / (B::R1 * npch);
        double2* blk = w1.data() + ((static_cast<size_t>(t) * B::R1 + q) * npch + pch) * B::BLOCK_ELEMS;
        for (int a = 0; a < B::NA; ++a) std::memcpy(&L[a * B::RSL], blk + a * B::COLS, B::ROW_BYTES);   // TMA bulk row loads
        if (!scratch) {
            for (int w = 0; w < B::ITEMS_IO; ++w) { const IoIdx x = io_index<B>(w); b0_compute<B>(L.data() + x.l, W.data() + x.s); }
            for (int cg = 0; cg < B::NGRP; ++cg) {
                for (int w = 0; w < B::ITEMS_Q; ++w) { const ColAIdx x = colq_index<B>(cg, w); b1_compute<B>(W.data() + x.base, twa + x.k, B::QA); }
                for (int w = 0; w < B::ITEMS_P; ++w) {
                    const ColAIdx x = colp_index<B>(cg, w);
                    const int r = x.col / CHUNK, pin = x.col % CHUNK;
                    const int kb = q + B::R1 * r;
                    const int sb = kb <= TB - kb ? kb : TB - kb;
                    double kv[B::QA];
                    b2_load_k<B>(ks.data() + (static_cast<size_t>(sb) * TC + pch * CHUNK + pin) * B::NSA, x.k, kv);
                    b2_compute<B>(W.data() + x.base, kv, twa2.data() + x.k, B::PA, x.k);
                }
                for (int w = 0; w < B::ITEMS_Q; ++w) b3_compute<B>(W.data() + colq_index<B>(cg, w).base);
            }
            for (int w = 0; w < B::ITEMS_IO; ++w) { const IoIdx x = io_index<B>(w); b4_compute<B>(W.data() + x.s, blk + x.g); }
        } else {
            // the warp-specialised kernels: the block lands straight in the padded layout, B0 in place; with the free-BC
            // expansion scratch the buffer holds NA rows and every column group expands into E
            for (int a = 0; a < B::NA; ++a) std::memcpy(&W[B::row_off(a)], blk + a * B::COLS, B::ROW_BYTES);
            for (int w = 0; w < B::ITEMS_IO; ++w) { const IoIdx x = io_index<B>(w); b0_compute<B>(W.data() + x.s, W.data() + x.s); }
            for (int cg = 0; cg < B::NGRP; ++cg) {
                for (int w = 0; w < B::ITEMS_Q; ++w) { const ColAIdx x = colq_index<B>(cg, w); b1e_compute<B>(W.data() + x.base, E.data() + w, twa + x.k, B::QA); }
                for (int w = 0; w < B::ITEMS_P; ++w) {
                    const ColAIdx x = colp_index<B>(cg, w);
                    const int r = x.col / CHUNK, pin = x.col % CHUNK;
                    const int kb = q + B::R1 * r;
                    const int sb = kb <= TB - kb ? kb : TB - kb;
                    double kv[B::QA];
                    b2_load_k<B>(ks.data() + (static_cast<size_t>(sb) * TC + pch * CHUNK + pin) * B::NSA, x.k, kv);
                    b2e_compute<B>(E.data() + x.k * B::QRSE + w % B::NCW, kv, twa2.data() + x.k, B::PA, x.k);
                }
                for (int w = 0; w < B::ITEMS_Q; ++w) b3e_compute<B>(E.data() + w, W.data() + colq_index<B>(cg, w).base);
            }
            for (int w = 0; w < B::ITEMS_IO; ++w) { const IoIdx x = io_index<B>(w); b4_compute<B>(W.data() + x.s, blk + x.g); }
        }
    }
    // pass C: the W1 columns land in place in the work buffer (the kernel's cp.async gather); psi_j / psi_l lines are
    // resident, the psi_i lines are staged in an operand buffer that C2 overwrites with the K psi_i increment (the
    // kernel's TMA bulk loads and bulk reduce-adds are plain copies / adds here).
    for (int tile = 0; tile < ntiles; ++tile) {
        const int a = tile / AC::TILES_PER_A, b2base = (tile % AC::TILES_PER_A) * G;
        std::fill(accj.begin(), accj.end(), 0.0);
        std::fill(accl.begin(), accl.end(), 0.0);
        stage_lines(j, res.data(), a, b2base);
        stage_lines(lsafe, res.data() + AC::LINES * AC::LS, a, b2base);
        for (int t = 0; t < count; ++t) {
            for (int w = 0; w < AC::ITEMS_POS; ++w) {
                const ColIdx x = col_index<AC, true>(w, a, b2base, na);
                for (int q = 0; q < AC::R1; ++q) SC[x.col + q * AC::ROW] = w1[t * tstride + x.w1 + q * qstride];
            }
            for (int w = 0; w < AC::ITEMS_POS; ++w) {
                const ColIdx x = col_index<AC, true>(w, a, b2base, na);
                c0_compute<AC>(SC.data() + x.col, twb.data() + x.b2 * AC::R1);
            }
            for (int w = 0; w < AC::ITEMS_LINE_P; ++w) {
                const LinePIdx x = linep_index<AC, true>(w);
                c1_compute<AC>(SC.data() + x.seg, twc + x.k1 * AC::QC, 1, x.k1);
            }
            const XformDesc d = desc[t];
            stage_lines(d.i, op.data(), a, b2base);
            double e1 = 0.0, e2 = 0.0;
            for (int w = 0; w < AC::ITEMS_LINE_Q; ++w) {
                const LineQIdx x = lineq_index<AC, true>(w, a, b2base);
                c2_compute<AC>(SC.data() + x.row, d, l, fj, fl, &res[x.op], &res[AC::LINES * AC::LS + x.op], &op[x.op],
                               &accj[static_cast<size_t>(w) * AC::PCN], &accl[static_cast<size_t>(w) * AC::PCN], e1, e2);
            }
            e_out[2 * t] += e1;
            e_out[2 * t + 1] += e2;
            if (d.flags != 0 && d.i != j && d.i != l)
                for (int ln = 0; ln < AC::LINES; ++ln)
                    for (int c = 0; c < AC::NC; ++c)
                        kpsi[static_cast<size_t>(d.i) * m_points + line_offset<AC>(ln, a, b2base) + c] += op[ln * AC::LS + c];
        }
        for (int w = 0; w < AC::ITEMS_LINE_Q; ++w) {
            const LineQIdx x = lineq_index<AC, true>(w, a, b2base);
            for (int n1 = 0; n1 < AC::PCN; ++n1) {
                kpsi[static_cast<size_t>(j) * m_points + x.gofs + AC::QC * n1] -= accj[static_cast<size_t>(w) * AC::PCN + n1];
                if (l >= 0) kpsi[static_cast<size_t>(l) * m_points + x.gofs + AC::QC * n1] -= accl[static_cast<size_t>(w) * AC::PCN + n1];
            }
        }
    }
    return 0;
}

#define EMU_CASE(TA_, TB_, TC_, FREE_, G_, CH_)                                                              \
    if (ta == TA_ && tb == TB_ && tc == TC_ && free_bc == FREE_ && g == G_ && chunk == CH_)                    \
        return emu_batch<TA_, TB_, TC_, FREE_ != 0, G_, CH_>(variant != 0, psi, kpsi, j, l, fj, fl, count, desc, twa, twc, rootsb, ks, e_out);

// variant 0: pass B with landing + work buffer (pass_b_kernel); 1: in-place landing with the expansion scratch
// (pass_b_ws_kernel<SCRATCH>; for periodic grids the scratch path is still a valid evaluation order)
extern "C" int exx_emu_batch(int variant, int ta, int tb, int tc, int free_bc, int g, int chunk, const double* psi, double* kpsi,
                             int j, int l, double fj, double fl, int count, const int* iflags /*[count][2]*/,
                             const double* fis /*[count]*/, const double* twa_, const double* twc_, const double* rootsb_,
                             const double* ks, double* e_out) {
    std::vector<XformDesc> dv(count);
    for (int t = 0; t < count; ++t) { dv[t].i = iflags[2 * t]; dv[t].flags = iflags[2 * t + 1]; dv[t].fi = fis[t]; }
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
    EMU_CASE(48, 48, 48, 0, 3, 4)
    EMU_CASE(48, 16, 16, 1, 1, 4)
    EMU_CASE(16, 48, 16, 1, 2, 2)
    EMU_CASE(16, 16, 48, 0, 1, 4)
    EMU_CASE(144, 16, 16, 0, 1, 4)
    EMU_CASE(16, 144, 16, 1, 3, 2)
    EMU_CASE(16, 16, 144, 1, 1, 4)
    EMU_CASE(24, 24, 24, 0, 2, 4)
    EMU_CASE(24, 24, 24, 1, 3, 2)
    EMU_CASE(72, 72, 72, 1, 2, 4)
    EMU_CASE(72, 72, 72, 0, 1, 2)
    return -1;
}
