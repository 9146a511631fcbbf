// exx_passes.cuh -- the three fused pass kernels of the exact-exchange hot path (sm_100a, fp64).
//
// One packed complex transform carries two real co-densities (Eq. 8):
//     z(r) = psi_i(r) psi_j(r) + i psi_i(r) psi_l(r)
// and is convolved with the Green's function (PAPER.md:73-75 Eq. 4, :125-127) by a 3-D FFT that crosses HBM
// only twice per direction ("4-step" split of the middle axis b):
//
//   pass A  (PAPER "Kernel 1" fused into the first FFT pass): co-density + zero padding, full FFT along c
//           (contiguous axis), first stage (R1-point) of the FFT along b, twiddle  ->  workspace W1
//   pass B  ("Kernel 2" core): second stage (R2-point) along b, full FFT along a, multiply by the Fourier-space
//           kernel K^, inverse FFT along a, inverse R2 stage                     ->  W1 (in place)
//   pass C  (inverse + "Kernel 3"): inverse R1 stage along b, inverse FFT along c, then
//           K psi_i += -(f_j V_ij psi_j + f_l V_il psi_l), K psi_j += -f_i V_ij psi_i, K psi_l += -f_i V_il psi_i,
//           and block-reduced partial sums of rho_ij V_ij (PAPER.md:67-69 Eq. 3, :81-82 Eq. 5).
//           One CTA owns a grid tile for ALL transforms of a same-i batch, so K psi_i accumulates in registers.
//
// 1-D FFT of length T = P*Q inside a tile (in place in shared memory, output in digit-scrambled order):
//     n = Q n1 + n2,  k = k1 + P k2,   position p = k1*Q + k2 holds X[k]
//     stage 1: P-point DFT over n1 in registers, twiddle W_T^{n2 k1};  stage 2: Q-point DFT over n2.
// The inverse runs the stages backwards, so no reordering pass is ever needed; K^ is indexed through the
// scramble.  Free boundary conditions (Hockney padding to 2n) prune the zero half of every first stage and the
// discarded half of every last stage.
//
// Every phase is written as a per-work-item function usable on host and device: the kernels run the items
// strided over the CTA's threads with __syncthreads() between phases; tests/emu runs the very same item
// functions sequentially on the CPU to validate the index algebra without a GPU.
#pragma once

#include <cuda_runtime.h>

#include "exx_async.cuh"
#include "exx_dft.cuh"

namespace exx {

// ---------------------------------------------------------------------------------------- compile-time splits
template <int T> struct Split;      // line FFT inside a tile: T = P*Q
template <> struct Split<16>  { static constexpr int P = 4,  Q = 4;  };
template <> struct Split<32>  { static constexpr int P = 4,  Q = 8;  };
template <> struct Split<64>  { static constexpr int P = 8,  Q = 8;  };
template <> struct Split<96>  { static constexpr int P = 8,  Q = 12; };
template <> struct Split<128> { static constexpr int P = 8,  Q = 16; };
template <> struct Split<192> { static constexpr int P = 12, Q = 16; };
template <> struct Split<256> { static constexpr int P = 16, Q = 16; };

template <int T> struct BSplit;     // middle axis split across passes: T = R1*R2 (R1 in pass A/C, R2 in pass B)
template <> struct BSplit<16>  { static constexpr int R1 = 4,  R2 = 4;  };
template <> struct BSplit<32>  { static constexpr int R1 = 8,  R2 = 4;  };
template <> struct BSplit<64>  { static constexpr int R1 = 8,  R2 = 8;  };
template <> struct BSplit<96>  { static constexpr int R1 = 8,  R2 = 12; };
template <> struct BSplit<128> { static constexpr int R1 = 16, R2 = 8;  };
template <> struct BSplit<192> { static constexpr int R1 = 16, R2 = 12; };
template <> struct BSplit<256> { static constexpr int R1 = 16, R2 = 16; };

// One packed transform of a same-i batch: pairs (i,j) and (i,l); l < 0 = the imaginary slot is empty.
struct XformDesc {
    int j, l;
    double fj, fl;
};

// Workspace W1 element index: [t][q][pch][a][b2][pin]  (pass B reads/writes contiguous [a][b2][pin] blocks).
template <int R1, int R2>
EXX_HD size_t w1_index(int t, int q, int pch, int a, int b2, int pin, int npch, int na, int chunk) {
    return ((((static_cast<size_t>(t) * R1 + q) * npch + pch) * na + a) * R2 + b2) * chunk + pin;
}

EXX_HD double2 ld_ro(const double2* p) {
#ifdef __CUDA_ARCH__
    return __ldg(p);
#else
    return *p;
#endif
}
EXX_HD double ld_ro(const double* p) {
#ifdef __CUDA_ARCH__
    return __ldg(p);
#else
    return *p;
#endif
}

// (xr + i xi) *= (w.x + i w.y)      /     *= conj(w)
EXX_HD void cmul(double& xr, double& xi, double2 w) {
    double t = xr * w.x - xi * w.y;
    xi = xr * w.y + xi * w.x;
    xr = t;
}
EXX_HD void cmul_conj(double& xr, double& xi, double2 w) {
    double t = xr * w.x + xi * w.y;
    xi = xi * w.x - xr * w.y;
    xr = t;
}

// ---------------------------------------------------------------------------------------- pass A / C geometry
template <int TC_, int TB_, bool FREE_, int G_>
struct CfgAC {
    static constexpr int TC = TC_, TB = TB_, G = G_;
    static constexpr bool FREE = FREE_;
    static constexpr int PC = Split<TC>::P, QC = Split<TC>::Q;
    static constexpr int R1 = BSplit<TB>::R1, R2 = BSplit<TB>::R2;
    static constexpr int NC = FREE ? TC / 2 : TC;          // grid points along c
    static constexpr int NB = FREE ? TB / 2 : TB;          // grid points along b
    static constexpr int NB1 = FREE ? R1 / 2 : R1;         // non-zero lines (b1) per (a,b2) tile
    static constexpr int PCN = FREE ? PC / 2 : PC;         // non-zero n1 per line
    static constexpr int QCP = QC | 1;                     // padded row of the [k1][n2] layout (bank conflicts)
    static constexpr int ROW = PC * QCP;                   // shared-memory elements per line
    static constexpr int LINES = G * NB1;
    static constexpr int SMEM_ELEMS = LINES * ROW;
    static constexpr int TILES_PER_A = R2 / G;             // CTAs per a-plane
    static constexpr int ITEMS_LINE_Q = LINES * QC;        // (line, n2) items: phases A0, C2
    static constexpr int ITEMS_LINE_P = LINES * PC;        // (line, k1) items: phases A1, C1
    static constexpr int ITEMS_POS = G * TC;               // (g, position) items: phases A2, C0
    static_assert(R2 % G == 0, "G must divide R2");
    EXX_HD static int spos(int p) { return (p / QC) * QCP + (p % QC); }
    // ---- pass C (v2): the W1 tile lands in place in the work buffer, which therefore has R1 lines per b2 of the tile
    static constexpr int GPAD = G > 1 ? 4 : 0;             // shifts consecutive b2 groups by 64 B (bank conflicts)
    static constexpr int GSTR_C = R1 * ROW + GPAD;         // elements between the line blocks of consecutive gi
    static constexpr int SMEM_C = G * GSTR_C;              // elements of one pass-C work buffer
    static constexpr int TILE_ELEMS = G * R1 * TC;         // complex values of one W1 tile
    // operand lines (psi_j, psi_l; overwritten with the K psi_j, K psi_l increments) staged in shared memory:
    // line stride LS doubles, LS = QC (mod 16) keeps the (line, n2)-mapped 8-byte accesses conflict-free
    static constexpr int LS = NC + (((QC - NC % 16) % 16) + 16) % 16;
    static constexpr int OP_DOUBLES = 2 * LINES * LS;      // one stage: [slot j|l][line][LS]
    static_assert(LS % 2 == 0 && NC % 2 == 0, "16-byte alignment of operand lines");
    EXX_HD static int line_c(int gi, int q) { return gi * GSTR_C + q * ROW; }
};

struct ArgsAC {
    const double* psi;          // [N][na][nb][nc]
    double* kpsi;               // pass C only
    double2* w1;
    const XformDesc* desc;      // first transform of this batch
    const double2* twc;         // [k1*QC + n2] = W_TC^{n2 k1}
    const double2* rootsb;      // [m] = W_TB^m
    double* epart;              // pass C: [count][ntiles][2] partial sums of rho*V
    long long m_points;         // na*nb*nc
    int na;
    int chunk_log2;             // W1 layout: CHUNK = 1 << chunk_log2 contiguous c-positions per (a,b2)
    int i;                      // common orbital of the batch
    double fi;
    int count;                  // transforms in the batch
};

// ---- A0: co-density (Eq. 8) + zero padding + stage 1 of the c-axis FFT
template <class C>
EXX_HD void a0_item(int w, double2* S, const ArgsAC& g, const XformDesc& d, int a, int b2base) {
    const int l = w / C::QC, n2 = w % C::QC;
    const int gi = l / C::NB1, b1 = l % C::NB1;
    const int b = C::R2 * b1 + b2base + gi;
    const size_t base = (static_cast<size_t>(a) * C::NB + b) * C::NC + n2;
    const double* pi = g.psi + static_cast<size_t>(g.i) * g.m_points + base;
    const double* pj = g.psi + static_cast<size_t>(d.j) * g.m_points + base;
    const double* pl = g.psi + static_cast<size_t>(d.l < 0 ? d.j : d.l) * g.m_points + base;
    const double lmask = d.l < 0 ? 0.0 : 1.0;
    double xr[C::PC], xi[C::PC];
#pragma unroll
    for (int n1 = 0; n1 < C::PCN; ++n1) {
        const double vi = ld_ro(pi + C::QC * n1);
        xr[n1] = vi * ld_ro(pj + C::QC * n1);
        xi[n1] = vi * ld_ro(pl + C::QC * n1) * lmask;
    }
#pragma unroll
    for (int n1 = C::PCN; n1 < C::PC; ++n1) { xr[n1] = 0.0; xi[n1] = 0.0; }
    dft_fwd<C::PC, C::FREE>(xr, xi);
    double2* row = S + l * C::ROW + n2;
#pragma unroll
    for (int k1 = 0; k1 < C::PC; ++k1) {
        if (k1 > 0) cmul(xr[k1], xi[k1], ld_ro(g.twc + k1 * C::QC + n2));
        row[k1 * C::QCP] = make_double2(xr[k1], xi[k1]);
    }
}

// ---- A1: stage 2 of the c-axis FFT (in place; the item reads and writes only its own row segment)
template <class C>
EXX_HD void a1_item(int w, double2* S) {
    const int l = w / C::PC, k1 = w % C::PC;
    double2* seg = S + l * C::ROW + k1 * C::QCP;
    double xr[C::QC], xi[C::QC];
#pragma unroll
    for (int n2 = 0; n2 < C::QC; ++n2) { double2 v = seg[n2]; xr[n2] = v.x; xi[n2] = v.y; }
    Dft<C::QC>::run(xr, xi);
#pragma unroll
    for (int k2 = 0; k2 < C::QC; ++k2) seg[k2] = make_double2(xr[k2], xi[k2]);
}

// ---- A2: stage 1 (R1-point) of the b-axis FFT + twiddle W_TB^{b2 q}, store to W1
template <class C>
EXX_HD void a2_item(int w, const double2* S, const ArgsAC& g, int t, int a, int b2base) {
    const int gi = w / C::TC, p = w % C::TC;
    const int b2 = b2base + gi;
    const double2* col = S + gi * C::NB1 * C::ROW + C::spos(p);
    double xr[C::R1], xi[C::R1];
#pragma unroll
    for (int b1 = 0; b1 < C::NB1; ++b1) { double2 v = col[b1 * C::ROW]; xr[b1] = v.x; xi[b1] = v.y; }
#pragma unroll
    for (int b1 = C::NB1; b1 < C::R1; ++b1) { xr[b1] = 0.0; xi[b1] = 0.0; }
    dft_fwd<C::R1, C::FREE>(xr, xi);
    const int chunk = 1 << g.chunk_log2;
    const int pch = p >> g.chunk_log2, pin = p & (chunk - 1);
    const int npch = C::TC >> g.chunk_log2;
#pragma unroll
    for (int q = 0; q < C::R1; ++q) {
        if (q > 0) cmul(xr[q], xi[q], ld_ro(g.rootsb + (b2 * q) % C::TB));
        g.w1[w1_index<C::R1, C::R2>(t, q, pch, a, b2, pin, npch, g.na, chunk)] = make_double2(xr[q], xi[q]);
    }
}

// ---- C landing: element e of the W1 tile of (t, a, b2base) -> (index in W1, element offset in the work buffer).
//      e enumerates (q, pch, gi, pin) with pin fastest, then gi: consecutive e are consecutive in W1 for G*CHUNK
//      elements (128 B runs for G*CHUNK = 8), so a warp's 16-byte cp.async requests coalesce into full lines.
template <class C>
EXX_HD void c_land_map(int e, const ArgsAC& g, int t, int a, int b2base, size_t* src, int* dst) {
    const int chunk = 1 << g.chunk_log2;
    const int npch = C::TC >> g.chunk_log2;
    const int pin = e & (chunk - 1);
    int r = e >> g.chunk_log2;
    const int gi = r % C::G; r /= C::G;
    const int pch = r % npch;
    const int q = r / npch;
    *src = w1_index<C::R1, C::R2>(t, q, pch, a, b2base + gi, pin, npch, g.na, chunk);
    *dst = C::line_c(gi, q) + C::spos(pch * chunk + pin);
}

// ---- C0: conj twiddle + inverse R1 stage of the b axis, in place in the work buffer (q lines -> b1 lines)
template <class C>
EXX_HD void c0_item(int w, double2* S, const ArgsAC& g, int b2base) {
    const int gi = w / C::TC, p = w % C::TC;
    const int b2 = b2base + gi;
    double2* col = S + C::line_c(gi, 0) + C::spos(p);
    double xr[C::R1], xi[C::R1];
#pragma unroll
    for (int q = 0; q < C::R1; ++q) {
        double2 v = col[q * C::ROW];
        xr[q] = v.x; xi[q] = v.y;
        if (q > 0) cmul_conj(xr[q], xi[q], ld_ro(g.rootsb + (b2 * q) % C::TB));
    }
    dft_inv<C::R1, C::FREE>(xr, xi);
#pragma unroll
    for (int b1 = 0; b1 < C::NB1; ++b1) col[b1 * C::ROW] = make_double2(xr[b1], xi[b1]);
}

// ---- C1: inverse stage over k2 (Q-point) of the c axis + conj twiddle
template <class C>
EXX_HD void c1_item(int w, double2* S, const ArgsAC& g) {
    const int l = w / C::PC, k1 = w % C::PC;
    double2* seg = S + C::line_c(l / C::NB1, l % C::NB1) + k1 * C::QCP;
    double xr[C::QC], xi[C::QC];
#pragma unroll
    for (int k2 = 0; k2 < C::QC; ++k2) { double2 v = seg[k2]; xr[k2] = v.x; xi[k2] = v.y; }
    dft_inv<C::QC, false>(xr, xi);
#pragma unroll
    for (int n2 = 0; n2 < C::QC; ++n2) {
        if (k1 > 0) cmul_conj(xr[n2], xi[n2], ld_ro(g.twc + k1 * C::QC + n2));
        seg[n2] = make_double2(xr[n2], xi[n2]);
    }
}

// ---- C2: inverse stage over k1 (P-point) of the c axis, then "Kernel 3" for the PCN points
//      c = QC n1 + n2 of line l that this item owns:
//      acc   += f_j V_ij psi_j + f_l V_il psi_l                 (K psi_i -= acc after the batch)
//      oj    <- -f_i V_ij psi_i ,  ol <- -f_i V_il psi_i         increments of K psi_j, K psi_l, written over the
//               staged psi_j / psi_l values and added to K psi by the memory system   PAPER.md:67-69 Eq. 3, :111
//      e1    += rho_ij V_ij,  e2 += rho_il V_il                                        PAPER.md:81-82 Eq. 5
//      vi = psi_i at the item's points; oj / ol = operand lines of this item at offset n2 (stride QC between n1).
template <class C>
EXX_HD void c2_item(int w, const double2* S, const XformDesc& d, double fi, const double* vi /*[PCN]*/, double* oj,
                    double* ol, double* acc /*[PCN]*/, double& e1, double& e2) {
    const int l = w / C::QC, n2 = w % C::QC;
    const double2* row = S + C::line_c(l / C::NB1, l % C::NB1) + n2;
    double xr[C::PC], xi[C::PC];
#pragma unroll
    for (int k1 = 0; k1 < C::PC; ++k1) { double2 v = row[k1 * C::QCP]; xr[k1] = v.x; xi[k1] = v.y; }
    dft_inv<C::PC, C::FREE>(xr, xi);
    const bool has_l = d.l >= 0;
    const double fl = has_l ? d.fl : 0.0;
    double s1 = 0.0, s2 = 0.0;
#pragma unroll
    for (int n1 = 0; n1 < C::PCN; ++n1) {
        const int off = C::QC * n1;
        const double v1 = xr[n1], v2 = xi[n1];
        const double vj = oj[off];
        const double vl = has_l ? ol[off] : 0.0;
        acc[n1] += d.fj * v1 * vj + fl * v2 * vl;
        oj[off] = -(fi * v1 * vi[n1]);
        if (has_l) ol[off] = -(fi * v2 * vi[n1]);
        s1 += vi[n1] * vj * v1;
        s2 += vi[n1] * vl * v2;
    }
    e1 += s1;
    e2 += s2;
}

template <class C>
EXX_HD void c_flush_item(int w, const ArgsAC& g, int a, int b2base, const double* acc) {
    const int l = w / C::QC, n2 = w % C::QC;
    const int gi = l / C::NB1, b1 = l % C::NB1;
    const int b = C::R2 * b1 + b2base + gi;
    double* ki = g.kpsi + static_cast<size_t>(g.i) * g.m_points + (static_cast<size_t>(a) * C::NB + b) * C::NC + n2;
#pragma unroll
    for (int n1 = 0; n1 < C::PCN; ++n1) ki[C::QC * n1] -= acc[n1];
}

// ---------------------------------------------------------------------------------------- pass B geometry
template <int TA_, int TB_, bool FREE_, int CHUNK_>
struct CfgB {
    static constexpr int TA = TA_, TB = TB_, CHUNK = CHUNK_;
    static constexpr bool FREE = FREE_;
    static constexpr int PA = Split<TA>::P, QA = Split<TA>::Q;
    static constexpr int R1 = BSplit<TB>::R1, R2 = BSplit<TB>::R2;
    static constexpr int NA = FREE ? TA / 2 : TA;
    static constexpr int PAN = FREE ? PA / 2 : PA;
    static constexpr int COLS = R2 * CHUNK;
    // row stride == CHUNK (mod 8) elements keeps the (a,pin)-mapped phases B0/B4 conflict-free
    static constexpr int RS = COLS + ((CHUNK - COLS % 8) + 8) % 8;
    static constexpr int SMEM_ELEMS = TA * RS;
    static constexpr int ITEMS_IO = NA * CHUNK;            // (a, pin): B0, B4
    static constexpr int ITEMS_Q = COLS * QA;              // (n2, col): B1, B3
    static constexpr int ITEMS_P = COLS * PA;              // (k1, col): B2
};

struct ArgsB {
    double2* w1;
    const double2* twa;         // [k1*QA + n2] = W_TA^{n2 k1}
    const double* ks;           // symmetric Fourier kernel [TA/2+1][TB/2+1][TC/2+1], includes 1/T_tot (and dV)
    int tc, pc, qc;             // c-axis transform length and its split (to unscramble kc)
    int npch;
};

template <class C>
EXX_HD void b0_item(int w, double2* S, const ArgsB& g, int t, int q, int pch) {
    const int a = w / C::CHUNK, pin = w % C::CHUNK;
    double xr[C::R2], xi[C::R2];
    const double2* src = g.w1 + w1_index<C::R1, C::R2>(t, q, pch, a, 0, pin, g.npch, C::NA, C::CHUNK);
#pragma unroll
    for (int b2 = 0; b2 < C::R2; ++b2) { double2 v = src[b2 * C::CHUNK]; xr[b2] = v.x; xi[b2] = v.y; }
    Dft<C::R2>::run(xr, xi);
    double2* dst = S + a * C::RS + pin;
#pragma unroll
    for (int r = 0; r < C::R2; ++r) dst[r * C::CHUNK] = make_double2(xr[r], xi[r]);
}

template <class C>
EXX_HD void b1_item(int w, double2* S, const ArgsB& g) {
    const int col = w % C::COLS, n2 = w / C::COLS;
    double xr[C::PA], xi[C::PA];
#pragma unroll
    for (int n1 = 0; n1 < C::PAN; ++n1) { double2 v = S[(C::QA * n1 + n2) * C::RS + col]; xr[n1] = v.x; xi[n1] = v.y; }
#pragma unroll
    for (int n1 = C::PAN; n1 < C::PA; ++n1) { xr[n1] = 0.0; xi[n1] = 0.0; }
    dft_fwd<C::PA, C::FREE>(xr, xi);
#pragma unroll
    for (int k1 = 0; k1 < C::PA; ++k1) {
        if (k1 > 0) cmul(xr[k1], xi[k1], ld_ro(g.twa + k1 * C::QA + n2));
        S[(k1 * C::QA + n2) * C::RS + col] = make_double2(xr[k1], xi[k1]);
    }
}

// B2: last forward stage along a, multiply by K^ ("convolving the density with the appropriate
// Green's function"), first inverse stage along a.
template <class C>
EXX_HD void b2_item(int w, double2* S, const ArgsB& g, int q, int pch) {
    const int col = w % C::COLS, k1 = w / C::COLS;
    double xr[C::QA], xi[C::QA];
#pragma unroll
    for (int n2 = 0; n2 < C::QA; ++n2) { double2 v = S[(k1 * C::QA + n2) * C::RS + col]; xr[n2] = v.x; xi[n2] = v.y; }
    Dft<C::QA>::run(xr, xi);
    const int r = col / C::CHUNK, pin = col % C::CHUNK;
    const int kb = q + C::R1 * r;
    const int p = pch * C::CHUNK + pin;
    const int kc = (p / g.qc) + g.pc * (p % g.qc);
    const int sb = kb <= C::TB - kb ? kb : C::TB - kb;
    const int sc = kc <= g.tc - kc ? kc : g.tc - kc;
    const int nbh = C::TB / 2 + 1, nch = g.tc / 2 + 1;
#pragma unroll
    for (int k2 = 0; k2 < C::QA; ++k2) {
        const int ka = k1 + C::PA * k2;
        const int sa = ka <= C::TA - ka ? ka : C::TA - ka;
        const double kv = ld_ro(g.ks + (static_cast<size_t>(sa) * nbh + sb) * nch + sc);
        xr[k2] *= kv; xi[k2] *= kv;
    }
    dft_inv<C::QA, false>(xr, xi);
#pragma unroll
    for (int n2 = 0; n2 < C::QA; ++n2) {
        if (k1 > 0) cmul_conj(xr[n2], xi[n2], ld_ro(g.twa + k1 * C::QA + n2));
        S[(k1 * C::QA + n2) * C::RS + col] = make_double2(xr[n2], xi[n2]);
    }
}

template <class C>
EXX_HD void b3_item(int w, double2* S) {
    const int col = w % C::COLS, n2 = w / C::COLS;
    double xr[C::PA], xi[C::PA];
#pragma unroll
    for (int k1 = 0; k1 < C::PA; ++k1) { double2 v = S[(k1 * C::QA + n2) * C::RS + col]; xr[k1] = v.x; xi[k1] = v.y; }
    dft_inv<C::PA, C::FREE>(xr, xi);
#pragma unroll
    for (int n1 = 0; n1 < C::PAN; ++n1) S[(C::QA * n1 + n2) * C::RS + col] = make_double2(xr[n1], xi[n1]);
}

template <class C>
EXX_HD void b4_item(int w, const double2* S, const ArgsB& g, int t, int q, int pch) {
    const int a = w / C::CHUNK, pin = w % C::CHUNK;
    double xr[C::R2], xi[C::R2];
    const double2* src = S + a * C::RS + pin;
#pragma unroll
    for (int r = 0; r < C::R2; ++r) { double2 v = src[r * C::CHUNK]; xr[r] = v.x; xi[r] = v.y; }
    dft_inv<C::R2, false>(xr, xi);
    double2* dst = g.w1 + w1_index<C::R1, C::R2>(t, q, pch, a, 0, pin, g.npch, C::NA, C::CHUNK);
#pragma unroll
    for (int b2 = 0; b2 < C::R2; ++b2) dst[b2 * C::CHUNK] = make_double2(xr[b2], xi[b2]);
}

// ---------------------------------------------------------------------------------------- kernels
#ifdef __CUDACC__

template <class C, int NT>
__global__ void __launch_bounds__(NT) pass_a_kernel(const ArgsAC g) {
    extern __shared__ double2 S[];
    const int tile = blockIdx.x, t = blockIdx.y;
    const int a = tile / C::TILES_PER_A, b2base = (tile % C::TILES_PER_A) * C::G;
    const XformDesc d = g.desc[t];
    for (int w = threadIdx.x; w < C::ITEMS_LINE_Q; w += NT) a0_item<C>(w, S, g, d, a, b2base);
    __syncthreads();
    for (int w = threadIdx.x; w < C::ITEMS_LINE_P; w += NT) a1_item<C>(w, S);
    __syncthreads();
    for (int w = threadIdx.x; w < C::ITEMS_POS; w += NT) a2_item<C>(w, S, g, t, a, b2base);
}

template <class C, int NT>
__global__ void __launch_bounds__(NT) pass_b_kernel(const ArgsB g) {
    extern __shared__ double2 S[];
    const int q = blockIdx.x % C::R1, pch = blockIdx.x / C::R1, t = blockIdx.y;
    for (int w = threadIdx.x; w < C::ITEMS_IO; w += NT) b0_item<C>(w, S, g, t, q, pch);
    __syncthreads();
    for (int w = threadIdx.x; w < C::ITEMS_Q; w += NT) b1_item<C>(w, S, g);
    __syncthreads();
    for (int w = threadIdx.x; w < C::ITEMS_P; w += NT) b2_item<C>(w, S, g, q, pch);
    __syncthreads();
    for (int w = threadIdx.x; w < C::ITEMS_Q; w += NT) b3_item<C>(w, S);
    __syncthreads();
    for (int w = threadIdx.x; w < C::ITEMS_IO; w += NT) b4_item<C>(w, S, g, t, q, pch);
}

// Pass C.  One CTA per (a, b2-group) tile; it loops over the transforms of the same-i batch, keeps the K psi_i
// accumulator and psi_i of its points in registers, and is software-pipelined:
//   * the W1 tile of transform t+1 is gathered into the second work buffer with 16-byte cp.async while t is computed;
//   * psi_j / psi_l lines arrive NSTG transforms ahead by TMA bulk copies (mbarrier completion) into operand stages;
//   * the K psi_j / K psi_l increments overwrite those lines and leave by TMA bulk reduce-add (fp64) -- each K psi
//     address receives exactly one add per launch (the j of a batch are distinct), so the result is deterministic.
// NT >= ITEMS_LINE_Q (one epilogue item per thread).
template <class C, int NT, int NSTG>
__global__ void __launch_bounds__(NT, 1) pass_c_kernel(const ArgsAC g) {
    static_assert(NT >= C::ITEMS_LINE_Q, "pass C needs one thread per epilogue item");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* const S0 = reinterpret_cast<double2*>(smem_raw);
    double* const OP = reinterpret_cast<double*>(S0 + 2 * C::SMEM_C);
    __shared__ uint64_t full[NSTG];
    __shared__ double red[2][NT / 32];
    const int tile = blockIdx.x;
    const int a = tile / C::TILES_PER_A, b2base = (tile % C::TILES_PER_A) * C::G;
    const int tid = threadIdx.x;
    constexpr uint32_t LINE_BYTES = C::NC * sizeof(double);

    if (tid == 0) {
        for (int s = 0; s < NSTG; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // operand traffic of transform t (warp 0): loads of psi_j / psi_l lines, later reduce-adds of the increments
    auto line_gmem = [&](int orb, int l) -> size_t {
        const int gi = l / C::NB1, b1 = l % C::NB1;
        const int b = C::R2 * b1 + b2base + gi;
        return static_cast<size_t>(orb) * g.m_points + (static_cast<size_t>(a) * C::NB + b) * C::NC;
    };
    auto issue_operand_loads = [&](int t) {          // called by all lanes of warp 0
        const XformDesc d = g.desc[t];
        const int s = t % NSTG;
        double* stage = OP + static_cast<size_t>(s) * C::OP_DOUBLES;
        const int nops = (d.l >= 0 ? 2 : 1) * C::LINES;
        if (tid == 0) mbar_arrive_expect_tx(&full[s], nops * LINE_BYTES);
        __syncwarp();
        for (int o = tid; o < nops; o += 32) {
            const int slot = o / C::LINES, l = o % C::LINES;
            bulk_g2s(stage + (slot * C::LINES + l) * C::LS, g.psi + line_gmem(slot ? d.l : d.j, l), LINE_BYTES, &full[s]);
        }
    };
    auto issue_w1_gather = [&](int t) {              // all threads
        double2* dstbuf = S0 + (t & 1) * C::SMEM_C;
        for (int e = tid; e < C::TILE_ELEMS; e += NT) {
            size_t src; int dst;
            c_land_map<C>(e, g, t, a, b2base, &src, &dst);
            cp_async16(dstbuf + dst, g.w1 + src);
        }
    };

    issue_w1_gather(0);
    cp_async_commit();
    if (tid < 32)
        for (int t = 0; t < NSTG && t < g.count; ++t) issue_operand_loads(t);

    // this thread's epilogue item: PCN points of one line
    const int my_l = tid / C::QC, my_n2 = tid % C::QC;
    double vi[C::PCN], acc[C::PCN];
#pragma unroll
    for (int n1 = 0; n1 < C::PCN; ++n1) { vi[n1] = 0.0; acc[n1] = 0.0; }
    if (tid < C::ITEMS_LINE_Q) {
        const double* pi = g.psi + line_gmem(g.i, my_l) + my_n2;
#pragma unroll
        for (int n1 = 0; n1 < C::PCN; ++n1) vi[n1] = ld_ro(pi + C::QC * n1);
    }

    for (int t = 0; t < g.count; ++t) {
        double2* S = S0 + (t & 1) * C::SMEM_C;
        const int s = t % NSTG;
        double* stage = OP + static_cast<size_t>(s) * C::OP_DOUBLES;
        const XformDesc d = g.desc[t];
        if (t + 1 < g.count) issue_w1_gather(t + 1);
        cp_async_commit();
        cp_async_wait<1>();                                // this thread's part of tile t has landed
        __syncthreads();
        for (int w = tid; w < C::ITEMS_POS; w += NT) c0_item<C>(w, S, g, b2base);
        __syncthreads();
        for (int w = tid; w < C::ITEMS_LINE_P; w += NT) c1_item<C>(w, S, g);
        __syncthreads();
        mbar_wait(&full[s], (t / NSTG) & 1);               // psi_j / psi_l lines of transform t have landed
        double e1 = 0.0, e2 = 0.0;
        if (tid < C::ITEMS_LINE_Q) {
            double* oj = stage + my_l * C::LS + my_n2;
            c2_item<C>(tid, S, d, g.fi, vi, oj, oj + C::LINES * C::LS, acc, e1, e2);
        }
        fence_proxy_async();                               // increments visible to the TMA reads below
        // block reduction of the energy partials in a fixed order (deterministic)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            e1 += __shfl_xor_sync(0xffffffffu, e1, o);
            e2 += __shfl_xor_sync(0xffffffffu, e2, o);
        }
        if ((tid & 31) == 0) { red[0][tid >> 5] = e1; red[1][tid >> 5] = e2; }
        __syncthreads();                                   // also: S and the operand stage are no longer read
        if (tid == 0) {
            double s1 = 0.0, s2 = 0.0;
#pragma unroll
            for (int k = 0; k < NT / 32; ++k) { s1 += red[0][k]; s2 += red[1][k]; }
            double* ep = g.epart + (static_cast<size_t>(t) * gridDim.x + tile) * 2;
            ep[0] = s1; ep[1] = s2;
        }
        if (tid < 32) {
            // K psi_j += -f_i V_ij psi_i,  K psi_l += -f_i V_il psi_i   (the same V_ij serves both orbitals)
            const bool upd_j = d.j != g.i, upd_l = d.l >= 0 && d.l != g.i;
            for (int o = tid; o < 2 * C::LINES; o += 32) {
                const int slot = o / C::LINES, l = o % C::LINES;
                if (slot ? upd_l : upd_j)
                    bulk_red_add_f64(g.kpsi + line_gmem(slot ? d.l : d.j, l), stage + (slot * C::LINES + l) * C::LS, LINE_BYTES);
            }
            bulk_commit();
            if (t + NSTG < g.count) {
                bulk_wait_read_all();                      // the stage may be overwritten
                __syncwarp();
                issue_operand_loads(t + NSTG);
            }
        }
    }
    if (tid < C::ITEMS_LINE_Q) c_flush_item<C>(tid, g, a, b2base, acc);
    if (tid < 32) bulk_wait_read_all();                    // shared memory must outlive the TMA reads
}

#endif  // __CUDACC__

}  // namespace exx
