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
//
// 1-D FFT of length T = P*Q inside a tile (in place in shared memory, output in digit-scrambled order):
//     n = Q n1 + n2,  k = k1 + P k2,   position p = k1*Q + k2 holds X[k]
//     stage 1: P-point DFT over n1 in registers, twiddle W_T^{n2 k1};  stage 2: Q-point DFT over n2.
// The inverse runs the stages backwards, so no reordering pass is ever needed; K^ is indexed through the
// scramble.  Free boundary conditions (Hockney padding to 2n) prune the zero half of every first stage and the
// discarded half of every last stage.
//
// Data movement (exx_async.cuh): all three kernels are software-pipelined loops.  Passes A and C: one CTA owns a
// grid tile for ALL transforms of a same-i batch (psi_i and the K psi_i accumulator of its points stay in
// registers); psi_j / psi_l lines arrive by TMA bulk copies into shared-memory stages one or two transforms
// ahead; pass C gathers the W1 tile of the next transform with cp.async while it computes the current one and
// sends the K psi_j / K psi_l increments out as TMA bulk reduce-adds.  Pass B: persistent CTAs; the next
// [a][b2][pin] block lands by TMA bulk row copies while the current one is transformed.
//
// Every phase is split into an *_index function (thread -> shared/global offsets; evaluated ONCE per thread,
// outside the loops) and a *_compute function (pure arithmetic on those offsets).  Both are __host__ __device__:
// tests/emu runs the very same functions sequentially on the CPU to validate the index algebra without a GPU.
#pragma once

#include <cuda_runtime.h>

#include "exx_async.cuh"
#include "exx_dft.cuh"

namespace exx {

// ---------------------------------------------------------------------------------------- compile-time splits
// Transform lengths T = 2^a 3^b the FFT covers (reading A9).  "Main" lengths may be mixed freely over the
// three axes; the "extra" ones are compiled for cubic transform grids only.
//   line FFT inside a tile:  T = P * Q   (stage 1: P-point in registers, stage 2: Q-point)
//   middle axis across passes: T = R1 * R2 (R1-point stage in passes A / C, R2-point stage in pass B)
constexpr bool is_main_length(int t) { return t == 16 || t == 32 || t == 48 || t == 64 || t == 96 || t == 128 || t == 144 || t == 192 || t == 256; }
constexpr bool is_extra_length(int t) { return t == 24 || t == 72; }
constexpr bool is_length(int t) { return is_main_length(t) || is_extra_length(t); }
constexpr int split_p(int t) {
    return t == 16 ? 4 : t == 24 ? 2 : t == 32 ? 4 : t == 48 ? 4 : t == 64 ? 8 : t == 72 ? 6 : t == 96 ? 8 : t == 128 ? 8 : t == 144 ? 12 :
           t == 192 ? 12 : t == 256 ? 16 : 0;
}
constexpr int split_q(int t) { return split_p(t) ? t / split_p(t) : 0; }
constexpr int r1_of(int tb) {     // 192 = 12 * 16: 12 lines per A/C tile, two CTAs per SM
    return tb == 16 ? 4 : tb == 24 ? 2 : tb == 32 ? 8 : tb == 48 ? 4 : tb == 64 ? 8 : tb == 72 ? 6 : tb == 96 ? 8 : tb == 128 ? 16 :
           tb == 144 ? 12 : tb == 192 ? 12 : tb == 256 ? 16 : 0;
}
constexpr int r2_of(int tb) { return r1_of(tb) ? tb / r1_of(tb) : 0; }
template <int T> struct Split  { static constexpr int P = split_p(T), Q = split_q(T); static_assert(is_length(T), "unsupported transform length"); };
template <int T> struct BSplit { static constexpr int R1 = r1_of(T), R2 = r2_of(T); static_assert(is_length(T), "unsupported transform length"); };
constexpr int chunk_for(int ta, int tb, bool free_bc);     // defined after the pass-B geometry helpers

// One packed transform of a same-(j,l) batch: the streamed orbital i forms the pairs (j,i) [real part] and (l,i)
// [imaginary part] with the two resident orbitals of the batch.
struct XformDesc {
    int i;
    int flags;                  // bit 0: pair (j,i) present, bit 1: pair (l,i) present
    double fi;
};

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
template <int TC_, int TB_, bool FREE_, int G_, int CHUNK_>
struct CfgAC {
    static constexpr int TC = TC_, TB = TB_, G = G_, CHUNK = CHUNK_;
    static constexpr bool FREE = FREE_;
    static constexpr int PC = Split<TC>::P, QC = Split<TC>::Q;
    static constexpr int R1 = BSplit<TB>::R1, R2 = BSplit<TB>::R2;
    static constexpr int NC = FREE ? TC / 2 : TC;          // grid points along c
    static constexpr int NB = FREE ? TB / 2 : TB;          // grid points along b
    static constexpr int NB1 = FREE ? R1 / 2 : R1;         // non-zero lines (b1) per (a,b2) tile
    static constexpr int PCN = FREE ? PC / 2 : PC;         // non-zero n1 per line
    static constexpr int NPCH = TC / CHUNK;
    static constexpr int QCP = QC | 1;                     // padded row of the [k1][n2] layout (bank conflicts)
    static constexpr int ROW = PC * QCP;                   // shared-memory elements per line
    static constexpr int LINES = G * NB1;                  // real-space lines of the tile
    static constexpr int TILES_PER_A = R2 / G;             // CTAs per a-plane
    static constexpr int ITEMS_LINE_Q = LINES * QC;        // (line, n2) items: phases A0, C2
    static constexpr int ITEMS_LINE_P = LINES * PC;        // (line, k1) items: phases A1, C1
    static constexpr int ITEMS_POS = G * TC;               // (gi, position) columns: phases A2, C0
    static_assert(R2 % G == 0, "G must divide R2");
    static_assert(TC % CHUNK == 0, "CHUNK must divide TC");
    // work buffers: the lines of consecutive gi are GPAD elements (64 B) apart so that the (pin, gi)-ordered
    // column accesses of A2 / C0 / the W1 gather hit disjoint banks
    static constexpr int GPAD = G > 1 ? 4 : 0;
    static constexpr int GSTR_A = NB1 * ROW + GPAD;        // pass A: NB1 lines per gi
    static constexpr int SMEM_A = G * GSTR_A;
    static constexpr int GSTR_C = R1 * ROW + GPAD;         // pass C: the W1 tile lands in place, R1 lines per gi
    static constexpr int SMEM_C = G * GSTR_C;
    // operand lines (the streamed psi_i; pass C overwrites them with the K psi_i increment) staged in shared memory:
    // line stride LS doubles, LS = QC (mod 16) keeps the (line, n2)-mapped 8-byte accesses conflict-free
    static constexpr int LS = NC + (((QC - NC % 16) % 16) + 16) % 16;
    static constexpr int OP_DOUBLES = LINES * LS;          // one stage: [line][LS]
    static constexpr int RES_DOUBLES = 2 * LINES * LS;     // pass C: the resident psi_j, psi_l lines [slot j|l][line][LS]
    static constexpr int LINE_BYTES = NC * 8;
    static_assert(LS % 2 == 0 && NC % 2 == 0, "16-byte alignment of operand lines");
    // W1 strides in elements ([t][q][pch][a][b2][pin], na = grid points along a)
    EXX_HD static size_t w1_a() { return static_cast<size_t>(R2) * CHUNK; }
    EXX_HD static size_t w1_pch(int na) { return static_cast<size_t>(na) * R2 * CHUNK; }
    EXX_HD static size_t w1_q(int na) { return static_cast<size_t>(NPCH) * na * R2 * CHUNK; }
    EXX_HD static size_t w1_t(int na) { return static_cast<size_t>(R1) * NPCH * na * R2 * CHUNK; }
    EXX_HD static int spos(int p) { return (p / QC) * QCP + (p % QC); }
};

struct ArgsAC {
    const double* psi;          // streamed set [N][na][nb][nc]: the orbitals i of the transform descriptors
    const double* psi_r;        // resident set: the orbitals j, l of the batch (== psi for the square apply)
    double* kpsi;               // pass C: K psi of the streamed set (reduce-add target); nullptr: no streamed update
    double* kpsi_r;             // pass C: K psi of the resident set (read-modify-write); nullptr: no resident update
    double2* w1;
    const XformDesc* desc;      // first transform of this batch
    const double2* twc;         // [k1*QC + n2] = W_TC^{n2 k1}
    const double2* twb;         // [b2*R1 + q]  = W_TB^{b2 q}
    double* epart;              // pass C: [count][ntiles][2] partial sums of rho*V
    long long m_points;         // na*nb*nc
    int na;
    int j, l;                   // resident orbitals of the batch (l < 0: none; the imaginary slot is then never present)
    int jd, ld;                 // j, l in the numbering of the STREAMED set (square apply: jd = j, ld = l), or negative
                                // values when the two sets are distinct (rectangular pair block: no diagonal pair exists)
    double fj, fl;
    int count;                  // transforms in the batch
};
// Extra arguments of pass C's TMA-gather variant, a kernel parameter of their own: ArgsAC must not grow -- pass A at 256^3
// free runs twice as long with 128 more bytes of kernel parameters (measured; same SASS up to register names).
struct ArgsCX {
    // CUtensorMap of W1 (5-D: [pin (2 CHUNK doubles)][b2][a][pch][q + R1 t]); opaque bytes here so that this header needs no
    // driver types.  Valid only for the geometries whose pass C uses it (KernelInfo::needs_w1_map).
    alignas(64) unsigned char w1_map[128];
    const double2* twc_rot;     // [n2*NCLS + cls] = W_TC^{n2 (k1 + PC r)}, cls = k1-and-rotation class of a C1 item
                                // (k1 = cls % PC, r = cls & 7, NCLS = lcm(8, PC)); see c1_compute_tg
};

// Offset (doubles) of real-space line l = gi*NB1 + b1 of tile (a, b2base) inside one orbital.
template <class C>
EXX_HD size_t line_offset(int l, int a, int b2base) {
    const int gi = l / C::NB1, b1 = l % C::NB1;
    const int b = C::R2 * b1 + b2base + gi;
    return (static_cast<size_t>(a) * C::NB + b) * C::NC;
}

// ---- (line, n2) items of A0 / C2: work-buffer row offset, operand offset, global offset of the item's first point
struct LineQIdx { int row; int op; int n2; size_t gofs; };
template <class C, bool PASS_C>
EXX_HD LineQIdx lineq_index(int w, int a, int b2base) {
    const int l = w / C::QC, n2 = w % C::QC;
    const int gi = l / C::NB1, b1 = l % C::NB1;
    LineQIdx x;
    x.row = gi * (PASS_C ? C::GSTR_C : C::GSTR_A) + b1 * C::ROW + n2;
    x.op = l * C::LS + n2;
    x.n2 = n2;
    x.gofs = line_offset<C>(l, a, b2base) + n2;
    return x;
}

// ---- (line, k1) items of A1 / C1: offset of the [k1] segment of the line, and k1 (twiddle row)
struct LinePIdx { int seg; int k1; };
template <class C, bool PASS_C>
EXX_HD LinePIdx linep_index(int w) {
    const int l = w / C::PC, k1 = w % C::PC;
    const int gi = l / C::NB1, b1 = l % C::NB1;
    LinePIdx x;
    x.seg = gi * (PASS_C ? C::GSTR_C : C::GSTR_A) + b1 * C::ROW + k1 * C::QCP;
    x.k1 = k1;
    return x;
}

// ---- column items of A2 / C0 / the W1 gather, enumerated (pch, gi, pin) with pin fastest, then gi: consecutive
//      items are consecutive in W1 for G*CHUNK elements (128 B for G*CHUNK = 8), so warp accesses coalesce.
struct ColIdx { int col; int b2; size_t w1; };     // work-buffer column offset, b2, W1 offset at (t = 0, q = 0)
template <class C, bool PASS_C>
EXX_HD ColIdx col_index(int w, int a, int b2base, int na) {
    const int pin = w % C::CHUNK;
    const int gi = (w / C::CHUNK) % C::G;
    const int pch = w / (C::CHUNK * C::G);
    ColIdx x;
    x.col = gi * (PASS_C ? C::GSTR_C : C::GSTR_A) + C::spos(pch * C::CHUNK + pin);
    x.b2 = b2base + gi;
    x.w1 = pch * C::w1_pch(na) + a * C::w1_a() + static_cast<size_t>(x.b2) * C::CHUNK + pin;
    return x;
}

// ---------------------------------------------------------------------------------------- pass A phases
// ---- A0: co-densities (Eq. 8) z = psi_i psi_j + i psi_i psi_l + zero padding + stage 1 of the c-axis FFT.
//      vj / vl = psi_j / psi_l at the item's PCN points (registers); pi = the streamed psi_i at the item's first point,
//      stride QC doubles between the points; row = work-buffer row of the item; tw = twc + n2.
template <class C>
EXX_HD void a0_compute(const double* vj, const double* vl, const double* pi, int flags, double2* row, const double2* tw) {
    double xr[C::PC], xi[C::PC];
#pragma unroll
    for (int n1 = 0; n1 < C::PCN; ++n1) {
        const double p = pi[C::QC * n1];
        xr[n1] = vj[n1] * p;
        xi[n1] = vl[n1] * p;
    }
    if (flags != 3) {                                          // an absent pair contributes an exactly zero co-density
        const double m1 = (flags & 1) ? 1.0 : 0.0, m2 = (flags & 2) ? 1.0 : 0.0;
#pragma unroll
        for (int n1 = 0; n1 < C::PCN; ++n1) { xr[n1] *= m1; xi[n1] *= m2; }
    }
#pragma unroll
    for (int n1 = C::PCN; n1 < C::PC; ++n1) { xr[n1] = 0.0; xi[n1] = 0.0; }
    dft_fwd<C::PC, C::FREE>(xr, xi);
#pragma unroll
    for (int k1 = 0; k1 < C::PC; ++k1) {
        if (k1 > 0) cmul(xr[k1], xi[k1], tw[k1 * C::QC]);
        row[k1 * C::QCP] = make_double2(xr[k1], xi[k1]);
    }
}

// ---- A1: stage 2 of the c-axis FFT (in place; the item reads and writes only its own row segment)
template <class C>
EXX_HD void a1_compute(double2* seg) {
    double xr[C::QC], xi[C::QC];
#pragma unroll
    for (int n2 = 0; n2 < C::QC; ++n2) { double2 v = seg[n2]; xr[n2] = v.x; xi[n2] = v.y; }
    Dft<C::QC>::run(xr, xi);
#pragma unroll
    for (int k2 = 0; k2 < C::QC; ++k2) seg[k2] = make_double2(xr[k2], xi[k2]);
}

// ---- A2: stage 1 (R1-point) of the b-axis FFT + twiddle W_TB^{b2 q}, store to W1.
//      col = work-buffer column; tw = twb + b2*R1; dst = W1 element (t, q = 0) of the column; qstride = C::w1_q(na)
template <class C>
EXX_HD void a2_compute(const double2* col, const double2* tw, double2* dst, size_t qstride) {
    double xr[C::R1], xi[C::R1];
#pragma unroll
    for (int b1 = 0; b1 < C::NB1; ++b1) { double2 v = col[b1 * C::ROW]; xr[b1] = v.x; xi[b1] = v.y; }
#pragma unroll
    for (int b1 = C::NB1; b1 < C::R1; ++b1) { xr[b1] = 0.0; xi[b1] = 0.0; }
    dft_fwd<C::R1, C::FREE>(xr, xi);
#pragma unroll
    for (int q = 0; q < C::R1; ++q) {
        if (q > 0) cmul(xr[q], xi[q], tw[q]);
        dst[q * qstride] = make_double2(xr[q], xi[q]);
    }
}

// ---------------------------------------------------------------------------------------- pass C phases
// ---- C0: conj twiddle + inverse R1 stage of the b axis, in place in the work buffer (q lines -> b1 lines)
template <class C>
EXX_HD void c0_compute(double2* col, const double2* tw) {
    double xr[C::R1], xi[C::R1];
#pragma unroll
    for (int q = 0; q < C::R1; ++q) {
        double2 v = col[q * C::ROW];
        xr[q] = v.x; xi[q] = v.y;
        if (q > 0) cmul_conj(xr[q], xi[q], tw[q]);
    }
    dft_inv<C::R1, C::FREE>(xr, xi);
#pragma unroll
    for (int b1 = 0; b1 < C::NB1; ++b1) col[b1 * C::ROW] = make_double2(xr[b1], xi[b1]);
}

// ---- C1: inverse stage over k2 (Q-point) of the c axis + conj twiddle W_TC^{-n2 k1} = conj(tw[n2*tws])
template <class C>
EXX_HD void c1_compute(double2* seg, const double2* tw, int tws, int k1) {
    double xr[C::QC], xi[C::QC];
#pragma unroll
    for (int k2 = 0; k2 < C::QC; ++k2) { double2 v = seg[k2]; xr[k2] = v.x; xi[k2] = v.y; }
    dft_inv<C::QC, false>(xr, xi);
#pragma unroll
    for (int n2 = 0; n2 < C::QC; ++n2) {
        if (k1 > 0) cmul_conj(xr[n2], xi[n2], tw[n2 * tws]);
        seg[n2] = make_double2(xr[n2], xi[n2]);
    }
}

// ---- C2: inverse stage over k1 (P-point) of the c axis, then "Kernel 3" for the PCN points
//      c = QC n1 + n2 of the line that this item owns, with V1 = V_ji = Re, V2 = V_li = Im:
//      accj  += f_i V1 psi_i ,  accl += f_i V2 psi_i            (K psi_j -= accj, K psi_l -= accl after the batch)
//      oi    <- -(f_j V1 psi_j + f_l V2 psi_l)                   increment of K psi_i, written over the staged psi_i
//               values and added to K psi_i by the memory system          PAPER.md:67-69 Eq. 3, :111
//      e1    += rho_ji V1,  e2 += rho_li V2                                         PAPER.md:81-82 Eq. 5
//      i == j (diagonal pair (j,j), imaginary slot absent) and i == l (pairs (j,l) and (l,l)) produce no increment
//      of K psi_i: the cross term f_j V_jl psi_j of K psi_l goes into accl instead, so every K psi address receives
//      exactly one reduce-add per launch.
//      rj / rl = resident psi_j / psi_l lines, oi = operand line, all at the item's first point (stride QC doubles).
//      The phase comes in two halves so that a single-buffered kernel can release the work buffer early: c2_load reads the
//      item's PC inputs into registers (after it, nothing of transform t is left in the buffer that this item needs),
//      c2_finish does the arithmetic.
template <class C>
EXX_HD void c2_load(const double2* row, double* xr /*[PC]*/, double* xi /*[PC]*/) {
#pragma unroll
    for (int k1 = 0; k1 < C::PC; ++k1) { double2 v = row[k1 * C::QCP]; xr[k1] = v.x; xi[k1] = v.y; }
}
template <class C>
EXX_HD void c2_finish(double* xr, double* xi, const XformDesc& d, int l, double fj, double fl, const double* rj, const double* rl,
                      double* oi, double* accj /*[PCN]*/, double* accl /*[PCN]*/, double& e1, double& e2) {
    dft_inv<C::PC, C::FREE>(xr, xi);
    const double m1 = (d.flags & 1) ? 1.0 : 0.0, m2 = (d.flags & 2) ? 1.0 : 0.0;
    const double fjl = d.i == l ? fj : 0.0;
    double s1 = 0.0, s2 = 0.0;
#pragma unroll
    for (int n1 = 0; n1 < C::PCN; ++n1) {
        const int off = C::QC * n1;
        const double v1 = xr[n1] * m1, v2 = xi[n1] * m2;
        const double pi = oi[off], pj = rj[off], pl = rl[off];
        const double a1 = v1 * pi, a2 = v2 * pi;              // V_ji psi_i, V_li psi_i
        const double b1 = v1 * pj, b2 = v2 * pl;              // V_ji psi_j, V_li psi_l
        accj[n1] += d.fi * a1;
        accl[n1] += d.fi * a2 + fjl * b1;
        oi[off] = -(fj * b1 + fl * b2);
        s1 += a1 * pj;
        s2 += a2 * pl;
    }
    e1 += s1;
    e2 += s2;
}
template <class C>
EXX_HD void c2_compute(const double2* row, const XformDesc& d, int l, double fj, double fl, const double* rj, const double* rl,
                       double* oi, double* accj /*[PCN]*/, double* accl /*[PCN]*/, double& e1, double& e2) {
    double xr[C::PC], xi[C::PC];
    c2_load<C>(row, xr, xi);
    c2_finish<C>(xr, xi, d, l, fj, fl, rj, rl, oi, accj, accl, e1, e2);
}

// ---- pass C with the TMA tile gather (TG).  ONE 5-D tensor-box copy brings the whole W1 tile of a transform; it lands
//      dense and unpadded, rows q of TC elements (a tensor box cannot carry the bank-conflict padding of the layout above, and
//      the hardware swizzles need a 128-byte contiguous inner dimension, which a 32-byte W1 run is not).  C0 and C2 run their
//      lanes along a row and stay conflict-free; the lanes of C1 own one k1 segment each, 128 or 256 bytes apart, so lane
//      item w reads and writes its segment ROTATED by r = w & 7 elements: at every step the 8 lanes of a quarter warp then
//      touch 8 different bank groups.  An inverse DFT of the rotated input Y[j] = X[(j + r) mod QC] is the wanted output times
//      a phase, x[n] = w_QC^{n r} IDFT(Y)[n], which together with the stage twiddle conj(W_TC^{n k1}) is conj(W_TC^{n (k1 + PC r)}):
//      one table entry (ArgsCX::twc_rot, [n2][class], class = w mod lcm(8, PC)), so the rotation costs no arithmetic.  C1
//      stores output n2 at position (n2 + r) mod QC of its segment, where C2 picks it up.
//      Why: a cp.async gather writes shared memory sector by sector -- 17 to 24 wavefronts per warp instruction instead of
//      4 -- and was the largest consumer of the shared-memory pipe in pass C.
__host__ __device__ constexpr int tg_classes(int pc) { return pc % 8 == 0 ? pc : pc % 4 == 0 ? 2 * pc : pc % 2 == 0 ? 4 * pc : 8 * pc; }   // lcm(8, pc)
template <class C>
EXX_HD void c0_compute_tg(double2* col /* S + w */, const double2* tw) {
    double xr[C::R1], xi[C::R1];
#pragma unroll
    for (int q = 0; q < C::R1; ++q) {
        double2 v = col[q * C::TC];
        xr[q] = v.x; xi[q] = v.y;
        if (q > 0) cmul_conj(xr[q], xi[q], tw[q]);
    }
    dft_inv<C::R1, C::FREE>(xr, xi);
#pragma unroll
    for (int b1 = 0; b1 < C::NB1; ++b1) col[b1 * C::TC] = make_double2(xr[b1], xi[b1]);
}
// seg = S + line*TC + k1*QC; r = item & 7; tw = twc_rot + class, stride tws = number of classes
template <class C>
EXX_HD void c1_compute_tg(double2* seg, int r, const double2* tw, int tws) {
    static_assert(C::QC == 8 || C::QC == 16, "the rotation needs a power-of-two segment of at least 8 elements");
    double xr[C::QC], xi[C::QC];
#pragma unroll
    for (int j = 0; j < C::QC; ++j) { double2 v = seg[(j + r) & (C::QC - 1)]; xr[j] = v.x; xi[j] = v.y; }
    dft_inv<C::QC, false>(xr, xi);
#pragma unroll
    for (int n2 = 0; n2 < C::QC; ++n2) {
        cmul_conj(xr[n2], xi[n2], tw[n2 * tws]);
        seg[(n2 + r) & (C::QC - 1)] = make_double2(xr[n2], xi[n2]);
    }
}
// row = S + line*TC; the element n2 of segment k1 of line `line` sits at position (n2 + ((line*PC + k1) & 7)) mod QC
template <class C>
EXX_HD void c2_load_tg(const double2* row, int line, int n2, double* xr /*[PC]*/, double* xi /*[PC]*/) {
#pragma unroll
    for (int k1 = 0; k1 < C::PC; ++k1) {
        double2 v = row[k1 * C::QC + ((n2 + ((line * C::PC + k1) & 7)) & (C::QC - 1))];
        xr[k1] = v.x; xi[k1] = v.y;
    }
}

// ---- pass A with the TMA tile store (TS), the mirror of the gather above: the (R1 x TC) output tile of a transform leaves by
//      ONE tensor-box store out of a dense shared-memory tile, rows of TC elements, instead of R1 scattered 16-byte stores
//      per column (32-byte runs in W1: one LSU wavefront per sector, 16 per warp instruction; the LSU data pipe of pass A stood
//      at 87 % at 192^3).  The work buffer is that dense tile; A0 stores, and A1 works on, every k1 segment ROTATED by
//      r = (line*PC + k1) & 7 elements (element n2 / k2 of the segment sits at position (index + r) mod QC), which keeps the
//      segment-per-lane accesses of A1 conflict-free without padding; A2 reads through the rotation and writes its R1 outputs
//      in place at the natural position.  Pure address arithmetic: no phase enters (unlike C1, where the rotation is applied to
//      the transform's input order).
template <class C>
EXX_HD int ts_pos(int line, int k1, int i) { return k1 * C::QC + ((i + ((line * C::PC + k1) & 7)) & (C::QC - 1)); }
template <class C>
EXX_HD void a0_compute_ts(const double* vj, const double* vl, const double* pi, int flags, double2* row /* S + line*TC */, int line, int n2,
                          const double2* tw /* twc + n2 */) {
    double xr[C::PC], xi[C::PC];
#pragma unroll
    for (int n1 = 0; n1 < C::PCN; ++n1) {
        const double p = pi[C::QC * n1];
        xr[n1] = vj[n1] * p;
        xi[n1] = vl[n1] * p;
    }
    if (flags != 3) {
        const double m1 = (flags & 1) ? 1.0 : 0.0, m2 = (flags & 2) ? 1.0 : 0.0;
#pragma unroll
        for (int n1 = 0; n1 < C::PCN; ++n1) { xr[n1] *= m1; xi[n1] *= m2; }
    }
#pragma unroll
    for (int n1 = C::PCN; n1 < C::PC; ++n1) { xr[n1] = 0.0; xi[n1] = 0.0; }
    dft_fwd<C::PC, C::FREE>(xr, xi);
#pragma unroll
    for (int k1 = 0; k1 < C::PC; ++k1) {
        if (k1 > 0) cmul(xr[k1], xi[k1], tw[k1 * C::QC]);
        row[ts_pos<C>(line, k1, n2)] = make_double2(xr[k1], xi[k1]);
    }
}
template <class C>
EXX_HD void a1_compute_ts(double2* seg /* S + line*TC + k1*QC */, int r) {
    double xr[C::QC], xi[C::QC];
#pragma unroll
    for (int n2 = 0; n2 < C::QC; ++n2) { double2 v = seg[(n2 + r) & (C::QC - 1)]; xr[n2] = v.x; xi[n2] = v.y; }
    Dft<C::QC>::run(xr, xi);
#pragma unroll
    for (int k2 = 0; k2 < C::QC; ++k2) seg[(k2 + r) & (C::QC - 1)] = make_double2(xr[k2], xi[k2]);
}
// column p = k1*QC + k2 of the tile: loads (through the rotation), transform, then -- after the caller's __syncwarp, since
// another lane of the warp may still have to read the element this one overwrites -- a2_store_ts
template <class C>
EXX_HD void a2_load_ts(const double2* S, int k1, int k2, double* xr /*[R1]*/, double* xi /*[R1]*/) {
#pragma unroll
    for (int b1 = 0; b1 < C::NB1; ++b1) { double2 v = S[b1 * C::TC + ts_pos<C>(b1, k1, k2)]; xr[b1] = v.x; xi[b1] = v.y; }
#pragma unroll
    for (int b1 = C::NB1; b1 < C::R1; ++b1) { xr[b1] = 0.0; xi[b1] = 0.0; }
}
template <class C>
EXX_HD void a2_store_ts(double* xr, double* xi, const double2* tw /* twb + b2*R1 */, double2* col /* S + p */) {
    dft_fwd<C::R1, C::FREE>(xr, xi);
#pragma unroll
    for (int q = 0; q < C::R1; ++q) {
        if (q > 0) cmul(xr[q], xi[q], tw[q]);
        col[q * C::TC] = make_double2(xr[q], xi[q]);
    }
}

// ---------------------------------------------------------------------------------------- pass B geometry
// Shared-memory bank model for 16-byte accesses: a warp request is served quarter-warp by quarter-warp (8 lanes,
// 128 bytes); lanes of a quarter that hit the same 16-byte bank group (offset mod 8) at different addresses
// serialise.  wavefronts32() counts the wavefronts of one warp-wide access (4 = conflict-free).
constexpr int wavefronts32(const int (&off)[32], int n_active) {
    int total = 0;
    for (int qw = 0; qw < 4; ++qw) {
        int worst = 0;
        for (int bank = 0; bank < 8; ++bank) {
            int cnt = 0;
            for (int l = 0; l < 8; ++l) {
                const int lane = qw * 8 + l;
                if (lane >= n_active || ((off[lane] % 8) + 8) % 8 != bank) continue;
                bool dup = false;
                for (int l2 = 0; l2 < l; ++l2)
                    if (off[qw * 8 + l2] == off[lane]) dup = true;
                if (!dup) ++cnt;
            }
            if (cnt > worst) worst = cnt;
        }
        total += worst;
    }
    return total;
}

// Work-buffer layout of pass B: element (row a, column col) at (a / QA) * QRS + (a % QA) * RS + col, QRS = QA*RS + PADK.
// The three warp access patterns that must be conflict-free:
//   io  (B0/B4): lane -> (a = lane / CHUNK, pin = lane % CHUNK)
//   q   (B1/B3): lane -> (n2 = lane / NCW, cw = lane % NCW), rows QA*n1 + n2   -> offset n2*RS + cw  (+ n1*QRS)
//   p   (B2)   : lane -> (k1 = lane / NCW, cw = lane % NCW), rows k1*QA + n2   -> offset k1*QRS + cw (+ n2*RS)
constexpr int padb_cost(int rs, int padk, int qa, int pa, int ncw, int chunk) {
    const int qrs = qa * rs + padk;
    int o_io[32] = {}, o_q[32] = {}, o_p[32] = {};
    for (int l = 0; l < 32; ++l) {
        const int a = l / chunk;
        o_io[l] = (a / qa) * qrs + (a % qa) * rs + l % chunk;
        o_q[l] = (l / ncw) * rs + l % ncw;
        o_p[l] = (l / ncw) * qrs + l % ncw;
    }
    const int nq = qa * ncw < 32 ? qa * ncw : 32, np = pa * ncw < 32 ? pa * ncw : 32;
    return wavefronts32(o_io, 32) + 2 * wavefronts32(o_q, nq) + 2 * wavefronts32(o_p, np);
}
struct PadB { int rs, padk; };
constexpr PadB pick_padb(int cols, int qa, int pa, int ncw, int chunk) {
    PadB best{cols, 0};
    int best_cost = 1 << 30;
    for (int rs = cols; rs < cols + 8; ++rs)
        for (int padk = 0; padk < 8; ++padk) {
            const int c = padb_cost(rs, padk, qa, pa, ncw, chunk) * 1024 + (rs - cols) * 16 + padk;
            if (c < best_cost) { best_cost = c; best = PadB{rs, padk}; }
        }
    return best;
}
// landing buffer: rows a*RSL, lanes (a, pin)
constexpr int pick_rsl(int cols, int chunk) {
    int best = cols, best_cost = 1 << 30;
    for (int rs = cols; rs < cols + 8; ++rs) {
        int o[32] = {};
        for (int l = 0; l < 32; ++l) o[l] = (l / chunk) * rs + l % chunk;
        const int c = wavefronts32(o, 32) * 1024 + (rs - cols);
        if (c < best_cost) { best_cost = c; best = rs; }
    }
    return best;
}
// columns owned by one warp in the a-axis phases: the divisor of COLS that best fills the 32 lanes in B2 (PA*NCW
// items, the heaviest phase) while leaving at least 8 column groups (warps) where possible; ties -> fewer columns
constexpr int pick_ncw(int pa, int cols) {
    int best = 1, best_score = -1;
    for (int n = 1; n <= cols; ++n) {
        if (cols % n != 0) continue;
        const int items = pa * n, rounds = (items + 31) / 32, ngrp = cols / n;
        const int score = items * 1000 / (32 * rounds) * (ngrp < 8 ? ngrp : 8);
        if (score > best_score) { best_score = score; best = n; }
    }
    return best;
}

// bytes of dynamic shared memory of pass B for a [NA][R2][chunk] block (mirrors CfgB::SMEM_BYTES)
constexpr int smem_b_bytes(int ta, int tb, bool free_bc, int chunk) {
    const int pa = split_p(ta), qa = split_q(ta), cols = r2_of(tb) * chunk;
    const int ncw = pick_ncw(pa, cols);
    const PadB pad = pick_padb(cols, qa, pa, ncw, chunk);
    return (pa * (qa * pad.rs + pad.padk) + (free_bc ? ta / 2 : ta) * pick_rsl(cols, chunk) + 2 * ta) * 16;
}
constexpr int kMaxSmemB = 224 * 1024;
// W1 stores CHUNK consecutive (scrambled) c-positions contiguously: the largest of 4, 2, 1 for which the pass-B work +
// landing buffers of a (TA x R2 x CHUNK)-point block fit shared memory.  It depends on (TA, TB); passes A / C are
// instantiated for every value it can take for their TB (exx_inst.cuh chunk_possible).
constexpr int chunk_for(int ta, int tb, bool free_bc) {
    return smem_b_bytes(ta, tb, free_bc, 4) <= kMaxSmemB ? 4 : smem_b_bytes(ta, tb, free_bc, 2) <= kMaxSmemB ? 2 : 1;
}

// skew between the k1-blocks of the expansion scratch: B2's lanes (k1 = lane / NCW, cw = lane % NCW) must not collide
constexpr int pick_pade(int qa, int pa, int ncw) {
    int best = 0, best_cost = 1 << 30;
    for (int pad = 0; pad < 8; ++pad) {
        int o[32] = {};
        for (int l = 0; l < 32; ++l) o[l] = (l / ncw) * (qa * ncw + pad) + l % ncw;
        const int c = wavefronts32(o, pa * ncw < 32 ? pa * ncw : 32) * 16 + pad;
        if (c < best_cost) { best_cost = c; best = pad; }
    }
    return best;
}

template <int TA_, int TB_, bool FREE_, int CHUNK_>
struct CfgB {
    static constexpr int TA = TA_, TB = TB_, CHUNK = CHUNK_;
    static constexpr bool FREE = FREE_;
    static constexpr int PA = Split<TA>::P, QA = Split<TA>::Q;
    static constexpr int R1 = BSplit<TB>::R1, R2 = BSplit<TB>::R2;
    static constexpr int NA = FREE ? TA / 2 : TA;
    static constexpr int PAN = FREE ? PA / 2 : PA;
    static constexpr int COLS = R2 * CHUNK;
    static constexpr int NCW = pick_ncw(PA, COLS);         // columns per warp (column group)
    static constexpr int NGRP = COLS / NCW;                // column groups
    static constexpr PadB PAD = pick_padb(COLS, QA, PA, NCW, CHUNK);
    static constexpr int RS = PAD.rs;                      // row stride inside a block of QA rows
    static constexpr int QRS = QA * RS + PAD.padk;         // stride between blocks of QA rows
    static constexpr int RSL = pick_rsl(COLS, CHUNK);      // landing-buffer row stride
    static constexpr int WORK_ELEMS = PA * QRS;            // work buffer (all TA rows)
    static constexpr int LAND_ELEMS = NA * RSL;            // landing buffer (the NA rows that exist in W1)
    static constexpr int ROW_BYTES = COLS * 16;            // one [b2][pin] row of W1
    static constexpr int BLOCK_ELEMS = NA * COLS;          // one contiguous [a][b2][pin] block of W1
    static constexpr int ITEMS_IO = NA * CHUNK;            // (a, pin): B0, B4
    static constexpr int ITEMS_Q = QA * NCW;               // (n2, cw) per column group: B1, B3
    static constexpr int ITEMS_P = PA * NCW;               // (k1, cw) per column group: B2
    static constexpr int NSA = TA / 2 + 1;                 // symmetric a-range of K^
    static constexpr int SMEM_BYTES = (WORK_ELEMS + LAND_ELEMS + 2 * TA) * 16;
    EXX_HD static int row_off(int a) { return (a / QA) * QRS + (a % QA) * RS; }
    // warp-private expansion scratch of the free-BC warp-specialised variant: the TA rows of the NCW columns a warp
    // owns, element (row k1*QA + n2, column cw) at k1*QRSE + n2*NCW + cw; the block buffers then hold NA rows only
    static constexpr int QRSE = QA * NCW + pick_pade(QA, PA, NCW);
    static constexpr int E_ELEMS = PA * QRSE;
    static constexpr int P_ELEMS = PAN * QRS;              // block buffer with the NA rows that exist in W1
};

struct ArgsB {
    double2* w1;
    const double2* twa;         // [k1*QA + n2] = W_TA^{n2 k1}
    const double* ks;           // Fourier kernel [TB/2+1][tc][TA/2+1]: symmetric index along b, SCRAMBLED position p
                                // along c (the order pass B meets it), symmetric index along a fastest; includes
                                // 1/T_tot (and dV).  fullk: [TB][tc][TA], every frequency index along a and b
    int fullk;
    int tc;                     // c-axis transform length
    int npch;                   // tc / CHUNK
    int count;                  // transforms in the batch
    int ntiles;                 // count * R1 * npch blocks in this launch
};

// (a, pin) items of B0 / B4: offsets in the landing buffer, the work buffer and the W1 block
struct IoIdx { int l; int s; int g; };
template <class C>
EXX_HD IoIdx io_index(int w) {
    const int a = w / C::CHUNK, pin = w % C::CHUNK;
    IoIdx x;
    x.l = a * C::RSL + pin;
    x.s = C::row_off(a) + pin;
    x.g = a * C::COLS + pin;
    return x;
}
// items of the a-axis phases inside column group cg: B1/B3 item w -> (n2, cw), B2 item w -> (k1, cw)
struct ColAIdx { int base; int k; int col; };
template <class C>
EXX_HD ColAIdx colq_index(int cg, int w) {                // rows QA*n1 + n2, n1 = 0..PA-1 (stride QRS)
    ColAIdx x;
    x.k = w / C::NCW; x.col = cg * C::NCW + w % C::NCW;
    x.base = x.k * C::RS + x.col;
    return x;
}
template <class C>
EXX_HD ColAIdx colp_index(int cg, int w) {                // rows k1*QA + n2, n2 = 0..QA-1 (stride RS)
    ColAIdx x;
    x.k = w / C::NCW; x.col = cg * C::NCW + w % C::NCW;
    x.base = x.k * C::QRS + x.col;
    return x;
}

// ---- B0: second (R2-point) stage of the b-axis FFT: landing buffer -> work buffer (row a, all r, one pin)
template <class C>
EXX_HD void b0_compute(const double2* src, double2* dst) {
    double xr[C::R2], xi[C::R2];
#pragma unroll
    for (int b2 = 0; b2 < C::R2; ++b2) { double2 v = src[b2 * C::CHUNK]; xr[b2] = v.x; xi[b2] = v.y; }
    Dft<C::R2>::run(xr, xi);
#pragma unroll
    for (int r = 0; r < C::R2; ++r) dst[r * C::CHUNK] = make_double2(xr[r], xi[r]);
}

// ---- B1: stage 1 of the a-axis FFT (P-point over n1, zero-padded half pruned) + twiddle W_TA^{n2 k1} = tw[k1*tws]
template <class C>
EXX_HD void b1_compute(double2* colp, const double2* tw, int tws) {
    double xr[C::PA], xi[C::PA];
#pragma unroll
    for (int n1 = 0; n1 < C::PAN; ++n1) { double2 v = colp[n1 * C::QRS]; xr[n1] = v.x; xi[n1] = v.y; }
#pragma unroll
    for (int n1 = C::PAN; n1 < C::PA; ++n1) { xr[n1] = 0.0; xi[n1] = 0.0; }
    dft_fwd<C::PA, C::FREE>(xr, xi);
#pragma unroll
    for (int k1 = 0; k1 < C::PA; ++k1) {
        if (k1 > 0) cmul(xr[k1], xi[k1], tw[k1 * tws]);
        colp[k1 * C::QRS] = make_double2(xr[k1], xi[k1]);
    }
}

// ---- B2: last forward stage along a, multiply by K^ ("convolving the density with the appropriate
//      Green's function"), first inverse stage along a.  kcol = K^ line [sa] of this column (symmetric a index);
//      conj twiddle W_TA^{-n2 k1} = conj(tw[n2*tws]).
// K^ values of one B2 item (frequencies ka = k1 + PA k2, symmetric index): issued well before they are used so that
// the L2 latency hides behind the FFT stages in between
// K^ comes in two layouts (ArgsB::fullk): folded -- symmetric index ranges along a and b, for kernels that are even in
// every index (the analytic and the tabulated ones of an orthorhombic cell, every free-BC kernel) -- and full -- every
// frequency index of a and b, for general periodic cells whose K^(m) = K^(-m) only (exx_plan_create_general).
template <class C>
EXX_HD const double* k_line(const double* ks, int fullk, int kb, int tc, int p) {
    const int sb = fullk ? kb : (kb <= C::TB - kb ? kb : C::TB - kb);
    return ks + (static_cast<size_t>(sb) * tc + p) * (fullk ? C::TA : C::NSA);
}
template <class C>
EXX_HD void b2_load_k(const double* kcol, int k1, double* kv /*[QA]*/, int fullk = 0) {
#pragma unroll
    for (int k2 = 0; k2 < C::QA; ++k2) {
        const int ka = k1 + C::PA * k2;
        kv[k2] = ld_ro(kcol + (fullk || ka <= C::TA - ka ? ka : C::TA - ka));
    }
}
template <class C>
EXX_HD void b2_compute(double2* colp, const double* kv, const double2* tw, int tws, int k1) {
    double xr[C::QA], xi[C::QA];
#pragma unroll
    for (int n2 = 0; n2 < C::QA; ++n2) { double2 v = colp[n2 * C::RS]; xr[n2] = v.x; xi[n2] = v.y; }
    Dft<C::QA>::run(xr, xi);
#pragma unroll
    for (int k2 = 0; k2 < C::QA; ++k2) { xr[k2] *= kv[k2]; xi[k2] *= kv[k2]; }
    dft_inv<C::QA, false>(xr, xi);
#pragma unroll
    for (int n2 = 0; n2 < C::QA; ++n2) {
        if (k1 > 0) cmul_conj(xr[n2], xi[n2], tw[n2 * tws]);
        colp[n2 * C::RS] = make_double2(xr[n2], xi[n2]);
    }
}

// ---- B3: last inverse stage along a (outputs beyond the grid pruned)
template <class C>
EXX_HD void b3_compute(double2* colp) {
    double xr[C::PA], xi[C::PA];
#pragma unroll
    for (int k1 = 0; k1 < C::PA; ++k1) { double2 v = colp[k1 * C::QRS]; xr[k1] = v.x; xi[k1] = v.y; }
    dft_inv<C::PA, C::FREE>(xr, xi);
#pragma unroll
    for (int n1 = 0; n1 < C::PAN; ++n1) colp[n1 * C::QRS] = make_double2(xr[n1], xi[n1]);
}

// ---- B4: inverse R2 stage of the b axis: work buffer -> W1 block
template <class C>
EXX_HD void b4_compute(const double2* src, double2* dst) {
    double xr[C::R2], xi[C::R2];
#pragma unroll
    for (int r = 0; r < C::R2; ++r) { double2 v = src[r * C::CHUNK]; xr[r] = v.x; xi[r] = v.y; }
    dft_inv<C::R2, false>(xr, xi);
#pragma unroll
    for (int b2 = 0; b2 < C::R2; ++b2) dst[b2 * C::CHUNK] = make_double2(xr[b2], xi[b2]);
}

// ---- free-BC variants with the expansion scratch E (warp-private, see CfgB::QRSE): B1 block buffer -> E, B2 in E,
//      B3 E -> block buffer.  in / out point at the item's first element; strides as in the in-place versions.
template <class C>
EXX_HD void b1e_compute(const double2* in, double2* out, const double2* tw, int tws) {
    double xr[C::PA], xi[C::PA];
#pragma unroll
    for (int n1 = 0; n1 < C::PAN; ++n1) { double2 v = in[n1 * C::QRS]; xr[n1] = v.x; xi[n1] = v.y; }
#pragma unroll
    for (int n1 = C::PAN; n1 < C::PA; ++n1) { xr[n1] = 0.0; xi[n1] = 0.0; }
    dft_fwd<C::PA, C::FREE>(xr, xi);
#pragma unroll
    for (int k1 = 0; k1 < C::PA; ++k1) {
        if (k1 > 0) cmul(xr[k1], xi[k1], tw[k1 * tws]);
        out[k1 * C::QRSE] = make_double2(xr[k1], xi[k1]);
    }
}
template <class C>
EXX_HD void b2e_compute(double2* colp, const double* kv, const double2* tw, int tws, int k1) {
    double xr[C::QA], xi[C::QA];
#pragma unroll
    for (int n2 = 0; n2 < C::QA; ++n2) { double2 v = colp[n2 * C::NCW]; xr[n2] = v.x; xi[n2] = v.y; }
    Dft<C::QA>::run(xr, xi);
#pragma unroll
    for (int k2 = 0; k2 < C::QA; ++k2) { xr[k2] *= kv[k2]; xi[k2] *= kv[k2]; }
    dft_inv<C::QA, false>(xr, xi);
#pragma unroll
    for (int n2 = 0; n2 < C::QA; ++n2) {
        if (k1 > 0) cmul_conj(xr[n2], xi[n2], tw[n2 * tws]);
        colp[n2 * C::NCW] = make_double2(xr[n2], xi[n2]);
    }
}
template <class C>
EXX_HD void b3e_compute(const double2* in, double2* out) {
    double xr[C::PA], xi[C::PA];
#pragma unroll
    for (int k1 = 0; k1 < C::PA; ++k1) { double2 v = in[k1 * C::QRSE]; xr[k1] = v.x; xi[k1] = v.y; }
    dft_inv<C::PA, C::FREE>(xr, xi);
#pragma unroll
    for (int n1 = 0; n1 < C::PAN; ++n1) out[n1 * C::QRS] = make_double2(xr[n1], xi[n1]);
}

// ---------------------------------------------------------------------------------------- kernels
#ifdef __CUDACC__

__host__ __device__ constexpr int ceil_div(int a, int b) { return (a + b - 1) / b; }

// TMA bulk loads of the LINES lines of orbital `orb` of tile (a, b2base) into [line][LS] shared memory; the caller has
// armed `bar` with the byte count (all 32 lanes of one warp call this)
template <class C>
__device__ __forceinline__ void issue_line_loads(const ArgsAC& g, const double* set, int orb, double* dst, uint64_t* bar, int a, int b2base,
                                                 int lane) {
    const double* base = set + static_cast<size_t>(orb) * g.m_points;
    for (int l = lane; l < C::LINES; l += 32) bulk_g2s(dst + l * C::LS, base + line_offset<C>(l, a, b2base), C::LINE_BYTES, bar);
}
// the streamed psi_i lines of one transform into an operand stage
template <class C>
__device__ __forceinline__ void issue_operand_loads(const ArgsAC& g, const XformDesc& d, double* stage, uint64_t* bar, int a,
                                                    int b2base, int lane) {
    if (lane == 0) mbar_arrive_expect_tx(bar, C::LINES * C::LINE_BYTES);
    __syncwarp();
    issue_line_loads<C>(g, g.psi, d.i, stage, bar, a, b2base, lane);
}

// Pass A with a single operand stage (the geometries where a second one would cost the second CTA of an SM): the load
// of transform t+1 can only be issued once A0 of t has consumed the stage, so its full DRAM latency would sit on the
// critical path of every iteration.  The lines of transform t+2 are therefore prefetched into L2 at that point (no
// shared-memory destination): the later bulk copy then meets an L2 hit.  Measured at 192^3: pass A -3 %; the same in
// pass C (+6 %) and with two stages (256^3 free: pass A +29 %) is slower -- the prefetches compete with the bulk
// copies and reduce-adds for the TMA unit -- so it stays confined to this case.
#ifndef EXX_PF_MODE
#define EXX_PF_MODE 1            // 0: never, 1: pass A with one operand stage, 2: pass A always
#endif
template <int NSTG>
__host__ __device__ constexpr bool prefetch_operands() { return EXX_PF_MODE == 2 || (EXX_PF_MODE == 1 && NSTG == 1); }
template <class C>
__device__ __forceinline__ void issue_operand_prefetch(const ArgsAC& g, const XformDesc& d, int a, int b2base, int lane) {
    const double* base = g.psi + static_cast<size_t>(d.i) * g.m_points;
    for (int l = lane; l < C::LINES; l += 32) bulk_prefetch_l2(base + line_offset<C>(l, a, b2base), C::LINE_BYTES);
}

// Pass A.  One CTA per (a, b2-group) tile, looping over the transforms of the same-(j,l) batch.  psi_j and psi_l of the
// thread's points live in registers; the streamed psi_i lines arrive NSTG transforms ahead by TMA bulk copies.
template <class C, int NT, int NSTG, int MINB>
__global__ void __launch_bounds__(NT, MINB) pass_a_kernel(const ArgsAC g) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* const S = reinterpret_cast<double2*>(smem_raw);
    double* const OP = reinterpret_cast<double*>(S + C::SMEM_A);
    __shared__ uint64_t full[NSTG];
    __shared__ double2 s_twc[C::TC], s_twb[C::TB];         // twiddle tables (shared-memory reads instead of L1 hits)
    const int tile = blockIdx.x, tid = threadIdx.x;
    const int a = tile / C::TILES_PER_A, b2base = (tile % C::TILES_PER_A) * C::G;
    constexpr int NI0 = ceil_div(C::ITEMS_LINE_Q, NT), NI1 = ceil_div(C::ITEMS_LINE_P, NT), NI2 = ceil_div(C::ITEMS_POS, NT);

    if (tid == 0) {
        for (int s = 0; s < NSTG; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    for (int x = tid; x < C::TC; x += NT) s_twc[x] = g.twc[x];
    for (int x = tid; x < C::TB; x += NT) s_twb[x] = g.twb[x];
    __syncthreads();
    if (tid < 32)
        for (int t = 0; t < NSTG && t < g.count; ++t)
            issue_operand_loads<C>(g, g.desc[t], OP + static_cast<size_t>(t) * C::OP_DOUBLES, &full[t], a, b2base, tid);
    if (prefetch_operands<NSTG>() && tid < 32 && NSTG < g.count) issue_operand_prefetch<C>(g, g.desc[NSTG], a, b2base, tid);

    // per-thread items, resolved once
    LineQIdx q0[NI0];
    double vj[NI0][C::PCN], vl[NI0][C::PCN];
#pragma unroll
    for (int m = 0; m < NI0; ++m) {
        const int w = tid + m * NT;
        q0[m] = lineq_index<C, false>(w < C::ITEMS_LINE_Q ? w : 0, a, b2base);
        const double* pj = g.psi_r + static_cast<size_t>(g.j) * g.m_points + q0[m].gofs;
        const double* pl = g.psi_r + static_cast<size_t>(g.l >= 0 ? g.l : g.j) * g.m_points + q0[m].gofs;
#pragma unroll
        for (int n1 = 0; n1 < C::PCN; ++n1) { vj[m][n1] = ld_ro(pj + C::QC * n1); vl[m][n1] = ld_ro(pl + C::QC * n1); }
    }
    LinePIdx p1[NI1];
#pragma unroll
    for (int m = 0; m < NI1; ++m) p1[m] = linep_index<C, false>(tid + m * NT < C::ITEMS_LINE_P ? tid + m * NT : 0);
    ColIdx c2[NI2];
#pragma unroll
    for (int m = 0; m < NI2; ++m) c2[m] = col_index<C, false>(tid + m * NT < C::ITEMS_POS ? tid + m * NT : 0, a, b2base, g.na);
    const size_t qstride = C::w1_q(g.na), tstride = C::w1_t(g.na);

    int flags_next = g.desc[0].flags;                          // descriptor of the next transform, one iteration ahead
    for (int t = 0; t < g.count; ++t) {
        const int s = t % NSTG;
        double* stage = OP + static_cast<size_t>(s) * C::OP_DOUBLES;
        const int flags = flags_next;
        if (t + 1 < g.count) flags_next = g.desc[t + 1].flags;
        mbar_wait(&full[s], (t / NSTG) & 1);
#pragma unroll
        for (int m = 0; m < NI0; ++m)
            if (tid + m * NT < C::ITEMS_LINE_Q)
                a0_compute<C>(vj[m], vl[m], stage + q0[m].op, flags, S + q0[m].row, s_twc + q0[m].n2);
        __syncthreads();
        if (tid < 32 && t + NSTG < g.count) {                  // the stage has been consumed: refill it
            issue_operand_loads<C>(g, g.desc[t + NSTG], stage, &full[s], a, b2base, tid);
            if (prefetch_operands<NSTG>() && t + NSTG + 1 < g.count) issue_operand_prefetch<C>(g, g.desc[t + NSTG + 1], a, b2base, tid);
        }
#pragma unroll
        for (int m = 0; m < NI1; ++m)
            if (tid + m * NT < C::ITEMS_LINE_P) a1_compute<C>(S + p1[m].seg);
        __syncthreads();
        double2* w1t = g.w1 + static_cast<size_t>(t) * tstride;
#pragma unroll
        for (int m = 0; m < NI2; ++m)
            if (tid + m * NT < C::ITEMS_POS) a2_compute<C>(S + c2[m].col, s_twb + c2[m].b2 * C::R1, w1t + c2[m].w1, qstride);
        __syncthreads();
    }
}


// Pass A, warp-specialised variant (transform lengths >= 96).  NAW "line" warps run the co-density + c-axis FFT phases
// A0, A1 of transform t+1 in one work buffer while NBW "column" warps run the first b-axis stage A2 of transform t out
// of the other buffer and store it to W1, so the global-store-heavy phase overlaps the FP64-heavy ones and the CTA
// needs no CTA-wide barrier: the buffers are handed over with mbarriers (sready: line -> column warps, sfree: back),
// the line warps synchronise among themselves with a named barrier between A0 and A1.
template <class C, int NAW, int NBW, int NSTG, int MINB>
__global__ void __launch_bounds__(32 * (NAW + NBW), MINB) pass_a_ws_kernel(const ArgsAC g) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* const S0 = reinterpret_cast<double2*>(smem_raw);            // two work buffers of SMEM_A
    double* const OP = reinterpret_cast<double*>(S0 + 2 * C::SMEM_A);
    __shared__ uint64_t full[NSTG], sready[2], sfree[2];
    __shared__ double2 s_twc[C::TC], s_twb[C::TB];
    constexpr int NT = 32 * (NAW + NBW), AT = 32 * NAW, BT = 32 * NBW;
    const int tile = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
    const int a = tile / C::TILES_PER_A, b2base = (tile % C::TILES_PER_A) * C::G;

    if (tid == 0) {
        for (int s = 0; s < NSTG; ++s) mbar_init(&full[s], 1);
        for (int b = 0; b < 2; ++b) { mbar_init(&sready[b], NAW); mbar_init(&sfree[b], NBW); }
        mbar_fence_init();
    }
    for (int x = tid; x < C::TC; x += NT) s_twc[x] = g.twc[x];
    for (int x = tid; x < C::TB; x += NT) s_twb[x] = g.twb[x];
    __syncthreads();

    if (tid < AT) {
        // ------------------------------------------------------------------ line warps: A0, A1
        constexpr int NI0 = ceil_div(C::ITEMS_LINE_Q, AT), NI1 = ceil_div(C::ITEMS_LINE_P, AT);
        if (tid < 32)
            for (int t = 0; t < NSTG && t < g.count; ++t)
                issue_operand_loads<C>(g, g.desc[t], OP + static_cast<size_t>(t) * C::OP_DOUBLES, &full[t], a, b2base, tid);
        if (prefetch_operands<NSTG>() && tid < 32 && NSTG < g.count) issue_operand_prefetch<C>(g, g.desc[NSTG], a, b2base, tid);
        LineQIdx q0[NI0];
        double vj[NI0][C::PCN], vl[NI0][C::PCN];
#pragma unroll
        for (int m = 0; m < NI0; ++m) {
            const int w = tid + m * AT;
            q0[m] = lineq_index<C, false>(w < C::ITEMS_LINE_Q ? w : 0, a, b2base);
            const double* pj = g.psi_r + static_cast<size_t>(g.j) * g.m_points + q0[m].gofs;
            const double* pl = g.psi_r + static_cast<size_t>(g.l >= 0 ? g.l : g.j) * g.m_points + q0[m].gofs;
#pragma unroll
            for (int n1 = 0; n1 < C::PCN; ++n1) { vj[m][n1] = ld_ro(pj + C::QC * n1); vl[m][n1] = ld_ro(pl + C::QC * n1); }
        }
        LinePIdx p1[NI1];
#pragma unroll
        for (int m = 0; m < NI1; ++m) p1[m] = linep_index<C, false>(tid + m * AT < C::ITEMS_LINE_P ? tid + m * AT : 0);

        int flags_next = g.desc[0].flags;
        for (int t = 0; t < g.count; ++t) {
            const int s = t % NSTG, b = t & 1;
            double2* const S = S0 + b * C::SMEM_A;
            double* stage = OP + static_cast<size_t>(s) * C::OP_DOUBLES;
            const int flags = flags_next;
            if (t + 1 < g.count) flags_next = g.desc[t + 1].flags;
            if (t >= 2) mbar_wait(&sfree[b], ((t >> 1) - 1) & 1);      // the column warps have drained this buffer
            mbar_wait(&full[s], (t / NSTG) & 1);
#pragma unroll
            for (int m = 0; m < NI0; ++m)
                if (tid + m * AT < C::ITEMS_LINE_Q)
                    a0_compute<C>(vj[m], vl[m], stage + q0[m].op, flags, S + q0[m].row, s_twc + q0[m].n2);
            asm volatile("bar.sync 1, %0;" ::"n"(AT) : "memory");
            if (tid < 32 && t + NSTG < g.count) {                      // the stage has been consumed: refill it
                issue_operand_loads<C>(g, g.desc[t + NSTG], stage, &full[s], a, b2base, tid);
                if (prefetch_operands<NSTG>() && t + NSTG + 1 < g.count) issue_operand_prefetch<C>(g, g.desc[t + NSTG + 1], a, b2base, tid);
            }
#pragma unroll
            for (int m = 0; m < NI1; ++m)
                if (tid + m * AT < C::ITEMS_LINE_P) a1_compute<C>(S + p1[m].seg);
            __syncwarp();
            if (lane == 0) mbar_arrive(&sready[b]);
        }
    } else {
        // ------------------------------------------------------------------ column warps: A2 -> W1
        const int bt = tid - AT;
        constexpr int NI2 = ceil_div(C::ITEMS_POS, BT);
        ColIdx c2[NI2];
#pragma unroll
        for (int m = 0; m < NI2; ++m) c2[m] = col_index<C, false>(bt + m * BT < C::ITEMS_POS ? bt + m * BT : 0, a, b2base, g.na);
        const size_t qstride = C::w1_q(g.na), tstride = C::w1_t(g.na);
        for (int t = 0; t < g.count; ++t) {
            const int b = t & 1;
            double2* const S = S0 + b * C::SMEM_A;
            double2* w1t = g.w1 + static_cast<size_t>(t) * tstride;
            mbar_wait(&sready[b], (t >> 1) & 1);
#pragma unroll
            for (int m = 0; m < NI2; ++m)
                if (bt + m * BT < C::ITEMS_POS) a2_compute<C>(S + c2[m].col, s_twb + c2[m].b2 * C::R1, w1t + c2[m].w1, qstride);
            __syncwarp();
            if (lane == 0) mbar_arrive(&sfree[b]);
        }
    }
}

// Pass A with the TMA tile store (see the *_ts phase functions): the warp-specialised structure of pass_a_ws_kernel with dense
// R1 x TC work buffers.  The column warps run A2 in place, synchronise among themselves, and one thread sends the tile out
// with a tensor-box store; the buffer goes back to the line warps once the store has READ it.
template <class C>
__host__ __device__ constexpr bool pass_a_tma_store() {
#ifdef EXX_NO_TS
    return false;
#else
    return C::G == 1 && C::TC % 64 == 0 && (C::QC == 8 || C::QC == 16) && !C::FREE;
#endif
}
template <class C, int NAW, int NBW, int NSTG, int MINB>
__global__ void __launch_bounds__(32 * (NAW + NBW), MINB) pass_a_ts_kernel(const ArgsAC g, const __grid_constant__ ArgsCX gx) {
    extern __shared__ __align__(128) unsigned char smem_raw_a[];
    constexpr int BUF = C::R1 * C::TC;                                   // one dense work buffer = one W1 tile
    double2* const S0 = reinterpret_cast<double2*>(smem_raw_a);
    double* const OP = reinterpret_cast<double*>(S0 + 2 * BUF);
    __shared__ uint64_t full[NSTG], sready[2], sfree[2];
    __shared__ double2 s_twc[C::TC], s_twb[C::TB];
    constexpr int NT = 32 * (NAW + NBW), AT = 32 * NAW, BT = 32 * NBW;
    const int tile = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
    const int a = tile / C::TILES_PER_A, b2base = (tile % C::TILES_PER_A) * C::G;

    if (tid == 0) {
        for (int s = 0; s < NSTG; ++s) mbar_init(&full[s], 1);
        for (int b = 0; b < 2; ++b) { mbar_init(&sready[b], NAW); mbar_init(&sfree[b], 1); }
        mbar_fence_init();
    }
    for (int x = tid; x < C::TC; x += NT) s_twc[x] = g.twc[x];
    for (int x = tid; x < C::TB; x += NT) s_twb[x] = g.twb[x];
    __syncthreads();

    if (tid < AT) {
        // ------------------------------------------------------------------ line warps: A0, A1
        constexpr int NI0 = ceil_div(C::ITEMS_LINE_Q, AT), NI1 = ceil_div(C::ITEMS_LINE_P, AT);
        if (tid < 32) {
            for (int t = 0; t < NSTG && t < g.count; ++t)
                issue_operand_loads<C>(g, g.desc[t], OP + static_cast<size_t>(t) * C::OP_DOUBLES, &full[t], a, b2base, tid);
            if (prefetch_operands<NSTG>() && NSTG < g.count) issue_operand_prefetch<C>(g, g.desc[NSTG], a, b2base, tid);
        }
        LineQIdx q0[NI0];
        double vj[NI0][C::PCN], vl[NI0][C::PCN];
#pragma unroll
        for (int m = 0; m < NI0; ++m) {
            const int w = tid + m * AT;
            q0[m] = lineq_index<C, false>(w < C::ITEMS_LINE_Q ? w : 0, a, b2base);
            const double* pj = g.psi_r + static_cast<size_t>(g.j) * g.m_points + q0[m].gofs;
            const double* pl = g.psi_r + static_cast<size_t>(g.l >= 0 ? g.l : g.j) * g.m_points + q0[m].gofs;
#pragma unroll
            for (int n1 = 0; n1 < C::PCN; ++n1) { vj[m][n1] = ld_ro(pj + C::QC * n1); vl[m][n1] = ld_ro(pl + C::QC * n1); }
        }
        int flags_next = g.desc[0].flags;
        for (int t = 0; t < g.count; ++t) {
            const int s = t % NSTG, b = t & 1;
            double2* const S = S0 + b * BUF;
            double* stage = OP + static_cast<size_t>(s) * C::OP_DOUBLES;
            const int flags = flags_next;
            if (t + 1 < g.count) flags_next = g.desc[t + 1].flags;
            if (t >= 2) mbar_wait(&sfree[b], ((t >> 1) - 1) & 1);      // the tile store of t-2 has read this buffer
            mbar_wait(&full[s], (t / NSTG) & 1);
#pragma unroll
            for (int m = 0; m < NI0; ++m) {
                const int w = tid + m * AT;
                if (w < C::ITEMS_LINE_Q)
                    a0_compute_ts<C>(vj[m], vl[m], stage + q0[m].op, flags, S + (w / C::QC) * C::TC, w / C::QC, q0[m].n2, s_twc + q0[m].n2);
            }
            asm volatile("bar.sync 1, %0;" ::"n"(AT) : "memory");
            if (tid < 32 && t + NSTG < g.count) {                      // the stage has been consumed: refill it
                issue_operand_loads<C>(g, g.desc[t + NSTG], stage, &full[s], a, b2base, tid);
                if (prefetch_operands<NSTG>() && t + NSTG + 1 < g.count) issue_operand_prefetch<C>(g, g.desc[t + NSTG + 1], a, b2base, tid);
            }
#pragma unroll
            for (int m = 0; m < NI1; ++m) {
                const int w = tid + m * AT;                            // item (line, k1)
                if (w < C::ITEMS_LINE_P) a1_compute_ts<C>(S + (w / C::PC) * C::TC + (w % C::PC) * C::QC, w & 7);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&sready[b]);
        }
    } else {
        // ------------------------------------------------------------------ column warps: A2 in place, tile store
        const int bt = tid - AT;
        constexpr int NI2 = ceil_div(C::ITEMS_POS, BT);
        static_assert(C::ITEMS_POS % 32 == 0, "whole k1 segments per warp");
        for (int t = 0; t < g.count; ++t) {
            const int b = t & 1;
            double2* const S = S0 + b * BUF;
            mbar_wait(&sready[b], (t >> 1) & 1);
#pragma unroll
            for (int m = 0; m < NI2; ++m) {
                const int p = bt + m * BT;                             // warp-uniform condition: BT and ITEMS_POS are multiples of 32
                if (p < C::ITEMS_POS) {
                    double xr[C::R1], xi[C::R1];
                    a2_load_ts<C>(S, p / C::QC, p % C::QC, xr, xi);
                    __syncwarp();                                      // every lane of the warp has read its column
                    a2_store_ts<C>(xr, xi, s_twb + b2base * C::R1, S + p);
                }
            }
            fence_proxy_async();                                       // the tile is read by the TMA below
            asm volatile("bar.sync 2, %0;" ::"n"(BT) : "memory");
            if (bt == 0) {
                tensor5_s2g(gx.w1_map, 0, b2base, a, 0, t * C::R1, S);
                bulk_commit();
                bulk_wait_read_all();
                mbar_arrive(&sfree[b]);
            }
        }
        if (bt == 0) bulk_wait_all();
    }
}

// Pass B.  Persistent CTAs over the (pch, q, t) blocks of the launch, t fastest (CTAs that run at the same time
// share a K^ slice in L2).  The next block lands in a separate buffer by TMA bulk row copies while the current one is
// transformed.  B0 / B4 map a thread to the rows (a, pin) it alone reads and writes, and the a-axis phases B1..B3 map
// a WARP to the NCW columns it alone owns (only __syncwarp between them), so a block costs two CTA barriers:
//     wait(landing) -> B0 -> barrier -> [issue next load] B1 ~ B2 ~ B3 -> barrier -> B4 -> next block.
// The a-axis twiddles live in shared memory in both index orders ([k1*QA+n2] for B1, [n2*PA+k1] for B2).
template <class C, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) pass_b_kernel(const ArgsB g) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* const W = reinterpret_cast<double2*>(smem_raw);
    double2* const L = W + C::WORK_ELEMS;
    double2* const TW1 = L + C::LAND_ELEMS;
    double2* const TW2 = TW1 + C::TA;
    __shared__ uint64_t full;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int NW = NT / 32;
    constexpr int NIO = ceil_div(C::ITEMS_IO, NT), NQ = ceil_div(C::ITEMS_Q, 32), NP = ceil_div(C::ITEMS_P, 32);

    if (tid == 0) { mbar_init(&full, 1); mbar_fence_init(); }
    for (int x = tid; x < C::TA; x += NT) {
        const double2 v = g.twa[x];
        TW1[x] = v;
        TW2[(x % C::QA) * C::PA + x / C::QA] = v;
    }
    __syncthreads();
    auto block_ptr = [&](int id) -> double2* {             // id -> (pch, q, t), t fastest
        const int t = id % g.count, rest = id / g.count;
        const int q = rest % C::R1, pch = rest / C::R1;
        return g.w1 + ((static_cast<size_t>(t) * C::R1 + q) * g.npch + pch) * C::BLOCK_ELEMS;
    };
    auto issue_block_load = [&](int id) {                  // all lanes of warp 0
        const double2* src = block_ptr(id);
        if (tid == 0) mbar_arrive_expect_tx(&full, C::NA * C::ROW_BYTES);
        __syncwarp();
        for (int a = tid; a < C::NA; a += 32) bulk_g2s(L + a * C::RSL, src + a * C::COLS, C::ROW_BYTES, &full);
    };
    if (tid < 32 && static_cast<int>(blockIdx.x) < g.ntiles) issue_block_load(blockIdx.x);

    int it = 0;
    for (int id = blockIdx.x; id < g.ntiles; id += gridDim.x, ++it) {
        const int rest = id / g.count;
        const int q = rest % C::R1, pch = rest / C::R1;
        double2* blk = block_ptr(id);
        mbar_wait(&full, it & 1);
#pragma unroll
        for (int m = 0; m < NIO; ++m)
            if (tid + m * NT < C::ITEMS_IO) {
                const IoIdx x = io_index<C>(tid + m * NT);
                b0_compute<C>(L + x.l, W + x.s);
            }
        __syncthreads();
        if (tid < 32 && id + static_cast<int>(gridDim.x) < g.ntiles) issue_block_load(id + gridDim.x);
        for (int cg = wid; cg < C::NGRP; cg += NW) {
#pragma unroll
            for (int m = 0; m < NQ; ++m)
                if (lane + m * 32 < C::ITEMS_Q) {
                    const ColAIdx x = colq_index<C>(cg, lane + m * 32);
                    b1_compute<C>(W + x.base, TW1 + x.k, C::QA);
                }
            __syncwarp();
#pragma unroll
            for (int m = 0; m < NP; ++m)
                if (lane + m * 32 < C::ITEMS_P) {
                    const ColAIdx x = colp_index<C>(cg, lane + m * 32);
                    const int r = x.col / C::CHUNK, pin = x.col % C::CHUNK;
                    const int kb = q + C::R1 * r;
                    double kv[C::QA];
                    b2_load_k<C>(k_line<C>(g.ks, g.fullk, kb, g.tc, pch * C::CHUNK + pin), x.k, kv, g.fullk);
                    b2_compute<C>(W + x.base, kv, TW2 + x.k, C::PA, x.k);
                }
            __syncwarp();
#pragma unroll
            for (int m = 0; m < NQ; ++m)
                if (lane + m * 32 < C::ITEMS_Q) b3_compute<C>(W + colq_index<C>(cg, lane + m * 32).base);
        }
        __syncthreads();
#pragma unroll
        for (int m = 0; m < NIO; ++m)
            if (tid + m * NT < C::ITEMS_IO) {
                const IoIdx x = io_index<C>(tid + m * NT);
                b4_compute<C>(W + x.s, blk + x.g);
            }
    }
}

// Pass B, warp-specialised variant (used where two work buffers fit shared memory: the periodic geometries).
// NY "column" warps run the a-axis phases B1..B3 of block k while NX "row" warps run the b-axis phases of its
// neighbours -- B0 of block k+1 in place in the OTHER buffer as soon as it has landed, B4 of block k-1 out of that
// buffer before -- so the FP64-heavy and the load/store-heavy halves of the pass overlap inside one CTA.  There is no
// CTA-wide barrier: blocks are handed over with mbarriers
//     full[b]   TMA rows of a block have landed in buf[b] (straight into the padded work layout)   -> row warps
//     ready[b]  B0 done on buf[b]  (row warps arrive)                                                -> column warps
//     done[b]   B1..B3 done on buf[b] (column warps arrive)                                          -> row warps
// and the row warps refill buf[b] with block k+2 once B4 of block k has drained it.
// SCRATCH (free BC, where two TA-row buffers do not fit): the block buffers hold only the NA rows that exist in W1 and
// every column warp expands its NCW columns to TA rows in a private scratch (B1 buffer -> scratch, B2 in the scratch,
// B3 scratch -> buffer).
template <class C, int NY, int NX, int MINB, bool SCRATCH>
__global__ void __launch_bounds__(32 * (NY + NX), MINB) pass_b_ws_kernel(const ArgsB g) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int BUF_ELEMS = SCRATCH ? C::P_ELEMS : C::WORK_ELEMS;
    double2* const BUF = reinterpret_cast<double2*>(smem_raw);           // two block buffers
    double2* const ESC = BUF + 2 * BUF_ELEMS;                            // NY scratch areas (SCRATCH only)
    double2* const TW1 = ESC + (SCRATCH ? NY * C::E_ELEMS : 0);
    double2* const TW2 = TW1 + C::TA;
    __shared__ uint64_t full[2], ready[2], done[2];
    constexpr int NT = 32 * (NY + NX), NXT = 32 * NX;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int NQ = ceil_div(C::ITEMS_Q, 32), NP = ceil_div(C::ITEMS_P, 32), NIO = ceil_div(C::ITEMS_IO, NXT);
    // ROWST: B4 writes its result back into the rows and every row leaves by one TMA bulk store.  A direct B4 store is a
    // scattered 16-byte STG whose warp instruction touches 32 / CHUNK different 32 * CHUNK-byte runs: with CHUNK = 2 that is one
    // LSU wavefront per 32-byte sector, 16 per instruction, where the in-place shared-memory store costs 4 (the LSU data
    // pipe of pass B stood at 82 %).  Measured: pass B -11 % at 256^3 free, -3 % at 192^3; with CHUNK = 4 (64-byte runs, 96^3)
    // the direct stores are cheap enough and the extra shared-memory round trip loses (+12 %).
    constexpr bool ROWST = C::CHUNK <= 2;

    if (tid == 0) {
        for (int b = 0; b < 2; ++b) { mbar_init(&full[b], NX); mbar_init(&ready[b], NX); mbar_init(&done[b], NY); }
        mbar_fence_init();
    }
    for (int x = tid; x < C::TA; x += NT) {
        const double2 v = g.twa[x];
        TW1[x] = v;
        TW2[(x % C::QA) * C::PA + x / C::QA] = v;
    }
    __syncthreads();
    auto block_ptr = [&](int id) -> double2* {             // id -> (pch, q, t), t fastest
        const int t = id % g.count, rest = id / g.count;
        const int q = rest % C::R1, pch = rest / C::R1;
        return g.w1 + ((static_cast<size_t>(t) * C::R1 + q) * g.npch + pch) * C::BLOCK_ELEMS;
    };
    // KREUSE (one column group per column warp, one B2 item per lane): every CTA takes a CONTIGUOUS range of block ids
    // (t fastest), so consecutive blocks of a CTA are the same (q, pch) slice of consecutive transforms and the K^ values
    // a column-warp lane needs stay in its registers for a whole run of blocks (96^3: pass B -7.5 %).  With two column
    // groups per warp the values alternate anyway; there the blocks stay interleaved over the CTAs (CTAs that run at the
    // same time share a K^ slice in L2) and the loads are issued ahead of B1 (measured: contiguous ranges +2..4 %).
    constexpr bool KREUSE = C::NGRP == NY && NP == 1;
    const int per_cta = (g.ntiles + static_cast<int>(gridDim.x) - 1) / static_cast<int>(gridDim.x);
    const int stride = KREUSE ? 1 : static_cast<int>(gridDim.x);
    const int id0 = KREUSE ? static_cast<int>(blockIdx.x) * per_cta : static_cast<int>(blockIdx.x);
    const int nk = id0 >= g.ntiles ? 0 : KREUSE ? (g.ntiles - id0 < per_cta ? g.ntiles - id0 : per_cta) : (g.ntiles - id0 + stride - 1) / stride;

    if (wid >= NY) {
        // ------------------------------------------------------------------ row warps: landing, B0, B4, refill
        // A row warp owns the rows a of its (a, pin) items for the whole kernel: it alone reads and writes them in B0
        // and B4, and it alone refills them, so the row warps never wait for one another.
        const int xt = tid - 32 * NY;
        int my_rows = 0;                                   // rows this warp refills (for the transaction count)
#pragma unroll
        for (int m = 0; m < NIO; ++m) {
            const int first = (xt - lane) + m * NXT;       // first item of this warp in round m
            const int n_items = C::ITEMS_IO - first < 32 ? C::ITEMS_IO - first : 32;
            if (n_items > 0) my_rows += (n_items + C::CHUNK - 1) / C::CHUNK;
        }
        auto issue_row_loads = [&](int k) {                // all lanes of this warp
            const double2* src = block_ptr(id0 + k * stride);
            double2* dst = BUF + (k & 1) * BUF_ELEMS;
            if (lane == 0) mbar_arrive_expect_tx(&full[k & 1], my_rows * C::ROW_BYTES);
            __syncwarp();
#pragma unroll
            for (int m = 0; m < NIO; ++m) {
                const int idx = xt + m * NXT;
                if (idx < C::ITEMS_IO && idx % C::CHUNK == 0) {
                    const int a = idx / C::CHUNK;
                    bulk_g2s(dst + C::row_off(a), src + a * C::COLS, C::ROW_BYTES, &full[k & 1]);
                }
            }
        };
        auto b4_block = [&](int k) {
            double2* const W = BUF + (k & 1) * BUF_ELEMS;
            double2* blk = block_ptr(id0 + k * stride);
            mbar_wait(&done[k & 1], (k >> 1) & 1);
            if constexpr (ROWST) {
                // B4 back into the rows (in place), then one TMA bulk store per row
#pragma unroll
                for (int m = 0; m < NIO; ++m)
                    if (xt + m * NXT < C::ITEMS_IO) {
                        const IoIdx x = io_index<C>(xt + m * NXT);
                        b4_compute<C>(W + x.s, W + x.s);
                    }
                fence_proxy_async();                       // generic-proxy writes of the rows precede the TMA reads
                __syncwarp();
#pragma unroll
                for (int m = 0; m < NIO; ++m) {
                    const int idx = xt + m * NXT;
                    if (idx < C::ITEMS_IO && idx % C::CHUNK == 0) {
                        const int a = idx / C::CHUNK;
                        bulk_s2g(blk + a * C::COLS, W + C::row_off(a), C::ROW_BYTES);
                    }
                }
                bulk_commit();
            } else {
#pragma unroll
                for (int m = 0; m < NIO; ++m)
                    if (xt + m * NXT < C::ITEMS_IO) {
                        const IoIdx x = io_index<C>(xt + m * NXT);
                        b4_compute<C>(W + x.s, blk + x.g);
                    }
            }
        };
        if (nk > 0) issue_row_loads(0);
        if (nk > 1) issue_row_loads(1);
        for (int k = 0; k < nk; ++k) {
            double2* const W = BUF + (k & 1) * BUF_ELEMS;
            mbar_wait(&full[k & 1], (k >> 1) & 1);
#pragma unroll
            for (int m = 0; m < NIO; ++m)
                if (xt + m * NXT < C::ITEMS_IO) {
                    const IoIdx x = io_index<C>(xt + m * NXT);
                    b0_compute<C>(W + x.s, W + x.s);       // in place
                }
            __syncwarp();
            if (lane == 0) mbar_arrive(&ready[k & 1]);
            if (k >= 1) {
                b4_block(k - 1);
                if (k + 1 < nk) {
                    if (ROWST) bulk_wait_read_all();       // the row stores of block k-1 have read their rows
                    fence_proxy_async();                   // this warp's reads of its rows precede the TMA writes
                    __syncwarp();
                    issue_row_loads(k + 1);
                }
            }
        }
        if (nk > 0) b4_block(nk - 1);
        if (ROWST) bulk_wait_all();                        // shared memory must outlive the row stores
    } else {
        // ------------------------------------------------------------------ column warps: a-axis phases
        // K^ of this lane's B2 item (one item per lane, NP = 1) is requested ahead of B1 so that the L2 latency hides
        // behind it.  KREUSE: nothing is requested when the values in the registers are the right ones already (same
        // (q, pch) slice: the usual case inside a contiguous run of blocks), and the first block of a new slice requests
        // its values as soon as B2 of the previous block has consumed the old ones.
        double kv0[C::QA];
        int k_slice = -1, k_cg = -1;                       // (q, pch) slice and column group the values in kv0 belong to
        auto kcol_of = [&](int slice, int cg, int w) {
            const int q = slice % C::R1, pch = slice / C::R1;
            const ColAIdx x = colp_index<C>(cg, w);
            const int r = x.col / C::CHUNK, pin = x.col % C::CHUNK;
            const int kb = q + C::R1 * r;
            return k_line<C>(g.ks, g.fullk, kb, g.tc, pch * C::CHUNK + pin);
        };
        auto request_k = [&](int slice, int cg) {
            if (NP != 1 || (slice == k_slice && cg == k_cg)) return;
            if (lane < C::ITEMS_P) b2_load_k<C>(kcol_of(slice, cg, lane), colp_index<C>(cg, lane).k, kv0, g.fullk);
            k_slice = slice; k_cg = cg;
        };
        if (nk > 0 && wid < C::NGRP) request_k(id0 / g.count, wid);
        for (int k = 0; k < nk; ++k) {
            const int id = id0 + k * stride;
            double2* const W = BUF + (k & 1) * BUF_ELEMS;
            const int slice = id / g.count;
            mbar_wait(&ready[k & 1], (k >> 1) & 1);
            for (int cg = wid; cg < C::NGRP; cg += NY) {
                double2* const E = ESC + wid * C::E_ELEMS;
                request_k(slice, cg);
#pragma unroll
                for (int m = 0; m < NQ; ++m)
                    if (lane + m * 32 < C::ITEMS_Q) {
                        const int w = lane + m * 32;
                        const ColAIdx x = colq_index<C>(cg, w);
                        if (SCRATCH) b1e_compute<C>(W + x.base, E + w, TW1 + x.k, C::QA);     // E offset n2*NCW + cw = w
                        else b1_compute<C>(W + x.base, TW1 + x.k, C::QA);
                    }
                __syncwarp();
#pragma unroll
                for (int m = 0; m < NP; ++m)
                    if (lane + m * 32 < C::ITEMS_P) {
                        const int w = lane + m * 32;
                        const ColAIdx x = colp_index<C>(cg, w);
                        double kvm[C::QA];
                        if (NP != 1) b2_load_k<C>(kcol_of(slice, cg, w), x.k, kvm, g.fullk);
                        const double* kv = NP == 1 ? kv0 : kvm;
                        if (SCRATCH) b2e_compute<C>(E + x.k * C::QRSE + w % C::NCW, kv, TW2 + x.k, C::PA, x.k);
                        else b2_compute<C>(W + x.base, kv, TW2 + x.k, C::PA, x.k);
                    }
                if (KREUSE && k + 1 < nk) request_k((id + stride) / g.count, wid);
                __syncwarp();
#pragma unroll
                for (int m = 0; m < NQ; ++m)
                    if (lane + m * 32 < C::ITEMS_Q) {
                        const int w = lane + m * 32;
                        const ColAIdx x = colq_index<C>(cg, w);
                        if (SCRATCH) b3e_compute<C>(E + w, W + x.base);
                        else b3_compute<C>(W + x.base);
                    }
                if (SCRATCH) __syncwarp();                 // the scratch is reused by this warp's next column group
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&done[k & 1]);
        }
    }
}

// Pass C.  One CTA per (a, b2-group) tile; it loops over the transforms of the same-(j,l) batch, keeps the K psi_j and
// K psi_l accumulators of its points in registers and the psi_j / psi_l lines of the tile resident in shared memory,
// and is software-pipelined:
//   * every thread gathers the W1 columns it will transform (C0) for transform t+1 into the second work buffer with
//     16-byte cp.async while t is computed (128-byte runs, see col_index);
//   * the streamed psi_i lines arrive NSTG transforms ahead by TMA bulk copies (mbarrier completion) into operand stages;
//   * the K psi_i increment overwrites those lines and leaves by TMA bulk reduce-add (fp64) -- each K psi address
//     receives exactly one add per launch (the i of a batch are distinct and never j or l), so the result is
//     deterministic.
//   * EARLY (single work buffer only): C2 first takes its inputs into registers, which frees the buffer, and the gather
//     of transform t+1 is issued from there, so that its latency hides behind the P-point stage and the epilogue of t.
//   * TG (single work buffer, one b2 per tile, rows of a multiple of 64 elements): the tile arrives by ONE TMA tensor-box
//     copy issued by thread 0 (mbarrier completion) instead of R1 cp.async per column, in the swizzled dense layout of
//     the *_tg phase functions.
template <class C, int NBUF>
__host__ __device__ constexpr bool pass_c_tma_gather() {
#ifdef EXX_NO_TG
    return false;
#else
    return C::G == 1 && C::TC % 64 == 0 && NBUF == 1;
#endif
}
template <class C, int NT, int NSTG, int NBUF, int MINB, bool EARLY>
__global__ void __launch_bounds__(NT, MINB) pass_c_kernel(const ArgsAC g, const __grid_constant__ ArgsCX gx) {
    static_assert(!EARLY || NBUF == 1, "the early gather is the single-buffer scheme");
    constexpr bool TG = pass_c_tma_gather<C, NBUF>();
    extern __shared__ __align__(128) unsigned char smem_raw_c[];        // tensor-box destination: 128-byte aligned
    double2* const S0 = reinterpret_cast<double2*>(smem_raw_c);
    double* const OP = reinterpret_cast<double*>(S0 + NBUF * C::SMEM_C);
    double* const RES = OP + NSTG * C::OP_DOUBLES;
    __shared__ uint64_t full[NSTG];
    __shared__ uint64_t resbar, gbar;
    __shared__ double red[2][NT / 32];
    constexpr int NCLS = tg_classes(C::PC);
    __shared__ double2 s_twct[TG ? C::QC * NCLS : C::TC], s_twb[C::TB];   // twiddle tables; the c-axis one transposed to [n2*PC + k1]
                                                                          // (TG: the rotated one, [n2*NCLS + class])
    const int tile = blockIdx.x, tid = threadIdx.x;
    const int a = tile / C::TILES_PER_A, b2base = (tile % C::TILES_PER_A) * C::G;
    constexpr int NI0 = ceil_div(C::ITEMS_POS, NT), NI1 = ceil_div(C::ITEMS_LINE_P, NT), NI2 = ceil_div(C::ITEMS_LINE_Q, NT);

    if (tid == 0) {
        for (int s = 0; s < NSTG; ++s) mbar_init(&full[s], 1);
        mbar_init(&resbar, 1);
        mbar_init(&gbar, 1);
        mbar_fence_init();
    }
    if (TG) { for (int x = tid; x < C::QC * NCLS; x += NT) s_twct[x] = gx.twc_rot[x]; }
    else { for (int x = tid; x < C::TC; x += NT) s_twct[(x % C::QC) * C::PC + x / C::QC] = g.twc[x]; }
    for (int x = tid; x < C::TB; x += NT) s_twb[x] = g.twb[x];
    __syncthreads();

    ColIdx c0[NI0];
#pragma unroll
    for (int m = 0; m < NI0; ++m) c0[m] = col_index<C, true>(tid + m * NT < C::ITEMS_POS ? tid + m * NT : 0, a, b2base, g.na);
    const size_t qstride = C::w1_q(g.na), tstride = C::w1_t(g.na);
    auto issue_w1_gather = [&](int t) {
        if (TG) {                                          // one tensor box: (pin, b2, a, all pch, the R1 q-rows of transform t)
            if (tid == 0) {
                fence_proxy_async();                       // the buffer was last written by generic stores (C0 / C1 of t-1)
                mbar_arrive_expect_tx(&gbar, C::R1 * C::TC * 16);
                tensor5_g2s(S0, gx.w1_map, 0, b2base, a, 0, t * C::R1, &gbar);
            }
            return;
        }
        double2* dstbuf = S0 + (NBUF == 2 ? (t & 1) : 0) * C::SMEM_C;
        const double2* w1t = g.w1 + static_cast<size_t>(t) * tstride;
#pragma unroll
        for (int m = 0; m < NI0; ++m)
            if (tid + m * NT < C::ITEMS_POS) {
#pragma unroll
                for (int q = 0; q < C::R1; ++q) cp_async16(dstbuf + c0[m].col + q * C::ROW, w1t + c0[m].w1 + q * qstride);
            }
    };
    if (NBUF == 2 || EARLY) {
        issue_w1_gather(0);
        cp_async_commit();
    }
    if (tid < 32) {
        if (tid == 0) mbar_arrive_expect_tx(&resbar, 2 * C::LINES * C::LINE_BYTES);
        __syncwarp();
        issue_line_loads<C>(g, g.psi_r, g.j, RES, &resbar, a, b2base, tid);
        issue_line_loads<C>(g, g.psi_r, g.l >= 0 ? g.l : g.j, RES + C::LINES * C::LS, &resbar, a, b2base, tid);
        for (int t = 0; t < NSTG && t < g.count; ++t)
            issue_operand_loads<C>(g, g.desc[t], OP + static_cast<size_t>(t) * C::OP_DOUBLES, &full[t], a, b2base, tid);
    }

    LinePIdx p1[NI1];
#pragma unroll
    for (int m = 0; m < NI1; ++m) p1[m] = linep_index<C, true>(tid + m * NT < C::ITEMS_LINE_P ? tid + m * NT : 0);
    LineQIdx q2[NI2];
    double accj[NI2][C::PCN], accl[NI2][C::PCN];
#pragma unroll
    for (int m = 0; m < NI2; ++m) {
        const int w = tid + m * NT;
        q2[m] = lineq_index<C, true>(w < C::ITEMS_LINE_Q ? w : 0, a, b2base);
#pragma unroll
        for (int n1 = 0; n1 < C::PCN; ++n1) { accj[m][n1] = 0.0; accl[m][n1] = 0.0; }
    }

    XformDesc d_next = g.desc[0];                              // descriptor of the next transform, one iteration ahead
    // The operand stage of transform t is refilled (for t + NSTG) by warp 0 once the reduce-adds of t have READ it.  Waiting
    // for that right after issuing them would idle warp 0 while the other warps already run C0 of t+1 and then wait for it
    // at the next barrier; instead the refill is deferred to after warp 0's own C0 of t+1, when the reads are long done.
    // (with a single stage the operand of t+1 would then arrive late: measured +3 % at 192^3, so only with two stages)
    constexpr bool DEFER = NSTG >= 2;
    int refill_t = -1, refill_s = 0;
    for (int t = 0; t < g.count; ++t) {
        double2* S = S0 + (NBUF == 2 ? (t & 1) : 0) * C::SMEM_C;
        const int s = t % NSTG;
        double* stage = OP + static_cast<size_t>(s) * C::OP_DOUBLES;
        const XformDesc d = d_next;
        if (t + 1 < g.count) d_next = g.desc[t + 1];
        if (NBUF == 2) {
            if (t + 1 < g.count) issue_w1_gather(t + 1);
            cp_async_commit();
            cp_async_wait<1>();                            // this thread's columns of transform t have landed
        } else if (EARLY) {                                // single work buffer, gather of t issued from inside C2 of t-1
            if (TG) mbar_wait(&gbar, t & 1); else cp_async_wait<0>();
        } else {                                           // single work buffer: no overlap of the gather
            issue_w1_gather(t);
            cp_async_commit();
            if (TG) mbar_wait(&gbar, t & 1); else cp_async_wait<0>();
        }
#pragma unroll
        for (int m = 0; m < NI0; ++m)
            if (tid + m * NT < C::ITEMS_POS) {
                if constexpr (TG) c0_compute_tg<C>(S + tid + m * NT, s_twb + c0[m].b2 * C::R1);
                else c0_compute<C>(S + c0[m].col, s_twb + c0[m].b2 * C::R1);
            }
        if (DEFER && tid < 32 && refill_t >= 0) {
            bulk_wait_read_all();                          // the stage may be overwritten
            __syncwarp();
            issue_operand_loads<C>(g, g.desc[refill_t], OP + static_cast<size_t>(refill_s) * C::OP_DOUBLES, &full[refill_s], a, b2base, tid);
            refill_t = -1;
        }
        __syncthreads();
#pragma unroll
        for (int m = 0; m < NI1; ++m)
            if (tid + m * NT < C::ITEMS_LINE_P) {
                if constexpr (TG) c1_compute_tg<C>(S + ((tid + m * NT) / C::PC) * C::TC + p1[m].k1 * C::QC, (tid + m * NT) & 7, s_twct + (tid + m * NT) % NCLS, NCLS);
                else c1_compute<C>(S + p1[m].seg, s_twct + p1[m].k1, C::PC, p1[m].k1);
            }
        __syncthreads();
        double e1 = 0.0, e2 = 0.0;
        if (!EARLY) {
            if (t == 0) mbar_wait(&resbar, 0);             // psi_j / psi_l lines of the tile
            mbar_wait(&full[s], (t / NSTG) & 1);           // psi_i lines of transform t have landed
#pragma unroll
            for (int m = 0; m < NI2; ++m)
                if (tid + m * NT < C::ITEMS_LINE_Q) {
                    if constexpr (TG) {
                        double xr[C::PC], xi[C::PC];
                        c2_load_tg<C>(S + ((tid + m * NT) / C::QC) * C::TC, (tid + m * NT) / C::QC, q2[m].n2, xr, xi);
                        c2_finish<C>(xr, xi, d, g.ld, g.fj, g.fl, RES + q2[m].op, RES + C::LINES * C::LS + q2[m].op, stage + q2[m].op,
                                     accj[m], accl[m], e1, e2);
                    } else {
                        c2_compute<C>(S + q2[m].row, d, g.ld, g.fj, g.fl, RES + q2[m].op, RES + C::LINES * C::LS + q2[m].op, stage + q2[m].op,
                                      accj[m], accl[m], e1, e2);
                    }
                }
        } else {
            // single work buffer: every item first takes its inputs into registers; after the barrier nothing of transform
            // t is left in the buffer, so the W1 tile of t+1 is gathered into it while the P-point stage and the Kernel-3
            // epilogue of t run out of registers (the gather latency hides behind them)
            double xr[NI2][C::PC], xi[NI2][C::PC];
#pragma unroll
            for (int m = 0; m < NI2; ++m)
                if (tid + m * NT < C::ITEMS_LINE_Q) {
                    if constexpr (TG) c2_load_tg<C>(S + ((tid + m * NT) / C::QC) * C::TC, (tid + m * NT) / C::QC, q2[m].n2, xr[m], xi[m]);
                    else c2_load<C>(S + q2[m].row, xr[m], xi[m]);
                }
            __syncthreads();
            if (t + 1 < g.count) issue_w1_gather(t + 1);
            cp_async_commit();
            if (t == 0) mbar_wait(&resbar, 0);
            mbar_wait(&full[s], (t / NSTG) & 1);
#pragma unroll
            for (int m = 0; m < NI2; ++m)
                if (tid + m * NT < C::ITEMS_LINE_Q)
                    c2_finish<C>(xr[m], xi[m], d, g.ld, g.fj, g.fl, RES + q2[m].op, RES + C::LINES * C::LS + q2[m].op, stage + q2[m].op,
                                 accj[m], accl[m], e1, e2);
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
        if (tid == NT - 32) {                              // first lane of the last warp: warp 0 has the TMA traffic to issue
            double s1 = 0.0, s2 = 0.0;
#pragma unroll
            for (int k = 0; k < NT / 32; ++k) { s1 += red[0][k]; s2 += red[1][k]; }
            double* ep = g.epart + (static_cast<size_t>(t) * gridDim.x + tile) * 2;
            ep[0] = s1; ep[1] = s2;
        }
        if (tid < 32) {
            // K psi_i += -(f_j V_ji psi_j + f_l V_li psi_l)   (the same V serves both orbitals of a pair)
            if (g.kpsi != nullptr && d.flags != 0 && d.i != g.jd && d.i != g.ld) {
                double* ki = g.kpsi + static_cast<size_t>(d.i) * g.m_points;
                for (int l = tid; l < C::LINES; l += 32)
                    bulk_red_add_f64(ki + line_offset<C>(l, a, b2base), stage + l * C::LS, C::LINE_BYTES);
            }
            bulk_commit();
            if (t + NSTG < g.count) {
                if (DEFER) {
                    refill_t = t + NSTG; refill_s = s;
                } else {
                    bulk_wait_read_all();                  // the stage may be overwritten
                    __syncwarp();
                    issue_operand_loads<C>(g, g.desc[t + NSTG], stage, &full[s], a, b2base, tid);
                }
            }
        }
    }
    // K psi_j -= accj, K psi_l -= accl (this CTA is the only writer of its tile of K psi_j, K psi_l in this launch)
#pragma unroll
    for (int m = 0; m < NI2; ++m)
        if (g.kpsi_r != nullptr && tid + m * NT < C::ITEMS_LINE_Q) {
            double* kj = g.kpsi_r + static_cast<size_t>(g.j) * g.m_points + q2[m].gofs;
#pragma unroll
            for (int n1 = 0; n1 < C::PCN; ++n1) kj[C::QC * n1] -= accj[m][n1];
            if (g.l >= 0) {
                double* kl = g.kpsi_r + static_cast<size_t>(g.l) * g.m_points + q2[m].gofs;
#pragma unroll
                for (int n1 = 0; n1 < C::PCN; ++n1) kl[C::QC * n1] -= accl[m][n1];
            }
        }
    if (tid < 32) bulk_wait_read_all();                    // shared memory must outlive the TMA reads
}

// Pass C, warp-specialised variant (used where two W1 tile buffers, two operand stages and two CTAs fit an SM).
// NAW "column" warps gather the W1 tile of transform t+1 (16-byte cp.async) and run the inverse b-axis stage C0 in one
// work buffer while NBW "line" warps run the inverse c-axis FFT C1, C2 and the Kernel-3 epilogue of transform t out of
// the other, so the gather latency and the load-heavy phase overlap the FP64-heavy ones.  Buffers are handed over with
// mbarriers (c0done: column -> line warps, sfree: back); the line warps synchronise among themselves with a named
// barrier.  Arithmetic, accumulation order and the one-reduce-add-per-address rule are those of pass_c_kernel.
template <class C, int NAW, int NBW, int NSTG, int MINB>
__global__ void __launch_bounds__(32 * (NAW + NBW), MINB) pass_c_ws_kernel(const ArgsAC g) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* const S0 = reinterpret_cast<double2*>(smem_raw);
    double* const OP = reinterpret_cast<double*>(S0 + 2 * C::SMEM_C);
    double* const RES = OP + NSTG * C::OP_DOUBLES;
    __shared__ uint64_t full[NSTG], resbar, c0done[2], sfree[2];
    __shared__ double red[2][NBW];
    __shared__ double2 s_twct[C::TC], s_twb[C::TB];
    constexpr int NT = 32 * (NAW + NBW), AT = 32 * NAW, BT = 32 * NBW;
    const int tile = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
    const int a = tile / C::TILES_PER_A, b2base = (tile % C::TILES_PER_A) * C::G;

    if (tid == 0) {
        for (int s = 0; s < NSTG; ++s) mbar_init(&full[s], 1);
        mbar_init(&resbar, 1);
        for (int b = 0; b < 2; ++b) { mbar_init(&c0done[b], NAW); mbar_init(&sfree[b], NBW); }
        mbar_fence_init();
    }
    for (int x = tid; x < C::TC; x += NT) s_twct[(x % C::QC) * C::PC + x / C::QC] = g.twc[x];
    for (int x = tid; x < C::TB; x += NT) s_twb[x] = g.twb[x];
    __syncthreads();

    if (tid >= BT) {
        // ------------------------------------------------------------------ column warps: W1 gather + C0
        const int at = tid - BT;
        constexpr int NI0 = ceil_div(C::ITEMS_POS, AT);
        ColIdx c0[NI0];
#pragma unroll
        for (int m = 0; m < NI0; ++m) c0[m] = col_index<C, true>(at + m * AT < C::ITEMS_POS ? at + m * AT : 0, a, b2base, g.na);
        const size_t qstride = C::w1_q(g.na), tstride = C::w1_t(g.na);
        for (int t = 0; t < g.count; ++t) {
            const int b = t & 1;
            double2* const S = S0 + b * C::SMEM_C;
            const double2* w1t = g.w1 + static_cast<size_t>(t) * tstride;
            if (t >= 2) mbar_wait(&sfree[b], ((t >> 1) - 1) & 1);      // the line warps have drained this buffer
#pragma unroll
            for (int m = 0; m < NI0; ++m)
                if (at + m * AT < C::ITEMS_POS) {
#pragma unroll
                    for (int q = 0; q < C::R1; ++q) cp_async16(S + c0[m].col + q * C::ROW, w1t + c0[m].w1 + q * qstride);
                }
            cp_async_commit();
            cp_async_wait<0>();
#pragma unroll
            for (int m = 0; m < NI0; ++m)
                if (at + m * AT < C::ITEMS_POS) c0_compute<C>(S + c0[m].col, s_twb + c0[m].b2 * C::R1);
            __syncwarp();
            if (lane == 0) mbar_arrive(&c0done[b]);
        }
    } else {
        // ------------------------------------------------------------------ line warps: C1, C2, epilogue
        constexpr int NI1 = ceil_div(C::ITEMS_LINE_P, BT), NI2 = ceil_div(C::ITEMS_LINE_Q, BT);
        if (tid < 32) {
            if (tid == 0) mbar_arrive_expect_tx(&resbar, 2 * C::LINES * C::LINE_BYTES);
            __syncwarp();
            issue_line_loads<C>(g, g.psi_r, g.j, RES, &resbar, a, b2base, tid);
            issue_line_loads<C>(g, g.psi_r, g.l >= 0 ? g.l : g.j, RES + C::LINES * C::LS, &resbar, a, b2base, tid);
            for (int t = 0; t < NSTG && t < g.count; ++t)
                issue_operand_loads<C>(g, g.desc[t], OP + static_cast<size_t>(t) * C::OP_DOUBLES, &full[t], a, b2base, tid);
        }
        LinePIdx p1[NI1];
#pragma unroll
        for (int m = 0; m < NI1; ++m) p1[m] = linep_index<C, true>(tid + m * BT < C::ITEMS_LINE_P ? tid + m * BT : 0);
        LineQIdx q2[NI2];
        double accj[NI2][C::PCN], accl[NI2][C::PCN];
#pragma unroll
        for (int m = 0; m < NI2; ++m) {
            const int w = tid + m * BT;
            q2[m] = lineq_index<C, true>(w < C::ITEMS_LINE_Q ? w : 0, a, b2base);
#pragma unroll
            for (int n1 = 0; n1 < C::PCN; ++n1) { accj[m][n1] = 0.0; accl[m][n1] = 0.0; }
        }
        XformDesc d_next = g.desc[0];
        for (int t = 0; t < g.count; ++t) {
            const int b = t & 1, s = t % NSTG;
            double2* const S = S0 + b * C::SMEM_C;
            double* stage = OP + static_cast<size_t>(s) * C::OP_DOUBLES;
            const XformDesc d = d_next;
            if (t + 1 < g.count) d_next = g.desc[t + 1];
            mbar_wait(&c0done[b], (t >> 1) & 1);
#pragma unroll
            for (int m = 0; m < NI1; ++m)
                if (tid + m * BT < C::ITEMS_LINE_P) c1_compute<C>(S + p1[m].seg, s_twct + p1[m].k1, C::PC, p1[m].k1);
            asm volatile("bar.sync 1, %0;" ::"n"(BT) : "memory");
            if (t == 0) mbar_wait(&resbar, 0);
            mbar_wait(&full[s], (t / NSTG) & 1);
            double e1 = 0.0, e2 = 0.0;
#pragma unroll
            for (int m = 0; m < NI2; ++m)
                if (tid + m * BT < C::ITEMS_LINE_Q)
                    c2_compute<C>(S + q2[m].row, d, g.ld, g.fj, g.fl, RES + q2[m].op, RES + C::LINES * C::LS + q2[m].op, stage + q2[m].op,
                                  accj[m], accl[m], e1, e2);
            fence_proxy_async();
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                e1 += __shfl_xor_sync(0xffffffffu, e1, o);
                e2 += __shfl_xor_sync(0xffffffffu, e2, o);
            }
            if (lane == 0) {
                red[0][tid >> 5] = e1; red[1][tid >> 5] = e2;
                mbar_arrive(&sfree[b]);                                // this warp no longer reads the work buffer
            }
            asm volatile("bar.sync 1, %0;" ::"n"(BT) : "memory");      // operand stage and red[] complete
            if (tid == 0) {
                double s1 = 0.0, s2 = 0.0;
#pragma unroll
                for (int k = 0; k < NBW; ++k) { s1 += red[0][k]; s2 += red[1][k]; }
                double* ep = g.epart + (static_cast<size_t>(t) * gridDim.x + tile) * 2;
                ep[0] = s1; ep[1] = s2;
            }
            if (tid < 32) {
                if (g.kpsi != nullptr && d.flags != 0 && d.i != g.jd && d.i != g.ld) {
                    double* ki = g.kpsi + static_cast<size_t>(d.i) * g.m_points;
                    for (int l = tid; l < C::LINES; l += 32)
                        bulk_red_add_f64(ki + line_offset<C>(l, a, b2base), stage + l * C::LS, C::LINE_BYTES);
                }
                bulk_commit();
                if (t + NSTG < g.count) {
                    bulk_wait_read_all();
                    __syncwarp();
                    issue_operand_loads<C>(g, g.desc[t + NSTG], stage, &full[s], a, b2base, tid);
                }
            }
            // red[] is rewritten only after the next named barrier pair, the stage only after its mbarrier: no hazard
        }
#pragma unroll
        for (int m = 0; m < NI2; ++m)
            if (g.kpsi_r != nullptr && tid + m * BT < C::ITEMS_LINE_Q) {
                double* kj = g.kpsi_r + static_cast<size_t>(g.j) * g.m_points + q2[m].gofs;
#pragma unroll
                for (int n1 = 0; n1 < C::PCN; ++n1) kj[C::QC * n1] -= accj[m][n1];
                if (g.l >= 0) {
                    double* kl = g.kpsi_r + static_cast<size_t>(g.l) * g.m_points + q2[m].gofs;
#pragma unroll
                    for (int n1 = 0; n1 < C::PCN; ++n1) kl[C::QC * n1] -= accl[m][n1];
                }
            }
        if (tid < 32) bulk_wait_read_all();
    }
}

#endif  // __CUDACC__

}  // namespace exx
