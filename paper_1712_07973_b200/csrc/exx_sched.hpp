// exx_sched.hpp -- host-side pair scheduler (pure C++, no CUDA): "form all the N(N+1)/2 charge
// densities rho_ij ... and then solve the Poisson's equation for each of them"; Table 1.
//
// SQUARE schedule (exx_apply: one orbital set on both sides).  Orbitals are taken two at a time: block-row
// m = {j, l} = {2m, 2m+1} (l = -1 for the last orbital of an odd N) owns the pairs (j,i), i >= j, and (l,i), i >= l.
// One complex transform carries the two pairs that the streamed orbital i forms with the block-row (real part: (j,i),
// imaginary part: (l,i)); i = j has only the diagonal pair (j,j).  A pair is skipped only if both occupations are zero
// (reading A15) or if an optional pair mask excludes it (localised orbitals, Eq. 6-7: the
// caller lists the pairs whose co-density does not vanish).  Block-rows are cut into batches of at most max_batch
// transforms; all transforms of a batch share (j,l), so pass C keeps K psi_j and K psi_l on chip and the K psi_i updates
// of one batch never collide (the i of a block-row are distinct).
//
// RECTANGULAR schedule (exx_apply_to / exx_apply_block: pairs between two DIFFERENT sets, Fig. 1 "each
// process ... calculates the co-densities between its own orbitals and the received ones"): block-rows {j, l} run over the
// RESIDENT set, every orbital i of the STREAMED set forms the pairs (j,i) and (l,i); there is no diagonal.
//
// The builders only clear and refill the vectors of a caller-owned Schedule: once those have been reserved for the
// largest apply of a plan (reserve_schedule), building a schedule allocates nothing.
#pragma once

#include <vector>

#include "exx_passes.cuh"

namespace exx {

struct Batch {
    int j, l;         // resident orbitals (l < 0: none)
    double fj, fl;
    int first;        // index of the first transform descriptor
    int count;        // transforms in this batch
};

struct Schedule {
    std::vector<XformDesc> xforms;
    std::vector<Batch> batches;
    long long n_pairs = 0;
};

// upper bounds for n_res resident x n_str streamed orbitals (square: n_res = n_str = N): one transform per (block-row,
// streamed orbital); every batch holds at least one transform
inline size_t max_transforms(size_t n_res, size_t n_str) { return ((n_res + 1) / 2) * n_str; }

inline void reserve_schedule(Schedule& s, size_t n_res, size_t n_str) {
    s.xforms.reserve(max_transforms(n_res, n_str));
    s.batches.reserve(max_transforms(n_res, n_str));
}

inline void cut_batches(Schedule& s, int j, int l, double fj, double fl, int row_first, int max_batch) {
    const int row_count = static_cast<int>(s.xforms.size()) - row_first;
    for (int off = 0; off < row_count; off += max_batch) {
        Batch b;
        b.j = j; b.l = l;
        b.fj = fj; b.fl = fl;
        b.first = row_first + off;
        b.count = row_count - off < max_batch ? row_count - off : max_batch;
        s.batches.push_back(b);
    }
}

// mask: optional [n_orb][n_orb] bytes, pair (a,b) is solved iff mask[a*n_orb+b] != 0 (the caller passes a symmetric mask)
inline void build_schedule(Schedule& s, int n_orb, const double* occ, int max_batch, const unsigned char* mask = nullptr) {
    s.xforms.clear();
    s.batches.clear();
    s.n_pairs = 0;
    if (max_batch < 1) max_batch = 1;
    for (int j = 0; j < n_orb; j += 2) {
        const int l = j + 1 < n_orb ? j + 1 : -1;
        const int row_first = static_cast<int>(s.xforms.size());
        for (int i = j; i < n_orb; ++i) {
            int flags = 0;
            if (!(occ[j] == 0.0 && occ[i] == 0.0) && (!mask || mask[static_cast<size_t>(j) * n_orb + i])) flags |= 1;
            if (l >= 0 && i >= l && !(occ[l] == 0.0 && occ[i] == 0.0) && (!mask || mask[static_cast<size_t>(l) * n_orb + i])) flags |= 2;
            if (flags == 0) continue;
            s.n_pairs += (flags & 1) + ((flags >> 1) & 1);
            s.xforms.push_back(XformDesc{i, flags, occ[i]});
        }
        cut_batches(s, j, l, occ[j], l >= 0 ? occ[l] : 0.0, row_first, max_batch);
    }
}

// occ_res may be nullptr (exx_apply_to: the resident set carries no occupations -- it only receives);
// skip_empty_streamed: streamed orbitals with f_i = 0 contribute nothing when only the resident side is updated
inline void build_schedule_rect(Schedule& s, int n_res, const double* occ_res, int n_str, const double* occ_str, bool skip_empty_streamed,
                                int max_batch) {
    s.xforms.clear();
    s.batches.clear();
    s.n_pairs = 0;
    if (max_batch < 1) max_batch = 1;
    for (int j = 0; j < n_res; j += 2) {
        const int l = j + 1 < n_res ? j + 1 : -1;
        const double fj = occ_res ? occ_res[j] : 0.0, fl = (occ_res && l >= 0) ? occ_res[l] : 0.0;
        const int row_first = static_cast<int>(s.xforms.size());
        for (int i = 0; i < n_str; ++i) {
            int flags = 0;
            if (skip_empty_streamed) {
                if (occ_str[i] != 0.0) flags = l >= 0 ? 3 : 1;
            } else {
                if (!(fj == 0.0 && occ_str[i] == 0.0)) flags |= 1;
                if (l >= 0 && !(fl == 0.0 && occ_str[i] == 0.0)) flags |= 2;
            }
            if (flags == 0) continue;
            s.n_pairs += (flags & 1) + ((flags >> 1) & 1);
            s.xforms.push_back(XformDesc{i, flags, occ_str[i]});
        }
        cut_batches(s, j, l, fj, fl, row_first, max_batch);
    }
}

}  // namespace exx
