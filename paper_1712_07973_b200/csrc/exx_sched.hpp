// exx_sched.hpp -- host-side pair scheduler (pure C++, no CUDA): "form all the N(N+1)/2 charge
// densities rho_ij ... and then solve the Poisson's equation for each of them"; Table 1.
//
// Orbitals are taken two at a time: block-row m = {j, l} = {2m, 2m+1} (l = -1 for the last orbital of an odd N) owns
// the pairs (j,i), i >= j, and (l,i), i >= l.  One complex transform carries the two pairs that the streamed orbital i
// forms with the block-row (real part: (j,i), imaginary part: (l,i)); i = j has only the diagonal pair (j,j).  A pair
// is skipped only if both occupations are zero (reading A15).  Block-rows are cut into batches of at most
// max_batch transforms; all transforms of a batch share (j,l), so pass C keeps K psi_j and K psi_l on chip and the
// K psi_i updates of one batch never collide (the i of a block-row are distinct).
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

inline Schedule build_schedule(int n_orb, const double* occ, int max_batch) {
    Schedule s;
    if (max_batch < 1) max_batch = 1;
    for (int j = 0; j < n_orb; j += 2) {
        const int l = j + 1 < n_orb ? j + 1 : -1;
        const int row_first = static_cast<int>(s.xforms.size());
        for (int i = j; i < n_orb; ++i) {
            int flags = 0;
            if (!(occ[j] == 0.0 && occ[i] == 0.0)) flags |= 1;
            if (l >= 0 && i >= l && !(occ[l] == 0.0 && occ[i] == 0.0)) flags |= 2;
            if (flags == 0) continue;
            s.n_pairs += (flags & 1) + ((flags >> 1) & 1);
            s.xforms.push_back(XformDesc{i, flags, occ[i]});
        }
        const int row_count = static_cast<int>(s.xforms.size()) - row_first;
        for (int off = 0; off < row_count; off += max_batch) {
            Batch b;
            b.j = j; b.l = l;
            b.fj = occ[j]; b.fl = l >= 0 ? occ[l] : 0.0;
            b.first = row_first + off;
            b.count = row_count - off < max_batch ? row_count - off : max_batch;
            s.batches.push_back(b);
        }
    }
    return s;
}

}  // namespace exx
