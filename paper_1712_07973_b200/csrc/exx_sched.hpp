// exx_sched.hpp -- host-side pair scheduler (pure C++, no CUDA): "form all the N(N+1)/2 charge
// densities rho_ij ... and then solve the Poisson's equation for each of them"; Table 1.
//
// Row i owns the pairs (i,j), j >= i.  A pair is skipped only if f_i = f_j = 0 (reading A15).
// Two pairs of the same row share one complex transform (real part: (i,j), imaginary part: (i,l)); a row with an
// odd number of pairs ends with a half-empty transform (l = -1).  Rows are cut into batches of at most
// max_batch transforms; all transforms of a batch share i, so pass C can keep K psi_i on chip and the
// K psi_j updates of one batch never collide (the j of a row are distinct).
#pragma once

#include <vector>

#include "exx_passes.cuh"

namespace exx {

struct Batch {
    int i;            // common orbital
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
    for (int i = 0; i < n_orb; ++i) {
        const int row_first = static_cast<int>(s.xforms.size());
        XformDesc cur{-1, -1, 0.0, 0.0};
        for (int j = i; j < n_orb; ++j) {
            if (occ[i] == 0.0 && occ[j] == 0.0) continue;
            ++s.n_pairs;
            if (cur.j < 0) {
                cur.j = j; cur.fj = occ[j];
            } else {
                cur.l = j; cur.fl = occ[j];
                s.xforms.push_back(cur);
                cur = XformDesc{-1, -1, 0.0, 0.0};
            }
        }
        if (cur.j >= 0) s.xforms.push_back(cur);
        const int row_count = static_cast<int>(s.xforms.size()) - row_first;
        for (int off = 0; off < row_count; off += max_batch) {
            Batch b;
            b.i = i;
            b.first = row_first + off;
            b.count = row_count - off < max_batch ? row_count - off : max_batch;
            s.batches.push_back(b);
        }
    }
    return s;
}

}  // namespace exx
