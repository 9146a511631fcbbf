// exx_inst.cuh -- which (TA | TC, TB) kernel geometries are compiled, shared by the instantiation files.
// Main lengths: every mix over the three axes.  Extra lengths: cubic transform grids only.  Each instantiation file
// (exx_pass_{a,b,c}.cu) is compiled once per middle-axis length with -DEXX_TB=<length> (paper_1712_07973_b200/build.py),
// so the template instantiations spread over many translation units that build in parallel.
#pragma once

#include "exx_passes.cuh"

#ifdef EXX_DEV_LENGTHS_LIST
// development builds only (EXX_DEV_LENGTHS=96,192 python -m paper_1712_07973_b200.build): a subset of the main lengths,
// no extra lengths; every other geometry then reports EXX_ERR_UNSUPPORTED_SIZE.  Never the shipped configuration.
#define EXX_MAIN_LENGTHS(X) EXX_DEV_LENGTHS_LIST
#define EXX_EXTRA_LENGTHS(X)
#else
#define EXX_MAIN_LENGTHS(X) X(16) X(32) X(48) X(64) X(96) X(128) X(144) X(192) X(256)
#define EXX_EXTRA_LENGTHS(X) X(24) X(72)
#endif
#define EXX_ALL_LENGTHS(X) EXX_MAIN_LENGTHS(X) EXX_EXTRA_LENGTHS(X)

#define EXX_CAT2(a, b) a##b
#define EXX_CAT(a, b) EXX_CAT2(a, b)

namespace exx {

// chunk_for() runs a compile-time search over shared-memory paddings: evaluate it once per (TA, TB, BC) as a static
// member (one constant expression each) instead of inside larger constant expressions.
template <int TA, int TB, bool FREE>
struct ChunkOf { static constexpr int value = chunk_for(TA, TB, FREE); };

// Can a plan with middle-axis length TB have the W1 layout parameter CHUNK = CH (for ANY admissible a-axis length)?
// Passes A / C are instantiated for exactly these values.
template <int TB, bool FREE, int CH>
constexpr bool chunk_possible() {
    if constexpr (is_extra_length(TB)) {
        return ChunkOf<TB, TB, FREE>::value == CH;
    } else {
#define X(TA_) || ChunkOf<TA_, TB, FREE>::value == CH
        return false EXX_MAIN_LENGTHS(X);
#undef X
    }
}

}  // namespace exx
