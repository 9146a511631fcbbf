// exx_inst.cuh -- list of compiled (TA|TC, TB) kernel geometries, shared by the three instantiation files.
// Cubic grids of every supported length, plus every mix of the lengths 16, 32, 64.
#pragma once

#define EXX_FOR_EACH_PAIR(X) \
    X(16, 16) X(16, 32) X(16, 64) X(32, 16) X(32, 32) X(32, 64) X(64, 16) X(64, 32) X(64, 64) \
    X(96, 96) X(128, 128) X(192, 192) X(256, 256)
