"""CPU emulation of the CUDA pass kernels vs the oracle (no GPU needed).

tests/emu/emu_passes.cu runs the very same per-work-item phase functions the kernels run
(paper_1712_07973_b200/csrc/exx_passes.cuh), sequentially on the host.  This checks the index algebra of the
4-step FFT split, the digit-scrambled K^ lookup, the Hockney pruning and the fused prologue/epilogue against
oracle.poisson -- the GPU parity tests (-m gpu) then only have to catch what is specific to the device.
"""
import ctypes as C
import os
import shutil
import subprocess

import numpy as np
import pytest

from oracle import Oracle
from workloads import make_workload, small_spec

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = os.path.join(HERE, "emu", "emu_passes.cu")
LIB = os.path.join(HERE, "emu", "libexx_emu.so")
CSRC = os.path.join(ROOT, "paper_1712_07973_b200", "csrc")

SPLIT = {16: (4, 4), 32: (4, 8), 64: (8, 8), 96: (8, 12), 128: (8, 16), 192: (12, 16), 256: (16, 16)}


def _build():
    deps = [SRC] + [os.path.join(CSRC, f) for f in ("exx_passes.cuh", "exx_dft.cuh")]
    if os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    subprocess.run([nvcc, "-std=c++17", "-O1", "-x", "cu", "-Wno-deprecated-gpu-targets", "-Xcompiler", "-fPIC", "-shared",
                    "-I", CSRC, "-o", LIB, SRC], check=True)
    return LIB


@pytest.fixture(scope="module")
def emu():
    lib = C.CDLL(_build())
    dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
    lib.exx_emu_batch.argtypes = [C.c_int] * 6 + [dp, dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, ip, dp, dp, dp, dp, dp, dp]
    return lib


def _tw(T):
    P, Q = SPLIT[T]
    k1 = np.arange(P)[:, None]
    n2 = np.arange(Q)[None, :]
    return np.ascontiguousarray(np.exp(-2j * np.pi * ((k1 * n2) % T) / T).reshape(-1))


def _roots(T):
    return np.ascontiguousarray(np.exp(-2j * np.pi * np.arange(T) / T))


CASES = [
    # ta, tb, tc, free, G, chunk
    (16, 16, 16, 0, 1, 4), (16, 16, 16, 0, 2, 2), (16, 16, 16, 1, 2, 4), (32, 32, 32, 0, 4, 4), (32, 32, 32, 1, 1, 2),
    (16, 32, 64, 0, 2, 4), (64, 16, 32, 1, 4, 4), (16, 96, 16, 1, 3, 2), (16, 16, 128, 0, 1, 4), (128, 16, 16, 1, 1, 4),
    (16, 192, 16, 0, 1, 4), (192, 16, 16, 0, 1, 4), (16, 16, 192, 1, 1, 4), (16, 256, 16, 1, 1, 2),
    (256, 16, 16, 0, 1, 2), (16, 16, 256, 1, 1, 2), (96, 96, 96, 0, 2, 4),
]


@pytest.mark.parametrize("ta,tb,tc,free,G,chunk", CASES)
def test_emulated_batch_matches_oracle(emu, ta, tb, tc, free, G, chunk):
    dims = tuple(t // 2 if free else t for t in (ta, tb, tc))
    base = "C2" if free else "C1"
    n_orb = 4 if max(ta, tb, tc) < 96 or min(ta, tb, tc) < 96 else 3
    w = make_workload(small_spec(base, dims=dims, n_orb=n_orb, spacing=(0.45, 0.5, 0.4), number=100 + ta + tb + tc))
    psi = np.ascontiguousarray(w["psi"].numpy())
    o = Oracle(dims, w["spec"].spacing, "free" if free else "periodic", w["kernel"])
    occ = np.array([2.0, 1.5, 0.75, 1.0])[:n_orb]
    # the same-(j,l) batch of block-row {0,1}: i = 0 carries only the diagonal pair (0,0); i = 1 the pairs (0,1), (1,1);
    # i >= 2 the pairs (0,i), (1,i).  N = 3 cases also run the odd tail block-row {2} (l = -1).
    batches = [(0, 1, [(i, 1 if i == 0 else 3) for i in range(n_orb)])]
    if n_orb == 3:
        batches.append((2, -1, [(2, 1)]))
    khat = o.khat()
    T_tot = ta * tb * tc
    ks = np.ascontiguousarray(khat.real[: ta // 2 + 1, : tb // 2 + 1, : tc // 2 + 1]) / T_tot
    kpsi = np.zeros_like(psi)
    twa, twc, rootsb = _tw(ta), _tw(tc), _roots(tb)
    d = lambda x: x.ctypes.data_as(C.POINTER(C.c_double))
    ref = np.zeros_like(psi)
    for j, l, xf in batches:
        count = len(xf)
        iflags = np.array(xf, dtype=np.int32)
        fis = np.array([occ[i] for i, _ in xf])
        e_out = np.zeros(2 * count)
        rc = emu.exx_emu_batch(ta, tb, tc, free, G, chunk, d(psi), d(kpsi), j, l, float(occ[j]), float(occ[l]) if l >= 0 else 0.0,
                               count, iflags.ctypes.data_as(C.POINTER(C.c_int)), d(fis), d(twa.view(np.float64)),
                               d(twc.view(np.float64)), d(rootsb.view(np.float64)), d(ks), d(e_out))
        assert rc == 0, "case not instantiated in tests/emu/emu_passes.cu"
        e_ref = []
        for i, flags in xf:
            for bit, x in ((1, j), (2, l)):
                if not flags & bit:
                    e_ref.append(0.0)
                    continue
                rho = psi[x] * psi[i]
                v = o.poisson(rho)
                ref[x] -= occ[i] * v * psi[i]
                if x != i:
                    ref[i] -= occ[x] * v * psi[x]
                e_ref.append(np.sum(rho * v))
        e_ref = np.array(e_ref)
        assert np.max(np.abs(e_out - e_ref)) <= 1e-12 * np.max(np.abs(e_ref))
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(kpsi - ref)) <= 1e-12 * scale
