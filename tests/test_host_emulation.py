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

SPLIT = {16: (4, 4), 24: (2, 12), 32: (4, 8), 48: (4, 12), 64: (8, 8), 72: (6, 12), 96: (8, 12), 128: (8, 16), 144: (12, 12), 192: (12, 16),
         256: (16, 16)}


def _build():
    deps = [SRC] + [os.path.join(CSRC, f) for f in ("exx_passes.cuh", "exx_dft.cuh", "exx_async.cuh")]
    if os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    subprocess.run([nvcc, "-std=c++17", "-O1", "-x", "cu", "-arch=sm_100a", "-Wno-deprecated-gpu-targets", "-Xcompiler", "-fPIC", "-shared",
                    "-I", CSRC, "-o", LIB, SRC], check=True)
    return LIB


@pytest.fixture(scope="module")
def emu():
    lib = C.CDLL(_build())
    dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
    lib.exx_emu_batch.argtypes = [C.c_int] * 7 + [dp, dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, ip, dp, dp, dp, dp, dp, dp]
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
    # lengths added in round 2 (radix-3 heavy: 48 = 4*12, 144 = 12*12, 24 = 2*12, 72 = 6*12) on every axis role
    (48, 48, 48, 0, 3, 4), (48, 16, 16, 1, 1, 4), (16, 48, 16, 1, 2, 2), (16, 16, 48, 0, 1, 4),
    (144, 16, 16, 0, 1, 4), (16, 144, 16, 1, 3, 2), (16, 16, 144, 1, 1, 4), (24, 24, 24, 0, 2, 4), (24, 24, 24, 1, 3, 2),
    (72, 72, 72, 1, 2, 4), (72, 72, 72, 0, 1, 2),
]


def _run_case(emu, ta, tb, tc, free, G, chunk, n_orb, occ, max_batch=0, variant=0):
    """Runs the library's own schedule (exx_schedule_list) for these occupations through the emulated passes and
    compares K psi and the pair energies with the oracle, pair by pair."""
    import paper_1712_07973_b200 as exx
    dims = tuple(t // 2 if free else t for t in (ta, tb, tc))
    base = "C2" if free else "C1"
    w = make_workload(small_spec(base, dims=dims, n_orb=n_orb, spacing=(0.45, 0.5, 0.4), number=100 + ta + tb + tc))
    psi = np.ascontiguousarray(w["psi"].numpy())
    o = Oracle(dims, w["spec"].spacing, "free" if free else "periodic", w["kernel"])
    occ = np.asarray(occ, dtype=np.float64)
    rows = exx.exx_schedule_list(occ, max_batch)
    batches = {}
    for j, l, i, flags, b in rows.tolist():
        batches.setdefault(b, (j, l, []))[2].append((i, flags))
    khat = o.khat()
    T_tot = ta * tb * tc
    ks = np.ascontiguousarray(khat.real[: ta // 2 + 1, : tb // 2 + 1, : tc // 2 + 1]) / T_tot
    kpsi = np.zeros_like(psi)
    twa, twc, rootsb = _tw(ta), _tw(tc), _roots(tb)
    d = lambda x: x.ctypes.data_as(C.POINTER(C.c_double))
    ref = np.zeros_like(psi)
    for b in sorted(batches):
        j, l, xf = batches[b]
        count = len(xf)
        iflags = np.array(xf, dtype=np.int32)
        fis = np.array([occ[i] for i, _ in xf])
        e_out = np.zeros(2 * count)
        rc = emu.exx_emu_batch(variant, ta, tb, tc, free, G, chunk, d(psi), d(kpsi), j, l, float(occ[j]), float(occ[l]) if l >= 0 else 0.0,
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
        assert np.max(np.abs(e_out - e_ref)) <= 1e-12 * max(np.max(np.abs(e_ref)), 1e-300)
    # the batches together are the whole operator: compare with the oracle's definition as well
    k_def, _, _ = o.apply(psi, occ, symmetric=False)
    scale = np.max(np.abs(k_def))
    assert np.max(np.abs(ref - k_def)) <= 1e-12 * scale
    assert np.max(np.abs(kpsi - ref)) <= 1e-12 * scale


@pytest.mark.parametrize("ta,tb,tc,free,G,chunk", CASES)
def test_emulated_batch_matches_oracle(emu, ta, tb, tc, free, G, chunk):
    big = max(ta, tb, tc) >= 96 and min(ta, tb, tc) >= 96
    n_orb = 3 if big else 4                              # N = 3: odd tail block-row {2} with l = -1
    _run_case(emu, ta, tb, tc, free, G, chunk, n_orb, [2.0, 1.5, 0.75, 1.0][:n_orb])


@pytest.mark.parametrize("ta,tb,tc,free,G,chunk", [c for c in CASES if c[3] == 1][:6] + [(32, 32, 32, 0, 4, 4)])
def test_emulated_scratch_variant_matches_oracle(emu, ta, tb, tc, free, G, chunk):
    """The warp-specialised pass B: block landed in place, a-axis phases through the per-warp expansion scratch."""
    _run_case(emu, ta, tb, tc, free, G, chunk, 3, [2.0, 1.5, 0.75], variant=1)


@pytest.mark.parametrize("occ,max_batch", [([0.0, 1.2, 0.0, 0.0, 2.0], 0),      # imaginary-slot-only transforms (flags = 2), odd N
                                           ([2.0, 0.0, 1.0, 0.0, 0.0, 0.3], 2),  # real-slot-only transforms, block-rows cut in batches
                                           ([1.0, 2.0, 0.5], 1)])                # one transform per batch: i = j and i = l alone
def test_emulated_schedule_edge_cases(emu, occ, max_batch):
    _run_case(emu, 16, 16, 16, 0, 2, 2, len(occ), occ, max_batch)
    _run_case(emu, 16, 16, 16, 1, 2, 4, len(occ), occ, max_batch)
