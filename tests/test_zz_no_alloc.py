"""The allocation-free entry point exx_exchange_energy_noalloc (include/exx.h; csrc/exx_noalloc.cu) against the existing path.

Collected last on purpose (the suite runs with `pytest -x`: a failure here must not hide other tests).  The entry point
evaluates E_x = 1/2 dV sum_i f_i <psi_i|K psi_i> with its scratch in a static __device__ array; the existing path's E_x is the
one exx_apply reduces from the pair energies (Eq. 5).  Two calls in a row on different inputs: the scratch keeps
the previous call's contents, which must not leak into the next result.  Tolerance: north_star's 1e-11 on E_x.
"""
import ctypes as C

import numpy as np
import pytest
import torch

import paper_1712_07973_b200 as exx
from workloads import make_workload, small_spec

E_RTOL = 1e-11


@pytest.mark.gpu
def test_noalloc_energy_matches_apply_on_two_calls_in_a_row():
    cases = [("C1", (32, 32, 32), 6, np.array([2.0, 1.0, 0.0, 0.5, 1.5, 2.0])),
             ("C2", (16, 32, 16), 3, np.array([2.0, 0.7, 1.3])),            # fewer orbitals, fewer blocks than the call before
             ("C1", (96, 96, 96), 4, np.array([2.0, 2.0, 1.0, 0.25]))]
    ex_dev = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    for base, dims, n_orb, occ in cases:
        w = make_workload(small_spec(base, dims=dims, n_orb=n_orb, number=2600 + sum(dims)))
        spec = w["spec"]
        plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=n_orb)
        psi = w["psi"].cuda()
        kpsi, ex_ref = plan.apply(psi, occ)
        before = torch.cuda.memory_allocated()
        exx.exx_exchange_energy_noalloc(psi, kpsi, occ, spec.dV, ex_dev)
        exx.exx_exchange_energy_noalloc(psi, kpsi, occ, spec.dV, ex_dev)          # second call in a row, same stream: same result
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before
        assert abs(float(ex_dev[0]) - ex_ref) <= E_RTOL * abs(ex_ref)
        plan.destroy()


@pytest.mark.gpu
def test_noalloc_rejects_sizes_beyond_the_static_scratch():
    lib = exx.load_library()
    x = torch.zeros(8, dtype=torch.float64, device="cuda")
    occ = np.ones(exx.binding.EXX_NOALLOC_MAX_ORBITALS + 1)
    st = lib.exx_exchange_energy_noalloc(occ.size, 1, 1.0, C.c_void_p(x.data_ptr()), C.c_void_p(x.data_ptr()),
                                         occ.ctypes.data_as(C.POINTER(C.c_double)), C.c_void_p(x.data_ptr()), None)
    assert st == 2 and b"EXX_NOALLOC_MAX_ORBITALS" in lib.exx_noalloc_last_error()
    st = lib.exx_exchange_energy_noalloc(1, 8, 1.0, C.c_void_p(x.data_ptr()), C.c_void_p(x.data_ptr()),
                                         C.cast(C.c_void_p(x.data_ptr()), C.POINTER(C.c_double)), C.c_void_p(x.data_ptr()), None)
    assert st == 3                                                              # occupations must be host memory


def test_noalloc_argument_errors_need_no_gpu():
    lib = exx.load_library()
    occ = np.ones(4)
    p = occ.ctypes.data_as(C.POINTER(C.c_double))
    assert lib.exx_exchange_energy_noalloc(4, 8, 1.0, None, None, p, None, None) == 1
    assert lib.exx_exchange_energy_noalloc(exx.binding.EXX_NOALLOC_MAX_ORBITALS + 1, 8, 1.0, C.c_void_p(16), C.c_void_p(16), p, C.c_void_p(16), None) == 2
    assert b"exceeds" in lib.exx_noalloc_last_error()
