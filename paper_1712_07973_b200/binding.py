"""ctypes binding of libexx_b200.so -- same names as include/exx.h, marshalling only.

There is no fallback of any kind: if the shared library cannot be built/loaded, or no CUDA device is usable,
the calls raise.  Nothing here imports the CPU oracle.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from .build import LIB, build

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)

EXX_BC_PERIODIC, EXX_BC_FREE = 0, 1
_STATUS = ["EXX_OK", "EXX_ERR_INVALID_ARG", "EXX_ERR_UNSUPPORTED_SIZE", "EXX_ERR_BAD_POINTER", "EXX_ERR_ALLOC",
           "EXX_ERR_CUDA", "EXX_ERR_INTERNAL"]

EXPORTS = [
    "exx_plan_create", "exx_apply", "exx_apply_async", "exx_apply_host", "exx_get_pair_energies",
    "exx_schedule_pairs", "exx_schedule_list", "exx_plan_transform_dims", "exx_plan_workspace_bytes", "exx_plan_launch_count", "exx_plan_kernel_name",
    "exx_plan_set_batch", "exx_plan_set_profiling", "exx_plan_get_profile", "exx_plan_destroy", "exx_status_string", "exx_last_error", "exx_version",
]

_lib = None


class ExxError(RuntimeError):
    def __init__(self, status: int, detail: str):
        name = _STATUS[status] if 0 <= status < len(_STATUS) else f"status {status}"
        super().__init__(f"{name}: {detail}" if detail else name)
        self.status = status
        self.status_name = name


def library_path() -> str:
    return LIB


def load_library():
    """Build (if stale) and load libexx_b200.so.  Raises if the CUDA extension is missing."""
    global _lib
    if _lib is not None:
        return _lib
    path = build() if os.environ.get("EXX_NO_BUILD") != "1" else LIB
    if not os.path.exists(path):
        raise ExxError(5, f"CUDA extension {path} is missing; run paper_1712_07973_b200.build()")
    lib = C.CDLL(path)
    lib.exx_plan_create.argtypes = [C.POINTER(C.c_void_p), _ip, _dp, C.c_int, _dp, C.c_int, C.c_void_p]
    lib.exx_plan_create.restype = C.c_int
    for name in ("exx_apply", "exx_apply_async", "exx_apply_host"):
        fn = getattr(lib, name)
        fn.argtypes = [C.c_void_p, C.c_int, C.c_void_p, _dp, C.c_void_p, C.c_void_p]
        fn.restype = C.c_int
    lib.exx_get_pair_energies.argtypes = [C.c_void_p, _dp]
    lib.exx_get_pair_energies.restype = C.c_int
    lib.exx_schedule_pairs.argtypes = [C.c_int, _dp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    lib.exx_schedule_pairs.restype = C.c_int
    lib.exx_schedule_list.argtypes = [C.c_int, _dp, C.c_int, _ip, C.c_longlong, C.POINTER(C.c_longlong)]
    lib.exx_schedule_list.restype = C.c_int
    lib.exx_plan_transform_dims.argtypes = [C.c_void_p, _ip]
    lib.exx_plan_transform_dims.restype = C.c_int
    lib.exx_plan_workspace_bytes.argtypes = [C.c_void_p]
    lib.exx_plan_workspace_bytes.restype = C.c_size_t
    lib.exx_plan_kernel_name.argtypes = [C.c_void_p, C.c_int]
    lib.exx_plan_kernel_name.restype = C.c_char_p
    lib.exx_plan_launch_count.argtypes = [C.c_void_p]
    lib.exx_plan_launch_count.restype = C.c_longlong
    lib.exx_plan_set_batch.argtypes = [C.c_void_p, C.c_int]
    lib.exx_plan_set_batch.restype = C.c_int
    lib.exx_plan_set_profiling.argtypes = [C.c_void_p, C.c_int]
    lib.exx_plan_set_profiling.restype = C.c_int
    lib.exx_plan_get_profile.argtypes = [C.c_void_p, _dp, C.POINTER(C.c_longlong)]
    lib.exx_plan_get_profile.restype = C.c_int
    lib.exx_plan_destroy.argtypes = [C.c_void_p]
    lib.exx_plan_destroy.restype = C.c_int
    lib.exx_status_string.argtypes = [C.c_int]
    lib.exx_status_string.restype = C.c_char_p
    lib.exx_last_error.argtypes = [C.c_void_p]
    lib.exx_last_error.restype = C.c_char_p
    lib.exx_version.argtypes = []
    lib.exx_version.restype = C.c_char_p
    _lib = lib
    return lib


def exx_version() -> str:
    return load_library().exx_version().decode()


def exx_schedule_pairs(occ: Sequence[float]):
    """(n_pairs, n_transforms) an apply with these occupations performs -- host only, no GPU needed."""
    occ = np.ascontiguousarray(np.asarray(occ, dtype=np.float64))
    n_pairs, n_x = C.c_longlong(), C.c_longlong()
    st = load_library().exx_schedule_pairs(int(occ.size), occ.ctypes.data_as(_dp), C.byref(n_pairs), C.byref(n_x))
    if st:
        raise ExxError(st, "exx_schedule_pairs")
    return n_pairs.value, n_x.value


def exx_schedule_list(occ: Sequence[float], max_batch: int = 0):
    """int32 array [n_transforms][5] of {j, l, i, flags, batch} -- host only, no GPU needed (see include/exx.h)."""
    occ = np.ascontiguousarray(np.asarray(occ, dtype=np.float64))
    lib = load_library()
    n_x = C.c_longlong()
    st = lib.exx_schedule_list(int(occ.size), occ.ctypes.data_as(_dp), int(max_batch), None, 0, C.byref(n_x))
    if st:
        raise ExxError(st, "exx_schedule_list")
    out = np.zeros((n_x.value, 5), dtype=np.int32)
    if n_x.value:
        st = lib.exx_schedule_list(int(occ.size), occ.ctypes.data_as(_dp), int(max_batch), out.ctypes.data_as(_ip), n_x.value, C.byref(n_x))
        if st:
            raise ExxError(st, "exx_schedule_list")
    return out


class ExxPlan:
    """Owns an exx_plan*.  Tensors passed to apply() must be CUDA fp64, contiguous, shape (N, n1, n2, n3)."""

    def __init__(self, dims, spacing, bc, kernel=None, max_orbitals=1, stream: Optional[int] = None):
        lib = load_library()
        self.dims = tuple(int(d) for d in dims)
        self.spacing = tuple(float(h) for h in spacing)
        self.bc = {"periodic": EXX_BC_PERIODIC, "free": EXX_BC_FREE}[bc] if isinstance(bc, str) else int(bc)
        self.max_orbitals = int(max_orbitals)
        d = (C.c_int * 3)(*self.dims)
        h = (C.c_double * 3)(*self.spacing)
        kptr = None
        if kernel is not None:
            self._kernel = np.ascontiguousarray(np.asarray(kernel, dtype=np.float64))
            if self._kernel.size != self.dims[0] * self.dims[1] * self.dims[2]:
                raise ValueError("kernel table must have n1*n2*n3 entries")
            kptr = self._kernel.ctypes.data_as(_dp)
        self._h = C.c_void_p()
        st = lib.exx_plan_create(C.byref(self._h), d, h, self.bc, kptr, self.max_orbitals,
                                 C.c_void_p(stream) if stream else None)
        if st:
            raise ExxError(st, lib.exx_last_error(None).decode())

    # -- helpers
    def _check(self, st):
        if st:
            raise ExxError(st, load_library().exx_last_error(self._h).decode())

    @property
    def handle(self):
        return self._h

    def transform_dims(self):
        t = (C.c_int * 3)()
        self._check(load_library().exx_plan_transform_dims(self._h, t))
        return tuple(t)

    def workspace_bytes(self) -> int:
        return int(load_library().exx_plan_workspace_bytes(self._h))

    def launch_count(self) -> int:
        return int(load_library().exx_plan_launch_count(self._h))

    def kernel_name(self, pass_index: int) -> str:
        """Kernel this plan dispatches to for pass 0 (A), 1 (B), 2 (C)."""
        return load_library().exx_plan_kernel_name(self._h, int(pass_index)).decode()

    def set_batch(self, n: int):
        self._check(load_library().exx_plan_set_batch(self._h, int(n)))

    def set_profiling(self, enable: bool):
        self._check(load_library().exx_plan_set_profiling(self._h, 1 if enable else 0))

    def get_profile(self):
        """Per-pass (A, B, C, reduce) summed device milliseconds and launch counts of the most recent apply."""
        ms = (C.c_double * 4)()
        n = (C.c_longlong * 4)()
        self._check(load_library().exx_plan_get_profile(self._h, ms, n))
        return list(ms), list(n)

    # -- the hot path
    def apply(self, psi, occ, kpsi=None):
        """exx_apply: returns (kpsi, E_x).  psi/kpsi are CUDA tensors (data_ptr is handed to the library)."""
        import torch
        if not (psi.is_cuda and psi.dtype == torch.float64 and psi.is_contiguous()):
            raise ValueError("psi must be a contiguous CUDA float64 tensor")
        if tuple(psi.shape[1:]) != self.dims:
            raise ValueError("psi grid shape does not match the plan")
        if kpsi is None:
            kpsi = torch.empty_like(psi)
        occ = np.ascontiguousarray(np.asarray(occ, dtype=np.float64))
        ex = C.c_double()
        st = load_library().exx_apply(self._h, int(psi.shape[0]), C.c_void_p(psi.data_ptr()), occ.ctypes.data_as(_dp),
                                      C.c_void_p(kpsi.data_ptr()), C.cast(C.byref(ex), C.c_void_p))
        self._check(st)
        return kpsi, ex.value

    def apply_async(self, psi, occ, kpsi, ex_dev):
        """exx_apply_async: no synchronisation, E_x lands in the 1-element CUDA tensor ex_dev."""
        occ = np.ascontiguousarray(np.asarray(occ, dtype=np.float64))
        st = load_library().exx_apply_async(self._h, int(psi.shape[0]), C.c_void_p(psi.data_ptr()), occ.ctypes.data_as(_dp),
                                            C.c_void_p(kpsi.data_ptr()), C.c_void_p(ex_dev.data_ptr()))
        self._check(st)

    def apply_host(self, psi_host: np.ndarray, occ, kpsi_host: Optional[np.ndarray] = None):
        """exx_apply_host: host buffers in, host buffers out (copies inside the library)."""
        if not (psi_host.dtype == np.float64 and psi_host.flags.c_contiguous):
            raise ValueError("psi_host must be C-contiguous float64")
        if kpsi_host is None:
            kpsi_host = np.empty_like(psi_host)
        occ = np.ascontiguousarray(np.asarray(occ, dtype=np.float64))
        ex = C.c_double()
        st = load_library().exx_apply_host(self._h, int(psi_host.shape[0]), C.c_void_p(psi_host.ctypes.data),
                                           occ.ctypes.data_as(_dp), C.c_void_p(kpsi_host.ctypes.data),
                                           C.cast(C.byref(ex), C.c_void_p))
        self._check(st)
        return kpsi_host, ex.value

    def pair_energies(self, n_orb: int) -> np.ndarray:
        e = np.empty((n_orb, n_orb))
        self._check(load_library().exx_get_pair_energies(self._h, e.ctypes.data_as(_dp)))
        return e

    def destroy(self):
        if getattr(self, "_h", None):
            load_library().exx_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# Function-style aliases with the names of include/exx.h.
def exx_plan_create(dims, spacing, bc, kernel=None, max_orbitals=1, stream=None) -> ExxPlan:
    return ExxPlan(dims, spacing, bc, kernel, max_orbitals, stream)


def exx_apply(plan: ExxPlan, psi, occ, kpsi=None):
    return plan.apply(psi, occ, kpsi)


def exx_plan_destroy(plan: ExxPlan):
    plan.destroy()
