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

EXX_BLOCK_ACCUMULATE_RESIDENT, EXX_BLOCK_ACCUMULATE_STREAMED = 1, 2

EXPORTS = [
    "exx_plan_create", "exx_plan_create_general", "exx_apply", "exx_apply_async", "exx_apply_host", "exx_apply_pairs", "exx_apply_to", "exx_apply_to_cross", "exx_apply_complex", "exx_apply_block",
    "exx_get_pair_energies", "exx_get_block_energies", "exx_plan_release_staging",
    "exx_schedule_pairs", "exx_schedule_list", "exx_schedule_list_masked", "exx_schedule_list_block", "exx_round_robin_step",
    "exx_plan_transform_dims", "exx_plan_workspace_bytes", "exx_plan_launch_count", "exx_plan_device", "exx_plan_kernel_name",
    "exx_plan_set_batch", "exx_plan_set_profiling", "exx_plan_get_profile", "exx_plan_destroy", "exx_status_string", "exx_last_error", "exx_version", "exx_diag_fp64", "exx_diag_shfl",
    "exx_exchange_energy_noalloc", "exx_noalloc_last_error",
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
    lib.exx_plan_create_general.argtypes = [C.POINTER(C.c_void_p), _ip, C.c_double, _dp, C.c_int, C.c_void_p]
    lib.exx_plan_create_general.restype = C.c_int
    for name in ("exx_apply", "exx_apply_async", "exx_apply_host"):
        fn = getattr(lib, name)
        fn.argtypes = [C.c_void_p, C.c_int, C.c_void_p, _dp, C.c_void_p, C.c_void_p]
        fn.restype = C.c_int
    lib.exx_get_pair_energies.argtypes = [C.c_void_p, C.c_int, _dp]
    lib.exx_get_pair_energies.restype = C.c_int
    lib.exx_get_block_energies.argtypes = [C.c_void_p, C.c_int, C.c_int, _dp]
    lib.exx_get_block_energies.restype = C.c_int
    lib.exx_plan_release_staging.argtypes = [C.c_void_p]
    lib.exx_plan_release_staging.restype = C.c_int
    lib.exx_apply_pairs.argtypes = [C.c_void_p, C.c_int, C.c_void_p, _dp, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.exx_apply_pairs.restype = C.c_int
    lib.exx_apply_to.argtypes = [C.c_void_p, C.c_int, C.c_void_p, _dp, C.c_int, C.c_void_p, C.c_void_p]
    lib.exx_apply_to.restype = C.c_int
    lib.exx_apply_to_cross.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, _dp, C.c_int, C.c_void_p, C.c_void_p]
    lib.exx_apply_to_cross.restype = C.c_int
    lib.exx_apply_complex.argtypes = [C.c_void_p, C.c_int, C.c_void_p, _dp, C.c_void_p, C.c_void_p, C.POINTER(C.c_double)]
    lib.exx_apply_complex.restype = C.c_int
    lib.exx_apply_block.argtypes = [C.c_void_p, C.c_int, C.c_void_p, _dp, C.c_void_p, C.c_int, C.c_void_p, _dp, C.c_void_p, C.c_int,
                                    C.c_void_p]
    lib.exx_apply_block.restype = C.c_int
    lib.exx_schedule_list_masked.argtypes = [C.c_int, _dp, C.c_void_p, C.c_int, _ip, C.c_longlong, C.POINTER(C.c_longlong)]
    lib.exx_schedule_list_masked.restype = C.c_int
    lib.exx_schedule_list_block.argtypes = [C.c_int, _dp, C.c_int, _dp, C.c_int, _ip, C.c_longlong, C.POINTER(C.c_longlong)]
    lib.exx_schedule_list_block.restype = C.c_int
    lib.exx_round_robin_step.argtypes = [C.c_int, C.c_int, C.c_int, _ip, _ip, _ip]
    lib.exx_round_robin_step.restype = C.c_int
    lib.exx_plan_device.argtypes = [C.c_void_p]
    lib.exx_plan_device.restype = C.c_int
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
    lib.exx_diag_fp64.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
    lib.exx_diag_fp64.restype = C.c_int
    lib.exx_diag_shfl.argtypes = [C.c_void_p, _dp, _dp]
    lib.exx_diag_shfl.restype = C.c_int
    lib.exx_exchange_energy_noalloc.argtypes = [C.c_int, C.c_longlong, C.c_double, C.c_void_p, C.c_void_p, _dp, C.c_void_p, C.c_void_p]
    lib.exx_exchange_energy_noalloc.restype = C.c_int
    lib.exx_noalloc_last_error.argtypes = []
    lib.exx_noalloc_last_error.restype = C.c_char_p
    lib.exx_version.argtypes = []
    lib.exx_version.restype = C.c_char_p
    _lib = lib
    return lib


def exx_version() -> str:
    return load_library().exx_version().decode()


def exx_diag_fp64(stream: Optional[int] = None) -> dict:
    """Measured FP64 / shared-memory pipe rates of the current device (include/exx.h exx_diag_fp64)."""
    v = [C.c_double() for _ in range(4)]
    st = load_library().exx_diag_fp64(C.c_void_p(stream) if stream else None, *[C.byref(x) for x in v])
    if st:
        raise ExxError(st, "exx_diag_fp64")
    return {"dfma_tflops": v[0].value, "dadd_tera_inst_per_s": v[1].value, "lds_gbs": v[2].value, "fp64_lds_overlap": v[3].value}


def exx_diag_shfl(stream: Optional[int] = None) -> dict:
    """Measured warp-shuffle bandwidth and its overlap with shared-memory loads (include/exx.h exx_diag_shfl)."""
    v = [C.c_double() for _ in range(2)]
    st = load_library().exx_diag_shfl(C.c_void_p(stream) if stream else None, *[C.byref(x) for x in v])
    if st:
        raise ExxError(st, "exx_diag_shfl")
    return {"shfl_gbs": v[0].value, "shfl_lds_overlap": v[1].value}


EXX_NOALLOC_MAX_ORBITALS = 4096


def exx_exchange_energy_noalloc(psi, kpsi, occ, dV: float, ex_dev, stream: Optional[int] = None) -> None:
    """include/exx.h exx_exchange_energy_noalloc: E_x = 1/2 dV sum_i f_i <psi_i|K psi_i> into ex_dev (CUDA fp64, 1 element), with
    no allocation anywhere (static device scratch; calls that overlap on the GPU race on it).  Does not synchronise."""
    import torch
    for name, t in (("psi", psi), ("kpsi", kpsi), ("ex_dev", ex_dev)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise ValueError(f"{name} must be a contiguous CUDA float64 tensor")
    if psi.shape != kpsi.shape or psi.dim() < 2 or ex_dev.numel() < 1:
        raise ValueError("psi and kpsi must have the same shape (N, ...) and ex_dev at least one element")
    n_orb = int(psi.shape[0])
    occ = np.ascontiguousarray(np.asarray(occ, dtype=np.float64))
    if occ.ndim != 1 or occ.size != n_orb:
        raise ValueError(f"occ must hold one occupation per orbital ({n_orb})")
    lib = load_library()
    st = lib.exx_exchange_energy_noalloc(n_orb, psi[0].numel(), float(dV), C.c_void_p(psi.data_ptr()), C.c_void_p(kpsi.data_ptr()),
                                         occ.ctypes.data_as(_dp), C.c_void_p(ex_dev.data_ptr()), C.c_void_p(stream) if stream else None)
    if st:
        raise ExxError(st, lib.exx_noalloc_last_error().decode())


def exx_schedule_pairs(occ: Sequence[float]):
    """(n_pairs, n_transforms) an apply with these occupations performs -- host only, no GPU needed."""
    occ = np.ascontiguousarray(np.asarray(occ, dtype=np.float64))
    n_pairs, n_x = C.c_longlong(), C.c_longlong()
    st = load_library().exx_schedule_pairs(int(occ.size), occ.ctypes.data_as(_dp), C.byref(n_pairs), C.byref(n_x))
    if st:
        raise ExxError(st, "exx_schedule_pairs")
    return n_pairs.value, n_x.value


def _mask_array(mask, n_orb: int) -> np.ndarray:
    m = np.ascontiguousarray((np.asarray(mask) != 0).astype(np.uint8))
    if m.shape != (n_orb, n_orb):
        raise ValueError("pair mask must have shape (n_orb, n_orb)")
    return m


def exx_schedule_list(occ: Sequence[float], max_batch: int = 0, pair_mask=None):
    """int32 array [n_transforms][5] of {j, l, i, flags, batch} -- host only, no GPU needed (see include/exx.h).
    pair_mask: optional (n_orb, n_orb) symmetric mask of the pairs to solve (exx_schedule_list_masked)."""
    occ = np.ascontiguousarray(np.asarray(occ, dtype=np.float64))
    lib = load_library()
    n_x = C.c_longlong()
    m = _mask_array(pair_mask, occ.size) if pair_mask is not None else None
    mp = C.c_void_p(m.ctypes.data) if m is not None else None

    def call(buf, cap):
        st = lib.exx_schedule_list_masked(int(occ.size), occ.ctypes.data_as(_dp), mp, int(max_batch), buf, cap, C.byref(n_x))
        if st:
            raise ExxError(st, "exx_schedule_list")
    call(None, 0)
    out = np.zeros((n_x.value, 5), dtype=np.int32)
    if n_x.value:
        call(out.ctypes.data_as(_ip), n_x.value)
    return out


def exx_schedule_list_block(occ_res, occ_str: Sequence[float], n_res: Optional[int] = None, max_batch: int = 0):
    """Listing of the rectangular schedule of exx_apply_block (occ_res given) or exx_apply_to (occ_res None, n_res given)."""
    occ_str = np.ascontiguousarray(np.asarray(occ_str, dtype=np.float64))
    occ_r = None if occ_res is None else np.ascontiguousarray(np.asarray(occ_res, dtype=np.float64))
    n_res = int(occ_r.size) if occ_r is not None else int(n_res)
    lib = load_library()
    n_x = C.c_longlong()

    def call(buf, cap):
        st = lib.exx_schedule_list_block(n_res, occ_r.ctypes.data_as(_dp) if occ_r is not None else None, int(occ_str.size),
                                         occ_str.ctypes.data_as(_dp), int(max_batch), buf, cap, C.byref(n_x))
        if st:
            raise ExxError(st, "exx_schedule_list_block")
    call(None, 0)
    out = np.zeros((n_x.value, 5), dtype=np.int32)
    if n_x.value:
        call(out.ctypes.data_as(_ip), n_x.value)
    return out


def exx_round_robin_step(n_ranks: int, rank: int, step: int):
    """(send_to, recv_from, what) of step `step` of the round-robin block exchange (include/exx.h) -- host only."""
    a, b, w = C.c_int(), C.c_int(), C.c_int()
    st = load_library().exx_round_robin_step(int(n_ranks), int(rank), int(step), C.byref(a), C.byref(b), C.byref(w))
    if st:
        raise ExxError(st, "exx_round_robin_step")
    return a.value, b.value, w.value


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
            if self.bc == EXX_BC_FREE:
                want = self.dims[0] * self.dims[1] * self.dims[2]
            else:                                       # periodic: Fourier-space filter on the symmetric index range
                want = (self.dims[0] // 2 + 1) * (self.dims[1] // 2 + 1) * (self.dims[2] // 2 + 1)
            if self._kernel.size != want:
                raise ValueError(f"kernel table must have {want} entries for this boundary condition")
            kptr = self._kernel.ctypes.data_as(_dp)
        self._h = C.c_void_p()
        st = lib.exx_plan_create(C.byref(self._h), d, h, self.bc, kptr, self.max_orbitals,
                                 C.c_void_p(stream) if stream else None)
        if st:
            raise ExxError(st, lib.exx_last_error(None).decode())

    @classmethod
    def general(cls, dims, cell_volume, khat_full, max_orbitals=1, stream: Optional[int] = None):
        """Periodic cell of any shape (exx_plan_create_general): khat_full = K^[m1][m2][m3] on the full FFT index grid."""
        lib = load_library()
        self = cls.__new__(cls)
        self.dims = tuple(int(d) for d in dims)
        self.bc = EXX_BC_PERIODIC
        self.max_orbitals = int(max_orbitals)
        h = (float(cell_volume) / (self.dims[0] * self.dims[1] * self.dims[2])) ** (1.0 / 3.0)
        self.spacing = (h, h, h)
        self._kernel = np.ascontiguousarray(np.asarray(khat_full, dtype=np.float64))
        if self._kernel.shape != self.dims:
            raise ValueError(f"khat_full must have shape {self.dims}")
        self._h = C.c_void_p()
        st = lib.exx_plan_create_general(C.byref(self._h), (C.c_int * 3)(*self.dims), C.c_double(float(cell_volume)),
                                         self._kernel.ctypes.data_as(_dp), self.max_orbitals, C.c_void_p(stream) if stream else None)
        if st:
            raise ExxError(st, lib.exx_last_error(None).decode())
        return self

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

    # -- argument checks of the binding (shape / dtype / residency; the library re-checks pointers, alignment, overlap)
    def _check_dev(self, t, name, n_orb=None):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise ValueError(f"{name} must be a contiguous CUDA float64 tensor")
        if t.dim() != 4 or tuple(t.shape[1:]) != self.dims:
            raise ValueError(f"{name} must have shape (N, {self.dims[0]}, {self.dims[1]}, {self.dims[2]})")
        if n_orb is not None and t.shape[0] != n_orb:
            raise ValueError(f"{name} must hold {n_orb} orbitals")
        if t.device.index != self.device:
            raise ValueError(f"{name} lives on cuda:{t.device.index}, the plan on cuda:{self.device}")
        return t

    @staticmethod
    def _occ(occ, n_orb, name="occ"):
        occ = np.ascontiguousarray(np.asarray(occ, dtype=np.float64))
        if occ.ndim != 1 or occ.size != n_orb:
            raise ValueError(f"{name} must hold one occupation per orbital ({n_orb})")
        return occ

    @property
    def device(self) -> int:
        return int(load_library().exx_plan_device(self._h))

    # -- the hot path
    def apply(self, psi, occ, kpsi=None, pair_mask=None):
        """exx_apply (or exx_apply_pairs with a pair mask): returns (kpsi, E_x).  psi/kpsi are CUDA tensors whose
        data_ptr is handed to the library."""
        import torch
        self._check_dev(psi, "psi")
        n_orb = int(psi.shape[0])
        kpsi = torch.empty_like(psi) if kpsi is None else self._check_dev(kpsi, "kpsi", n_orb)
        occ = self._occ(occ, n_orb)
        ex = C.c_double()
        lib = load_library()
        if pair_mask is None:
            st = lib.exx_apply(self._h, n_orb, C.c_void_p(psi.data_ptr()), occ.ctypes.data_as(_dp), C.c_void_p(kpsi.data_ptr()),
                               C.cast(C.byref(ex), C.c_void_p))
        else:
            m = _mask_array(pair_mask, n_orb)
            st = lib.exx_apply_pairs(self._h, n_orb, C.c_void_p(psi.data_ptr()), occ.ctypes.data_as(_dp), C.c_void_p(m.ctypes.data),
                                     C.c_void_p(kpsi.data_ptr()), C.cast(C.byref(ex), C.c_void_p))
        self._check(st)
        self._last_n_orb = n_orb
        return kpsi, ex.value

    def apply_async(self, psi, occ, kpsi, ex_dev):
        """exx_apply_async: no synchronisation, E_x lands in the 1-element CUDA tensor ex_dev."""
        import torch
        self._check_dev(psi, "psi")
        n_orb = int(psi.shape[0])
        self._check_dev(kpsi, "kpsi", n_orb)
        if not (isinstance(ex_dev, torch.Tensor) and ex_dev.is_cuda and ex_dev.dtype == torch.float64 and ex_dev.numel() >= 1):
            raise ValueError("ex_dev must be a CUDA float64 tensor with at least one element")
        occ = self._occ(occ, n_orb)
        st = load_library().exx_apply_async(self._h, n_orb, C.c_void_p(psi.data_ptr()), occ.ctypes.data_as(_dp),
                                            C.c_void_p(kpsi.data_ptr()), C.c_void_p(ex_dev.data_ptr()))
        self._check(st)
        self._last_n_orb = n_orb

    def apply_host(self, psi_host: np.ndarray, occ, kpsi_host: Optional[np.ndarray] = None):
        """exx_apply_host: host buffers in, host buffers out (copies inside the library)."""
        if not (psi_host.dtype == np.float64 and psi_host.flags.c_contiguous and psi_host.ndim == 4 and tuple(psi_host.shape[1:]) == self.dims):
            raise ValueError("psi_host must be C-contiguous float64 of shape (N, n1, n2, n3)")
        if kpsi_host is None:
            kpsi_host = np.empty_like(psi_host)
        elif not (kpsi_host.dtype == np.float64 and kpsi_host.flags.c_contiguous and kpsi_host.shape == psi_host.shape and kpsi_host.flags.writeable):
            raise ValueError("kpsi_host must be writable C-contiguous float64 with the shape of psi_host")
        n_orb = int(psi_host.shape[0])
        occ = self._occ(occ, n_orb)
        ex = C.c_double()
        st = load_library().exx_apply_host(self._h, n_orb, C.c_void_p(psi_host.ctypes.data), occ.ctypes.data_as(_dp),
                                           C.c_void_p(kpsi_host.ctypes.data), C.cast(C.byref(ex), C.c_void_p))
        self._check(st)
        self._last_n_orb = n_orb
        return kpsi_host, ex.value

    def release_staging(self):
        self._check(load_library().exx_plan_release_staging(self._h))

    def apply_to(self, psi, occ, phi, kphi=None):
        """exx_apply_to: K (built from the occupied psi, occ) applied to the orbitals phi; returns kphi."""
        import torch
        self._check_dev(psi, "psi")
        self._check_dev(phi, "phi")
        kphi = torch.empty_like(phi) if kphi is None else self._check_dev(kphi, "kphi", int(phi.shape[0]))
        occ = self._occ(occ, int(psi.shape[0]))
        st = load_library().exx_apply_to(self._h, int(psi.shape[0]), C.c_void_p(psi.data_ptr()), occ.ctypes.data_as(_dp),
                                         int(phi.shape[0]), C.c_void_p(phi.data_ptr()), C.c_void_p(kphi.data_ptr()))
        self._check(st)
        return kphi

    def apply_to_cross(self, psi, chi, occ, phi, kphi=None):
        """exx_apply_to_cross: kphi_t = - sum_j f_j V[phi_t psi_j] chi_j."""
        import torch
        self._check_dev(psi, "psi")
        self._check_dev(chi, "chi", int(psi.shape[0]))
        self._check_dev(phi, "phi")
        kphi = torch.empty_like(phi) if kphi is None else self._check_dev(kphi, "kphi", int(phi.shape[0]))
        occ = self._occ(occ, int(psi.shape[0]))
        st = load_library().exx_apply_to_cross(self._h, int(psi.shape[0]), C.c_void_p(psi.data_ptr()), C.c_void_p(chi.data_ptr()),
                                               occ.ctypes.data_as(_dp), int(phi.shape[0]), C.c_void_p(phi.data_ptr()),
                                               C.c_void_p(kphi.data_ptr()))
        self._check(st)
        return kphi

    def apply_complex(self, psi_planar, occ, kpsi_planar=None, work=None):
        """exx_apply_complex: psi_planar = CUDA fp64 [2, N, n1, n2, n3] (real parts, imaginary parts); returns (kpsi_planar, E_x)."""
        import torch
        if not (isinstance(psi_planar, torch.Tensor) and psi_planar.dim() == 5 and psi_planar.shape[0] == 2):
            raise ValueError("psi_planar must have shape (2, N, n1, n2, n3)")
        n = int(psi_planar.shape[1])
        x = self._check_dev(psi_planar.view(2 * n, *self.dims), "psi_planar")
        kpsi_planar = torch.empty_like(psi_planar) if kpsi_planar is None else kpsi_planar
        k = self._check_dev(kpsi_planar.view(2 * n, *self.dims), "kpsi_planar", 2 * n)
        work = torch.empty(6 * n * x[0].numel(), dtype=torch.float64, device=psi_planar.device) if work is None else work
        if not (work.is_cuda and work.dtype == torch.float64 and work.is_contiguous() and work.numel() >= 6 * n * x[0].numel()):
            raise ValueError("work must be a contiguous CUDA float64 tensor of at least 6 N n1 n2 n3 elements")
        occ = self._occ(occ, n)
        ex = C.c_double()
        st = load_library().exx_apply_complex(self._h, n, C.c_void_p(x.data_ptr()), occ.ctypes.data_as(_dp), C.c_void_p(k.data_ptr()),
                                              C.c_void_p(work.data_ptr()), C.byref(ex))
        self._check(st)
        return kpsi_planar, ex.value

    def apply_block(self, psi_res, occ_res, kpsi_res, psi_str, occ_str, kpsi_str, flags=0):
        """exx_apply_block: all pairs between two disjoint blocks; returns the block's contribution to E_x."""
        self._check_dev(psi_res, "psi_res")
        self._check_dev(psi_str, "psi_str")
        self._check_dev(kpsi_res, "kpsi_res", int(psi_res.shape[0]))
        self._check_dev(kpsi_str, "kpsi_str", int(psi_str.shape[0]))
        occ_res = self._occ(occ_res, int(psi_res.shape[0]), "occ_res")
        occ_str = self._occ(occ_str, int(psi_str.shape[0]), "occ_str")
        ex = C.c_double()
        st = load_library().exx_apply_block(self._h, int(psi_res.shape[0]), C.c_void_p(psi_res.data_ptr()), occ_res.ctypes.data_as(_dp),
                                            C.c_void_p(kpsi_res.data_ptr()), int(psi_str.shape[0]), C.c_void_p(psi_str.data_ptr()),
                                            occ_str.ctypes.data_as(_dp), C.c_void_p(kpsi_str.data_ptr()), int(flags),
                                            C.cast(C.byref(ex), C.c_void_p))
        self._check(st)
        return ex.value

    def pair_energies(self, n_orb: Optional[int] = None) -> np.ndarray:
        """e_ij of the most recent square apply; n_orb defaults to that apply's orbital count (the library checks it)."""
        n_orb = int(n_orb if n_orb is not None else getattr(self, "_last_n_orb", 0))
        if n_orb < 1:
            raise ValueError("no apply has run on this plan")
        e = np.empty((n_orb, n_orb))
        self._check(load_library().exx_get_pair_energies(self._h, n_orb, e.ctypes.data_as(_dp)))
        return e

    def block_energies(self, n_res: int, n_str: int) -> np.ndarray:
        e = np.empty((int(n_res), int(n_str)))
        self._check(load_library().exx_get_block_energies(self._h, int(n_res), int(n_str), e.ctypes.data_as(_dp)))
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
