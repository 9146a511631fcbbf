"""ctypes binding of the CPU oracle (oracle/exx_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It shares no code with paper_1712_07973_b200.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as build_oracle

_lib = None

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_lp = C.POINTER(C.c_longlong)


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build_oracle())
        lib.exx_oracle_create.argtypes = [C.POINTER(C.c_void_p), _ip, _dp, C.c_int, _dp]
        lib.exx_oracle_destroy.argtypes = [C.c_void_p]
        lib.exx_oracle_destroy.restype = None
        lib.exx_oracle_fft1d.argtypes = [C.c_int, _dp, C.c_int]
        lib.exx_oracle_transform_dims.argtypes = [C.c_void_p, _ip]
        lib.exx_oracle_transform_dims.restype = None
        lib.exx_oracle_get_khat.argtypes = [C.c_void_p, _dp]
        lib.exx_oracle_poisson.argtypes = [C.c_void_p, _dp, _dp]
        lib.exx_oracle_apply.argtypes = [C.c_void_p, C.c_int, _dp, _dp, _dp, _dp, _dp, C.c_int]
        lib.exx_oracle_rows.argtypes = [C.c_void_p, C.c_int, _dp, _dp, C.c_int, _ip, _dp, _dp]
        lib.exx_oracle_pair_energies.argtypes = [C.c_void_p, C.c_int, _dp, C.c_int, _ip, _ip, _dp]
        lib.exx_oracle_realspace_kernel.argtypes = [C.c_void_p, _dp]
        lib.exx_oracle_poisson_direct.argtypes = [C.c_void_p, _dp, _dp]
        lib.exx_oracle_kpsi_points.argtypes = [C.c_void_p, C.c_int, _dp, _dp, C.c_int, _ip, _lp, _dp]
        lib.exx_oracle_apply_masked.argtypes = [C.c_void_p, C.c_int, _dp, _dp, C.c_void_p, _dp, _dp, _dp]
        lib.exx_oracle_apply_to.argtypes = [C.c_void_p, C.c_int, _dp, _dp, C.c_int, _dp, _dp]
        lib.exx_oracle_apply_block.argtypes = [C.c_void_p, C.c_int, _dp, _dp, _dp, C.c_int, _dp, _dp, _dp, _dp, _dp]
        lib.exx_oracle_set_periodic_filter.argtypes = [C.c_void_p, _dp]
        lib.exx_oracle_set_periodic_filter_full.argtypes = [C.c_void_p, _dp]
        lib.exx_oracle_poisson_direct_mixed.argtypes = [_ip, _dp, _ip, _dp, _dp, _dp]
        lib.exx_oracle_threads.argtypes = []
        _lib = lib
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def fft1d(x, sign=-1):
    """Unnormalised 1-D DFT by the oracle's own FFT (complex128 in, complex128 out)."""
    z = np.ascontiguousarray(np.asarray(x, dtype=np.complex128)).copy()
    buf = z.view(np.float64)
    rc = _load().exx_oracle_fft1d(int(z.size), _d(buf), int(sign))
    if rc:
        raise RuntimeError(f"exx_oracle_fft1d failed ({rc})")
    return z


class Oracle:
    """Plain CPU exact-exchange oracle for one grid / boundary condition / Green's function."""

    def __init__(self, dims, spacing, bc, kernel=None):
        """kernel: free BC -> real-space table g[n1][n2][n3]; periodic BC -> None (analytic 4 pi/|G|^2) or a
        Fourier-space filter table on the symmetric index range [n1/2+1][n2/2+1][n3/2+1]."""
        lib = _load()
        self.dims = tuple(int(d) for d in dims)
        self.spacing = tuple(float(h) for h in spacing)
        self.bc = {"periodic": 0, "free": 1}[bc] if isinstance(bc, str) else int(bc)
        self.M = self.dims[0] * self.dims[1] * self.dims[2]
        self.dV = self.spacing[0] * self.spacing[1] * self.spacing[2]
        d = (C.c_int * 3)(*self.dims)
        h = (C.c_double * 3)(*self.spacing)
        k = None
        filt = None
        if kernel is not None and self.bc == 1:
            k = _f64(kernel)
            if k.size != self.M:
                raise ValueError("kernel table must have n1*n2*n3 entries")
        elif kernel is not None:
            filt = _f64(kernel)
            if filt.size != (self.dims[0] // 2 + 1) * (self.dims[1] // 2 + 1) * (self.dims[2] // 2 + 1):
                raise ValueError("periodic filter table must have (n1/2+1)(n2/2+1)(n3/2+1) entries")
        self._h = C.c_void_p()
        rc = lib.exx_oracle_create(C.byref(self._h), d, h, self.bc, _d(k) if k is not None else None)
        if rc:
            raise RuntimeError(f"exx_oracle_create failed ({rc})")
        if filt is not None and lib.exx_oracle_set_periodic_filter(self._h, _d(filt)):
            raise RuntimeError("exx_oracle_set_periodic_filter failed")
        t = (C.c_int * 3)()
        lib.exx_oracle_transform_dims(self._h, t)
        self.tdims = tuple(t)

    @classmethod
    def general(cls, dims, cell_volume, khat_full):
        """Periodic cell of any shape: khat_full = K^ on the full FFT index grid [n1][n2][n3]; dV = cell_volume / M."""
        dims = tuple(int(d) for d in dims)
        h = (float(cell_volume) / (dims[0] * dims[1] * dims[2])) ** (1.0 / 3.0)
        o = cls(dims, (h, h, h), "periodic")
        t = _f64(khat_full)
        if t.shape != dims:
            raise ValueError("khat_full must have shape dims")
        if _load().exx_oracle_set_periodic_filter_full(o._h, _d(t)):
            raise RuntimeError("exx_oracle_set_periodic_filter_full failed")
        return o

    def close(self):
        if self._h:
            _load().exx_oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def khat(self):
        out = np.empty(self.tdims, dtype=np.complex128)
        rc = _load().exx_oracle_get_khat(self._h, _d(out.view(np.float64)))
        if rc:
            raise RuntimeError("exx_oracle_get_khat failed")
        return out

    def poisson(self, rho):
        rho = _f64(rho).reshape(self.dims)
        v = np.empty(self.dims)
        rc = _load().exx_oracle_poisson(self._h, _d(rho), _d(v))
        if rc:
            raise RuntimeError("exx_oracle_poisson failed")
        return v

    def poisson_direct(self, rho):
        rho = _f64(rho).reshape(self.dims)
        v = np.empty(self.dims)
        rc = _load().exx_oracle_poisson_direct(self._h, _d(rho), _d(v))
        if rc:
            raise RuntimeError("exx_oracle_poisson_direct failed")
        return v

    def realspace_kernel(self):
        g = np.empty(self.dims)
        rc = _load().exx_oracle_realspace_kernel(self._h, _d(g))
        if rc:
            raise RuntimeError("exx_oracle_realspace_kernel failed")
        return g

    def apply(self, psi, occ, symmetric=False):
        """Returns (kpsi[N,n1,n2,n3], E_x, e_pair[N,N])."""
        psi = _f64(psi)
        n_orb = psi.shape[0]
        psi = psi.reshape(n_orb, self.M)
        occ = _f64(occ)
        kpsi = np.empty_like(psi)
        ex = C.c_double()
        e = np.empty((n_orb, n_orb))
        rc = _load().exx_oracle_apply(self._h, n_orb, _d(psi), _d(occ), _d(kpsi), C.byref(ex), _d(e),
                                      1 if symmetric else 0)
        if rc:
            raise RuntimeError(f"exx_oracle_apply failed ({rc})")
        return kpsi.reshape((n_orb,) + self.dims), ex.value, e

    def apply_masked(self, psi, occ, mask):
        """As apply() with the ordered pairs whose mask entry is 0 left out.  Returns (kpsi, E_x, e_pair)."""
        psi = _f64(psi)
        n_orb = psi.shape[0]
        psi = psi.reshape(n_orb, self.M)
        occ = _f64(occ)
        m = np.ascontiguousarray((np.asarray(mask) != 0).astype(np.uint8))
        if m.shape != (n_orb, n_orb):
            raise ValueError("mask must have shape (n_orb, n_orb)")
        kpsi = np.empty_like(psi)
        ex = C.c_double()
        e = np.empty((n_orb, n_orb))
        rc = _load().exx_oracle_apply_masked(self._h, n_orb, _d(psi), _d(occ), C.c_void_p(m.ctypes.data), _d(kpsi), C.byref(ex), _d(e))
        if rc:
            raise RuntimeError(f"exx_oracle_apply_masked failed ({rc})")
        return kpsi.reshape((n_orb,) + self.dims), ex.value, e

    def apply_to(self, psi, occ, phi):
        """K of the occupied set (psi, occ) applied to phi: returns kphi[n_tgt, n1, n2, n3]."""
        psi = _f64(psi)
        phi = _f64(phi)
        n_occ, n_tgt = psi.shape[0], phi.shape[0]
        psi = psi.reshape(n_occ, self.M)
        phi = phi.reshape(n_tgt, self.M)
        occ = _f64(occ)
        kphi = np.empty_like(phi)
        rc = _load().exx_oracle_apply_to(self._h, n_occ, _d(psi), _d(occ), n_tgt, _d(phi), _d(kphi))
        if rc:
            raise RuntimeError(f"exx_oracle_apply_to failed ({rc})")
        return kphi.reshape((n_tgt,) + self.dims)

    def apply_to_cross(self, psi, chi, occ, phi):
        """K phi_t = - sum_j f_j V[phi_t psi_j] chi_j: the potential of the co-density (phi_t, psi_j) multiplied by a partner
        orbital chi_j (chi = psi gives apply_to).  Plain numpy loop over the pairs on top of the pinned Poisson solve."""
        psi, chi, phi = (_f64(x).reshape((-1,) + self.dims) for x in (psi, chi, phi))
        occ = _f64(occ)
        out = np.zeros_like(phi)
        for t in range(phi.shape[0]):
            for j in range(psi.shape[0]):
                if occ[j] != 0.0:
                    out[t] -= occ[j] * self.poisson(phi[t] * psi[j]) * chi[j]
        return out

    def apply_complex(self, psi, occ):
        """Complex orbitals (Eq. 8 with its conjugate; reading A26), the definition over all ordered
        pairs:  rho = conj(psi_j) psi_i,  V = Poisson(Re rho) + i Poisson(Im rho)  (the Green's function is real),
        K psi_i -= f_j V psi_j,  E_x -= 1/2 f_i f_j dV sum_r conj(rho) V.  Returns (K psi complex, E_x)."""
        psi = np.ascontiguousarray(np.asarray(psi, dtype=np.complex128)).reshape((-1,) + self.dims)
        occ = _f64(occ)
        n = psi.shape[0]
        kpsi = np.zeros_like(psi)
        ex = 0.0
        for i in range(n):
            for j in range(n):
                if occ[i] == 0.0 and occ[j] == 0.0:
                    continue
                rho = np.conj(psi[j]) * psi[i]
                v = self.poisson(rho.real) + 1j * self.poisson(rho.imag)
                kpsi[i] -= occ[j] * v * psi[j]
                ex -= 0.5 * occ[i] * occ[j] * self.dV * float(np.sum(np.conj(rho) * v).real)
        return kpsi, ex

    def apply_block(self, psi_a, occ_a, psi_b, occ_b):
        """All pairs between two disjoint blocks: returns (ka, kb, ex, e_block[n_a, n_b])."""
        psi_a = _f64(psi_a)
        psi_b = _f64(psi_b)
        n_a, n_b = psi_a.shape[0], psi_b.shape[0]
        psi_a = psi_a.reshape(n_a, self.M)
        psi_b = psi_b.reshape(n_b, self.M)
        occ_a, occ_b = _f64(occ_a), _f64(occ_b)
        ka, kb = np.empty_like(psi_a), np.empty_like(psi_b)
        ex = C.c_double()
        e = np.empty((n_a, n_b))
        rc = _load().exx_oracle_apply_block(self._h, n_a, _d(psi_a), _d(occ_a), _d(ka), n_b, _d(psi_b), _d(occ_b), _d(kb),
                                            C.byref(ex), _d(e))
        if rc:
            raise RuntimeError(f"exx_oracle_apply_block failed ({rc})")
        return ka.reshape((n_a,) + self.dims), kb.reshape((n_b,) + self.dims), ex.value, e

    def rows(self, psi, occ, rows):
        """Complete rows K psi_i for listed i: returns (kpsi_rows[len(rows),n1,n2,n3], e_rows[len(rows),N])."""
        psi = _f64(psi)
        n_orb = psi.shape[0]
        psi = psi.reshape(n_orb, self.M)
        occ = _f64(occ)
        rows = np.ascontiguousarray(np.asarray(rows, dtype=np.int32))
        out = np.empty((rows.size, self.M))
        e = np.empty((rows.size, n_orb))
        rc = _load().exx_oracle_rows(self._h, n_orb, _d(psi), _d(occ), int(rows.size),
                                     rows.ctypes.data_as(_ip), _d(out), _d(e))
        if rc:
            raise RuntimeError(f"exx_oracle_rows failed ({rc})")
        return out.reshape((rows.size,) + self.dims), e

    def pair_energies(self, psi, pairs):
        psi = _f64(psi)
        n_orb = psi.shape[0]
        psi = psi.reshape(n_orb, self.M)
        pairs = np.asarray(pairs, dtype=np.int32).reshape(-1, 2)
        pi = np.ascontiguousarray(pairs[:, 0])
        pj = np.ascontiguousarray(pairs[:, 1])
        e = np.empty(pairs.shape[0])
        rc = _load().exx_oracle_pair_energies(self._h, n_orb, _d(psi), int(e.size), pi.ctypes.data_as(_ip),
                                              pj.ctypes.data_as(_ip), _d(e))
        if rc:
            raise RuntimeError(f"exx_oracle_pair_energies failed ({rc})")
        return e

    def kpsi_points(self, psi, occ, orbs, points):
        """Sampled K psi entries by direct real-space summation (no FFT in the convolution)."""
        psi = _f64(psi)
        n_orb = psi.shape[0]
        psi = psi.reshape(n_orb, self.M)
        occ = _f64(occ)
        orbs = np.ascontiguousarray(np.asarray(orbs, dtype=np.int32))
        points = np.ascontiguousarray(np.asarray(points, dtype=np.int64))
        out = np.empty(orbs.size)
        rc = _load().exx_oracle_kpsi_points(self._h, n_orb, _d(psi), _d(occ), int(orbs.size),
                                            orbs.ctypes.data_as(_ip), points.ctypes.data_as(_lp), _d(out))
        if rc:
            raise RuntimeError(f"exx_oracle_kpsi_points failed ({rc})")
        return out


def poisson_direct_mixed(dims, spacing, periodic, table, rho):
    """Mixed boundary conditions by the O(M^2) definition (exx_oracle_poisson_direct_mixed): periodic[a] truthy = axis a
    is periodic (the table holds one full period there), else isolated."""
    dims = tuple(int(d) for d in dims)
    rho = _f64(rho).reshape(dims)
    table = _f64(table).reshape(dims)
    v = np.empty(dims)
    d = np.asarray(dims, dtype=np.int32)
    h = np.asarray(spacing, dtype=np.float64)
    per = np.asarray([1 if x else 0 for x in periodic], dtype=np.int32)
    rc = _load().exx_oracle_poisson_direct_mixed(d.ctypes.data_as(_ip), _d(h), per.ctypes.data_as(_ip), _d(table), _d(rho), _d(v))
    if rc:
        raise RuntimeError("exx_oracle_poisson_direct_mixed failed")
    return v


def threads_used() -> int:
    return int(_load().exx_oracle_threads())
