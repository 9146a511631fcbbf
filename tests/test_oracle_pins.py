"""Pins of the CPU oracle against things other than itself.  CPU only.

Each pin is chosen so that a plausible mistake in oracle/exx_oracle.c (a dropped factor, a wrong sign or index,
a transposed axis, a wrong embedding) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
from scipy.special import erf

from oracle import Oracle, fft1d
from workloads import cell_average_inverse_r, free_kernel_table, make_workload, small_spec

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rng(seed):
    return np.random.default_rng(seed)


# ------------------------------------------------------------------ P1: the oracle's own FFT
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8, 12, 30, 32, 96, 192, 256])
def test_p1_fft_vs_direct_dft(n):
    x = _rng(n).standard_normal(n) + 1j * _rng(n + 1000).standard_normal(n)
    k = np.arange(n)
    # direct O(n^2) DFT with exactly reduced phases
    phase = (np.outer(k, k) % n) / n
    F = np.exp(-2j * np.pi * phase)
    ref = F @ x
    got = fft1d(x, -1)
    assert np.max(np.abs(got - ref)) <= 1e-13 * np.max(np.abs(ref)) * max(1, math.log2(n + 1))
    # inverse sign and round trip
    back = fft1d(got, +1) / n
    assert np.max(np.abs(back - x)) <= 1e-13
    # Parseval
    assert abs(np.sum(np.abs(got) ** 2) - n * np.sum(np.abs(x) ** 2)) <= 1e-12 * n * np.sum(np.abs(x) ** 2)
    # delta -> constant, shifted delta -> pure phase with the forward sign e^{-i...}
    d = np.zeros(n, dtype=complex)
    d[0] = 1.0
    assert np.max(np.abs(fft1d(d, -1) - 1.0)) <= 1e-15
    if n > 2:
        d = np.zeros(n, dtype=complex)
        d[1] = 1.0
        assert np.max(np.abs(fft1d(d, -1) - np.exp(-2j * np.pi * k / n))) <= 2e-15 * n


@pytest.mark.parametrize("n", [32, 96, 192, 256])
def test_p1_fft_vs_library(n):
    x = _rng(7 * n).standard_normal(n) + 1j * _rng(7 * n + 1).standard_normal(n)
    assert np.max(np.abs(fft1d(x, -1) - np.fft.fft(x))) <= 2e-13 * np.max(np.abs(x)) * math.sqrt(n)


# ------------------------------------------------------------------ P2: free BC vs brute-force O(M^2)
def _brute_free(rho, g, dV):
    n1, n2, n3 = rho.shape
    ia = np.abs(np.arange(n1)[:, None] - np.arange(n1)[None, :])
    ib = np.abs(np.arange(n2)[:, None] - np.arange(n2)[None, :])
    ic = np.abs(np.arange(n3)[:, None] - np.arange(n3)[None, :])
    v = np.zeros_like(rho)
    for a in range(n1):
        for b in range(n2):
            for c in range(n3):
                # V(r) = dV sum_r' g(|r - r'|) rho(r')
                v[a, b, c] = dV * np.sum(g[ia[a][:, None, None], ib[b][None, :, None], ic[c][None, None, :]] * rho)
    return v


@pytest.mark.parametrize("dims,h", [((4, 4, 4), (0.5, 0.5, 0.5)), ((5, 5, 5), (0.4, 0.4, 0.4)),
                                    ((4, 6, 8), (0.3, 0.45, 0.25)), ((6, 3, 2), (0.7, 0.2, 0.5))])
def test_p2_free_bruteforce(dims, h):
    g = free_kernel_table(dims, h)
    o = Oracle(dims, h, "free", g)
    rho = _rng(11).standard_normal(dims)
    v = o.poisson(rho)
    ref = _brute_free(rho, g, h[0] * h[1] * h[2])
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(v - ref)) <= 1e-13 * scale
    # the oracle's own direct-sum routine agrees too (it is what sampled parity at full size uses)
    assert np.max(np.abs(o.poisson_direct(rho) - ref)) <= 1e-13 * scale


def test_p2_free_table_is_data():
    """The free-BC kernel is host data: an arbitrary (non-Coulomb, asymmetric-in-axes) table must work the same."""
    dims, h = (3, 4, 5), (0.5, 0.6, 0.7)
    g = _rng(5).standard_normal(dims)
    o = Oracle(dims, h, "free", g)
    rho = _rng(6).standard_normal(dims)
    ref = _brute_free(rho, g, h[0] * h[1] * h[2])
    assert np.max(np.abs(o.poisson(rho) - ref)) <= 1e-13 * np.max(np.abs(ref))


# ------------------------------------------------------------------ P3: periodic vs brute-force
def _khat_periodic(dims, h):
    ks = []
    for n, hh in zip(dims, h):
        m = np.arange(n)
        m = np.where(2 * m <= n, m, m - n)
        ks.append(2 * np.pi * m / (n * hh))
    g2 = ks[0][:, None, None] ** 2 + ks[1][None, :, None] ** 2 + ks[2][None, None, :] ** 2
    g2[0, 0, 0] = 1.0
    k = 4 * np.pi / g2
    k[0, 0, 0] = 0.0
    return k


def _brute_periodic(rho, dims, h):
    n1, n2, n3 = dims
    khat = _khat_periodic(dims, h)
    M = n1 * n2 * n3
    # real-space kernel by direct O(M^2) sum: g_per(r) = (1/M) sum_G K^(G) e^{iG.r}
    e1 = np.exp(2j * np.pi * np.outer(np.arange(n1), np.arange(n1)) / n1)
    e2 = np.exp(2j * np.pi * np.outer(np.arange(n2), np.arange(n2)) / n2)
    e3 = np.exp(2j * np.pi * np.outer(np.arange(n3), np.arange(n3)) / n3)
    gper = np.einsum("abc,ax,by,cz->xyz", khat, e1, e2, e3).real / M
    v = np.zeros(dims)
    A, B, Cc = np.arange(n1), np.arange(n2), np.arange(n3)
    for a in range(n1):
        for b in range(n2):
            for c in range(n3):
                v[a, b, c] = np.sum(gper[(a - A)[:, None, None] % n1, (b - B)[None, :, None] % n2,
                                         (c - Cc)[None, None, :] % n3] * rho)
    return v, gper


@pytest.mark.parametrize("dims,h", [((6, 6, 6), (0.4, 0.4, 0.4)), ((4, 6, 3), (0.3, 0.5, 0.7)),
                                    ((12, 2, 5), (0.25, 0.6, 0.35))])
def test_p3_periodic_bruteforce(dims, h):
    o = Oracle(dims, h, "periodic")
    rho = _rng(21).standard_normal(dims)
    v = o.poisson(rho)
    ref, gper = _brute_periodic(rho, dims, h)
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(v - ref)) <= 1e-12 * scale
    assert abs(np.sum(v)) <= 1e-12 * scale * rho.size          # K^(0)=0 -> zero-mean potential (A6)
    assert np.max(np.abs(o.realspace_kernel() - gper)) <= 1e-12 * np.max(np.abs(gper))
    assert np.max(np.abs(o.poisson_direct(rho) - ref)) <= 1e-12 * scale


# ------------------------------------------------------------------ P4: plane wave closed form
@pytest.mark.parametrize("dims,h,m", [((12, 12, 12), (0.4, 0.4, 0.4), (1, 0, 0)), ((8, 12, 6), (0.3, 0.5, 0.45), (1, -2, 1)),
                                      ((32, 32, 32), (0.4, 0.4, 0.4), (3, 5, -7))])
def test_p4_plane_wave(dims, h, m):
    o = Oracle(dims, h, "periodic")
    kvec = [2 * np.pi * mi / (n * hh) for mi, n, hh in zip(m, dims, h)]
    x = [np.arange(n) * hh for n, hh in zip(dims, h)]
    phase = kvec[0] * x[0][:, None, None] + kvec[1] * x[1][None, :, None] + kvec[2] * x[2][None, None, :]
    rho = np.cos(phase)
    k2 = sum(k * k for k in kvec)
    ref = 4 * np.pi / k2 * rho
    assert np.max(np.abs(o.poisson(rho) - ref)) <= 1e-13 * np.max(np.abs(ref))
    # a sine with the same k checks the sign convention of the imaginary parts
    rho_s = np.sin(phase)
    assert np.max(np.abs(o.poisson(rho_s) - 4 * np.pi / k2 * rho_s)) <= 1e-13 * np.max(np.abs(ref))


# ------------------------------------------------------------------ P5: whole path, N=2, closed form
def test_p5_two_orbital_closed_form():
    dims, h, m = (12, 12, 12), (0.4, 0.35, 0.5), (1, 2, 0)
    o = Oracle(dims, h, "periodic")
    vol = np.prod([n * hh for n, hh in zip(dims, h)])
    kvec = [2 * np.pi * mi / (n * hh) for mi, n, hh in zip(m, dims, h)]
    k2 = sum(k * k for k in kvec)
    x = [np.arange(n) * hh for n, hh in zip(dims, h)]
    cosk = np.cos(kvec[0] * x[0][:, None, None] + kvec[1] * x[1][None, :, None] + kvec[2] * x[2][None, None, :])
    psi1 = np.full(dims, vol ** -0.5)
    psi2 = math.sqrt(2.0 / vol) * cosk
    f1, f2 = 2.0, 1.25
    kpsi, ex, e = o.apply(np.stack([psi1, psi2]), [f1, f2])
    e11, e12, e22 = 0.0, 4 * np.pi / (k2 * vol), np.pi / (2 * k2 * vol)
    assert abs(e[0, 0] - e11) <= 1e-15
    assert abs(e[0, 1] - e12) <= 1e-13 * e12 and abs(e[1, 0] - e12) <= 1e-13 * e12
    assert abs(e[1, 1] - e22) <= 1e-13 * e22
    ex_ref = -0.5 * (2 * f1 * f2 * e12 + f2 * f2 * e22)
    assert abs(ex - ex_ref) <= 1e-13 * abs(ex_ref)
    # K psi_1 = -f2 V12 psi2 (V11 = 0);  V12 = (4 pi/k^2) sqrt(2)/vol cos(k.r)
    v12 = 4 * np.pi / k2 * math.sqrt(2.0) / vol * cosk
    ref1 = -f2 * v12 * psi2
    assert np.max(np.abs(kpsi[0] - ref1)) <= 1e-13 * np.max(np.abs(ref1))
    # K psi_2 = -f1 V12 psi1 - f2 V22 psi2;  rho22 = (1 + cos 2k.r)/vol -> V22 = (4 pi/(4 k^2)) cos(2k.r)/vol
    cos2k = 2 * cosk * cosk - 1
    v22 = np.pi / k2 * cos2k / vol
    ref2 = -f1 * v12 * psi1 - f2 * v22 * psi2
    assert np.max(np.abs(kpsi[1] - ref2)) <= 1e-13 * np.max(np.abs(ref2))


# ------------------------------------------------------------------ P6: Gaussian, free BC -> erf(r/(sqrt2 s))/r
def _gaussian_free_errors(n, h, sigma):
    dims, hs = (n, n, n), (h, h, h)
    g = free_kernel_table(dims, hs)
    o = Oracle(dims, hs, "free", g)
    c = 0.5 * (n - 1) * h
    x = np.arange(n) * h - c
    r2 = x[:, None, None] ** 2 + x[None, :, None] ** 2 + x[None, None, :] ** 2
    rho = (2 * np.pi * sigma ** 2) ** -1.5 * np.exp(-r2 / (2 * sigma ** 2))
    v = o.poisson(rho)
    r = np.sqrt(r2)
    with np.errstate(divide="ignore", invalid="ignore"):
        ref = np.where(r > 0, erf(r / (math.sqrt(2) * sigma)) / r, math.sqrt(2 / np.pi) / sigma)
    self_energy = h ** 3 * np.sum(rho * v)
    return np.max(np.abs(v - ref)), abs(self_energy - 1.0 / (math.sqrt(np.pi) * sigma))


def test_p6_gaussian_free_converges():
    sigma = 1.0
    ev1, ee1 = _gaussian_free_errors(24, 0.5, sigma)      # box half-width 5.75 sigma
    ev2, ee2 = _gaussian_free_errors(48, 0.25, sigma)
    assert ev1 < 1.5e-2 and ev2 < 4e-3
    assert ee1 < 6e-3 and ee2 < 1.5e-3
    assert 3.0 <= ev1 / ev2 <= 5.0                        # second-order discretisation of the point-sampled 1/r
    assert 3.0 <= ee1 / ee2 <= 5.0


def test_p6_cell_average_constant():
    with open(os.path.join(GOLDEN, "constants.txt")) as fh:
        c0 = [float(line.split()[1]) for line in fh if line.startswith("c0")][0]
    assert abs(c0 - (3 * math.log(2 + math.sqrt(3)) - math.pi / 2)) < 1e-15
    for h in (0.25, 0.35, 1.0):
        assert abs(cell_average_inverse_r((h, h, h)) - c0 / h) <= 1e-12 / h


# ------------------------------------------------------------------ P7-P9 on seeded synthetic orbitals
@pytest.fixture(scope="module")
def small_periodic():
    w = make_workload(small_spec("C1", dims=(12, 8, 6), n_orb=4, spacing=(0.5, 0.6, 0.7)))
    w["occ"] = np.array([2.0, 1.5, 0.0, 0.7])
    o = Oracle(w["spec"].dims, w["spec"].spacing, "periodic")
    return w, o, o.apply(w["psi"].numpy(), w["occ"])


@pytest.fixture(scope="module")
def small_free():
    w = make_workload(small_spec("C2", dims=(6, 8, 10), n_orb=3, spacing=(0.5, 0.45, 0.4)))
    w["occ"] = np.array([2.0, 1.0, 0.5])
    o = Oracle(w["spec"].dims, w["spec"].spacing, "free", w["kernel"])
    return w, o, o.apply(w["psi"].numpy(), w["occ"])


@pytest.mark.parametrize("which", ["periodic", "free"])
def test_p7_invariants(which, small_periodic, small_free):
    w, o, (kpsi, ex, e) = small_periodic if which == "periodic" else small_free
    psi, occ, dV = w["psi"].numpy(), w["occ"], w["spec"].dV
    n_orb = psi.shape[0]
    assert np.array_equal(e, e.T)                               # e_ij = e_ji (rho_ij = rho_ji exactly, A2)
    assert ex <= 0.0
    assert np.all(np.diag(e) > 0)
    if which == "periodic":
        assert np.all(e >= -1e-16)                              # K^ >= 0
    # i<=j shortcut (what the GPU does) reproduces the definition
    kpsi_s, ex_s, e_s = o.apply(psi, occ, symmetric=True)
    scale = np.max(np.abs(kpsi))
    assert np.max(np.abs(kpsi_s - kpsi)) <= 1e-13 * scale
    assert abs(ex_s - ex) <= 1e-13 * abs(ex)
    live = (occ[:, None] != 0) | (occ[None, :] != 0)            # a pair with f_i = f_j = 0 is skipped (A15)
    assert np.max(np.abs(e_s - e)[live]) <= 1e-13 * np.max(np.abs(e))
    assert np.all(e_s[~live] == 0.0)
    # <psi_k|K psi_l> = <psi_l|K psi_k>
    kmat = dV * psi.reshape(n_orb, -1) @ kpsi.reshape(n_orb, -1).T
    assert np.max(np.abs(kmat - kmat.T)) <= 1e-12 * np.max(np.abs(kmat))


@pytest.mark.parametrize("which", ["periodic", "free"])
def test_p8_energy_operator_consistency(which, small_periodic, small_free):
    w, o, (kpsi, ex, e) = small_periodic if which == "periodic" else small_free
    psi, occ, dV = w["psi"].numpy(), w["occ"], w["spec"].dV
    # E_x = 1/2 dV sum_i f_i <psi_i|K psi_i>
    ex2 = 0.5 * dV * sum(occ[i] * np.sum(psi[i] * kpsi[i]) for i in range(psi.shape[0]))
    assert abs(ex2 - ex) <= 1e-13 * abs(ex)
    # E_x recomputed from the e-matrix
    ex3 = -0.5 * np.einsum("i,j,ij->", occ, occ, e)
    assert abs(ex3 - ex) <= 1e-13 * abs(ex)
    # directional derivative: dE_x[psi_i + eps d]/d eps = 2 f_i dV <d|K psi_i>  (static form of PAPER.md:161)
    i, eps = 1, 1e-5
    d = _rng(3).standard_normal(psi[i].shape)
    pp, pm = psi.copy(), psi.copy()
    pp[i] += eps * d
    pm[i] -= eps * d
    fd = (o.apply(pp, occ)[1] - o.apply(pm, occ)[1]) / (2 * eps)
    an = 2 * occ[i] * dV * np.sum(d * kpsi[i])
    assert abs(fd - an) <= 1e-7 * abs(an)


@pytest.mark.parametrize("which", ["periodic", "free"])
def test_p9_hartree_and_packing(which, small_periodic, small_free):
    w, o, _ = small_periodic if which == "periodic" else small_free
    psi, dV = w["psi"].numpy(), w["spec"].dV
    # N=1: K psi = -f V[psi^2] psi, E_x = -1/2 f^2 dV sum rho V (the Hartree energy of rho = psi^2)
    f = 1.7
    kpsi, ex, e = o.apply(psi[:1], [f])
    v = o.poisson(psi[0] ** 2)
    assert np.max(np.abs(kpsi[0] + f * v * psi[0])) <= 1e-14 * np.max(np.abs(kpsi))
    assert abs(ex + 0.5 * f * f * dV * np.sum(psi[0] ** 2 * v)) <= 1e-13 * abs(ex)
    # two real co-densities in one complex transform (the GPU's packing), done here with the LIBRARY FFT and the
    # oracle's K^: Re / Im must equal the oracle's two separate real solves.
    r1, r2 = psi[0] * psi[1], psi[1] * psi[2]
    t = o.tdims
    z = np.zeros(t, dtype=complex)
    z[:r1.shape[0], :r1.shape[1], :r1.shape[2]] = r1 + 1j * r2
    c = np.fft.ifftn(np.fft.fftn(z) * o.khat())[:r1.shape[0], :r1.shape[1], :r1.shape[2]]
    v1, v2 = o.poisson(r1), o.poisson(r2)
    scale = max(np.max(np.abs(v1)), np.max(np.abs(v2)))
    assert np.max(np.abs(c.real - v1)) <= 1e-13 * scale
    assert np.max(np.abs(c.imag - v2)) <= 1e-13 * scale
    # K^ is real and even up to rounding -> the symmetric (T/2+1)^3 real table the GPU keeps is lossless
    k = o.khat()
    assert np.max(np.abs(k.imag)) <= 1e-12 * np.max(np.abs(k.real))
    assert np.max(np.abs(k.real - np.roll(k.real[::-1, ::-1, ::-1], 1, axis=(0, 1, 2)))) <= 1e-12 * np.max(np.abs(k.real))


@pytest.mark.parametrize("which", ["periodic", "free"])
def test_rows_pairs_points_agree_with_apply(which, small_periodic, small_free):
    """The sampled-parity entry points (rows, pair energies, direct-sum points) reproduce the full apply."""
    w, o, (kpsi, ex, e) = small_periodic if which == "periodic" else small_free
    psi, occ = w["psi"].numpy(), w["occ"]
    rows, e_rows = o.rows(psi, occ, [2, 0])
    scale = np.max(np.abs(kpsi))
    assert np.max(np.abs(rows[0] - kpsi[2])) <= 1e-13 * scale
    assert np.max(np.abs(rows[1] - kpsi[0])) <= 1e-13 * scale
    assert np.max(np.abs(e_rows[0] - e[2])) <= 1e-13 * np.max(np.abs(e))
    pe = o.pair_energies(psi, [(0, 1), (2, 2), (1, 0)])
    assert np.max(np.abs(pe - np.array([e[0, 1], e[2, 2], e[1, 0]]))) <= 1e-13 * np.max(np.abs(e))
    orbs = [0, 1, 2, 1]
    pts = [0, 17, psi[0].size - 1, 123]
    got = o.kpsi_points(psi, occ, orbs, pts)
    ref = np.array([kpsi[i].reshape(-1)[p] for i, p in zip(orbs, pts)])
    assert np.max(np.abs(got - ref)) <= 1e-12 * scale


def test_generator_is_seeded_and_normalised():
    a = make_workload("C1")
    b = make_workload("C1")
    assert np.array_equal(a["psi"].numpy(), b["psi"].numpy())
    psi, dV = a["psi"].numpy(), a["spec"].dV
    assert np.allclose(dV * np.sum(psi.reshape(psi.shape[0], -1) ** 2, axis=1), 1.0, atol=1e-13)
    w = make_workload(small_spec("C3", dims=(16, 16, 16), n_orb=6))
    p = w["psi"].numpy().reshape(6, -1)
    assert np.max(np.abs(w["spec"].dV * p @ p.T - np.eye(6))) <= 1e-12


def test_full_c1_oracle_sanity():
    """C1 (BASELINE.json configs[0]) runs through the oracle in seconds; E_x < 0, all e_ij >= 0."""
    w = make_workload("C1")
    o = Oracle(w["spec"].dims, w["spec"].spacing, "periodic")
    kpsi, ex, e = o.apply(w["psi"].numpy(), w["occ"])
    assert ex < 0 and np.all(e >= 0) and np.isfinite(kpsi).all()
    ex2 = 0.5 * w["spec"].dV * sum(w["occ"][i] * np.sum(w["psi"].numpy()[i] * kpsi[i]) for i in range(8))
    assert abs(ex2 - ex) <= 1e-13 * abs(ex)
