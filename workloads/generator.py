"""Seeded synthetic orbitals and Green's-function tables (recipe: SURVEY.md 8(d)).

Stands in for the paper's converged BigDFT Kohn-Sham orbitals of water boxes and UO2 supercells
(PAPER.md:159, :179-185 Table 1, :202-210), which are not available.  Every step of the hot path is
data-oblivious, so only shapes, smoothness, normalisation and (for C3/C5) orthonormality matter.

Nothing here belongs to the method: no co-density, no transform, no Poisson solve.  Both the CUDA path and
the CPU oracle receive the *same bytes* produced here (generate once, copy).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace
from typing import Dict, Optional, Tuple

import numpy as np
import torch

_MASK64 = (1 << 64) - 1
SEED_BASE = 171207973 * 10  # + config number


class SplitMix64:
    """Self-written SplitMix64 stream; `uniform()` returns the top 53 bits as a double in [0,1)."""

    def __init__(self, seed: int):
        self.state = seed & _MASK64

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _MASK64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK64
        return z ^ (z >> 31)

    def uniform(self) -> float:
        return (self.next_u64() >> 11) * (1.0 / 9007199254740992.0)


@dataclass(frozen=True)
class WorkloadSpec:
    name: str
    number: int                      # seed = SEED_BASE + number
    bc: str                          # "periodic" | "free"
    dims: Tuple[int, int, int]       # n1, n2, n3 (last index fastest in memory)
    spacing: Tuple[float, float, float]
    n_orb: int
    n_gauss: int                     # Gaussians per orbital
    sigma: Tuple[float, float]       # uniform range, bohr
    inner_fraction: float            # centres uniform in the inner fraction of each axis (1.0 = whole box)
    n_centres: Optional[int]         # shared pool of centres ("atoms"); None = one private centre per Gaussian
    orthonormalize: bool             # Loewdin on the grid
    occupation: float = 2.0

    @property
    def n_pairs(self) -> int:
        return self.n_orb * (self.n_orb + 1) // 2

    @property
    def n_points(self) -> int:
        return self.dims[0] * self.dims[1] * self.dims[2]

    @property
    def dV(self) -> float:
        return self.spacing[0] * self.spacing[1] * self.spacing[2]


# The five configs of BASELINE.json, made concrete as in SURVEY.md 8(d).
CONFIGS: Dict[str, WorkloadSpec] = {
    "C1": WorkloadSpec("C1", 1, "periodic", (32, 32, 32), (0.4, 0.4, 0.4), 8, 4, (0.8, 1.5), 1.0, None, False),
    "C2": WorkloadSpec("C2", 2, "free", (64, 64, 64), (0.35, 0.35, 0.35), 32, 6, (0.6, 1.2), 0.6, None, False),
    "C3": WorkloadSpec("C3", 3, "periodic", (96, 96, 96), (0.3, 0.3, 0.3), 128, 4, (0.8, 1.5), 1.0, None, True),
    "C4": WorkloadSpec("C4", 4, "free", (128, 128, 128), (0.3, 0.3, 0.3), 256, 6, (0.6, 1.2), 0.6, 128, False),
    "C5": WorkloadSpec("C5", 5, "periodic", (192, 192, 192), (0.25, 0.25, 0.25), 1024, 4, (0.8, 1.5), 1.0, 512, True),
}


def small_spec(base: str, *, dims=None, n_orb=None, number=None, spacing=None, name=None,
               orthonormalize=None, n_centres="keep") -> WorkloadSpec:
    """A reduced variant of a named config (same recipe, other sizes) for parity cases the oracle finishes fast."""
    s = CONFIGS[base]
    kw = {}
    if dims is not None:
        kw["dims"] = tuple(int(d) for d in dims)
    if n_orb is not None:
        kw["n_orb"] = int(n_orb)
    if number is not None:
        kw["number"] = int(number)
    if spacing is not None:
        kw["spacing"] = tuple(float(x) for x in spacing)
    if orthonormalize is not None:
        kw["orthonormalize"] = bool(orthonormalize)
    if n_centres != "keep":
        kw["n_centres"] = n_centres
    kw["name"] = name or f"{base}-small"
    return replace(s, **kw)


def _draw_parameters(spec: WorkloadSpec):
    """Fixed draw order: all centres first, then per orbital and per Gaussian (centre choice, sigma, coefficient)."""
    rng = SplitMix64(SEED_BASE + spec.number)
    box = [n * h for n, h in zip(spec.dims, spec.spacing)]
    lo = [(1.0 - spec.inner_fraction) * 0.5 * L for L in box]
    span = [spec.inner_fraction * L for L in box]
    n_pool = spec.n_centres if spec.n_centres is not None else spec.n_orb * spec.n_gauss
    centres = np.empty((n_pool, 3))
    for p in range(n_pool):
        for ax in range(3):
            centres[p, ax] = lo[ax] + span[ax] * rng.uniform()
    which = np.empty((spec.n_orb, spec.n_gauss), dtype=np.int64)
    sigma = np.empty((spec.n_orb, spec.n_gauss))
    coeff = np.empty((spec.n_orb, spec.n_gauss))
    for i in range(spec.n_orb):
        for g in range(spec.n_gauss):
            if spec.n_centres is not None:
                which[i, g] = min(int(rng.uniform() * n_pool), n_pool - 1)
            else:
                which[i, g] = i * spec.n_gauss + g
            sigma[i, g] = spec.sigma[0] + (spec.sigma[1] - spec.sigma[0]) * rng.uniform()
            sign = 1.0 if rng.uniform() < 0.5 else -1.0
            coeff[i, g] = sign * (0.5 + 0.5 * rng.uniform())
    return centres, which, sigma, coeff


def make_orbitals(spec: WorkloadSpec, device="cpu") -> torch.Tensor:
    """psi[N][n1][n2][n3], fp64, C order; each orbital normalised so that dV * sum(psi^2) = 1.

    Gaussian term: a * (pi sigma^2)^(-3/4) * exp(-|r-c|^2 / (2 sigma^2)); periodic boxes use the
    minimum-image distance.  The product form exp(-dx^2..)exp(-dy^2..)exp(-dz^2..) is evaluated per axis.
    """
    centres, which, sigma, coeff = _draw_parameters(spec)
    dev = torch.device(device)
    n1, n2, n3 = spec.dims
    axes = [torch.arange(n, dtype=torch.float64, device=dev) * h for n, h in zip(spec.dims, spec.spacing)]
    box = [n * h for n, h in zip(spec.dims, spec.spacing)]
    psi = torch.empty((spec.n_orb, n1, n2, n3), dtype=torch.float64, device=dev)
    dV = spec.dV
    for i in range(spec.n_orb):
        c = torch.as_tensor(centres[which[i]], dtype=torch.float64, device=dev)          # (G,3)
        s = torch.as_tensor(sigma[i], dtype=torch.float64, device=dev)                    # (G,)
        a = torch.as_tensor(coeff[i], dtype=torch.float64, device=dev) * (math.pi * s * s) ** (-0.75)
        fac = []
        for ax in range(3):
            d = axes[ax][None, :] - c[:, ax:ax + 1]                                       # (G,n)
            if spec.bc == "periodic":
                L = box[ax]
                d = torch.remainder(d + 0.5 * L, L) - 0.5 * L
            fac.append(torch.exp(-(d * d) / (2.0 * s[:, None] ** 2)))
        orb = torch.einsum("ga,gb,gc->abc", fac[0] * a[:, None], fac[1], fac[2])
        orb = orb / torch.sqrt(dV * torch.sum(orb * orb))
        psi[i] = orb
    if spec.orthonormalize:
        _loewdin_inplace(psi, dV)
    return psi


def _loewdin_inplace(psi: torch.Tensor, dV: float, chunk_points: int = 1 << 22) -> None:
    """Psi <- S^(-1/2) Psi with S = dV Psi Psi^T (harness only).  Applied in grid chunks, in place."""
    n_orb = psi.shape[0]
    flat = psi.view(n_orb, -1)
    m = flat.shape[1]
    S = torch.zeros((n_orb, n_orb), dtype=torch.float64, device=psi.device)
    for lo in range(0, m, chunk_points):
        blk = flat[:, lo:lo + chunk_points]
        S += blk @ blk.T
    S *= dV
    lam, U = torch.linalg.eigh(S)
    if float(lam.min()) < 1e-8:
        raise ValueError(f"overlap matrix nearly singular (lambda_min={float(lam.min()):.3e}); choose another seed")
    S_inv_half = (U * lam.rsqrt()[None, :]) @ U.T
    for lo in range(0, m, chunk_points):
        flat[:, lo:lo + chunk_points] = S_inv_half @ flat[:, lo:lo + chunk_points]


def _pyramid(a: float, b: float, c: float, nodes: int = 96) -> float:
    """Integral of 1/r over the pyramid with apex at the origin and base {x=a, 0<=y<=b, 0<=z<=c}.

    With y = x s, z = x t the integrand becomes x / sqrt(1+s^2+t^2): smooth, Gauss-Legendre converges fast.
    """
    x, w = np.polynomial.legendre.leggauss(nodes)
    s = 0.5 * (x + 1.0) * (b / a)
    ws = 0.5 * w * (b / a)
    t = 0.5 * (x + 1.0) * (c / a)
    wt = 0.5 * w * (c / a)
    val = np.sum(ws[:, None] * wt[None, :] / np.sqrt(1.0 + s[:, None] ** 2 + t[None, :] ** 2))
    return 0.5 * a * a * float(val)


def cell_average_inverse_r(spacing) -> float:
    """(1/dV) * integral of 1/|x| over the grid cell centred at the origin.

    For a cubic cell this is c0/h with c0 = 3 ln(2+sqrt 3) - pi/2 = 2.380077363979553.
    """
    a, b, c = (0.5 * float(h) for h in spacing)
    octant = _pyramid(a, b, c) + _pyramid(b, c, a) + _pyramid(c, a, b)
    return 8.0 * octant / (8.0 * a * b * c)


def free_kernel_table(dims, spacing) -> np.ndarray:
    """Host table g[a][b][c] = 1/|d|, d = (a h1, b h2, c h3), d = 0 entry cell-averaged (BASELINE.json C2/C4)."""
    n1, n2, n3 = (int(d) for d in dims)
    h1, h2, h3 = (float(h) for h in spacing)
    x = (np.arange(n1) * h1)[:, None, None]
    y = (np.arange(n2) * h2)[None, :, None]
    z = (np.arange(n3) * h3)[None, None, :]
    r2 = x * x + y * y + z * z
    r2[0, 0, 0] = 1.0
    g = 1.0 / np.sqrt(r2)
    g[0, 0, 0] = cell_average_inverse_r((h1, h2, h3))
    return np.ascontiguousarray(g)


def mixed_bc_kernel_table(dims, spacing, periodic, mu: float, images: int = 2) -> np.ndarray:
    """Host table for slab / wire boundary conditions, handed to a FREE-BC plan as data: the short-range
    screened Coulomb kernel erfc(mu r)/r (the HSE-type filter of PAPER.md:236 in real space) summed over the periodic
    images along the axes marked periodic,
        g[a][b][c] = sum_{m} erfc(mu |d + m L|) / |d + m L|,   d = (a h1, b h2, c h3),  m_axis = -images..images,
    where L_axis = n_axis h_axis on periodic axes and m_axis = 0 on isolated ones.  Along a periodic axis the table holds
    one full period and is even under index -> n - index (up to the truncated image sum, which erfc makes negligible
    for mu L >= 4); the d = 0 entry takes the cell average of 1/r minus the r -> 0 limit 2 mu / sqrt(pi) of
    (1 - erfc)/r.  Input data only: none of the method's arithmetic."""
    from math import erfc, pi, sqrt
    n = [int(d) for d in dims]
    h = [float(x) for x in spacing]
    per = [bool(x) for x in periodic]
    rng = [range(-images, images + 1) if per[ax] else range(0, 1) for ax in range(3)]
    ax_d = [np.arange(n[ax]) * h[ax] for ax in range(3)]
    verfc = np.vectorize(erfc)
    g = np.zeros(n, dtype=np.float64)
    for m0 in rng[0]:
        for m1 in rng[1]:
            for m2 in rng[2]:
                x = (ax_d[0] + m0 * n[0] * h[0])[:, None, None]
                y = (ax_d[1] + m1 * n[1] * h[1])[None, :, None]
                z = (ax_d[2] + m2 * n[2] * h[2])[None, None, :]
                r = np.sqrt(x * x + y * y + z * z)
                home = m0 == 0 and m1 == 0 and m2 == 0
                if home:
                    r[0, 0, 0] = 1.0
                term = verfc(mu * r) / r
                if home:
                    term[0, 0, 0] = cell_average_inverse_r(h) - 2.0 * mu / sqrt(pi)
                g += term
    # make the evenness along periodic axes exact (the truncated image sum breaks it at the 1e-16..1e-12 level)
    for ax in range(3):
        if per[ax]:
            idx = (-np.arange(n[ax])) % n[ax]
            g = 0.5 * (g + np.take(g, idx, axis=ax))
    return np.ascontiguousarray(g)


def general_cell_khat(dims, lattice) -> tuple:
    """Fourier-space Coulomb kernel of a periodic cell of any shape, for exx_plan_create_general: lattice = rows a1, a2, a3
    (bohr).  Returns (K^ on the full FFT index grid [n1][n2][n3], cell volume):  K^(m) = 4 pi / |m1 b1 + m2 b2 + m3 b3|^2
    with the reciprocal vectors b_a (a_a . b_b = 2 pi delta_ab) and signed frequencies m_a in (-n_a/2, n_a/2], K^(0) = 0.
    An index n_a/2 is its own negative, so the table is symmetrised, K^(m) <- (K^(m) + K^(-m mod n)) / 2, which makes
    K^(-m) = K^(m) hold exactly (real potentials).  Input data only: none of the method's arithmetic."""
    n = [int(d) for d in dims]
    a = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
    vol = abs(float(np.linalg.det(a)))
    b = 2.0 * np.pi * np.linalg.inv(a).T                    # rows b1, b2, b3
    m = [np.where(np.arange(k) <= k // 2, np.arange(k), np.arange(k) - k).astype(np.float64) for k in n]
    g = (m[0][:, None, None, None] * b[0] + m[1][None, :, None, None] * b[1] + m[2][None, None, :, None] * b[2])
    g2 = np.sum(g * g, axis=-1)
    khat = np.where(g2 > 0, 4.0 * np.pi / np.where(g2 > 0, g2, 1.0), 0.0)
    neg = khat
    for ax in range(3):
        neg = np.take(neg, (-np.arange(n[ax])) % n[ax], axis=ax)
    return np.ascontiguousarray(0.5 * (khat + neg)), vol


def make_workload(spec_or_name, device="cpu") -> dict:
    """Orbitals, occupations and (free BC) the Green's-function table for a config name or a WorkloadSpec."""
    spec = CONFIGS[spec_or_name] if isinstance(spec_or_name, str) else spec_or_name
    psi = make_orbitals(spec, device=device)
    occ = np.full((spec.n_orb,), spec.occupation, dtype=np.float64)
    kernel = free_kernel_table(spec.dims, spec.spacing) if spec.bc == "free" else None
    return {"spec": spec, "psi": psi, "occ": occ, "kernel": kernel}
