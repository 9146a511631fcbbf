"""GPU parity of the SURVEY.md 8(f) entry points (through the C ABI) against the oracle functions pinned in
tests/test_oracle_pins_ext.py.  Tolerances as in test_gpu_parity.py (north_star): 1e-10 max|K psi|, 1e-11 on energies.

  exx_apply_to      K of the occupied set applied to another orbital set        (NEXT-1)
  exx_apply_complex complex orbitals through the real kernels (+ exx_apply_to_cross)  (NEXT-1; Eq. 8)
  periodic filter   host-supplied Fourier-space table (screened kernel)          (NEXT-2)
  slab / wire BC    FREE plan + one period of the mixed Green's function as data (NEXT-2)
  general cells     non-orthorhombic periodic cell: K^ on the full FFT index grid   (NEXT-2)
  exx_apply_block   all pairs between two disjoint blocks + round-robin schedule (NEXT-3)
  exx_apply_pairs   sparse pair list for localised orbitals                      (NEXT-4)
"""
import ctypes as C

import numpy as np
import pytest
import torch

import paper_1712_07973_b200 as exx
from oracle import Oracle
from paper_1712_07973_b200.distributed import block_range
from workloads import make_workload, small_spec

pytestmark = pytest.mark.gpu

E_RTOL = 1e-11
K_RTOL = 1e-10


def _setup(base, dims, n_orb, number, kernel=None):
    w = make_workload(small_spec(base, dims=dims, n_orb=n_orb, spacing=(0.45, 0.4, 0.5), number=number))
    spec = w["spec"]
    kern = w["kernel"] if kernel is None else kernel
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, kern, max_orbitals=n_orb)
    o = Oracle(spec.dims, spec.spacing, spec.bc, kern)
    return w, spec, plan, o


# ------------------------------------------------------------------ NEXT-1: exx_apply_to
@pytest.mark.parametrize("base,dims,n_occ,n_tgt,batch", [("C1", (16, 16, 16), 4, 3, 0), ("C2", (8, 16, 8), 3, 4, 2), ("C1", (16, 32, 64), 5, 2, 3),
                                                         ("C1", (96, 96, 96), 5, 3, 2), ("C2", (48, 48, 48), 4, 3, 0)])
def test_apply_to_matches_oracle(base, dims, n_occ, n_tgt, batch):
    w, spec, plan, o = _setup(base, dims, n_occ + n_tgt, 500 + sum(dims))
    if batch:
        plan.set_batch(batch)
    allpsi = w["psi"].cuda()
    psi, phi = allpsi[:n_occ].contiguous(), allpsi[n_occ:].contiguous()
    occ = np.array([2.0, 0.0, 1.3, 0.6, 1.0][:n_occ])                    # a zero occupation: that orbital is skipped
    kphi = plan.apply_to(psi, occ, phi)
    ref = o.apply_to(w["psi"][:n_occ].numpy(), occ, w["psi"][n_occ:].numpy())
    assert np.max(np.abs(kphi.cpu().numpy() - ref)) <= K_RTOL * np.max(np.abs(ref))
    # phi = psi: the operator applied to its own occupied set is exx_apply's K psi
    k_self = plan.apply_to(psi, occ, psi)
    k_sq, _ = plan.apply(psi, occ)
    assert float((k_self - k_sq).abs().max()) <= 1e-12 * float(k_sq.abs().max())
    # a second "spin channel" is a second call with other occupied orbitals on the same plan: results are independent
    kphi2 = plan.apply_to(psi, occ, phi)
    assert torch.equal(kphi, kphi2)
    plan.destroy()


# ------------------------------------------------------------------ the TMA-tile kernels under the rectangular entry points
@pytest.mark.parametrize("base,dims", [("C1", (16, 192, 192)), ("C1", (32, 64, 128)), ("C2", (8, 64, 128)), ("C2", (16, 96, 96))])
def test_tma_tile_geometries_under_apply_to_block_and_complex(base, dims):
    """Geometries whose pass C gathers its W1 tile by a TMA tensor-box copy (c-axis transform length 128 / 192 / 256, one b2 per
    tile) and whose pass A (periodic) sends it by a tensor-box store, driven through exx_apply_to, exx_apply_block and
    exx_apply_complex: resident and streamed sets differ, so the partner-set and accumulate paths of those kernels run too."""
    n_a, n_b = 3, 2
    w = make_workload(small_spec(base, dims=dims, n_orb=n_a + n_b + 1, spacing=(0.45, 0.4, 0.5), number=1900 + sum(dims)))
    spec = w["spec"]
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=n_a + n_b + 1)
    plan.set_batch(2)
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    allp = w["psi"].cuda()
    pa, pb = allp[:n_a].contiguous(), allp[n_a:n_a + n_b].contiguous()
    ha, hb = w["psi"][:n_a].numpy(), w["psi"][n_a:n_a + n_b].numpy()
    occ_a, occ_b = np.array([2.0, 0.0, 1.3]), np.array([0.6, 1.0])
    # apply_to
    kphi = plan.apply_to(pa, occ_a, pb)
    ref = o.apply_to(ha, occ_a, hb)
    assert np.max(np.abs(kphi.cpu().numpy() - ref)) <= K_RTOL * np.max(np.abs(ref))
    # apply_block
    ka, kb = torch.empty_like(pa), torch.empty_like(pb)
    ex = plan.apply_block(pa, occ_a, ka, pb, occ_b, kb)
    ka_ref, kb_ref, ex_ref, _ = o.apply_block(ha, occ_a, hb, occ_b)
    assert np.max(np.abs(ka.cpu().numpy() - ka_ref)) <= K_RTOL * np.max(np.abs(ka_ref))
    assert np.max(np.abs(kb.cpu().numpy() - kb_ref)) <= K_RTOL * np.max(np.abs(kb_ref))
    assert abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    # complex orbitals: 3 complex = 6 real
    planar = w["psi"].reshape(2, 3, *dims)
    occ_c = np.array([2.0, 0.9, 0.4])
    k_ref, exc_ref = o.apply_complex(planar[0].numpy() + 1j * planar[1].numpy(), occ_c)
    kpl, exc = plan.apply_complex(planar.cuda(), occ_c)
    k_gpu = kpl[0].cpu().numpy() + 1j * kpl[1].cpu().numpy()
    assert np.max(np.abs(k_gpu - k_ref)) <= K_RTOL * np.max(np.abs(k_ref))
    assert abs(exc - exc_ref) <= E_RTOL * abs(exc_ref)
    plan.destroy()


# ------------------------------------------------------------------ NEXT-1: complex orbitals
@pytest.mark.parametrize("base,dims,n_orb,batch", [("C1", (16, 16, 16), 3, 0), ("C2", (8, 16, 8), 3, 2), ("C1", (96, 96, 96), 3, 3),
                                                   ("C2", (48, 48, 48), 2, 0)])
def test_apply_complex_matches_oracle(base, dims, n_orb, batch):
    """exx_apply_complex (planar real / imaginary parts) against the oracle's complex definition (P17), and its building
    block exx_apply_to_cross against the oracle's cross apply."""
    w = make_workload(small_spec(base, dims=dims, n_orb=2 * n_orb, spacing=(0.45, 0.4, 0.5), number=1700 + sum(dims)))
    spec = w["spec"]
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=2 * n_orb)
    if batch:
        plan.set_batch(batch)
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    planar = w["psi"].reshape(2, n_orb, *dims)                              # seeded real / imaginary parts
    psi_c = planar[0].numpy() + 1j * planar[1].numpy()
    occ = np.array([2.0, 0.9, 0.0][:n_orb])
    k_ref, ex_ref = o.apply_complex(psi_c, occ)
    kpl, ex = plan.apply_complex(planar.cuda(), occ)
    k_gpu = kpl[0].cpu().numpy() + 1j * kpl[1].cpu().numpy()
    assert np.max(np.abs(k_gpu - k_ref)) <= K_RTOL * np.max(np.abs(k_ref))
    assert abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    # the building block on its own
    x = w["psi"].cuda()
    chi = torch.flip(x, dims=[0]).contiguous()
    occ2 = np.concatenate([occ, occ])
    kx = plan.apply_to_cross(x, chi, occ2, x[:2].contiguous())
    ref = o.apply_to_cross(w["psi"].numpy(), chi.cpu().numpy(), occ2, w["psi"][:2].numpy())
    assert np.max(np.abs(kx.cpu().numpy() - ref)) <= K_RTOL * np.max(np.abs(ref))
    plan.destroy()


# ------------------------------------------------------------------ NEXT-2: periodic Fourier-space filter table
def _screened_table(dims, spacing, omega):
    g = [2 * np.pi * np.arange(n // 2 + 1) / (n * h) for n, h in zip(dims, spacing)]
    g2 = g[0][:, None, None] ** 2 + g[1][None, :, None] ** 2 + g[2][None, None, :] ** 2
    safe = np.where(g2 > 0, g2, 1.0)
    return np.where(g2 > 0, 4 * np.pi / safe * (1 - np.exp(-safe / (4 * omega ** 2))), np.pi / omega ** 2)


@pytest.mark.parametrize("dims", [(16, 32, 64), (96, 96, 96)])
def test_periodic_filter_table_matches_oracle_and_closed_form(dims):
    spacing = (0.45, 0.4, 0.5)
    table = _screened_table(dims, spacing, 0.3)
    w, spec, plan, o = _setup("C1", dims, 4, 600 + sum(dims), kernel=table)
    occ = np.array([2.0, 1.0, 0.5, 1.5])
    kpsi, ex = plan.apply(w["psi"].cuda(), occ)
    e = plan.pair_energies()
    k_ref, ex_ref, e_ref = o.apply(w["psi"].numpy(), occ, symmetric=True)
    assert np.max(np.abs(kpsi.cpu().numpy() - k_ref)) <= K_RTOL * np.max(np.abs(k_ref))
    assert abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    assert np.max(np.abs(e - e_ref)) <= E_RTOL * np.max(np.abs(e_ref))
    # closed form on the GPU itself: psi_1 = Vol^-1/2, psi_2 = sqrt(2/Vol) cos(k.r)  ->  e_12 = K^(k)/Vol, e_22 = K^(2k)/(2 Vol) + K^(0)/Vol
    L = [n * h for n, h in zip(dims, spacing)]
    vol = L[0] * L[1] * L[2]
    m = (3, 1, 2)
    k = np.array([2 * np.pi * m[a] / L[a] for a in range(3)])
    ax = [np.arange(n) * h for n, h in zip(dims, spacing)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    two = np.stack([np.full(dims, vol ** -0.5), np.sqrt(2 / vol) * np.cos(k[0] * X + k[1] * Y + k[2] * Z)])
    plan.apply(torch.from_numpy(two).cuda(), [1.0, 1.0])
    e2 = plan.pair_energies()
    khat = lambda q: 4 * np.pi / (q @ q) * (1 - np.exp(-(q @ q) / (4 * 0.3 ** 2)))
    k0 = np.pi / 0.3 ** 2
    assert abs(e2[0, 1] - khat(k) / vol) <= 1e-12 * khat(k) / vol
    assert abs(e2[0, 0] - k0 / vol) <= 1e-12 * k0 / vol
    assert abs(e2[1, 1] - (khat(2 * k) / (2 * vol) + k0 / vol)) <= 1e-12 * k0 / vol
    plan.destroy()


# ------------------------------------------------------------------ NEXT-2: slab / wire boundary conditions
@pytest.mark.parametrize("dims,periodic,n_orb", [((8, 16, 8), (1, 1, 0), 3), ((8, 8, 16), (0, 0, 1), 3)])
def test_slab_and_wire_match_the_direct_mixed_definition(dims, periodic, n_orb):
    """Slab (two periodic axes) and wire (one) boundary conditions are a FREE plan whose host table holds one period of
    the mixed Green's function along the periodic axes (A24).  Reference: the oracle's O(M^2)
    wrap-around direct sum, pair by pair (P15), combined by Eq. 3 / Eq. 5 in numpy."""
    from oracle import poisson_direct_mixed
    from workloads import mixed_bc_kernel_table
    spacing = (0.45, 0.4, 0.5)
    w = make_workload(small_spec("C2", dims=dims, n_orb=n_orb, spacing=spacing, number=700 + sum(dims)))
    spec = w["spec"]
    table = mixed_bc_kernel_table(dims, spacing, periodic, mu=1.2)
    occ = np.array([2.0, 1.1, 0.4][:n_orb])
    psi = w["psi"].numpy()
    k_ref = np.zeros_like(psi)
    ex_ref = 0.0
    for i in range(n_orb):
        for j in range(n_orb):
            v = poisson_direct_mixed(dims, spacing, periodic, table, psi[i] * psi[j])
            k_ref[i] -= occ[j] * v * psi[j]
            ex_ref -= 0.5 * occ[i] * occ[j] * spec.dV * float(np.sum(psi[i] * psi[j] * v))
    plan = exx.ExxPlan(spec.dims, spec.spacing, "free", table, max_orbitals=n_orb)
    kpsi, ex = plan.apply(w["psi"].cuda(), occ)
    assert np.max(np.abs(kpsi.cpu().numpy() - k_ref)) <= K_RTOL * np.max(np.abs(k_ref))
    assert abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    plan.destroy()


def test_slab_at_a_warp_specialised_size_matches_the_oracle():
    """The same at 48 x 48 x 24 (transform grid 96 x 96 x 48) against the oracle's FFT path with the same table -- which
    P15 ties to the wrap-around definition."""
    from workloads import mixed_bc_kernel_table
    dims, n_orb = (48, 48, 24), 4
    w = make_workload(small_spec("C2", dims=dims, n_orb=n_orb, spacing=(0.45, 0.4, 0.5), number=777))
    spec = w["spec"]
    table = mixed_bc_kernel_table(dims, spec.spacing, (1, 1, 0), mu=0.8)
    occ = np.array([2.0, 1.0, 0.0, 1.5])
    plan = exx.ExxPlan(spec.dims, spec.spacing, "free", table, max_orbitals=n_orb)
    kpsi, ex = plan.apply(w["psi"].cuda(), occ)
    k_ref, ex_ref, _ = Oracle(spec.dims, spec.spacing, "free", table).apply(w["psi"].numpy(), occ)
    assert np.max(np.abs(kpsi.cpu().numpy() - k_ref)) <= K_RTOL * np.max(np.abs(k_ref))
    assert abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    plan.destroy()


# ------------------------------------------------------------------ NEXT-2: general (non-orthorhombic) periodic cells
@pytest.mark.parametrize("dims,n_orb,batch", [((16, 32, 64), 4, 0), ((96, 96, 96), 4, 2), ((48, 96, 32), 3, 0), ((192, 48, 96), 3, 2)])
def test_general_cell_matches_oracle(dims, n_orb, batch):
    """exx_plan_create_general: a triclinic cell -- K^ on the full FFT index grid, even only under inversion (DESIGN.md
    A25) -- against the oracle with the same table (P16).  Orbitals: the seeded Gaussian sums sampled on the
    index grid."""
    from workloads import general_cell_khat
    lattice = np.array([[0.5 * dims[0], 0.0, 0.0], [0.13 * dims[1], 0.45 * dims[1], 0.0], [-0.07 * dims[2], 0.1 * dims[2], 0.4 * dims[2]]])
    khat, vol = general_cell_khat(dims, lattice)
    w = make_workload(small_spec("C1", dims=dims, n_orb=n_orb, spacing=(0.45, 0.4, 0.5), number=1600 + sum(dims)))
    occ = np.array([2.0, 1.2, 0.0, 0.7][:n_orb])
    plan = exx.ExxPlan.general(dims, vol, khat, max_orbitals=n_orb)
    if batch:
        plan.set_batch(batch)
    kpsi, ex = plan.apply(w["psi"].cuda(), occ)
    k_ref, ex_ref, e_ref = Oracle.general(dims, vol, khat).apply(w["psi"].numpy(), occ)
    assert np.max(np.abs(kpsi.cpu().numpy() - k_ref)) <= K_RTOL * np.max(np.abs(k_ref))
    assert abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    e = plan.pair_energies(n_orb)
    live = (occ[:, None] != 0) | (occ[None, :] != 0)
    assert np.all((np.abs(e - e_ref) <= E_RTOL * np.max(np.abs(e_ref)))[live])
    plan.destroy()


# ------------------------------------------------------------------ NEXT-3: exx_apply_block + the round-robin schedule
@pytest.mark.parametrize("base,dims,n_a,n_b,batch", [("C1", (16, 16, 16), 3, 4, 0), ("C2", (16, 8, 8), 2, 3, 2), ("C1", (96, 96, 96), 3, 4, 3),
                                                     ("C2", (48, 48, 48), 3, 2, 0)])
def test_apply_block_matches_oracle(base, dims, n_a, n_b, batch):
    w, spec, plan, o = _setup(base, dims, n_a + n_b, 700 + sum(dims))
    if batch:
        plan.set_batch(batch)
    allpsi = w["psi"].cuda()
    occ = np.array([2.0, 0.0, 1.3, 0.6, 0.0, 1.0, 1.7][: n_a + n_b])
    a, b = allpsi[:n_a], allpsi[n_a:]                                    # sub-ranges of ONE array
    ka, kb = torch.empty_like(a), torch.empty_like(b)
    ex = plan.apply_block(a, occ[:n_a], ka, b, occ[n_a:], kb)
    e = plan.block_energies(n_a, n_b)
    ka_ref, kb_ref, ex_ref, e_ref = o.apply_block(w["psi"][:n_a].numpy(), occ[:n_a], w["psi"][n_a:].numpy(), occ[n_a:])
    scale = max(np.max(np.abs(ka_ref)), np.max(np.abs(kb_ref)))
    assert np.max(np.abs(ka.cpu().numpy() - ka_ref)) <= K_RTOL * scale
    assert np.max(np.abs(kb.cpu().numpy() - kb_ref)) <= K_RTOL * scale
    assert abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    live = (occ[:n_a, None] != 0) | (occ[None, n_a:] != 0)
    assert np.all((np.abs(e - e_ref) <= E_RTOL * np.max(np.abs(e_ref)))[live]) and not e[~live].any()
    # accumulate flags: partial results of successive steps add up
    ka2, kb2 = torch.full_like(a, 0.25), torch.full_like(b, -0.5)
    ex2 = plan.apply_block(a, occ[:n_a], ka2, b, occ[n_a:], kb2, flags=exx.EXX_BLOCK_ACCUMULATE_RESIDENT | exx.EXX_BLOCK_ACCUMULATE_STREAMED)
    assert ex2 == ex
    # (pre-filled value + increment) is rounded at the magnitude of the pre-filled value: allow a few ulps of 0.5 on top
    assert float((ka2 - 0.25 - ka).abs().max()) <= 1e-13 * scale + 4e-16 and float((kb2 + 0.5 - kb).abs().max()) <= 1e-13 * scale + 4e-16
    # the same block memory on both sides is refused (the diagonal belongs to exx_apply)
    with pytest.raises(exx.ExxError):
        plan.apply_block(a, occ[:n_a], ka, a, occ[:n_a], torch.empty_like(a))
    plan.destroy()


@pytest.mark.parametrize("n_ranks,n_orb", [(2, 5), (3, 7), (4, 6)])
def test_round_robin_blocks_sum_to_the_full_apply(n_ranks, n_orb):
    """All ranks of the round-robin schedule, run one after the other on this GPU with the product's block calls:
    diagonal blocks by exx_apply, every scheduled block (full / half, `what` 1..3) by exx_apply_block with accumulation;
    the sum equals exx_apply of the whole set and the oracle."""
    w, spec, plan, o = _setup("C2", (16, 16, 16), n_orb, 800 + n_ranks)
    psi = w["psi"].cuda()
    occ = np.array([2.0, 0.7, 0.0, 1.3, 0.4, 1.1, 0.9][:n_orb])
    kpsi = torch.zeros_like(psi)
    ex = 0.0
    rng = [block_range(n_orb, n_ranks, r) for r in range(n_ranks)]
    for rank in range(n_ranks):
        lo, hi = rng[rank]
        kd, e0 = plan.apply(psi[lo:hi], occ[lo:hi])
        kpsi[lo:hi] += kd
        ex += e0
        for step in range(1, n_ranks // 2 + 1):
            _, src, what = exx.exx_round_robin_step(n_ranks, rank, step)
            vlo, vhi = rng[src]
            if what == 2:
                hi_r, vlo_s = lo + (hi - lo + 1) // 2, vlo
            elif what == 3:
                hi_r, vlo_s = hi, vlo + (vhi - vlo + 1) // 2
            else:
                hi_r, vlo_s = hi, vlo
            if hi_r == lo or vlo_s == vhi:
                continue
            ex += plan.apply_block(psi[lo:hi_r], occ[lo:hi_r], kpsi[lo:hi_r], psi[vlo_s:vhi], occ[vlo_s:vhi], kpsi[vlo_s:vhi],
                                   flags=exx.EXX_BLOCK_ACCUMULATE_RESIDENT | exx.EXX_BLOCK_ACCUMULATE_STREAMED)
    k_full, ex_full = plan.apply(psi, occ)
    k_ref, ex_ref, _ = o.apply(w["psi"].numpy(), occ, symmetric=False)
    scale = np.max(np.abs(k_ref))
    assert float((kpsi - k_full).abs().max()) <= 1e-12 * scale and abs(ex - ex_full) <= 1e-12 * abs(ex_full)
    assert np.max(np.abs(kpsi.cpu().numpy() - k_ref)) <= K_RTOL * scale and abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    plan.destroy()


# ------------------------------------------------------------------ NEXT-4: exx_apply_pairs
@pytest.mark.parametrize("base,dims,batch", [("C1", (16, 16, 16), 0), ("C2", (8, 8, 16), 2), ("C1", (96, 96, 96), 0)])
def test_apply_pairs_matches_masked_oracle(base, dims, batch):
    n = 6
    w, spec, plan, o = _setup(base, dims, n, 900 + sum(dims))
    if batch:
        plan.set_batch(batch)
    psi = w["psi"].cuda()
    occ = np.array([2.0, 1.0, 0.0, 0.6, 1.4, 0.8])
    rng = np.random.default_rng(9)
    mask = rng.random((n, n)) < 0.55
    mask = mask | mask.T
    mask[0, 0] = False                                                   # a diagonal pair can be excluded too
    mask[4, :] = mask[:, 4] = False                                      # an orbital without any partner: K psi_4 = 0
    mask[2, 3] = mask[3, 2] = True
    kpsi, ex = plan.apply(psi, occ, pair_mask=mask)
    e = plan.pair_energies()
    k_ref, ex_ref, e_ref = o.apply_masked(w["psi"].numpy(), occ, mask)
    scale = np.max(np.abs(k_ref))
    assert np.max(np.abs(kpsi.cpu().numpy() - k_ref)) <= K_RTOL * scale
    assert abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    live = mask & ((occ[:, None] != 0) | (occ[None, :] != 0))
    assert np.all((np.abs(e - e_ref) <= E_RTOL * np.max(np.abs(e_ref)))[live]) and not e[~live].any()
    assert float(kpsi[4].abs().max()) == 0.0
    # schedule listing agrees with the mask; a full mask is plain exx_apply; an asymmetric mask is refused
    rows = exx.exx_schedule_list(occ, 0, pair_mask=mask)
    got = {(j, i) for j, l, i, f, b in rows.tolist() if f & 1} | {(l, i) for j, l, i, f, b in rows.tolist() if f & 2}
    assert got == {(a, b) for a in range(n) for b in range(a, n) if live[a, b]}
    k_all, ex_all = plan.apply(psi, occ, pair_mask=np.ones((n, n)))
    k_std, ex_std = plan.apply(psi, occ)
    assert torch.equal(k_all, k_std) and ex_all == ex_std
    bad = np.ones((n, n))
    bad[1, 2] = 0
    with pytest.raises(exx.ExxError):
        plan.apply(psi, occ, pair_mask=bad)
    plan.destroy()


# ------------------------------------------------------------------ boundary: status codes that need a device
def test_boundary_status_paths_on_device():
    w = make_workload(small_spec("C1", dims=(16, 16, 16), n_orb=3, number=79))
    plan = exx.ExxPlan((16, 16, 16), w["spec"].spacing, "periodic", None, max_orbitals=3)
    lib = exx.load_library()
    dp = C.POINTER(C.c_double)
    psi = w["psi"].cuda()
    occ = np.array([2.0, 1.0, 0.5])
    ex = C.c_double()
    exp = C.cast(C.byref(ex), C.c_void_p)
    kpsi, ex_ok = plan.apply(psi, occ)
    M = 16 ** 3
    # pair energies: the caller states n_orb, a mismatch is an error (no silent overrun)
    buf = np.empty(9)
    assert lib.exx_get_pair_energies(plan.handle, 2, buf.ctypes.data_as(dp)) == 1
    assert lib.exx_get_pair_energies(plan.handle, 3, buf.ctypes.data_as(dp)) == 0
    assert lib.exx_get_block_energies(plan.handle, 3, 3, buf.ctypes.data_as(dp)) == 1     # last apply was not a block
    # misaligned psi (offset by one double) and partially overlapping kpsi are rejected, not faulted on
    big = torch.zeros(4 * M + 2, dtype=torch.float64, device="cuda")
    odd = C.c_void_p(big.data_ptr() + 8)
    k = torch.empty_like(psi)
    assert lib.exx_apply(plan.handle, 3, odd, occ.ctypes.data_as(dp), C.c_void_p(k.data_ptr()), exp) == 1
    assert b"aligned" in lib.exx_last_error(plan.handle)
    over = C.c_void_p(big.data_ptr() + 16 * (M // 2))
    assert lib.exx_apply(plan.handle, 3, C.c_void_p(big.data_ptr()), occ.ctypes.data_as(dp), over, exp) == 1
    assert b"overlap" in lib.exx_last_error(plan.handle)
    # an absurd batch size fails with EXX_ERR_ALLOC and leaves the plan fully usable with its previous workspace
    ws = plan.workspace_bytes()
    with pytest.raises(exx.ExxError) as ei:
        plan.set_batch(4096 * 4096)                                     # clamped to 4096 transforms -> still fits 16^3 ...
        big_plan = exx.ExxPlan((256, 256, 256), (0.3, 0.3, 0.3), "periodic", None, max_orbitals=2)
        try:
            big_plan.set_batch(4096)                                    # 4096 x 268 MB = 1.1 TB
        finally:
            assert big_plan.workspace_bytes() > 0
            k2, _ = big_plan.apply(torch.zeros((1, 256, 256, 256), dtype=torch.float64, device="cuda"), [1.0])
            big_plan.destroy()
    assert ei.value.status_name == "EXX_ERR_ALLOC"
    plan.set_batch(0)
    assert plan.workspace_bytes() == ws
    k3, ex3 = plan.apply(psi, occ)
    assert torch.equal(k3, kpsi) and ex3 == ex_ok
    # binding-side validation
    with pytest.raises(ValueError):
        plan.apply(psi, occ[:2])
    with pytest.raises(ValueError):
        plan.apply(psi, occ, kpsi=torch.empty((2, 16, 16, 16), dtype=torch.float64, device="cuda"))
    with pytest.raises(ValueError):
        plan.apply(psi.float(), occ)
    assert plan.device == torch.cuda.current_device()
    plan.destroy()
