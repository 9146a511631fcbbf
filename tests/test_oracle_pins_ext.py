"""Pins P11-P14 of the oracle functions behind the SURVEY.md 8(f) rows (no GPU): every function is tied to something
other than itself -- a closed form, an identity that reduces it to the already pinned exx_oracle_apply / poisson, or an
independently built table.

P11  exx_oracle_apply_to       K of the occupied set applied to another set (PAPER.md:67-69 Eq. 3; :210, :244)
P12  exx_oracle_apply_block    all pairs between two disjoint blocks (Fig. 1)
P13  exx_oracle_apply_masked   sparse pair list for localised orbitals (Eq. 6-7)
P14  periodic filter table     "only the filter F of kernel 2 would be different"
"""
import numpy as np
import pytest

from oracle import Oracle
from workloads import make_workload, small_spec


def _grid(dims, spacing):
    ax = [np.arange(n) * h for n, h in zip(dims, spacing)]
    return np.meshgrid(*ax, indexing="ij")


# ------------------------------------------------------------------------------------------------ P11 apply_to
def test_p11_apply_to_reduces_to_apply_when_sets_coincide():
    for base, dims in (("C1", (6, 8, 12)), ("C2", (4, 6, 8))):
        w = make_workload(small_spec(base, dims=dims, n_orb=4, spacing=(0.5, 0.45, 0.4), number=1101))
        spec = w["spec"]
        occ = np.array([2.0, 0.5, 0.0, 1.25])
        o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
        psi = w["psi"].numpy()
        k_ref, _, _ = o.apply(psi, occ, symmetric=False)
        k_to = o.apply_to(psi, occ, psi)
        assert np.max(np.abs(k_to - k_ref)) <= 1e-13 * np.max(np.abs(k_ref))


def test_p11_apply_to_two_cosine_closed_form():
    """Periodic box, occupied psi_1 = Vol^-1/2 (f_1), psi_2 = sqrt(2/Vol) cos(k2.r) (f_2); target phi = sqrt(2/Vol) cos(k.r):
    rho_1 = phi psi_1 = (sqrt2/Vol) cos(k.r)                      -> V_1 = (4 pi/k^2) rho_1
    rho_2 = phi psi_2 = (1/Vol)[cos((k+k2).r) + cos((k-k2).r)]    -> V_2 = (4 pi/Vol)[cos((k+k2).r)/|k+k2|^2 + cos((k-k2).r)/|k-k2|^2]
    K phi = -f_1 V_1 psi_1 - f_2 V_2 psi_2."""
    dims, spacing = (12, 8, 6), (0.4, 0.5, 0.45)
    L = [n * h for n, h in zip(dims, spacing)]
    vol = L[0] * L[1] * L[2]
    X, Y, Z = _grid(dims, spacing)
    kvec = lambda m: np.array([2 * np.pi * m[a] / L[a] for a in range(3)])
    k, k2 = kvec((2, 1, 0)), kvec((1, 0, 1))
    ph = lambda q: q[0] * X + q[1] * Y + q[2] * Z
    psi = np.stack([np.full(dims, vol ** -0.5), np.sqrt(2 / vol) * np.cos(ph(k2))])
    phi = (np.sqrt(2 / vol) * np.cos(ph(k)))[None]
    f1, f2 = 1.7, 0.6
    o = Oracle(dims, spacing, "periodic")
    got = o.apply_to(psi, [f1, f2], phi)[0]
    v1 = 4 * np.pi / (k @ k) * (np.sqrt(2) / vol) * np.cos(ph(k))
    kp, km = k + k2, k - k2
    v2 = 4 * np.pi / vol * (np.cos(ph(kp)) / (kp @ kp) + np.cos(ph(km)) / (km @ km))
    want = -f1 * v1 * psi[0] - f2 * v2 * psi[1]
    assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(want))


def test_p11_apply_to_is_linear_and_symmetric():
    w = make_workload(small_spec("C2", dims=(6, 4, 8), n_orb=5, spacing=(0.5, 0.45, 0.4), number=1102))
    spec = w["spec"]
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    all_orb = w["psi"].numpy()
    psi, phi = all_orb[:3], all_orb[3:]
    occ = np.array([2.0, 1.0, 0.3])
    kphi = o.apply_to(psi, occ, phi)
    combo = (0.7 * phi[0] - 1.9 * phi[1])[None]
    k_combo = o.apply_to(psi, occ, combo)[0]
    assert np.max(np.abs(k_combo - (0.7 * kphi[0] - 1.9 * kphi[1]))) <= 1e-13 * np.max(np.abs(kphi))
    # <phi_s | K phi_t> = <phi_t | K phi_s>   (K is a symmetric operator: the Green's function is even)
    m = np.einsum("sabc,tabc->st", phi, kphi)
    assert abs(m[0, 1] - m[1, 0]) <= 1e-13 * np.max(np.abs(m))
    assert m[0, 0] < 0 and m[1, 1] < 0                      # -sum_j f_j e_tj with e >= 0 for this kernel


# ------------------------------------------------------------------------------------------------ P12 apply_block
@pytest.mark.parametrize("base,dims", [("C1", (6, 6, 8)), ("C2", (4, 6, 4))])
def test_p12_block_is_union_minus_parts(base, dims):
    """apply(A u B) = apply(A) (+) apply(B) + block(A, B) for K psi, E_x and the pair-energy matrix."""
    w = make_workload(small_spec(base, dims=dims, n_orb=5, spacing=(0.5, 0.45, 0.4), number=1201))
    spec = w["spec"]
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    psi = w["psi"].numpy()
    occ = np.array([2.0, 0.7, 0.0, 1.3, 0.4])
    na = 2
    k_u, ex_u, e_u = o.apply(psi, occ, symmetric=False)
    k_a, ex_a, e_a = o.apply(psi[:na], occ[:na], symmetric=False)
    k_b, ex_b, e_b = o.apply(psi[na:], occ[na:], symmetric=False)
    ka, kb, ex_blk, e_blk = o.apply_block(psi[:na], occ[:na], psi[na:], occ[na:])
    scale = np.max(np.abs(k_u))
    assert np.max(np.abs(k_u[:na] - (k_a + ka))) <= 1e-13 * scale
    assert np.max(np.abs(k_u[na:] - (k_b + kb))) <= 1e-13 * scale
    assert abs(ex_u - (ex_a + ex_b + ex_blk)) <= 1e-13 * abs(ex_u)
    assert np.max(np.abs(e_u[:na, na:] - e_blk)) <= 1e-13 * np.max(np.abs(e_u))
    # swapping the roles of the blocks transposes the result
    kb2, ka2, ex2, e2 = o.apply_block(psi[na:], occ[na:], psi[:na], occ[:na])
    assert np.max(np.abs(ka2 - ka)) <= 1e-13 * scale and np.max(np.abs(kb2 - kb)) <= 1e-13 * scale
    assert abs(ex2 - ex_blk) <= 1e-13 * abs(ex_blk) and np.max(np.abs(e2.T - e_blk)) <= 1e-13 * np.max(np.abs(e_blk))


# ------------------------------------------------------------------------------------------------ P13 masked apply
def test_p13_mask_of_ones_and_block_diagonal_mask():
    w = make_workload(small_spec("C1", dims=(6, 8, 6), n_orb=5, spacing=(0.5, 0.45, 0.4), number=1301))
    spec = w["spec"]
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    psi = w["psi"].numpy()
    occ = np.array([2.0, 0.7, 1.1, 1.3, 0.4])
    k_ref, ex_ref, e_ref = o.apply(psi, occ, symmetric=False)
    k1, ex1, e1 = o.apply_masked(psi, occ, np.ones((5, 5)))
    assert np.array_equal(k1, k_ref) and ex1 == ex_ref and np.array_equal(e1, e_ref)
    # two groups that do not talk to each other = two independent systems
    groups = [[0, 3], [1, 2, 4]]
    mask = np.zeros((5, 5))
    for g in groups:
        mask[np.ix_(g, g)] = 1
    k_m, ex_m, e_m = o.apply_masked(psi, occ, mask)
    ex_sum = 0.0
    for g in groups:
        k_g, ex_g, e_g = o.apply(psi[g], occ[g], symmetric=False)
        assert np.max(np.abs(k_m[g] - k_g)) <= 1e-14 * np.max(np.abs(k_ref))
        assert np.max(np.abs(e_m[np.ix_(g, g)] - e_g)) <= 1e-14 * np.max(np.abs(e_ref))
        ex_sum += ex_g
    assert abs(ex_m - ex_sum) <= 1e-14 * abs(ex_ref)
    assert not e_m[mask == 0].any()
    # a single excluded pair removes exactly its two terms:  K psi_0 += f_3 V_03 psi_3,  E_x += f_0 f_3 e_03
    mask = np.ones((5, 5))
    mask[0, 3] = mask[3, 0] = 0
    k_x, ex_x, _ = o.apply_masked(psi, occ, mask)
    v03 = o.poisson(psi[0] * psi[3])
    assert np.max(np.abs(k_x[0] - (k_ref[0] + occ[3] * v03 * psi[3]))) <= 1e-13 * np.max(np.abs(k_ref))
    assert np.max(np.abs(k_x[3] - (k_ref[3] + occ[0] * v03 * psi[0]))) <= 1e-13 * np.max(np.abs(k_ref))
    assert abs(ex_x - (ex_ref + occ[0] * occ[3] * e_ref[0, 3])) <= 1e-13 * abs(ex_ref)


# ------------------------------------------------------------------------------------------------ P14 periodic filter table
def _sym_g2(dims, spacing):
    """|G|^2 on the symmetric index range, built here with numpy (independent of the oracle's index map)."""
    g = [2 * np.pi * np.arange(n // 2 + 1) / (n * h) for n, h in zip(dims, spacing)]
    return g[0][:, None, None] ** 2 + g[1][None, :, None] ** 2 + g[2][None, None, :] ** 2


def test_p14_coulomb_table_reproduces_the_analytic_kernel():
    dims, spacing = (6, 8, 12), (0.5, 0.4, 0.45)
    g2 = _sym_g2(dims, spacing)
    table = np.where(g2 > 0, 4 * np.pi / np.where(g2 > 0, g2, 1.0), 0.0)
    rng = np.random.default_rng(14)
    rho = rng.standard_normal(dims)
    v_tab = Oracle(dims, spacing, "periodic", table).poisson(rho)
    v_ana = Oracle(dims, spacing, "periodic").poisson(rho)
    assert np.max(np.abs(v_tab - v_ana)) <= 1e-14 * np.max(np.abs(v_ana))


def test_p14_screened_plane_wave_closed_form():
    """Short-range (erfc-screened) Coulomb filter K^(G) = (4 pi/G^2)(1 - exp(-G^2/(4 w^2))), K^(0) = pi/w^2:
    rho = cos(k.r) -> V = K^(k) cos(k.r).  Non-cubic grid, unequal spacings, k with three different indices: a
    transposed or mis-indexed table gives another K^(k)."""
    dims, spacing, omega = (12, 6, 8), (0.4, 0.5, 0.45), 0.11 * 4
    g2 = _sym_g2(dims, spacing)
    safe = np.where(g2 > 0, g2, 1.0)
    table = np.where(g2 > 0, 4 * np.pi / safe * (1 - np.exp(-safe / (4 * omega ** 2))), np.pi / omega ** 2)
    o = Oracle(dims, spacing, "periodic", table)
    L = [n * h for n, h in zip(dims, spacing)]
    X, Y, Z = _grid(dims, spacing)
    for m in ((3, 1, 2), (5, 0, 1), (0, 2, 3), (0, 0, 0)):
        k = np.array([2 * np.pi * m[a] / L[a] for a in range(3)])
        phase = k[0] * X + k[1] * Y + k[2] * Z
        rho = np.cos(phase)
        kk = k @ k
        khat = 4 * np.pi / kk * (1 - np.exp(-kk / (4 * omega ** 2))) if kk > 0 else np.pi / omega ** 2
        v = o.poisson(rho)
        assert np.max(np.abs(v - khat * rho)) <= 1e-13 * abs(khat)
    # negative-frequency half of the index range maps to the same table entry (even filter): sin component too
    k = np.array([2 * np.pi * 4 / L[0], 2 * np.pi * 2 / L[1], 2 * np.pi * 3 / L[2]])
    rho = np.sin(k[0] * X - k[1] * Y + k[2] * Z)
    kk = k @ k
    v = o.poisson(rho)
    assert np.max(np.abs(v - 4 * np.pi / kk * (1 - np.exp(-kk / (4 * omega ** 2))) * rho)) <= 1e-13 * (4 * np.pi / kk)


# ------------------------------------------------------------------------------------------------ P15 mixed BC (slab / wire)
def _even_table(rng, dims, periodic):
    """Random positive table, made even under index -> n - index along the periodic axes (what a Green's function is)."""
    g = rng.random(dims) + 0.1
    for ax in range(3):
        if periodic[ax]:
            g = 0.5 * (g + np.take(g, (-np.arange(dims[ax])) % dims[ax], axis=ax))
    return g


@pytest.mark.parametrize("dims,periodic", [((4, 6, 3), (1, 1, 0)), ((3, 4, 6), (0, 0, 1)), ((4, 3, 5), (1, 0, 1)), ((3, 4, 4), (0, 0, 0))])
def test_p15_point_charge_reads_the_table_with_wrap(dims, periodic):
    """A unit point charge at r0 gives V(r) = dV g(d(r, r0)): periodic axes wrap (roll), isolated axes take |r - r0|."""
    from oracle import poisson_direct_mixed
    rng = np.random.default_rng(1501)
    spacing = (0.5, 0.4, 0.3)
    g = _even_table(rng, dims, periodic)
    r0 = (dims[0] - 1, 1, dims[2] // 2)
    rho = np.zeros(dims)
    rho[r0] = 1.0
    got = poisson_direct_mixed(dims, spacing, periodic, g, rho)
    want = g
    for ax in range(3):
        n = dims[ax]
        idx = (np.arange(n) - r0[ax]) % n if periodic[ax] else np.abs(np.arange(n) - r0[ax])
        want = np.take(want, idx, axis=ax)
    want = want * np.prod(spacing)
    assert np.max(np.abs(got - want)) <= 1e-15 * np.max(np.abs(want))


@pytest.mark.parametrize("dims,periodic", [((4, 6, 3), (1, 1, 0)), ((3, 4, 6), (0, 0, 1)), ((4, 4, 4), (1, 1, 1))])
def test_p15_free_path_with_a_periodic_even_table_is_the_mixed_solver(dims, periodic):
    """The claim behind slab / wire support (A24): zero-padded (Hockney) convolution with table[|d|] equals the
    wrap-around convolution along every axis on which the table is even under d -> n - d."""
    from oracle import poisson_direct_mixed
    rng = np.random.default_rng(1502)
    spacing = (0.5, 0.4, 0.3)
    g = _even_table(rng, dims, periodic)
    rho = rng.standard_normal(dims)
    want = poisson_direct_mixed(dims, spacing, periodic, g, rho)
    got = Oracle(dims, spacing, "free", g).poisson(rho)
    assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(want))


def test_p15_all_axes_periodic_reproduces_the_periodic_solver():
    """With the real-space image of 4 pi/|G|^2 as the table, the mixed solver with three periodic axes -- by the direct
    sum and through the FREE path -- is the (pinned: P3, P4) periodic Poisson solver."""
    from oracle import poisson_direct_mixed
    dims, spacing = (4, 6, 4), (0.5, 0.4, 0.45)
    o = Oracle(dims, spacing, "periodic")
    table = o.realspace_kernel() / np.prod(spacing)
    rng = np.random.default_rng(1503)
    rho = rng.standard_normal(dims)
    want = o.poisson(rho)
    got_direct = poisson_direct_mixed(dims, spacing, (1, 1, 1), table, rho)
    got_free = Oracle(dims, spacing, "free", table).poisson(rho)
    scale = np.max(np.abs(want))
    assert np.max(np.abs(got_direct - want)) <= 1e-12 * scale
    assert np.max(np.abs(got_free - want)) <= 1e-12 * scale


def test_p15_screened_image_table_is_even_and_decays():
    from workloads import mixed_bc_kernel_table
    dims, spacing = (8, 6, 8), (0.5, 0.6, 0.5)
    g = mixed_bc_kernel_table(dims, spacing, (1, 0, 1), mu=2.0)
    for ax in (0, 2):
        assert np.array_equal(g, np.take(g, (-np.arange(dims[ax])) % dims[ax], axis=ax))
    assert g[0, 0, 0] > g[1, 0, 0] > g[2, 0, 0] > 0 and g[0, 5, 0] < 1e-3 * g[0, 1, 0]


# ------------------------------------------------------------------------------------------------ P16 general periodic cells
TRICLINIC = np.array([[4.0, 0.0, 0.0], [1.1, 3.6, 0.0], [-0.7, 0.9, 4.4]])


def test_p16_full_grid_filter_of_an_orthorhombic_cell_is_the_analytic_kernel():
    from workloads import general_cell_khat
    dims, spacing = (6, 4, 8), (0.5, 0.45, 0.4)
    lattice = np.diag([n * h for n, h in zip(dims, spacing)])
    khat, vol = general_cell_khat(dims, lattice)
    rng = np.random.default_rng(1601)
    rho = rng.standard_normal(dims)
    want = Oracle(dims, spacing, "periodic").poisson(rho)
    got = Oracle.general(dims, vol, khat).poisson(rho)
    assert abs(vol - np.prod(lattice.diagonal())) <= 1e-12 * vol
    assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(want))


def test_p16_triclinic_plane_waves_read_their_own_table_entry():
    """rho = cos / sin of the plane wave with FFT index m on the index grid -> V = K^[m] rho: the entry of exactly that
    index (an asymmetric table would expose a transposed or mirrored lookup), for a cosine and -- since K^(-m) = K^(m) --
    for a sine."""
    from workloads import general_cell_khat
    dims = (6, 8, 10)
    khat, vol = general_cell_khat(dims, TRICLINIC)
    o = Oracle.general(dims, vol, khat)
    i, j, k = np.meshgrid(*[np.arange(n) for n in dims], indexing="ij")
    for m in [(1, 2, 3), (5, 1, 0), (2, 7, 9), (0, 3, 8)]:
        theta = 2 * np.pi * (m[0] * i / dims[0] + m[1] * j / dims[1] + m[2] * k / dims[2])
        for f in (np.cos, np.sin):
            v = o.poisson(f(theta))
            assert np.max(np.abs(v - khat[m] * f(theta))) <= 1e-13 * khat[m]
    # the table is not even in each index separately (that is what makes the cell "general") but inversion-symmetric
    assert abs(khat[1, 2, 3] - khat[5, 2, 3]) > 1e-3 * khat[1, 2, 3]
    assert khat[1, 2, 3] == khat[5, 6, 7]


def test_p16_triclinic_fft_path_is_the_brute_force_convolution():
    from workloads import general_cell_khat
    dims = (4, 6, 4)
    khat, vol = general_cell_khat(dims, TRICLINIC)
    o = Oracle.general(dims, vol, khat)
    rng = np.random.default_rng(1602)
    rho = rng.standard_normal(dims)
    v, vd = o.poisson(rho), o.poisson_direct(rho)
    assert np.max(np.abs(v - vd)) <= 1e-12 * np.max(np.abs(v))


def test_p16_triclinic_coulomb_entry_is_four_pi_over_g_squared():
    """One entry of the seeded table against the textbook reciprocal-lattice construction b1 = 2 pi (a2 x a3) / V, ..."""
    from workloads import general_cell_khat
    dims = (6, 8, 10)
    khat, vol = general_cell_khat(dims, TRICLINIC)
    a1, a2, a3 = TRICLINIC
    v = float(np.dot(a1, np.cross(a2, a3)))
    b1, b2, b3 = (2 * np.pi * np.cross(a2, a3) / v, 2 * np.pi * np.cross(a3, a1) / v, 2 * np.pi * np.cross(a1, a2) / v)
    g = 1 * b1 + (-2) * b2 + 3 * b3                      # index (1, 6, 3) <-> frequencies (1, -2, 3)
    assert abs(vol - abs(v)) <= 1e-12 * abs(v)
    assert abs(khat[1, 6, 3] - 4 * np.pi / np.dot(g, g)) <= 1e-13 * khat[1, 6, 3]


# ------------------------------------------------------------------------------------------------ P17 complex orbitals
def _complex_set(seed, dims, n):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n,) + dims) + 1j * rng.standard_normal((n,) + dims)


def test_p17_real_orbitals_reduce_to_the_real_apply():
    for bc, dims in (("periodic", (6, 4, 8)), ("free", (4, 6, 4))):
        w = make_workload(small_spec("C1" if bc == "periodic" else "C2", dims=dims, n_orb=3, spacing=(0.5, 0.45, 0.4), number=1701))
        o = Oracle(dims, w["spec"].spacing, bc, w["kernel"])
        occ = np.array([2.0, 0.0, 1.1])
        k_ref, ex_ref, _ = o.apply(w["psi"].numpy(), occ)
        k, ex = o.apply_complex(w["psi"].numpy().astype(np.complex128), occ)
        assert np.max(np.abs(k.imag)) == 0.0
        assert np.max(np.abs(k.real - k_ref)) <= 1e-13 * np.max(np.abs(k_ref))
        assert abs(ex - ex_ref) <= 1e-13 * abs(ex_ref)


def test_p17_plane_wave_exchange_closed_form():
    """psi_n = Vol^-1/2 exp(i k_n.r): rho_ij = exp(i (k_i - k_j).r) / Vol, V_ij = 4 pi / |k_i - k_j|^2 rho_ij (0 for i = j), so
    K psi_i = - [sum_{j != i} f_j 4 pi / (|k_i - k_j|^2 Vol)] psi_i  and  E_x = -1/2 sum_{i != j} f_i f_j 4 pi / (|k_i - k_j|^2 Vol):
    the textbook exchange of plane waves.  A missing conjugate turns k_i - k_j into k_i + k_j."""
    dims, spacing = (8, 6, 10), (0.5, 0.45, 0.4)
    L = np.array([n * h for n, h in zip(dims, spacing)])
    vol = float(np.prod(L))
    ms = [(1, 0, 2), (2, 1, 0), (-1, 2, 1)]
    ks = [2 * np.pi * np.array(m) / L for m in ms]
    X, Y, Z = _grid(dims, spacing)
    psi = np.stack([np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z)) / np.sqrt(vol) for k in ks])
    occ = np.array([2.0, 1.0, 0.5])
    k_got, ex_got = Oracle(dims, spacing, "periodic").apply_complex(psi, occ)
    ex_want = 0.0
    for i in range(3):
        lam = sum(occ[j] * 4 * np.pi / (np.dot(ks[i] - ks[j], ks[i] - ks[j]) * vol) for j in range(3) if j != i)
        assert np.max(np.abs(k_got[i] + lam * psi[i])) <= 1e-13 * lam * np.max(np.abs(psi[i]))
        ex_want -= 0.5 * occ[i] * lam
    assert abs(ex_got - ex_want) <= 1e-13 * abs(ex_want)


def test_p17_phase_covariance_hermiticity_and_energy_identity():
    dims, spacing = (4, 6, 4), (0.5, 0.45, 0.4)
    w = make_workload(small_spec("C2", dims=dims, n_orb=3, spacing=spacing, number=1702))
    o = Oracle(dims, spacing, "free", w["kernel"])
    psi = _complex_set(1703, dims, 3)
    occ = np.array([2.0, 0.8, 1.4])
    k, ex = o.apply_complex(psi, occ)
    # every orbital may carry its own phase: K (e^{i t_i} psi_i) = e^{i t_i} K psi_i, E_x unchanged
    ph = np.exp(1j * np.array([0.3, -1.1, 2.0]))[:, None, None, None]
    k2, ex2 = o.apply_complex(ph * psi, occ)
    assert np.max(np.abs(k2 - ph * k)) <= 1e-12 * np.max(np.abs(k))
    assert abs(ex2 - ex) <= 1e-12 * abs(ex)
    # <psi_a|K psi_b> is Hermitian;  E_x = 1/2 dV sum f_i Re<psi_i|K psi_i> <= 0
    m = np.einsum("axyz,bxyz->ab", np.conj(psi), k)
    assert np.max(np.abs(m - m.conj().T)) <= 1e-12 * np.max(np.abs(m))
    assert ex < 0 and abs(ex - 0.5 * o.dV * float(np.sum(occ * np.diag(m).real))) <= 1e-12 * abs(ex)


def test_p17_cross_apply_reduces_to_apply_to_and_is_linear_in_the_partner():
    dims, spacing = (4, 6, 4), (0.5, 0.45, 0.4)
    w = make_workload(small_spec("C2", dims=dims, n_orb=5, spacing=spacing, number=1704))
    o = Oracle(dims, spacing, "free", w["kernel"])
    allp = w["psi"].numpy()
    psi, phi = allp[:3], allp[3:]
    occ = np.array([2.0, 0.0, 1.3])
    assert np.max(np.abs(o.apply_to_cross(psi, psi, occ, phi) - o.apply_to(psi, occ, phi))) <= 1e-13 * np.max(np.abs(phi))
    rng = np.random.default_rng(1705)
    c1, c2 = rng.standard_normal(psi.shape), rng.standard_normal(psi.shape)
    lhs = o.apply_to_cross(psi, 2.0 * c1 - 0.5 * c2, occ, phi)
    rhs = 2.0 * o.apply_to_cross(psi, c1, occ, phi) - 0.5 * o.apply_to_cross(psi, c2, occ, phi)
    assert np.max(np.abs(lhs - rhs)) <= 1e-12 * np.max(np.abs(rhs))
