"""GPU parity: the CUDA path (through the C ABI) vs the CPU oracle on the same seeded inputs.  Needs a B200.

Tolerances are north_star's: |E_gpu - E_orc| <= 1e-11 |E_orc|;  max|dKpsi| <= 1e-10 max|Kpsi_orc|;
pair energies: 1e-11 * max(|e_ij|, 1e-3 sqrt(e_ii e_jj)).
"""
import os

import numpy as np
import pytest
import torch

import paper_1712_07973_b200 as exx
from oracle import Oracle
from workloads import CONFIGS, make_workload, small_spec

pytestmark = pytest.mark.gpu

E_RTOL = 1e-11
K_RTOL = 1e-10


def _run_gpu(w, occ=None, batch=None):
    spec = w["spec"]
    occ = w["occ"] if occ is None else occ
    psi = w["psi"].cuda()
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=spec.n_orb)
    if batch:
        plan.set_batch(batch)
    kpsi, ex = plan.apply(psi, occ)
    e = plan.pair_energies(spec.n_orb)
    torch.cuda.synchronize()
    return plan, psi, kpsi, ex, e


def _pair_tol(e_ref, diag=None):
    d = np.sqrt(np.abs(np.diag(e_ref) if diag is None else diag))
    return E_RTOL * np.maximum(np.abs(e_ref), 1e-3 * d[:, None] * d[None, :])


def _check_full(w, occ=None, symmetric=True, batch=None):
    spec = w["spec"]
    occ = np.asarray(w["occ"] if occ is None else occ, dtype=np.float64)
    plan, psi, kpsi, ex, e = _run_gpu(w, occ, batch)
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    k_ref, ex_ref, e_ref = o.apply(w["psi"].numpy(), occ, symmetric=symmetric)
    scale = np.max(np.abs(k_ref))
    assert np.max(np.abs(kpsi.cpu().numpy() - k_ref)) <= K_RTOL * scale
    assert abs(ex - ex_ref) <= E_RTOL * abs(ex_ref)
    live = (occ[:, None] != 0) | (occ[None, :] != 0)        # a pair with f_i = f_j = 0 is skipped and reads 0 (A15)
    # the tolerance floor needs every self-energy e_ii; the oracle's symmetric mode skips the doubly-empty ones
    n = len(occ)
    diag = o.pair_energies(w["psi"].numpy(), [(i, i) for i in range(n)]) if symmetric and np.any(occ == 0) else None
    assert np.all((np.abs(e - e_ref) <= _pair_tol(e_ref, diag))[live])
    assert not e[~live].any()
    assert np.array_equal(e, e.T)
    plan.destroy()
    return ex


# ------------------------------------------------------------------ full element-by-element comparisons
def test_c1_full_definition():
    """BASELINE.json configs[0]: periodic 32^3, 8 orbitals, all N^2 ordered pairs in the oracle."""
    _check_full(make_workload("C1"), symmetric=False)


@pytest.mark.parametrize("dims", [(16, 16, 16), (16, 32, 64), (64, 16, 32), (32, 64, 16), (64, 64, 64)])
def test_periodic_small_and_mixed(dims):
    w = make_workload(small_spec("C1", dims=dims, n_orb=5, spacing=(0.45, 0.4, 0.5), number=40 + sum(dims)))
    _check_full(w, occ=[2.0, 1.0, 0.5, 2.0, 1.5], symmetric=False)


@pytest.mark.parametrize("dims", [(8, 8, 8), (16, 16, 16), (8, 16, 32), (32, 8, 16), (16, 32, 8), (32, 32, 32)])
def test_free_small_and_mixed(dims):
    w = make_workload(small_spec("C2", dims=dims, n_orb=4, spacing=(0.5, 0.45, 0.4), number=60 + sum(dims)))
    _check_full(w, occ=[2.0, 1.0, 0.5, 2.0], symmetric=False)


def test_edge_cases_occupations_and_batching():
    w = make_workload(small_spec("C1", dims=(16, 16, 16), n_orb=7, number=77))
    # zero occupations (pairs with f_i = f_j = 0 skipped), odd pair counts, batch size 1 and 2 (rows split)
    occ = [2.0, 0.0, 1.0, 0.0, 0.0, 0.3, 1.7]
    ex_a = _check_full(w, occ=occ, symmetric=False)
    ex_b = _check_full(w, occ=occ, symmetric=False, batch=1)
    ex_c = _check_full(w, occ=occ, symmetric=False, batch=2)
    assert abs(ex_a - ex_b) <= 1e-13 * abs(ex_a) and abs(ex_a - ex_c) <= 1e-13 * abs(ex_a)
    # imaginary-slot-only transforms (f_j = f_i = 0, f_l != 0) and an even N with empty block-rows
    w8 = make_workload(small_spec("C2", dims=(8, 16, 8), n_orb=8, number=76))
    _check_full(w8, occ=[0.0, 1.2, 0.0, 0.0, 2.0, 0.0, 0.0, 0.7], symmetric=False, batch=3)
    # N = 1: Hartree special case
    w1 = make_workload(small_spec("C1", dims=(16, 16, 16), n_orb=1, number=78))
    _check_full(w1, occ=[1.3], symmetric=False)
    # all occupations zero: nothing to do, K psi = 0, E_x = 0
    plan, psi, kpsi, ex, e = _run_gpu(w, occ=[0.0] * 7)
    assert ex == 0.0 and float(kpsi.abs().max()) == 0.0 and not e.any()
    plan.destroy()


def test_apply_is_repeatable_and_overwrites():
    w = make_workload("C1")
    spec = w["spec"]
    psi = w["psi"].cuda()
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, None, max_orbitals=spec.n_orb)
    k1 = torch.full_like(psi, 123.0)
    k1, ex1 = plan.apply(psi, w["occ"], k1)
    k2, ex2 = plan.apply(psi, w["occ"])
    assert torch.equal(k1, k2) and ex1 == ex2           # deterministic, output overwritten not accumulated
    # async variant and host-buffer variant agree
    ex_dev = torch.zeros(1, dtype=torch.float64, device="cuda")
    k3 = torch.empty_like(psi)
    plan.apply_async(psi, w["occ"], k3, ex_dev)
    torch.cuda.synchronize()
    assert torch.equal(k3, k1) and float(ex_dev[0]) == ex1
    k4, ex4 = plan.apply_host(w["psi"].numpy(), w["occ"])
    assert np.array_equal(k4, k1.cpu().numpy()) and ex4 == ex1
    assert plan.launch_count() > 0 and plan.workspace_bytes() > 0
    plan.destroy()


@pytest.mark.parametrize("base,dims", [("C1", (96, 96, 96)), ("C2", (48, 48, 48))])
def test_warp_specialised_kernels_repeat_bitwise(base, dims):
    """Transform length 96: all three passes run their warp-specialised kernels (mbarrier hand-over between warp
    roles).  A race there shows up as run-to-run differences: five applies, several batch cuts, bit-identical."""
    w = make_workload(small_spec(base, dims=dims, n_orb=7, number=91))
    spec = w["spec"]
    psi = w["psi"].cuda()
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=spec.n_orb)
    ref_k, ref_ex = plan.apply(psi, w["occ"])
    ref_k = ref_k.clone()
    for batch in (0, 1, 2, 3, 5):
        plan.set_batch(batch)
        k, ex = plan.apply(psi, w["occ"])
        if batch == 0:
            assert torch.equal(k, ref_k) and ex == ref_ex
        else:                                               # other batch cuts change the accumulation order of K psi_j only
            assert float((k - ref_k).abs().max()) <= 1e-13 * float(ref_k.abs().max())
            k2, ex2 = plan.apply(psi, w["occ"])
            assert torch.equal(k, k2) and ex == ex2
    plan.destroy()


@pytest.mark.parametrize("base,dims", [("C1", (96, 96, 96)), ("C2", (48, 48, 48))])
def test_warp_specialised_kernels_edge_schedule(base, dims):
    """Odd N, zero occupations (absent real / imaginary slots, skipped transforms) and one- and three-transform batches
    through the warp-specialised kernels, element by element against the oracle's N^2 definition."""
    w = make_workload(small_spec(base, dims=dims, n_orb=7, number=92))
    occ = [0.0, 1.2, 0.0, 2.0, 0.0, 0.0, 0.7]
    ex_a = _check_full(w, occ=occ, symmetric=False)
    ex_b = _check_full(w, occ=occ, symmetric=False, batch=1)
    ex_c = _check_full(w, occ=occ, symmetric=False, batch=3)
    assert abs(ex_a - ex_b) <= 1e-13 * abs(ex_a) and abs(ex_a - ex_c) <= 1e-13 * abs(ex_a)


@pytest.mark.parametrize("base,dims,n_orb,batch", [("C1", (32, 32, 32), 5, 2), ("C1", (96, 96, 96), 5, 3), ("C2", (48, 48, 48), 4, 0),
                                                   ("C1", (192, 96, 48), 3, 2), ("C2", (16, 64, 32), 3, 0),
                                                   ("C1", (192, 192, 192), 3, 2), ("C2", (128, 128, 128), 2, 0)])   # TMA tile gather
def test_guard_bands_and_poisoned_outputs(base, dims, n_orb, batch):
    """Memory-safety evidence that needs no tool (compute-sanitizer is closed on this pool): psi and K psi live in the
    middle of larger allocations whose guard bands hold a sentinel, K psi starts as NaN, and E_x / e_ij start as NaN.
    After the apply the guard bands and psi must be bit-for-bit what they were (no stray store, no stray reduce-add:
    an add onto the sentinel would change it), and the outputs must be finite everywhere and equal to those of a plain
    run (every output element was written, nothing read an output before writing it)."""
    w = make_workload(small_spec(base, dims=dims, n_orb=n_orb, number=1300 + sum(dims)))
    spec = w["spec"]
    m = spec.n_orb * spec.n_points
    guard = 1 << 16
    sentinel = 1.2345678901234567e+100
    buf_p = torch.full((m + 2 * guard,), sentinel, dtype=torch.float64, device="cuda")
    buf_k = torch.full((m + 2 * guard,), sentinel, dtype=torch.float64, device="cuda")
    psi = buf_p[guard:guard + m].view(spec.n_orb, *spec.dims)
    kpsi = buf_k[guard:guard + m].view(spec.n_orb, *spec.dims)
    psi.copy_(w["psi"].cuda())
    psi_before = psi.clone()
    kpsi.fill_(float("nan"))
    ex_dev = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=spec.n_orb)
    if batch:
        plan.set_batch(batch)
    occ = np.array([2.0, 1.0, 0.0, 0.5, 1.5][:n_orb])
    plan.apply_async(psi, occ, kpsi, ex_dev)
    torch.cuda.synchronize()
    for buf in (buf_p, buf_k):
        assert bool((buf[:guard] == sentinel).all()) and bool((buf[guard + m:] == sentinel).all())
    assert torch.equal(psi, psi_before)
    assert bool(torch.isfinite(kpsi).all()) and bool(torch.isfinite(ex_dev).all())
    k_plain, ex_plain = plan.apply(w["psi"].cuda(), occ)
    assert torch.equal(kpsi, k_plain) and float(ex_dev[0]) == ex_plain
    plan.destroy()


def test_pointer_and_argument_errors():
    w = make_workload(small_spec("C1", dims=(16, 16, 16), n_orb=2, number=79))
    plan = exx.ExxPlan((16, 16, 16), w["spec"].spacing, "periodic", None, max_orbitals=2)
    psi = w["psi"].cuda()
    import ctypes as C
    lib = exx.load_library()
    occ = np.array([2.0, 2.0])
    ex = C.c_double()
    host = w["psi"].numpy()
    dp = C.POINTER(C.c_double)
    # host pointer where a device pointer is required
    st = lib.exx_apply(plan.handle, 2, C.c_void_p(host.ctypes.data), occ.ctypes.data_as(dp), C.c_void_p(psi.data_ptr()),
                       C.cast(C.byref(ex), C.c_void_p))
    assert st == 3
    k = torch.empty_like(psi)
    st = lib.exx_apply(plan.handle, 3, C.c_void_p(psi.data_ptr()), occ.ctypes.data_as(dp), C.c_void_p(k.data_ptr()),
                       C.cast(C.byref(ex), C.c_void_p))
    assert st == 1                                       # n_orb > max_orbitals
    st = lib.exx_apply(plan.handle, 2, C.c_void_p(psi.data_ptr()), occ.ctypes.data_as(dp), C.c_void_p(psi.data_ptr()),
                       C.cast(C.byref(ex), C.c_void_p))
    assert st == 1                                       # aliasing
    plan.destroy()


# ------------------------------------------------------------------ every supported transform length
@pytest.mark.parametrize("bc,n,n_orb", [("periodic", 96, 4), ("periodic", 128, 3), ("periodic", 192, 3),
                                        ("free", 48, 4), ("free", 64, 4), ("free", 96, 3), ("free", 128, 2),
                                        ("periodic", 256, 2)])
def test_every_length(bc, n, n_orb):
    base = "C1" if bc == "periodic" else "C2"
    w = make_workload(small_spec(base, dims=(n, n, n), n_orb=n_orb, spacing=(0.3, 0.3, 0.3), number=200 + n))
    _check_full(w, occ=[2.0, 1.0, 1.5, 0.5][:n_orb], symmetric=True)


# ------------------------------------------------------------------ lengths and mixes added in round 2 (reading A9)
@pytest.mark.parametrize("bc,dims,n_orb", [("periodic", (48, 48, 48), 4), ("periodic", (144, 144, 144), 3), ("free", (24, 24, 24), 4),
                                           ("free", (72, 72, 72), 3), ("periodic", (24, 24, 24), 5), ("free", (12, 12, 12), 4),
                                           ("periodic", (72, 72, 72), 3), ("free", (36, 36, 36), 3)])
def test_new_lengths(bc, dims, n_orb):
    """Transform lengths 48 = 4*12, 144 = 12*12 (main: free mixes too) and 24 = 2*12, 72 = 6*12 (cubic transform grids)."""
    base = "C1" if bc == "periodic" else "C2"
    w = make_workload(small_spec(base, dims=dims, n_orb=n_orb, spacing=(0.3, 0.35, 0.3), number=400 + sum(dims)))
    _check_full(w, occ=[2.0, 1.0, 1.5, 0.5, 0.7][:n_orb], symmetric=True, batch=2)


@pytest.mark.parametrize("bc,dims,n_orb", [("periodic", (96, 128, 192), 3), ("periodic", (192, 96, 48), 3), ("periodic", (16, 256, 144), 3),
                                           ("free", (64, 96, 128), 2), ("free", (96, 16, 72), 3), ("free", (24, 128, 48), 3),
                                           ("periodic", (256, 32, 96), 3)])
def test_noncubic_large_grids(bc, dims, n_orb):
    """Non-cubic grids with lengths above 64 on every axis role (a: pass B lines, b: split middle axis, c: contiguous):
    each (TA, TB) picks its own W1 chunk, each (TC, TB, chunk) its own pass A / C instantiation."""
    base = "C1" if bc == "periodic" else "C2"
    w = make_workload(small_spec(base, dims=dims, n_orb=n_orb, spacing=(0.3, 0.35, 0.4), number=450 + sum(dims)))
    _check_full(w, occ=[2.0, 1.0, 1.5][:n_orb], symmetric=True, batch=2)


# ------------------------------------------------------------------ large lengths, multi-batch block-rows, element by element
@pytest.mark.parametrize("bc,n,n_orb,batch", [("periodic", 192, 9, 4), ("free", 128, 9, 4)])
def test_large_lengths_multibatch_full(bc, n, n_orb, batch):
    """T = 192 (periodic 192^3) and T = 256 (free 128^3 -> 256^3) with N = 9 orbitals and batches of 4 transforms: the
    first block-rows are cut into 3 / 2 batches (9, 7, 5 ... streamed orbitals), the last one is the odd tail {8}, so the
    batch cuts, the scratch pass B and pass C of those lengths are compared element by element with the oracle."""
    base = "C1" if bc == "periodic" else "C2"
    w = make_workload(small_spec(base, dims=(n, n, n), n_orb=n_orb, spacing=(0.3, 0.3, 0.3), number=300 + n))
    occ = [2.0, 1.0, 1.5, 0.5, 2.0, 0.0, 1.25, 0.75, 1.0][:n_orb]
    _check_full(w, occ=occ, symmetric=True, batch=batch)


# ------------------------------------------------------------------ full-size configs, sampled (SURVEY.md 8(d) protocol)
def _check_sampled(name, rows, n_pairs, point_orbs, seed):
    """rows: orbitals i whose complete K psi_i (all j) and e_i* come from the oracle; n_pairs seeded random pair
    energies; point_orbs: orbitals of the sampled K psi entries (one seeded random grid point each), computed by the
    oracle's direct real-space sum."""
    w = make_workload(name, device="cuda")
    spec = w["spec"]
    psi = w["psi"]
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=spec.n_orb)
    kpsi, ex = plan.apply(psi, w["occ"])
    e = plan.pair_energies(spec.n_orb)
    occ = w["occ"]
    n_orb = spec.n_orb
    # (iii) global identities on the GPU result: a missed or doubled pair breaks these
    ex_from_e = -0.5 * np.einsum("i,j,ij->", occ, occ, e)
    assert abs(ex_from_e - ex) <= 1e-12 * abs(ex)
    ex_from_k = 0.5 * spec.dV * float(sum(occ[i] * torch.sum(psi[i] * kpsi[i]) for i in range(n_orb)))
    assert abs(ex_from_k - ex) <= 1e-11 * abs(ex)
    assert np.array_equal(e, e.T) and ex < 0
    assert plan_pairs(occ) == spec.n_pairs
    # oracle on sampled outputs
    psi_h = psi.cpu().numpy()
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    rng = np.random.default_rng(seed)
    kmax = float(kpsi.abs().max())
    d = np.sqrt(np.abs(np.diag(e)))
    if rows:
        rows = sorted(int(r) for r in rows)
        k_rows, e_rows = o.rows(psi_h, occ, rows)
        for s, i in enumerate(rows):
            assert np.max(np.abs(kpsi[i].cpu().numpy() - k_rows[s])) <= K_RTOL * kmax
            tol = E_RTOL * np.maximum(np.abs(e_rows[s]), 1e-3 * d[i] * d)
            assert np.all(np.abs(e[i] - e_rows[s]) <= tol)
    if n_pairs:
        pairs = [(int(a), int(b)) for a, b in rng.integers(0, n_orb, size=(n_pairs, 2))]
        e_ref = o.pair_energies(psi_h, pairs)
        for (a, b), er in zip(pairs, e_ref):
            assert abs(e[a, b] - er) <= E_RTOL * max(abs(er), 1e-3 * d[a] * d[b])
    if len(point_orbs):
        orbs = np.asarray(point_orbs, dtype=np.int64)
        pts = rng.integers(0, spec.n_points, size=orbs.size)
        ref = o.kpsi_points(psi_h, occ, orbs, pts)
        got = np.array([float(kpsi[int(i)].reshape(-1)[int(p)]) for i, p in zip(orbs, pts)])
        assert np.max(np.abs(got - ref)) <= K_RTOL * kmax
    plan.destroy()


def plan_pairs(occ):
    return exx.exx_schedule_pairs(occ)[0]


def _spread_orbitals(n_orb, count):
    """Orbitals from the first, a middle and the last block-rows (both members of a block-row), then evenly spread: the
    first block-row is cut into the most batches, the last ones are shorter than one batch, and at C5 the rows beyond
    orbital 75 start more than 4 GiB into psi / K psi."""
    fixed = [0, 1, n_orb // 2 - 1, n_orb // 2, n_orb - 2, n_orb - 1]
    rest = np.linspace(2, n_orb - 3, max(0, count - len(fixed))).astype(int).tolist()
    return (fixed + rest)[:count]


def test_c2_full_size_sampled():
    """BASELINE.json configs[1]: free 64^3 -> 128^3, 32 orbitals, 528 pairs."""
    _check_sampled("C2", rows=[3, 30], n_pairs=16, point_orbs=_spread_orbitals(32, 8), seed=2)


def test_c3_full_size_sampled():
    """BASELINE.json configs[2]: periodic 96^3, 128 Loewdin-orthonormal orbitals, 8256 pairs."""
    _check_sampled("C3", rows=[0, 77], n_pairs=64, point_orbs=_spread_orbitals(128, 16), seed=3)


def test_c4_full_size_sampled():
    """BASELINE.json configs[3]: free 128^3 -> 256^3, 256 orbitals, 32896 pairs: one complete oracle row (256 solves),
    64 pair energies, 16 K psi entries."""
    _check_sampled("C4", rows=[131], n_pairs=64, point_orbs=_spread_orbitals(256, 16), seed=4)


def _c5_fits():
    """C5 needs ~125 GB of device memory (psi, K psi, workspace) and a 58 GB host copy of psi for the oracle."""
    if os.environ.get("EXX_TEST_C5") == "0" or not torch.cuda.is_available():
        return False
    try:
        host_gb = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES") / 1e9
    except (ValueError, OSError):
        host_gb = 0.0
    return torch.cuda.get_device_properties(0).total_memory / 1e9 >= 150 and host_gb >= 120


@pytest.mark.skipif(not _c5_fits(), reason="C5 needs >= 150 GB of device memory and >= 120 GB of host memory (EXX_TEST_C5=0 skips it)")
def test_c5_full_size_sampled():
    """BASELINE.json configs[4] (the bench workload): periodic 192^3, 1024 orbitals, 524800 pairs.  One complete oracle
    row (1024 solves; orbital 517 is streamed by 258 block-rows and resident in its own), 64 pair energies and 32 K psi
    entries on orbitals of the first, a middle and the last block-rows (offsets beyond 4 GiB, every batch cut)."""
    _check_sampled("C5", rows=[517], n_pairs=64, point_orbs=_spread_orbitals(1024, 32), seed=5)
