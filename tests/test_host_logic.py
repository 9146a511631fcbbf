"""Host-side logic of the CUDA library that needs no GPU: exported symbols, scheduler counts, argument checks."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_1712_07973_b200 as exx
from paper_1712_07973_b200.binding import EXPORTS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLDEN = os.path.join(ROOT, "tests", "golden")


def test_library_loads_and_exports_every_declared_symbol():
    lib = exx.load_library()
    header = open(os.path.join(ROOT, "include", "exx.h")).read()
    declared = set(re.findall(r"\b(exx_[a-z0-9_]+)\s*\(", header))
    declared -= {"exx_plan", "exx_status", "exx_bc"}
    assert declared, "no declarations found in include/exx.h"
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in include/exx.h but not exported"
    assert declared == set(EXPORTS), "binding.EXPORTS out of sync with include/exx.h"
    assert "sm_100a" in exx.exx_version()


def test_p10_pair_counts_match_table1():
    """Scheduler count = N(N+1)/2 = PAPER.md:179-185 Table 1 (H2O columns)."""
    rows = [line.split() for line in open(os.path.join(GOLDEN, "table1_pair_counts.txt")) if line[0].isdigit()]
    assert len(rows) == 4
    for n_orb, solves in rows:
        n_orb, solves = int(n_orb), int(solves)
        n_pairs, n_x = exx.exx_schedule_pairs([2.0] * n_orb)
        assert n_pairs == solves == n_orb * (n_orb + 1) // 2
        # block-row {j, j+1} holds one transform per streamed orbital i >= j (i = j carries only the diagonal pair)
        assert n_x == sum(n_orb - j for j in range(0, n_orb, 2))


def test_scheduler_skips_only_doubly_empty_pairs():
    occ = [2.0, 0.0, 1.0, 0.0, 0.0]
    n_pairs, n_x = exx.exx_schedule_pairs(occ)
    expect = sum(1 for i in range(5) for j in range(i, 5) if not (occ[i] == 0 and occ[j] == 0))
    assert n_pairs == expect == 9
    assert exx.exx_schedule_pairs([0.0, 0.0]) == (0, 0)
    assert exx.exx_schedule_pairs([1.0]) == (1, 1)


@pytest.mark.parametrize("occ,max_batch", [([2.0] * 7, 0), ([2.0] * 8, 3), ([2.0, 0.0, 1.0, 0.0, 0.0, 1.5], 2), ([0.0, 0.0, 1.0], 0),
                                           ([1.0], 0), ([2.0] * 33, 5)])
def test_schedule_covers_every_pair_exactly_once(occ, max_batch):
    """Row-pair schedule (include/exx.h exx_schedule_list): every unordered pair that is not doubly empty is carried by
    exactly one transform slot; batches share (j,l), never stream j or l as an update target twice, and respect max_batch."""
    n = len(occ)
    rows = exx.exx_schedule_list(occ, max_batch)
    seen = {}
    per_batch = {}
    for j, l, i, flags, b in rows.tolist():
        assert flags in (1, 2, 3) and 0 <= j <= i < n and (l == -1 or l == j + 1)
        per_batch.setdefault(b, []).append((j, l, i))
        if flags & 1:
            seen[(j, i)] = seen.get((j, i), 0) + 1
        if flags & 2:
            assert l >= 0 and i >= l
            seen[(l, i)] = seen.get((l, i), 0) + 1
    expect = {(x, y) for x in range(n) for y in range(x, n) if not (occ[x] == 0 and occ[y] == 0)}
    assert set(seen) == expect and all(v == 1 for v in seen.values())
    assert exx.exx_schedule_pairs(occ) == (len(expect), len(rows))
    for b, items in per_batch.items():
        assert len({(j, l) for j, l, _ in items}) == 1, "a batch shares its resident orbitals"
        streamed = [i for _, _, i in items]
        assert len(set(streamed)) == len(streamed), "K psi_i targets of a batch are distinct"
        if max_batch > 0:
            assert len(items) <= max_batch


def test_status_codes_without_compute():
    lib = exx.load_library()
    assert lib.exx_status_string(0) == b"EXX_OK"
    assert lib.exx_status_string(2) == b"EXX_ERR_UNSUPPORTED_SIZE"
    h = C.c_void_p()
    d = (C.c_int * 3)(30, 32, 32)          # 30 = 2*3*5: not a supported length
    sp = (C.c_double * 3)(0.4, 0.4, 0.4)
    assert lib.exx_plan_create(C.byref(h), d, sp, 0, None, 4, None) == 2
    assert b"transform lengths" in lib.exx_last_error(None)
    d = (C.c_int * 3)(32, 32, 32)
    assert lib.exx_plan_create(C.byref(h), d, sp, 7, None, 4, None) == 1          # bad enum
    assert lib.exx_plan_create(C.byref(h), d, sp, 1, None, 4, None) == 1          # free BC without a table
    sp_bad = (C.c_double * 3)(0.4, -1.0, 0.4)
    assert lib.exx_plan_create(C.byref(h), d, sp_bad, 0, None, 4, None) == 1
    assert lib.exx_plan_create(C.byref(h), d, sp, 0, None, 0, None) == 1          # max_orbitals < 1
    d = (C.c_int * 3)(32, 64, 72)                                                 # 24 and 72 only as cubic transform grids
    assert lib.exx_plan_create(C.byref(h), d, sp, 0, None, 4, None) == 2
    d = (C.c_int * 3)(512, 512, 512)                                              # longer than any compiled length
    assert lib.exx_plan_create(C.byref(h), d, sp, 0, None, 4, None) == 2
    d = (C.c_int * 3)(36, 16, 16)                                                 # free BC: 2n = 72 mixed with 32
    g = np.ones(36 * 16 * 16)
    assert lib.exx_plan_create(C.byref(h), d, sp, 1, g.ctypes.data_as(C.POINTER(C.c_double)), 4, None) == 2
    # exx_plan_create_general: argument checks come before any device work
    d = (C.c_int * 3)(32, 32, 32)
    k = np.ones(32 ** 3)
    kp = k.ctypes.data_as(C.POINTER(C.c_double))
    assert lib.exx_plan_create_general(C.byref(h), d, C.c_double(100.0), None, 4, None) == 1      # no table
    assert lib.exx_plan_create_general(C.byref(h), d, C.c_double(-1.0), kp, 4, None) == 1         # volume <= 0
    assert lib.exx_plan_create_general(C.byref(h), d, C.c_double(100.0), kp, 0, None) == 1        # max_orbitals < 1
    d = (C.c_int * 3)(30, 32, 32)
    assert lib.exx_plan_create_general(C.byref(h), d, C.c_double(100.0), kp, 4, None) == 2        # unsupported length
    assert lib.exx_plan_destroy(None) == 0
    assert lib.exx_plan_workspace_bytes(None) == 0


def test_no_cpu_fallback():
    """Without a GPU the product path fails loudly (EXX_ERR_CUDA); with one it must succeed.  Never a CPU result."""
    import torch
    if torch.cuda.is_available():
        plan = exx.ExxPlan((16, 16, 16), (0.4, 0.4, 0.4), "periodic", max_orbitals=2)
        plan.destroy()
    else:
        with pytest.raises(exx.ExxError) as ei:
            exx.ExxPlan((16, 16, 16), (0.4, 0.4, 0.4), "periodic", max_orbitals=2)
        assert ei.value.status_name == "EXX_ERR_CUDA"


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1712_07973_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".hpp", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f
                assert "exx_oracle" not in src, f


@pytest.mark.parametrize("occ_res,occ_str,max_batch", [([2.0, 1.0, 0.0], [1.0, 0.0, 2.0, 0.5], 0), ([0.0, 0.0], [0.0, 1.0, 0.0], 2),
                                                       ([1.0], [2.0] * 5, 2), (None, [1.0, 0.0, 2.0], 0)])
def test_block_schedule_covers_the_rectangle_exactly_once(occ_res, occ_str, max_batch):
    """Rectangular schedule of exx_apply_block / exx_apply_to (include/exx.h exx_schedule_list_block): every pair
    (resident j, streamed i) that is not doubly empty appears once; exx_apply_to (no resident occupations) skips the
    streamed orbitals with f = 0, which contribute nothing to K phi."""
    n_res = 3 if occ_res is None else len(occ_res)
    rows = exx.exx_schedule_list_block(occ_res, occ_str, n_res=n_res, max_batch=max_batch)
    seen = {}
    per_batch = {}
    for j, l, i, flags, b in rows.tolist():
        assert flags in (1, 2, 3) and 0 <= j < n_res and (l == -1 or l == j + 1) and 0 <= i < len(occ_str)
        per_batch.setdefault(b, []).append((j, l, i))
        if flags & 1:
            seen[(j, i)] = seen.get((j, i), 0) + 1
        if flags & 2:
            seen[(l, i)] = seen.get((l, i), 0) + 1
    if occ_res is None:
        expect = {(j, i) for j in range(n_res) for i in range(len(occ_str)) if occ_str[i] != 0}
    else:
        expect = {(j, i) for j in range(n_res) for i in range(len(occ_str)) if not (occ_res[j] == 0 and occ_str[i] == 0)}
    assert set(seen) == expect and all(v == 1 for v in seen.values())
    for items in per_batch.values():
        assert len({(j, l) for j, l, _ in items}) == 1
        assert len({i for _, _, i in items}) == len(items)
        if max_batch > 0:
            assert len(items) <= max_batch


def test_masked_schedule_lists_exactly_the_masked_pairs():
    occ = [2.0, 0.0, 1.0, 0.0, 1.5]
    n = len(occ)
    mask = np.zeros((n, n), dtype=np.uint8)
    for a, b in [(0, 0), (0, 2), (1, 3), (1, 4), (3, 4), (2, 2)]:        # (1,3) is doubly empty: skipped although listed
        mask[a, b] = mask[b, a] = 1
    rows = exx.exx_schedule_list(occ, 2, pair_mask=mask)
    got = sorted([(j, i) for j, l, i, f, b in rows.tolist() if f & 1] + [(l, i) for j, l, i, f, b in rows.tolist() if f & 2])
    assert got == [(0, 0), (0, 2), (1, 4), (2, 2), (3, 4)]
    assert np.array_equal(exx.exx_schedule_list(occ, 3, pair_mask=np.ones((n, n))), exx.exx_schedule_list(occ, 3))
