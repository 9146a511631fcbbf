"""NEXT-3: the round-robin orbital-block distribution of PAPER.md:105-111 / Fig. 1, without GPUs.

* the schedule exported by the C ABI (exx_round_robin_step) covers every pair of orbitals in different blocks exactly
  once, for odd and even rank counts and ragged block sizes;
* paper_1712_07973_b200.distributed.round_robin_apply, run under real torch.distributed process groups (gloo, world
  sizes 2, 3 and 4 on 127.0.0.1) with a CPU backend that evaluates each block with the ORACLE, reproduces the oracle's
  single-process apply: what is tested is the exchange / send-back / accumulation logic of the product's driver, the pair
  solves themselves are covered by the GPU parity tests of exx_apply_block.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import paper_1712_07973_b200 as exx                                      # noqa: E402
from paper_1712_07973_b200.distributed import block_counts, block_range    # noqa: E402


@pytest.mark.parametrize("n_ranks,n_orb", [(1, 3), (2, 5), (2, 2), (3, 7), (4, 9), (4, 4), (5, 11), (8, 19), (8, 8)])
def test_schedule_covers_every_cross_block_pair_once(n_ranks, n_orb):
    seen = {}
    for rank in range(n_ranks):
        lo, hi = block_range(n_orb, n_ranks, rank)
        for step in range(n_ranks // 2 + 1):
            send_to, recv_from, what = exx.exx_round_robin_step(n_ranks, rank, step)
            assert send_to == (rank + step) % n_ranks and recv_from == (rank - step) % n_ranks
            # the peer I send to must expect my block at this step
            assert exx.exx_round_robin_step(n_ranks, send_to, step)[1] == rank
            if step == 0:
                assert what == 0
                continue
            vlo, vhi = block_range(n_orb, n_ranks, recv_from)
            own, vis = list(range(lo, hi)), list(range(vlo, vhi))
            if what == 2:
                own = own[: (len(own) + 1) // 2]
            elif what == 3:
                vis = vis[(len(vis) + 1) // 2:]
            else:
                assert what == 1
            for a in own:
                for b in vis:
                    key = (min(a, b), max(a, b))
                    seen[key] = seen.get(key, 0) + 1
    owner = lambda x: next(r for r in range(n_ranks) if block_range(n_orb, n_ranks, r)[0] <= x < block_range(n_orb, n_ranks, r)[1])
    expect = {(a, b) for a in range(n_orb) for b in range(a + 1, n_orb) if owner(a) != owner(b)}
    assert set(seen) == expect and all(v == 1 for v in seen.values())
    assert sum(block_counts(n_orb, n_ranks)) == n_orb


def test_schedule_argument_errors():
    lib = exx.load_library()
    import ctypes as C
    a, b, w = C.c_int(), C.c_int(), C.c_int()
    assert lib.exx_round_robin_step(4, 4, 0, C.byref(a), C.byref(b), C.byref(w)) == 1      # rank out of range
    assert lib.exx_round_robin_step(4, 0, 3, C.byref(a), C.byref(b), C.byref(w)) == 1      # step > floor(P/2)
    assert lib.exx_round_robin_step(0, 0, 0, C.byref(a), C.byref(b), C.byref(w)) == 1
    assert lib.exx_round_robin_step(4, 0, 1, None, C.byref(b), C.byref(w)) == 1


class OracleBlockBackend:
    """CPU stand-in for CudaBlockBackend used ONLY by this test: every block is evaluated by the oracle."""

    def __init__(self, dims, spacing, bc, kernel):
        from oracle import Oracle
        self.o = Oracle(dims, spacing, bc, kernel)

    def apply_diag(self, psi, occ):
        k, ex, _ = self.o.apply(psi.numpy(), occ, symmetric=False)
        return torch.from_numpy(k), ex

    def apply_block(self, psi_res, occ_res, kpsi_res, psi_str, occ_str):
        ka, kb, ex, _ = self.o.apply_block(psi_res.numpy(), occ_res, psi_str.numpy(), occ_str)
        kpsi_res += torch.from_numpy(ka)
        return torch.from_numpy(kb), ex


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, spec_args, occ, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1712_07973_b200.distributed import round_robin_apply
    from workloads import make_workload, small_spec
    w = make_workload(small_spec(*spec_args[0], **spec_args[1]))
    spec = w["spec"]
    lo, hi = block_range(spec.n_orb, world, rank)
    backend = OracleBlockBackend(spec.dims, spec.spacing, spec.bc, w["kernel"])
    kpsi, ex = round_robin_apply(backend, w["psi"][lo:hi].contiguous(), occ, rank, world, dist)
    out[rank] = (kpsi.numpy(), ex)
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,base,dims,n_orb", [(2, "C1", (6, 6, 8), 5), (3, "C2", (4, 4, 6), 7), (4, "C1", (4, 6, 4), 6)])
def test_round_robin_driver_matches_single_process_oracle(world, base, dims, n_orb):
    from oracle import Oracle
    from workloads import make_workload, small_spec
    spec_args = ((base,), dict(dims=dims, n_orb=n_orb, spacing=(0.5, 0.45, 0.4), number=3300 + world))
    occ = np.array([2.0, 0.7, 0.0, 1.3, 0.4, 1.1, 0.9][:n_orb])
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), spec_args, occ, out), nprocs=world, join=True)
    w = make_workload(small_spec(*spec_args[0], **spec_args[1]))
    spec = w["spec"]
    k_ref, ex_ref, _ = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"]).apply(w["psi"].numpy(), occ, symmetric=False)
    scale = np.max(np.abs(k_ref))
    for rank in range(world):
        lo, hi = block_range(n_orb, world, rank)
        kpsi, ex = out[rank]
        assert np.max(np.abs(kpsi - k_ref[lo:hi])) <= 1e-13 * scale
        assert abs(ex - ex_ref) <= 1e-13 * abs(ex_ref)
