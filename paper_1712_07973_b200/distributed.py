"""Round-robin distribution of the orbitals over the GPUs of one node.

PAPER.md:105-111 (section 2.1, Fig. 1): "each process ... owns a subset of orbitals"; at step s it exchanges blocks with
the ranks p +- s, "calculates the co-densities between its own orbitals and the received ones", and the results that
belong to the received orbitals are "sent back to the owner"; floor(P/2)+1 steps.  Here: one process per GPU,
`torch.distributed` point-to-point transfers (NCCL over NVLink/NVSwitch on the GPU box, gloo in the CPU tests) for the
plumbing, and the library's own kernels for every pair solve: exx_apply for the diagonal block, exx_apply_block for a
received block.  The receive of step s+1 is posted before step s is computed, so the transfer overlaps the pair solves
("overlap of communication and computation").

The step logic is written against two small interfaces so that it can be exercised without GPUs:
  * a BACKEND with  apply_diag(psi, occ) -> (kpsi, ex)  and
                    apply_block(psi_res, occ_res, kpsi_res, psi_str, occ_str) -> (kpsi_str_partial, ex)
    (kpsi_res is accumulated into in place);  CudaBlockBackend is the product one (ExxPlan), the CPU tests pass their own;
  * `torch.distributed` itself (any initialised backend; tensors live wherever the backend's tensors live).
There is no CPU fallback here: CudaBlockBackend needs the CUDA library and a device.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np

from .binding import EXX_BLOCK_ACCUMULATE_RESIDENT, ExxPlan, exx_round_robin_step


def block_counts(n_orb: int, n_ranks: int) -> List[int]:
    """Contiguous blocks, the first n_orb % n_ranks ranks hold one orbital more."""
    return [n_orb // n_ranks + (1 if r < n_orb % n_ranks else 0) for r in range(n_ranks)]


def block_range(n_orb: int, n_ranks: int, rank: int) -> Tuple[int, int]:
    counts = block_counts(n_orb, n_ranks)
    lo = sum(counts[:rank])
    return lo, lo + counts[rank]


class CudaBlockBackend:
    """Pair solves of one rank on its GPU through the C ABI (exx_apply / exx_apply_block)."""

    def __init__(self, plan: ExxPlan):
        self.plan = plan

    def apply_diag(self, psi, occ):
        kpsi, ex = self.plan.apply(psi, occ)
        return kpsi, ex

    def apply_block(self, psi_res, occ_res, kpsi_res, psi_str, occ_str):
        import torch
        kpsi_str = torch.empty_like(psi_str)
        ex = self.plan.apply_block(psi_res, occ_res, kpsi_res, psi_str, occ_str, kpsi_str, flags=EXX_BLOCK_ACCUMULATE_RESIDENT)
        return kpsi_str, ex


def round_robin_apply(backend, psi_own, occ_all: Sequence[float], rank: int, n_ranks: int, dist=None):
    """K psi of this rank's orbital block and the total E_x.

    psi_own   this rank's block [n_own, n1, n2, n3] (orbitals block_range(N, P, rank) of the global set)
    occ_all   occupations of ALL N orbitals (host, replicated: N doubles)
    dist      torch.distributed (initialised) or None for a single rank
    Returns (kpsi_own, E_x) with E_x summed over all ranks.
    """
    import torch
    occ_all = np.ascontiguousarray(np.asarray(occ_all, dtype=np.float64))
    n_orb = int(occ_all.size)
    counts = block_counts(n_orb, n_ranks)
    lo, hi = block_range(n_orb, n_ranks, rank)
    if psi_own.shape[0] != hi - lo:
        raise ValueError("psi_own does not hold this rank's block")
    occ_own = occ_all[lo:hi]
    grid = tuple(psi_own.shape[1:])

    def occ_of(r):
        a, b = block_range(n_orb, n_ranks, r)
        return occ_all[a:b]

    n_steps = n_ranks // 2
    # post the receive of the first visiting block before the diagonal block is computed
    def post_exchange(step):
        send_to, recv_from, what = exx_round_robin_step(n_ranks, rank, step)
        buf = torch.empty((counts[recv_from],) + grid, dtype=psi_own.dtype, device=psi_own.device)
        reqs = dist.batch_isend_irecv([dist.P2POp(dist.isend, psi_own, send_to), dist.P2POp(dist.irecv, buf, recv_from)])
        return send_to, recv_from, what, buf, reqs

    pending = post_exchange(1) if (n_steps >= 1 and dist is not None) else None
    kpsi_own, ex = backend.apply_diag(psi_own, occ_own)                      # step 0: the diagonal block
    for step in range(1, n_steps + 1):
        send_to, recv_from, what, visiting, reqs = pending
        for r in reqs:
            r.wait()
        pending = post_exchange(step + 1) if step + 1 <= n_steps else None   # overlaps this step's pair solves
        occ_vis = occ_of(recv_from)
        n_vis = counts[recv_from]
        if what == 1:                                                        # full block: own (resident) x visiting (streamed)
            part, e = backend.apply_block(psi_own, occ_own, kpsi_own, visiting, occ_vis)
        elif what == 2:                                                      # even P, last step: first half of the own rows
            h = (hi - lo + 1) // 2
            part, e = backend.apply_block(psi_own[:h], occ_own[:h], kpsi_own[:h], visiting, occ_vis)
        else:                                                                # what == 3: second half of the visiting rows
            h = (n_vis + 1) // 2
            if n_vis - h > 0:
                part, e = backend.apply_block(psi_own, occ_own, kpsi_own, visiting[h:], occ_vis[h:])
            else:
                part, e = visiting[h:].clone(), 0.0
        ex += e
        # the partial K psi of the visiting orbitals goes back to their owner; mine arrives from the
        # rank that worked on my block in this step (= send_to)
        _, _, what_peer = exx_round_robin_step(n_ranks, send_to, step)
        if what_peer == 3:
            mine_lo = (hi - lo + 1) // 2
        else:
            mine_lo = 0
        back = torch.empty((hi - lo - mine_lo,) + grid, dtype=psi_own.dtype, device=psi_own.device)
        ops = []
        if part.shape[0] > 0:
            ops.append(dist.P2POp(dist.isend, part.contiguous(), recv_from))
        if back.shape[0] > 0:
            ops.append(dist.P2POp(dist.irecv, back, send_to))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        if back.shape[0] > 0:
            kpsi_own[mine_lo:] += back
    if dist is not None and n_ranks > 1:
        t = torch.tensor([ex], dtype=torch.float64, device=psi_own.device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        ex = float(t[0])
    return kpsi_own, ex
