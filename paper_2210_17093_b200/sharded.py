"""Pole-sharded Sigma^c build over several GPUs: one process per GPU, torch.distributed plumbing.

Sigma is a plain sum over the poles s (Eq. (17)), so rank r runs the unchanged single-GPU build
(qsgw_sigma_begin / _add_poles / _finish) on its contiguous slice of Omega / Z columns -- the partition is
qsgw_sigma_pole_slice of the C library -- with B, eps, occ replicated, and ONE all-reduce(sum) of the N x N FP64 matrix
(<= 8 MB) finishes the build.  There is no other exchange step, so the collective is a plain NCCL (or gloo) all-reduce;
no arithmetic of the method happens here.
"""
from __future__ import annotations

from typing import Optional

import torch
import torch.distributed as dist

from . import binding


def allreduce_sigma(Sigma: torch.Tensor, group=None) -> torch.Tensor:
    """In-place sum over the ranks of `group` of a bit-symmetric N x N matrix, keeping it bit-symmetric.

    Only the upper triangle travels (a ring all-reduce adds the ranks in a different order in different parts of the
    buffer, so reducing both triangles would break Sigma[p][q] == Sigma[q][p] in the last bit) and is mirrored
    afterwards.  With one rank (or no process group) this is the identity.
    """
    if not dist.is_available() or not dist.is_initialized() or dist.get_world_size(group) == 1:
        return Sigma
    N = Sigma.shape[0]
    iu = torch.triu_indices(N, N, device=Sigma.device)
    packed = Sigma[iu[0], iu[1]].contiguous()
    if Sigma.is_cuda and dist.get_backend(group) == "gloo":       # gloo reduces host buffers
        host = packed.cpu()
        dist.all_reduce(host, op=dist.ReduceOp.SUM, group=group)
        packed = host.to(Sigma.device)
    else:
        dist.all_reduce(packed, op=dist.ReduceOp.SUM, group=group)
    Sigma[iu[0], iu[1]] = packed
    Sigma[iu[1], iu[0]] = packed
    return Sigma


def qsgw_sigma_build_pole_sharded(plan: binding.Plan, B, eps, occ, Omega_local, Z_local, eta: float, group=None,
                                  Sigma: Optional[torch.Tensor] = None, max_poles_per_call: Optional[int] = None) -> torch.Tensor:
    """This rank's part of a pole-sharded build, then the all-reduce: every rank returns the full Sigma.

    Omega_local [n], Z_local [n_ov, n] are this rank's slice (s0, n) = qsgw_sigma_pole_slice(n_pole, world, rank) of the
    poles; n may be 0.  Poles are handed to qsgw_sigma_add_poles in pieces of at most plan.n_pole_max.
    """
    n = int(Omega_local.shape[0])
    step = int(max_poles_per_call or plan.n_pole_max)
    binding.qsgw_sigma_begin(plan, B, eps, occ, eta)
    for a in range(0, n, step):
        b = min(n, a + step)
        binding.qsgw_sigma_add_poles(plan, Omega_local[a:b], Z_local[:, a:b])
    Sigma = binding.qsgw_sigma_finish(plan, Sigma)
    stream = plan.stream if plan.stream is not None else torch.cuda.current_stream()
    with torch.cuda.stream(stream):                                # the reduction follows the build on the plan's stream
        allreduce_sigma(Sigma, group)
    return Sigma
