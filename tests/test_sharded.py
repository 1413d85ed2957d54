"""Row 8(f).4 (s-sharded multi-GPU build), the parts that need no GPU: the pole partition of the C library
(qsgw_sigma_pole_slice, pure host arithmetic) and the combine step (allreduce_sigma) over gloo with world_size 2, the
CPU oracle standing in for each rank's local build: the sum of the ranks' partial Sigmas is the oracle's Sigma of all poles
(Eq. (17): Sigma is a plain sum over s)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("n_pole", [1, 31, 32, 33, 95, 2000, 10400, 41600, 127500])
@pytest.mark.parametrize("n_ranks", [1, 2, 3, 4, 7, 8])
def test_pole_slices_are_contiguous_disjoint_aligned_and_balanced(n_pole, n_ranks):
    import paper_2210_17093_b200 as pkg
    slices = [pkg.qsgw_sigma_pole_slice(n_pole, n_ranks, r) for r in range(n_ranks)]
    pos = 0
    for s0, n in slices:
        assert n >= 0 and s0 == pos and (s0 % 32 == 0 or n == 0)     # contiguous, in rank order, 32-pole aligned starts
        pos += n
    assert pos == n_pole                                             # cover [0, n_pole) exactly
    lens = [n for _, n in slices]
    assert max(lens) - min(lens) <= 32 or n_pole < 32 * n_ranks      # balanced to one 32-pole group
    if n_pole >= 32 * n_ranks:
        assert min(lens) > 0


def test_pole_slice_rejects_bad_arguments():
    import paper_2210_17093_b200 as pkg
    for args in ((0, 2, 0), (10, 0, 0), (10, 2, 2), (10, 2, -1)):
        with pytest.raises(pkg.QsgwSigmaError) as ei:
            pkg.qsgw_sigma_pole_slice(*args)
        assert ei.value.code == pkg.QSGW_SIGMA_ERR_INVALID_ARG


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import oracle
    import qsgw_inputs as qi
    import paper_2210_17093_b200 as pkg
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = qi.custom_config(30, 6, 25, n_pole=101, seed=21)          # 101 poles: slices of 64 and 37
    inp = qi.make_inputs(cfg)
    s0, n = pkg.qsgw_sigma_pole_slice(cfg.n_pole, world, rank)
    args = (inp.B.numpy(), inp.eps.numpy(), inp.occ.numpy())
    local = oracle.sigma(*args, inp.Omega.numpy()[s0:s0 + n], inp.Z.numpy()[:, s0:s0 + n], cfg.eta, cfg.n_occ)
    local = 0.5 * (local + local.T)                                  # each rank's build is bit-symmetric (epilogue)
    S = pkg.allreduce_sigma(torch.from_numpy(local.copy()))
    out[rank] = (s0, n, S.numpy().copy())
    dist.destroy_process_group()


def test_partial_sigmas_of_two_ranks_sum_to_the_oracle_gloo_world2():
    import oracle
    import qsgw_inputs as qi
    world, port = 2, 31500 + (os.getpid() % 2000)
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    cfg = qi.custom_config(30, 6, 25, n_pole=101, seed=21)
    inp = qi.make_inputs(cfg)
    ref = oracle.sigma(inp.B.numpy(), inp.eps.numpy(), inp.occ.numpy(), inp.Omega.numpy(), inp.Z.numpy(), cfg.eta, cfg.n_occ)
    assert (out[0][0], out[0][1]) == (0, 64) and (out[1][0], out[1][1]) == (64, 37)
    for rank in range(world):
        S = out[rank][2]
        assert np.max(np.abs(S - ref)) <= 1e-12 * np.abs(ref).max()
        assert np.array_equal(S, S.T)                                # the reduction keeps Sigma bit-symmetric
    assert np.array_equal(out[0][2], out[1][2])                      # every rank holds the same matrix


def test_allreduce_sigma_is_the_identity_without_a_process_group():
    import paper_2210_17093_b200 as pkg
    S = torch.arange(9, dtype=torch.float64).reshape(3, 3)
    assert pkg.allreduce_sigma(S) is S
