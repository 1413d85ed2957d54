"""Row 8(f).4 on the GPU: two processes (world_size 2, gloo for the one all-reduce) share cuda:0, each builds its pole
slice with the unchanged single-GPU library (qsgw_sigma_build_pole_sharded), and the reduced Sigma is compared with the
oracle's Sigma of ALL poles.  The ranks only meet at the all-reduce after their builds (no kernel waits on another rank)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import qsgw_inputs as qi

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CASES = {"small": qi.CONFIGS["small"], "medium": qi.CONFIGS["medium"],
         "uneven": qi.custom_config(70, 9, 45, n_pole=333, s_block=64, seed=31)}


def _worker(rank, world, port, name, out):
    sys.path.insert(0, ROOT)
    import paper_2210_17093_b200 as pkg
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    cfg = CASES[name]
    s0, n = pkg.qsgw_sigma_pole_slice(cfg.n_pole, world, rank)
    B = qi.make_B(cfg).cuda()                       # host-drawn: every rank (and the oracle) sees the same arrays
    eps, occ, Om = qi.make_eps(cfg).cuda(), qi.make_occ(cfg).cuda(), qi.make_omega(cfg).cuda()
    Z = qi.make_Z(cfg, s0, s0 + n).cuda()
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, max(n, 1), cfg.s_block)
    S = pkg.qsgw_sigma_build_pole_sharded(plan, B, eps, occ, Om[s0:s0 + n], Z, cfg.eta)
    torch.cuda.synchronize()
    out[rank] = (s0, n, S.cpu().numpy())
    pkg.qsgw_sigma_destroy(plan)
    dist.destroy_process_group()


@pytest.mark.parametrize("name", ["uneven", "small", "medium"])
def test_two_ranks_build_pole_slices_and_all_reduce(name):
    world, port = 2, 33500 + (os.getpid() % 2000)
    out = mp.Manager().dict()
    mp.spawn(_worker, args=(world, port, name, out), nprocs=world, join=True)
    cfg = CASES[name]
    assert out[0][0] == 0 and out[1][0] == out[0][1] and out[0][1] + out[1][1] == cfg.n_pole
    states = None if cfg.n_mo <= 120 else sorted({0, cfg.n_occ - 1, cfg.n_occ, 63, 64, 255, 256, cfg.n_mo - 1, 101, 202})
    ref = oracle.sigma(qi.make_B(cfg).numpy(), qi.make_eps(cfg).numpy(), qi.make_occ(cfg).numpy(), qi.make_omega(cfg).numpy(),
                       qi.make_Z(cfg).numpy(), cfg.eta, cfg.n_occ, states=states)
    for rank in range(world):
        S = out[rank][2]
        assert np.array_equal(S, S.T)
        got = S if states is None else S[np.ix_(states, states)]
        err, scale = np.max(np.abs(got - ref)), np.abs(ref).max()
        assert err <= 1e-9 * scale, f"rank {rank}: {err:.3e} vs {scale:.3e}"
    assert np.array_equal(out[0][2], out[1][2])
