"""Parity of qsgw_mp2_direct_build (row 8(f).3, first half: the direct term of the qsMP2 self-energy, Eq. (20) first
sum in Eq. (21)) against oracle.mp2_direct, element by element.  Bar: 1e-9 * max|ref|."""
import numpy as np
import pytest
import torch

import oracle
import qsgw_inputs as qi

pytestmark = pytest.mark.gpu


def _pkg():
    import paper_2210_17093_b200 as pkg
    return pkg


@pytest.mark.parametrize("n_mo,n_occ,n_aux,s_block", [
    (24, 5, 80, 0),        # tiny config shapes, one chunk
    (37, 7, 53, 64),       # odd sizes, several chunks with a short last one (210 pairs)
    (120, 20, 400, 512),   # small config shapes (2000 pairs, 4 chunks)
    (131, 64, 33, 1000),   # N just over two p tiles, many pairs (4288)
    (2, 1, 1, 0),
])
def test_parity(n_mo, n_occ, n_aux, s_block):
    pkg = _pkg()
    cfg = qi.custom_config(n_mo, n_occ, n_aux, s_block=s_block, seed=500 + n_mo)
    B, eps, occ = qi.make_B(cfg), qi.make_eps(cfg), qi.make_occ(cfg)
    plan = pkg.qsgw_sigma_create(n_mo, n_occ, n_aux, cfg.n_ov, s_block)
    S = pkg.qsgw_mp2_direct_build(plan, B.cuda(), eps.cuda(), occ.cuda(), cfg.eta)
    torch.cuda.synchronize()
    ref = oracle.mp2_direct(B.numpy(), eps.numpy(), occ.numpy(), cfg.eta, n_occ)
    err = np.max(np.abs(S.cpu().numpy() - ref))
    assert err <= 1e-9 * np.abs(ref).max(), f"{err:.3e} vs {np.abs(ref).max():.3e}"
    assert torch.equal(S, S.T)
    # the plan still serves the GW build afterwards, and the two paths agree on their common ground
    Om = torch.tensor([float(eps[a] - eps[i]) for i in range(n_occ) for a in range(n_occ, n_mo)], dtype=torch.float64)
    S_gw = pkg.qsgw_sigma_build(plan, B.cuda(), eps.cuda(), occ.cuda(), Om.cuda(),
                                torch.eye(cfg.n_ov, dtype=torch.float64, device="cuda"), cfg.eta)
    assert float((S_gw - S).abs().max()) <= 1e-11 * float(S.abs().max())
    pkg.qsgw_sigma_destroy(plan)


@pytest.mark.parametrize("n_mo,n_occ,n_aux,s_block", [
    (24, 5, 80, 0),        # odd n_occ: the exchange loop starts one (zero-weight) state early to stay aligned
    (37, 7, 53, 8),        # odd N (padded exchange-integral rows, scalar GEMM loads), virtual range cut into several chunks
    (120, 20, 400, 512),   # small config shapes
    (70, 64, 33, 0),       # few virtual states
    (2, 1, 1, 0),
])
def test_full_qsmp2_parity(n_mo, n_occ, n_aux, s_block):
    """direct + second-order exchange (qsgw_mp2_build) against oracle.mp2; the exchange part alone as the difference of
    the two entry points against the oracle's sox_only mode."""
    pkg = _pkg()
    cfg = qi.custom_config(n_mo, n_occ, n_aux, s_block=s_block, seed=700 + n_mo)
    B, eps, occ = qi.make_B(cfg), qi.make_eps(cfg), qi.make_occ(cfg)
    plan = pkg.qsgw_sigma_create(n_mo, n_occ, n_aux, cfg.n_ov, s_block)
    Bd, ed, od = B.cuda(), eps.cuda(), occ.cuda()
    S = pkg.qsgw_mp2_build(plan, Bd, ed, od, cfg.eta)
    Sd = pkg.qsgw_mp2_direct_build(plan, Bd, ed, od, cfg.eta)
    torch.cuda.synchronize()
    ref = oracle.mp2(B.numpy(), eps.numpy(), occ.numpy(), cfg.eta, n_occ)
    ref_sox = oracle.mp2(B.numpy(), eps.numpy(), occ.numpy(), cfg.eta, n_occ, sox_only=True)
    scale = np.abs(ref).max()
    assert np.max(np.abs(S.cpu().numpy() - ref)) <= 1e-9 * scale
    assert np.max(np.abs((S - Sd).cpu().numpy() - ref_sox)) <= 1e-9 * max(np.abs(ref_sox).max(), 1e-300) + 1e-12 * scale
    assert torch.equal(S, S.T)
    assert torch.equal(S, pkg.qsgw_mp2_build(plan, Bd, ed, od, cfg.eta))       # reproducible
    pkg.qsgw_sigma_destroy(plan)


def _mp2_sampled(cfg_name, states):
    """qsgw_mp2_build on the WHOLE config (the GPU runs its full build, as bench.py --path mp2 does); the oracle computes
    the sampled S x S block with every internal sum (i, a, p, P) over its full range (oracle.mp2(states=...))."""
    pkg = _pkg()
    cfg = qi.CONFIGS[cfg_name]
    B, eps, occ = qi.make_B(cfg, "cuda"), qi.make_eps(cfg), qi.make_occ(cfg)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_ov, cfg.s_block)
    S = pkg.qsgw_mp2_build(plan, B, eps.cuda(), occ.cuda(), cfg.eta)
    torch.cuda.synchronize()
    assert torch.equal(S, S.T)
    B_h = B.cpu().numpy()
    pkg.qsgw_sigma_destroy(plan)
    ref = oracle.mp2(B_h, eps.numpy(), occ.numpy(), cfg.eta, cfg.n_occ, states=states)
    got = S.cpu().numpy()[np.ix_(states, states)]
    err, scale = np.max(np.abs(got - ref)), np.abs(ref).max()
    assert err <= 1e-9 * scale, f"{cfg_name}: {err:.3e} vs {scale:.3e}"


def test_medium_config_qsmp2_sampled_states():
    """`medium` (N = 300, o = 40, naux = 1100, s-block 2048: 10400 (ia) pairs in 6 chunks for the direct term, 40 exchange
    passes).  24 output states: deepest, HOMO-1, HOMO, LUMO, LUMO+1, highest, the 64/256 tile edges and a regular grid."""
    cfg = qi.CONFIGS["medium"]
    o, N = cfg.n_occ, cfg.n_mo
    states = sorted({0, 1, o - 2, o - 1, o, o + 1, 63, 64, 127, 128, 255, 256, N - 2, N - 1} | set(range(7, N, 29)))
    _mp2_sampled("medium", states)


def test_large_config_qsmp2_sampled_states():
    """`large` (N = 600, o = 80, naux = 2400, s-block 4096), the size bench.py --path mp2 reports: 41600 pairs in 11 chunks,
    80 exchange passes with the [N][N][N] exchange-integral buffer.  5 output states (the oracle's cost is
    41600 x 3 x |S| x 600 x 2400 multiply-adds)."""
    cfg = qi.CONFIGS["large"]
    _mp2_sampled("large", [0, cfg.n_occ - 1, cfg.n_occ, 256, cfg.n_mo - 1])
