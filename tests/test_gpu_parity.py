"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Bar (BASELINE.json north_star): max|Sigma_gpu - Sigma_ref| <= 1e-9 * max|Sigma_ref|."""
import numpy as np
import pytest
import torch

import oracle
import qsgw_inputs as qi

pytestmark = pytest.mark.gpu

TOL = 1e-9


def _pkg():
    import paper_2210_17093_b200 as pkg
    return pkg


def _to_dev(inp):
    return [t.cuda() for t in (inp.B, inp.eps, inp.occ, inp.Omega, inp.Z)]


def _gpu_sigma(cfg, dev, s_block=None, n_pole_max=None):
    pkg = _pkg()
    B, eps, occ, Om, Z = dev
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, n_pole_max or Om.shape[0],
                                 cfg.s_block if s_block is None else s_block)
    S = pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta)
    torch.cuda.synchronize()
    return S, plan


def _ref_sigma(cfg, inp, states=None):
    return oracle.sigma(inp.B.numpy(), inp.eps.numpy(), inp.occ.numpy(), inp.Omega.numpy(), inp.Z.numpy(),
                        cfg.eta, cfg.n_occ, states=states)


def _assert_parity(S_gpu, S_ref, tol=TOL):
    S_gpu = S_gpu.cpu().numpy() if isinstance(S_gpu, torch.Tensor) else S_gpu
    err = np.max(np.abs(S_gpu - S_ref))
    scale = np.max(np.abs(S_ref))
    assert np.all(np.isfinite(S_gpu))
    assert err <= tol * scale, f"max|dSigma| = {err:.3e} > {tol:g} * max|Sigma_ref| = {tol * scale:.3e}"


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_config_full_parity(name):
    cfg = qi.CONFIGS[name]
    inp = qi.make_inputs(cfg)
    S, plan = _gpu_sigma(cfg, _to_dev(inp))
    _assert_parity(S, _ref_sigma(cfg, inp))
    assert torch.equal(S, S.T), "Sigma must be bit-symmetric"
    _pkg().qsgw_sigma_destroy(plan)


# ragged shapes: odd N (scalar epilogues), odd naux, pole counts that leave ragged k / n tails, several
# chunks with a short last chunk, N spanning 2-3 tiles with a ragged last tile
RAGGED = [
    # n_mo n_occ n_aux n_pole s_block
    (37, 7, 53, 210, 64),
    (130, 3, 17, 381, 128),
    (131, 64, 33, 150, 0),
    (257, 5, 40, 300, 100),
    (250, 20, 40, 200, 64),      # one 256-column q-tile: the stage-3 instance for 8 column fragments per warp
    (233, 9, 24, 130, 0),        # the same instance with 8 / 8 / 7 / 7 column fragments
    (24, 23, 9, 23, 0),
    (2, 1, 1, 1, 0),
]


@pytest.mark.parametrize("n_mo,n_occ,n_aux,n_pole,s_block", RAGGED)
def test_ragged_shapes_parity(n_mo, n_occ, n_aux, n_pole, s_block):
    cfg = qi.custom_config(n_mo, n_occ, n_aux, n_pole=n_pole, s_block=s_block, seed=100 + n_mo)
    inp = qi.make_inputs(cfg)
    S, plan = _gpu_sigma(cfg, _to_dev(inp))
    _assert_parity(S, _ref_sigma(cfg, inp))
    assert torch.equal(S, S.T)
    _pkg().qsgw_sigma_destroy(plan)


def test_stage_outputs_match_oracle_steps():
    """a1/a2: V and the w chunk, element by element, against oracle steps 1 and 2 (through the test build of the library,
    which adds the qsgw_sigma_copy_workspace hook; the same sources otherwise)."""
    from testhooks import HookedPlan, WORKSPACE_V, WORKSPACE_W
    cfg = qi.custom_config(70, 9, 45, n_pole=200, s_block=0, seed=5)
    inp = qi.make_inputs(cfg)
    B, eps, occ, Om, Z = _to_dev(inp)
    plan = HookedPlan(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, cfg.s_block)
    S = plan.build(B, eps, occ, Om, Z, cfg.eta)
    V = plan.copy_workspace(WORKSPACE_V, cfg.n_aux, cfg.n_pole).cpu().numpy()
    W = plan.copy_workspace(WORKSPACE_W, cfg.n_mo ** 2, cfg.n_pole).cpu().numpy()
    torch.cuda.synchronize()
    _assert_parity(S, _ref_sigma(cfg, inp))
    V_ref = oracle.pole_weights(inp.B.numpy(), inp.Z.numpy(), cfg.n_occ)
    assert np.max(np.abs(V - V_ref)) <= 1e-13 * np.max(np.abs(V_ref))
    W = W.reshape(cfg.n_mo, cfg.n_mo, cfg.n_pole)              # [m][p][s]
    for s in (0, 1, 77, 199):
        w_ref = oracle.residues(inp.B.numpy(), V_ref, s)       # [p][m]
        assert np.max(np.abs(W[:, :, s].T - w_ref)) <= 1e-13 * np.max(np.abs(w_ref))
    plan.destroy()


def test_general_occupations_and_unsorted_inputs():
    cfg = qi.custom_config(40, 6, 20, n_pole=90, seed=9)
    inp = qi.make_inputs(cfg)
    g = torch.Generator().manual_seed(3)
    inp.occ = torch.rand(cfg.n_mo, generator=g, dtype=torch.float64)          # fractional f_m: both terms of D
    inp.occ[0], inp.occ[1] = 1.0, 0.0
    inp.Omega = inp.Omega[torch.randperm(cfg.n_pole, generator=g)]            # sorting is not required
    S, plan = _gpu_sigma(cfg, _to_dev(inp))
    _assert_parity(S, _ref_sigma(cfg, inp))
    _pkg().qsgw_sigma_destroy(plan)


def test_exact_power_of_two_scaling_and_reproducibility():
    pkg = _pkg()
    cfg = qi.CONFIGS["tiny"]
    inp = qi.make_inputs(cfg)
    B, eps, occ, Om, Z = _to_dev(inp)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, 32)
    S = pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta).clone()
    S2 = pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta).clone()
    assert torch.equal(S, S2), "same inputs, same plan: results must be bitwise reproducible"
    assert torch.equal(pkg.qsgw_sigma_build(plan, B, eps, occ, Om, 2.0 * Z, cfg.eta), 4.0 * S)
    assert torch.equal(pkg.qsgw_sigma_build(plan, 2.0 * B, eps, occ, Om, Z, cfg.eta), 16.0 * S)
    pkg.qsgw_sigma_destroy(plan)


def test_additive_over_pole_ranges_and_chunkings():
    pkg = _pkg()
    cfg = qi.custom_config(96, 12, 60, n_pole=700, seed=12)
    inp = qi.make_inputs(cfg)
    B, eps, occ, Om, Z = _to_dev(inp)
    ref = _ref_sigma(cfg, inp)
    scale = np.abs(ref).max()
    results = []
    for s_block in (0, 64, 250, 700):
        S, plan = _gpu_sigma(cfg, (B, eps, occ, Om, Z), s_block=s_block)
        _assert_parity(S, ref)
        results.append(S.cpu().numpy())
        pkg.qsgw_sigma_destroy(plan)
    for r in results[1:]:
        assert np.max(np.abs(r - results[0])) <= 1e-12 * scale
    # streaming API over ragged ranges (pointer offsets into the full Z, ldz = full n_pole)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, 300, 128)
    pkg.qsgw_sigma_begin(plan, B, eps, occ, cfg.eta)
    for a, b in [(0, 1), (1, 300), (300, 555), (555, 700)]:
        pkg.qsgw_sigma_add_poles(plan, Om[a:b], Z[:, a:b])
    S = pkg.qsgw_sigma_finish(plan)
    _assert_parity(S, ref)
    # the one-shot call on a sub-range equals the oracle on that sub-range
    S_r = pkg.qsgw_sigma_build(plan, B, eps, occ, Om[101:400], Z[:, 101:400], cfg.eta)
    ref_r = oracle.sigma(inp.B.numpy(), inp.eps.numpy(), inp.occ.numpy(), inp.Omega.numpy()[101:400],
                         inp.Z.numpy()[:, 101:400], cfg.eta, cfg.n_occ)
    _assert_parity(S_r, ref_r)
    pkg.qsgw_sigma_destroy(plan)


def test_stage1_in_several_pole_batches():
    """more poles in one call than one stage-1 launch takes (V capacity): the v-range loop of add_poles"""
    pkg = _pkg()
    cfg = qi.custom_config(50, 8, 31, n_pole=330, s_block=64, seed=44)
    inp = qi.make_inputs(cfg)
    dev = _to_dev(inp)
    ref = _ref_sigma(cfg, inp)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, cfg.s_block)
    S_one = pkg.qsgw_sigma_build(plan, *dev, cfg.eta).clone()
    for batch in (1, 64, 100, 256):                       # rounded up to 64, 64, 128, 256 poles per stage-1 launch
        pkg.qsgw_sigma_limit_pole_batch(plan, batch)
        S = pkg.qsgw_sigma_build(plan, *dev, cfg.eta)
        _assert_parity(S, ref)
        assert float((S - S_one).abs().max()) <= 1e-12 * float(S_one.abs().max())
    pkg.qsgw_sigma_destroy(plan)


def test_host_buffer_entry_point_matches_device_entry_point():
    pkg = _pkg()
    cfg = qi.custom_config(64, 10, 48, n_pole=540, s_block=128, seed=21)
    inp = qi.make_inputs(cfg)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, cfg.s_block)
    S_dev = pkg.qsgw_sigma_build(plan, *_to_dev(inp), cfg.eta)
    torch.cuda.synchronize()
    pinned = [t.pin_memory() for t in (inp.B, inp.eps, inp.occ, inp.Omega, inp.Z)]
    S_host = pkg.qsgw_sigma_build_host(plan, *pinned, cfg.eta)
    assert torch.equal(S_host, S_dev.cpu())
    S_host2 = pkg.qsgw_sigma_build_host(plan, inp.B, inp.eps, inp.occ, inp.Omega, inp.Z, cfg.eta)   # pageable
    assert torch.equal(S_host2, S_host)
    _assert_parity(S_host, _ref_sigma(cfg, inp))
    pkg.qsgw_sigma_destroy(plan)


def test_host_buffer_entry_point_with_more_poles_than_the_plan_capacity_and_unequal_ranges():
    """n_pole > n_pole_max through the host path: the library uploads one s-block first and then ranges of four s-blocks
    (64, 256 and 220 poles here), each with its own stage 1; compared with the oracle, and twice for reproducibility."""
    pkg = _pkg()
    cfg = qi.custom_config(70, 9, 45, n_pole=540, s_block=64, seed=23)
    inp = qi.make_inputs(cfg)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, 256, cfg.s_block)
    S1 = pkg.qsgw_sigma_build_host(plan, inp.B, inp.eps, inp.occ, inp.Omega, inp.Z, cfg.eta)
    S2 = pkg.qsgw_sigma_build_host(plan, inp.B, inp.eps, inp.occ, inp.Omega, inp.Z, cfg.eta)
    assert torch.equal(S1, S2) and torch.equal(S1, S1.T)
    _assert_parity(S1, _ref_sigma(cfg, inp))
    pkg.qsgw_sigma_destroy(plan)


def test_null_case_and_error_codes():
    pkg = _pkg()
    cfg = qi.CONFIGS["tiny"]
    inp = qi.make_inputs(cfg)
    B, eps, occ, Om, Z = _to_dev(inp)
    B0 = B.clone()
    B0[:, :cfg.n_occ, cfg.n_occ:] = 0.0
    B0[:, cfg.n_occ:, :cfg.n_occ] = 0.0
    S, plan = _gpu_sigma(cfg, (B0, eps, occ, Om, Z))
    assert torch.count_nonzero(S) == 0
    with pytest.raises(pkg.QsgwSigmaError) as ei:
        pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, 0.0)
    assert ei.value.code == pkg.QSGW_SIGMA_ERR_INVALID_ARG
    with pytest.raises(pkg.QsgwSigmaError):
        pkg.qsgw_sigma_finish(plan)                           # finish without begin
    with pytest.raises(pkg.QsgwSigmaError):
        pkg.qsgw_sigma_add_poles(plan, Om, Z)                 # add_poles without begin
    small_plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, 10)
    with pytest.raises(pkg.QsgwSigmaError):
        pkg.qsgw_sigma_build(small_plan, B, eps, occ, Om, Z, cfg.eta)   # n_pole > n_pole_max
    # the plan is still usable after errors
    S2 = pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta)
    _assert_parity(S2, _ref_sigma(cfg, inp))
    pkg.qsgw_sigma_destroy(plan)
    pkg.qsgw_sigma_destroy(small_plan)


def test_repeated_build_on_a_side_stream_replays_as_a_cuda_graph():
    """Identical calls on a capturable stream: the third call on is one CUDA graph launch; results are bitwise those of
    the launch-by-launch path, and they follow the CONTENTS of the caller's buffers (refreshed in place)."""
    pkg = _pkg()
    cfg = qi.custom_config(150, 11, 70, n_pole=300, s_block=128, seed=77)
    inp = qi.make_inputs(cfg)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        B, eps, occ, Om, Z = _to_dev(inp)
        plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, cfg.s_block, stream=stream)
        S = torch.empty((cfg.n_mo, cfg.n_mo), dtype=torch.float64, device="cuda")
        outs = []
        for _ in range(4):
            pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta, S)
            stream.synchronize()
            outs.append(S.clone())
        st = pkg.qsgw_sigma_get_stats(plan)
        assert st["builds"] == 4 and st["poles"] == 4 * cfg.n_pole
        assert all(torch.equal(outs[0], o) for o in outs[1:])
        _assert_parity(outs[3], _ref_sigma(cfg, inp))
        Z.mul_(2.0)                                              # same pointers, new contents: the graph must see them
        pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta, S)
        stream.synchronize()
        assert torch.equal(S, 4.0 * outs[0])
        Z.mul_(0.5)
        S2 = pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta)        # other output pointer: launch by launch again
        stream.synchronize()
        assert torch.equal(S2, outs[0])
        pkg.qsgw_sigma_destroy(plan)


def test_debug_mode_checks_the_device_side_preconditions():
    """occ in [0,1], Omega > 0 and B symmetric are documented preconditions, verified only in debug mode."""
    pkg = _pkg()
    cfg = qi.custom_config(40, 6, 20, n_pole=90, seed=12)
    inp = qi.make_inputs(cfg)
    B, eps, occ, Om, Z = _to_dev(inp)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole)
    S = pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta)
    pkg.qsgw_sigma_set_debug(plan, True)
    assert torch.equal(pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta), S)     # valid inputs pass, same result
    B_bad = B.clone(); B_bad[3, 5, 17] += 1e-3
    occ_bad = occ.clone(); occ_bad[7] = 1.5
    occ_nan = occ.clone(); occ_nan[0] = float("nan")
    Om_bad = Om.clone(); Om_bad[11] = -Om_bad[11]
    Om_zero = Om.clone(); Om_zero[0] = 0.0
    B_inf = B.clone(); B_inf[0, 1, 1] = float("inf")
    for args, word in (((B_bad, eps, occ, Om, Z), "symmetric"), ((B, eps, occ_bad, Om, Z), "occupations"),
                       ((B, eps, occ_nan, Om, Z), "occupations"), ((B, eps, occ, Om_bad, Z), "Omega"),
                       ((B, eps, occ, Om_zero, Z), "Omega"), ((B_inf, eps, occ, Om, Z), "non-finite")):
        with pytest.raises(pkg.QsgwSigmaError) as ei:
            pkg.qsgw_sigma_build(plan, *args, cfg.eta)
        assert ei.value.code == pkg.QSGW_SIGMA_ERR_INVALID_ARG and word in str(ei.value), str(ei.value)
    assert torch.equal(pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta), S)     # the plan survives the refusals
    pkg.qsgw_sigma_set_debug(plan, False)
    pkg.qsgw_sigma_build(plan, B_bad, eps, occ, Om, Z, cfg.eta)                        # outside debug mode: not checked
    torch.cuda.synchronize()
    pkg.qsgw_sigma_destroy(plan)


def test_medium_config_full_parity():
    cfg = qi.CONFIGS["medium"]
    inp = qi.make_inputs(cfg)
    S, plan = _gpu_sigma(cfg, _to_dev(inp))
    _assert_parity(S, _ref_sigma(cfg, inp))
    assert torch.equal(S, S.T)
    _pkg().qsgw_sigma_destroy(plan)
