"""Parity of the CUDA path at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(plan created with the config's n_pole and s_block; one-shot qsgw_sigma_build for `large`, the streaming
begin/add_poles/finish calls with 8192-pole ranges for `xl`, whose Z is 130 GB).

The full oracle is unaffordable there (1e14 - 1e15 flops), so (SURVEY.md 8(c) "Oracle affordability"):
  * sampled outputs the oracle can compute one by one: a pole sub-range x a sampled set of states at the full
    N and naux with the config's random inputs, the GPU building the same sub-range -- more than one s-block of poles in
    ONE call, so that the library's chunk loop runs -- through pointer offsets into the full-size arrays;
  * a property that holds at any size: the separable closed form (pin 9 of tests/test_oracle_pins.py, where the
    oracle itself is checked against it) evaluated in numpy for sampled states, the GPU doing its full dense work;
  * additivity over pole ranges, bit-symmetry, reproducibility.
Bar: max|Sigma_gpu - Sigma_ref| <= 1e-9 * max|Sigma_ref| (BASELINE.json north_star).
"""
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


def _sample_states(cfg, n_random=10, seed=0):
    """deepest, HOMO-1, HOMO, LUMO, LUMO+1, highest, tile-edge neighbours, and a few random states"""
    N, o = cfg.n_mo, cfg.n_occ
    fixed = [0, 1, o - 2, o - 1, o, o + 1, 63, 64, 255, 256, N - 2, N - 1]
    rng = np.random.default_rng(seed)
    extra = rng.choice(N, size=n_random, replace=False).tolist()
    return sorted({s for s in fixed + extra if 0 <= s < N})


def _separable_reference(c, u, z, t, eps, occ, Om, eta, o, states):
    """Sigma_pq = kappa^2 C2^2 u_p u_q [h(eps_p) + h(eps_q)], h(w) = sum_m u_m^2 sum_s t_s^2 D_ms(w), for p, q in
    `states` (SURVEY.md 8(c) pin 9).  numpy FP64, the (m, s) sum in long double."""
    N = len(u)
    v = N - o
    kappa = float(np.sum(np.outer(u[:o], u[o:]).reshape(-1).astype(np.longdouble) * z.astype(np.longdouble)))
    C2 = float(np.sum(c.astype(np.longdouble) ** 2))
    t2 = (t * t)
    h = np.zeros(len(states), dtype=np.longdouble)
    for k, p in enumerate(states):
        acc = np.longdouble(0)
        for m in range(N):
            d = eps[p] - eps[m]
            x1 = d + Om
            x2 = d - Om
            Dm = occ[m] * (x1 / (x1 * x1 + eta * eta)) + (1.0 - occ[m]) * (x2 / (x2 * x2 + eta * eta))
            acc += np.longdouble(u[m] * u[m]) * np.sum((t2 * Dm).astype(np.longdouble))
        h[k] = acc
    us = u[states]
    ref = (kappa ** 2) * (C2 ** 2) * np.outer(us, us) * (h[:, None] + h[None, :]).astype(np.float64)
    return ref


def _assert_parity(got, ref, what):
    err = float(np.max(np.abs(got - ref)))
    scale = float(np.max(np.abs(ref)))
    assert np.all(np.isfinite(got)), what
    assert err <= TOL * scale, f"{what}: max|dSigma| = {err:.3e} > {TOL:g} * max|Sigma_ref| = {TOL * scale:.3e}"
    return err / scale


def _separable_inputs(cfg, dev, seed):
    g = torch.Generator().manual_seed(seed)
    c = torch.randn(cfg.n_aux, generator=g, dtype=torch.float64) * 0.3
    u = torch.randn(cfg.n_mo, generator=g, dtype=torch.float64)
    z = torch.randn(cfg.n_ov, generator=g, dtype=torch.float64)
    t = torch.randn(cfg.n_pole, generator=g, dtype=torch.float64) / np.sqrt(cfg.n_pole)
    B = (c.to(dev)[:, None, None] * u.to(dev)[None, :, None] * u.to(dev)[None, None, :]).contiguous()
    return c, u, z, t, B


def test_large_config_full_build_separable_closed_form():
    """`large`, exactly as bench.py runs it (one qsgw_sigma_build over all 41600 poles, s-block 4096)."""
    pkg = _pkg()
    cfg = qi.CONFIGS["large"]
    dev = torch.device("cuda", 0)
    c, u, z, t, B = _separable_inputs(cfg, dev, seed=1234)
    eps, occ, Om = qi.make_eps(cfg), qi.make_occ(cfg), qi.make_omega(cfg)
    Z = torch.outer(z.to(dev), t.to(dev))
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, cfg.s_block)
    S = pkg.qsgw_sigma_build(plan, B, eps.to(dev), occ.to(dev), Om.to(dev), Z, cfg.eta)
    torch.cuda.synchronize()
    assert torch.equal(S, S.T), "Sigma must be bit-symmetric"
    S2 = pkg.qsgw_sigma_build(plan, B, eps.to(dev), occ.to(dev), Om.to(dev), Z, cfg.eta)
    assert torch.equal(S, S2), "same inputs, same plan: bitwise reproducible"
    states = _sample_states(cfg)
    ref = _separable_reference(c.numpy(), u.numpy(), z.numpy(), t.numpy(), eps.numpy(), occ.numpy(), Om.numpy(),
                               cfg.eta, cfg.n_occ, states)
    got = S.cpu().numpy()[np.ix_(states, states)]
    _assert_parity(got, ref, "large, separable closed form")
    pkg.qsgw_sigma_destroy(plan)


def test_large_config_multi_chunk_pole_range_vs_oracle_on_sampled_states():
    """Full N = 600, naux = 2400, (ia) = 41600 with the config's RANDOM inputs, plan as bench.py creates it (n_pole_max =
    41600, s-block 4096).  ONE qsgw_sigma_build call over 4096 + 160 poles that start at pole 3000 (pointer offset into
    a wider Z, full leading dimension), so that the library's own chunk loop runs twice -- a full 4096-pole w chunk and a
    ragged 160-pole one -- and, in a second pass with qsgw_sigma_limit_pole_batch(4096), its stage-1 range loop too.
    Sampled states S x S against oracle.sigma on exactly those poles (about a minute of oracle time)."""
    pkg = _pkg()
    cfg = qi.CONFIGS["large"]
    dev = torch.device("cuda", 0)
    s0 = 3000
    s1 = s0 + cfg.s_block + 160
    B = qi.make_B(cfg, dev)
    eps, occ, Om = qi.make_eps(cfg), qi.make_occ(cfg), qi.make_omega(cfg)
    eps_d, occ_d, Om_d = eps.to(dev), occ.to(dev), Om.to(dev)   # must outlive begin ... finish (include/qsgw_sigma.h)
    # one buffer holding the columns [0, s1): the sub-range is handed over by pointer offset with the full leading dimension
    Zfull = torch.zeros((cfg.n_ov, s1), dtype=torch.float64, device=dev)
    Zr = qi.make_Z(cfg, s0, s1, device=dev)
    Zfull[:, s0:s1] = Zr
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, cfg.s_block)
    pkg.qsgw_sigma_get_stats(plan, reset=True)
    S = pkg.qsgw_sigma_build(plan, B, eps_d, occ_d, Om_d[s0:s1], Zfull[:, s0:s1], cfg.eta)
    torch.cuda.synchronize()
    st = pkg.qsgw_sigma_get_stats(plan, reset=True)
    assert st["poles"] == s1 - s0
    assert st["kernel_launches"] >= 2 + 1 + 2 * 2 + 1, "one stage-1 launch and TWO stage-2/3 chunks must have run"
    assert torch.equal(S, S.T)
    states = _sample_states(cfg, n_random=4, seed=1)
    ref = oracle.sigma(B.cpu().numpy(), eps.numpy(), occ.numpy(), Om.numpy()[s0:s1], Zr.cpu().numpy(), cfg.eta,
                       cfg.n_occ, states=states)
    got = S.cpu().numpy()[np.ix_(states, states)]
    _assert_parity(got, ref, "large, multi-chunk pole range vs oracle")
    # the same call with stage 1 cut into two ranges (4096 + 160 poles)
    pkg.qsgw_sigma_limit_pole_batch(plan, cfg.s_block)
    S2 = pkg.qsgw_sigma_build(plan, B, eps_d, occ_d, Om_d[s0:s1], Zfull[:, s0:s1], cfg.eta)
    torch.cuda.synchronize()
    st2 = pkg.qsgw_sigma_get_stats(plan, reset=True)
    assert st2["kernel_launches"] > st["kernel_launches"], "a second stage-1 launch"
    _assert_parity(S2.cpu().numpy()[np.ix_(states, states)], ref, "large, two stage-1 ranges vs oracle")
    pkg.qsgw_sigma_limit_pole_batch(plan, cfg.n_pole)
    # additivity: the same range in two pieces through the streaming calls
    pkg.qsgw_sigma_begin(plan, B, eps_d, occ_d, cfg.eta)
    mid = 4096
    pkg.qsgw_sigma_add_poles(plan, Om_d[s0:mid], Zfull[:, s0:mid])
    pkg.qsgw_sigma_add_poles(plan, Om_d[mid:s1], Zfull[:, mid:s1])
    S_parts = pkg.qsgw_sigma_finish(plan)
    torch.cuda.synchronize()
    scale = float(S.abs().max())
    assert float((S_parts - S).abs().max()) <= 1e-12 * scale
    pkg.qsgw_sigma_destroy(plan)


XL_RANGE = 2 * qi.CONFIGS["xl"].s_block     # poles per qsgw_sigma_add_poles call of the xl runs (bench.py uses the same)


def test_xl_config_multi_chunk_pole_range_vs_oracle_on_sampled_states():
    """`xl` (N = 1000, naux = 4000, (ia) = 127500) with the config's RANDOM B and Z, plan as bench.py creates it for the
    streamed build (n_pole_max = 8192 = two s-blocks).  begin, ONE qsgw_sigma_add_poles call over 4096 + 128 poles (a full
    w chunk and a ragged one: the chunk loop runs twice; row offsets (m N + p) ldw reach 4.1e9 > 2^32), finish.  Sampled
    states S x S -- deepest, HOMO, LUMO, highest, tile-edge neighbours, random -- against oracle.sigma on those poles
    (SURVEY.md 8(c) "xl parity (i)")."""
    pkg = _pkg()
    cfg = qi.CONFIGS["xl"]
    dev = torch.device("cuda", 0)
    free, _ = torch.cuda.mem_get_info()
    if free < 120e9:
        pytest.skip("needs ~110 GB of free device memory")
    s0 = 61000                                                   # mid-spectrum poles (Omega ~ 3 Ha)
    s1 = s0 + cfg.s_block + 128
    B = qi.make_B(cfg, dev)
    eps, occ, Om = qi.make_eps(cfg), qi.make_occ(cfg), qi.make_omega(cfg)
    eps_d, occ_d, Om_d = eps.to(dev), occ.to(dev), Om.to(dev)
    Zr = qi.make_Z(cfg, s0, s1, device=dev)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, XL_RANGE, cfg.s_block)
    pkg.qsgw_sigma_get_stats(plan, reset=True)
    pkg.qsgw_sigma_begin(plan, B, eps_d, occ_d, cfg.eta)
    pkg.qsgw_sigma_add_poles(plan, Om_d[s0:s1], Zr)
    S = pkg.qsgw_sigma_finish(plan)
    torch.cuda.synchronize()
    st = pkg.qsgw_sigma_get_stats(plan, reset=True)
    assert st["poles"] == s1 - s0 and st["kernel_launches"] >= 2 + 1 + 2 * 2 + 1
    assert torch.equal(S, S.T)
    N, o = cfg.n_mo, cfg.n_occ
    states = sorted({0, o - 1, o, N - 1, 63, 64, 255, 256, 959, 960, 417, 702})
    B_h = B.cpu().numpy()
    pkg.qsgw_sigma_destroy(plan)
    del B
    torch.cuda.empty_cache()
    ref = oracle.sigma(B_h, eps.numpy(), occ.numpy(), Om.numpy()[s0:s1], Zr.cpu().numpy(), cfg.eta, cfg.n_occ, states=states)
    got = S.cpu().numpy()[np.ix_(states, states)]
    _assert_parity(got, ref, "xl, multi-chunk pole range vs oracle")


def test_xl_config_streamed_build_separable_closed_form():
    """`xl` as bench.py runs it: begin, 16 add_poles calls of <= 8192 poles = two s-blocks each (Z produced range by
    range on the device: 130 GB whole), finish.  Separable inputs, closed form on sampled states."""
    pkg = _pkg()
    cfg = qi.CONFIGS["xl"]
    dev = torch.device("cuda", 0)
    free, _ = torch.cuda.mem_get_info()
    if free < 120e9:
        pytest.skip("needs ~110 GB of free device memory")
    c, u, z, t, B = _separable_inputs(cfg, dev, seed=4321)
    eps, occ, Om = qi.make_eps(cfg), qi.make_occ(cfg), qi.make_omega(cfg)
    eps_d, occ_d, Om_d, z_d, t_d = eps.to(dev), occ.to(dev), Om.to(dev), z.to(dev), t.to(dev)
    rng = XL_RANGE
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, rng, cfg.s_block)
    Zbuf = [torch.empty((cfg.n_ov, rng), dtype=torch.float64, device=dev) for _ in range(2)]
    pkg.qsgw_sigma_begin(plan, B, eps_d, occ_d, cfg.eta)
    for k, a in enumerate(range(0, cfg.n_pole, rng)):
        b = min(cfg.n_pole, a + rng)
        zb = Zbuf[k % 2][:, : b - a]
        torch.outer(z_d, t_d[a:b], out=zb)
        pkg.qsgw_sigma_add_poles(plan, Om_d[a:b], zb)
    S = pkg.qsgw_sigma_finish(plan)
    torch.cuda.synchronize()
    assert torch.equal(S, S.T)
    states = _sample_states(cfg, n_random=4, seed=2)
    ref = _separable_reference(c.numpy(), u.numpy(), z.numpy(), t.numpy(), eps.numpy(), occ.numpy(), Om.numpy(),
                               cfg.eta, cfg.n_occ, states)
    got = S.cpu().numpy()[np.ix_(states, states)]
    _assert_parity(got, ref, "xl, separable closed form")
    pkg.qsgw_sigma_destroy(plan)


def test_large_config_g0w0_diagonal_pole_subrange_vs_oracle_on_sampled_states():
    """Row 8(f).1 at the full N, naux, (ia) of `large`: 1024 poles straddling the s-block edge, 8 grid points, sampled
    states against oracle.sigma_diag."""
    pkg = _pkg()
    cfg = qi.CONFIGS["large"]
    dev = torch.device("cuda", 0)
    s0, s1 = 4096 - 500, 4096 + 524
    B = qi.make_B(cfg, dev)
    eps, occ, Om = qi.make_eps(cfg), qi.make_occ(cfg), qi.make_omega(cfg)
    eps_d, occ_d, Om_d = eps.to(dev), occ.to(dev), Om.to(dev)
    Zr = qi.make_Z(cfg, s0, s1, device=dev)
    grid = np.array([-2.0, float(eps[cfg.n_occ - 1]), float(eps[cfg.n_occ]), 0.0, 0.731, float(eps[0] - Om[s0 + 3]), 3.3, 6.5])
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, cfg.s_block)
    re, im = pkg.qsgw_sigma_diag_build(plan, B, eps_d, occ_d, Om_d[s0:s1], Zr, cfg.eta, torch.from_numpy(grid).to(dev))
    torch.cuda.synchronize()
    states = _sample_states(cfg, n_random=2, seed=3)
    ref_re, ref_im = oracle.sigma_diag(B.cpu().numpy(), eps.numpy(), occ.numpy(), Om.numpy()[s0:s1], Zr.cpu().numpy(),
                                       cfg.eta, cfg.n_occ, grid, states=states)
    _assert_parity(re.cpu().numpy()[states], ref_re, "large, G0W0 diagonal Re")
    _assert_parity(im.cpu().numpy()[states], ref_im, "large, G0W0 diagonal Im")
    pkg.qsgw_sigma_destroy(plan)


def test_large_config_ao_to_mo_sampled_auxiliary_functions():
    """Row 8(f).2 at `large` (n_ao = N = 600, naux = 2400), as bench.py --path aomo runs it; the oracle transforms
    a sample of the auxiliary functions (each P is independent)."""
    pkg = _pkg()
    cfg = qi.CONFIGS["large"]
    dev = torch.device("cuda", 0)
    B_ao = qi.make_B(cfg, dev)
    g = torch.Generator(device=dev); g.manual_seed(11)
    C, _ = torch.linalg.qr(torch.randn((cfg.n_mo, cfg.n_mo), generator=g, dtype=torch.float64, device=dev))
    C = C.contiguous()
    B_mo = pkg.qsgw_ri_ao_to_mo(B_ao, C)
    torch.cuda.synchronize()
    sample = [0, 127, 1199, 2399]                    # the oracle is the O(N^4) double sum per auxiliary function
    ref = oracle.ao_to_mo(B_ao[sample].cpu().numpy(), C.cpu().numpy())
    _assert_parity(B_mo[sample].cpu().numpy(), ref, "large, AO->MO")
    # an orthogonal C preserves the trace of every B[P]: a property checked on ALL 2400 auxiliary functions
    tr_ao = torch.diagonal(B_ao, dim1=1, dim2=2).sum(-1)
    tr_mo = torch.diagonal(B_mo, dim1=1, dim2=2).sum(-1)
    assert float((tr_ao - tr_mo).abs().max()) <= 1e-10 * float(B_ao.abs().max()) * cfg.n_mo
