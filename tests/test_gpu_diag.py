"""Parity of the G0W0 diagonal path (qsgw_sigma_diag_build: Eq. (17) with m = n on a frequency grid, SURVEY.md
8(f).1) against the CPU oracle (oracle.sigma_diag), element by element on the same seeded inputs.
Bar, as for the qsGW matrix: max|got - ref| <= 1e-9 * max|ref|, separately for the real and the imaginary part."""
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


def _grid(cfg, inp, n_omega, seed=0):
    """A grid spanning the QP energies, plus points ON poles (omega = eps_m -+ Omega_s exactly) and the eps themselves."""
    rng = np.random.default_rng(seed)
    eps, Om = inp.eps.numpy(), inp.Omega.numpy()
    g = list(np.linspace(eps.min() - 1.0, eps.max() + 1.0, max(n_omega - 4, 1)))
    g += [eps[0] - Om[0], eps[-1] + Om[-1], eps[cfg.n_occ - 1], eps[cfg.n_occ]]
    g = np.array(g[:n_omega]) if len(g) >= n_omega else np.array(g)
    rng.shuffle(g)                                   # the grid need not be sorted
    return np.ascontiguousarray(g)


def _run(cfg, inp, omega, s_block=None):
    pkg = _pkg()
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, cfg.s_block if s_block is None else s_block)
    dev = [t.cuda() for t in (inp.B, inp.eps, inp.occ, inp.Omega, inp.Z)]
    re, im = pkg.qsgw_sigma_diag_build(plan, *dev, cfg.eta, torch.from_numpy(omega).cuda())
    torch.cuda.synchronize()
    return re, im, plan, dev


def _assert_parity(got, ref, what):
    got = got.cpu().numpy()
    assert np.all(np.isfinite(got)), what
    err, scale = np.max(np.abs(got - ref)), np.max(np.abs(ref))
    assert err <= TOL * scale, f"{what}: max|d| = {err:.3e} > {TOL:g} * {scale:.3e}"


def _ref(cfg, inp, omega):
    return oracle.sigma_diag(inp.B.numpy(), inp.eps.numpy(), inp.occ.numpy(), inp.Omega.numpy(), inp.Z.numpy(),
                             cfg.eta, cfg.n_occ, omega)


@pytest.mark.parametrize("name,n_omega", [("tiny", 13), ("small", 24)])
def test_config_parity(name, n_omega):
    cfg = qi.CONFIGS[name]
    inp = qi.make_inputs(cfg)
    omega = _grid(cfg, inp, n_omega)
    re, im, plan, _ = _run(cfg, inp, omega)
    ref_re, ref_im = _ref(cfg, inp, omega)
    _assert_parity(re, ref_re, f"{name} Re")
    _assert_parity(im, ref_im, f"{name} Im")
    _pkg().qsgw_sigma_destroy(plan)


@pytest.mark.parametrize("n_mo,n_occ,n_aux,n_pole,s_block,n_omega", [
    (37, 7, 53, 210, 64, 1),          # one grid point; several chunks with a short last one
    (130, 3, 17, 381, 128, 9),        # n_omega = 8 + 1: a second, nearly empty grid tile
    (24, 23, 9, 23, 0, 16),
    (2, 1, 1, 1, 0, 3),
])
def test_ragged_shapes_parity(n_mo, n_occ, n_aux, n_pole, s_block, n_omega):
    cfg = qi.custom_config(n_mo, n_occ, n_aux, n_pole=n_pole, s_block=s_block, seed=300 + n_mo)
    inp = qi.make_inputs(cfg)
    omega = _grid(cfg, inp, n_omega, seed=n_mo)
    re, im, plan, _ = _run(cfg, inp, omega)
    ref_re, ref_im = _ref(cfg, inp, omega)
    _assert_parity(re, ref_re, "Re")
    _assert_parity(im, ref_im, "Im")
    _pkg().qsgw_sigma_destroy(plan)


def test_fractional_occupations():
    cfg = qi.custom_config(40, 6, 20, n_pole=90, seed=9)
    inp = qi.make_inputs(cfg)
    g = torch.Generator().manual_seed(3)
    inp.occ = torch.rand(cfg.n_mo, generator=g, dtype=torch.float64)
    inp.occ[0], inp.occ[1] = 1.0, 0.0
    omega = _grid(cfg, inp, 11)
    re, im, plan, _ = _run(cfg, inp, omega)
    ref_re, ref_im = _ref(cfg, inp, omega)
    _assert_parity(re, ref_re, "Re")
    _assert_parity(im, ref_im, "Im")
    _pkg().qsgw_sigma_destroy(plan)


def test_real_part_at_qp_energies_is_the_diagonal_of_the_qsgw_matrix_and_runs_are_reproducible():
    pkg = _pkg()
    cfg = qi.custom_config(96, 12, 60, n_pole=700, s_block=250, seed=12)
    inp = qi.make_inputs(cfg)
    omega = inp.eps.numpy().copy()                       # grid = the QP energies: Eq. (19) with m = n
    re, im, plan, dev = _run(cfg, inp, omega)
    S = pkg.qsgw_sigma_build(plan, *dev, cfg.eta)
    torch.cuda.synchronize()
    d_gw = torch.diagonal(re).cpu().numpy()
    d_qs = torch.diagonal(S).cpu().numpy()
    assert np.max(np.abs(d_gw - d_qs)) <= 1e-11 * np.abs(d_qs).max()
    re2, im2 = pkg.qsgw_sigma_diag_build(plan, *dev, cfg.eta, torch.from_numpy(omega).cuda())
    assert torch.equal(re, re2) and torch.equal(im, im2)
    with pytest.raises(pkg.QsgwSigmaError):
        pkg.qsgw_sigma_diag_build(plan, *dev, 0.0, torch.from_numpy(omega).cuda())      # eta <= 0
    pkg.qsgw_sigma_destroy(plan)


def test_medium_config_sampled_grid_parity():
    """N = 300, n_s = 10400, s-block 2048 (6 chunks); the oracle computes 12 sampled states x 8 grid points."""
    pkg = _pkg()
    cfg = qi.CONFIGS["medium"]
    inp = qi.make_inputs(cfg)
    omega = _grid(cfg, inp, 8)
    re, im, plan, _ = _run(cfg, inp, omega)
    states = [0, 1, 38, 39, 40, 41, 127, 128, 200, 255, 298, 299]
    ref_re, ref_im = oracle.sigma_diag(inp.B.numpy(), inp.eps.numpy(), inp.occ.numpy(), inp.Omega.numpy(),
                                       inp.Z.numpy(), cfg.eta, cfg.n_occ, omega, states=states)
    _assert_parity(re[states], ref_re, "medium Re")
    _assert_parity(im[states], ref_im, "medium Im")
    pkg.qsgw_sigma_destroy(plan)
