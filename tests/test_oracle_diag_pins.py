"""Pins of the oracle's G0W0 diagonal self-energy on a frequency grid (oracle.sigma_diag; SURVEY.md 8(f).1,
Eq. (17) of the paper with m = n) against things other than itself.  No CUDA path involved."""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rand_case(rng, N, o, naux, n_s, frac_occ=False):
    v = N - o
    G = rng.normal(0, 0.3, (naux, N, N))
    B = 0.5 * (G + G.transpose(0, 2, 1))
    eps = np.concatenate([np.sort(rng.uniform(-1.5, -0.2, o)), np.sort(rng.uniform(0.05, 5.0, v))])
    occ = rng.uniform(0, 1, N) if frac_occ else np.concatenate([np.ones(o), np.zeros(v)])
    Om = np.sort(rng.uniform(0.2, 6.0, n_s))
    Z = rng.normal(0, 1, (o * v, n_s)) / np.sqrt(n_s)
    return B, eps, occ, Om, Z


def _golden_rows():
    rows = []
    for line in open(os.path.join(GOLDEN, "two_state_diag_grid.txt")):
        if line.strip() and not line.startswith("#"):
            rows.append([Fraction(t) for t in line.split()])
    return rows


@pytest.mark.parametrize("row", _golden_rows())
def test_hand_solved_two_state_case_on_grid(row):
    om, re00, im00, re11, im11 = row
    B = np.array([[[1.0, 0.5], [0.5, 2.0]]])
    re, im = oracle.sigma_diag(B, np.array([-0.5, 0.5]), np.array([1.0, 0.0]), np.array([1.0]), np.array([[1.0]]),
                               0.1, 1, np.array([float(om)]))
    assert re[0, 0] == pytest.approx(float(re00), rel=1e-14, abs=1e-15)
    assert im[0, 0] == pytest.approx(float(im00), rel=1e-14, abs=1e-15)
    assert re[1, 0] == pytest.approx(float(re11), rel=1e-14, abs=1e-15)
    assert im[1, 0] == pytest.approx(float(im11), rel=1e-14, abs=1e-15)


def _bruteforce_diag(B, eps, occ, Om, Z, eta, o, omega):
    """Eq. (18) verbatim through the 4-index (pm|ia), then Eq. (17) with m = n = p as Python complex numbers."""
    naux, N, _ = B.shape
    v = N - o
    out = np.zeros((N, len(omega)), dtype=complex)
    for p in range(N):
        for m in range(N):
            for s in range(len(Om)):
                w = 0.0
                for i in range(o):
                    for a in range(o, N):
                        pmia = sum(B[P, p, m] * B[P, i, a] for P in range(naux))
                        w += pmia * Z[i * v + (a - o), s]
                w *= np.sqrt(2.0)
                for k, om in enumerate(omega):
                    out[p, k] += w * w * (occ[m] / complex(om - eps[m] + Om[s], -eta)
                                          + (1.0 - occ[m]) / complex(om - eps[m] - Om[s], +eta))
    return out


@pytest.mark.parametrize("N,o,naux,n_s,seed,frac", [(4, 1, 3, 3, 1, False), (5, 2, 2, 4, 2, False), (6, 3, 4, 3, 3, True)])
def test_literal_complex_eq17_non_ri_bruteforce(N, o, naux, n_s, seed, frac):
    rng = np.random.default_rng(seed)
    B, eps, occ, Om, Z = _rand_case(rng, N, o, naux, n_s, frac_occ=frac)
    omega = np.array([-2.0, -0.3, 0.0, 0.77, 3.1])
    want = _bruteforce_diag(B, eps, occ, Om, Z, 0.05, o, omega)
    re, im = oracle.sigma_diag(B, eps, occ, Om, Z, 0.05, o, omega)
    scale = np.abs(want).max()
    assert np.max(np.abs(re - want.real)) <= 1e-12 * scale
    assert np.max(np.abs(im - want.imag)) <= 1e-12 * scale


def test_real_part_at_qp_energies_is_the_diagonal_of_the_qsgw_matrix():
    """Eq. (19) with m = n: Sigma^qsGW_pp = Re Sigma^GW_pp(eps_p).  oracle.sigma is pinned on its own
    (tests/test_oracle_pins.py); the two functions share only steps 1-2."""
    rng = np.random.default_rng(7)
    N, o = 11, 4
    B, eps, occ, Om, Z = _rand_case(rng, N, o, 6, 25)
    full = oracle.sigma(B, eps, occ, Om, Z, 1e-3, o)
    re, _ = oracle.sigma_diag(B, eps, occ, Om, Z, 1e-3, o, eps)       # grid = the QP energies themselves
    assert np.max(np.abs(np.diag(re) - np.diag(full))) <= 1e-12 * np.abs(np.diag(full)).max()


def test_exact_scaling_additivity_and_state_subset():
    rng = np.random.default_rng(9)
    N, o = 9, 3
    B, eps, occ, Om, Z = _rand_case(rng, N, o, 5, 12)
    omega = np.linspace(-3.0, 3.0, 7)
    re, im = oracle.sigma_diag(B, eps, occ, Om, Z, 0.02, o, omega)
    re2, im2 = oracle.sigma_diag(B, eps, occ, Om, 2.0 * Z, 0.02, o, omega)
    assert np.array_equal(re2, 4.0 * re) and np.array_equal(im2, 4.0 * im)          # w ~ Z, Sigma ~ w^2: exact
    ra, ia = oracle.sigma_diag(B, eps, occ, Om[:5], Z[:, :5], 0.02, o, omega)
    rb, ib = oracle.sigma_diag(B, eps, occ, Om[5:], Z[:, 5:], 0.02, o, omega)
    assert np.max(np.abs(ra + rb - re)) <= 1e-13 * np.abs(re).max()                 # plain sum over poles
    assert np.max(np.abs(ia + ib - im)) <= 1e-13 * max(np.abs(im).max(), 1e-300)
    rs, is_ = oracle.sigma_diag(B, eps, occ, Om, Z, 0.02, o, omega, states=[8, 0, 4])
    assert np.array_equal(rs, re[[8, 0, 4]]) and np.array_equal(is_, im[[8, 0, 4]])


def test_sign_of_imaginary_part_and_eta_to_zero_limit():
    """Occupied poles (omega - eps_i + Omega - i eta) give Im >= 0, empty ones (+ i eta) give Im <= 0; away from every
    pole Re -> sum w^2 / x with error <= eta^2/|x|^3 per term and Im = O(eta)."""
    rng = np.random.default_rng(11)
    N, o = 8, 3
    B, eps, occ, Om, Z = _rand_case(rng, N, o, 4, 10)
    omega = np.array([-9.0, 12.0])          # x1 = w - eps_i + Om and x2 = w - eps_a - Om are all far from zero
    only_occ = np.concatenate([np.ones(o), np.ones(N - o)])     # every state treated as occupied: one-signed Im
    _, im_occ = oracle.sigma_diag(B, eps, only_occ, Om, Z, 0.05, o, omega)
    _, im_emp = oracle.sigma_diag(B, eps, 0.0 * only_occ, Om, Z, 0.05, o, omega)
    assert np.all(im_occ >= 0.0) and np.all(im_emp <= 0.0) and im_occ.max() > 0.0 and im_emp.min() < 0.0
    V = oracle.pole_weights(B, Z, o)
    re, im = oracle.sigma_diag(B, eps, occ, Om, Z, 1e-6, o, omega)
    want = np.zeros((N, 2))
    for s in range(len(Om)):
        w = oracle.residues(B, V, s)                                   # [p][m]
        for k, om in enumerate(omega):
            x = om - eps[None, :] + np.where(occ[None, :] > 0.5, Om[s], -Om[s])
            want[:, k] += np.sum(w * w / x, axis=1)
    assert np.max(np.abs(re - want)) <= 1e-10 * np.abs(want).max()
    assert np.abs(im).max() <= 1e-5 * np.abs(want).max()
