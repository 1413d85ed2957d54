"""Pins of oracle.mp2_direct (second-order Coulomb term of the qsMP2 self-energy, first sum of Eq. (20) in Eq. (21),
PAPER.md:174-186) against things other than itself.  No CUDA path involved."""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _case(rng, N, o, naux, sym=True):
    G = rng.normal(0, 0.3, (naux, N, N))
    B = 0.5 * (G + G.transpose(0, 2, 1)) if sym else G
    eps = np.concatenate([np.sort(rng.uniform(-1.5, -0.2, o)), np.sort(rng.uniform(0.05, 5.0, N - o))])
    occ = np.concatenate([np.ones(o), np.zeros(N - o)])
    return B, eps, occ


def test_hand_solved_two_state_case():
    """N = 2, one (i, a) pair, eps_a - eps_i = 1: the direct MP2 term is the GW expression with Omega = 1 and
    w^2 = 2 (pm|ia)^2 (spin factor 2 here, sqrt(2)^2 there) -- the same exact rationals as
    tests/golden/two_state_single_pole.txt (Sigma = 1/4 sum_m B_pm B_qm [D_m(eps_p) + D_m(eps_q)] with B_01 = 1/2 ...)."""
    rows = [line.split() for line in open(os.path.join(GOLDEN, "two_state_single_pole.txt"))
            if line.strip() and not line.startswith("#")]
    eta, s00, s01, s11 = [Fraction(t) for t in rows[1]]           # the eta = 1/10 line
    # (mp|ia) = B_mp * B_01 with B_01 = 1/2; the golden example has V = B_01 * Z = 1/2, i.e. the same numbers
    B = np.array([[[1.0, 0.5], [0.5, 2.0]]])
    S = oracle.mp2_direct(B, np.array([-0.5, 0.5]), np.array([1.0, 0.0]), float(eta), 1)
    assert S[0, 0] == pytest.approx(float(s00), rel=1e-14)
    assert S[0, 1] == pytest.approx(float(s01), rel=1e-14) and S[1, 0] == pytest.approx(float(s01), rel=1e-14)
    assert S[1, 1] == pytest.approx(float(s11), rel=1e-14)


def _bruteforce(B, eps, occ, eta, o):
    """Eq. (20), first sum, literally: 4-index integrals, both spins of sigma' summed explicitly, complex denominators;
    then Eq. (21) and the real part."""
    naux, N, _ = B.shape
    eri = np.einsum("Pmp,Pia->mpia", B, B)                      # (mp|ia)
    def sigma_w(m, n, w):
        tot = 0.0 + 0.0j
        for spin in range(2):                                   # sigma' = up, down: same spatial integrals (closed shell)
            for i in range(o):
                for a in range(o, N):
                    for p in range(N):
                        num = eri[m, p, i, a] * eri[p, n, a, i]
                        tot += num * (occ[p] / complex(w + eps[a] - eps[i] - eps[p], -eta)
                                      + (1.0 - occ[p]) / complex(w + eps[i] - eps[a] - eps[p], +eta))
        return tot
    out = np.zeros((N, N))
    for m in range(N):
        for n in range(N):
            out[m, n] = 0.5 * (sigma_w(m, n, eps[n]) + sigma_w(n, m, eps[m])).real
    return out


@pytest.mark.parametrize("N,o,naux,seed,sym", [(4, 1, 3, 1, True), (5, 2, 2, 2, True), (5, 3, 3, 3, False)])
def test_literal_eq20_first_sum(N, o, naux, seed, sym):
    rng = np.random.default_rng(seed)
    B, eps, occ = _case(rng, N, o, naux, sym)
    want = _bruteforce(B, eps, occ, 0.05, o)
    got = oracle.mp2_direct(B, eps, occ, 0.05, o)
    assert np.max(np.abs(got - want)) <= 1e-12 * np.abs(want).max()


def test_equals_the_gw_expression_with_unit_z_and_orbital_energy_differences():
    """(mp|ia) is the GW residue of Eq. (18) for X+Y = 1 and Omega_s = eps_a - eps_i: oracle.sigma (pinned on its own)
    with Z = identity reproduces the direct MP2 term -- which is how the CUDA path computes it."""
    rng = np.random.default_rng(5)
    N, o, naux = 9, 3, 6
    B, eps, occ = _case(rng, N, o, naux)
    Om = np.array([eps[a] - eps[i] for i in range(o) for a in range(o, N)])
    want = oracle.sigma(B, eps, occ, Om, np.eye(o * (N - o)), 1e-3, o)
    got = oracle.mp2_direct(B, eps, occ, 1e-3, o)
    assert np.max(np.abs(got - want)) <= 1e-12 * np.abs(want).max()
    assert np.max(np.abs(got - got.T)) <= 1e-13 * np.abs(got).max()
