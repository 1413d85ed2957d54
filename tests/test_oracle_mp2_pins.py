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


# ---------------------------------------------------------------- whole qsMP2: direct + second-order exchange
def _bruteforce_spin_orbital(B, eps, occ, eta, o):
    """Eq. (20) in spin orbitals, both sums literally: the direct sum runs over sigma' in {up, down}, the SOX sum has all
    spins equal; 4-index integrals (xy|zw) = sum_P B_xy B_zw; complex denominators; Eq. (21); real part."""
    naux, N, _ = B.shape
    eri = np.einsum("Pxy,Pzw->xyzw", B, B)
    def den(w, i, a, p):
        return (occ[p] / complex(w + eps[a] - eps[i] - eps[p], -eta)
                + (1.0 - occ[p]) / complex(w + eps[i] - eps[a] - eps[p], +eta))
    def sigma_w(m, n, w):
        tot = 0.0 + 0.0j
        for i in range(o):
            for a in range(o, N):
                for p in range(N):
                    d = den(w, i, a, p)
                    for spin in range(2):
                        tot += eri[m, p, i, a] * eri[p, n, a, i] * d          # direct, sigma' = spin
                    tot -= eri[m, p, i, a] * eri[p, i, a, n] * d              # SOX, one spin
        return tot
    out = np.zeros((N, N))
    for m in range(N):
        for n in range(N):
            out[m, n] = 0.5 * (sigma_w(m, n, eps[n]) + sigma_w(n, m, eps[m])).real
    return out


@pytest.mark.parametrize("N,o,naux,seed,sym", [(4, 1, 3, 1, True), (5, 2, 2, 2, True), (5, 3, 3, 3, False)])
def test_literal_eq20_both_sums(N, o, naux, seed, sym):
    rng = np.random.default_rng(seed)
    B, eps, occ = _case(rng, N, o, naux, sym)
    want = _bruteforce_spin_orbital(B, eps, occ, 0.05, o)
    got = oracle.mp2(B, eps, occ, 0.05, o)
    assert np.max(np.abs(got - want)) <= 1e-12 * np.abs(want).max()
    # the parts add up, and the direct part is the function pinned above
    sox = oracle.mp2(B, eps, occ, 0.05, o, sox_only=True)
    assert np.max(np.abs(oracle.mp2_direct(B, eps, occ, 0.05, o) + sox - got)) <= 1e-13 * np.abs(got).max()


def test_one_auxiliary_function_sox_is_minus_half_the_direct_term():
    """naux = 1: (mp|ia)(pi|an) = B_mp B_ia B_pi B_an and (mp|ia)(pn|ai) = B_mp B_ia B_pn B_ai; no general relation, but
    with a rank-one B = u u^T every 4-index integral factorises, (xy|zw) = u_x u_y u_z u_w, so SOX = -1/2 direct exactly."""
    rng = np.random.default_rng(8)
    N, o = 6, 2
    u = rng.normal(0, 1, N)
    B = np.outer(u, u)[None, :, :]
    _, eps, occ = _case(rng, N, o, 1)
    d = oracle.mp2_direct(B, eps, occ, 0.01, o)
    sox = oracle.mp2(B, eps, occ, 0.01, o, sox_only=True)
    assert np.max(np.abs(sox + 0.5 * d)) <= 1e-13 * np.abs(d).max()


@pytest.mark.parametrize("sym,sox_only", [(True, False), (False, False), (False, True)])
def test_states_restriction_equals_the_full_call(sym, sox_only):
    """oracle.mp2(states=S) (the gathered-copy variant used at sizes where the full sum is unaffordable) is the S x S
    block of the full literal call, for unsorted S with B NOT symmetric (so a row gather taken for a column gather, or
    (p S|ai) read as (S p|ai), shows), and for the exchange part alone."""
    rng = np.random.default_rng(11)
    N, o, naux = 9, 4, 5
    B, eps, occ = _case(rng, N, o, naux, sym=sym)
    full = oracle.mp2(B, eps, occ, 0.05, o, sox_only=sox_only)
    S = [7, 0, 3, 4]
    part = oracle.mp2(B, eps, occ, 0.05, o, sox_only=sox_only, states=S)
    assert part.shape == (4, 4)
    assert np.max(np.abs(part - full[np.ix_(S, S)])) <= 1e-13 * np.abs(full).max()
    one = oracle.mp2(B, eps, occ, 0.05, o, sox_only=sox_only, states=[5])
    assert one[0, 0] == pytest.approx(full[5, 5], rel=1e-12)
    allS = oracle.mp2(B, eps, occ, 0.05, o, sox_only=sox_only, states=list(range(N)))
    assert np.max(np.abs(allS - full)) <= 1e-13 * np.abs(full).max()
