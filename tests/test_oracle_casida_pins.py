"""Pins of the Casida / RPA oracle (oracle.casida_matrix, casida_z, casida; Eqs. (12)-(14), closed shell,
direct RPA, RI integrals) against things other than itself.  No CUDA path involved."""
import math

import numpy as np
import pytest

import oracle


def _case(rng, N, o, naux, scale=0.3):
    G = rng.normal(0, scale, (naux, N, N))
    B = 0.5 * (G + G.transpose(0, 2, 1))
    eps = np.concatenate([np.sort(rng.uniform(-1.5, -0.2, o)), np.sort(rng.uniform(0.05, 5.0, N - o))])
    return B, eps


def _delta_and_K(B, eps, o):
    N = B.shape[1]
    d = np.array([eps[a] - eps[i] for i in range(o) for a in range(o, N)])
    Bov = B[:, :o, o:].reshape(B.shape[0], -1)
    return d, Bov.T @ Bov                                         # K[ia,jb] = (ia|jb)


def test_hand_solved_single_pair():
    """N = 2, one (i, a) pair: Delta = 1, (ia|ia) = B_01^2 = 1/4.  A = Delta + 2K, B = 2K (singlet), so
    Omega^2 = (A-B)(A+B) = Delta (Delta + 4K) = 2, Omega = sqrt(2), and X + Y = sqrt(Delta / Omega) = 2^(-1/4)."""
    B = np.array([[[1.0, 0.5], [0.5, 2.0]]])
    eps = np.array([-0.5, 0.5])
    C = oracle.casida_matrix(B, eps, 1)
    assert C.shape == (1, 1) and C[0, 0] == 2.0
    Om, Z = oracle.casida(B, eps, 1)
    assert Om[0] == pytest.approx(math.sqrt(2.0), rel=1e-15)
    assert abs(Z[0, 0]) == pytest.approx(2.0 ** -0.25, rel=1e-15)


def test_hand_solved_two_pairs():
    """N = 3, o = 1: pairs (0,1), (0,2) with Delta = (1, 4) and one auxiliary function with B_01 = 1/2, B_02 = 1/4:
    K = [[1/4, 1/8], [1/8, 1/16]], C = diag(1, 16) + 4 sqrt(D) K sqrt(D) = [[2, 1], [1, 17]].
    Eigenvalues of [[2, 1], [1, 17]]: (19 -+ sqrt(229)) / 2."""
    B = np.zeros((1, 3, 3))
    B[0, 0, 1] = B[0, 1, 0] = 0.5
    B[0, 0, 2] = B[0, 2, 0] = 0.25
    eps = np.array([-1.0, 0.0, 3.0])
    C = oracle.casida_matrix(B, eps, 1)
    assert np.array_equal(C, np.array([[2.0, 1.0], [1.0, 17.0]]))
    Om, Z = oracle.casida(B, eps, 1)
    lam = np.array([(19 - math.sqrt(229)) / 2, (19 + math.sqrt(229)) / 2])
    assert np.max(np.abs(Om - np.sqrt(lam))) <= 1e-14
    # eigenvector of the lower root: (1, lam0 - 2) normalised; Z = sqrt(Delta) xi / sqrt(Omega)
    xi0 = np.array([1.0, lam[0] - 2.0]); xi0 /= np.linalg.norm(xi0)
    z0 = np.sqrt(np.array([1.0, 4.0])) * xi0 / math.sqrt(Om[0])
    assert min(np.max(np.abs(Z[:, 0] - z0)), np.max(np.abs(Z[:, 0] + z0))) <= 1e-14


@pytest.mark.parametrize("N,o,naux,seed", [(5, 2, 3, 1), (7, 3, 6, 2), (6, 1, 2, 3)])
def test_literal_non_symmetric_casida_equation(N, o, naux, seed):
    """Eq. (12) itself: the 2n x 2n matrix [[A, B], [-B, -A]] with A = Delta + 2K, B = 2K, diagonalised by a general
    (non-symmetric) library eigensolver.  Its positive eigenvalues are the oracle's Omega, and X + Y of the eigenvectors
    normalised to X^T X - Y^T Y = 1 is the oracle's Z up to the sign of each column."""
    rng = np.random.default_rng(seed)
    B, eps = _case(rng, N, o, naux)
    d, K = _delta_and_K(B, eps, o)
    n = len(d)
    A_, B_ = np.diag(d) + 2 * K, 2 * K
    M = np.block([[A_, B_], [-B_, -A_]])
    w, V = np.linalg.eig(M)
    assert np.max(np.abs(w.imag)) < 1e-12
    w, V = w.real, V.real
    pos = np.argsort(w)[n:]                                       # the n positive roots, ascending
    Om, Z = oracle.casida(B, eps, o)
    assert np.max(np.abs(w[pos] - Om)) <= 1e-11 * Om.max()
    for k, col in enumerate(pos):
        X, Y = V[:n, col], V[n:, col]
        nrm = X @ X - Y @ Y
        assert nrm > 0
        z = (X + Y) / math.sqrt(nrm)
        assert min(np.max(np.abs(z - Z[:, k])), np.max(np.abs(z + Z[:, k]))) <= 1e-9 * np.abs(Z[:, k]).max()


def test_sum_rules_and_bounds():
    """sum_s Omega_s Z_s Z_s^T = A - B = Delta and sum_s Z_s Z_s^T / Omega_s = (A + B)^-1 (completeness of the RPA
    eigenvectors); every Omega_s >= min Delta (the Coulomb kernel is positive semidefinite)."""
    rng = np.random.default_rng(7)
    B, eps = _case(rng, 9, 3, 8)
    d, K = _delta_and_K(B, eps, 3)
    Om, Z = oracle.casida(B, eps, 3)
    assert np.all(np.diff(Om) >= 0) and Om[0] >= d.min() * (1 - 1e-12)
    S1 = (Z * Om[None, :]) @ Z.T
    assert np.max(np.abs(S1 - np.diag(d))) <= 1e-12 * d.max()
    Sm1 = (Z / Om[None, :]) @ Z.T
    assert np.max(np.abs(Sm1 - np.linalg.inv(np.diag(d) + 4 * K))) <= 1e-11 * np.abs(Sm1).max()


def test_no_coupling_limit_and_scaling_of_the_kernel():
    """Zero ov block: Omega = sorted Delta and Z is a signed permutation.  C - Delta^2 is linear in K: scaling B by 2
    multiplies it by 4 exactly (power of two)."""
    rng = np.random.default_rng(9)
    B, eps = _case(rng, 6, 2, 4)
    d, _ = _delta_and_K(B, eps, 2)
    B0 = B.copy()
    B0[:, :2, 2:] = 0.0
    B0[:, 2:, :2] = 0.0
    Om, Z = oracle.casida(B0, eps, 2)
    assert np.max(np.abs(Om - np.sort(d))) <= 1e-14
    assert np.allclose(np.abs(Z).sum(axis=0), 1.0) and np.allclose(np.abs(Z).sum(axis=1), 1.0)
    C1, C2 = oracle.casida_matrix(B, eps, 2), oracle.casida_matrix(2.0 * B, eps, 2)
    D2 = np.diag(np.diag(oracle.casida_matrix(B0, eps, 2)))
    assert np.max(np.abs((C2 - D2) - 4.0 * (C1 - D2))) <= 1e-13 * np.abs(C1).max()
    assert np.max(np.abs(C1 - C1.T)) <= 1e-15 * np.abs(C1).max()


def test_matrix_agrees_with_a_library_restatement_and_feeds_the_sigma_oracle():
    rng = np.random.default_rng(11)
    N, o, naux = 8, 3, 5
    B, eps = _case(rng, N, o, naux)
    d, K = _delta_and_K(B, eps, o)
    want = np.diag(d * d) + 4 * np.sqrt(d)[:, None] * K * np.sqrt(d)[None, :]
    assert np.max(np.abs(oracle.casida_matrix(B, eps, o) - want)) <= 1e-13 * np.abs(want).max()
    Om, Z = oracle.casida(B, eps, o)
    occ = np.concatenate([np.ones(o), np.zeros(N - o)])
    S = oracle.sigma(B, eps, occ, Om, Z, 1e-3, o)                  # Omega > 0, Z of the right shape: the chain closes
    assert np.all(np.isfinite(S)) and np.max(np.abs(S - S.T)) <= 1e-12 * np.abs(S).max()
