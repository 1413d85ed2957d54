"""Pins of oracle.ao_to_mo (RI AO->MO transformation of B; RI analogue of Eq. (16))
against things other than itself.  No CUDA path involved."""
import numpy as np

import oracle


def _case(rng, naux, nao, n_mo, sym=True):
    G = rng.normal(0, 1, (naux, nao, nao))
    B = 0.5 * (G + G.transpose(0, 2, 1)) if sym else G
    C = rng.normal(0, 1, (nao, n_mo))
    return B, C


def test_literal_double_sum_on_tiny_inputs():
    """B^P_pq = sum_mu sum_nu C[mu][p] C[nu][q] B^P_mu,nu written as four nested Python loops; B NOT symmetric, nao != n_mo,
    so a transposed operand or swapped index shows."""
    rng = np.random.default_rng(1)
    naux, nao, n_mo = 3, 5, 4
    B, C = _case(rng, naux, nao, n_mo, sym=False)
    want = np.zeros((naux, n_mo, n_mo))
    for P in range(naux):
        for p in range(n_mo):
            for q in range(n_mo):
                acc = 0.0
                for mu in range(nao):
                    for nu in range(nao):
                        acc += C[mu, p] * C[nu, q] * B[P, mu, nu]
                want[P, p, q] = acc
    got = oracle.ao_to_mo(B, C)
    assert got.shape == (naux, n_mo, n_mo)
    assert np.max(np.abs(got - want)) <= 1e-13 * np.abs(want).max()


def test_hand_solved_two_by_two():
    """nao = n_mo = 2, B = [[1, 2], [3, 4]] (unsymmetric), C = [[1, 2], [3, 5]]: C^T B C by hand.
    B C = [[7, 12], [15, 26]];  C^T (B C) = [[1*7 + 3*15, 1*12 + 3*26], [2*7 + 5*15, 2*12 + 5*26]] = [[52, 90], [89, 154]]."""
    B = np.array([[[1.0, 2.0], [3.0, 4.0]]])
    C = np.array([[1.0, 2.0], [3.0, 5.0]])
    assert np.array_equal(oracle.ao_to_mo(B, C), np.array([[[52.0, 90.0], [89.0, 154.0]]]))


def test_agrees_with_library_matmul():
    """C^T B C through numpy's matmul (a library routine the oracle does not call) on a non-square C."""
    rng = np.random.default_rng(5)
    B, C = _case(rng, 4, 11, 7, sym=False)
    want = np.matmul(C.T[None], np.matmul(B, C[None]))
    assert np.max(np.abs(oracle.ao_to_mo(B, C) - want)) <= 1e-13 * np.abs(want).max()


def test_identity_permutation_and_selection():
    rng = np.random.default_rng(2)
    B, _ = _case(rng, 4, 6, 6)
    assert np.array_equal(oracle.ao_to_mo(B, np.eye(6)), B)                      # C = 1
    perm = rng.permutation(6)
    Pm = np.eye(6)[:, perm]                                                     # orbital p = AO perm[p]
    assert np.array_equal(oracle.ao_to_mo(B, Pm), B[:, perm][:, :, perm])
    sel = np.eye(6)[:, [4, 1]]                                                  # two orbitals only: a 2 x 2 block
    assert np.array_equal(oracle.ao_to_mo(B, sel), B[:, [4, 1]][:, :, [4, 1]])


def test_composition_symmetry_linearity_and_trace():
    rng = np.random.default_rng(3)
    B, C1 = _case(rng, 3, 7, 7)
    C2 = rng.normal(0, 1, (7, 5))
    two_steps = oracle.ao_to_mo(oracle.ao_to_mo(B, C1), C2)
    one_step = oracle.ao_to_mo(B, C1 @ C2)                                      # (C1 C2)^T B (C1 C2)
    assert np.max(np.abs(two_steps - one_step)) <= 1e-12 * np.abs(one_step).max()
    out = oracle.ao_to_mo(B, C1)
    assert np.max(np.abs(out - out.transpose(0, 2, 1))) <= 1e-13 * np.abs(out).max()   # symmetric in, symmetric out
    assert np.array_equal(oracle.ao_to_mo(2.0 * B, C1), 2.0 * out)              # linear in B (exact for a power of two)
    assert np.array_equal(oracle.ao_to_mo(B, 2.0 * C1), 4.0 * out)              # quadratic in C
    Q, _ = np.linalg.qr(rng.normal(0, 1, (7, 7)))                               # orthogonal C preserves the trace
    tr = np.trace(oracle.ao_to_mo(B, Q), axis1=1, axis2=2)
    assert np.max(np.abs(tr - np.trace(B, axis1=1, axis2=2))) <= 1e-12 * np.abs(B).max() * 7
