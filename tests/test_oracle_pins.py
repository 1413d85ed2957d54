"""Pins of the CPU oracle (oracle/qsgw_oracle.c) against things other than itself.

Every test here checks the oracle against something the paper's equations and plain
mathematics fix independently (SURVEY.md 8(c) "What pins each part"): a hand-solved case
with exact rationals, a literal complex evaluation of Eq. (17), the non-RI 4-index form of
Eq. (18), closed forms, invariants.  None of them calls the CUDA path.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
import qsgw_inputs as qi

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rand_case(rng, N, o, naux, n_s, sym=True, frac_occ=False):
    v = N - o
    G = rng.normal(0, 0.3, (naux, N, N))
    B = 0.5 * (G + G.transpose(0, 2, 1)) if sym else G
    eps = np.concatenate([np.sort(rng.uniform(-1.5, -0.2, o)), np.sort(rng.uniform(0.05, 5.0, v))])
    occ = np.concatenate([np.ones(o), np.zeros(v)])
    if frac_occ:
        occ = rng.uniform(0, 1, N)
    Om = np.sort(rng.uniform(0.2, 6.0, n_s))
    Z = rng.normal(0, 1, (o * v, n_s)) / np.sqrt(n_s)
    return B, eps, occ, Om, Z


def _tiny():
    cfg = qi.CONFIGS["tiny"]
    inp = qi.make_inputs(cfg, "cpu")
    return cfg, [t.numpy() for t in (inp.B, inp.eps, inp.occ, inp.Omega, inp.Z)]


# ---------------------------------------------------------------- pin 1: hand-solved two-state case
def _golden_rows():
    rows = []
    with open(os.path.join(GOLDEN, "two_state_single_pole.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            rows.append([Fraction(tok) for tok in line.split()])
    return rows


@pytest.mark.parametrize("row", _golden_rows())
def test_hand_solved_two_state_single_pole(row):
    eta, s00, s01, s11 = row
    B = np.array([[[1.0, 0.5], [0.5, 2.0]]])
    eta_f = float(eta) if eta != 0 else 1e-9           # eta -> 0 limit: |D(eta)-1/x| <= eta^2/|x|^3
    S = oracle.sigma(B, [-0.5, 0.5], [1.0, 0.0], [1.0], [[1.0]], eta_f, n_occ=1)
    want = np.array([[float(s00), float(s01)], [float(s01), float(s11)]])
    tol = 1e-14 if eta != 0 else 1e-15 + 4 * eta_f ** 2
    assert np.max(np.abs(S - want)) <= tol * max(1.0, np.abs(want).max())


def test_hand_solved_intermediates():
    B = np.array([[[1.0, 0.5], [0.5, 2.0]]])
    V = oracle.pole_weights(B, [[1.0]], n_occ=1)
    assert V.shape == (1, 1) and V[0, 0] == 0.5
    w = oracle.residues(B, V, 0)
    assert np.allclose(w, np.sqrt(2.0) / 2 * B[0], rtol=0, atol=1e-16)


# ---------------------------------------------------------------- pin 2: literal complex Eq. (17)
def test_D_is_real_part_of_eq17_terms():
    rng = np.random.default_rng(5)
    for _ in range(200):
        f = rng.choice([0.0, 1.0, rng.uniform()])
        em, Om, om = rng.uniform(-2, 5), rng.uniform(0.2, 6), rng.uniform(-2, 5)
        eta = 10 ** rng.uniform(-4, -1)
        lit = (f / complex(om - em + Om, -eta) + (1 - f) / complex(om - em - Om, +eta)).real
        got = oracle.D(f, em, Om, om, eta)
        assert abs(got - lit) <= 1e-13 * max(1.0, abs(lit))
    # the sign of i*eta does not matter for the real part (reading #3)
    assert oracle.D(1.0, 0.3, 1.0, 0.1, 0.05) == pytest.approx((1 / complex(0.1 - 0.3 + 1.0, +0.05)).real, rel=1e-14)
    # x == 0 gives 0, no singularity (reading #4)
    assert oracle.D(1.0, 1.0, 0.5, 0.5, 1e-3) == 0.0


# ---------------------------------------------------------------- pin 3: non-RI brute force of Eq. (18) + Eq. (17)/(19)
def _bruteforce_sigma(B, eps, occ, Om, Z, eta, o):
    """Eq. (18) verbatim with 4-index integrals, then Eqs. (17),(19) with complex arithmetic; pure Python loops."""
    naux, N, _ = B.shape
    v = N - o
    n_s = len(Om)
    eri = np.zeros((N, N, o, v))                       # (pm|ia) = sum_P B^P_pm B^P_ia
    for p in range(N):
        for m in range(N):
            for i in range(o):
                for a in range(v):
                    eri[p, m, i, a] = sum(B[P, p, m] * B[P, i, o + a] for P in range(naux))
    w = np.zeros((n_s, N, N))
    for s in range(n_s):
        for p in range(N):
            for m in range(N):
                w[s, p, m] = np.sqrt(2.0) * sum(eri[p, m, i, a] * Z[i * v + a, s] for i in range(o) for a in range(v))

    def sig_gw(p, q, omega):                           # Eq. (17), complex, then real part
        t = 0j
        for m in range(N):
            for s in range(n_s):
                t += w[s, p, m] * w[s, q, m] * (occ[m] / complex(omega - eps[m] + Om[s], -eta)
                                                + (1 - occ[m]) / complex(omega - eps[m] - Om[s], +eta))
        return t.real

    S = np.zeros((N, N))
    for p in range(N):
        for q in range(N):
            S[p, q] = 0.5 * (sig_gw(p, q, eps[q]) + sig_gw(q, p, eps[p]))   # Eq. (19)
    return S, w


@pytest.mark.parametrize("N,o,naux,n_s,seed", [(4, 1, 3, 3, 0), (5, 2, 4, 6, 1), (6, 3, 2, 5, 2), (7, 2, 5, 4, 3)])
def test_bruteforce_non_ri_small_random(N, o, naux, n_s, seed):
    rng = np.random.default_rng(seed)
    B, eps, occ, Om, Z = _rand_case(rng, N, o, naux, n_s, sym=(seed % 2 == 0))   # odd seeds: B NOT symmetric
    want, w_want = _bruteforce_sigma(B, eps, occ, Om, Z, 0.02, o)
    got = oracle.sigma(B, eps, occ, Om, Z, 0.02, o)
    assert np.max(np.abs(got - want)) <= 1e-12 * np.abs(want).max()
    V = oracle.pole_weights(B, Z, o)
    for s in range(n_s):
        assert np.max(np.abs(oracle.residues(B, V, s) - w_want[s])) <= 1e-13 * np.abs(w_want).max()


def test_einsum_restatement_tiny_config():
    """tiny config (N=24): same definition through numpy einsum on the 4-index integrals (non-RI route)."""
    cfg, (B, eps, occ, Om, Z) = _tiny()
    o, v, N = cfg.n_occ, cfg.n_virt, cfg.n_mo
    eri = np.einsum("Ppm,Pia->pmia", B, B[:, :o, o:])                       # (pm|ia)
    w = np.sqrt(2.0) * np.einsum("pmia,ias->spm", eri, Z.reshape(o, v, -1))  # Eq. (18)
    om_p = eps[:, None, None]                                               # omega = eps_p
    x1 = om_p - eps[None, :, None] + Om[None, None, :]
    x2 = om_p - eps[None, :, None] - Om[None, None, :]
    Dp = (occ[None, :, None] / (x1 - 1j * cfg.eta) + (1 - occ[None, :, None]) / (x2 + 1j * cfg.eta)).real  # [p,m,s]
    T = np.einsum("spm,sqm,pms->pq", w, w, Dp)
    want = 0.5 * (T + T.T)
    got = oracle.sigma(B, eps, occ, Om, Z, cfg.eta, o)
    assert np.max(np.abs(got - want)) <= 1e-12 * np.abs(want).max()


# ---------------------------------------------------------------- pins 4-8: invariants
def test_symmetric_output():
    cfg, (B, eps, occ, Om, Z) = _tiny()
    S = oracle.sigma(B, eps, occ, Om, Z, cfg.eta, cfg.n_occ)
    assert np.max(np.abs(S - S.T)) <= 1e-13 * np.abs(S).max()


def test_exact_power_of_two_scaling():
    cfg, (B, eps, occ, Om, Z) = _tiny()
    S = oracle.sigma(B, eps, occ, Om, Z, cfg.eta, cfg.n_occ)
    assert np.array_equal(oracle.sigma(B, eps, occ, Om, 2.0 * Z, cfg.eta, cfg.n_occ), 4.0 * S)      # Sigma ~ Z^2
    assert np.array_equal(oracle.sigma(2.0 * B, eps, occ, Om, Z, cfg.eta, cfg.n_occ), 16.0 * S)     # Sigma ~ B^4


def test_additive_over_poles_and_quadratic_per_pole():
    cfg, (B, eps, occ, Om, Z) = _tiny()
    S = oracle.sigma(B, eps, occ, Om, Z, cfg.eta, cfg.n_occ)
    cuts = [0, 7, 40, 41, cfg.n_pole]
    parts = [oracle.sigma(B, eps, occ, Om[a:b], Z[:, a:b], cfg.eta, cfg.n_occ) for a, b in zip(cuts[:-1], cuts[1:])]
    assert np.max(np.abs(sum(parts) - S)) <= 1e-13 * np.abs(S).max()
    # scaling ONE pole's eigenvector by c scales that pole's contribution by c^2
    s, c = 13, 3.0
    Zc = Z.copy()
    Zc[:, s] *= c
    S_one = oracle.sigma(B, eps, occ, Om[s:s + 1], Z[:, s:s + 1], cfg.eta, cfg.n_occ)
    assert np.max(np.abs(oracle.sigma(B, eps, occ, Om, Zc, cfg.eta, cfg.n_occ) - (S + (c * c - 1) * S_one))) \
        <= 1e-12 * np.abs(S).max()


def test_eta_to_zero_limit_away_from_poles():
    rng = np.random.default_rng(11)
    N, o, naux, n_s = 9, 3, 6, 12
    B, eps, occ, Om, Z = _rand_case(rng, N, o, naux, n_s)
    Om = np.sort(rng.uniform(8.0, 12.0, n_s))            # Omega_min > eps_max - eps_min: every x1 > 0, every x2 < 0
    V = oracle.pole_weights(B, Z, o)
    w = np.stack([oracle.residues(B, V, s) for s in range(n_s)])
    sign = np.where(occ > 0.5, 1.0, -1.0)
    x = eps[:, None, None] - eps[None, :, None] + sign[None, :, None] * Om[None, None, :]   # [p,m,s]
    assert np.abs(x).min() > 2.0
    T = np.einsum("spm,sqm,pms->pq", w, w, 1.0 / x)
    want = 0.5 * (T + T.T)
    got = oracle.sigma(B, eps, occ, Om, Z, 1e-6, o)
    assert np.max(np.abs(got - want)) <= 1e-11 * np.abs(want).max()


def test_null_case_zero_ov_block():
    cfg, (B, eps, occ, Om, Z) = _tiny()
    B0 = B.copy()
    B0[:, :cfg.n_occ, cfg.n_occ:] = 0.0                  # stage 1 reads exactly B[P][i][a], i<o<=a
    assert np.array_equal(oracle.sigma(B0, eps, occ, Om, Z, cfg.eta, cfg.n_occ), np.zeros((cfg.n_mo, cfg.n_mo)))
    B1 = B.copy()
    B1[:, cfg.n_occ:, :cfg.n_occ] = 0.0                  # ...and NOT the transposed block B[P][a][i]
    S1 = oracle.sigma(B1, eps, occ, Om, Z, cfg.eta, cfg.n_occ)
    assert np.abs(S1).max() > 0


# ---------------------------------------------------------------- pin 9: separable closed form
def separable_case(rng, N, o, naux, n_s):
    v = N - o
    c = rng.normal(0, 1, naux)
    u = rng.normal(0, 1, N)
    z = rng.normal(0, 1, o * v)
    t = rng.normal(0, 1, n_s)
    B = c[:, None, None] * u[None, :, None] * u[None, None, :]
    Z = z[:, None] * t[None, :]
    return c, u, z, t, B, Z


def separable_sigma(c, u, z, t, eps, occ, Om, eta, o):
    """Sigma_pq = kappa^2 C2^2 u_p u_q [h(eps_p) + h(eps_q)],  h(w) = sum_m u_m^2 sum_s t_s^2 D_ms(w)."""
    N = len(u)
    v = N - o
    kappa = sum(u[i] * u[o + a] * z[i * v + a] for i in range(o) for a in range(v))
    C2 = float(np.sum(c * c))
    x1 = eps[:, None, None] - eps[None, :, None] + Om[None, None, :]
    x2 = eps[:, None, None] - eps[None, :, None] - Om[None, None, :]
    Dm = occ[None, :, None] * x1 / (x1 * x1 + eta * eta) + (1 - occ[None, :, None]) * x2 / (x2 * x2 + eta * eta)
    h = np.einsum("m,s,pms->p", u * u, t * t, Dm)
    return kappa ** 2 * C2 ** 2 * np.outer(u, u) * (h[:, None] + h[None, :])


def test_separable_closed_form():
    rng = np.random.default_rng(21)
    N, o, naux, n_s = 13, 4, 7, 30
    _, eps, occ, Om, _ = _rand_case(rng, N, o, naux, n_s)
    c, u, z, t, B, Z = separable_case(rng, N, o, naux, n_s)
    want = separable_sigma(c, u, z, t, eps, occ, Om, 1e-3, o)
    got = oracle.sigma(B, eps, occ, Om, Z, 1e-3, o)
    assert np.max(np.abs(got - want)) <= 1e-12 * np.abs(want).max()


# ---------------------------------------------------------------- pin 10: metamorphic permutations
def test_permutation_invariances():
    rng = np.random.default_rng(31)
    N, o, naux, n_s = 10, 4, 6, 15
    v = N - o
    B, eps, occ, Om, Z = _rand_case(rng, N, o, naux, n_s)
    eta = 5e-3
    S = oracle.sigma(B, eps, occ, Om, Z, eta, o)
    tol = 1e-12 * np.abs(S).max()
    ps = rng.permutation(n_s)                                   # poles: columns of Z together with Omega
    assert np.max(np.abs(oracle.sigma(B, eps, occ, Om[ps], Z[:, ps], eta, o) - S)) <= tol
    pP = rng.permutation(naux)                                  # auxiliary index
    assert np.max(np.abs(oracle.sigma(B[pP], eps, occ, Om, Z, eta, o) - S)) <= tol
    po, pv = rng.permutation(o), o + rng.permutation(v)         # states within the occupied / virtual sets
    perm = np.concatenate([po, pv])
    Bp = B[:, perm][:, :, perm]
    Zp = Z.reshape(o, v, n_s)[po][:, pv - o].reshape(o * v, n_s)
    Sp = oracle.sigma(Bp, eps[perm], occ[perm], Om, Zp, eta, o)
    assert np.max(np.abs(Sp - S[np.ix_(perm, perm)])) <= tol


# ---------------------------------------------------------------- pin 11: diagonal == G0W0 expression
def test_diagonal_reduces_to_g0w0():
    cfg, (B, eps, occ, Om, Z) = _tiny()
    S = oracle.sigma(B, eps, occ, Om, Z, cfg.eta, cfg.n_occ)
    V = oracle.pole_weights(B, Z, cfg.n_occ)
    w = np.stack([oracle.residues(B, V, s) for s in range(cfg.n_pole)])          # [s,p,m]
    for p in (0, cfg.n_occ - 1, cfg.n_occ, cfg.n_mo - 1):
        lit = 0.0
        for m in range(cfg.n_mo):                                               # Eq. (17) with m=n=p, omega=eps_p
            for s in range(cfg.n_pole):
                if occ[m] > 0.5:
                    lit += (w[s, p, m] ** 2 / complex(eps[p] - eps[m] + Om[s], -cfg.eta)).real
                else:
                    lit += (w[s, p, m] ** 2 / complex(eps[p] - eps[m] - Om[s], +cfg.eta)).real
        assert abs(S[p, p] - lit) <= 1e-12 * np.abs(S).max()


# ---------------------------------------------------------------- restricted-output mode used for sampled parity
def test_state_subset_matches_full():
    cfg, (B, eps, occ, Om, Z) = _tiny()
    S = oracle.sigma(B, eps, occ, Om, Z, cfg.eta, cfg.n_occ)
    st = [0, 4, 5, 23, 11]
    Ss = oracle.sigma(B, eps, occ, Om, Z, cfg.eta, cfg.n_occ, states=st)
    assert np.array_equal(Ss, S[np.ix_(st, st)])


def test_fractional_occupations_general_D():
    rng = np.random.default_rng(41)
    N, o, naux, n_s = 6, 2, 3, 4
    B, eps, occ, Om, Z = _rand_case(rng, N, o, naux, n_s, frac_occ=True)
    want, _ = _bruteforce_sigma(B, eps, occ, Om, Z, 0.03, o)
    got = oracle.sigma(B, eps, occ, Om, Z, 0.03, o)
    assert np.max(np.abs(got - want)) <= 1e-12 * np.abs(want).max()
