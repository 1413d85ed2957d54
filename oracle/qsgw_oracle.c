/*
 * qsgw_oracle.c -- TEST INFRASTRUCTURE, not product code.
 *
 * Plain, slow, obviously-correct CPU FP64 statement of what the qsGW correlation
 * self-energy path computes, written from the paper's equations (arxiv 2210.17093,
 * /root/reference/PAPER.md) in its resolution-of-identity (RI) form.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or helper with the
 * CUDA path under paper_2210_17093_b200/csrc/, and neither includes the other.
 *
 * What it computes (Eqs. (17)-(19); RI remark PAPER.md:120):
 *
 *   1. V[P][s]    = sum_{i<o} sum_{a>=o} B[P][i][a] * Z[i*v + (a-o)][s]        first half of Eq. (18)
 *   2. w[s][p][m] = sqrt(2) * sum_P B[P][p][m] * V[P][s]                        second half of Eq. (18)
 *   3. Sigma[p][q] = 1/2 * sum_m sum_s w[s][p][m] w[s][q][m] (D(m,s,eps[p]) + D(m,s,eps[q]))
 *                                                                              Eq. (17) put into Eq. (19)
 *      D(m,s,omega) = occ[m]     * x1/(x1*x1 + eta*eta),  x1 = omega - eps[m] + Omega[s]
 *                   + (1-occ[m]) * x2/(x2*x2 + eta*eta),  x2 = omega - eps[m] - Omega[s]
 *      (real part of the two terms of Eq. (17); Re[1/(x -+ i eta)] = x/(x^2+eta^2)).
 *
 * Readings of the paper taken here are the ones listed in DESIGN.md ("Readings"):
 * the (ia) composite index is i*v + (a-o) with a fastest; closed shell, one spin channel,
 * prefactor sqrt(2) on w; eta is a finite positive input; one array eps serves as the
 * poles eps[m] and as the evaluation points eps[p], eps[q]; p, q, m run over all N states.
 * The oracle does NOT assume B symmetric in its last two indices: it reads B[P][p][m]
 * literally.
 *
 * Layouts (row-major C arrays): B[naux][N][N], Z[o*v][ldz], V[naux][ldv], Sigma[N][N].
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): hand-solved two-state case with
 * exact rationals (tests/golden/two_state_single_pole.txt), literal complex evaluation of
 * Eq. (17), non-RI 4-index brute force of Eq. (18) on tiny inputs, symmetry, exact
 * power-of-two scaling, additivity over poles, eta->0 limit, null case, separable closed
 * form, permutation invariances, diagonal == G0W0 expression.
 *
 * Next row, at the end of this file: qsgw_oracle_sigma_diag, the G0W0 diagonal Sigma_pp(omega) of
 * Eq. (17) with m = n on a real frequency grid, complex.  Pins (tests/test_oracle_diag_pins.py): the
 * same hand-solved two-state system on a grid in exact rationals (tests/golden/two_state_diag_grid.txt), literal
 * Python-complex evaluation of Eq. (17) through the non-RI 4-index form, Re Sigma_pp(eps_p) == diagonal of the
 * (separately pinned) qsGW matrix, exact power-of-two scaling, additivity over poles, sign of Im, eta -> 0 limit.
 *
 * Further rows at the end of this file: qsgw_oracle_mp2_direct and qsgw_oracle_mp2 (Eqs. (20)-(21), PAPER.md:174-186;
 * pins in tests/test_oracle_mp2_pins.py: the hand-solved two-state rationals, a literal complex spin-orbital brute force
 * of both sums incl. unsymmetric B, identity with the GW oracle at Z = 1, SOX = -direct/2 for rank-one B);
 * qsgw_oracle_mp2_states (the same sums for sampled output states, pinned by equality with qsgw_oracle_mp2); and
 * qsgw_oracle_ao_to_mo, the RI AO->MO transformation as its defining double sum (pins in tests/test_oracle_aomo_pins.py).
 *
 * Floating point: products and the P-, ia- and m-sums are plain double; the running sum
 * over poles s of step 3 is kept in long double so that the oracle's own rounding is far
 * below the 1e-9 parity budget.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int qsgw_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* D(m,s,omega): real part of the two Lehmann terms of Eq. (17). */
double qsgw_oracle_D(double occ_m, double eps_m, double Omega_s, double omega, double eta) {
  double x1 = omega - eps_m + Omega_s;
  double x2 = omega - eps_m - Omega_s;
  return occ_m * (x1 / (x1 * x1 + eta * eta)) + (1.0 - occ_m) * (x2 / (x2 * x2 + eta * eta));
}

/* Step 1, first half of Eq. (18) after (pm|ia) = sum_P B^P_pm B^P_ia (RI):
 *   V[P][s] = sum_i sum_a B[P][i][a] * Z[i*v + (a-o)][s],   i < o <= a < N,  s in [0, n_pole). */
void qsgw_oracle_pole_weights(int N, int o, int naux, int64_t n_pole, const double *B, const double *Z,
                              int64_t ldz, double *V, int64_t ldv) {
  const int v = N - o;
#pragma omp parallel for schedule(static)
  for (int P = 0; P < naux; ++P) {
    double *Vrow = V + (size_t)P * ldv;
    for (int64_t s = 0; s < n_pole; ++s) Vrow[s] = 0.0;
    for (int i = 0; i < o; ++i) {
      for (int a = o; a < N; ++a) {
        const double b = B[((size_t)P * N + i) * N + a];
        const double *Zrow = Z + ((size_t)i * v + (a - o)) * ldz;
        for (int64_t s = 0; s < n_pole; ++s) Vrow[s] += b * Zrow[s];
      }
    }
  }
}

/* Step 2, second half of Eq. (18) for ONE pole s and the listed rows p (rows == NULL: all p):
 *   w[r][m] = sqrt(2) * sum_P B[P][p_r][m] * V[P][s]. */
void qsgw_oracle_residues(int N, int naux, const double *B, const double *V, int64_t ldv, int64_t s,
                          int n_rows, const int *rows, double *w) {
  const double sqrt2 = sqrt(2.0);
#pragma omp parallel for schedule(static)
  for (int r = 0; r < n_rows; ++r) {
    const int p = rows ? rows[r] : r;
    double *wr = w + (size_t)r * N;
    for (int m = 0; m < N; ++m) wr[m] = 0.0;
    for (int P = 0; P < naux; ++P) {
      const double vps = V[(size_t)P * ldv + s];
      const double *Brow = B + ((size_t)P * N + p) * N;
      for (int m = 0; m < N; ++m) wr[m] += Brow[m] * vps;
    }
    for (int m = 0; m < N; ++m) wr[m] *= sqrt2;
  }
}

/* Steps 1-3 restricted to the output rows/columns listed in `states` (n_states entries; NULL: all N
 * states, n_states = N) and to the poles [0, n_pole) of the arrays handed in:
 *   Sigma[r][c] = 1/2 sum_m sum_s w[s][p_r][m] w[s][p_c][m] (D(m,s,eps[p_r]) + D(m,s,eps[p_c]))
 * Sigma is n_states x n_states, row-major.  Loop order: s outermost; w^s is built, used, discarded
 * (w is never held whole).  Returns 0, or -1 on allocation failure / bad arguments. */
int qsgw_oracle_sigma(int N, int o, int naux, int64_t n_pole, const double *B, const double *eps,
                      const double *occ, const double *Omega, const double *Z, int64_t ldz, double eta,
                      int n_states, const int *states, double *Sigma) {
  if (N < 2 || o < 1 || o >= N || naux < 1 || n_pole < 1 || ldz < n_pole || !(eta > 0.0)) return -1;
  if (!states) n_states = N;
  if (n_states < 1) return -1;
  const size_t nS = (size_t)n_states;
  double *V = (double *)malloc(sizeof(double) * (size_t)naux * (size_t)n_pole);
  double *w = (double *)malloc(sizeof(double) * nS * N);
  double *Dm = (double *)malloc(sizeof(double) * nS * N);
  long double *acc = (long double *)malloc(sizeof(long double) * nS * nS);
  if (!V || !w || !Dm || !acc) { free(V); free(w); free(Dm); free(acc); return -1; }
  for (size_t k = 0; k < nS * nS; ++k) acc[k] = 0.0L;

  qsgw_oracle_pole_weights(N, o, naux, n_pole, B, Z, ldz, V, n_pole);            /* step 1 */

  for (int64_t s = 0; s < n_pole; ++s) {
    qsgw_oracle_residues(N, naux, B, V, n_pole, s, n_states, states, w);        /* step 2 */
#pragma omp parallel for schedule(static)
    for (int r = 0; r < n_states; ++r) {                                         /* D(m,s,eps[p_r]) */
      const int p = states ? states[r] : r;
      for (int m = 0; m < N; ++m) Dm[(size_t)r * N + m] = qsgw_oracle_D(occ[m], eps[m], Omega[s], eps[p], eta);
    }
#pragma omp parallel for schedule(static)
    for (int r = 0; r < n_states; ++r) {                                         /* step 3, this pole */
      for (int c = 0; c < n_states; ++c) {
        double t = 0.0;
        for (int m = 0; m < N; ++m)
          t += w[(size_t)r * N + m] * w[(size_t)c * N + m] * (Dm[(size_t)r * N + m] + Dm[(size_t)c * N + m]);
        acc[(size_t)r * nS + c] += 0.5L * (long double)t;
      }
    }
  }
  for (size_t k = 0; k < nS * nS; ++k) Sigma[k] = (double)acc[k];
  free(V); free(w); free(Dm); free(acc);
  return 0;
}

/* ---- next row: G0W0 diagonal self-energy on a real frequency grid ------------------------
 * "The conventional G0W0 method uses only diagonal elements (m = n) of Eq. (17)".  For the listed
 * states p (states == NULL: all N) and the grid points omega[k], Eq. (17) with m = n = p, written out literally as a
 * complex number (RI residues w of Eq. (18) as in steps 1-2 above):
 *   Sigma_pp(omega) = sum_m sum_s w[s][p][m]^2 * ( occ[m] / (omega - eps[m] + Omega[s] - i eta)
 *                                               + (1-occ[m]) / (omega - eps[m] - Omega[s] + i eta) )
 * 1/(x - i eta) = (x + i eta)/(x^2+eta^2),  1/(x + i eta) = (x - i eta)/(x^2+eta^2).
 * Re[r][k], Im[r][k] are n_states x n_omega, row-major.  Loop order: s outermost, w^s built, used, discarded; the
 * pole sum is kept in long double.  Returns 0, or -1 on allocation failure / bad arguments. */
int qsgw_oracle_sigma_diag(int N, int o, int naux, int64_t n_pole, const double *B, const double *eps,
                           const double *occ, const double *Omega, const double *Z, int64_t ldz, double eta,
                           int n_omega, const double *omega, int n_states, const int *states, double *Re, double *Im) {
  if (N < 2 || o < 1 || o >= N || naux < 1 || n_pole < 1 || ldz < n_pole || !(eta > 0.0) || n_omega < 1) return -1;
  if (!states) n_states = N;
  if (n_states < 1) return -1;
  const size_t nS = (size_t)n_states, nW = (size_t)n_omega;
  double *V = (double *)malloc(sizeof(double) * (size_t)naux * (size_t)n_pole);
  double *w = (double *)malloc(sizeof(double) * nS * N);
  long double *accR = (long double *)malloc(sizeof(long double) * nS * nW);
  long double *accI = (long double *)malloc(sizeof(long double) * nS * nW);
  if (!V || !w || !accR || !accI) { free(V); free(w); free(accR); free(accI); return -1; }
  for (size_t k = 0; k < nS * nW; ++k) accR[k] = accI[k] = 0.0L;

  qsgw_oracle_pole_weights(N, o, naux, n_pole, B, Z, ldz, V, n_pole);            /* step 1 */

  for (int64_t s = 0; s < n_pole; ++s) {
    qsgw_oracle_residues(N, naux, B, V, n_pole, s, n_states, states, w);        /* step 2 */
#pragma omp parallel for schedule(static)
    for (int r = 0; r < n_states; ++r) {
      for (int k = 0; k < n_omega; ++k) {
        double tr = 0.0, ti = 0.0;
        for (int m = 0; m < N; ++m) {
          const double w2 = w[(size_t)r * N + m] * w[(size_t)r * N + m];
          const double x1 = omega[k] - eps[m] + Omega[s];
          const double x2 = omega[k] - eps[m] - Omega[s];
          const double d1 = x1 * x1 + eta * eta, d2 = x2 * x2 + eta * eta;
          tr += w2 * (occ[m] * (x1 / d1) + (1.0 - occ[m]) * (x2 / d2));
          ti += w2 * (occ[m] * (eta / d1) - (1.0 - occ[m]) * (eta / d2));
        }
        accR[(size_t)r * nW + k] += (long double)tr;
        accI[(size_t)r * nW + k] += (long double)ti;
      }
    }
  }
  for (size_t k = 0; k < nS * nW; ++k) { Re[k] = (double)accR[k]; Im[k] = (double)accI[k]; }
  free(V); free(w); free(accR); free(accI);
  return 0;
}

/* ---- row 8(f).3, first half: the second-order Coulomb (direct) term of the qsMP2 self-energy ----------------
 * First sum of Eq. (20) put into Eq. (21), closed shell (the spin sum over sigma'
 * gives a factor 2), RI integrals (mp|ia) = sum_P B[P][m][p] B[P][i][a], real part as for qsGW:
 *   Sigma[m][n] = 1/2 * sum_i sum_a sum_p 2 [ (mp|ia)(pn|ai) Dd(i,a,p,eps[n]) + (np|ia)(pm|ai) Dd(i,a,p,eps[m]) ]
 *   Dd(i,a,p,omega) = occ[p]     * x1/(x1^2+eta^2),  x1 = omega + eps[a] - eps[i] - eps[p]
 *                   + (1-occ[p]) * x2/(x2^2+eta^2),  x2 = omega + eps[i] - eps[a] - eps[p]
 * i < o <= a, p over all N states; (pn|ai) is read literally as sum_P B[P][p][n] B[P][a][i].
 * The second sum of Eq. (20) (second-order exchange, SOX) is NOT part of this function.
 * Sigma is N x N row-major.  Returns 0, or -1 on allocation failure / bad arguments. */
int qsgw_oracle_mp2_direct(int N, int o, int naux, const double *B, const double *eps, const double *occ, double eta,
                           double *Sigma) {
  if (N < 2 || o < 1 || o >= N || naux < 1 || !(eta > 0.0)) return -1;
  long double *acc = (long double *)malloc(sizeof(long double) * (size_t)N * N);
  double *L = (double *)malloc(sizeof(double) * (size_t)N * N);   /* L[m][p] = (mp|ia) */
  double *R = (double *)malloc(sizeof(double) * (size_t)N * N);   /* R[p][n] = (pn|ai) */
  if (!acc || !L || !R) { free(acc); free(L); free(R); return -1; }
  for (size_t k = 0; k < (size_t)N * N; ++k) acc[k] = 0.0L;
  for (int i = 0; i < o; ++i) {
    for (int a = o; a < N; ++a) {
#pragma omp parallel for schedule(static)
      for (int m = 0; m < N; ++m) {
        for (int p = 0; p < N; ++p) {
          double l = 0.0, r = 0.0;
          for (int P = 0; P < naux; ++P) {
            const double *BP = B + (size_t)P * N * N;
            l += BP[(size_t)m * N + p] * BP[(size_t)i * N + a];
            r += BP[(size_t)m * N + p] * BP[(size_t)a * N + i];     /* here m, p play the roles of p, n */
          }
          L[(size_t)m * N + p] = l;
          R[(size_t)m * N + p] = r;
        }
      }
#pragma omp parallel for schedule(static)
      for (int m = 0; m < N; ++m) {
        for (int n = 0; n < N; ++n) {
          double t = 0.0;
          for (int p = 0; p < N; ++p) {
            /* <m|Sigma(eps_n)|n> uses (mp|ia)(pn|ai); <n|Sigma(eps_m)|m> uses (np|ia)(pm|ai)   (Eq. (21)) */
            const double om[2] = {eps[n], eps[m]};
            const double num[2] = {L[(size_t)m * N + p] * R[(size_t)p * N + n], L[(size_t)n * N + p] * R[(size_t)p * N + m]};
            for (int k = 0; k < 2; ++k) {
              const double x1 = om[k] + eps[a] - eps[i] - eps[p];
              const double x2 = om[k] + eps[i] - eps[a] - eps[p];
              t += 2.0 * num[k] * (occ[p] * (x1 / (x1 * x1 + eta * eta)) + (1.0 - occ[p]) * (x2 / (x2 * x2 + eta * eta)));
            }
          }
          acc[(size_t)m * N + n] += 0.5L * (long double)t;
        }
      }
    }
  }
  for (size_t k = 0; k < (size_t)N * N; ++k) Sigma[k] = (double)acc[k];
  free(acc); free(L); free(R);
  return 0;
}

/* ---- row 8(f).3, whole: the qsMP2 correlation self-energy, direct + second-order exchange (SOX) ------------------
 * Both sums of Eq. (20) put into Eq. (21), closed shell: the direct sum runs over both
 * spins sigma' (factor 2), the SOX sum over the same spin only (factor 1, sign -), RI integrals, real part:
 *   Sigma[m][n] = 1/2 sum_i sum_a sum_p ( [2 (mp|ia)(pn|ai) - (mp|ia)(pi|an)] Dd(i,a,p,eps[n])
 *                                       + [2 (np|ia)(pm|ai) - (np|ia)(pi|am)] Dd(i,a,p,eps[m]) )
 * with Dd as in qsgw_oracle_mp2_direct; every integral is read literally, (xy|zw) = sum_P B[P][x][y] B[P][z][w].
 * sox_only != 0 drops the direct part.  Returns 0 / -1 as above. */
int qsgw_oracle_mp2(int N, int o, int naux, const double *B, const double *eps, const double *occ, double eta,
                    int sox_only, double *Sigma) {
  if (N < 2 || o < 1 || o >= N || naux < 1 || !(eta > 0.0)) return -1;
  const size_t NN = (size_t)N * N;
  long double *acc = (long double *)malloc(sizeof(long double) * NN);
  double *L = (double *)malloc(sizeof(double) * NN);    /* L[x][y]  = (xy|ia) */
  double *R = (double *)malloc(sizeof(double) * NN);    /* R[x][y]  = (xy|ai) */
  double *E = (double *)malloc(sizeof(double) * NN);    /* E[p][n]  = (pi|an) */
  if (!acc || !L || !R || !E) { free(acc); free(L); free(R); free(E); return -1; }
  for (size_t k = 0; k < NN; ++k) acc[k] = 0.0L;
  const double cd = sox_only ? 0.0 : 2.0;
  for (int i = 0; i < o; ++i) {
    for (int a = o; a < N; ++a) {
#pragma omp parallel for schedule(static)
      for (int x = 0; x < N; ++x) {
        for (int y = 0; y < N; ++y) {
          double l = 0.0, r = 0.0, e = 0.0;
          for (int P = 0; P < naux; ++P) {
            const double *BP = B + (size_t)P * NN;
            l += BP[(size_t)x * N + y] * BP[(size_t)i * N + a];
            r += BP[(size_t)x * N + y] * BP[(size_t)a * N + i];
            e += BP[(size_t)x * N + i] * BP[(size_t)a * N + y];
          }
          L[(size_t)x * N + y] = l; R[(size_t)x * N + y] = r; E[(size_t)x * N + y] = e;
        }
      }
#pragma omp parallel for schedule(static)
      for (int m = 0; m < N; ++m) {
        for (int n = 0; n < N; ++n) {
          double t = 0.0;
          for (int p = 0; p < N; ++p) {
            const double om[2] = {eps[n], eps[m]};
            const double num[2] = {L[(size_t)m * N + p] * (cd * R[(size_t)p * N + n] - E[(size_t)p * N + n]),
                                   L[(size_t)n * N + p] * (cd * R[(size_t)p * N + m] - E[(size_t)p * N + m])};
            for (int k = 0; k < 2; ++k) {
              const double x1 = om[k] + eps[a] - eps[i] - eps[p];
              const double x2 = om[k] + eps[i] - eps[a] - eps[p];
              t += num[k] * (occ[p] * (x1 / (x1 * x1 + eta * eta)) + (1.0 - occ[p]) * (x2 / (x2 * x2 + eta * eta)));
            }
          }
          acc[(size_t)m * N + n] += 0.5L * (long double)t;
        }
      }
    }
  }
  for (size_t k = 0; k < NN; ++k) Sigma[k] = (double)acc[k];
  free(acc); free(L); free(R); free(E);
  return 0;
}

/* ---- qsMP2 restricted to sampled output states (for parity checks at sizes where the full sum is unaffordable) ------
 * The same sums as qsgw_oracle_mp2 -- Eq. (20) in Eq. (21), every integral read literally,
 * (xy|zw) = sum_P B[P][x][y] B[P][z][w] -- for the outputs Sigma[r][c] = <S_r|Sigma|S_c> with S = states[0..n_states).
 * All internal sums (i, a, p, P) run over their full ranges.  The only difference from qsgw_oracle_mp2 is data movement:
 * the entries of B that the restricted outputs need are first COPIED (no arithmetic) into dense arrays with the
 * auxiliary index P contiguous,
 *   Brow[r][y][P] = B[P][S_r][y],   Bcol[y][r][P] = B[P][y][S_r],   Bi[y][P] = B[P][y][i] (per i),
 *   bia[P] = B[P][i][a],  bai[P] = B[P][a][i] (per pair),
 * so that the sums over P do not stride through all of B for every (i, a) pair.  Per pair (i, a):
 *   L[r][p] = (S_r p|ia)  = sum_P Brow[r][p][P] bia[P]
 *   R[p][r] = (p S_r|ai)  = sum_P Bcol[p][r][P] bai[P]
 *   E[p][r] = (p i|a S_r) = sum_P Bi[p][P]      Bcol[a][r][P]
 *   Sigma[r][c] += 1/2 sum_p ( L[r][p] (cd R[p][c] - E[p][c]) Dd(i,a,p,eps[S_c]) + L[c][p] (cd R[p][r] - E[p][r]) Dd(i,a,p,eps[S_r]) )
 * with cd = 2 (0 if sox_only) and Dd as in qsgw_oracle_mp2_direct.  Pinned by equality with qsgw_oracle_mp2 on small
 * inputs incl. unsymmetric B (tests/test_oracle_mp2_pins.py).  Sigma is n_states x n_states row-major.  Returns 0 / -1. */
int qsgw_oracle_mp2_states(int N, int o, int naux, const double *B, const double *eps, const double *occ, double eta,
                           int sox_only, int n_states, const int *states, double *Sigma) {
  if (N < 2 || o < 1 || o >= N || naux < 1 || !(eta > 0.0) || n_states < 1 || !states) return -1;
  for (int r = 0; r < n_states; ++r) if (states[r] < 0 || states[r] >= N) return -1;
  const size_t NN = (size_t)N * N, nS = (size_t)n_states, nP = (size_t)naux;
  long double *acc = (long double *)malloc(sizeof(long double) * nS * nS);
  double *Brow = (double *)malloc(sizeof(double) * nS * N * nP);
  double *Bcol = (double *)malloc(sizeof(double) * (size_t)N * nS * nP);
  double *Bi = (double *)malloc(sizeof(double) * (size_t)N * nP);
  double *bia = (double *)malloc(sizeof(double) * nP);
  double *bai = (double *)malloc(sizeof(double) * nP);
  double *L = (double *)malloc(sizeof(double) * nS * N);
  double *R = (double *)malloc(sizeof(double) * (size_t)N * nS);
  double *E = (double *)malloc(sizeof(double) * (size_t)N * nS);
  if (!acc || !Brow || !Bcol || !Bi || !bia || !bai || !L || !R || !E) {
    free(acc); free(Brow); free(Bcol); free(Bi); free(bia); free(bai); free(L); free(R); free(E);
    return -1;
  }
  for (size_t k = 0; k < nS * nS; ++k) acc[k] = 0.0L;
#pragma omp parallel for schedule(static)
  for (int y = 0; y < N; ++y)                                        /* copies only */
    for (int r = 0; r < n_states; ++r)
      for (int P = 0; P < naux; ++P) {
        Brow[((size_t)r * N + y) * nP + P] = B[(size_t)P * NN + (size_t)states[r] * N + y];
        Bcol[((size_t)y * nS + r) * nP + P] = B[(size_t)P * NN + (size_t)y * N + states[r]];
      }
  const double cd = sox_only ? 0.0 : 2.0;
  for (int i = 0; i < o; ++i) {
#pragma omp parallel for schedule(static)
    for (int y = 0; y < N; ++y)                                      /* copy */
      for (int P = 0; P < naux; ++P) Bi[(size_t)y * nP + P] = B[(size_t)P * NN + (size_t)y * N + i];
    for (int a = o; a < N; ++a) {
      for (int P = 0; P < naux; ++P) {                               /* copies */
        bia[P] = B[(size_t)P * NN + (size_t)i * N + a];
        bai[P] = B[(size_t)P * NN + (size_t)a * N + i];
      }
#pragma omp parallel for schedule(static)
      for (int p = 0; p < N; ++p) {
        for (int r = 0; r < n_states; ++r) {
          const double *brow = Brow + ((size_t)r * N + p) * nP, *bcol = Bcol + ((size_t)p * nS + r) * nP;
          const double *bi = Bi + (size_t)p * nP, *bax = Bcol + ((size_t)a * nS + r) * nP;
          double l = 0.0, rr = 0.0, e = 0.0;
          for (int P = 0; P < naux; ++P) {
            l += brow[P] * bia[P];
            rr += bcol[P] * bai[P];
            e += bi[P] * bax[P];
          }
          L[(size_t)r * N + p] = l; R[(size_t)p * nS + r] = rr; E[(size_t)p * nS + r] = e;
        }
      }
#pragma omp parallel for schedule(static)
      for (int r = 0; r < n_states; ++r) {
        for (int c = 0; c < n_states; ++c) {
          const int m = states[r], n = states[c];
          double t = 0.0;
          for (int p = 0; p < N; ++p) {
            const double om[2] = {eps[n], eps[m]};
            const double num[2] = {L[(size_t)r * N + p] * (cd * R[(size_t)p * nS + c] - E[(size_t)p * nS + c]),
                                   L[(size_t)c * N + p] * (cd * R[(size_t)p * nS + r] - E[(size_t)p * nS + r])};
            for (int k = 0; k < 2; ++k) {
              const double x1 = om[k] + eps[a] - eps[i] - eps[p];
              const double x2 = om[k] + eps[i] - eps[a] - eps[p];
              t += num[k] * (occ[p] * (x1 / (x1 * x1 + eta * eta)) + (1.0 - occ[p]) * (x2 / (x2 * x2 + eta * eta)));
            }
          }
          acc[(size_t)r * nS + c] += 0.5L * (long double)t;
        }
      }
    }
  }
  for (size_t k = 0; k < nS * nS; ++k) Sigma[k] = (double)acc[k];
  free(acc); free(Brow); free(Bcol); free(Bi); free(bia); free(bai); free(L); free(R); free(E);
  return 0;
}

/* ---- row 8(f).2: RI AO->MO transformation of the three-index factors ------------------------------------------------
 * The RI analogue of Eq. (16) (RI remark PAPER.md:120), the defining double sum written out for every
 * auxiliary function P and every orbital pair (p, q):
 *   B_mo[P][p][q] = sum_mu sum_nu C[mu][p] * C[nu][q] * B_ao[P][mu][nu]
 * B_ao [naux][nao][nao] (not assumed symmetric), C [nao][nmo] (column p = orbital p), B_mo [naux][nmo][nmo], row-major.
 * O(naux nmo^2 nao^2): callers sample the auxiliary index at large sizes (each P is independent).  Returns 0 / -1. */
int qsgw_oracle_ao_to_mo(int naux, int nao, int nmo, const double *B_ao, const double *C, double *B_mo) {
  if (naux < 1 || nao < 1 || nmo < 1) return -1;
#pragma omp parallel for collapse(2) schedule(static)
  for (int P = 0; P < naux; ++P) {
    for (int p = 0; p < nmo; ++p) {
      double *row = B_mo + ((size_t)P * nmo + p) * nmo;              /* row[q] = B_mo[P][p][q], all q at once */
      for (int q = 0; q < nmo; ++q) row[q] = 0.0;
      for (int mu = 0; mu < nao; ++mu) {
        for (int nu = 0; nu < nao; ++nu) {
          const double cb = C[(size_t)mu * nmo + p] * B_ao[((size_t)P * nao + mu) * nao + nu];
          for (int q = 0; q < nmo; ++q) row[q] += cb * C[(size_t)nu * nmo + q];
        }
      }
    }
  }
  return 0;
}

/* Number of OpenMP threads the oracle uses from now on (n < 1: leave unchanged).  Not arithmetic: bench.py uses it to time
 * the oracle on one host core next to the all-cores figure. */
void qsgw_oracle_set_num_threads(int n) {
#ifdef _OPENMP
  if (n >= 1) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ---- row 8(f).4, second half: the Casida / RPA step that produces Omega and Z = X + Y ---------------------------------
 * Eqs. (12)-(14), closed shell, real orbitals, RI integrals (ia|jb) = sum_P B[P][i][a] B[P][j][b]
 * (PAPER.md:120), direct RPA (no exchange kernel).  Spin-adapted singlet block: A = Delta + 2K, B = 2K with
 * Delta_ia = eps[a] - eps[i] (diagonal) and K[ia][jb] = (ia|jb), hence
 *   A - B = Delta (diagonal),   A + B = Delta + 4 K.
 * Sign reading: Eqs. (13)-(14) print the Coulomb terms with a minus sign; the RPA polarizability
 * chi = chi0 + chi0 v chi of Eq. (11) gives A = Delta + K, B = K per spin pair, and only that sign keeps every Omega_s real
 * and >= min Delta > 0 for the positive semidefinite RI kernel -- the precondition Omega > 0 of the Sigma build.
 * For real orbitals Eq. (12) reduces to the symmetric problem (the standard Casida reduction)
 *   C xi_s = Omega_s^2 xi_s,   C = (A-B)^(1/2) (A+B) (A-B)^(1/2),   C[ia][jb] = Delta_ia^2 delta + 4 sqrt(Delta_ia) K[ia][jb] sqrt(Delta_jb)
 *   X^s + Y^s = (A-B)^(1/2) xi_s / sqrt(Omega_s)            (normalisation (X+Y)^T (X-Y) = 1, xi_s orthonormal)
 * This function writes C (step before the eigensolve); qsgw_oracle_casida_z does the step after it.  The symmetric
 * eigensolve in between is a library routine (numpy.linalg.eigh in qsgw_oracle.py).  Composite index ia = i*v + (a-o).
 * C is n_ov x n_ov row-major.  Returns 0 / -1. */
int qsgw_oracle_casida_matrix(int N, int o, int naux, const double *B, const double *eps, double *C) {
  if (N < 2 || o < 1 || o >= N || naux < 1) return -1;
  const int v = N - o;
  const size_t nov = (size_t)o * v;
#pragma omp parallel for schedule(static)
  for (int i = 0; i < o; ++i) {
    for (int a = o; a < N; ++a) {
      const size_t ia = (size_t)i * v + (a - o);
      const double d_ia = eps[a] - eps[i];
      for (int j = 0; j < o; ++j) {
        for (int b = o; b < N; ++b) {
          const size_t jb = (size_t)j * v + (b - o);
          const double d_jb = eps[b] - eps[j];
          double k = 0.0;                                                        /* (ia|jb) */
          for (int P = 0; P < naux; ++P) k += B[((size_t)P * N + i) * N + a] * B[((size_t)P * N + j) * N + b];
          C[ia * nov + jb] = (ia == jb ? d_ia * d_ia : 0.0) + 4.0 * sqrt(d_ia) * k * sqrt(d_jb);
        }
      }
    }
  }
  return 0;
}

/* After the eigensolve: lambda[s] (eigenvalues of C, = Omega_s^2) and xi[ia][s] (orthonormal eigenvectors in the columns,
 * leading dimension ldxi) -> Omega[s] = sqrt(lambda[s]),  Z[ia][s] = sqrt(Delta_ia) * xi[ia][s] / sqrt(Omega[s]).
 * n_pole <= n_ov columns are converted.  Z is [n_ov][ldz].  Returns 0, or -1 on bad arguments or a non-positive lambda. */
int qsgw_oracle_casida_z(int N, int o, const double *eps, int64_t n_pole, const double *lambda, const double *xi,
                         int64_t ldxi, double *Omega, double *Z, int64_t ldz) {
  if (N < 2 || o < 1 || o >= N || n_pole < 1 || ldxi < n_pole || ldz < n_pole) return -1;
  const int v = N - o;
  for (int64_t s = 0; s < n_pole; ++s) {
    if (!(lambda[s] > 0.0)) return -1;
    Omega[s] = sqrt(lambda[s]);
  }
  for (int i = 0; i < o; ++i)
    for (int a = o; a < N; ++a) {
      const size_t ia = (size_t)i * v + (a - o);
      const double sd = sqrt(eps[a] - eps[i]);
      for (int64_t s = 0; s < n_pole; ++s) Z[ia * ldz + s] = sd * xi[ia * ldxi + s] / sqrt(Omega[s]);
    }
  return 0;
}
