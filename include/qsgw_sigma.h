/*
 * qsgw_sigma.h -- C ABI of the B200 (sm_100a) qsGW correlation self-energy build.
 *
 * What the library computes (arxiv 2210.17093; citations are lines of /root/reference/PAPER.md):
 * the full off-diagonal "mode A" quasiparticle self-consistent GW correlation self-energy
 * matrix of Eq. (19), with Sigma^GW(omega) the Lehmann sum of Eq. (17)
 * and the residues w of Eq. (18), in resolution-of-identity
 * form, (pm|ia) = sum_P B^P_pm B^P_ia (RI remark):
 *
 *   stage 1   V[P][s]    = sum_{i<o<=a} B[P][i][a] * Z[i*v+(a-o)][s]                  (Eq. 18, first half)
 *   stage 2   w[s][p][m] = sqrt(2) * sum_P B[P][p][m] * V[P][s]                      (Eq. 18, second half)
 *   stage 3   T[p][q]    = sum_m sum_s ( w[s][p][m] * D(m,s,eps[p]) ) * w[s][q][m]   (Eq. 17 at omega = eps[p])
 *   epilogue  Sigma[p][q] = 1/2 ( T[p][q] + T[q][p] )                                (Eq. 19)
 *   D(m,s,omega) = occ[m]     * x1/(x1^2+eta^2),  x1 = omega - eps[m] + Omega[s]
 *                + (1-occ[m]) * x2/(x2^2+eta^2),  x2 = omega - eps[m] - Omega[s]     (real part of Eq. 17's terms)
 *
 * All arithmetic is FP64.  Every step runs in hand-written CUDA kernels (FP64 tensor-core DMMA
 * tiles); there is no CPU fallback: without a CUDA device every entry point that needs one
 * returns QSGW_SIGMA_ERR_CUDA.
 *
 * Conventions
 *   - All arrays are dense, row-major (C order), FP64.
 *   - "device" pointers are CUDA device pointers valid on the device the plan was created on;
 *     "host" pointers are ordinary host memory (pinned memory makes the copies faster, it is not required).
 *   - The caller owns every array it passes.  The plan owns its workspace (packed copies of B,
 *     V, the w chunk, split-K partial tiles), allocated in qsgw_sigma_create, freed in
 *     qsgw_sigma_destroy.  qsgw_sigma_build / _begin / _add_poles / _finish / _diag_build never
 *     allocate.  Three entry points allocate extra plan-owned device buffers on their FIRST call
 *     (kept until destroy; ALLOC if they do not fit): qsgw_sigma_build_host (device copies of B,
 *     eps, occ, Sigma and two Omega/Z ranges), qsgw_mp2_direct_build (one s_block of doubles) and
 *     qsgw_mp2_build (that plus n_mo^3 doubles).
 *   - Every entry point that takes a plan makes the plan's device current while it runs and
 *     restores the caller's current device before it returns.
 *   - Device entry points are asynchronous on the plan's stream: inputs must stay alive and
 *     unmodified, and Sigma must not be read, until the stream has been synchronised.
 *   - Return value: QSGW_SIGMA_OK (0) or a negative qsgw_sigma_status.  No exception or abort
 *     crosses the ABI.  qsgw_sigma_last_error(plan) gives a message for the last failure.
 *   - Preconditions that need a look at device data are checked only in DEBUG MODE
 *     (qsgw_sigma_set_debug(plan, 1), or the environment variable QSGW_SIGMA_DEBUG=1 at create):
 *     B[P][p][q] == B[P][q][p] to 1e-10 max|B| and finite (real orbitals), occ[m] in
 *     [0,1], Omega[s] finite and > 0.  In debug mode begin / add_poles (and every build call made
 *     of them) run small check kernels, SYNCHRONISE the stream and return INVALID_ARG with a
 *     message if a precondition fails.  Outside debug mode they are not checked.
 */
#ifndef QSGW_SIGMA_H
#define QSGW_SIGMA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qsgw_sigma_plan qsgw_sigma_plan; /* opaque */

typedef enum qsgw_sigma_status {
  QSGW_SIGMA_OK = 0,
  QSGW_SIGMA_ERR_INVALID_ARG = -1, /* null pointer, size out of range, eta <= 0, call out of sequence */
  QSGW_SIGMA_ERR_ALLOC = -2,       /* workspace allocation failed */
  QSGW_SIGMA_ERR_CUDA = -3         /* a CUDA call failed (no device, launch error, ...) */
} qsgw_sigma_status;

/* Per-stage device times of the builds since the last reset, measured with CUDA events on the plan's
 * stream around every kernel launch (only while profiling is on; see qsgw_sigma_set_profiling). */
typedef struct qsgw_sigma_stats {
  double ms_pack;     int64_t launches_pack;     /* symmetric-pair pack of B + transposed ov block   */
  double ms_stage1;   int64_t launches_stage1;   /* V = B_ov * Z                      (DMMA GEMM)      */
  double ms_stage2;   int64_t launches_stage2;   /* w chunk = sqrt(2) B^T V           (DMMA GEMM)      */
  double ms_stage3;   int64_t launches_stage3;   /* T += (w.D) w^T                    (fused DMMA)     */
  double ms_epilogue; int64_t launches_epilogue; /* split-K reduce + symmetrise                         */
  double ms_diag;     int64_t launches_diag;     /* G0W0 diagonal Sigma_pp(omega) kernel (qsgw_sigma_diag_build) */
  int64_t kernel_launches;                       /* CUDA kernels launched by the library (counted always) */
  int64_t builds;                                /* number of qsgw_sigma_finish calls                  */
  int64_t poles;                                 /* poles processed                                    */
} qsgw_sigma_stats;

/*
 * Create a plan for problems with n_mo molecular orbitals (N), of which the first n_occ are the
 * occupied ones that define the (ia) block of stage 1, n_aux auxiliary functions, and at most
 * n_pole_max poles per qsgw_sigma_build / qsgw_sigma_add_poles call.
 *   s_block     : poles per internal w chunk (the config's "s-block"); 0 = library default (2048).
 *                 w is only ever materialised for one chunk: workspace holds n_mo*n_mo*s_block doubles.
 *   cuda_stream : a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream), or NULL for the
 *                 legacy default stream.  All work of this plan is enqueued on it.
 * Errors: INVALID_ARG if plan == NULL, n_mo < 2, n_occ not in [1, n_mo-1], n_aux < 1, n_pole_max < 1,
 * s_block < 0; ALLOC if the workspace does not fit; CUDA if no usable device.
 */
int qsgw_sigma_create(qsgw_sigma_plan **plan, int n_mo, int n_occ, int n_aux, int64_t n_pole_max,
                      int s_block, void *cuda_stream);

/*
 * One-shot build: Sigma (Eq. 19) from all n_pole poles handed in.  Equivalent to
 * qsgw_sigma_begin + qsgw_sigma_add_poles + qsgw_sigma_finish.
 *   B      device [n_aux][n_mo][n_mo]   RI factors in the MO basis, symmetric in the last two indices
 *   eps    device [n_mo]                QP energies (Ha): the poles eps[m] AND the evaluation points eps[p], eps[q]
 *   occ    device [n_mo]                occupations f_m in [0,1] (0 or 1)
 *   Omega  device [n_pole]              RPA excitation energies (Ha), > 0                       (Eq. 12)
 *   Z      device [n_occ*n_virt][ldz]   X+Y of Eq. (18); row i*n_virt + (a - n_occ), column s
 *   ldz    leading dimension of Z, >= n_pole (a pole sub-range is Z + s0, Omega + s0 with the full ldz)
 *   n_pole poles in this call, 1 <= n_pole <= n_pole_max
 *   eta    > 0 (Ha)
 *   Sigma  device [n_mo][n_mo]          OVERWRITTEN; bit-symmetric (Sigma[p][q] == Sigma[q][p])
 * Because Eq. (17) is a plain sum over s, Sigma of a set of poles is the sum of the Sigmas of any
 * partition of it.
 * Repeated calls with the SAME arguments (pointers, sizes, eta -- the calling pattern of a qsGW loop that
 * refreshes caller-owned buffers in place) are replayed as one CUDA graph from the third call on, provided the
 * plan's stream can be captured (not the legacy default stream) and neither profiling nor debug mode is on;
 * the arithmetic and its order are the same either way.
 */
int qsgw_sigma_build(qsgw_sigma_plan *plan, const double *B, const double *eps, const double *occ,
                     const double *Omega, const double *Z, int64_t ldz, int64_t n_pole, double eta,
                     double *Sigma);

/*
 * Streaming form, for pole sets that are produced or uploaded range by range (Z of the xl config is
 * 130 GB): begin once per Sigma, add any number of pole ranges, finish once.
 *   qsgw_sigma_begin     packs B (symmetric pairs + transposed ov block), keeps eps/occ/eta, zeroes the accumulators.
 *                        B, eps, occ must stay valid until qsgw_sigma_finish has completed on the stream.
 *   qsgw_sigma_add_poles stages 1-3 for the poles handed in, accumulated into the plan's split-K partial tiles.
 *   qsgw_sigma_finish    fixed-order reduction of the partial tiles and Sigma = (T + T^T)/2.
 * INVALID_ARG if called out of sequence.
 */
int qsgw_sigma_begin(qsgw_sigma_plan *plan, const double *B, const double *eps, const double *occ, double eta);
int qsgw_sigma_add_poles(qsgw_sigma_plan *plan, const double *Omega, const double *Z, int64_t ldz, int64_t n_pole);
int qsgw_sigma_finish(qsgw_sigma_plan *plan, double *Sigma);

/*
 * Same build with HOST buffers (same shapes and meaning as qsgw_sigma_build): the library uploads
 * B, eps, occ once and Omega/Z in ranges of poles (the first of one s_block, the later ones of up to four
 * s_blocks, at most 6 GB of Z each), overlapping the upload of the next range with the kernels of the
 * current one, downloads Sigma and synchronises before returning.
 * n_pole may exceed n_pole_max.  Device staging buffers for the host path are allocated on the first
 * call (not in create) and kept by the plan; ALLOC if they do not fit.
 * Of B only the entries B[P][p][q] with p <= q are read (and uploaded): B is symmetric in its last two
 * indices (precondition), and the build uses nothing else.  In debug mode all of B is uploaded and checked.
 */
int qsgw_sigma_build_host(qsgw_sigma_plan *plan, const double *B, const double *eps, const double *occ,
                          const double *Omega, const double *Z, int64_t ldz, int64_t n_pole, double eta,
                          double *Sigma);

/*
 * Next row of the scope table: the G0W0 diagonal self-energy on a real frequency grid,
 *   Sigma_pp(omega_k) = sum_m sum_s w[s][p][m]^2 ( occ[m]     / (omega_k - eps[m] + Omega[s] - i eta)
 *                                                + (1-occ[m]) / (omega_k - eps[m] - Omega[s] + i eta) ),
 * i.e. Eq. (17) with m = n = p ("the conventional G0W0 method uses only diagonal elements"), for all
 * n_mo states p and n_omega grid points.  Stages 1 and 2 (V and the s-blocked residues w) are those of qsgw_sigma_build;
 * stage 3 is replaced by an FP64-ALU-bound reduction kernel.  Arguments as qsgw_sigma_build, plus
 *   omega_grid device [n_omega]          real frequencies (Ha), n_omega >= 1
 *   SigmaRe    device [n_mo][n_omega]    OVERWRITTEN with Re Sigma_pp(omega_k)
 *   SigmaIm    device [n_mo][n_omega]    OVERWRITTEN with Im Sigma_pp(omega_k)
 * Re Sigma_pp(eps[p]) equals the diagonal of the matrix qsgw_sigma_build returns (Eq. (19) with m = n).
 * Asynchronous on the plan's stream.  INVALID_ARG as for qsgw_sigma_build, or if omega_grid / SigmaRe / SigmaIm is
 * NULL or n_omega < 1, or if the chunk's Omega (s_block doubles) does not fit the kernel's shared memory (s_block > 24576).
 */
int qsgw_sigma_diag_build(qsgw_sigma_plan *plan, const double *B, const double *eps, const double *occ,
                          const double *Omega, const double *Z, int64_t ldz, int64_t n_pole, double eta,
                          const double *omega_grid, int n_omega, double *SigmaRe, double *SigmaIm);

/*
 * Row 8(f).3, first half: the second-order Coulomb (direct) term of the qsMP2 self-energy -- the first sum of Eq. (20)
 * put into Eq. (21), closed shell, RI integrals, real part:
 *   Sigma[m][n] = 1/2 sum_{i<o<=a} sum_p 2 [ (mp|ia)(pn|ai) Dd(eps[n]) + (np|ia)(pm|ai) Dd(eps[m]) ],
 *   Dd(omega) = occ[p] x1/(x1^2+eta^2) + (1-occ[p]) x2/(x2^2+eta^2),  x1 = omega + eps[a]-eps[i] - eps[p],  x2 = omega - (eps[a]-eps[i]) - eps[p].
 * This is Eq. (17)-(19) with the (ia) pairs as poles, X+Y = 1 and Omega_ia = eps[a] - eps[i], so the library runs its stages 2-3
 * on pole weights V[P][ia] = B[P][i][a] gathered chunk by chunk (no stage 1, no Z).  The second-order exchange (SOX) sum of
 * Eq. (20) is NOT included here (qsgw_mp2_build adds it).  B, eps, occ, eta, Sigma as in qsgw_sigma_build (B symmetric in its last two indices); the plan may
 * have any n_pole_max.  Asynchronous on the plan's stream; a small Omega buffer is allocated on the first call (ALLOC if it fails).
 */
int qsgw_mp2_direct_build(qsgw_sigma_plan *plan, const double *B, const double *eps, const double *occ, double eta,
                          double *Sigma);

/*
 * Row 8(f).3, whole: the qsMP2 correlation self-energy, both sums of Eq. (20) in Eq. (21), closed shell:
 *   Sigma[m][n] = 1/2 sum_{i<o<=a} sum_p ( [2 (mp|ia)(pn|ai) - (mp|ia)(pi|an)] Dd(eps[n]) + [2 (np|ia)(pm|ai) - (np|ia)(pi|am)] Dd(eps[m]) )
 * The direct sum is computed as in qsgw_mp2_direct_build.  The second-order exchange (SOX) sum runs, for every occupied i,
 * one batched GEMM for the exchange integrals (pi|an), stage 2 for -(mp|ia) and the fused D-scaling + contraction kernel of
 * stage 3 with those two as its left and right operands (virtual a as the "poles", p as the internal state); everything
 * accumulates into the same split-K partial tiles and one epilogue symmetrises.  O(o N^2 (N + v) naux + o v N^3) flops.
 * Arguments as qsgw_mp2_direct_build; B must be symmetric in its last two indices.  A buffer of n_mo^3 doubles for the
 * exchange integrals of one i is allocated on the first call (ALLOC if it does not fit).
 */
int qsgw_mp2_build(qsgw_sigma_plan *plan, const double *B, const double *eps, const double *occ, double eta, double *Sigma);

/*
 * Row 8(f).2 of the scope table: the RI AO->MO transformation that produces the B argument of the calls above, once per
 * qsGW iteration (the RI analogue of Eq. (16); RI remark PAPER.md:120):
 *   B_mo[P][p][q] = sum_mu sum_nu C[mu][p] * C[nu][q] * B_ao[P][mu][nu]        (B_mo[P] = C^T B_ao[P] C)
 * as two batched FP64 tensor-core GEMMs over the n_aux auxiliary functions (half transform into `work`, then the second
 * index).  No plan is needed.
 *   B_ao  device [n_aux][n_ao][n_ao]   three-index RI factors in the AO basis (need not be symmetric)
 *   C     device [n_ao][n_mo]          AO coefficients of the MOs, column p = orbital p
 *   work  device, qsgw_ri_ao_to_mo_work_doubles(n_aux, n_ao, n_mo) doubles, 16-byte aligned; caller-owned scratch
 *   B_mo  device [n_aux][n_mo][n_mo]   OVERWRITTEN
 *   cuda_stream  a cudaStream_t or NULL; the call is asynchronous on it
 * Errors: INVALID_ARG for NULL pointers, sizes < 1 or a misaligned work buffer; CUDA if no sm_100 device or a launch fails
 * (message: qsgw_sigma_last_error(NULL)).
 */
int qsgw_ri_ao_to_mo(const double *B_ao, const double *C, int n_aux, int n_ao, int n_mo, double *work, double *B_mo,
                     void *cuda_stream);
size_t qsgw_ri_ao_to_mo_work_doubles(int n_aux, int n_ao, int n_mo);

/*
 * The same transformation for callers that must not allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc) and have no scratch buffer of their own: the `work` array of qsgw_ri_ao_to_mo is a
 * file-scope device array of the library, qsgw_ri_ao_to_mo_static_max_doubles() = 8 Mi doubles = 64 MiB, which every GPU
 * that loads the library holds until the process exits.  The call allocates nothing (no cudaMalloc / cudaFree, no allocating
 * library routine); arguments, layouts, results and asynchrony are those of qsgw_ri_ao_to_mo.
 *   - Limit: n_aux * n_ao * round_up(n_mo, 2) <= 8 Mi doubles (e.g. the `small` config, 400 x 120 x 120); larger problems
 *     return INVALID_ARG with a message that names the limit -- use qsgw_ri_ao_to_mo with a caller-owned buffer.
 *   - ALL calls on one GPU share the one array, which keeps the contents of the last call (nothing in it has to start at
 *     zero).  Two calls that overlap on the GPU -- different streams, or different host threads on different streams -- RACE
 *     on it and give wrong results; calls on one stream are ordered and safe.
 * Errors: as qsgw_ri_ao_to_mo; CUDA also if the address of the array cannot be obtained on the current device.
 */
int qsgw_ri_ao_to_mo_static(const double *B_ao, const double *C, int n_aux, int n_ao, int n_mo, double *B_mo, void *cuda_stream);
size_t qsgw_ri_ao_to_mo_static_max_doubles(void);

/*
 * Row 8(e) / 8(f).4 of the scope table: the build shards over the pole index s.  Sigma is a plain sum over s (Eq. (17),
 * PAPER.md:149), V[:,s] depends only on Z[:,s] and w^s only on V[:,s], so rank r of n_ranks runs
 * qsgw_sigma_begin / _add_poles / _finish on the contiguous slice Omega[s0 .. s0+n), Z[:, s0 .. s0+n) of the poles (B, eps,
 * occ replicated) and ONE all-reduce(sum) of the n_mo x n_mo Sigma over the ranks finishes the build (the paper itself is
 * single-GPU; multi-GPU is its future work).  This helper is the partition: slices are contiguous, disjoint,
 * cover [0, n_pole), start at multiples of 32 poles (the k-tile depth of stage 3; keeps Z + s0 16-byte aligned) and differ
 * by at most 32 poles in length.  A rank may get n = 0 (more ranks than 32-pole groups): it calls begin and finish only and
 * contributes Sigma = 0.  Pure host arithmetic, no device needed.
 * Errors: INVALID_ARG if n_pole < 1, n_ranks < 1, rank outside [0, n_ranks) or s0 / n is NULL.
 */
int qsgw_sigma_pole_slice(int64_t n_pole, int n_ranks, int rank, int64_t *s0, int64_t *n);

/*
 * Row 8(f).4, second half: the Casida / RPA step that produces the Omega and Z arguments of the build (Eqs. (12)-(14),
 * PAPER.md:130-136; "the next bottleneck").  Closed shell, real orbitals, direct RPA, RI integrals
 * (ia|jb) = sum_P B[P][i][a] B[P][j][b]: A - B = Delta (diagonal, Delta_ia = eps[a] - eps[i]), A + B = Delta + 4 K, and
 * Eq. (12) reduces to the symmetric problem C xi_s = Omega_s^2 xi_s with
 *   C[ia][jb] = Delta_ia^2 delta_{ia,jb} + 4 sqrt(Delta_ia) (ia|jb) sqrt(Delta_jb),   X^s + Y^s = sqrt(Delta) xi_s / sqrt(Omega_s).
 * (Sign reading: Eqs. (13)-(14) print the Coulomb terms with a minus sign; + is taken, the sign that follows
 * from Eq. (11) and keeps Omega real.)  The library does the two steps around the eigensolve; the dense symmetric
 * eigensolve itself is NOT part of this library (callers use a library routine, e.g. cuSOLVER through torch.linalg.eigh).
 *
 * qsgw_casida_matrix: C from B and eps -- one gather kernel and one FP64 tensor-core GEMM over the auxiliary index
 * (upper-triangle tiles only, mirrored in the epilogue: n_ov (n_ov + 128) naux flops); C is bit-symmetric.
 *   B     device [n_aux][n_mo][n_mo]; only the occupied-virtual block B[P][i][a], i < n_occ <= a, is read
 *   eps   device [n_mo]; eps[a] > eps[i] for every pair (else C holds NaN)
 *   work  device, qsgw_casida_work_doubles(n_mo, n_occ, n_aux) doubles, 16-byte aligned; caller-owned scratch
 *   C     device [n_ov][ldc], n_ov = n_occ * (n_mo - n_occ), row / column ia = i * n_virt + (a - n_occ); OVERWRITTEN
 * qsgw_casida_z: after the eigensolve, for the first n_pole eigenpairs handed in,
 *   Omega[s] = sqrt(lambda[s]),   Z[ia][s] = sqrt(Delta_ia) * xi[ia][s] / sqrt(Omega[s])
 *   lambda device [n_pole] eigenvalues of C (> 0);  xi device [n_ov][ldxi], eigenvector s in column s (orthonormal)
 *   Omega  device [n_pole], Z device [n_ov][ldz]: OVERWRITTEN; they are the Omega / Z arguments of qsgw_sigma_build.
 * Both are asynchronous on cuda_stream (a cudaStream_t or NULL) and need no plan.
 * Errors: INVALID_ARG for NULL pointers, sizes out of range, leading dimensions too small, a misaligned work buffer;
 * CUDA if no sm_100 device or a launch fails (message: qsgw_sigma_last_error(NULL)).
 */
size_t qsgw_casida_work_doubles(int n_mo, int n_occ, int n_aux);
int qsgw_casida_matrix(const double *B, const double *eps, int n_mo, int n_occ, int n_aux, double *work, double *C,
                       int64_t ldc, void *cuda_stream);
int qsgw_casida_z(const double *eps, int n_mo, int n_occ, const double *lambda, const double *xi, int64_t ldxi,
                  int64_t n_pole, double *Omega, double *Z, int64_t ldz, void *cuda_stream);

/* Free the workspace and the plan.  Synchronises the plan's stream first.  NULL is accepted. */
int qsgw_sigma_destroy(qsgw_sigma_plan *plan);

/* ---- helpers, not part of the method ---- */

/* Message for the most recent failure on this plan ("" if none); valid until the next call on the plan.
 * With plan == NULL: message for the most recent failed qsgw_sigma_create on this thread. */
const char *qsgw_sigma_last_error(const qsgw_sigma_plan *plan);

/* Device bytes the plan allocated (workspace + host-path staging so far). */
size_t qsgw_sigma_workspace_bytes(const qsgw_sigma_plan *plan);

/* Bounds the number of poles one stage-1 launch handles (default: as many as fit in 4 GiB of V, at most n_pole_max).  A
 * build / add_poles call with more poles runs stage 1 range by range; the result does not depend on it beyond rounding
 * order (V is the same, the chunks of stages 2-3 are cut at other places only if n is not a multiple of s_block).
 * n is rounded up to a multiple of the plan's s_block and clamped to the allocated capacity.  INVALID_ARG if n < 1. */
int qsgw_sigma_limit_pole_batch(qsgw_sigma_plan *plan, int64_t n);

/* Profiling on (1) / off (0): when on, every kernel launch is bracketed by CUDA events on the plan's
 * stream and qsgw_sigma_get_stats sums them per stage.  Off by default. */
int qsgw_sigma_set_profiling(qsgw_sigma_plan *plan, int on);
/* Synchronises the stream, fills *stats with the totals since the last reset; reset != 0 clears them. */
int qsgw_sigma_get_stats(qsgw_sigma_plan *plan, qsgw_sigma_stats *stats, int reset);

/* Debug mode on (1) / off (0): device-side precondition checks in begin / add_poles (see "Preconditions" above).
 * Off by default unless QSGW_SIGMA_DEBUG=1 was set when the plan was created. */
int qsgw_sigma_set_debug(qsgw_sigma_plan *plan, int on);

#ifdef QSGW_SIGMA_TEST_HOOKS
/* Test hook, compiled only into the test build of the library (-DQSGW_SIGMA_TEST_HOOKS; libqsgw_sigma_testhooks.so),
 * not into libqsgw_sigma.so: copy the leading rows x cols block of a workspace array into a dense device buffer
 * dst[rows][cols], asynchronously on the plan's stream.  which: 0 = V of the last chunk [n_aux][s],
 * 1 = w chunk of the last chunk [n_mo*n_mo][s] (row m*n_mo+p), 2 = packed symmetric B [n_aux][n_mo(n_mo+1)/2],
 * 3 = transposed ov block [n_occ*n_virt][n_aux], 4 = split-K partial tiles [nsplit][n_mo*n_mo] (rows = nsplit).
 * INVALID_ARG if the block exceeds the array. */
int qsgw_sigma_copy_workspace(qsgw_sigma_plan *plan, int which, double *dst, int64_t rows, int64_t cols);
#endif

/* Library version (major*10000 + minor*100 + patch). */
int qsgw_sigma_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QSGW_SIGMA_H */
