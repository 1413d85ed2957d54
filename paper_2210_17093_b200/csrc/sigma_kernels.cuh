// sigma_kernels.cuh -- pack kernels, the fused denominator-scaling + contraction kernel (stage 3) and
// the split-K reduce + symmetrise epilogue of the qsGW Sigma^c build.
//
// Stage 3 evaluates Eq. (17) of the paper at omega = eps_p for every (p, q):
//   T[p][q] = sum_m sum_s ( w[s][p][m] * D(m,s,eps_p) ) * w[s][q][m]
// as ONE GEMM T = A W^T over k = (m, s) whose left operand A[p][k] = w * D is formed in shared memory by
// the operand producer of the same kernel: the scaled operand never exists in HBM.  Eq. (19)
// is then Sigma = (T + T^T)/2 (epilogue).
#pragma once
#include "dmma_gemm.cuh"

namespace qsgw {

// ---------------------------------------------------------------- pack kernels
// Symmetric-pair index: r(p, m) = p*N - p(p-1)/2 + (m - p),  0 <= p <= m < N.
__host__ __device__ __forceinline__ int64_t pair_offset(int p, int n_mo) {
  return (int64_t)p * n_mo - ((int64_t)p * (p - 1)) / 2;
}

// Bp[P][r(p,m)] = B[P][p][m] for p <= m: the A operand of stage 2 with the p<->m symmetry of
// w (B^P_pm = B^P_mp, real orbitals) folded in, so stage 2 does N(N+1)/2 rows, not N^2.
__global__ void pack_pairs_kernel(const double *__restrict__ B, int n_mo, double *__restrict__ Bp, int64_t ldp) {
  const int p = blockIdx.x, P = blockIdx.y;
  const double *src = B + ((int64_t)P * n_mo + p) * n_mo;
  double *dst = Bp + (int64_t)P * ldp + pair_offset(p, n_mo) - p;
  for (int m = p + threadIdx.x; m < n_mo; m += blockDim.x) dst[m] = src[m];
}

__global__ void pair_table_kernel(int n_mo, int2 *__restrict__ pairs) {
  const int p = blockIdx.x;
  int2 *dst = pairs + pair_offset(p, n_mo) - p;
  for (int m = p + threadIdx.x; m < n_mo; m += blockDim.x) dst[m] = make_int2(p, m);
}

// BovT[i*v + (a-o)][P] = B[P][i][a], i < o <= a: the (ia) block of Eq. (18), k-major for the stage-1 GEMM.
__global__ void pack_ov_transposed_kernel(const double *__restrict__ B, int n_mo, int n_occ, int n_aux,
                                          double *__restrict__ BovT, int64_t ld_aux) {
  __shared__ double tile[32][33];
  const int v = n_mo - n_occ;
  const int i = blockIdx.z;
  const int a0 = blockIdx.x * 32, P0 = blockIdx.y * 32;
  for (int y = threadIdx.y; y < 32; y += blockDim.y) {
    const int P = P0 + y, a = a0 + threadIdx.x;
    tile[y][threadIdx.x] = (P < n_aux && a < v) ? B[((int64_t)P * n_mo + i) * n_mo + n_occ + a] : 0.0;
  }
  __syncthreads();
  for (int y = threadIdx.y; y < 32; y += blockDim.y) {
    const int a = a0 + y, P = P0 + threadIdx.x;
    if (a < v && P < n_aux) BovT[((int64_t)i * v + a) * ld_aux + P] = tile[threadIdx.x][y];
  }
}

// Row 8(f).3 (direct term of qsMP2): the (ia) pairs s = i*v + (a-o) take the place of the poles.  blockIdx.y < n_aux:
// V[P][s - s0] = B[P][i][a] (the residues (mp|ia) are then w with X+Y = 1); blockIdx.y == n_aux: Omega[s - s0] = eps_a - eps_i.
__global__ void mp2_chunk_kernel(const double *__restrict__ B, const double *__restrict__ eps, int n_mo, int n_occ, int n_aux,
                                 int64_t s0, int sc, double *__restrict__ V, int64_t ldv, double *__restrict__ Omega) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= sc) return;
  const int v = n_mo - n_occ;
  const int64_t s = s0 + j;
  const int i = (int)(s / v), a = n_occ + (int)(s - (int64_t)i * v);
  const int P = blockIdx.y;
  if (P < n_aux) V[(int64_t)P * ldv + j] = B[((int64_t)P * n_mo + i) * n_mo + a];
  else Omega[j] = eps[a] - eps[i];
}

// Exchange (SOX) term of qsMP2 at fixed occupied i: the virtual states a = a0 + j take the place of the poles.
// blockIdx.y < n_aux: V[P][j] = B[P][i][a] (0 for a < n_occ: a0 may start one state early to stay 16-byte aligned);
// blockIdx.y == n_aux: Omega[j] = eps_a - eps_i.
__global__ void mp2_sox_chunk_kernel(const double *__restrict__ B, const double *__restrict__ eps, int n_mo, int n_occ, int n_aux,
                                     int i, int a0, int sc, double *__restrict__ V, int64_t ldv, double *__restrict__ Omega) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= sc) return;
  const int a = a0 + j, P = blockIdx.y;
  if (P < n_aux) V[(int64_t)P * ldv + j] = (a >= n_occ) ? B[((int64_t)P * n_mo + i) * n_mo + a] : 0.0;
  else Omega[j] = eps[a] - eps[i];
}

// ---------------------------------------------------------------- debug-mode precondition checks (include/qsgw_sigma.h)
// out[0] = max |B[P][p][q] - B[P][q][p]|, out[1] = max |B| as the bit patterns of non-negative doubles (which order
// like unsigned integers, so atomicMax on the bits is the max of the values); out[2] = number of NaN/Inf entries.
__global__ void check_B_symmetry_kernel(const double *__restrict__ B, int n_mo, int n_aux, unsigned long long *out) {
  const int p = blockIdx.x, P = blockIdx.y;
  const double *BP = B + (int64_t)P * n_mo * n_mo;
  double dmax = 0.0, amax = 0.0;
  unsigned long long bad = 0;
  for (int q = threadIdx.x; q < n_mo; q += blockDim.x) {
    const double a = BP[(int64_t)p * n_mo + q], b = BP[(int64_t)q * n_mo + p];
    if (!isfinite(a)) ++bad;
    else {
      dmax = fmax(dmax, fabs(a - b));
      amax = fmax(amax, fabs(a));
    }
  }
  if (dmax > 0.0) atomicMax(out + 0, (unsigned long long)__double_as_longlong(dmax));
  if (amax > 0.0) atomicMax(out + 1, (unsigned long long)__double_as_longlong(amax));
  if (bad) atomicAdd(out + 2, bad);
}

// out[0] += number of entries of x[0..n) outside [lo, hi] (NaN counts as outside); lo_open: the lower bound is excluded.
__global__ void check_range_kernel(const double *__restrict__ x, int64_t n, double lo, double hi, int lo_open,
                                   unsigned long long *out) {
  unsigned long long bad = 0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double v = x[i];
    const bool ok = (lo_open ? v > lo : v >= lo) && v <= hi;
    if (!ok) ++bad;
  }
  if (bad) atomicAdd(out, bad);
}

// ---------------------------------------------------------------- stage 3
// D(m,s,omega) = occ_m * x1/(x1^2+eta^2) + (1-occ_m) * x2/(x2^2+eta^2),  x1 = (omega-eps_m)+Omega_s,
// x2 = (omega-eps_m)-Omega_s: real part of the two terms of Eq. (17).  d = omega - eps_m.
// x/(x^2+eta^2) without the IEEE division's slow path: y = x^2+eta^2, r = MUFU.RCP64H(y) (relative error
// e = 1 - y r, |e| <= 2^-20 measured), 1/y = r (1 + e + e^2 + O(e^3)), so x/y = q + q (e + e^2) with q = x r:
// 5 FP64-pipe instructions, error <= 1 ulp (|e|^3 = 2^-60).  y >= eta^2 > 0 is never subnormal for physical energies.
__device__ __forceinline__ double lehmann_term_old(double x, double eta2) {
  const double y = fma(x, x, eta2);
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(y));
  const double q = x * r;
  const double e = fma(-y, r, 1.0);
  const double t = fma(e, e, e);
  return fma(q, t, q);
}

// OCC: 1 = f_m == 1 (occupied), 0 = f_m == 0 (virtual), 2 = fractional (both terms)
template <int OCC>
__device__ __forceinline__ double denominator_D(double d, double Omega_s, double occ_m, double eta2) {
  if (OCC == 1) return lehmann_term_old(d + Omega_s, eta2);
  if (OCC == 0) return lehmann_term_old(d - Omega_s, eta2);
  return occ_m * lehmann_term_old(d + Omega_s, eta2) + (1.0 - occ_m) * lehmann_term_old(d - Omega_s, eta2);
}

// Stage-3 CTA tile: 64 p rows x 256 q columns, k-tiles of 16 poles at one internal state m.  The tile is wide
// in q because the D evaluations of a k-tile (one per element of the p operand) are amortised over the q width:
// 64 x 16 evaluations against 64 x 256 x 16 FMA.  The 8 consumer warps are laid out 2 (p) x 4 (q), each owning
// 4 x 8 DMMA fragments interleaved across the tile (p rows 16i + 8wmi + g, q columns 32j + 8wni + g), so ragged
// edge tiles shed whole fragments evenly: granule 16 rows x 32 columns.
constexpr int kOldTP = 64;
constexpr int kOldTQ = 256;
constexpr int kSigmaStages = 5;
constexpr int kSigmaStageDoubles = (kOldTP + kOldTQ) * kBK;   // unpadded [row][16] tiles, XOR-swizzled (see sw_col)
constexpr size_t kOldSigmaSmemBytes = (size_t)kSigmaStages * kSigmaStageDoubles * sizeof(double) + 2 * kSigmaStages * sizeof(uint64_t);

// Shared tiles of stage 3 are [row][16] doubles with the column index XOR-swizzled by 4 * (row & 3): a DMMA fragment
// load (lanes g = 0..7 rows, t = 0..3 columns 4kk + t) then hits 16 distinct 8-byte bank pairs per half warp, and a
// 16-byte cp.async chunk (2 columns) stays contiguous.  No padding: 5 stages of (64 + 256) x 16 doubles fit.
__device__ __forceinline__ int sw_col(int row, int col) { return col ^ ((row & 3) << 2); }

struct OldSigmaFragMap {
  int wmi, wni, g, t;
  int mi_cnt, nj_cnt;   // fragments of this warp with at least one valid row / column (warp-uniform)
  __device__ __forceinline__ OldSigmaFragMap(int warp, int lane, int rows_valid, int cols_valid) {
    wmi = warp & 1; wni = warp >> 1; g = lane >> 2; t = lane & 3;
    const int rb = min(kOldTP / 8, (max(rows_valid, 0) + 7) >> 3), cb = min(kOldTQ / 8, (max(cols_valid, 0) + 7) >> 3);
    mi_cnt = max(0, (rb - wmi + 1) >> 1);
    nj_cnt = max(0, (cb - wni + 3) >> 2);
  }
  __device__ __forceinline__ int row(int i) const { return 16 * i + 8 * wmi + g; }
  __device__ __forceinline__ int out_col(int j) const { return 32 * j + 8 * wni + 2 * t; }
};

// One k-tile of DMMA work: acc[i][j] += A[p rows of fragment i][k] * Wq[q rows of fragment j][k], k = 0..15, for the
// first MI x NJ fragments of the warp.  MI, NJ are compile-time: a predicated-off DMMA still occupies the FP64 pipe
// for its full issue time (measured: ncu counts it in sm__ops_path_tensor_src_fp64), so ragged edge tiles must
// BRANCH around the fragments they do not own, not predicate them.
template <int MI, int NJ>
__device__ __forceinline__ void mma_ktile_sigma(double (&acc)[4][8][2], const double *ap, const double *bp, int gs) {
#pragma unroll
  for (int kk = 0; kk < kBK / 4; ++kk) {
    const int off = (kk ^ gs) << 2;
    double a[MI], b[NJ];
#pragma unroll
    for (int i = 0; i < MI; ++i) a[i] = ap[16 * i * kBK + off];
#pragma unroll
    for (int j = 0; j < NJ; ++j) b[j] = bp[32 * j * kBK + off];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int j = 0; j < NJ; ++j) dmma_m8n8k4(acc[i][j], a[i], b[j]);
  }
}

template <int MI>
__device__ __forceinline__ void mma_ktile_sigma_nj(double (&acc)[4][8][2], const double *ap, const double *bp, int gs, int nj) {
  switch (nj) {
    case 1: mma_ktile_sigma<MI, 1>(acc, ap, bp, gs); break;
    case 2: mma_ktile_sigma<MI, 2>(acc, ap, bp, gs); break;
    case 3: mma_ktile_sigma<MI, 3>(acc, ap, bp, gs); break;
    case 4: mma_ktile_sigma<MI, 4>(acc, ap, bp, gs); break;
    case 5: mma_ktile_sigma<MI, 5>(acc, ap, bp, gs); break;
    case 6: mma_ktile_sigma<MI, 6>(acc, ap, bp, gs); break;
    case 7: mma_ktile_sigma<MI, 7>(acc, ap, bp, gs); break;
    case 8: mma_ktile_sigma<MI, 8>(acc, ap, bp, gs); break;
    default: break;
  }
}

// Ragged tile: dispatch (warp-uniform) on the fragment counts of this warp.
__device__ __forceinline__ void mma_ktile_sigma_ragged(double (&acc)[4][8][2], const double *ap, const double *bp, int gs,
                                                       int mi, int nj) {
  switch (mi) {
    case 1: mma_ktile_sigma_nj<1>(acc, ap, bp, gs, nj); break;
    case 2: mma_ktile_sigma_nj<2>(acc, ap, bp, gs, nj); break;
    case 3: mma_ktile_sigma_nj<3>(acc, ap, bp, gs, nj); break;
    case 4: mma_ktile_sigma_nj<4>(acc, ap, bp, gs, nj); break;
    default: break;
  }
}

// One CTA: output tile (tp, tq) of T, 64 x 256, for the internal states m in [z*m_per_split, ...) and all
// s_c poles of the chunk.  k-tiles of 16 poles at fixed m, so eps_m / occ_m are CTA-uniform per k-tile.
//   WA    [N*N][ldA]  left operand (scaled by D): row m*N + p, column s.  qsGW: the w chunk of stage 2 (both mirrors present)
//   WB    [N*N][ldB]  right operand, same indexing.  qsGW: the same array; qsMP2 exchange term: (pi|an) left, -(mp|ia) right
//   Omega [s_c]       excitation energies of the chunk
//   Tpart [nsplit][N][N]  split-K partial tiles; slot z is owned by the CTAs with blockIdx.y == z and is
//                     read-modify-written once per launch -> accumulation order is fixed, results reproducible.
// Roles: the 4 producer warps form the operands -- both row blocks of w go global -> shared by cp.async, two k-tiles
// ahead; each producer thread then multiplies the chunks of the p rows it copied itself by D(m, s, eps_p) in
// place: the scaled operand A = w.D exists only in shared memory.  The 8 consumer warps run LDS + DMMA only.
__global__ void __launch_bounds__(kThreads, 1)
sigma_accumulate_cpasync_kernel(const double *__restrict__ WA, int64_t ldA, const double *__restrict__ WB, int64_t ldB,
                        const double *__restrict__ eps, const double *__restrict__ occ, const double *__restrict__ Omega,
                        int n_mo, int s_c, double eta2, int m_per_split, int ntq, double *__restrict__ Tpart) {
  extern __shared__ __align__(16) double smem[];
  // stage st: p rows at smem + st*kSigmaStageDoubles (already scaled by D when released), q rows kOldTP*kBK further
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + kSigmaStages * kSigmaStageDoubles);
  uint64_t *empty = full + kSigmaStages;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tp = blockIdx.x / ntq, tq = blockIdx.x - tp * ntq;
  const int p0 = tp * kOldTP, q0 = tq * kOldTQ;
  const int m_begin = blockIdx.y * m_per_split;
  const int m_end = min(n_mo, m_begin + m_per_split);
  const int KTS = (s_c + kBK - 1) / kBK;         // k-tiles per m
  const int KT = (m_end - m_begin) * KTS;

  if (tid == 0) {
    for (int s = 0; s < kSigmaStages; ++s) {
      mbar_init(full + s, kProducerThreads);
      mbar_init(empty + s, kConsumerWarps);
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (warp >= kConsumerWarps) {
    // ------------------------------------------------ producers
    reg_dec<136>();
    const int pt = tid - kConsumerThreads, pw = pt >> 5;
    const int c2 = (lane & 7) * 2;                // this thread's two columns of every k-tile
    const int rsub = lane >> 3;                   // rows rA0 + 4j (j < 4) of the p tile, rB0 + 4j (j < 16) of the q tile
    const int rA0 = pw * (kOldTP / 4) + rsub, rB0 = pw * (kOldTQ / 4) + rsub;
    const int nrowA = max(0, min(kOldTP / 16, (n_mo - p0 - rA0 + 3) >> 2));   // valid rows among its 4 / 16
    const int nrowB = max(0, min(kOldTQ / 16, (n_mo - q0 - rB0 + 3) >> 2));
    // all of a thread's rows are congruent to rsub mod 4, so one swizzled column offset serves them all
    const int csw = sw_col(rsub, c2);
    double eps_p[kOldTP / 16];
#pragma unroll
    for (int j = 0; j < kOldTP / 16; ++j) eps_p[j] = (j < nrowA) ? __ldg(eps + p0 + rA0 + 4 * j) : 0.0;
    const int64_t stepA = 4 * ldA, stepB = 4 * ldB;
    constexpr int kAhead = 2;                     // k-tiles whose cp.async are in flight ahead of the scaling

    // loader: raw w rows of both operands, global -> shared (cp.async); every thread later scales exactly the
    // 16-byte chunks of the p rows it copied itself, so no producer-side barrier is needed
    int ld_st = 0, ld_m = m_begin, ld_ks = 0;
    uint32_t ld_ph = 1;                           // a fresh barrier passes a wait on parity 1
    auto issue = [&](int kt) {
      if (kt < KT) {
        mbar_wait(empty + ld_st, ld_ph);
        const int s = ld_ks * kBK + c2;
        const int ncol = min(2, max(0, s_c - s));
        const double *srcA = WA + ((int64_t)ld_m * n_mo + p0 + rA0) * ldA + s;
        const double *srcB = WB + ((int64_t)ld_m * n_mo + q0 + rB0) * ldB + s;
        double *dstA = smem + ld_st * kSigmaStageDoubles + rA0 * kBK + csw;
        double *dstB = smem + ld_st * kSigmaStageDoubles + (kOldTP + rB0) * kBK + csw;
#pragma unroll
        for (int j = 0; j < kOldTP / 16; ++j) {
          const int nb = (j < nrowA) ? ncol * 8 : 0;
          cp_async_16(dstA + 4 * j * kBK, nb ? srcA + j * stepA : WA, nb);
        }
#pragma unroll
        for (int j = 0; j < kOldTQ / 16; ++j) {
          const int nb = (j < nrowB) ? ncol * 8 : 0;
          cp_async_16(dstB + 4 * j * kBK, nb ? srcB + j * stepB : WB, nb);
        }
        if (++ld_ks == KTS) { ld_ks = 0; ++ld_m; }
        if (++ld_st == kSigmaStages) { ld_st = 0; ld_ph ^= 1; }
      }
      cp_async_commit();
    };
#pragma unroll
    for (int i = 0; i < kAhead; ++i) issue(i);

    int st = 0, kt = 0;
#pragma unroll 1
    for (int m = m_begin; m < m_end; ++m) {
      const double em = __ldg(eps + m), fo = __ldg(occ + m);
      const long long fbits = __double_as_longlong(fo);
      // occupation class by bit pattern (no FP64-pipe compare): 1.0 -> occupied term only, +-0.0 -> virtual term only
      const int occ_class = (fbits == 0x3FF0000000000000LL) ? 1 : (((unsigned long long)fbits << 1) == 0ULL ? 0 : 2);
      const double sgn = occ_class == 1 ? 1.0 : -1.0;
      double d[kOldTP / 16];
#pragma unroll
      for (int j = 0; j < kOldTP / 16; ++j) d[j] = eps_p[j] - em;
      // Omega_s of the next k-tile is fetched one k-tile ahead (a new 128-byte line per k-tile: an L2 round trip)
      double om0n = __ldg(Omega + min(c2, s_c - 1)), om1n = __ldg(Omega + min(c2 + 1, s_c - 1));
#pragma unroll 1
      for (int ks = 0; ks < KTS; ++ks, ++kt) {
        issue(kt + kAhead);
        const double om0 = om0n, om1 = om1n;
        const int sn = min(ks + 1, KTS - 1) * kBK + c2;
        om0n = __ldg(Omega + min(sn, s_c - 1));
        om1n = __ldg(Omega + min(sn + 1, s_c - 1));
        cp_async_wait<kAhead>();                  // this thread's copies of k-tile kt have landed
        double *rowA = smem + st * kSigmaStageDoubles + rA0 * kBK + csw;
        double2 cur[kOldTP / 16];
#pragma unroll
        for (int j = 0; j < kOldTP / 16; ++j) cur[j] = *reinterpret_cast<const double2 *>(rowA + 4 * j * kBK);
        if (occ_class != 2) {
          // f_m in {0, 1}: one Lehmann term, x = d + sgn * Omega_s.  The 8 evaluations advance together, stage by
          // stage, so that each dependent step is ONE burst of 8 independent FP64 instructions: the producer warp
          // shares its sub-partition's FP64 pipe with two DMMA streams and pays an arbitration wait per burst.
          constexpr int E = kOldTP / 8;
          double x[E], y[E], r[E];
#pragma unroll
          for (int e = 0; e < E; ++e) x[e] = fma(sgn, (e & 1) ? om1 : om0, d[e >> 1]);
#pragma unroll
          for (int e = 0; e < E; ++e) y[e] = fma(x[e], x[e], eta2);
#pragma unroll
          for (int e = 0; e < E; ++e) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r[e]) : "d"(y[e]));
#pragma unroll
          for (int e = 0; e < E; ++e) x[e] *= r[e];                      // q = x r
#pragma unroll
          for (int e = 0; e < E; ++e) y[e] = fma(-y[e], r[e], 1.0);      // e = 1 - y r
#pragma unroll
          for (int e = 0; e < E; ++e) y[e] = fma(y[e], y[e], y[e]);      // t = e + e^2
#pragma unroll
          for (int e = 0; e < E; ++e) x[e] = fma(x[e], y[e], x[e]);      // D = q + q t
#pragma unroll
          for (int j = 0; j < kOldTP / 16; ++j) {
            cur[j].x *= x[2 * j];
            cur[j].y *= x[2 * j + 1];
          }
        } else {
#pragma unroll
          for (int j = 0; j < kOldTP / 16; ++j) {
            cur[j].x *= denominator_D<2>(d[j], om0, fo, eta2);
            cur[j].y *= denominator_D<2>(d[j], om1, fo, eta2);
          }
        }
#pragma unroll
        for (int j = 0; j < kOldTP / 16; ++j) *reinterpret_cast<double2 *>(rowA + 4 * j * kBK) = cur[j];
        mbar_arrive(full + st);                   // release: the scaled p rows and the landed q rows of this thread
        if (++st == kSigmaStages) st = 0;
      }
    }
    cp_async_wait_all();
  } else {
    // ------------------------------------------------ consumers
    reg_inc<184>();
    const OldSigmaFragMap fm(warp, lane, n_mo - p0, n_mo - q0);
    const bool full_tile = fm.mi_cnt == 4 && fm.nj_cnt == 8;
    double acc[4][8][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    int st = 0;
    uint32_t ph = 0;
#pragma unroll 1
    for (int kt = 0; kt < KT; ++kt) {
      mbar_wait(full + st, ph);
      const double *ap = smem + st * kSigmaStageDoubles + (8 * fm.wmi + fm.g) * kBK + fm.t;
      const double *bp = smem + st * kSigmaStageDoubles + (kOldTP + 8 * fm.wni + fm.g) * kBK + fm.t;
      if (full_tile) mma_ktile_sigma<4, 8>(acc, ap, bp, fm.g & 3);
      else mma_ktile_sigma_ragged(acc, ap, bp, fm.g & 3, fm.mi_cnt, fm.nj_cnt);
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + st);
      if (++st == kSigmaStages) { st = 0; ph ^= 1; }
    }

    double *Tz = Tpart + (int64_t)blockIdx.y * n_mo * n_mo;
    const bool vec_ok = (n_mo & 1) == 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int p = p0 + fm.row(i);
      if (p < n_mo) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const int q = q0 + fm.out_col(j);
          if (q < n_mo) {
            double *dst = Tz + (int64_t)p * n_mo + q;
            if (vec_ok) {
              double2 t = *reinterpret_cast<double2 *>(dst);
              t.x += acc[i][j][0];
              t.y += acc[i][j][1];
              *reinterpret_cast<double2 *>(dst) = t;
            } else {
              dst[0] += acc[i][j][0];
              if (q + 1 < n_mo) dst[1] += acc[i][j][1];
            }
          }
        }
      }
    }
  }
}

// ---------------------------------------------------------------- epilogue
// T = sum_z Tpart[z] in the fixed order z = 0..nsplit-1, then Eq. (19): Sigma[p][q] = Sigma[q][p] = (T[p][q]+T[q][p])/2,
// both written from the same expression so the output is bit-symmetric.  grid = (nt, nt), blocks below the
// diagonal return at once; block = (32, 8).
__global__ void sigma_epilogue_kernel(const double *__restrict__ Tpart, int nsplit, int n_mo, double *__restrict__ Sigma) {
  if (blockIdx.y > blockIdx.x) return;
  __shared__ double Tu[32][33];   // T[p-block rows][q-block cols]
  __shared__ double Tl[32][33];   // T[q-block rows][p-block cols]
  const int pb = blockIdx.y * 32, qb = blockIdx.x * 32;
  const int64_t nn = (int64_t)n_mo * n_mo;
  for (int y = threadIdx.y; y < 32; y += blockDim.y) {
    const int x = threadIdx.x;
    double su = 0.0, sl = 0.0;
    if (pb + y < n_mo && qb + x < n_mo)
      for (int z = 0; z < nsplit; ++z) su += Tpart[z * nn + (int64_t)(pb + y) * n_mo + qb + x];
    if (qb + y < n_mo && pb + x < n_mo)
      for (int z = 0; z < nsplit; ++z) sl += Tpart[z * nn + (int64_t)(qb + y) * n_mo + pb + x];
    Tu[y][x] = su;
    Tl[y][x] = sl;
  }
  __syncthreads();
  for (int y = threadIdx.y; y < 32; y += blockDim.y) {
    const int x = threadIdx.x;
    if (pb + y < n_mo && qb + x < n_mo) Sigma[(int64_t)(pb + y) * n_mo + qb + x] = 0.5 * (Tu[y][x] + Tl[x][y]);
    if (qb + y < n_mo && pb + x < n_mo) Sigma[(int64_t)(qb + y) * n_mo + pb + x] = 0.5 * (Tu[x][y] + Tl[y][x]);
  }
}

// ---------------------------------------------------------------- next row: G0W0 diagonal on a frequency grid
// Sigma_pp(omega_k) = sum_m sum_s w[s][p][m]^2 ( f_m / (omega_k - eps_m + Omega_s - i eta)
//                                              + (1 - f_m) / (omega_k - eps_m - Omega_s + i eta) )
// Eq. (17) with m = n = p, stages 1-2 unchanged.  No contraction is left: per (p, m, s, k) one
// complex reciprocal, so the kernel is bound by the FP64 ALU rate (8 FP64-pipe instructions per evaluation:
// x, y = x^2+eta^2, e, t, r (RCP64H seed + cubic correction as in stage 3), w^2 r, Re += (w^2 r) x, Im +-= w^2 r).
// One CTA = one state p and kDiagKW grid points, all m and all s_c poles of the chunk; each element of w is loaded
// once per CTA (coalesced along s) and used for kDiagKW evaluations.  The CTA owns its outputs and adds the chunk's
// contribution to them with a plain read-modify-write: fixed order, reproducible, no atomics.
constexpr int kDiagKW = 8;         // frequency points per thread
constexpr int kDiagThreads = 128;
constexpr size_t kDiagSmemMax = 200 * 1024;   // dynamic shared memory the kernel may be launched with (Omega of one chunk + scratch)

__device__ __forceinline__ void diag_term(double x, double eta2, double w2, double wim, double &re, double &im) {
  const double y = fma(x, x, eta2);
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(y));
  const double e = fma(-y, r, 1.0);
  const double t = fma(e, e, e);
  r = fma(r, t, r);                 // 1 / (x^2 + eta^2) to <= 1 ulp
  re = fma(w2 * r, x, re);          // Re 1/(x -+ i eta) = x / (x^2 + eta^2)
  im = fma(wim, r, im);             // Im 1/(x -+ i eta) = +-eta / (x^2 + eta^2); eta is applied once at the end
}

__global__ void __launch_bounds__(kDiagThreads)
sigma_diag_kernel(const double *__restrict__ W, int64_t ldw, const double *__restrict__ eps,
                  const double *__restrict__ occ, const double *__restrict__ Omega, int n_mo, int s_c, double eta,
                  const double *__restrict__ omega_grid, int n_omega, double *__restrict__ Re, double *__restrict__ Im) {
  extern __shared__ __align__(16) double smem[];     // [s_c] Omega of the chunk, then the cross-warp reduction scratch
  double *om_s = smem;
  double *red = smem + s_c;                          // [kDiagThreads / 32][2 * kDiagKW]
  const int p = blockIdx.x, k0 = blockIdx.y * kDiagKW;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int s = tid; s < s_c; s += kDiagThreads) om_s[s] = Omega[s];
  double wk[kDiagKW], re[kDiagKW], im[kDiagKW];
#pragma unroll
  for (int k = 0; k < kDiagKW; ++k) {
    wk[k] = __ldg(omega_grid + min(k0 + k, n_omega - 1));
    re[k] = im[k] = 0.0;
  }
  __syncthreads();
  const double eta2 = eta * eta;
  for (int m = 0; m < n_mo; ++m) {
    const double em = __ldg(eps + m), fo = __ldg(occ + m);
    const long long fbits = __double_as_longlong(fo);
    const int occ_class = (fbits == 0x3FF0000000000000LL) ? 1 : (((unsigned long long)fbits << 1) == 0ULL ? 0 : 2);
    const double *row = W + ((int64_t)m * n_mo + p) * ldw;
    if (occ_class != 2) {
      const double sgn = occ_class == 1 ? 1.0 : -1.0;      // x = omega - eps_m + sgn Omega_s; Im carries the same sign
      for (int s = tid; s < s_c; s += kDiagThreads) {
        const double w = __ldg(row + s);
        const double w2 = w * w, wim = sgn * w2;
        const double b = fma(-sgn, om_s[s], em);           // eps_m - sgn Omega_s
#pragma unroll
        for (int k = 0; k < kDiagKW; ++k) diag_term(wk[k] - b, eta2, w2, wim, re[k], im[k]);
      }
    } else {
      for (int s = tid; s < s_c; s += kDiagThreads) {
        const double w = __ldg(row + s);
        const double w2 = w * w;
        const double b1 = em - om_s[s], b2 = em + om_s[s];
#pragma unroll
        for (int k = 0; k < kDiagKW; ++k) {
          diag_term(wk[k] - b1, eta2, fo * w2, fo * w2, re[k], im[k]);
          diag_term(wk[k] - b2, eta2, (1.0 - fo) * w2, -(1.0 - fo) * w2, re[k], im[k]);
        }
      }
    }
  }
  // reduce over the CTA in a fixed order: butterfly inside each warp, then warps 0..3 in sequence
#pragma unroll
  for (int k = 0; k < kDiagKW; ++k) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      re[k] += __shfl_xor_sync(0xffffffffu, re[k], off);
      im[k] += __shfl_xor_sync(0xffffffffu, im[k], off);
    }
  }
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < kDiagKW; ++k) {
      red[warp * 2 * kDiagKW + k] = re[k];
      red[warp * 2 * kDiagKW + kDiagKW + k] = im[k];
    }
  }
  __syncthreads();
  if (tid < kDiagKW && k0 + tid < n_omega) {
    double r = 0.0, i = 0.0;
    for (int wv = 0; wv < kDiagThreads / 32; ++wv) {
      r += red[wv * 2 * kDiagKW + tid];
      i += red[wv * 2 * kDiagKW + kDiagKW + tid];
    }
    const int64_t o = (int64_t)p * n_omega + k0 + tid;
    Re[o] += r;
    Im[o] += eta * i;
  }
}

}  // namespace qsgw
