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

// ---------------------------------------------------------------- stage 3
// D(m,s,omega) = occ_m * x1/(x1^2+eta^2) + (1-occ_m) * x2/(x2^2+eta^2),  x1 = (omega-eps_m)+Omega_s,
// x2 = (omega-eps_m)-Omega_s: real part of the two terms of Eq. (17).  d = omega - eps_m.
__device__ __forceinline__ double lehmann_term(double x, double eta2) { return x / fma(x, x, eta2); }

__device__ __forceinline__ double denominator_D(double d, double Omega_s, double occ_m, double eta2) {
  if (occ_m == 1.0) return lehmann_term(d + Omega_s, eta2);
  if (occ_m == 0.0) return lehmann_term(d - Omega_s, eta2);
  return occ_m * lehmann_term(d + Omega_s, eta2) + (1.0 - occ_m) * lehmann_term(d - Omega_s, eta2);
}

constexpr size_t kSigmaSmemBytes = (size_t)kStages * 2 * kBM * kLdK * sizeof(double);

// One CTA: output tile (tp, tq) of T, 128 x 128, for the internal states m in [z*m_per_split, ...) and all
// s_c poles of the chunk.  k-tiles of 16 poles at fixed m, so eps_m / occ_m are CTA-uniform per k-tile.
//   W     [N*N][ldw]  chunk of residues, row m*N + p, column s (stage-2 output; both mirrors present)
//   Omega [s_c]       excitation energies of the chunk
//   Tpart [nsplit][N][N]  split-K partial tiles; slot z is owned by the CTAs with blockIdx.y == z and is
//                     read-modify-written once per launch -> accumulation order is fixed, results reproducible.
__global__ void __launch_bounds__(kThreads, 1)
sigma_accumulate_kernel(const double *__restrict__ W, int64_t ldw, const double *__restrict__ eps,
                        const double *__restrict__ occ, const double *__restrict__ Omega, int n_mo, int s_c,
                        double eta2, int m_per_split, int ntq, double *__restrict__ Tpart) {
  extern __shared__ __align__(16) double smem[];
  double *As = smem;                             // [stage][128][kLdK]  p rows, scaled in place by D
  double *Bs = smem + kStages * kBM * kLdK;      // [stage][128][kLdK]  q rows, raw
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tp = blockIdx.x / ntq, tq = blockIdx.x - tp * ntq;
  const int p0 = tp * kBM, q0 = tq * kBN;
  const int wm = (warp & 1) * 64, wn = (warp >> 1) * 32;
  const int m_begin = blockIdx.y * m_per_split;
  const int m_end = min(n_mo, m_begin + m_per_split);
  const int KTS = (s_c + kBK - 1) / kBK;         // k-tiles per m
  const int KT = (m_end - m_begin) * KTS;

  // ---- loader: thread owns 4 (row, 16-byte chunk) slots of each operand tile; counters (m, ks) advance per k-tile
  int ld_m = m_begin, ld_ks = 0;
  auto issue = [&](int kt) {
    if (kt < KT) {
      const int st = kt % kStages;
      const int s0 = ld_ks * kBK;
      const double *wm_base = W + (int64_t)ld_m * n_mo * ldw + s0;
#pragma unroll
      for (int j = 0; j < (kBM * kBK / 2) / kThreads; ++j) {
        const int id = tid + j * kThreads;
        const int r = id >> 3, c = (id & 7) * 2;
        int n = s_c - s0 - c;
        n = n < 0 ? 0 : (n > 2 ? 2 : n);
        const int nbA = (p0 + r < n_mo) ? n * 8 : 0;
        const int nbB = (q0 + r < n_mo) ? n * 8 : 0;
        cp_async_16(As + (st * kBM + r) * kLdK + c, nbA ? wm_base + (int64_t)(p0 + r) * ldw + c : W, nbA);
        cp_async_16(Bs + (st * kBM + r) * kLdK + c, nbB ? wm_base + (int64_t)(q0 + r) * ldw + c : W, nbB);
      }
      if (++ld_ks == KTS) { ld_ks = 0; ++ld_m; }
    }
    cp_async_commit();
  };

  // ---- operand producer: thread scales 8 consecutive k of one p row, A[p][k] *= D(m, s0+k, eps_p)
  const int sc_row = tid >> 1, sc_k = (tid & 1) * 8;
  const double eps_p = (p0 + sc_row < n_mo) ? __ldg(eps + p0 + sc_row) : 0.0;
  int sc_m = m_begin, sc_ks = 0;
  auto scale = [&](int kt) {
    if (kt < KT) {
      const int st = kt % kStages;
      const int s0 = sc_ks * kBK + sc_k;
      const double d = eps_p - __ldg(eps + sc_m);
      const double f = __ldg(occ + sc_m);
      double2 *row = reinterpret_cast<double2 *>(As + (st * kBM + sc_row) * kLdK + sc_k);
#pragma unroll
      for (int h = 0; h < 4; ++h) {
        const int s = s0 + 2 * h;
        const double om0 = (s < s_c) ? __ldg(Omega + s) : 1.0;
        const double om1 = (s + 1 < s_c) ? __ldg(Omega + s + 1) : 1.0;
        double2 wv = row[h];
        wv.x *= denominator_D(d, om0, f, eta2);
        wv.y *= denominator_D(d, om1, f, eta2);
        row[h] = wv;
      }
      if (++sc_ks == KTS) { sc_ks = 0; ++sc_m; }
    }
  };

  double acc[8][4][2];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
  for (int s = 0; s < kStages - 1; ++s) issue(s);
  cp_async_wait<kStages - 2>();   // k-tile 0 landed (this thread's copies)
  __syncthreads();
  scale(0);

  for (int kt = 0; kt < KT; ++kt) {
    cp_async_wait<kStages - 3>();  // k-tile kt+1 landed
    __syncthreads();               // ... for all threads; scale(kt) visible; compute(kt-1) finished everywhere
    issue(kt + kStages - 1);       // refills the buffer compute(kt-1) just released
    scale(kt + 1);
    const double *as = As + ((kt % kStages) * kBM + wm + (lane >> 2)) * kLdK + (lane & 3);
    const double *bs = Bs + ((kt % kStages) * kBM + wn + (lane >> 2)) * kLdK + (lane & 3);
#pragma unroll
    for (int kk = 0; kk < kBK / 4; ++kk) {
      double a[8], b[4];
#pragma unroll
      for (int i = 0; i < 8; ++i) a[i] = as[(8 * i) * kLdK + 4 * kk];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = bs[(8 * j) * kLdK + 4 * kk];
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma_m8n8k4(acc[i][j], a[i], b[j]);
    }
  }
  cp_async_wait<0>();

  double *Tz = Tpart + (int64_t)blockIdx.y * n_mo * n_mo;
  const bool vec_ok = (n_mo & 1) == 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int p = p0 + wm + 8 * i + (lane >> 2);
    if (p < n_mo) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int q = q0 + wn + 8 * j + 2 * (lane & 3);
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

}  // namespace qsgw
