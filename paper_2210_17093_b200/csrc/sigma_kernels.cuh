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
// x/(x^2+eta^2) without the IEEE division's slow path: MUFU.RCP64H seed + two Newton steps folded into the
// quotient (relative error ~2 ulp; x^2+eta^2 >= eta^2 > 0 is never subnormal for physical energies).
__device__ __forceinline__ double lehmann_term(double x, double eta2) {
  const double y = fma(x, x, eta2);
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(y));
  double e = fma(-y, r, 1.0);
  r = fma(r, e, r);
  const double q = x * r;
  e = fma(-y, r, 1.0);
  return fma(q, e, q);
}

// OCC: 1 = f_m == 1 (occupied), 0 = f_m == 0 (virtual), 2 = fractional (both terms)
template <int OCC>
__device__ __forceinline__ double denominator_D(double d, double Omega_s, double occ_m, double eta2) {
  if (OCC == 1) return lehmann_term(d + Omega_s, eta2);
  if (OCC == 0) return lehmann_term(d - Omega_s, eta2);
  return occ_m * lehmann_term(d + Omega_s, eta2) + (1.0 - occ_m) * lehmann_term(d - Omega_s, eta2);
}

constexpr int kSigmaStages = 5;
constexpr size_t kSigmaSmemBytes = (size_t)kSigmaStages * 2 * kBM * kLdK * sizeof(double) + 2 * kSigmaStages * sizeof(uint64_t);

// One CTA: output tile (tp, tq) of T, 128 x 128, for the internal states m in [z*m_per_split, ...) and all
// s_c poles of the chunk.  k-tiles of 16 poles at fixed m, so eps_m / occ_m are CTA-uniform per k-tile.
//   W     [N*N][ldw]  chunk of residues, row m*N + p, column s (stage-2 output; both mirrors present)
//   Omega [s_c]       excitation energies of the chunk
//   Tpart [nsplit][N][N]  split-K partial tiles; slot z is owned by the CTAs with blockIdx.y == z and is
//                     read-modify-written once per launch -> accumulation order is fixed, results reproducible.
// Roles: the 4 producer warps form the operands -- both row blocks of w go global -> shared by cp.async, two k-tiles
// ahead; each producer thread then multiplies the chunks of the p rows it copied itself by D(m, s, eps_p) in
// place: the scaled operand A = w.D exists only in shared memory.  The 8 consumer warps run LDS + DMMA only.
__global__ void __launch_bounds__(kThreads, 1)
sigma_accumulate_kernel(const double *__restrict__ W, int64_t ldw, const double *__restrict__ eps,
                        const double *__restrict__ occ, const double *__restrict__ Omega, int n_mo, int s_c,
                        double eta2, int m_per_split, int ntq, double *__restrict__ Tpart) {
  extern __shared__ __align__(16) double smem[];
  double *As = smem;                                  // [stage][128][kLdK]  p rows, already scaled by D
  double *Bs = smem + kSigmaStages * kBM * kLdK;      // [stage][128][kLdK]  q rows, raw
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + 2 * kSigmaStages * kBM * kLdK);
  uint64_t *empty = full + kSigmaStages;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tp = blockIdx.x / ntq, tq = blockIdx.x - tp * ntq;
  const int p0 = tp * kBM, q0 = tq * kBN;
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
    reg_dec<104>();
    const int pt = tid - kConsumerThreads, pw = pt >> 5;
    const int c2 = (lane & 7) * 2;                // this thread's two columns of every k-tile
    const int r0 = pw * 32 + (lane >> 3);         // its rows: r0 + 4j, j < 8
    int nrowA = (n_mo - p0 - r0 + 3) >> 2, nrowB = (n_mo - q0 - r0 + 3) >> 2;   // valid rows among its 8
    nrowA = max(0, min(8, nrowA));
    nrowB = max(0, min(8, nrowB));
    double eps_p[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) eps_p[j] = (j < nrowA) ? __ldg(eps + p0 + r0 + 4 * j) : 0.0;
    const int64_t row_step = 4 * ldw;
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
        const double *srcA = W + ((int64_t)ld_m * n_mo + p0 + r0) * ldw + s;
        const double *srcB = W + ((int64_t)ld_m * n_mo + q0 + r0) * ldw + s;
        double *dstA = As + (ld_st * kBM + r0) * kLdK + c2;
        double *dstB = Bs + (ld_st * kBM + r0) * kLdK + c2;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const int nbA = (j < nrowA) ? ncol * 8 : 0, nbB = (j < nrowB) ? ncol * 8 : 0;
          cp_async_16(dstA + 4 * j * kLdK, nbA ? srcA + j * row_step : W, nbA);
          cp_async_16(dstB + 4 * j * kLdK, nbB ? srcB + j * row_step : W, nbB);
        }
        if (++ld_ks == KTS) { ld_ks = 0; ++ld_m; }
        if (++ld_st == kSigmaStages) { ld_st = 0; ld_ph ^= 1; }
      }
      cp_async_commit();
    };
#pragma unroll
    for (int i = 0; i < kAhead; ++i) issue(i);

    int st = 0, sc_m = m_begin, sc_ks = 0;
#pragma unroll 1
    for (int kt = 0; kt < KT; ++kt) {
      issue(kt + kAhead);
      const int s = sc_ks * kBK + c2;
      const double om0 = __ldg(Omega + min(s, s_c - 1)), om1 = __ldg(Omega + min(s + 1, s_c - 1));
      const double em = __ldg(eps + sc_m), fo = __ldg(occ + sc_m);
      cp_async_wait<kAhead>();                    // this thread's copies of k-tile kt have landed
      double *rowA = As + (st * kBM + r0) * kLdK + c2;
      double2 cur[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) cur[j] = *reinterpret_cast<const double2 *>(rowA + 4 * j * kLdK);
      if (fo == 1.0) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const double d = eps_p[j] - em;
          cur[j].x *= denominator_D<1>(d, om0, fo, eta2);
          cur[j].y *= denominator_D<1>(d, om1, fo, eta2);
        }
      } else if (fo == 0.0) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const double d = eps_p[j] - em;
          cur[j].x *= denominator_D<0>(d, om0, fo, eta2);
          cur[j].y *= denominator_D<0>(d, om1, fo, eta2);
        }
      } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const double d = eps_p[j] - em;
          cur[j].x *= denominator_D<2>(d, om0, fo, eta2);
          cur[j].y *= denominator_D<2>(d, om1, fo, eta2);
        }
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) *reinterpret_cast<double2 *>(rowA + 4 * j * kLdK) = cur[j];
      mbar_arrive(full + st);                     // release: the scaled p rows and the landed q rows of this thread
      if (++sc_ks == KTS) { sc_ks = 0; ++sc_m; }
      if (++st == kSigmaStages) st = 0;
    }
    cp_async_wait_all();
  } else {
    // ------------------------------------------------ consumers
    reg_inc<200>();
    const FragMap fm(warp, lane, n_mo - p0, n_mo - q0);
    const bool full_tile = fm.mi_cnt == 8 && fm.nj_cnt == 4;
    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    int st = 0;
    uint32_t ph = 0;
#pragma unroll 1
    for (int kt = 0; kt < KT; ++kt) {
      mbar_wait(full + st, ph);
      if (full_tile) mma_ktile_rowmajor<true>(acc, As + st * kBM * kLdK, Bs + st * kBM * kLdK, fm);
      else mma_ktile_rowmajor<false>(acc, As + st * kBM * kLdK, Bs + st * kBM * kLdK, fm);
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + st);
      if (++st == kSigmaStages) { st = 0; ph ^= 1; }
    }

    double *Tz = Tpart + (int64_t)blockIdx.y * n_mo * n_mo;
    const bool vec_ok = (n_mo & 1) == 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int p = p0 + fm.row(i);
      if (p < n_mo) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
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

}  // namespace qsgw
