// sigma_kernels.cuh -- pack kernels, debug-mode checks, the split-K reduce + symmetrise epilogue of the qsGW Sigma^c
// build (Eq. (19): Sigma = (T + T^T)/2) and the G0W0 diagonal kernel.  Stage 3 itself (the fused
// denominator-scaling + contraction kernel) is in sigma_tma.cuh.
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
// One thread per pair and auxiliary function (4 pairs per thread): the pair table gives (p, m), consecutive pairs of a row p
// are consecutive m, so reads and writes are coalesced, and a small N (the paper's molecules) still fills its blocks.
constexpr int kPackPairsPerBlock = 1024;
__global__ void __launch_bounds__(256)
pack_pairs_kernel(const double *__restrict__ B, const int2 *__restrict__ pairs, int n_mo, int64_t n_pair, double *__restrict__ Bp,
                  int64_t ldp) {
  const int P = blockIdx.y;
  const double *src = B + (int64_t)P * n_mo * n_mo;
  double *dst = Bp + (int64_t)P * ldp;
  const int64_t r0 = (int64_t)blockIdx.x * kPackPairsPerBlock + threadIdx.x;
#pragma unroll
  for (int k = 0; k < kPackPairsPerBlock / 256; ++k) {
    const int64_t r = r0 + k * 256;
    if (r < n_pair) {
      const int2 pm = __ldg(pairs + r);
      dst[r] = __ldg(src + (int64_t)pm.x * n_mo + pm.y);
    }
  }
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

// ---------------------------------------------------------------- Casida / RPA step (row 8(f).4)
// Bov[P][ia] = B[P][i][a] (k-major operand of the C-matrix GEMM; ia = i*v + (a-o)), and for blockIdx.y == n_aux:
// d[ia] = Delta_ia = eps[a] - eps[i], sqd[ia] = sqrt(Delta_ia).
__global__ void casida_gather_kernel(const double *__restrict__ B, const double *__restrict__ eps, int n_mo, int n_occ, int n_aux,
                                     double *__restrict__ Bov, int64_t ld_ov, double *__restrict__ d, double *__restrict__ sqd) {
  const int v = n_mo - n_occ;
  const int64_t n_ov = (int64_t)n_occ * v;
  const int64_t ia = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (ia >= n_ov) return;
  const int i = (int)(ia / v), a = n_occ + (int)(ia - (int64_t)i * v);
  const int P = blockIdx.y;
  if (P < n_aux) {
    Bov[(int64_t)P * ld_ov + ia] = B[((int64_t)P * n_mo + i) * n_mo + a];
  } else {
    const double dd = eps[a] - eps[i];
    d[ia] = dd;
    sqd[ia] = sqrt(dd);
  }
}

// blockIdx.y == gridDim.y - 1 (one extra row of blocks): Omega[s] = sqrt(lambda[s]);
// otherwise Z[ia][s] = sqrt(Delta_ia) * xi[ia][s] / sqrt(Omega_s) for the rows ia = blockIdx.y * 8 .. + 7  (X + Y of Eq. (18)).
// HBM-bound (xi read once, Z written once): a thread owns two adjacent poles and issues the loads of its 8 rows before it
// uses any of them; VEC = 2 needs xi and Z 16-byte aligned with even leading dimensions.
template <int VEC>
__global__ void __launch_bounds__(128)
casida_z_kernel(const double *__restrict__ eps, int n_mo, int n_occ, const double *__restrict__ lambda,
                const double *__restrict__ xi, int64_t ldxi, int64_t n_pole, double *__restrict__ Omega,
                double *__restrict__ Z, int64_t ldz) {
  const int64_t s = 2 * (blockIdx.x * (int64_t)blockDim.x + threadIdx.x);
  if (s >= n_pole) return;
  const bool two = s + 1 < n_pole;
  const double om0 = sqrt(__ldg(lambda + s)), om1 = two ? sqrt(__ldg(lambda + s + 1)) : 1.0;
  if (blockIdx.y == gridDim.y - 1) {
    Omega[s] = om0;
    if (two) Omega[s + 1] = om1;
    return;
  }
  const double rs0 = 1.0 / sqrt(om0), rs1 = 1.0 / sqrt(om1);
  const int v = n_mo - n_occ;
  const int64_t n_ov = (int64_t)n_occ * v;
  const int64_t ia0 = (int64_t)blockIdx.y * 8;
  double x0[8], x1[8], sd[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int64_t ia = min(ia0 + r, n_ov - 1);
    const int i = (int)(ia / v), a = n_occ + (int)(ia - (int64_t)i * v);
    sd[r] = sqrt(__ldg(eps + a) - __ldg(eps + i));
    if (VEC == 2 && two) {
      const double2 t = *reinterpret_cast<const double2 *>(xi + ia * ldxi + s);
      x0[r] = t.x; x1[r] = t.y;
    } else {
      x0[r] = xi[ia * ldxi + s];
      x1[r] = two ? xi[ia * ldxi + s + 1] : 0.0;
    }
  }
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int64_t ia = ia0 + r;
    if (ia < n_ov) {
      const double z0 = sd[r] * x0[r] * rs0, z1 = sd[r] * x1[r] * rs1;
      if (VEC == 2 && two) {
        *reinterpret_cast<double2 *>(Z + ia * ldz + s) = make_double2(z0, z1);
      } else {
        Z[ia * ldz + s] = z0;
        if (two) Z[ia * ldz + s + 1] = z1;
      }
    }
  }
}

// ---------------------------------------------------------------- epilogue
// T = sum_z Tpart[z] in a fixed order, then Eq. (19): Sigma[p][q] = Sigma[q][p] = (T[p][q]+T[q][p])/2, both written
// from the same expression so the output is bit-symmetric.  grid = (nt, nt) tiles of 16 x 16, blocks below the
// diagonal return at once; block = (16, 16, 4): the four z groups each add a contiguous quarter of the slots in
// order, and the four partial sums are combined as ((s0 + s1) + s2) + s3 -- the same order in every run.
constexpr int kEpiTile = 16;
constexpr int kEpiGroups = 4;

__global__ void __launch_bounds__(kEpiTile * kEpiTile * kEpiGroups)
sigma_epilogue_kernel(const double *__restrict__ Tpart, int nsplit, int n_mo, double *__restrict__ Sigma) {
  if (blockIdx.y > blockIdx.x) return;
  __shared__ double Tu[kEpiGroups][kEpiTile][kEpiTile + 1];   // T[p-block rows][q-block cols], per z group
  __shared__ double Tl[kEpiGroups][kEpiTile][kEpiTile + 1];   // T[q-block rows][p-block cols]
  const int pb = blockIdx.y * kEpiTile, qb = blockIdx.x * kEpiTile;
  const int x = threadIdx.x, y = threadIdx.y, g = threadIdx.z;
  const int64_t nn = (int64_t)n_mo * n_mo;
  const int z0 = (int)((int64_t)nsplit * g / kEpiGroups), z1 = (int)((int64_t)nsplit * (g + 1) / kEpiGroups);
  double su = 0.0, sl = 0.0;
  if (pb + y < n_mo && qb + x < n_mo) {
    const double *src = Tpart + (int64_t)(pb + y) * n_mo + qb + x;
    for (int z = z0; z < z1; ++z) su += src[z * nn];
  }
  if (qb + y < n_mo && pb + x < n_mo) {
    const double *src = Tpart + (int64_t)(qb + y) * n_mo + pb + x;
    for (int z = z0; z < z1; ++z) sl += src[z * nn];
  }
  Tu[g][y][x] = su;
  Tl[g][y][x] = sl;
  __syncthreads();
  if (g == 0) {
    Tu[0][y][x] = ((Tu[0][y][x] + Tu[1][y][x]) + Tu[2][y][x]) + Tu[3][y][x];
    Tl[0][y][x] = ((Tl[0][y][x] + Tl[1][y][x]) + Tl[2][y][x]) + Tl[3][y][x];
  }
  __syncthreads();
  if (g == 0 && pb + y < n_mo && qb + x < n_mo) Sigma[(int64_t)(pb + y) * n_mo + qb + x] = 0.5 * (Tu[0][y][x] + Tl[0][x][y]);
  if (g == 1 && qb + y < n_mo && pb + x < n_mo) Sigma[(int64_t)(qb + y) * n_mo + pb + x] = 0.5 * (Tu[0][x][y] + Tl[0][y][x]);
}

// V[P][s] = sum_b Vpart[b][P][s], b = 0..nb-1 in order: the fixed-order reduction of a split-K stage 1 (small problems,
// whose stage-1 GEMM has fewer tiles than the GPU has SMs).  One thread per pair of poles.
__global__ void reduce_split_v_kernel(const double *__restrict__ Vpart, int nb, int64_t stride, int n_aux, int n_cols, int64_t ldv,
                                      double *__restrict__ V) {
  const int c = 2 * (blockIdx.x * blockDim.x + threadIdx.x), P = blockIdx.y;
  if (c >= n_cols || P >= n_aux) return;
  const double2 *src = reinterpret_cast<const double2 *>(Vpart + (int64_t)P * ldv + c);
  double2 acc = *src;
  for (int b = 1; b < nb; ++b) {
    const double2 v = *reinterpret_cast<const double2 *>(Vpart + b * stride + (int64_t)P * ldv + c);
    acc.x += v.x;
    acc.y += v.y;
  }
  *reinterpret_cast<double2 *>(V + (int64_t)P * ldv + c) = acc;
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
