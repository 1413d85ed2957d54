// dmma_gemm.cuh -- FP64 tensor-core (DMMA) building blocks and the "TN" GEMM used by stages 1 and 2.
//
// sm_100a has no tcgen05 kind for f64 (CUDA 12.9 lists f16/tf32/i8/f8f6f4/mx* only), so FP64
// contractions go through mma.sync.m8n8k4.f64, which assembles to DMMA.8x8x4.  Accumulators live in
// registers; operand tiles are staged global -> shared with a 4-deep cp.async (LDGSTS) ring and read
// as LDS.64 fragments from padded, bank-conflict-free layouts.  Measured on B200: an LDS-fed 64x32
// warp tile sustains 36.98 TFLOP/s = 99 % of 148 SM x 64 FMA/clk x 1.965 GHz (profiles/r01_fp64_peaks.md).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qsgw {

constexpr int kThreads = 256;   // 8 warps: 2 (M) x 4 (N), warp tile 64 x 32
constexpr int kBM = 128;
constexpr int kBN = 128;
constexpr int kBK = 16;
constexpr int kStages = 4;
constexpr int kLdT = kBM + 4;   // k-major tile rows [k][128 + 4]: ld = 4 (mod 16) doubles -> LDS.64 fragments conflict-free
constexpr int kLdK = kBK + 4;   // row-major tile rows [row][16 + 4]: same property for the [row][k] layout of stage 3

// D(2 regs) += A(8x4, row) * B(4x8, col); lane holds A[lane/4][lane%4], B[lane%4][lane/4],
// D[lane/4][2*(lane%4) + {0,1}].
__device__ __forceinline__ void dmma_m8n8k4(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(c[0]), "+d"(c[1])
      : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async_16(void *smem_dst, const void *gmem_src, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_8(void *smem_dst, const void *gmem_src, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(s), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// Stage one k-major operand tile: dst[k][c] = src[k*ld + c], k < kBK, c < 128; rows >= kvalid and
// columns >= cvalid are zero-filled.  VEC = doubles per cp.async (2 needs 16-byte aligned src rows).
template <int VEC>
__device__ __forceinline__ void load_tile_kmajor(double *dst, const double *src, int64_t ld, int kvalid, int cvalid,
                                                 const double *safe) {
  const int tid = threadIdx.x;
  if (VEC == 2) {
#pragma unroll
    for (int j = 0; j < (kBK * kBM / 2) / kThreads; ++j) {
      const int id = tid + j * kThreads;
      const int r = id >> 6, c = (id & 63) * 2;
      int n = cvalid - c;
      n = n < 0 ? 0 : (n > 2 ? 2 : n);
      const int nb = (r < kvalid) ? n * 8 : 0;
      cp_async_16(dst + r * kLdT + c, nb ? src + (int64_t)r * ld + c : safe, nb);
    }
  } else {
#pragma unroll
    for (int j = 0; j < (kBK * kBM) / kThreads; ++j) {
      const int id = tid + j * kThreads;
      const int r = id >> 7, c = id & 127;
      const int nb = (r < kvalid && c < cvalid) ? 8 : 0;
      cp_async_8(dst + r * kLdT + c, nb ? src + (int64_t)r * ld + c : safe, nb);
    }
  }
}

// ---------------------------------------------------------------- epilogues
// C[row][col] = alpha * acc   (stage 1: V)
struct EpiStore {
  double *C;
  int64_t ldc;
  double alpha;
  __device__ __forceinline__ void operator()(int row, int col, double v0, double v1, int ncols) const {
    double *dst = C + (int64_t)row * ldc + col;
    if (col + 1 < ncols && ((ldc & 1) == 0)) {
      *reinterpret_cast<double2 *>(dst) = make_double2(alpha * v0, alpha * v1);
    } else {
      dst[0] = alpha * v0;
      if (col + 1 < ncols) dst[1] = alpha * v1;
    }
  }
};

// Rows are symmetric pairs r -> (p <= m); write alpha*acc to W[(m*N+p)][col] and its mirror W[(p*N+m)][col]
// (stage 2: w chunk, w[s][p][m] = w[s][m][p] because B is symmetric).  ldw is even, W 16-byte aligned.
struct EpiPairScatter {
  double *W;
  int64_t ldw;
  const int2 *pairs;
  int n_mo;
  double alpha;
  __device__ __forceinline__ void operator()(int row, int col, double v0, double v1, int ncols) const {
    const int2 pm = __ldg(pairs + row);
    double *d0 = W + ((int64_t)pm.y * n_mo + pm.x) * ldw + col;
    double *d1 = W + ((int64_t)pm.x * n_mo + pm.y) * ldw + col;
    v0 *= alpha;
    v1 *= alpha;
    if (col + 1 < ncols) {
      *reinterpret_cast<double2 *>(d0) = make_double2(v0, v1);
      if (pm.x != pm.y) *reinterpret_cast<double2 *>(d1) = make_double2(v0, v1);
    } else {
      d0[0] = v0;
      if (pm.x != pm.y) d1[0] = v0;
    }
  }
};

constexpr size_t kGemmSmemBytes = (size_t)kStages * 2 * kBK * kLdT * sizeof(double);

// C(M x N) = epilogue( sum_k A[k][m] * B[k][n] ),  A stored [K][lda] (m contiguous), B stored [K][ldb] (n contiguous).
// A must be 16-byte aligned with even lda (library workspace); B may be arbitrary when VECB == 1.
// grid.x = ceil(M/128) * ceil(N/128), n-tile fastest so CTAs that share an A tile run together.
template <int VECB, class Epi>
__global__ void __launch_bounds__(kThreads, 1)
gemm_tn_dmma_kernel(const double *__restrict__ A, int64_t lda, const double *__restrict__ Bm, int64_t ldb, int M, int N,
                    int K, int ntn, Epi epi) {
  extern __shared__ __align__(16) double smem[];
  double *As = smem;
  double *Bs = smem + kStages * kBK * kLdT;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tm = blockIdx.x / ntn, tn = blockIdx.x - tm * ntn;
  const int m0 = tm * kBM, n0 = tn * kBN;
  const int wm = (warp & 1) * 64, wn = (warp >> 1) * 32;
  const int KT = (K + kBK - 1) / kBK;

  auto issue = [&](int kt) {
    if (kt < KT) {
      const int st = kt % kStages, k0 = kt * kBK;
      load_tile_kmajor<2>(As + st * kBK * kLdT, A + (int64_t)k0 * lda + m0, lda, K - k0, M - m0, A);
      load_tile_kmajor<VECB>(Bs + st * kBK * kLdT, Bm + (int64_t)k0 * ldb + n0, ldb, K - k0, N - n0, Bm);
    }
    cp_async_commit();
  };

  double acc[8][4][2];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
  for (int s = 0; s < kStages - 1; ++s) issue(s);

  for (int kt = 0; kt < KT; ++kt) {
    cp_async_wait<kStages - 2>();
    __syncthreads();
    issue(kt + kStages - 1);
    const double *as = As + (kt % kStages) * kBK * kLdT + wm + (lane >> 2);
    const double *bs = Bs + (kt % kStages) * kBK * kLdT + wn + (lane >> 2);
#pragma unroll
    for (int kk = 0; kk < kBK / 4; ++kk) {
      const int k = kk * 4 + (lane & 3);
      double a[8], b[4];
#pragma unroll
      for (int i = 0; i < 8; ++i) a[i] = as[k * kLdT + 8 * i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = bs[k * kLdT + 8 * j];
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma_m8n8k4(acc[i][j], a[i], b[j]);
    }
  }
  cp_async_wait<0>();

#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int row = m0 + wm + 8 * i + (lane >> 2);
    if (row < M) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int col = n0 + wn + 8 * j + 2 * (lane & 3);
        if (col < N) epi(row, col, acc[i][j][0], acc[i][j][1], N);
      }
    }
  }
}

}  // namespace qsgw
