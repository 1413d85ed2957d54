// dmma_gemm.cuh -- FP64 tensor-core (DMMA) building blocks and the warp-specialised "TN" GEMM of stages 1 and 2.
//
// sm_100a has no tcgen05 kind for f64 (CUDA 12.9 lists f16/tf32/i8/f8f6f4/mx* only), so FP64 contractions go
// through mma.sync.m8n8k4.f64, which assembles to DMMA.8x8x4 (256 FMA; 64 FMA/clk/SM).  Accumulators live in
// registers.  A CTA is 12 warps: 8 consumer warps (2 x 4, each a 64 x 32 warp tile of 8 x 4 DMMA fragments,
// fragments interleaved across warps so that ragged edge tiles shed work evenly) that do nothing but
// LDS.64 fragment loads + DMMA, and 4 producer warps (one per SM sub-partition) that stage the operand tiles
// global -> shared: with cp.async.bulk row copies of the TMA unit when both operands are 16-byte aligned (two of the
// warps, one lane per k-row), with 8 / 16-byte cp.async (LDGSTS) otherwise.  The two roles meet only through mbarriers (full[stage] /
// empty[stage]); there is no CTA-wide barrier in the main loop, so the DMMA pipe never drains at a k-tile edge.
// Registers are re-split with setmaxnreg (consumers up, producers down).  Shared tiles are padded so that every
// fragment load is bank-conflict free.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qsgw {

constexpr int kConsumerWarps = 8;                    // 2 (M) x 4 (N)
constexpr int kProducerWarps = 4;
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kProducerThreads = kProducerWarps * 32;
constexpr int kThreads = kConsumerThreads + kProducerThreads;   // 384
constexpr int kBM = 128;
constexpr int kBN = 128;
constexpr int kBK = 16;
constexpr int kLdT = kBM + 4;   // k-major tile rows [k][128 + 4]: ld = 4 (mod 16) doubles -> LDS.64 fragments conflict-free
constexpr int kGBK = 32;          // k depth of one ring stage of the stage-1/2 GEMM (two barrier round trips per 8 k4 steps cost ~2 %)
constexpr int kGemmStages = 3;

// D(2 regs) += A(8x4, row) * B(4x8, col); lane holds A[lane/4][lane%4], B[lane%4][lane/4],
// D[lane/4][2*(lane%4) + {0,1}].
__device__ __forceinline__ void dmma_m8n8k4(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(c[0]), "+d"(c[1])
      : "d"(a), "d"(b));
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void cp_async_16(void *smem_dst, const void *gmem_src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(src_bytes)
               : "memory");
}
__device__ __forceinline__ void cp_async_16_s(uint32_t smem_dst, const void *gmem_src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_dst), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_8_s(uint32_t smem_dst, const void *gmem_src, int src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(smem_dst), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// ---- mbarrier pipeline primitives (shared::cta)
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// one arrival on `bar` once all cp.async issued so far by this thread have landed (not counted as pending: the
// barrier's init count includes it)
__device__ __forceinline__ void cp_async_mbar_arrive_noinc(uint64_t *bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
template <int R>
__device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R)); }
template <int R>
__device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(R)); }

// Fragment geometry of consumer warp `warp` (0..7) and lane: warp (wmi, wni) = (warp & 1, warp >> 1) owns the
// 8-row blocks 2i + wmi (i < 8) and the 8-column blocks 4j + wni (j < 4) of the 128 x 128 CTA tile.
struct FragMap {
  int wmi, wni, g, t;      // g = lane / 4 (fragment row / column), t = lane % 4 (k within a k4 step)
  int mi_cnt, nj_cnt;      // fragments of this warp that hold at least one valid row / column (warp-uniform)
  __device__ __forceinline__ FragMap(int warp, int lane, int rows_valid, int cols_valid) {
    wmi = warp & 1; wni = warp >> 1; g = lane >> 2; t = lane & 3;
    const int rb = min(16, (max(rows_valid, 0) + 7) >> 3), cb = min(16, (max(cols_valid, 0) + 7) >> 3);
    mi_cnt = max(0, (rb - wmi + 1) >> 1);
    nj_cnt = max(0, (cb - wni + 3) >> 2);
  }
  __device__ __forceinline__ int row(int i) const { return 16 * i + 8 * wmi + g; }          // of fragment i, this lane's A row
  __device__ __forceinline__ int col(int j) const { return 32 * j + 8 * wni + g; }          // of fragment j, this lane's B column
  __device__ __forceinline__ int out_col(int j) const { return 32 * j + 8 * wni + 2 * t; }  // first of this lane's 2 accumulator columns
};

// The first MI x NJ fragments of the warp, MI and NJ compile-time constants -- a predicated-off DMMA still costs its pipe
// time, so the fragments a warp does not own in a ragged tile must be branched around, not predicated.
template <int MI, int NJ>
__device__ __forceinline__ void mma_ktile_kmajor_frag(double (&acc)[8][4][2], const double *as, const double *bs, const FragMap &fm) {
  const double *ap = as + 8 * fm.wmi + fm.g + fm.t * kLdT;
  const double *bp = bs + 8 * fm.wni + fm.g + fm.t * kLdT;
#pragma unroll
  for (int kk = 0; kk < kGBK / 4; ++kk) {
    double a[MI], b[NJ];
#pragma unroll
    for (int i = 0; i < MI; ++i) a[i] = ap[kk * 4 * kLdT + 16 * i];
#pragma unroll
    for (int j = 0; j < NJ; ++j) b[j] = bp[kk * 4 * kLdT + 32 * j];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int j = 0; j < NJ; ++j) dmma_m8n8k4(acc[i][j], a[i], b[j]);
  }
}

// A full tile's LAST k-tile when K is not a multiple of the ring depth: only the first nsteps k4 steps hold rows k < K (the
// producers zero-filled the rest), so the others are skipped instead of multiplied (K = 1100: 12 of the last 32 rows).
__device__ __forceinline__ void mma_ktile_kmajor_partial(double (&acc)[8][4][2], const double *as, const double *bs, const FragMap &fm,
                                                         int nsteps) {
  const double *ap = as + 8 * fm.wmi + fm.g + fm.t * kLdT;
  const double *bp = bs + 8 * fm.wni + fm.g + fm.t * kLdT;
#pragma unroll 1
  for (int kk = 0; kk < nsteps; ++kk) {
    double a[8], b[4];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = ap[kk * 4 * kLdT + 16 * i];
#pragma unroll
    for (int j = 0; j < 4; ++j) b[j] = bp[kk * 4 * kLdT + 32 * j];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) dmma_m8n8k4(acc[i][j], a[i], b[j]);
  }
}

template <int NJ>
__device__ __forceinline__ void mma_ktile_kmajor_mi(double (&acc)[8][4][2], const double *as, const double *bs, const FragMap &fm) {
  switch (fm.mi_cnt) {
    case 8: mma_ktile_kmajor_frag<8, NJ>(acc, as, bs, fm); break;
    case 7: mma_ktile_kmajor_frag<7, NJ>(acc, as, bs, fm); break;
    case 6: mma_ktile_kmajor_frag<6, NJ>(acc, as, bs, fm); break;
    case 5: mma_ktile_kmajor_frag<5, NJ>(acc, as, bs, fm); break;
    case 4: mma_ktile_kmajor_frag<4, NJ>(acc, as, bs, fm); break;
    case 3: mma_ktile_kmajor_frag<3, NJ>(acc, as, bs, fm); break;
    case 2: mma_ktile_kmajor_frag<2, NJ>(acc, as, bs, fm); break;
    case 1: mma_ktile_kmajor_frag<1, NJ>(acc, as, bs, fm); break;
    default: break;
  }
}

// Dispatch of one k-tile on the (warp-uniform) fragment counts of a ragged tile.
__device__ __forceinline__ void mma_ktile_kmajor_any(double (&acc)[8][4][2], const double *as, const double *bs, const FragMap &fm) {
  switch (fm.nj_cnt) {
    case 4: mma_ktile_kmajor_mi<4>(acc, as, bs, fm); break;
    case 3: mma_ktile_kmajor_mi<3>(acc, as, bs, fm); break;
    case 2: mma_ktile_kmajor_mi<2>(acc, as, bs, fm); break;
    case 1: mma_ktile_kmajor_mi<1>(acc, as, bs, fm); break;
    default: break;
  }
}

// Producer side: stage one k-major operand tile dst[k][c] = src[k*ld + c], k < kGBK, c < 128, with the 128 producer
// threads (pt = 0..127); rows >= kvalid and columns >= cvalid are zero-filled.  VEC = doubles per cp.async
// (2 needs 16-byte aligned src rows).
template <int VEC>
__device__ __forceinline__ void load_tile_kmajor(double *dst, const double *src, int64_t ld, int kvalid, int cvalid,
                                                 const double *safe, int pt) {
  // running source pointer / 32-bit shared address: few live registers, so the 40-72 register producers do not spill
  if (VEC == 2) {
    const int c = (pt & 63) * 2, r0 = pt >> 6;
    int n = cvalid - c;
    n = n < 0 ? 0 : (n > 2 ? 2 : n);
    const int nbytes = n * 8;
    const double *s = src + (int64_t)r0 * ld + c;
    uint32_t d = smem_u32(dst + r0 * kLdT + c);
    const int64_t step = 2 * ld;
#pragma unroll 4
    for (int j = 0; j < kGBK / 2; ++j) {
      const int nb = (r0 + 2 * j < kvalid) ? nbytes : 0;
      cp_async_16_s(d, nb ? s : safe, nb);
      s += step;
      d += 2 * kLdT * (int)sizeof(double);
    }
  } else {
    const int c = pt;
    const int nbc = (c < cvalid) ? 8 : 0;
    const double *s = src + c;
    uint32_t d = smem_u32(dst + c);
#pragma unroll 4
    for (int r = 0; r < kGBK; ++r) {
      const int nb = (r < kvalid) ? nbc : 0;
      cp_async_8_s(d, nb ? s : safe, nb);
      s += ld;
      d += kLdT * (int)sizeof(double);
    }
  }
}

// ---- bulk-copy producer (both operands 16-byte aligned with even leading dimensions)
// One k-row of an operand tile is 128 contiguous doubles in global memory and one padded row of the shared tile, so it
// travels as ONE cp.async.bulk (1 KB, the TMA unit's linear copy, completion counted in bytes on the stage's mbarrier)
// issued by the lane that owns the row: warp 0 of the producers moves the 32 rows of A, warp 1 those of B.  Against
// 16-byte LDGSTS copies through the LSU / L1 path this removes the producers' data return from the path of the DMMA
// warps' fragment loads (measured at the `large` config: the LDGSTS producers cost stage 2 2.3 %).
// Ragged tiles copy round_up(cvalid, 2) columns (the source row has an even leading dimension, so the extra column is
// inside it; columns >= cvalid only reach output columns that are not stored).  Rows k >= kvalid of a last k-tile are
// zero-filled by their lane with ordinary stores.
__device__ __forceinline__ void bulk_copy_row(uint32_t smem_dst, const double *src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_dst), "l"(src),
               "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx_u32(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// Lane `lane` (= k-row of the tile) of one producer warp: dst = shared tile [kGBK][kLdT], src = first valid element of the
// tile (row 0), ld its leading dimension.
__device__ __forceinline__ void bulk_load_tile_kmajor(double *dst, const double *src, int64_t ld, int kvalid, int cvalid, uint64_t *bar,
                                                      int lane) {
  const int cols = min(kBM, (max(cvalid, 0) + 1) & ~1);
  const int rows = min(kvalid, kGBK);
  const uint32_t bar32 = smem_u32(bar);
  if (lane == 0) mbar_arrive_expect_tx_u32(bar32, (uint32_t)(rows * cols * (int)sizeof(double)));
  __syncwarp();
  if (lane < rows) {
    bulk_copy_row(smem_u32(dst + lane * kLdT), src + (int64_t)lane * ld, (uint32_t)(cols * (int)sizeof(double)), bar32);
  } else {
    double2 *row = reinterpret_cast<double2 *>(dst + lane * kLdT);
#pragma unroll 4
    for (int c = 0; c < kBM / 2; ++c) row[c] = make_double2(0.0, 0.0);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // a later bulk copy (async proxy) reuses these rows
  }
  if (lane != 0) mbar_arrive(bar);
}

// ---------------------------------------------------------------- epilogues
// C[row][col] = alpha * acc   (stage 1: V, alpha = 1; AO->MO half transforms); batch b writes at C + b * strideC.
struct EpiStore {
  double *C;
  int64_t ldc;
  double alpha;
  int64_t strideC;   // doubles between the outputs of consecutive batches (0 when there is one batch)
  int vec;           // 1: C 16-byte aligned, ldc and strideC even -> double2 stores
  using RowCtx = int;
  __device__ __forceinline__ EpiStore for_batch(int b) const { return EpiStore{C + (int64_t)b * strideC, ldc, alpha, 0, vec}; }
  __device__ __forceinline__ RowCtx row_ctx(int) const { return 0; }
  __device__ __forceinline__ void operator()(RowCtx, int row, int col, double v0, double v1, int ncols) const {
    double *dst = C + (int64_t)row * ldc + col;
    if (vec && col + 1 < ncols) {
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
  using RowCtx = int2;
  __device__ __forceinline__ EpiPairScatter for_batch(int) const { return *this; }
  __device__ __forceinline__ RowCtx row_ctx(int row) const { return __ldg(pairs + row); }
  __device__ __forceinline__ void operator()(RowCtx pm, int, int col, double v0, double v1, int ncols) const {
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

// Tile t of a batch -> (tm, tn).  tri: only the tiles with tm <= tn of a square tile grid are enumerated (symmetric
// products: t = tn (tn + 1) / 2 + tm); otherwise all ntm x ntn tiles.  m_fastest > 0: tm varies fastest; 0: tn varies
// fastest; < 0: L2-aware order for many row tiles and few column tiles -- the column tiles are taken in groups of
// g = -m_fastest whose B panels (g x K x 128 doubles) fit in L2 together, and inside a group tn varies fastest, so the
// group's B panels stay resident while the A panels stream through once per group.
__device__ __forceinline__ void decode_tile(int t, int ntm, int ntn, int m_fastest, int tri, int &tm, int &tn) {
  if (tri) {
    tn = (int)((sqrtf(8.0f * (float)t + 1.0f) - 1.0f) * 0.5f);
    while (tn * (tn + 1) / 2 > t) --tn;
    while ((tn + 1) * (tn + 2) / 2 <= t) ++tn;
    tm = t - tn * (tn + 1) / 2;
  } else if (m_fastest > 0) {
    tn = t / ntm; tm = t - tn * ntm;
  } else if (m_fastest == 0) {
    tm = t / ntn; tn = t - tm * ntn;
  } else {
    const int g = -m_fastest, per_group = ntm * g;
    const int grp = t / per_group, r = t - grp * per_group;
    const int gsz = min(g, ntn - grp * g);
    tm = r / gsz;
    tn = grp * g + (r - tm * gsz);
  }
}

// Casida matrix (Eqs. (12)-(14)): C[r][c] = 4 sqrt(Delta_r) acc sqrt(Delta_c) + (r == c) Delta_r^2 from
// acc = K[r][c] = (ia|jb).  Launched over the upper-triangle tiles only; off-diagonal tiles also store the mirror element
// C[c][r].  The scale factor is formed as (4 acc) * (sqrt(Delta_r) sqrt(Delta_c)) -- symmetric in r <-> c to the last bit.
struct EpiCasida {
  double *C;
  int64_t ldc;
  const double *sqd;   // [n_ov] sqrt(Delta)
  const double *d;     // [n_ov] Delta
  using RowCtx = double;
  __device__ __forceinline__ EpiCasida for_batch(int) const { return *this; }
  __device__ __forceinline__ RowCtx row_ctx(int row) const { return __ldg(sqd + row); }
  __device__ __forceinline__ void one(double sr, int row, int col, double v) const {
    double c = (4.0 * v) * (sr * __ldg(sqd + col));
    if (row == col) { const double dr = __ldg(d + row); c += dr * dr; }
    C[(int64_t)row * ldc + col] = c;
    if ((row / kBM) != (col / kBN)) C[(int64_t)col * ldc + row] = c;
  }
  __device__ __forceinline__ void operator()(RowCtx sr, int row, int col, double v0, double v1, int ncols) const {
    one(sr, row, col, v0);
    if (col + 1 < ncols) one(sr, row, col + 1, v1);
  }
};

// contraction depth of batch b: K, or what is left of k_total when the batches are K-slices of one product
__device__ __forceinline__ int batch_depth(int K, int k_total, int batch) {
  return k_total > 0 ? max(0, min(K, k_total - batch * K)) : K;
}

constexpr size_t kGemmSmemBytes = (size_t)kGemmStages * 2 * kGBK * kLdT * sizeof(double) + 2 * kGemmStages * sizeof(uint64_t);

// C(M x N) = epilogue( sum_k A[k][m] * B[k][n] ),  A stored [K][lda] (m contiguous), B stored [K][ldb] (n contiguous).
// VECA / VECB = 2 need the operand 16-byte aligned with even leading dimension (and even batch stride); 1 takes anything.
// nbatch independent problems of the same shape (operands strideA / strideB doubles apart, 0 = shared) share one launch.
// k_total > 0 makes the batches the K-slices of ONE product (split-K: batch b contracts k in [b K, min((b+1) K, k_total)),
// the strides advancing K rows, the epilogue storing each slice's partial result).
// ntm * ntn tiles of 128 x 128 dealt round-robin to the grid; m_fastest picks which tile index varies fastest (the
// dimension with fewer tiles, so that concurrently running CTAs share operand panels in L2).
template <int VECA, int VECB, class Epi>
__global__ void __launch_bounds__(kThreads, 1)
gemm_tn_dmma_kernel(const double *__restrict__ A0, int64_t lda, const double *__restrict__ B0, int64_t ldb, int M, int N,
                    int K, int ntm, int ntn, int m_fastest, int nbatch, int64_t strideA, int64_t strideB, int k_total, int tri, Epi epi0) {
  extern __shared__ __align__(16) double smem[];
  double *As = smem;
  double *Bs = smem + kGemmStages * kGBK * kLdT;
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + 2 * kGemmStages * kGBK * kLdT);
  uint64_t *empty = full + kGemmStages;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tiles_per_batch = tri ? ntn * (ntn + 1) / 2 : ntm * ntn;
  const int ntiles = tiles_per_batch * nbatch;

  if (tid == 0) {
    for (int s = 0; s < kGemmStages; ++s) {
      mbar_init(full + s, (VECA == 2 && VECB == 2) ? 64 : kProducerThreads);   // bulk producers: the lanes of two warps
      mbar_init(empty + s, kConsumerWarps);
    }
    mbar_fence_init();
  }
  __syncthreads();

  // Tiles blockIdx.x, blockIdx.x + gridDim.x, ...: with gridDim.x = ntiles this is one tile per CTA; with one CTA per
  // SM it is a persistent kernel whose operand ring runs on across tile boundaries, so the producers prefetch the
  // next tile's first k-tiles while the consumers store the current tile.
  if (warp >= kConsumerWarps) {
    // ------------------------------------------------ producers: cp.async the k-tiles into the ring
    reg_dec<40>();
    const int pt = tid - kConsumerThreads;
    int st = 0;
    uint32_t ph = 1;   // a fresh barrier passes a wait on parity 1: the first pass over the ring does not block
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const int batch = tile / tiles_per_batch, t = tile - batch * tiles_per_batch;
      int tm, tn;
      decode_tile(t, ntm, ntn, m_fastest, tri, tm, tn);
      const int m0 = tm * kBM, n0 = tn * kBN;
      const double *A = A0 + batch * strideA, *Bm = B0 + batch * strideB;
      const int Kb = batch_depth(K, k_total, batch);
      const int KT = (Kb + kGBK - 1) / kGBK;
      for (int kt = 0; kt < KT; ++kt) {
        const int k0 = kt * kGBK;
        if (VECA == 2 && VECB == 2) {
          // bulk-copy producers: warp 0 owns A, warp 1 owns B, the other two have nothing to do
          if (pt < 64) {
            mbar_wait(empty + st, ph);
            if (pt < 32) bulk_load_tile_kmajor(As + st * kGBK * kLdT, A + (int64_t)k0 * lda + m0, lda, Kb - k0, M - m0, full + st, pt);
            else bulk_load_tile_kmajor(Bs + st * kGBK * kLdT, Bm + (int64_t)k0 * ldb + n0, ldb, Kb - k0, N - n0, full + st, pt - 32);
          }
        } else {
          mbar_wait(empty + st, ph);
          load_tile_kmajor<VECA>(As + st * kGBK * kLdT, A + (int64_t)k0 * lda + m0, lda, Kb - k0, M - m0, A, pt);
          load_tile_kmajor<VECB>(Bs + st * kGBK * kLdT, Bm + (int64_t)k0 * ldb + n0, ldb, Kb - k0, N - n0, Bm, pt);
          cp_async_mbar_arrive_noinc(full + st);
        }
        if (++st == kGemmStages) { st = 0; ph ^= 1; }
      }
    }
    cp_async_wait_all();
  } else {
    // ------------------------------------------------ consumers: LDS.64 fragments + DMMA
    reg_inc<232>();
    int st = 0;
    uint32_t ph = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const int batch = tile / tiles_per_batch, t = tile - batch * tiles_per_batch;
      int tm, tn;
      decode_tile(t, ntm, ntn, m_fastest, tri, tm, tn);
      const int m0 = tm * kBM, n0 = tn * kBN;
      const Epi epi = epi0.for_batch(batch);
      const int Kb = batch_depth(K, k_total, batch);
      const int KT = (Kb + kGBK - 1) / kGBK;
      const int last_steps = (Kb - (KT - 1) * kGBK + 3) >> 2;       // k4 steps of the last k-tile that hold rows k < K
      const FragMap fm(warp, lane, M - m0, N - n0);
      const bool full_tile = fm.mi_cnt == 8 && fm.nj_cnt == 4;
      // per-row epilogue context (stage 2: the (p, m) pair of the row), fetched now so its latency hides behind the k loop
      typename Epi::RowCtx rc[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) rc[i] = epi.row_ctx(min(m0 + fm.row(i), M - 1));
      double acc[8][4][2];
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll 1
      for (int kt = 0; kt < KT; ++kt) {
        mbar_wait(full + st, ph);
        if (full_tile && kt == KT - 1 && last_steps < kGBK / 4)
          mma_ktile_kmajor_partial(acc, As + st * kGBK * kLdT, Bs + st * kGBK * kLdT, fm, last_steps);
        else if (full_tile) mma_ktile_kmajor_frag<8, 4>(acc, As + st * kGBK * kLdT, Bs + st * kGBK * kLdT, fm);
        else mma_ktile_kmajor_any(acc, As + st * kGBK * kLdT, Bs + st * kGBK * kLdT, fm);
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + st);
        if (++st == kGemmStages) { st = 0; ph ^= 1; }
      }
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int row = m0 + fm.row(i);
        if (row < M) {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int col = n0 + fm.out_col(j);
            if (col < N) epi(rc[i], row, col, acc[i][j][0], acc[i][j][1], N);
          }
        }
      }
    }
  }
}

}  // namespace qsgw
