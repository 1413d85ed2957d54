// sigma_tma.cuh -- stage 3 of the qsGW Sigma^c build: the fused denominator-scaling + contraction kernel.
//
// Evaluates Eq. (17) of the paper at omega = eps_p for every (p, q):
//   T[p][q] = sum_m sum_s ( w[s][p][m] * D(m,s,eps_p) ) * w[s][q][m]
// as ONE GEMM T = A W^T over k = (m, s) whose left operand A[p][k] = w * D is formed in shared memory by the operand
// producers of the same kernel: the scaled operand never exists in HBM.  Eq. (19) is then
// Sigma = (T + T^T)/2 (epilogue kernel).
//
// Organisation (one CTA = one 64 (p) x tq (q <= 256) tile of T for the internal states m of one split-K slot):
//   * operand tiles travel global -> shared by TMA (cp.async.bulk.tensor, 3-D tensor maps [m][p][s] with the 128-byte
//     swizzle, out-of-range rows / poles zero-filled by the hardware), issued by ONE elected thread;
//   * k-tiles are 32 poles deep at one m (two 16-pole = 128-byte halves), so eps_m / f_m are CTA-uniform per k-tile;
//   * the two operands have their own rings: the p rows (16 KB per k-tile) sit in a DEEP ring, because they must be
//     scaled by D before use -- three producer warps multiply them in place, several k-tiles ahead of the DMMA
//     warps, so that the latency of their FP64 bursts (they share the FP64 pipe with the DMMAs and are served in its
//     gaps) stays off the critical path; the q rows go straight from TMA to the DMMA warps through a ring managed in
//     16-pole halves of a k-tile (a half is released, and its refill issued, as soon as it has been consumed);
//   * 8 consumer warps (2 x 4) run LDS.64 fragment loads + DMMA.8x8x4 only, software-pipelined across k4 steps and ring
//     stages (the next fragments, barrier waits included, are fetched under the current DMMAs); accumulators in registers;
//   * split-K over a linear (m, 32-pole group) index into slot-owned partial tiles (fixed accumulation order, no atomics);
//   * two instances: <true> for tiles of up to 224 columns (at most 7 column fragments per warp: 112 accumulator
//     registers, hand-pipelined DMMA loop), <false> for 256-column tiles (all 128 accumulator registers, plain loop).
#pragma once
#include <cuda.h>

#include "dmma_gemm.cuh"

namespace qsgw {

// D(m,s,omega) = occ_m * x1/(x1^2+eta^2) + (1-occ_m) * x2/(x2^2+eta^2),  x1 = (omega-eps_m)+Omega_s,
// x2 = (omega-eps_m)-Omega_s: real part of the two terms of Eq. (17).  d = omega - eps_m.
// x/(x^2+eta^2) without the IEEE division's slow path: y = x^2+eta^2, r = MUFU.RCP64H(y) (relative error
// e = 1 - y r, |e| <= 2^-20 measured), 1/y = r (1 + e + e^2 + O(e^3)), so x/y = q + q (e + e^2) with q = x r:
// 5 FP64-pipe instructions, error <= 1 ulp (|e|^3 = 2^-60).  y >= eta^2 > 0 is never subnormal for physical energies.
__device__ __forceinline__ double lehmann_term(double x, double eta2) {
  const double y = fma(x, x, eta2);
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(y));
  const double q = x * r;
  const double e = fma(-y, r, 1.0);
  const double t = fma(e, e, e);
  return fma(q, t, q);
}

// general occupation 0 <= f_m <= 1: both terms
__device__ __forceinline__ double denominator_D_fractional(double d, double Omega_s, double occ_m, double eta2) {
  return occ_m * lehmann_term(d + Omega_s, eta2) + (1.0 - occ_m) * lehmann_term(d - Omega_s, eta2);
}

constexpr int kTP = 64;                 // p rows of the CTA tile
constexpr int kTQMax = 256;             // q columns of the CTA tile, at most (a multiple of 8 chosen per N at launch)
constexpr int kKD = 32;                 // poles per k-tile: two halves of 16 doubles = 128 bytes (the TMA swizzle span)
constexpr int kHalfRowBytes = 128;
constexpr int kAStageBytes = 2 * kTP * kHalfRowBytes;   // 16 KB
constexpr int kMaxAStages = 6;
constexpr int kScaleWarps = 3;           // producer warps that scale (the fourth issues the TMA loads)
constexpr int kMaxBStages = 8;           // q-row ring stages (each ONE 16-pole half of a k-tile)
constexpr size_t kSigmaSmemBudget = 227 * 1024 - 1024;  // dynamic shared memory of one CTA, less the alignment slack

struct SigmaRings {
  int nA, nB;            // ring depths: p ring in k-tiles, q ring in 16-pole HALVES of a k-tile
  int b_stage_bytes;     // tq * 128: one half of a k-tile of q rows
  size_t smem_bytes;     // dynamic shared memory to launch with (includes 1 KB of alignment slack and the barriers)
};

// Ring depths for a tile tq columns wide.  The q rows go straight from TMA to the DMMA warps, so their ring is what hides
// the load latency: it is managed in half k-tiles (a stage is released -- and its refill issued -- as soon as its 16 poles
// are consumed) and gets the shared memory the p ring does not need.  The p ring keeps nA k-tiles: one being read, up to
// three being scaled by the three scaling warps, the rest landing.
inline SigmaRings sigma_rings(int tq) {
  SigmaRings r;
  r.b_stage_bytes = tq * kHalfRowBytes;
  const size_t bar_bytes = 1024;
  const size_t avail = kSigmaSmemBudget - bar_bytes;
  r.nA = 6;
  r.nB = (int)((avail - (size_t)r.nA * kAStageBytes) / r.b_stage_bytes);
  if (r.nB > kMaxBStages) r.nB = kMaxBStages;
  if (r.nB < 2) r.nB = 2;
  r.smem_bytes = 1024 + (size_t)r.nA * kAStageBytes + (size_t)r.nB * r.b_stage_bytes + bar_bytes;
  return r;
}

// ---- TMA / mbarrier primitives used here
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// non-blocking probe: has the phase with this parity completed?
__device__ __forceinline__ bool mbar_test(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "mbarrier.test_wait.parity.shared::cta.b64 P1, [%1], %2;\n"
      "selp.u32 %0, 1, 0, P1;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void tma_load_3d(uint32_t smem_dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(smem_dst), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

struct SigmaFragMap {
  int wmi, wni, g, t;
  int mi_cnt, nj_cnt;   // fragments of this warp with at least one valid row / column (warp-uniform)
  __device__ __forceinline__ SigmaFragMap(int warp, int lane, int rows_valid, int cols_valid) {
    wmi = warp & 1; wni = warp >> 1; g = lane >> 2; t = lane & 3;
    const int rb = min(kTP / 8, (max(rows_valid, 0) + 7) >> 3), cb = min(kTQMax / 8, (max(cols_valid, 0) + 7) >> 3);
    mi_cnt = max(0, (rb - wmi + 1) >> 1);
    nj_cnt = max(0, (cb - wni + 3) >> 2);
  }
  __device__ __forceinline__ int row(int i) const { return 16 * i + 8 * wmi + g; }
  __device__ __forceinline__ int out_col(int j) const { return 32 * j + 8 * wni + 2 * t; }
};

// Ring state of the DMMA warps, as 32-bit shared-window addresses (few registers: the accumulators take 128 of them).
struct SigmaConsumerRings {
  uint32_t a_ring, b_ring;            // ring bases plus this lane's row / byte offset
  uint32_t a_full, a_empty, b_full, b_empty;   // barrier arrays (8 bytes per stage)
  int nA, nB, b_stage_bytes;
};

__device__ __forceinline__ double lds_f64(uint32_t addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void mbar_wait_s(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive_s(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// The whole k loop of a CTA tile for the first MI x NJ fragments of the warp: acc[i][j] += A[p rows of fragment i][k] *
// Wq[q rows of fragment j][k] over the KT k-tiles of the split-K slot, two 16-pole halves per k-tile, four k4 steps per
// half.  Rows are 128 bytes; fragment i of the p operand is 16 rows further, fragment j of the q operand 32 rows; sw[kk]
// is the lane's swizzled 16-byte chunk offset of k4 step kk.  MI, NJ are compile-time: a predicated-off DMMA still
// occupies the FP64 pipe for its full issue time, so ragged edge tiles BRANCH around unowned fragments.
// Software-pipelined across k4 steps AND ring stages without a second set of fragment registers: the fragments of the
// next step are fetched into the registers of this step as they fall free (a[i] after the DMMAs of row i, b[j] during
// the last row); at the last step of a half the barrier waits of the next half come first.  The q-row stage of a half
// is released as soon as that half is consumed; the p-row stage after both halves.
template <int MI, int NJ, int NJM>
__device__ __forceinline__ void sigma_consumer_kloop(double (&acc)[4][NJM][2], const SigmaConsumerRings &r, uint32_t sw0, int KT, int lane) {
  int sa = 0, sb = 0;
  uint32_t pha = 0, phb = 0;
  double a[MI], b[NJ];
  mbar_wait_s(r.b_full, 0);
  mbar_wait_s(r.a_full, 0);
  uint32_t ap = r.a_ring, bp = r.b_ring;
#pragma unroll
  for (int i = 0; i < MI; ++i) a[i] = lds_f64((ap ^ sw0) + 16 * i * kHalfRowBytes);
#pragma unroll
  for (int j = 0; j < NJ; ++j) b[j] = lds_f64((bp ^ sw0) + 32 * j * kHalfRowBytes);
#pragma unroll 1
  for (int kt = 0; kt < KT; ++kt) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
#pragma unroll
      for (int kk = 0; kk < 4; ++kk) {
        // sw[kk] = sw0 ^ (kk << 4), applied with XOR: the lane offsets in ap / bp are multiples of 128 plus 0 or 8, so
        // bits 4..6 of the address are free
        const bool edge = (kk == 3);
        bool fetch = true;
        uint32_t apx, bpx;
        if (edge) {
          fetch = (h == 0) || (kt + 1 < KT);
          const int sb_n = (sb + 1 == r.nB) ? 0 : sb + 1;
          const int sa_n = h ? ((sa + 1 == r.nA) ? 0 : sa + 1) : sa;
          if (fetch) {
            mbar_wait_s(r.b_full + 8 * sb_n, (sb + 1 == r.nB) ? phb ^ 1 : phb);
            if (h) mbar_wait_s(r.a_full + 8 * sa_n, (sa + 1 == r.nA) ? pha ^ 1 : pha);
          }
          apx = (r.a_ring + sa_n * kAStageBytes + (h ? 0 : kTP * kHalfRowBytes));
          bpx = (r.b_ring + sb_n * r.b_stage_bytes);
        } else {
          apx = ap ^ ((kk + 1) << 4);
          bpx = bp ^ ((kk + 1) << 4);
        }
        apx ^= sw0;
        bpx ^= sw0;
#pragma unroll
        for (int i = 0; i < MI; ++i) {
#pragma unroll
          for (int j = 0; j < NJ; ++j) {
            dmma_m8n8k4(acc[i][j], a[i], b[j]);
            if (i == MI - 1 && fetch) b[j] = lds_f64(bpx + 32 * j * kHalfRowBytes);
          }
          if (fetch) a[i] = lds_f64(apx + 16 * i * kHalfRowBytes);
        }
      }
      __syncwarp();
      if (lane == 0) {
        mbar_arrive_s(r.b_empty + 8 * sb);         // this half of the q rows can be refilled while the other is in use
        if (h) mbar_arrive_s(r.a_empty + 8 * sa);
      }
      if (++sb == r.nB) { sb = 0; phb ^= 1; }
      if (h && ++sa == r.nA) { sa = 0; pha ^= 1; }
      ap = r.a_ring + sa * kAStageBytes + (h ? 0 : kTP * kHalfRowBytes);
      bp = r.b_ring + sb * r.b_stage_bytes;
    }
  }
}

// One 16-pole half of a k-tile: acc[i][j] += A[p rows of fragment i][k] * Wq[q rows of fragment j][k], k = 0..15, for
// the first MI x NJ fragments of the warp.  ap / bp: this lane's row (8 wmi + g resp. 8 wni + g) of the half, at byte
// offset 8 (t & 1); sw[kk]: the lane's swizzled 16-byte chunk offset of k4 step kk.  Rows are 128 bytes; fragment i of
// the p operand is 16 rows further, fragment j of the q operand 32 rows.  MI, NJ are compile-time: a predicated-off
// DMMA still occupies the FP64 pipe for its full issue time, so ragged edge tiles BRANCH around unowned fragments.
template <int MI, int NJ, int NJM>
__device__ __forceinline__ void mma_half_sigma(double (&acc)[4][NJM][2], const char *ap, const char *bp, const int (&sw)[4]) {
#pragma unroll
  for (int kk = 0; kk < 4; ++kk) {
    double a[MI], b[NJ];
#pragma unroll
    for (int i = 0; i < MI; ++i) a[i] = *reinterpret_cast<const double *>(ap + 16 * i * kHalfRowBytes + sw[kk]);
#pragma unroll
    for (int j = 0; j < NJ; ++j) b[j] = *reinterpret_cast<const double *>(bp + 32 * j * kHalfRowBytes + sw[kk]);
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int j = 0; j < NJ; ++j) dmma_m8n8k4(acc[i][j], a[i], b[j]);
  }
}

template <int MI, int NJM>
__device__ __forceinline__ void mma_half_sigma_nj(double (&acc)[4][NJM][2], const char *ap, const char *bp, const int (&sw)[4], int nj) {
  switch (nj) {
    case 1: if constexpr (NJM >= 1) mma_half_sigma<MI, 1>(acc, ap, bp, sw); break;
    case 2: if constexpr (NJM >= 2) mma_half_sigma<MI, 2>(acc, ap, bp, sw); break;
    case 3: if constexpr (NJM >= 3) mma_half_sigma<MI, 3>(acc, ap, bp, sw); break;
    case 4: if constexpr (NJM >= 4) mma_half_sigma<MI, 4>(acc, ap, bp, sw); break;
    case 5: if constexpr (NJM >= 5) mma_half_sigma<MI, 5>(acc, ap, bp, sw); break;
    case 6: if constexpr (NJM >= 6) mma_half_sigma<MI, 6>(acc, ap, bp, sw); break;
    case 7: if constexpr (NJM >= 7) mma_half_sigma<MI, 7>(acc, ap, bp, sw); break;
    case 8: if constexpr (NJM >= 8) mma_half_sigma<MI, 8>(acc, ap, bp, sw); break;
    default: break;
  }
}

// Ragged tile: dispatch (warp-uniform) on the fragment counts of this warp.
template <int NJM>
__device__ __forceinline__ void mma_half_sigma_ragged(double (&acc)[4][NJM][2], const char *ap, const char *bp, const int (&sw)[4],
                                                      int mi, int nj) {
  switch (mi) {
    case 1: mma_half_sigma_nj<1>(acc, ap, bp, sw, nj); break;
    case 2: mma_half_sigma_nj<2>(acc, ap, bp, sw, nj); break;
    case 3: mma_half_sigma_nj<3>(acc, ap, bp, sw, nj); break;
    case 4: mma_half_sigma_nj<4>(acc, ap, bp, sw, nj); break;
    default: break;
  }
}


// The k loop for every other fragment count (256-column tiles with all 8 column fragments, the short last p row, narrow
// last q-tiles): ONE loop with the (warp-uniform) dispatch on the fragment counts inside, barrier waits at the top of a
// half.  With all 128 accumulator registers in use the hand-pipelined loop above spills ~20 doubles per k-tile (xl: 7891 vs
// 7662 ms per build), and one loop per fragment-count pair makes ptxas spill in all of them, so only the hot
// pairs of the small-to-large sizes (4 x 4..7) get the pipelined loop.
template <int NJM>
__device__ __forceinline__ void sigma_consumer_kloop_generic(double (&acc)[4][NJM][2], const char *a_ring, const char *b_ring,
                                                             int b_stage_bytes, uint64_t *a_full, uint64_t *a_empty, uint64_t *b_full,
                                                             uint64_t *b_empty, int nA, int nB, const int (&sw)[4], int KT, int lane,
                                                             int mi, int nj) {
  const bool full_tile = mi == 4 && nj == 8;
  int sa = 0, sb = 0;
  uint32_t pha = 0, phb = 0;
#pragma unroll 1
  for (int kt = 0; kt < KT; ++kt) {
    mbar_wait(a_full + sa, pha);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      mbar_wait(b_full + sb, phb);
      const char *ap = a_ring + sa * kAStageBytes + h * (kTP * kHalfRowBytes);
      const char *bp = b_ring + (size_t)sb * b_stage_bytes;
      if (NJM == 8 && full_tile) mma_half_sigma<4, NJM>(acc, ap, bp, sw);
      else mma_half_sigma_ragged(acc, ap, bp, sw, mi, nj);
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(b_empty + sb);                 // this half of the q rows can be refilled while the other is in use
        if (h) mbar_arrive(a_empty + sa);
      }
      if (++sb == nB) { sb = 0; phb ^= 1; }
    }
    if (++sa == nA) { sa = 0; pha ^= 1; }
  }
}

// One CTA: output tile (tp, tq) of T, 64 x tq, for the k-tiles of split-K slot z: a contiguous range of the
// (m, 32-pole group) pairs of the chunk (s_c poles, all internal states m).
//   mapA  tensor map of the left operand (scaled by D)  [m][p][s], box {16 poles, 64 rows, 1}.  qsGW: the w chunk of
//         stage 2 (both mirrors present); qsMP2 exchange term: the exchange integrals (pi|an)
//   mapB  tensor map of the right operand, same indexing, box {16 poles, tq rows, 1}.  qsGW: the same array
//   Omega [s_c]  excitation energies of the chunk
//   Tpart [nsplit][N][N]  split-K partial tiles; slot z is owned by the CTAs of that slot and is
//         read-modify-written once per launch -> accumulation order is fixed, results reproducible.
// PIPE: the hand-pipelined DMMA loop for 4 x 4..7 fragments per warp (tiles of 104..224 columns); the host launches the
// PIPE = false instance for wider tiles (all 8 column fragments in use, see sigma_consumer_kloop_generic).
template <bool PIPE>
__global__ void __launch_bounds__(kThreads, 1)
sigma_accumulate_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                        const double *__restrict__ eps, const double *__restrict__ occ, const double *__restrict__ Omega,
                        int n_mo, int s_c, double eta2, int nsplit, int ntq, int tq, int nA, int nB,
                        double *__restrict__ Tpart) {
  extern __shared__ uint8_t smem_raw[];
  // the 128-byte swizzle pattern is a function of the shared-memory ADDRESS: stage bases must be 1024-byte aligned
  // (offset added to the __shared__ array itself, so that the compiler keeps emitting LDS / STS rather than generic accesses)
  uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int b_stage_bytes = tq * kHalfRowBytes;   // one 16-pole half of a k-tile
  uint8_t *a_ring = smem;
  uint8_t *b_ring = smem + nA * kAStageBytes;
  uint64_t *bars = reinterpret_cast<uint64_t *>(b_ring + (size_t)nB * b_stage_bytes);
  uint64_t *a_raw = bars;                       // [nA] TMA landed (tx bytes)            -> producers
  uint64_t *a_full = a_raw + kMaxAStages;       // [nA] scaled by all producer threads   -> consumers
  uint64_t *a_empty = a_full + kMaxAStages;     // [nA] read by all consumer warps       -> TMA issuer
  uint64_t *b_full = a_empty + kMaxAStages;     // [nB] TMA landed                       -> consumers
  uint64_t *b_empty = b_full + kMaxBStages;     // [nB] read by all consumer warps       -> TMA issuer

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // CTA -> (tile, split-K slot z).  CTAs start in the order of their linear index; the tiles of the last, short p row
  // (N mod 64 rows) run 2-3 times shorter than the others, so they are numbered LAST: the end of the launch is filled
  // with short CTAs instead of waiting for a long one.  Within either group the tile index varies fastest, so the CTAs
  // of one slot (same m range, same w rows) run at the same time and share those rows in L2.
  int tile, z;
  {
    const int ntiles = gridDim.x, nfull = (n_mo / kTP) * ntq, nrag = ntiles - nfull;
    const int lin = blockIdx.y * ntiles + blockIdx.x;
    if (lin < nfull * nsplit) { z = lin / nfull; tile = lin - z * nfull; }
    else { const int l2 = lin - nfull * nsplit; z = l2 / nrag; tile = nfull + (l2 - z * nrag); }
  }
  const int tp = tile / ntq, tqi = tile - tp * ntq;
  const int p0 = tp * kTP, q0 = tqi * tq;
  // split-K: the k-tiles (m, ks), numbered m * KTS + ks, are dealt to the nsplit slots in equal contiguous ranges
  const int KTS = (s_c + kKD - 1) / kKD;         // k-tiles per m
  const int kt_begin = (int)((int64_t)n_mo * KTS * z / nsplit);
  const int KT = (int)((int64_t)n_mo * KTS * (z + 1) / nsplit) - kt_begin;

  if (tid == 0) {
    for (int s = 0; s < nA; ++s) {
      mbar_init(a_raw + s, 1);
      mbar_init(a_full + s, 32);              // the 32 lanes of the scaling warp that owns the k-tile
      mbar_init(a_empty + s, kConsumerWarps);
    }
    for (int s = 0; s < nB; ++s) {
      mbar_init(b_full + s, 1);
      mbar_init(b_empty + s, kConsumerWarps);
    }
    mbar_fence_init();
  }
  __syncthreads();

  // registers are a per-sub-partition resource (16 K each, holding two DMMA warps and one producer warp): 2 x 184 + 136
  if (warp >= kConsumerWarps) reg_dec<136>();     // the whole producer warpgroup, one instruction
  if (warp == kConsumerWarps) {
    // ------------------------------------------------ TMA issuer (one elected thread of the first producer warp)
    // Its own warp, so that it never waits for the FP64 pipe: the scaling warps below are served only in the gaps of
    // the DMMA streams, and a load that waits behind their arithmetic would stall everybody.
    if (lane == 0) {
      int a_next = 0, a_st = 0, a_m = kt_begin / KTS, a_ks = kt_begin - (kt_begin / KTS) * KTS;
      uint32_t a_ph = 1;                          // a fresh barrier passes a wait on parity 1
      int b_next = 0, b_st = 0, b_m = a_m, b_s0 = a_ks * kKD;     // the q ring advances in halves of a k-tile
      uint32_t b_ph = 1;
      const int KTB = 2 * KT, s_end = KTS * kKD;
      // both rings in k-tile order, never blocking on one ring while the other has a free stage
      while (a_next < KT || b_next < KTB) {
        bool issued = false;
        if (a_next < KT && mbar_test(a_empty + a_st, a_ph)) {
          mbar_arrive_expect_tx(a_raw + a_st, kAStageBytes);
          const uint32_t dst = smem_u32(a_ring + a_st * kAStageBytes);
          tma_load_3d(dst, &mapA, a_raw + a_st, a_ks * kKD, p0, a_m);
          tma_load_3d(dst + kTP * kHalfRowBytes, &mapA, a_raw + a_st, a_ks * kKD + 16, p0, a_m);
          ++a_next;
          if (++a_ks == KTS) { a_ks = 0; ++a_m; }
          if (++a_st == nA) { a_st = 0; a_ph ^= 1; }
          issued = true;
        }
        if (b_next < KTB && mbar_test(b_empty + b_st, b_ph)) {
          mbar_arrive_expect_tx(b_full + b_st, b_stage_bytes);
          tma_load_3d(smem_u32(b_ring + (size_t)b_st * b_stage_bytes), &mapB, b_full + b_st, b_s0, q0, b_m);
          ++b_next;
          if ((b_s0 += 16) == s_end) { b_s0 = 0; ++b_m; }
          if (++b_st == nB) { b_st = 0; b_ph ^= 1; }
          issued = true;
        }
        if (!issued) __nanosleep(64);
      }
    }
  } else if (warp > kConsumerWarps) {
    // ------------------------------------------------ scaling warps: multiply the p rows of a k-tile by D in place
    // The three warps take whole k-tiles in turn (warp j: k-tiles j, j + 3, ...), so three k-tiles are in work at any
    // time and each warp has three k-tile periods for the dependent steps of its FP64 bursts.
    const int sw_id = warp - kConsumerWarps - 1;  // 0..2
    const int cc = lane & 7;                      // this lane's 16-byte chunk (2 poles) of every 16-pole half
    const int rsub = lane >> 3;                   // its rows: rsub + 4 j, j < 16
    double eps_p[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) eps_p[j] = (p0 + rsub + 4 * j < n_mo) ? __ldg(eps + p0 + rsub + 4 * j) : 0.0;
    // byte offset of its chunk in row rsub + 4 j of a half: rows alternate between r & 7 = rsub and rsub + 4
    const uint32_t off_even = rsub * kHalfRowBytes + ((cc ^ rsub) << 4);
    const uint32_t off_odd = (rsub + 4) * kHalfRowBytes + ((cc ^ (rsub + 4)) << 4);
    int st = sw_id % nA;
    uint32_t ph = (sw_id / nA) & 1;
#pragma unroll 1
    for (int kt = sw_id; kt < KT; kt += kScaleWarps) {
      const int m = (kt_begin + kt) / KTS, ks = (kt_begin + kt) - m * KTS;
      const double em = __ldg(eps + m), fo = __ldg(occ + m);
      const long long fbits = __double_as_longlong(fo);
      // occupation class by bit pattern (no FP64-pipe compare): 1.0 -> occupied term only, +-0.0 -> virtual term only
      const int occ_class = (fbits == 0x3FF0000000000000LL) ? 1 : (((unsigned long long)fbits << 1) == 0ULL ? 0 : 2);
      const double sgn = occ_class == 1 ? 1.0 : -1.0;
      double om[4];                               // Omega of this lane's 4 poles of the k-tile (2 per half)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        om[2 * h] = __ldg(Omega + min(ks * kKD + h * 16 + 2 * cc, s_c - 1));
        om[2 * h + 1] = __ldg(Omega + min(ks * kKD + h * 16 + 2 * cc + 1, s_c - 1));
      }
      mbar_wait(a_raw + st, ph);                  // the raw p rows of this k-tile have landed
      uint8_t *tile = a_ring + st * kAStageBytes;
      if (occ_class != 2) {
        // f_m in {0, 1}: one Lehmann term, x = d + sgn * Omega_s.  8 evaluations (2 rows x 2 halves x 2 poles) advance
        // together, stage by stage, so that each dependent step is ONE burst of 8 independent FP64 instructions.
#pragma unroll
        for (int b = 0; b < 8; ++b) {
          double x[8], y[8], r[8];                // element e = (row jj, half h, pole c): e = 4 jj + 2 h + c
#pragma unroll
          for (int e = 0; e < 8; ++e) x[e] = fma(sgn, om[e & 3], eps_p[2 * b + (e >> 2)] - em);
#pragma unroll
          for (int e = 0; e < 8; ++e) y[e] = fma(x[e], x[e], eta2);
#pragma unroll
          for (int e = 0; e < 8; ++e) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r[e]) : "d"(y[e]));
#pragma unroll
          for (int e = 0; e < 8; ++e) x[e] *= r[e];                      // q = x r
#pragma unroll
          for (int e = 0; e < 8; ++e) y[e] = fma(-y[e], r[e], 1.0);      // e = 1 - y r
#pragma unroll
          for (int e = 0; e < 8; ++e) y[e] = fma(y[e], y[e], y[e]);      // t = e + e^2
#pragma unroll
          for (int e = 0; e < 8; ++e) x[e] = fma(x[e], y[e], x[e]);      // D = q + q t
#pragma unroll
          for (int jj = 0; jj < 2; ++jj)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              double2 *ptr = reinterpret_cast<double2 *>(tile + h * (kTP * kHalfRowBytes) + b * (8 * kHalfRowBytes) +
                                                         (jj ? off_odd : off_even));
              double2 v = *ptr;
              v.x *= x[4 * jj + 2 * h];
              v.y *= x[4 * jj + 2 * h + 1];
              *ptr = v;
            }
        }
      } else {
#pragma unroll
        for (int j = 0; j < 16; ++j)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            double2 *ptr = reinterpret_cast<double2 *>(tile + h * (kTP * kHalfRowBytes) + (j >> 1) * (8 * kHalfRowBytes) +
                                                       ((j & 1) ? off_odd : off_even));
            double2 v = *ptr;
            const double dj = eps_p[j] - em;
            v.x *= denominator_D_fractional(dj, om[2 * h], fo, eta2);
            v.y *= denominator_D_fractional(dj, om[2 * h + 1], fo, eta2);
            *ptr = v;
          }
      }
      fence_proxy_async_smem();                   // these generic-proxy writes precede the TMA write that later reuses the stage
      mbar_arrive(a_full + st);                   // release: the scaled chunks of this lane
      // the warp's next k-tile is kScaleWarps stages further along the ring
      st += kScaleWarps;
      if (st >= nA) { st -= nA; ph ^= 1; }
    }
  } else {
    // ------------------------------------------------ consumers
    reg_inc<184>();
    const int cols_valid = min(tq, n_mo - q0);
    const SigmaFragMap fm(warp, lane, n_mo - p0, cols_valid);
    constexpr int NJM = PIPE ? 7 : 8;      // column fragments a warp can own: the accumulator registers follow
    double acc[4][NJM][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < NJM; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    // 128-byte swizzle: 16-byte chunk c of row r lives at chunk c ^ (r & 7); every fragment row of this lane has
    // r & 7 == g.  Which of the 16 poles of a half a lane feeds into which k4 step is free as long as both operands agree
    // (the contraction sums over all of them), so lane t of step kk takes pole 8 (t >> 1) + 2 kk + (t & 1): chunk
    // 4 (t >> 1) + kk, half (t & 1) of it.  The 16 lanes of a half warp (4 rows g x 4 t) then hit 16 distinct 8-byte
    // bank pairs -- with the natural choice 4 kk + t, rows g and g ^ 1 would collide on the same two chunks.
    const uint32_t sw = (uint32_t)(fm.g ^ ((fm.t >> 1) << 2)) << 4;   // k4 step kk reads chunk offset sw ^ (kk << 4)
    const int a_lane = (8 * fm.wmi + fm.g) * kHalfRowBytes + 8 * (fm.t & 1);
    const int b_lane = (8 * fm.wni + fm.g) * kHalfRowBytes + 8 * (fm.t & 1);
    if (KT > 0) {
      if (PIPE && fm.mi_cnt == 4 && fm.nj_cnt >= 4 && fm.nj_cnt <= 7) {
        SigmaConsumerRings rings;
        rings.a_ring = smem_u32(a_ring) + a_lane;
        rings.b_ring = smem_u32(b_ring) + b_lane;
        rings.a_full = smem_u32(a_full); rings.a_empty = smem_u32(a_empty);
        rings.b_full = smem_u32(b_full); rings.b_empty = smem_u32(b_empty);
        rings.nA = nA; rings.nB = nB; rings.b_stage_bytes = b_stage_bytes;
        if (fm.nj_cnt == 7) sigma_consumer_kloop<4, 7>(acc, rings, sw, KT, lane);
        else if (fm.nj_cnt == 6) sigma_consumer_kloop<4, 6>(acc, rings, sw, KT, lane);
        else if (fm.nj_cnt == 5) sigma_consumer_kloop<4, 5>(acc, rings, sw, KT, lane);
        else sigma_consumer_kloop<4, 4>(acc, rings, sw, KT, lane);
      } else {
        int swk[4];
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) swk[kk] = (int)(sw ^ (kk << 4));
        sigma_consumer_kloop_generic(acc, reinterpret_cast<const char *>(a_ring) + a_lane, reinterpret_cast<const char *>(b_ring) + b_lane,
                                     b_stage_bytes, a_full, a_empty, b_full, b_empty, nA, nB, swk, KT, lane, fm.mi_cnt, fm.nj_cnt);
      }
    }

    double *Tz = Tpart + (int64_t)z * n_mo * n_mo;
    const bool vec_ok = (n_mo & 1) == 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int p = p0 + fm.row(i);
      if (p < n_mo) {
#pragma unroll
        for (int j = 0; j < NJM; ++j) {
          const int qc = fm.out_col(j);
          const int q = q0 + qc;
          if (qc < cols_valid) {
            double *dst = Tz + (int64_t)p * n_mo + q;
            if (vec_ok) {
              double2 t = *reinterpret_cast<double2 *>(dst);
              t.x += acc[i][j][0];
              t.y += acc[i][j][1];
              *reinterpret_cast<double2 *>(dst) = t;
            } else {
              dst[0] += acc[i][j][0];
              if (qc + 1 < cols_valid) dst[1] += acc[i][j][1];
            }
          }
        }
      }
    }
  }
}

}  // namespace qsgw
