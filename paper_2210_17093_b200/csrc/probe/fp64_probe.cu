// fp64_probe.cu -- measures the FP64 issue rates the roofline of this library is quoted against.
// MEASUREMENT TOOL, not part of the product: built into its own libqsgw_fp64_probe.so (paper_2210_17093_b200/build.py),
// loaded only by bench.py; libqsgw_sigma.so neither contains nor calls it, and this file includes no product header.
//
// MEASURED_PEAKS.json carries no FP64 figure, so the denominator of the "fraction of FP64 tensor peak" is
// derived (SMs x 64 FMA/clk x 2 x max SM clock) and CHECKED on the box by these register-resident loops:
//   mode 0  DMMA.8x8x4 only, 32 independent accumulator fragments per warp (the 64x32 warp tile of the GEMMs)
//   mode 1  DFMA only, 32 independent chains per thread
//   mode 2  32 DMMA + `mix` DFMA per iteration: tells whether DMMA and DFMA share one pipe (time adds) or not
//   mode 3  DMMA fed by LDS.64 fragment loads from a padded shared tile (the inner loop of the GEMMs, no global traffic)
// One CTA of 256 threads per SM x `ctas_per_sm`; flops counted: 512 per DMMA per warp, 2 per DFMA per thread.
#include <cuda_runtime.h>
#include <stdint.h>

namespace qsgw_probe {

constexpr int kBK = 16;          // k depth and padded row length of the shared tile in mode 3 (the GEMM kernels' layout)
constexpr int kLdT = 128 + 4;

__device__ __forceinline__ void dmma_m8n8k4(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(c[0]), "+d"(c[1])
      : "d"(a), "d"(b));
}

template <int MODE>
__global__ void __launch_bounds__(256) fp64_probe_kernel(int iters, int mix, double seed, double *sink) {
  __shared__ double tile[2][kBK * kLdT];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double acc[8][4][2];
  double a[8], b[4], f[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    a[i] = seed * (i + 1 + lane);
    f[i] = seed * (i + 3);
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) b[j] = seed * (j + 2);
  if (MODE == 3) {
    for (int i = threadIdx.x; i < 2 * kBK * kLdT; i += blockDim.x) (&tile[0][0])[i] = seed * (i & 255);
    __syncthreads();
  }
  const int wm = (warp & 1) * 64, wn = (warp >> 1) * 32;
  for (int it = 0; it < iters; ++it) {
    if (MODE == 0 || MODE == 2) {
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma_m8n8k4(acc[i][j], a[i], b[j]);
    }
    if (MODE == 1) {
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          acc[i][j][0] = fma(acc[i][j][0], a[i], b[j]);
          acc[i][j][1] = fma(acc[i][j][1], a[i], b[j]);
        }
    }
    if (MODE == 2) {
      for (int r = 0; r < mix; r += 8) {   // mix is a multiple of 8
#pragma unroll
        for (int i = 0; i < 8; ++i) f[i] = fma(f[i], a[i], b[i & 3]);
      }
    }
    if (MODE == 3) {
      const double *as = tile[0] + wm + (lane >> 2), *bs = tile[1] + wn + (lane >> 2);
#pragma unroll
      for (int kk = 0; kk < kBK / 4; ++kk) {
        const int k = kk * 4 + (lane & 3);
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
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    s += f[i];
#pragma unroll
    for (int j = 0; j < 4; ++j) s += acc[i][j][0] + acc[i][j][1];
  }
  if (s == 12345.678) sink[0] = s;   // never true for the seeds used; keeps the loops alive
}

}  // namespace qsgw_probe

// Returns 0, or -1 bad argument, -2 allocation failure, -3 CUDA failure.  Synchronises the stream.
extern "C" int qsgw_fp64_probe(int mode, int iters, int mix, int ctas_per_sm, void *cuda_stream, double *tflops,
                               double *ms_out) {
  using namespace qsgw_probe;
  if (mode < 0 || mode > 3 || iters < 1 || mix < 0 || (mix & 7) || ctas_per_sm < 1 || !tflops) return -1;
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    cudaGetLastError();
    return -3;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double *sink = nullptr;
  if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return -2;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int grid = prop.multiProcessorCount * ctas_per_sm;
  auto launch = [&](int n) {
    switch (mode) {
      case 0: fp64_probe_kernel<0><<<grid, 256, 0, st>>>(n, mix, 1e-300, sink); break;
      case 1: fp64_probe_kernel<1><<<grid, 256, 0, st>>>(n, mix, 1e-300, sink); break;
      case 2: fp64_probe_kernel<2><<<grid, 256, 0, st>>>(n, mix, 1e-300, sink); break;
      default: fp64_probe_kernel<3><<<grid, 256, 0, st>>>(n, mix, 1e-300, sink); break;
    }
  };
  launch(iters / 8 + 1);   // warm-up
  cudaEventRecord(e0, st);
  launch(iters);
  cudaEventRecord(e1, st);
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = 0.f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (e != cudaSuccess) return -3;
  const double warps = (double)grid * 8;
  double flops = 0.0;
  if (mode == 0) flops = warps * iters * 32.0 * 512.0;
  if (mode == 1) flops = warps * iters * 32.0 * 64.0 * 2.0;
  if (mode == 2) flops = warps * iters * (32.0 * 512.0 + 32.0 * 2.0 * mix);
  if (mode == 3) flops = warps * iters * 4.0 * 32.0 * 512.0;
  *tflops = flops / (ms * 1e-3) / 1e12;
  if (ms_out) *ms_out = ms;
  return 0;
}
