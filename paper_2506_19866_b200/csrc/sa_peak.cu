// Integer issue-rate microbenchmark: the measured denominator of the ALU roofline
// (SURVEY.md §8(d) "Which roofline").  Independent dependency chains of one
// instruction kind, 8 chains per thread, 32 warps per SM, timed with CUDA events; the SM clock
// is read through clock64 / globaltimer inside the same launch.
#include <cuda_runtime.h>

#include <string>

#include "../../include/ternary_sa.h"

namespace {

constexpr int kChains = 8;
constexpr int kRepeat = 16;   // unrolled instructions per chain per loop trip

template <int OP>
__global__ void __launch_bounds__(256) peak_kernel(uint32_t* sink, int trips, unsigned long long* clk) {
  uint32_t a[kChains];
  const uint32_t b = threadIdx.x * 2654435761u + 12345u, c = blockIdx.x * 40503u + 977u;
#pragma unroll
  for (int i = 0; i < kChains; ++i) a[i] = threadIdx.x + i * 7919u;
  unsigned long long c0 = 0, t0 = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    c0 = clock64();
  }
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int r = 0; r < kRepeat; ++r) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) {
        if (OP == 0) asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(b));
        else if (OP == 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b), "r"(c));
        else if (OP == 2) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
        else if (i & 1) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
        else asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(b));
      }
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    unsigned long long c1 = clock64(), t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
    clk[0] = c1 - c0;
    clk[1] = t1 - t0;
  }
  uint32_t x = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) x ^= a[i];
  if (x == 0xDEADBEEFu) sink[0] = x;   // keeps the chains alive
}

template <int OP>
cudaError_t run_one(int sms, int trips, uint32_t* sink, unsigned long long* clk, double* rate, double* hz) {
  const int grid = sms * 4, block = 256;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  peak_kernel<OP><<<grid, block>>>(sink, trips / 8, clk);   // warm-up
  cudaEventRecord(e0);
  peak_kernel<OP><<<grid, block>>>(sink, trips, clk);
  cudaEventRecord(e1);
  cudaError_t err = cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (err != cudaSuccess) return err;
  unsigned long long h[2] = {0, 0};
  err = cudaMemcpy(h, clk, sizeof(h), cudaMemcpyDeviceToHost);
  if (err != cudaSuccess) return err;
  const double warp_instr = (double)grid * (block / 32) * (double)trips * kRepeat * kChains;
  *rate = warp_instr / (ms * 1e-3);
  if (hz && h[1] > 0) *hz = (double)h[0] / ((double)h[1] * 1e-9);
  return cudaGetLastError();
}

}  // namespace

extern "C" int sa_int32_peak(double out[6]) {
  if (!out) return SA_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return SA_ECUDA;
  uint32_t* sink = nullptr;
  unsigned long long* clk = nullptr;
  if (cudaMalloc(&sink, 16) != cudaSuccess || cudaMalloc(&clk, 16) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(sink);                                      // NULL if the first allocation is the one that failed
    cudaFree(clk);
    return SA_ENOMEM;
  }
  const int trips = 4096;
  double hz = 0.0;
  cudaError_t e = run_one<0>(sms, trips, sink, clk, &out[0], nullptr);
  if (e == cudaSuccess) e = run_one<1>(sms, trips, sink, clk, &out[1], nullptr);
  if (e == cudaSuccess) e = run_one<2>(sms, trips, sink, clk, &out[2], nullptr);
  if (e == cudaSuccess) e = run_one<3>(sms, trips, sink, clk, &out[3], &hz);
  out[4] = (double)sms;
  out[5] = hz;
  cudaFree(sink);
  cudaFree(clk);
  return e == cudaSuccess ? SA_OK : SA_ECUDA;
}

// Legacy tensor-path issue rates: the measured denominator of the dense kernel's second ceiling
// (DESIGN.md §7).  Independent accumulator tiles, 4 per warp, 16 warps per SM, event-timed.
namespace {

template <bool SPARSE>
__global__ void __launch_bounds__(512) imma_peak_kernel(int* sink, int trips, unsigned long long* clk) {
  const unsigned a[4] = {threadIdx.x, 1u, 2u, 3u}, b[4] = {threadIdx.x * 3u, 7u, 9u, 11u};
  const unsigned e = 0x44444444u;
  int c[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) c[i][j] = i + j;
  unsigned long long c0 = 0, t0 = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    c0 = clock64();
  }
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        if (SPARSE)
          asm volatile("mma.sp::ordered_metadata.sync.aligned.m16n8k64.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9,%10,%11}, {%0,%1,%2,%3}, %12, 0x0;"
                       : "+r"(c[i][0]), "+r"(c[i][1]), "+r"(c[i][2]), "+r"(c[i][3])
                       : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]), "r"(e));
        else
          asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                       : "+r"(c[i][0]), "+r"(c[i][1]), "+r"(c[i][2]), "+r"(c[i][3])
                       : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
      }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    unsigned long long c1 = clock64(), t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
    clk[0] = c1 - c0;
    clk[1] = t1 - t0;
  }
  int x = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) x ^= c[i][j];
  if (x == 0x7EADBEEF) sink[0] = x;
}

template <bool SPARSE>
cudaError_t run_imma(int sms, int trips, int* sink, unsigned long long* clk, double* rate, double* hz) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  imma_peak_kernel<SPARSE><<<sms, 512>>>(sink, trips / 8, clk);   // warm-up
  cudaEventRecord(e0);
  imma_peak_kernel<SPARSE><<<sms, 512>>>(sink, trips, clk);
  cudaEventRecord(e1);
  cudaError_t err = cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (err != cudaSuccess) return err;
  unsigned long long h[2] = {0, 0};
  err = cudaMemcpy(h, clk, sizeof(h), cudaMemcpyDeviceToHost);
  if (err != cudaSuccess) return err;
  *rate = (double)sms * 16.0 * (double)trips * 16.0 / (ms * 1e-3);
  if (hz && h[1] > 0) *hz = (double)h[0] / ((double)h[1] * 1e-9);
  return cudaGetLastError();
}

}  // namespace

extern "C" int sa_imma_peak(double out[4]) {
  if (!out) return SA_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return SA_ECUDA;
  int* sink = nullptr;
  unsigned long long* clk = nullptr;
  if (cudaMalloc(&sink, 16) != cudaSuccess || cudaMalloc(&clk, 16) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(sink);                                      // NULL if the first allocation is the one that failed
    cudaFree(clk);
    return SA_ENOMEM;
  }
  double hz = 0.0;
  cudaError_t e = run_imma<false>(sms, 8192, sink, clk, &out[0], nullptr);
  if (e == cudaSuccess) e = run_imma<true>(sms, 8192, sink, clk, &out[1], &hz);
  out[2] = (double)sms;
  out[3] = hz;
  cudaFree(sink);
  cudaFree(clk);
  return e == cudaSuccess ? SA_OK : SA_ECUDA;
}
