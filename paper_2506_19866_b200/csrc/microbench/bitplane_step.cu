// Microbenchmark (B200, sm_100a): latency of one simulated time step in a bit-plane formulation for networks of at
// most 32 nodes (one warp per condition, one lane per node; the states of t-1 as two ballots s >= 1, s == 2; a node's
// sum = popc(B0 & P) + popc(B1 & P) - popc(B0 & M) - popc(B1 & M) with its positive / negative in-edge masks P, M;
// every third step scored with one more ballot).  Measured 72 clocks per step against about 120 of the dense kernel's
// HPG-shaped step: DESIGN.md 11 weighs that against a second kernel family.  Not part of libternary_sa.so.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O2 -o bitplane_step bitplane_step.cu && ./bitplane_step
#include <cuda_runtime.h>
#include <cstdio>
__global__ void k(int* sink, int trips, long long* clk, unsigned seed) {
  const unsigned lane = threadIdx.x & 31;
  unsigned P = seed * (lane + 3) * 2654435761u, M = ~P & (seed * 7919u * (lane + 1));
  int lo = -1, hi = 1;
  int s = lane % 3;
  int mis = 0;
  long long c0; asm volatile("mov.u64 %0, %%clock64;" : "=l"(c0) :: "memory");
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int r = 0; r < 24; ++r) {
      const unsigned B0 = __ballot_sync(0xffffffffu, s >= 1), B1 = __ballot_sync(0xffffffffu, s == 2);
      const int sum = __popc(B0 & P) + __popc(B1 & P) - __popc(B0 & M) - __popc(B1 & M);
      s = (sum >= lo) + (sum > hi);
      if ((r % 3) == 2) mis += __popc(__ballot_sync(0xffffffffu, s != (int)((lane + r) % 3)));
    }
  }
  long long c1; asm volatile("mov.u64 %0, %%clock64;" : "=l"(c1) :: "memory");
  if (threadIdx.x == 0) clk[0] = c1 - c0;
  if (s + mis == 0x7fffffff) sink[0] = 1;
}
int main() {
  int* sink; long long* clk; cudaMalloc(&sink, 16); cudaMalloc(&clk, 8);
  k<<<1, 32>>>(sink, 16, clk, 5u); k<<<1, 32>>>(sink, 512, clk, 5u);
  cudaDeviceSynchronize();
  long long h; cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
  printf("bit-plane time step: %.1f clk (%s)\n", (double)h / (512.0 * 24), cudaGetErrorString(cudaGetLastError()));
  return 0;
}
