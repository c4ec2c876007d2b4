// Microbenchmark (B200, sm_100a): issue rate of the smaller legacy integer MMA shapes (sparse m16n8k32, dense m16n8k16)
// beside m16n8k64 sparse: the slot is per instruction, not per product, so the largest shape is the cheapest.
// Results: profiles/r2c_microbench.md.  Not part of libternary_sa.so.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O2 -o imma_shapes imma_shapes.cu && ./imma_shapes
#include <cuda_runtime.h>
#include <cstdio>
template <int V>
__global__ void __launch_bounds__(512) k(int* sink, int trips, long long* clk, const unsigned* src) {
  unsigned a[14][4], b[8], m[14];
  for (int i = 0; i < 14; ++i) { for (int j = 0; j < 4; ++j) a[i][j] = src[(i * 4 + j) * 32 + (threadIdx.x & 31)]; m[i] = 0x44444444u; }
  for (int j = 0; j < 8; ++j) b[j] = src[j * 32 + (threadIdx.x & 31)];
  int c[4][4];
  for (int i = 0; i < 4; ++i) c[i][0] = c[i][1] = c[i][2] = c[i][3] = 0;
  long long c0; asm volatile("mov.u64 %0, %%clock64;" : "=l"(c0) :: "memory");
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int i = 0; i < 14; ++i) {
      const int ci = i % 4, bi = (i & 1) * 4;
      if (V == 0) asm volatile("mma.sp::ordered_metadata.sync.aligned.m16n8k64.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9,%10,%11}, {%0,%1,%2,%3}, %12, 0x0;" : "+r"(c[ci][0]), "+r"(c[ci][1]), "+r"(c[ci][2]), "+r"(c[ci][3]) : "r"(a[i][0]), "r"(a[i][1]), "r"(a[i][2]), "r"(a[i][3]), "r"(b[bi]), "r"(b[bi + 1]), "r"(b[bi + 2]), "r"(b[bi + 3]), "r"(m[i]));
      if (V == 1) asm volatile("mma.sp::ordered_metadata.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5}, {%6,%7}, {%0,%1,%2,%3}, %8, 0x0;" : "+r"(c[ci][0]), "+r"(c[ci][1]), "+r"(c[ci][2]), "+r"(c[ci][3]) : "r"(a[i][0]), "r"(a[i][1]), "r"(b[bi]), "r"(b[bi + 1]), "r"(m[i]));
      if (V == 2) asm volatile("mma.sync.aligned.m16n8k16.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};" : "+r"(c[ci][0]), "+r"(c[ci][1]), "+r"(c[ci][2]), "+r"(c[ci][3]) : "r"(a[i][0]), "r"(a[i][1]), "r"(b[bi]));
    }
  }
  long long c1; asm volatile("mov.u64 %0, %%clock64;" : "=l"(c1) :: "memory");
  if (threadIdx.x == 0 && blockIdx.x == 0) clk[0] = c1 - c0;
  int x = 0; for (int i = 0; i < 4; ++i) x ^= c[i][0] ^ c[i][1] ^ c[i][2] ^ c[i][3];
  if (x == 0x01020301) sink[0] = x;
}
template <int V> void run(const char* n, int sms, int* sink, long long* clk, unsigned* src) {
  k<V><<<sms, 512>>>(sink, 256, clk, src); k<V><<<sms, 512>>>(sink, 2048, clk, src);
  cudaDeviceSynchronize(); long long h; cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
  printf("%-28s %.2f clk per MMA per SMSP (%s)\n", n, (double)h / (2048.0 * 14 * 4), cudaGetErrorString(cudaGetLastError()));
}
int main() {
  int sms; cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
  int* sink; long long* clk; unsigned* src; cudaMalloc(&sink, 16); cudaMalloc(&clk, 8); cudaMalloc(&src, 64 * 32 * 4);
  unsigned h[64 * 32]; for (int i = 0; i < 64 * 32; ++i) h[i] = (i * 2654435761u) & 0x01010101u;
  cudaMemcpy(src, h, sizeof(h), cudaMemcpyHostToDevice);
  run<0>("IMMA.SP m16n8k64", sms, sink, clk, src);
  run<1>("IMMA.SP m16n8k32", sms, sink, clk, src);
  run<2>("IMMA m16n8k16", sms, sink, clk, src);
  return 0;
}
