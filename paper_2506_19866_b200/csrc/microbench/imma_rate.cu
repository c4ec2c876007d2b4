// Microbenchmark (B200, sm_100a): issue rate of IMMA.16832 / IMMA.SP.16864 when the A fragment, the selector word or
// the number of accumulator chains changes, for 1, 2 and 4 warps per SM sub-partition.
// Results: profiles/r2c_microbench.md.  Not part of libternary_sa.so.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O2 -o imma_rate imma_rate.cu && ./imma_rate
#include <cuda_runtime.h>
#include <cstdio>
template <int SPARSE, int VARA, int NACC>
__global__ void __launch_bounds__(512) k(int* sink, int trips, long long* clk, const unsigned* src) {
  unsigned a[14][4], m[14], b[8];
#pragma unroll
  for (int i = 0; i < 14; ++i) {
#pragma unroll
    for (int j = 0; j < 4; ++j) a[i][j] = src[(i * 4 + j) * 32 + (threadIdx.x & 31)];
    m[i] = 0x44444444u;
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) b[j] = src[j * 32 + (threadIdx.x & 31)] & 0x03030303u;
  int c[NACC][4];
#pragma unroll
  for (int i = 0; i < NACC; ++i) { c[i][0] = c[i][1] = c[i][2] = c[i][3] = 0; }
  long long c0 = clock64();
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int i = 0; i < 14; ++i) {
      const int ai = VARA ? i : 0, bi = (i & 1) * 4, ci = i % NACC;
      if (SPARSE)
        asm volatile("mma.sp::ordered_metadata.sync.aligned.m16n8k64.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9,%10,%11}, {%0,%1,%2,%3}, %12, 0x0;" : "+r"(c[ci][0]), "+r"(c[ci][1]), "+r"(c[ci][2]), "+r"(c[ci][3]) : "r"(a[ai][0]), "r"(a[ai][1]), "r"(a[ai][2]), "r"(a[ai][3]), "r"(b[bi]), "r"(b[bi + 1]), "r"(b[bi + 2]), "r"(b[bi + 3]), "r"(m[ai]));
      else
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};" : "+r"(c[ci][0]), "+r"(c[ci][1]), "+r"(c[ci][2]), "+r"(c[ci][3]) : "r"(a[ai][0]), "r"(a[ai][1]), "r"(a[ai][2]), "r"(a[ai][3]), "r"(b[bi]), "r"(b[bi + 1]));
    }
  }
  long long c1 = clock64();
  if (threadIdx.x == 0 && blockIdx.x == 0) clk[0] = c1 - c0;
  int x = 0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) x ^= c[i][0] ^ c[i][1] ^ c[i][2] ^ c[i][3];
  if (x == 0x7EADBEEF) sink[0] = x;
}
template <int SPARSE, int VARA, int NACC>
void run(const char* name, int sms, int* sink, long long* clk, const unsigned* src) {
  for (int warps : {4, 8, 16}) {
    const int trips = 2048;
    k<SPARSE, VARA, NACC><<<sms, warps * 32>>>(sink, trips / 8, clk, src);
    k<SPARSE, VARA, NACC><<<sms, warps * 32>>>(sink, trips, clk, src);
    cudaDeviceSynchronize();
    long long h; cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
    printf("%-30s acc %d warps/SMSP %d: %.2f clk per IMMA per SMSP  (%s)\n", name, NACC, warps / 4, (double)h / (trips * 14.0 * (warps / 4)), cudaGetErrorString(cudaGetLastError()));
  }
}
int main() {
  int sms; cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
  int* sink; long long* clk; unsigned* src; cudaMalloc(&sink, 16); cudaMalloc(&clk, 8); cudaMalloc(&src, 64 * 32 * 4);
  unsigned h[64 * 32]; for (int i = 0; i < 64 * 32; ++i) h[i] = (i * 2654435761u) & 0x01010101u;
  cudaMemcpy(src, h, sizeof(h), cudaMemcpyHostToDevice);
  run<1, 0, 4>("sparse, constant A", sms, sink, clk, src);
  run<1, 1, 4>("sparse, A changes", sms, sink, clk, src);
  run<1, 1, 2>("sparse, A changes", sms, sink, clk, src);
  run<1, 1, 7>("sparse, A changes", sms, sink, clk, src);
  run<0, 0, 4>("dense, constant A", sms, sink, clk, src);
  run<0, 1, 4>("dense, A changes", sms, sink, clk, src);
  run<0, 1, 1>("dense, A changes", sms, sink, clk, src);
  return 0;
}
