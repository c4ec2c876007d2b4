// Microbenchmark (B200, sm_100a): what an IMMA.SP of the legacy tensor path costs the other instructions of its SM
// sub-partition.  Four warps per sub-partition; per loop trip 14 IMMA.SP.16864 (four accumulator chains, a different A
// fragment and selector word each, as in sa_dense_kernel.cu) and N integer operations of one kind in eight
// independent chains.  Prints clocks per warp-trip per sub-partition with and without the IMMAs.
// Results and reading: profiles/r2c_microbench.md, DESIGN.md 7.  Not part of libternary_sa.so.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O2 -o imma_dispatch imma_dispatch.cu && ./imma_dispatch
#include <cuda_runtime.h>
#include <cstdio>
template <int KIND, int NI, int NOPS>
__global__ void __launch_bounds__(512) k(int* sink, int trips, long long* clk, const unsigned* src) {
  unsigned a[4], m = 0x44444444u, b[4], x[8], A[14][4], B2[8];
  __shared__ unsigned sm[512];
  sm[threadIdx.x] = threadIdx.x;
  __syncthreads();
  const unsigned saddr = (unsigned)__cvta_generic_to_shared(&sm[threadIdx.x]);
#pragma unroll
  for (int j = 0; j < 4; ++j) { a[j] = src[j * 32 + (threadIdx.x & 31)]; b[j] = src[(j + 4) * 32 + (threadIdx.x & 31)]; }
#pragma unroll
  for (int i = 0; i < 14; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) A[i][j] = src[((i * 4 + j) % 60) * 32 + (threadIdx.x & 31)];
#pragma unroll
  for (int j = 0; j < 8; ++j) B2[j] = src[(j + 20) * 32 + (threadIdx.x & 31)];
#pragma unroll
  for (int j = 0; j < 8; ++j) x[j] = src[(j + 8) * 32 + (threadIdx.x & 31)];
  int c[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i) c[i][0] = c[i][1] = c[i][2] = c[i][3] = 0;
  long long c0; asm volatile("mov.u64 %0, %%clock64;" : "=l"(c0) :: "memory");
  for (int t = 0; t < trips; ++t) {
    constexpr int PER = NI > 0 ? (NOPS + NI - 1) / NI : NOPS;
    int done = 0;
#pragma unroll
    for (int i = 0; i < (NI > 0 ? NI : 1); ++i) {
      if (NI > 0) {
        const int ci = i % 4;
        asm volatile("mma.sp::ordered_metadata.sync.aligned.m16n8k64.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9,%10,%11}, {%0,%1,%2,%3}, %12, 0x0;" : "+r"(c[ci][0]), "+r"(c[ci][1]), "+r"(c[ci][2]), "+r"(c[ci][3]) : "r"(A[i % 14][0]), "r"(A[i % 14][1]), "r"(A[i % 14][2]), "r"(A[i % 14][3]), "r"(B2[(i & 1) * 4]), "r"(B2[(i & 1) * 4 + 1]), "r"(B2[(i & 1) * 4 + 2]), "r"(B2[(i & 1) * 4 + 3]), "r"(m));
      }
#pragma unroll
      for (int o = 0; o < PER; ++o) {
        if (done >= NOPS) break;
        unsigned& v = x[done % 8];
        const int kind = KIND == 8 ? (done & 1 ? 2 : 1) : KIND == 9 ? (done & 1 ? 2 : 0) : KIND;
        if (kind == 0) asm volatile("add.u32 %0, %0, %1;" : "+r"(v) : "r"(a[0]));
        if (kind == 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(v) : "r"(a[0]), "r"(a[1]));
        if (kind == 2) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(v) : "r"(a[0]), "r"(a[1]));
        if (kind == 3) asm volatile("shf.r.clamp.b32 %0, %0, %1, 6;" : "+r"(v) : "r"(a[0]));
        if (kind == 10) asm volatile("{ .reg .u32 t; shl.b32 t, %0, 16; add.u32 %0, t, %1; }" : "+r"(v) : "r"(a[0]));
        if (kind == 11) asm volatile("{ .reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2; }" : "+r"(v) : "r"(a[0]), "r"(a[1]));
        if (kind == 12) asm volatile("and.b32 %0, %0, 0x80808080;" : "+r"(v));
        if (kind == 13) asm volatile("vadd.u32.u32.u32 %0, %0, %1, %2;" : "+r"(v) : "r"(a[0]), "r"(a[1]));
        if (kind == 4) asm volatile("prmt.b32 %0, %0, %1, 0x5410;" : "+r"(v) : "r"(a[0]));
        if (kind == 5) asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %0;" : "+r"(v));
        if (kind == 6) asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
        if (kind == 7) asm volatile("mad.hi.u32 %0, %0, 0x80000000, %1;" : "+r"(v) : "r"(a[1]));
        ++done;
      }
    }
  }
  long long c1; asm volatile("mov.u64 %0, %%clock64;" : "=l"(c1) :: "memory");
  if (threadIdx.x == 0 && blockIdx.x == 0) clk[0] = c1 - c0;
  unsigned y = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) y ^= x[j];
#pragma unroll
  for (int i = 0; i < 4; ++i) y ^= c[i][0] ^ c[i][1] ^ c[i][2] ^ c[i][3];
  if (y == 0x01020301u) sink[0] = y;
}
template <int KIND, int NI, int NOPS>
double run(int sms, int* sink, long long* clk, const unsigned* src) {
  const int trips = 2048, warps = 16;
  k<KIND, NI, NOPS><<<sms, warps * 32>>>(sink, trips / 8, clk, src);
  k<KIND, NI, NOPS><<<sms, warps * 32>>>(sink, trips, clk, src);
  cudaDeviceSynchronize();
  long long h; cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
  return (double)h / trips / 4.0;   // per warp-iteration per SMSP
}
template <int KIND> void kind(const char* name, int sms, int* sink, long long* clk, const unsigned* src) {
  const double n0 = run<KIND, 0, 56>(sms, sink, clk, src), n1 = run<KIND, 0, 112>(sms, sink, clk, src);
  const double i0 = run<KIND, 14, 56>(sms, sink, clk, src), i1 = run<KIND, 14, 112>(sms, sink, clk, src);
  printf("%-14s alone: 56 ops %.1f, 112 ops %.1f clk (%.2f per op) | with 14 IMMA.SP: %.1f, %.1f clk (%.2f per op; IMMA adds %.1f = %.2f each)  %s\n", name, n0, n1,
         (n1 - n0) / 56.0, i0, i1, (i1 - i0) / 56.0, i1 - n1, (i1 - n1) / 14.0, cudaGetErrorString(cudaGetLastError()));
}
int main() {
  int sms; cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
  int* sink; long long* clk; unsigned* src; cudaMalloc(&sink, 16); cudaMalloc(&clk, 8); cudaMalloc(&src, 64 * 32 * 4);
  unsigned h[64 * 32]; for (int i = 0; i < 64 * 32; ++i) h[i] = (i * 2654435761u) & 0x01010101u;
  cudaMemcpy(src, h, sizeof(h), cudaMemcpyHostToDevice);
  printf("IMMA.SP only: %.1f clk per 14\n", run<0, 14, 0>(sms, sink, clk, src));
  kind<0>("IADD", sms, sink, clk, src);
  kind<1>("LOP3", sms, sink, clk, src);
  kind<2>("IMAD", sms, sink, clk, src);
  kind<3>("SHF", sms, sink, clk, src);
  kind<4>("PRMT", sms, sink, clk, src);
  kind<5>("MOVM", sms, sink, clk, src);
  kind<7>("IMAD.HI", sms, sink, clk, src);
  kind<10>("SHL+ADD", sms, sink, clk, src);
  kind<11>("ADD+ADD", sms, sink, clk, src);
  kind<8>("LOP3+IMAD", sms, sink, clk, src);
  kind<9>("IADD+IMAD", sms, sink, clk, src);
  return 0;
}
