// Microbenchmark (B200, sm_100a): dependent-issue latency of one warp: IMMA chained through C or through B, the
// integer operations of the dense kernel's time step, and chains that alternate between the tensor pipe and the ALU
// (the HPG-shaped time step: shift, two IMMAs, pack, two adds, two logic operations, LEA, PRMT, MOVM).
// Results: profiles/r2c_microbench.md.  Not part of libternary_sa.so.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O2 -o imma_latency imma_latency.cu && ./imma_latency
#include <cuda_runtime.h>
#include <cstdio>
template <int MODE>
__global__ void k(int* sink, int trips, long long* clk) {
  unsigned a[4] = {threadIdx.x, 1u, 2u, 3u}, b[4] = {threadIdx.x * 3u, 7u, 9u, 11u};
  const unsigned e = 0x44444444u;
  int c[4] = {0, 0, 0, 0};
  long long c0 = clock64();
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      if (MODE == 0)  // dependent through C, sparse
        asm volatile("mma.sp::ordered_metadata.sync.aligned.m16n8k64.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9,%10,%11}, {%0,%1,%2,%3}, %12, 0x0;" : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]), "r"(e));
      if (MODE == 1)  // dependent through C, dense
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};" : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
      if (MODE == 2) {  // dependent through B, dense, C = 0
        int d[4];
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};" : "=r"(d[0]), "=r"(d[1]), "=r"(d[2]), "=r"(d[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(0));
        b[0] = d[0]; b[1] = d[1];
      }
      if (MODE == 3) {  // dependent through B, sparse
        int d[4];
        asm volatile("mma.sp::ordered_metadata.sync.aligned.m16n8k64.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9,%10,%11}, {%13,%13,%13,%13}, %12, 0x0;" : "=r"(d[0]), "=r"(d[1]), "=r"(d[2]), "=r"(d[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]), "r"(e), "r"(0));
        b[0] = d[0]; b[1] = d[1]; b[2] = d[2]; b[3] = d[3];
      }
      if (MODE == 4) {  // ALU dependent chain reference: IMAD
        asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(c[0]) : "r"(a[0]), "r"(b[0]));
      }
      if (MODE == 5) {  // LOP3 chain
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(c[0]) : "r"(a[0]), "r"(b[0]));
      }
      if (MODE == 6) {  // IADD chain
        asm volatile("add.u32 %0, %0, %1;" : "+r"(c[0]) : "r"(a[0]));
      }
      if (MODE == 7) {  // PRMT chain
        asm volatile("prmt.b32 %0, %0, %1, 0x5410;" : "+r"(c[0]) : "r"(a[0]));
      }
      if (MODE == 8) {  // shift chain
        asm volatile("shr.u32 %0, %0, 6;" : "+r"(c[0]));
        asm volatile("add.u32 %0, %0, %1;" : "+r"(c[0]) : "r"(a[0]));
      }
    }
  }
  long long c1 = clock64();
  if (threadIdx.x == 0) clk[0] = c1 - c0;
  if ((c[0] ^ c[1] ^ c[2] ^ c[3] ^ b[0] ^ b[1] ^ b[2] ^ b[3]) == 0x7EADBEEF) sink[0] = 1;
}
template <int MODE> void run(const char* name, int* sink, long long* clk) {
  k<MODE><<<1, 32>>>(sink, 64, clk); k<MODE><<<1, 32>>>(sink, 1024, clk);
  cudaDeviceSynchronize();
  long long h; cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
  printf("%-34s %.1f clk per op (%s)\n", name, (double)h / (1024.0 * 16), cudaGetErrorString(cudaGetLastError()));
}
template <int MODE>
__global__ void kmix(int* sink, int trips, long long* clk, unsigned seed) {
  unsigned a[4] = {threadIdx.x & 1u, 1u, 0u, 1u}, a2[4] = {1u, threadIdx.x & 1u, 1u, 0u}, b[2] = {seed, seed * 3u};
  unsigned ta = 0x7f7f7f7fu, tb = 0x7e7e7e7eu;
  int c[4];
  long long c0 = clock64();
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      if (MODE == 0) {        // IMMA -> IADD -> IMMA
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};" : "=r"(c[0]), "=r"(c[1]), "=r"(c[2]), "=r"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(0));
        asm volatile("add.u32 %0, %1, %2;" : "=r"(b[0]) : "r"(c[0]), "r"(ta));
        asm volatile("add.u32 %0, %1, %2;" : "=r"(b[1]) : "r"(c[1]), "r"(tb));
      } else if (MODE == 1) { // IMMA -> IMMA (C) -> IADD -> IMMA
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};" : "=r"(c[0]), "=r"(c[1]), "=r"(c[2]), "=r"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(0));
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};" : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3]) : "r"(a2[0]), "r"(a2[1]), "r"(a2[2]), "r"(a2[3]), "r"(b[0]), "r"(b[1]));
        asm volatile("add.u32 %0, %1, %2;" : "=r"(b[0]) : "r"(c[0]), "r"(ta));
        asm volatile("add.u32 %0, %1, %2;" : "=r"(b[1]) : "r"(c[1]), "r"(tb));
      } else if (MODE == 2) { // the HPG time step: shift, 2 IMMA, pack, 2 add, 2 lop, lea, prmt, movm
        unsigned bl0 = b[0] >> 6, bl1 = b[1] >> 6;
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};" : "=r"(c[0]), "=r"(c[1]), "=r"(c[2]), "=r"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(bl0), "r"(bl1), "r"(0));
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};" : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3]) : "r"(a2[0]), "r"(a2[1]), "r"(a2[2]), "r"(a2[3]), "r"(b[0]), "r"(b[1]));
        unsigned ns[2];
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
          const unsigned pk = (unsigned)c[cc] + ((unsigned)c[2 + cc] << 16);
          const unsigned x = pk + ta, y = pk + tb;
          unsigned rr; asm("mad.hi.u32 %0, %1, 0x80000000, %2;" : "=r"(rr) : "r"((x ^ y) & 0x80808080u), "r"(y & 0x80808080u));
          ns[cc] = rr;
        }
        unsigned p0 = __byte_perm(ns[0], ns[1], 0x5410), p1 = __byte_perm(ns[0], ns[1], 0x7632);
        asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(b[0]) : "r"(p0));
        asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(b[1]) : "r"(p1));
      } else if (MODE == 3) { // same without the IMMAs
        unsigned bl0 = b[0] >> 6, bl1 = b[1] >> 6;
        c[0] = bl0 + a[0]; c[1] = bl1 + b[0]; c[2] = b[1] + a[1]; c[3] = bl0 ^ b[1];
        unsigned ns[2];
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
          const unsigned pk = (unsigned)c[cc] + ((unsigned)c[2 + cc] << 16);
          const unsigned x = pk + ta, y = pk + tb;
          unsigned rr; asm("mad.hi.u32 %0, %1, 0x80000000, %2;" : "=r"(rr) : "r"((x ^ y) & 0x80808080u), "r"(y & 0x80808080u));
          ns[cc] = rr;
        }
        unsigned p0 = __byte_perm(ns[0], ns[1], 0x5410), p1 = __byte_perm(ns[0], ns[1], 0x7632);
        asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(b[0]) : "r"(p0));
        asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(b[1]) : "r"(p1));
      }
    }
  }
  long long c1 = clock64();
  if (threadIdx.x == 0) clk[0] = c1 - c0;
  if ((c[0] ^ c[1] ^ c[2] ^ c[3] ^ b[0] ^ b[1]) == 0x7EADBEEF) sink[0] = 1;
}
template <int MODE> void run_mix(const char* name, int* sink, long long* clk) {
  kmix<MODE><<<1, 32>>>(sink, 64, clk, 5u); kmix<MODE><<<1, 32>>>(sink, 1024, clk, 5u);
  cudaDeviceSynchronize();
  long long h; cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
  printf("%-44s %.1f clk per iteration (%s)\n", name, (double)h / (1024.0 * 8), cudaGetErrorString(cudaGetLastError()));
}
int main() {
  int* sink; long long* clk; cudaMalloc(&sink, 16); cudaMalloc(&clk, 8);
  run<0>("IMMA.SP.16864 dep via C", sink, clk);
  run<1>("IMMA.16832 dep via C", sink, clk);
  run<2>("IMMA.16832 dep via B", sink, clk);
  run<3>("IMMA.SP.16864 dep via B", sink, clk);
  run<4>("IMAD chain", sink, clk);
  run<5>("LOP3 chain", sink, clk);
  run<6>("IADD chain", sink, clk);
  run<7>("PRMT chain", sink, clk);
  run<8>("SHF+IADD chain (per pair)", sink, clk);
  run_mix<0>("IMMA -> IADD -> IMMA", sink, clk);
  run_mix<1>("IMMA -> IMMA(C) -> IADD -> IMMA", sink, clk);
  run_mix<2>("HPG time step (2 IMMA + pack + movm)", sink, clk);
  run_mix<3>("HPG time step without the IMMAs", sink, clk);
  return 0;
}
