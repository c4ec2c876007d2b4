// Microbenchmark: one chain's synchronous time step on the Blackwell tensor path (tcgen05.mma.kind::i8, accumulator in
// TMEM), to set against the legacy IMMA.SP path the dense kernel uses (DESIGN.md §6.2 / §11).
//
// The step, per chain:  D[128 x N] = A[128 x 128] (s8 weights, one row per node) . B[128 x N] (u8 states, one column
// per condition), four K = 32 instructions issued by one thread; tcgen05.commit -> mbarrier; every thread of the CTA
// (128 = one TMEM lane = one node each) reads its row of D with tcgen05.ld, thresholds it to 0/1/2, stores the N new
// state bytes into the B tile, fence.proxy.async, barrier, next step.  A CTA carries C chains round-robin so that the
// MMA of one chain runs under the epilogue of the others; several CTAs per SM add more.
//
//   umma_step verify  N [a_tmem [split]]          one step, D compared with the host's A . B
//   umma_step ldtm    N ctas_per_sm               tcgen05.ld + wait alone: clocks per 128 x N tile per SM
//   umma_step step    N chains_per_cta ctas_per_sm steps [a_tmem [split]]
//
// a_tmem = 1: A lives in TMEM (32 columns per chain, written once with tcgen05.st) instead of shared memory.
// split = 1: the four K = 32 instructions write four accumulators (independent of one another), summed after tcgen05.ld.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O2 -lineinfo -o umma_step umma_step.cu
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

typedef uint32_t u32;
typedef uint64_t u64;

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA error %s at %s:%d\n", cudaGetErrorString(e_), __FILE__, __LINE__); return 1; } } while (0)

constexpr int M = 128, K = 128;
constexpr int A_BYTES = M * K;                 // 16 KB per chain
constexpr u32 LBO = 128, SBO = 1024;           // core matrix = 8 rows x 16 bytes, K-adjacent ones 128 B apart, 8-row groups 1024 B

// canonical K-major layout without swizzle: element (r, k) of a [rows x 128] byte matrix
__host__ __device__ inline u32 canon(u32 r, u32 k) { return (r >> 3) * SBO + (k >> 4) * LBO + (r & 7) * 16 + (k & 15); }

__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }

__device__ __forceinline__ u64 make_desc(u32 saddr) {
  // start address >> 4 | LBO >> 4 at bit 16 | SBO >> 4 at bit 32 | version 1 at bit 46 | SWIZZLE_NONE
  return (u64)((saddr & 0x3FFFFu) >> 4) | ((u64)(LBO >> 4) << 16) | ((u64)(SBO >> 4) << 32) | (1ull << 46);
}

__device__ __forceinline__ u32 make_idesc(int n) {
  // D = s32 (2 at bit 4), A = signed 8 bit (1 at bit 7), B = unsigned 8 bit (0 at bit 10), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
  return (2u << 4) | (1u << 7) | ((u32)(n >> 3) << 17) | ((u32)(M >> 4) << 24);
}

__device__ __forceinline__ void mma_ss(u32 d_tmem, u64 da, u64 db, u32 idesc, u32 accumulate) {
  asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n}\n"
               :: "r"(d_tmem), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void mma_ts(u32 d_tmem, u32 a_tmem, u64 db, u32 idesc, u32 accumulate) {
  asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p;\n}\n"
               :: "r"(d_tmem), "r"(a_tmem), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void commit(u32 bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" :: "r"(bar) : "memory");
}
__device__ __forceinline__ bool wait_parity(u32 bar, u32 parity, unsigned* err) {
  for (u32 spin = 0; spin < (1u << 24); ++spin) {
    u32 ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) return true;
  }
  atomicExch(err, 1u);                          // never hang the box: give up and say so
  return false;
}
template <int N>
__device__ __forceinline__ void ld_row(u32 taddr, u32 (&v)[N]) {
  if constexpr (N == 8)
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(taddr));
  else
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
                   "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]) : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
}

struct Args {
  const int8_t* A;       // [chains][128][128] row-major (host layout), the same for every CTA
  const uint8_t* B0;     // [chains][N][128]   row-major: state of node k in condition n
  int32_t* D;            // verify: [128][N] of chain 0 after the first step
  unsigned long long* clocks;   // [grid] clocks of the timed loop
  unsigned long long* phase;    // [6] thread 0 of CTA 0: clocks in wait / ld / threshold + store / proxy fence / barrier / issue
  unsigned* err;
  int chains, steps, a_tmem, tmem_cols;
  int split;             // 1: the four K = 32 instructions write four separate accumulators (no dependent accumulation), summed in the epilogue
};

// COLS (TMEM columns per CTA) is a compile-time constant: with a run-time operand the driver assumes all 512 columns
// and keeps one CTA per SM.
template <int N, int COLS>
__global__ void __launch_bounds__(128) step_kernel(Args a) {
  extern __shared__ __align__(1024) unsigned char smem[];
  const int C = a.chains, tid = threadIdx.x, warp = tid >> 5;
  const u32 b_bytes = N * K;
  unsigned char* sA = smem;                                   // [C][16 KB] canonical (unused with a_tmem)
  unsigned char* sB = smem + (a.a_tmem ? 0 : (size_t)C * A_BYTES);   // [C][N x 128] canonical
  u64* bars = (u64*)(sB + (size_t)C * b_bytes);
  u32* tmem_base_slot = (u32*)(bars + C);

  // stage the operands
  if (!a.a_tmem)
    for (int x = tid; x < C * A_BYTES; x += 128) {
      const int c = x / A_BYTES, r = (x % A_BYTES) / K, k = x % K;
      sA[(size_t)c * A_BYTES + canon(r, k)] = (unsigned char)a.A[x];
    }
  for (int x = tid; x < C * (int)b_bytes; x += 128) {
    const int c = x / b_bytes, n = (x % b_bytes) / K, k = x % K;
    sB[(size_t)c * b_bytes + canon(n, k)] = a.B0[x];
  }
  if (tid == 0)
    for (int c = 0; c < C; ++c) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(smem_u32(&bars[c])));
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" :: "r"(smem_u32(tmem_base_slot)), "n"(COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const u32 tbase = *tmem_base_slot;
  const u32 lane_off = (u32)(warp * 32) << 16;                // this warp's 32 TMEM lanes
  const u32 idesc = make_idesc(N);
  const int DW = a.split ? 4 * N : N;                         // accumulator columns per chain
  // columns: chain c has D at c*N, and with a_tmem its A at C*N + c*32 (128 bytes of row m in lane m)
  if (a.a_tmem) {
    for (int c = 0; c < C; ++c) {
      u32 w[32];
      const u32* row = (const u32*)(a.A + (size_t)c * A_BYTES + (size_t)tid * K);
#pragma unroll
      for (int j = 0; j < 32; ++j) w[j] = row[j];
      const u32 ta = tbase + lane_off + (u32)(C * DW + c * 32);
      asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,"
                   "%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};\n"
                   :: "r"(ta), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]), "r"(w[8]), "r"(w[9]),
                      "r"(w[10]), "r"(w[11]), "r"(w[12]), "r"(w[13]), "r"(w[14]), "r"(w[15]), "r"(w[16]), "r"(w[17]), "r"(w[18]), "r"(w[19]),
                      "r"(w[20]), "r"(w[21]), "r"(w[22]), "r"(w[23]), "r"(w[24]), "r"(w[25]), "r"(w[26]), "r"(w[27]), "r"(w[28]), "r"(w[29]),
                      "r"(w[30]), "r"(w[31]) : "memory");
    }
    asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  }

  auto issue = [&](int c) {                                   // thread 0: the four K = 32 instructions of chain c, then commit
    const u32 d = tbase + (u32)(c * DW);
    const u32 sb = smem_u32(sB + (size_t)c * b_bytes), sa = smem_u32(sA + (size_t)c * A_BYTES);
#pragma unroll
    for (int kb = 0; kb < K / 32; ++kb) {
      const u64 db = make_desc(sb + kb * 2 * LBO);
      const u32 dk = a.split ? d + (u32)(kb * N) : d;
      const u32 acc = a.split ? 0u : (u32)(kb > 0);
      if (a.a_tmem) mma_ts(dk, tbase + (u32)(C * DW + c * 32 + kb * 8), db, idesc, acc);
      else mma_ss(dk, make_desc(sa + kb * 2 * LBO), db, idesc, acc);
    }
    commit(smem_u32(&bars[c]));
  };

  if (tid == 0)
    for (int c = 0; c < C; ++c) issue(c);
  const long long t0 = clock64();
  u32 score = 0;
  bool alive = true;
  long long ph[6] = {0, 0, 0, 0, 0, 0}, tp = t0, tq;
#define PHASE(i) do { tq = clock64(); ph[i] += tq - tp; tp = tq; } while (0)
  for (int s = 0; s < a.steps && alive; ++s) {
    for (int c = 0; c < C; ++c) {
      if (!wait_parity(smem_u32(&bars[c]), (u32)(s & 1), a.err)) { alive = false; break; }
      asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
      PHASE(0);
      u32 v[N];
      ld_row<N>(tbase + lane_off + (u32)(c * DW), v);
      if (a.split) {
#pragma unroll
        for (int kb = 1; kb < 4; ++kb) {
          u32 w[N];
          ld_row<N>(tbase + lane_off + (u32)(c * DW + kb * N), w);
#pragma unroll
          for (int n = 0; n < N; ++n) v[n] += w[n];
        }
      }
      PHASE(1);
      if (a.D && s == 0 && c == 0 && blockIdx.x == 0)
        for (int n = 0; n < N; ++n) a.D[tid * N + n] = (int32_t)v[n];
      // threshold to 0 / 1 / 2 (two compares per value), score, write the node's N new state bytes into the B tile
      unsigned char* bt = sB + (size_t)c * b_bytes;
#pragma unroll
      for (int n = 0; n < N; ++n) {
        const int d = (int)v[n];
        const u32 st = (u32)(d > 1) + (u32)(d >= -1);
        score += st;
        bt[canon(n, tid)] = (unsigned char)st;
      }
      PHASE(2);
      asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
      PHASE(3);
      asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
      __syncthreads();
      PHASE(4);
      if (tid == 0 && s + 1 < a.steps) { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); issue(c); }
      PHASE(5);
    }
  }
  const long long t1 = clock64();
  if (tid == 0 && blockIdx.x == 0 && a.phase)
    for (int i = 0; i < 6; ++i) a.phase[i] = (unsigned long long)ph[i];
  if (score == 0xFFFFFFFFu) a.err[0] = 2;                     // keeps `score` live
  if (tid == 0) a.clocks[blockIdx.x] = (unsigned long long)(t1 - t0);
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" :: "r"(tbase), "n"(COLS));
}

template <int N>
__global__ void __launch_bounds__(128) ldtm_kernel(unsigned long long* clocks, unsigned* sink, int iters) {
  __shared__ u32 slot;
  const int warp = threadIdx.x >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" :: "r"(smem_u32(&slot)), "r"(32));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const u32 t = slot + ((u32)(warp * 32) << 16);
  u32 acc = 0;
  const long long t0 = clock64();
  for (int i = 0; i < iters; ++i) {
    u32 v[N];
    ld_row<N>(t, v);
#pragma unroll
    for (int n = 0; n < N; ++n) acc += v[n];
  }
  const long long t1 = clock64();
  if (acc == 0x12345678u) sink[0] = acc;
  if (threadIdx.x == 0) clocks[blockIdx.x] = (unsigned long long)(t1 - t0);
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" :: "r"(slot), "r"(32));
}

static int pow2_cols(int want) { int c = 32; while (c < want) c *= 2; return c; }

template <int N>
static void (*pick_kernel(int cols))(Args) {
  switch (cols) {
    case 32: return step_kernel<N, 32>;
    case 64: return step_kernel<N, 64>;
    case 128: return step_kernel<N, 128>;
    case 256: return step_kernel<N, 256>;
    default: return step_kernel<N, 512>;
  }
}

template <int N>
static int run(const char* mode, int chains, int ctas_per_sm, int steps, int a_tmem, int split) {
  int sms = 0;
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0));
  unsigned *d_err; unsigned long long* d_clk;
  const int grid = sms * ctas_per_sm;
  CK(cudaMalloc(&d_err, 8)); CK(cudaMemset(d_err, 0, 8));
  CK(cudaMalloc(&d_clk, sizeof(unsigned long long) * grid));
  std::vector<unsigned long long> clk(grid);
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  float ms = 0;
  if (!strcmp(mode, "ldtm")) {
    ldtm_kernel<N><<<grid, 128>>>(d_clk, d_err + 1, 100);
    CK(cudaEventRecord(e0));
    ldtm_kernel<N><<<grid, 128>>>(d_clk, d_err + 1, steps);
    CK(cudaEventRecord(e1));
    CK(cudaDeviceSynchronize());
    CK(cudaEventElapsedTime(&ms, e0, e1));
    CK(cudaMemcpy(clk.data(), d_clk, sizeof(unsigned long long) * grid, cudaMemcpyDeviceToHost));
    double mean = 0; for (auto c : clk) mean += (double)c; mean /= grid;
    printf("ldtm N=%d ctas_per_sm=%d: %.1f clocks per tcgen05.ld.32x32b.x%d + wait per CTA; per SM one 128 x %d tile (%d B) every %.1f clocks "
           "= %.1f B/clk/SM (%.3f ms)\n", N, ctas_per_sm, mean / steps, N, N, 128 * N * 4, mean / steps / ctas_per_sm,
           128.0 * N * 4 * ctas_per_sm / (mean / steps), ms);
    return 0;
  }
  std::vector<int8_t> A((size_t)chains * A_BYTES);
  std::vector<uint8_t> B((size_t)chains * N * K);
  u64 x = 88172645463325252ull;
  auto rnd = [&]() { x ^= x << 13; x ^= x >> 7; x ^= x << 17; return (u32)(x >> 33); };
  for (auto& v : A) { const u32 r = rnd() % 10; v = r == 0 ? 1 : r == 1 ? -1 : 0; }         // ~20 % non-zero weights
  for (auto& v : B) v = (uint8_t)(rnd() % 3);
  int8_t* dA; uint8_t* dB; int32_t* dD;
  CK(cudaMalloc(&dA, A.size())); CK(cudaMalloc(&dB, B.size())); CK(cudaMalloc(&dD, M * N * 4));
  CK(cudaMemcpy(dA, A.data(), A.size(), cudaMemcpyHostToDevice));
  CK(cudaMemcpy(dB, B.data(), B.size(), cudaMemcpyHostToDevice));
  unsigned long long* d_phase;
  CK(cudaMalloc(&d_phase, 48)); CK(cudaMemset(d_phase, 0, 48));
  Args a{dA, dB, !strcmp(mode, "verify") ? dD : nullptr, d_clk, d_phase, d_err, chains, steps, a_tmem, pow2_cols(chains * (N * (split ? 4 : 1) + (a_tmem ? 32 : 0))), split};
  if (a.tmem_cols > 512) { printf("TMEM: %d columns asked, 512 exist\n", a.tmem_cols); return 1; }
  void (*kernel)(Args) = pick_kernel<N>(a.tmem_cols);
  const size_t smem = (size_t)chains * ((a_tmem ? 0 : A_BYTES) + N * K) + 8 * chains + 16;
  if (a.tmem_cols * ctas_per_sm > 512) { printf("TMEM: %d columns x %d CTAs per SM do not fit 512\n", a.tmem_cols, ctas_per_sm); return 1; }
  CK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int occ = 0;
  CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, 128, smem));
  if (occ < ctas_per_sm) printf("(the occupancy query allows %d CTAs of %zu B shared memory per SM, %d asked: the rate below tells what ran)\n", occ, smem, ctas_per_sm);
  if (!strcmp(mode, "verify")) {
    kernel<<<1, 128, smem>>>(a);
    CK(cudaDeviceSynchronize());
    std::vector<int32_t> D(M * N);
    unsigned err = 0;
    CK(cudaMemcpy(D.data(), dD, D.size() * 4, cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(&err, d_err, 4, cudaMemcpyDeviceToHost));
    int bad = 0;
    for (int m = 0; m < M; ++m)
      for (int n = 0; n < N; ++n) {
        int ref = 0;
        for (int k = 0; k < K; ++k) ref += (int)A[m * K + k] * (int)B[n * K + k];
        if (ref != D[m * N + n] && bad++ < 4) printf("  D[%d][%d] = %d, host %d\n", m, n, D[m * N + n], ref);
      }
    printf("verify N=%d a_tmem=%d split=%d: %s (%d of %d entries differ, wait error %u)\n", N, a_tmem, split, bad == 0 && !err ? "D == A . B" : "MISMATCH", bad, M * N, err);
    return bad != 0 || err;
  }
  a.steps = 50;
  kernel<<<grid, 128, smem>>>(a);                              // warm-up
  a.steps = steps;
  CK(cudaEventRecord(e0));
  kernel<<<grid, 128, smem>>>(a);
  CK(cudaEventRecord(e1));
  CK(cudaDeviceSynchronize());
  CK(cudaEventElapsedTime(&ms, e0, e1));
  unsigned err = 0;
  CK(cudaMemcpy(&err, d_err, 4, cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(clk.data(), d_clk, sizeof(unsigned long long) * grid, cudaMemcpyDeviceToHost));
  double mean = 0; for (auto c : clk) mean += (double)c; mean /= grid;
  const double per_sm = mean / steps / (chains * ctas_per_sm);   // clocks per chain-time-step per SM
  const double rate = (double)grid * chains * steps / (ms * 1e-3) / sms;
  printf("step N=%d a_tmem=%d split=%d chains/CTA=%d CTAs/SM=%d (%d chains per SM): round trip %.0f clocks per chain step, %.1f clocks per "
         "chain-time-step per SM, %.2f M chain-time-steps/s per SM (kernel %.3f ms)%s\n", N, a_tmem, split, chains, ctas_per_sm,
         chains * ctas_per_sm, mean / steps, per_sm, rate / 1e6, ms, err ? "  WAIT ERROR" : "");
  unsigned long long ph[6];
  CK(cudaMemcpy(ph, d_phase, 48, cudaMemcpyDeviceToHost));
  const double per = (double)steps * chains;
  printf("    thread 0 of CTA 0, clocks per chain step: wait %.0f | tcgen05.ld %.0f | threshold + store %.0f | fence.proxy.async %.0f | "
         "barrier %.0f | issue 4 MMA + commit %.0f\n", ph[0] / per, ph[1] / per, ph[2] / per, ph[3] / per, ph[4] / per, ph[5] / per);
  return err ? 1 : 0;
}

int main(int argc, char** argv) {
  if (argc < 3) { printf("usage: umma_step verify|ldtm|step N ...\n"); return 2; }
  const char* mode = argv[1];
  const int n = atoi(argv[2]);
  int chains = 1, cps = 1, steps = 2000, a_tmem = 0, split = 0;
  if (!strcmp(mode, "verify")) { a_tmem = argc > 3 ? atoi(argv[3]) : 0; split = argc > 4 ? atoi(argv[4]) : 0; steps = 1; }
  else if (!strcmp(mode, "ldtm")) { cps = argc > 3 ? atoi(argv[3]) : 1; steps = 20000; }
  else { chains = atoi(argv[3]); cps = atoi(argv[4]); steps = atoi(argv[5]); a_tmem = argc > 6 ? atoi(argv[6]) : 0; split = argc > 7 ? atoi(argv[7]) : 0; }
  if (n == 8) return run<8>(mode, chains, cps, steps, a_tmem, split);
  if (n == 16) return run<16>(mode, chains, cps, steps, a_tmem, split);
  printf("N must be 8 or 16\n");
  return 2;
}
