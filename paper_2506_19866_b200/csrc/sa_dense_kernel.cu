// sa_run kernel v4 (sm_100a), for networks of at most 128 nodes and 8 conditions: the node update
// of one time step is ONE dense int8 product on the tensor pipe instead of E shared-memory gathers,
//
//     sum[i][k] = SUM_j  W[i][j] * s[j][k]      (PAPER.md :66-70: the image of node i is a sum over its sources)
//
// with W the chain's N x N weight matrix (w_e at [dst(e)][src(e)], structural zeros elsewhere, padded
// to 16*MT x 32*KS) and s the N x K state matrix of all conditions at t-1.  One warp = one chain.
// The warp keeps the WHOLE of W in registers as mma.sync m16n8k32 A fragments (MT*KS*4 registers per
// thread) for the entire sa_run, the states of t-1 as KS B fragments, and issues MT*KS IMMAs per time
// step.  The sums come back as C fragments, are packed four to a word (byte lanes), thresholded with
// the same biased-byte trick as the gather kernel, and go through a 1-2 KB shared-memory buffer laid
// out so that every lane writes its result words with one vector store and reads its next B
// fragments with two vector loads (row <-> column numbering chosen by the host, sa_dense_plan.cpp).
// Compiled at run time by NVRTC (sa_jit.cpp) with the problem's shape as -D constants, and ahead of
// time with the Mtb-shaped defaults below (build check, SASS inspection).  It includes nothing:
// sa_dense_params.h is prepended by whoever compiles it.
// (Table 1 :121-158 is the chain step, :86-111 the objective; SURVEY.md §8(c) the exact
// arithmetic.)  Shares nothing with oracle/.
#ifndef TSD_MT
#define TSD_MT 7
#define TSD_KS 4
#define TSD_T 32
#define TSD_NOBS 8
#define TSD_OBSMASK_LO 0x0000000111111110ull
#define TSD_OBSMASK_HI 0x0ull
#define TSD_CS 144
#define TSD_TS 32
#define TSD_NPAIRS 6
#define TSD_NE 900
#define TSD_NP 1000
#define TSD_EPADA 1408
#define TSD_NPADA 128
#define TSD_NFIX 1
#define TSD_MINBLOCKS 10
#endif

namespace tsa_dense {

constexpr int MT = TSD_MT, KS = TSD_KS, NW = TSD_KS, T = TSD_T, NOBS = TSD_NOBS;
constexpr int CS = TSD_CS, TS = TSD_TS, NFIX = TSD_NFIX;
constexpr int NA = MT * KS * 4;                 // A-fragment registers per thread
constexpr int STATE_BYTES = 8 * CS;             // one exchange buffer: 8 condition rows
constexpr u64 kObsLo = TSD_OBSMASK_LO, kObsHi = TSD_OBSMASK_HI;
constexpr u32 kOnes = 0x01010101u, kTwos = 0x02020202u;
constexpr bool kByteMism = NOBS * 2 * NW <= 255;   // mismatch counters stay in byte lanes
static_assert(KS == 1 || KS == 2 || KS == 4, "KS must be 1, 2 or 4");
static_assert(2 * KS >= MT && MT >= 1, "row <-> column numbering needs MT <= 2*KS");

// Philox4x32-10 (Salmon et al., SC'11)
__device__ __forceinline__ void philox4x32_10(u32 c0, u32 c1, u32 c2, u32 c3, u32 k0, u32 k1, u32 (&out)[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const u32 hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const u32 hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// 0xFF in every byte whose bit 7 is set, else 0x00
__device__ __forceinline__ u32 sign_mask(u32 x) {
  u32 r;
  asm("prmt.b32 %0, %1, 0, 0xBA98;" : "=r"(r) : "r"(x));
  return r;
}

// D (16 x 8, s32) += A (16 x 32, s8, row) * B (32 x 8, s8, col)
__device__ __forceinline__ void imma(int (&c)[4], const u32* a, u32 b0, u32 b1) {
  asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// shared memory through 32-bit shared-window addresses, NW words at a time
__device__ __forceinline__ void lds_vec(u32 a, u32 (&s)[1]) { asm volatile("ld.shared.u32 %0, [%1];" : "=r"(s[0]) : "r"(a) : "memory"); }
__device__ __forceinline__ void lds_vec(u32 a, u32 (&s)[2]) { asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(s[0]), "=r"(s[1]) : "r"(a) : "memory"); }
__device__ __forceinline__ void lds_vec(u32 a, u32 (&s)[4]) {
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(s[0]), "=r"(s[1]), "=r"(s[2]), "=r"(s[3]) : "r"(a) : "memory");
}
__device__ __forceinline__ void sts_vec(u32 a, const u32 (&s)[1]) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(s[0]) : "memory"); }
__device__ __forceinline__ void sts_vec(u32 a, const u32 (&s)[2]) { asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(a), "r"(s[0]), "r"(s[1]) : "memory"); }
__device__ __forceinline__ void sts_vec(u32 a, const u32 (&s)[4]) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(s[0]), "r"(s[1]), "r"(s[2]), "r"(s[3]) : "memory");
}
__device__ __forceinline__ void sts_u8(u32 a, u32 v) { asm volatile("st.shared.u8 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }

// a[sel] ^= x for a run-time sel (a jump table: registers cannot be indexed); sel outside [0, NA) does nothing
#define TSD_C1(i) case (i): if ((i) < NA) a[(i) < NA ? (i) : 0] ^= x; break;
#define TSD_C4(i) TSD_C1(i) TSD_C1((i) + 1) TSD_C1((i) + 2) TSD_C1((i) + 3)
#define TSD_C16(i) TSD_C4(i) TSD_C4((i) + 4) TSD_C4((i) + 8) TSD_C4((i) + 12)
#define TSD_C64(i) TSD_C16(i) TSD_C16((i) + 16) TSD_C16((i) + 32) TSD_C16((i) + 48)
__device__ __forceinline__ void xor_reg(u32 (&a)[NA], int sel, u32 x) {
  switch (sel) {
    TSD_C64(0)
    TSD_C64(64)
    default: break;
  }
}

// Everything a thread keeps in registers for the whole launch.
struct Regs {
  u32 A[NA];        // the chain's weight matrix: A fragments of tile (m, s) at [(m*KS + s)*4 .. +3]
  u32 TA[NW];       // per byte (row 32w + 8j' ... of this thread group): 0x80 - t_lo, padding rows 0
  u32 TD[NW];       // minus, per byte: t_hi - t_lo + 1, padding rows 0
  u32 fix[NFIX];    // clamp fix-ups of this lane
};

// a3 + a4 for the parameters now in registers: returns the warp's mismatch count.
// sbuf = shared address of the warp's exchange buffer.
__device__ __forceinline__ u32 simulate(const Params& p, const Regs& r, u32 sbuf, int lane) {
  const int g = lane >> 2, t4 = lane & 3;
  const u32 st_addr = sbuf + (u32)((2 * t4) * CS + (g & 3) * TS + (g >> 2) * NW * 4);
  const u32 ld_addr = sbuf + (u32)(g * CS + t4 * TS);
  u32 b[2 * KS];
  {
    const u32* src = p.init_frag + lane * 2 * KS;
#pragma unroll
    for (int i = 0; i < 2 * KS; ++i) b[i] = __ldg(src + i);
  }
  u32 mis[2 * NW];
#pragma unroll
  for (int i = 0; i < 2 * NW; ++i) mis[i] = 0u;
  int oj = 0;
#pragma unroll 1
  for (int t = 1; t <= T; ++t) {
    int acc[2 * NW][4];
#pragma unroll
    for (int m = 0; m < 2 * NW; ++m) { acc[m][0] = 0; acc[m][1] = 0; acc[m][2] = 0; acc[m][3] = 0; }
#pragma unroll
    for (int s = 0; s < KS; ++s)
#pragma unroll
      for (int m = 0; m < MT; ++m) imma(acc[m], &r.A[(m * KS + s) * 4], b[2 * s], b[2 * s + 1]);
    // pack four sums to a word on top of the biased thresholds, compare, encode 0 / 1 / 2 per byte
    u32 ns[2][NW];
#pragma unroll
    for (int w = 0; w < NW; ++w)
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const u32 x = r.TA[w] + (u32)acc[2 * w][c] + ((u32)acc[2 * w][2 + c] << 8) + ((u32)acc[2 * w + 1][c] << 16) +
                      ((u32)acc[2 * w + 1][2 + c] << 24);
        const u32 ge = sign_mask(x);
        const u32 gt = sign_mask(x + r.TD[w]);
        ns[c][w] = ((ge ^ gt) & kOnes) | (gt & kTwos);
      }
    const bool is_obs = t < 64 ? ((kObsLo >> t) & 1ull) : ((kObsHi >> (t - 64)) & 1ull);
    if (is_obs) {
      const u32* ow = p.obs_word + ((size_t)oj * 32 + lane) * (2 * NW);
#pragma unroll
      for (int i = 0; i < 2 * NW; ++i) {
        const u32 z = ns[i / NW][i % NW] ^ __ldg(ow + i);
        const u32 nz = (z | (z >> 1)) & kOnes;
        if (kByteMism) mis[i] += nz; else mis[i] += (u32)__popc(nz);
      }
      ++oj;
    }
    if (t < T) {
      __syncwarp();                       // every lane has its B fragments out of the buffer
      sts_vec(st_addr, ns[0]);
      sts_vec(st_addr + CS, ns[1]);
      __syncwarp();
#pragma unroll
      for (int f = 0; f < NFIX; ++f)
        if (r.fix[f] >> 31) sts_u8(sbuf + (r.fix[f] & 0xFFFFu), (r.fix[f] >> 16) & 3u);
      __syncwarp();
      u32 lo[NW], hi[NW];
      lds_vec(ld_addr, lo);
      lds_vec(ld_addr + NW * 4, hi);
#pragma unroll
      for (int i = 0; i < NW; ++i) { b[i] = lo[i]; b[NW + i] = hi[i]; }
    }
  }
  u32 m = 0;
#pragma unroll
  for (int i = 0; i < 2 * NW; ++i) m += kByteMism ? __dp4a(mis[i], kOnes, 0u) : mis[i];
  m = __reduce_add_sync(0xffffffffu, m);
  return (u32)((int)m + p.fit_const);
}

extern "C" __global__ void __launch_bounds__(32, TSD_MINBLOCKS) tsa_run_dense(const __grid_constant__ Params p) {
  extern __shared__ __align__(16) u32 smem[];
  const int lane = threadIdx.x, g = lane >> 2;
  const u32 chain = blockIdx.x;
  const u32 gchain = p.chain_id_base + chain;
  // shared memory: exchange buffer, then the chain's canonical weight and threshold rows
  i8* const cw = (i8*)smem + STATE_BYTES;
  i8* const cth = cw + TSD_EPADA;
  const u32 sbuf = (u32)__cvta_generic_to_shared(smem);
  i8* const cur_w = p.cur_w + (size_t)chain * TSD_EPADA;
  i8* const cur_th = p.cur_th + (size_t)chain * TSD_NPADA;
  i8* const best_w = p.best_w + (size_t)chain * TSD_EPADA;
  i8* const best_th = p.best_th + (size_t)chain * TSD_NPADA;

  // a0: stage the chain
  for (int x = lane; x < STATE_BYTES / 4; x += 32) smem[x] = 0u;
  for (int x = lane; x < TSD_EPADA / 4; x += 32) ((u32*)cw)[x] = ((const u32*)cur_w)[x];
  for (int x = lane; x < TSD_NPADA / 4; x += 32) ((u32*)cth)[x] = ((const u32*)cur_th)[x];
  __syncwarp();
  Regs r;
#pragma unroll
  for (int i = 0; i < NA; ++i) {
    const uint2 fs = __ldg((const uint2*)p.frag_slot + i * 32 + lane);
    const u32 o0 = fs.x & 0xFFFFu, o1 = fs.x >> 16, o2 = fs.y & 0xFFFFu, o3 = fs.y >> 16;
    const u32 b0 = o0 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o0];
    const u32 b1 = o1 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o1];
    const u32 b2 = o2 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o2];
    const u32 b3 = o3 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o3];
    r.A[i] = b0 | (b1 << 8) | (b2 << 16) | (b3 << 24);
  }
#pragma unroll
  for (int w = 0; w < NW; ++w) {
    u32 ta = 0u, td = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const u32 e = __ldg(p.th_entry + (g * NW + w) * 4 + j);
      if (e != 0xFFFFu) {
        const int q = cth[e];
        ta += (u32)(0x80 + (int)p.tha[q]) << (8 * j);
        td -= (u32)((int)p.tha[q] - (int)p.thb[q]) << (8 * j);
      }
    }
    r.TA[w] = ta; r.TD[w] = td;
  }
#pragma unroll
  for (int f = 0; f < NFIX; ++f) r.fix[f] = __ldg(p.fix + f * 32 + lane);

  u32 fcur = p.fit_cur[chain], fbest = p.fit_best[chain];
  const int trow = p.trace_row ? p.trace_row[chain] : -1;
  u64 level = p.g0 / (u64)p.steps_per_level;
  i64 left_in_level = p.steps_per_level - (i64)(p.g0 % (u64)p.steps_per_level);

#pragma unroll 1
  for (i64 it = 0; it < p.steps; ++it) {
    const u64 gs = p.g0 + (u64)it;
    u32 x[4];
    philox4x32_10((u32)gs, (u32)(gs >> 32), gchain, 0u, p.key0, p.key1, x);
    // a1 / a2: propose; apply in the registers of the lanes that hold the parameter and in the canonical row
    const u32 pidx = __umulhi(x[0], (u32)TSD_NP);
    const bool is_w = pidx < (u32)TSD_NE;
    const u32 loc = is_w ? __ldg(p.wloc + pidx) : __ldg(p.thloc + (pidx - (u32)TSD_NE));
    const u32 slot = loc >> 16;
    int oldv, newv;
    u32 code, wx = 0u;
    int wsel = -1;
    if (is_w) {
      oldv = cw[slot];
      newv = (oldv + 2 + (int)__umulhi(x[1], 2u)) % 3 - 1;          // (code + 1 + r) mod 3 - 1, code = old + 1
      code = (u32)(newv + 1);
      if (((loc >> 10) & 31u) == (u32)lane) { wsel = (int)(loc & 0xFFu); wx = ((u32)(oldv ^ newv) & 0xFFu) << (8 * ((loc >> 8) & 3u)); }
      xor_reg(r.A, wsel, wx);
      __syncwarp();
      if (lane == 0) cw[slot] = (i8)newv;
    } else {
      oldv = cth[slot];
      newv = (oldv + 1 + (int)__umulhi(x[1], (u32)(TSD_NPAIRS - 1))) % TSD_NPAIRS;
      code = (u32)newv;
      if ((loc & 7u) == (u32)g) {
        const int w = (int)((loc >> 3) & 3u), sh = 8 * (int)((loc >> 5) & 3u);
        const u32 da = (u32)((int)p.tha[newv] - (int)p.tha[oldv]) << sh;
        const u32 dd = (u32)(((int)p.tha[oldv] - (int)p.thb[oldv]) - ((int)p.tha[newv] - (int)p.thb[newv])) << sh;
#pragma unroll
        for (int i = 0; i < NW; ++i) if (i == w) { r.TA[i] += da; r.TD[i] += dd; }
      }
      __syncwarp();
      if (lane == 0) cth[slot] = (i8)newv;
    }
    // a3 / a4
    const u32 fcand = simulate(p, r, sbuf, lane);
    // a5
    const u64 lv = level < (u64)(p.n_levels - 1) ? level : (u64)(p.n_levels - 1);
    const i64 d = (i64)fcand - (i64)fcur;
    bool acc = d <= 0;
    if (!acc && d <= (i64)p.dmax) acc = x[2] < __ldg(p.accept + lv * (u64)p.dmax + (u64)(d - 1));
    bool new_best = false;
    // a6
    if (acc) {
      fcur = fcand;
      if (fcand < fbest) {
        fbest = fcand;
        new_best = true;
        __syncwarp();
        for (int i = lane; i < TSD_EPADA / 4; i += 32) ((u32*)best_w)[i] = ((const u32*)cw)[i];
        for (int i = lane; i < TSD_NPADA / 4; i += 32) ((u32*)best_th)[i] = ((const u32*)cth)[i];
      }
    } else if (is_w) {
      xor_reg(r.A, wsel, wx);
      if (lane == 0) cw[slot] = (i8)oldv;
    } else {
      if ((loc & 7u) == (u32)g) {
        const int w = (int)((loc >> 3) & 3u), sh = 8 * (int)((loc >> 5) & 3u);
        const u32 da = (u32)((int)p.tha[oldv] - (int)p.tha[newv]) << sh;
        const u32 dd = (u32)(((int)p.tha[newv] - (int)p.thb[newv]) - ((int)p.tha[oldv] - (int)p.thb[oldv])) << sh;
#pragma unroll
        for (int i = 0; i < NW; ++i) if (i == w) { r.TA[i] += da; r.TD[i] += dd; }
      }
      if (lane == 0) cth[slot] = (i8)oldv;
    }
    __syncwarp();
    if (trow >= 0 && lane == 0) {
      const u64 idx = gs - p.trace_g0;
      if (gs >= p.trace_g0 && idx < (u64)p.trace_max)
        p.trace_rec[(size_t)trow * (size_t)p.trace_max + idx] =
            (u64)fcand | ((u64)pidx << 32) | ((u64)code << 56) | ((u64)(acc ? 1 : 0) << 60) | ((u64)(new_best ? 1 : 0) << 61);
    }
    if (--left_in_level == 0) { ++level; left_in_level = p.steps_per_level; }
  }
  // a7
  __syncwarp();
  for (int i = lane; i < TSD_EPADA / 4; i += 32) ((u32*)cur_w)[i] = ((const u32*)cw)[i];
  for (int i = lane; i < TSD_NPADA / 4; i += 32) ((u32*)cur_th)[i] = ((const u32*)cth)[i];
  if (lane == 0) { p.fit_cur[chain] = fcur; p.fit_best[chain] = fbest; }
}

}  // namespace tsa_dense
