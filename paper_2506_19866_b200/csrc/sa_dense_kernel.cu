// sa_run kernel v4 (sm_100a), for networks of at most 128 nodes and 8 conditions: the node update
// of one time step is ONE dense int8 product on the tensor pipe instead of E shared-memory gathers,
//
//     sum[i][k] = SUM_j  W[i][j] * s[j][k]      (PAPER.md :66-70: the image of node i is a sum over its sources)
//
// with W the chain's N x N weight matrix (w_e at [dst(e)][src(e)], structural zeros elsewhere, padded
// to 16*MT x 32*KS) and s the N x K state matrix of all conditions at t-1.  One chain = one team of
// TW warps = one CTA; warp ww owns the row tiles of its NW/TW result words.  The team keeps the WHOLE
// of W in registers as mma.sync m16n8k32 A fragments (up to 2*NW/TW*KS*4 registers per thread) for
// the entire sa_run, every warp the states of t-1 as KS B fragments, and the team issues MT*KS IMMAs
// per time step.  The sums come back as C fragments, are packed four to a word (byte lanes), thresholded with
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
#define TSD_MINBLOCKS 8
#define TSD_W 2
#endif

namespace tsa_dense {

constexpr int MT = TSD_MT, KS = TSD_KS, NW = TSD_KS, T = TSD_T, NOBS = TSD_NOBS;
constexpr int CS = TSD_CS, TS = TSD_TS, NFIX = TSD_NFIX;
constexpr int TW = TSD_W, TEAM = TW * 32;       // warps / threads per chain
constexpr int WPW = NW / TW;                    // result words per condition a lane produces
constexpr int MTW = 2 * WPW;                    // row tiles per warp (the last warp's may lie beyond MT)
constexpr int NA = MTW * KS * 4;                // A-fragment registers per thread
constexpr int STATE_BYTES = 8 * CS;             // one exchange buffer: 8 condition rows
constexpr int NBUF = TW > 1 ? 2 : 1;            // teams alternate between two exchange buffers: one barrier per time step
constexpr u64 kObsLo = TSD_OBSMASK_LO, kObsHi = TSD_OBSMASK_HI;
constexpr u32 kOnes = 0x01010101u, kTwos = 0x02020202u;
constexpr bool kByteMism = NOBS * 2 * NW <= 255;   // mismatch counters stay in byte lanes
static_assert(KS == 1 || KS == 2 || KS == 4, "KS must be 1, 2 or 4");
static_assert(2 * KS >= MT && MT >= 1, "row <-> column numbering needs MT <= 2*KS");
static_assert(WPW >= 1 && WPW * TW == NW, "team width must divide the words per condition");

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

__device__ __forceinline__ void team_sync() {
  if (TW == 1) __syncwarp(); else __syncthreads();
}

// shared memory through 32-bit shared-window addresses, up to four words at a time
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
  u32 A[NA];        // the warp's rows of the weight matrix: A fragments of its tile (mi, s) at [(mi*KS + s)*4 .. +3]
  u32 TA[WPW];      // per byte (one row of this thread group): 0x80 - t_lo, padding rows 0
  u32 TD[WPW];      // minus, per byte: t_hi - t_lo + 1, padding rows 0
  u32 fix[NFIX];    // clamp fix-ups of this lane (entries of the warp's own rows)
};

// a3 + a4 for the parameters now in registers: returns the team's mismatch count.
// sbuf = shared address of the exchange buffer(s), red = the team's reduction words [2][TW].
__device__ __forceinline__ u32 simulate(const Params& p, const Regs& r, u32 sbuf, volatile u32* red, int parity, int lane, int ww) {
  const int g = lane >> 2, t4 = lane & 3;
  u32 st_addr = sbuf + (u32)((2 * t4) * CS + (g & 3) * TS + ((g >> 2) * NW + ww * WPW) * 4);
  u32 ld_addr = sbuf + (u32)(g * CS + t4 * TS);
  asm volatile("" : "+r"(st_addr), "+r"(ld_addr));      // keep them in registers (no S2R in the loop)
  const int n_tiles = MT - ww * MTW;                      // row tiles of this warp that exist (warp-uniform)
  u32 b[2 * KS];
  {
    const u32* src = p.init_frag + lane * 2 * KS;
#pragma unroll
    for (int i = 0; i < 2 * KS; ++i) b[i] = __ldg(src + i);
  }
  u32 mis = 0u;
  int oj = 0;
#pragma unroll 1
  for (int t = 1; t <= T; ++t) {
    int acc[MTW][4];
#pragma unroll
    for (int m = 0; m < MTW; ++m) { acc[m][0] = 0; acc[m][1] = 0; acc[m][2] = 0; acc[m][3] = 0; }
#pragma unroll
    for (int s = 0; s < KS; ++s)
#pragma unroll
      for (int m = 0; m < MTW; ++m)
        if (TW * MTW <= MT || m < n_tiles) imma(acc[m], &r.A[(m * KS + s) * 4], b[2 * s], b[2 * s + 1]);
    // pack four sums to a word on top of the biased thresholds, compare, encode 0 / 1 / 2 per byte
    u32 ns[2][WPW];
#pragma unroll
    for (int w = 0; w < WPW; ++w)
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
      const u32* ow = p.obs_word + ((size_t)oj * 32 + lane) * (2 * NW) + ww * WPW;
      u32 cnt = 0u;                                       // per byte at most 2*WPW <= 8
#pragma unroll
      for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int w = 0; w < WPW; ++w) {
          const u32 z = ns[c][w] ^ __ldg(ow + c * NW + w);
          cnt += (z | (z >> 1)) & kOnes;
        }
      if (kByteMism) mis += cnt; else mis += __dp4a(cnt, kOnes, 0u);
      ++oj;
    }
    if (t < T) {
      const u32 boff = NBUF == 2 ? (u32)(t & 1) * STATE_BYTES : 0u;
      if (TW == 1) __syncwarp();          // every lane has its B fragments out of the single buffer
      sts_vec(st_addr + boff, ns[0]);
      sts_vec(st_addr + boff + CS, ns[1]);
      __syncwarp();
#pragma unroll
      for (int f = 0; f < NFIX; ++f)
        if (r.fix[f] >> 31) sts_u8(sbuf + boff + (r.fix[f] & 0xFFFFu), (r.fix[f] >> 16) & 3u);
      team_sync();
      u32 lo[NW], hi[NW];
      lds_vec(ld_addr + boff, lo);
      lds_vec(ld_addr + boff + NW * 4, hi);
#pragma unroll
      for (int i = 0; i < NW; ++i) { b[i] = lo[i]; b[NW + i] = hi[i]; }
    }
  }
  u32 m = kByteMism ? __dp4a(mis, kOnes, 0u) : mis;
  m = __reduce_add_sync(0xffffffffu, m);
  if (TW > 1) {
    if (lane == 0) red[parity * TW + ww] = m;
    __syncthreads();
    m = 0;
#pragma unroll
    for (int i = 0; i < TW; ++i) m += red[parity * TW + i];
  }
  return (u32)((int)m + p.fit_const);
}

extern "C" __global__ void __launch_bounds__(TEAM, TSD_MINBLOCKS) tsa_run_dense(const __grid_constant__ Params p) {
  extern __shared__ __align__(16) u32 smem[];
  const int lane = threadIdx.x & 31, ww = threadIdx.x >> 5, g = lane >> 2, t4 = lane & 3;
  const u32 chain = blockIdx.x;
  const u32 gchain = p.chain_id_base + chain;
  // shared memory: exchange buffer(s), the chain's canonical weight and threshold rows, reduction words
  i8* const cw = (i8*)smem + NBUF * STATE_BYTES;
  i8* const cth = cw + TSD_EPADA;
  volatile u32* const red = (volatile u32*)(cth + TSD_NPADA);
  const u32 sbuf = (u32)__cvta_generic_to_shared(smem);
  i8* const cur_w = p.cur_w + (size_t)chain * TSD_EPADA;
  i8* const cur_th = p.cur_th + (size_t)chain * TSD_NPADA;
  i8* const best_w = p.best_w + (size_t)chain * TSD_EPADA;
  i8* const best_th = p.best_th + (size_t)chain * TSD_NPADA;

  // a0: stage the chain
  for (int x = threadIdx.x; x < NBUF * STATE_BYTES / 4; x += TEAM) smem[x] = 0u;
  for (int x = threadIdx.x; x < TSD_EPADA / 4; x += TEAM) ((u32*)cw)[x] = ((const u32*)cur_w)[x];
  for (int x = threadIdx.x; x < TSD_NPADA / 4; x += TEAM) ((u32*)cth)[x] = ((const u32*)cur_th)[x];
  team_sync();
  Regs r;
#pragma unroll
  for (int i = 0; i < NA; ++i) {
    const uint2 fs = __ldg((const uint2*)p.frag_slot + (ww * NA + i) * 32 + lane);
    const u32 o0 = fs.x & 0xFFFFu, o1 = fs.x >> 16, o2 = fs.y & 0xFFFFu, o3 = fs.y >> 16;
    const u32 b0 = o0 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o0];
    const u32 b1 = o1 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o1];
    const u32 b2 = o2 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o2];
    const u32 b3 = o3 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o3];
    r.A[i] = b0 | (b1 << 8) | (b2 << 16) | (b3 << 24);
  }
#pragma unroll
  for (int w = 0; w < WPW; ++w) {
    u32 ta = 0u, td = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const u32 e = __ldg(p.th_entry + (g * NW + ww * WPW + w) * 4 + j);
      if (e != 0xFFFFu) {
        const int q = cth[e];
        ta += (u32)(0x80 + (int)p.tha[q]) << (8 * j);
        td -= (u32)((int)p.tha[q] - (int)p.thb[q]) << (8 * j);
      }
    }
    r.TA[w] = ta; r.TD[w] = td;
  }
#pragma unroll
  for (int f = 0; f < NFIX; ++f) r.fix[f] = __ldg(p.fix + (ww * NFIX + f) * 32 + lane);

  u32 fcur = p.fit_cur[chain], fbest = p.fit_best[chain];
  const int trow = p.trace_row ? p.trace_row[chain] : -1;
  u64 level = p.g0 / (u64)p.steps_per_level;
  i64 left_in_level = p.steps_per_level - (i64)(p.g0 % (u64)p.steps_per_level);

#pragma unroll 1
  for (i64 it = 0; it < p.steps; ++it) {
    const u64 gs = p.g0 + (u64)it;
    u32 x[4];
    philox4x32_10((u32)gs, (u32)(gs >> 32), gchain, 0u, p.key0, p.key1, x);
    // a1 / a2: propose; the threads that hold the parameter apply it in their registers.  Only they
    // read or write its byte in the canonical row, so the row needs no barrier of its own.
    const u32 pidx = __umulhi(x[0], (u32)TSD_NP);
    const bool is_w = pidx < (u32)TSD_NE;
    const u32 loc = is_w ? __ldg(p.wloc + pidx) : __ldg(p.thloc + (pidx - (u32)TSD_NE));
    const u32 slot = loc >> 16;
    int oldv = 0, newv = 0, wsel = -1;
    u32 wx = 0u;
    bool mine;
    if (is_w) {
      mine = ((loc >> 9) & 31u) == (u32)lane && ((loc >> 14) & 3u) == (u32)ww;
      if (mine) {
        oldv = cw[slot];
        newv = (oldv + 2 + (int)__umulhi(x[1], 2u)) % 3 - 1;          // (code + 1 + r) mod 3 - 1, code = old + 1
        wsel = (int)(loc & 0x7Fu);
        wx = ((u32)(oldv ^ newv) & 0xFFu) << (8 * ((loc >> 7) & 3u));
      }
      xor_reg(r.A, wsel, wx);
    } else {
      const int w = (int)((loc >> 3) & 3u);
      mine = (loc & 7u) == (u32)g && w / WPW == ww;
      if (mine) {
        oldv = cth[slot];
        newv = (oldv + 1 + (int)__umulhi(x[1], (u32)(TSD_NPAIRS - 1))) % TSD_NPAIRS;
        const int sh = 8 * (int)((loc >> 5) & 3u);
        const u32 da = (u32)((int)p.tha[newv] - (int)p.tha[oldv]) << sh;
        const u32 dd = (u32)(((int)p.tha[oldv] - (int)p.thb[oldv]) - ((int)p.tha[newv] - (int)p.thb[newv])) << sh;
#pragma unroll
        for (int i = 0; i < WPW; ++i) if (i == w % WPW) { r.TA[i] += da; r.TD[i] += dd; }
      }
    }
    // a3 / a4
    const u32 fcand = simulate(p, r, sbuf, red, (int)(it & 1), lane, ww);
    // a5
    const u64 lv = level < (u64)(p.n_levels - 1) ? level : (u64)(p.n_levels - 1);
    const i64 d = (i64)fcand - (i64)fcur;
    bool acc = d <= 0;
    if (!acc && d <= (i64)p.dmax) acc = x[2] < __ldg(p.accept + lv * (u64)p.dmax + (u64)(d - 1));
    bool new_best = false;
    // a6
    if (acc) {
      fcur = fcand;
      if (mine) {
        if (is_w) cw[slot] = (i8)newv;
        else if (t4 == 0) cth[slot] = (i8)newv;
      }
      if (fcand < fbest) {
        fbest = fcand;
        new_best = true;
        team_sync();
        for (int i = threadIdx.x; i < TSD_EPADA / 4; i += TEAM) ((u32*)best_w)[i] = ((const u32*)cw)[i];
        for (int i = threadIdx.x; i < TSD_NPADA / 4; i += TEAM) ((u32*)best_th)[i] = ((const u32*)cth)[i];
      }
    } else if (is_w) {
      xor_reg(r.A, wsel, wx);
    } else if (mine) {
      const int w = (int)((loc >> 3) & 3u), sh = 8 * (int)((loc >> 5) & 3u);
      const u32 da = (u32)((int)p.tha[oldv] - (int)p.tha[newv]) << sh;
      const u32 dd = (u32)(((int)p.tha[newv] - (int)p.thb[newv]) - ((int)p.tha[oldv] - (int)p.thb[oldv])) << sh;
#pragma unroll
      for (int i = 0; i < WPW; ++i) if (i == w % WPW) { r.TA[i] += da; r.TD[i] += dd; }
    }
    __syncwarp();
    if (trow >= 0 && mine && (is_w || t4 == 0)) {
      const u64 idx = gs - p.trace_g0;
      const u32 code = is_w ? (u32)(newv + 1) : (u32)newv;
      if (gs >= p.trace_g0 && idx < (u64)p.trace_max)
        p.trace_rec[(size_t)trow * (size_t)p.trace_max + idx] =
            (u64)fcand | ((u64)pidx << 32) | ((u64)code << 56) | ((u64)(acc ? 1 : 0) << 60) | ((u64)(new_best ? 1 : 0) << 61);
    }
    if (--left_in_level == 0) { ++level; left_in_level = p.steps_per_level; }
  }
  // a7
  team_sync();
  for (int i = threadIdx.x; i < TSD_EPADA / 4; i += TEAM) ((u32*)cur_w)[i] = ((const u32*)cw)[i];
  for (int i = threadIdx.x; i < TSD_NPADA / 4; i += TEAM) ((u32*)cur_th)[i] = ((const u32*)cth)[i];
  if (threadIdx.x == 0) { p.fit_cur[chain] = fcur; p.fit_best[chain] = fbest; }
}

}  // namespace tsa_dense
