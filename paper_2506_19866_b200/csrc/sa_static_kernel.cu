// sa_run kernel v3 (sm_100a): the whole schedule of ONE problem is static.
//
// This file is compiled at run time by NVRTC (sa_jit.cpp) with the problem's schedule as -D
// constants, and ahead of time by build.py with the Mtb-shaped defaults below (build check, SASS
// inspection).  It includes nothing: sa_static_params.h is prepended by whoever compiles it.
//
// One chain = one team of W warps = one CTA.  Thread (warp, lane) owns, in REGISTERS for the whole
// sa_run: the byte offsets of the source entries of its edge slots, the chain's weights of those
// slots (4 per register), and per tier (a tier = one pass per warp) the threshold words (clamped
// conditions folded in) and the store offset of the row it finalises.  Shared memory holds only the
// node states (byte lanes, 4 conditions per 32-bit word, CG words per node): the t = 0 states and
// two buffers that alternate.  Per edge slot the inner loop is LDS + CG x IMAD plus, when the
// register budget does not let the compiler hoist them, one offset and one weight extraction.  All
// loops over tiers, slots and combine rounds are unrolled at compile time, so no schedule table is
// read at run time.
// (Table 1 :121-158 is the chain step, :66-70 the node update, :86-111 the objective;
// SURVEY.md §8(c) the exact arithmetic.)  Shares nothing with oracle/.
#ifndef TSA_CG
#define TSA_CG 2
#define TSA_W 1
#define TSA_NT 4
#define TSA_IT 13, 9, 6, 5
#define TSA_RND 2, 1, 0, 0
#define TSA_T 32
#define TSA_NOBS 8
#define TSA_OBSMASK_LO 0x0000000111111110ull
#define TSA_OBSMASK_HI 0x0ull
#define TSA_STATE_WORDS 256
#define TSA_NPAIRS 6
#define TSA_NE 900
#define TSA_NP 1000
#define TSA_EPADA 1408
#define TSA_NPADA 128
#define TSA_MINBLOCKS 16
#define TSA_TUNROLL 1
#define TSA_BATCH 8
#endif
#ifndef TSA_CONSTRAINED
#define TSA_CONSTRAINED 0
#define TSA_NN 100
#endif

namespace tsa_static {

constexpr int CG = TSA_CG, W = TSA_W, NT = TSA_NT, T = TSA_T, NOBS = TSA_NOBS;
constexpr int STATE_WORDS = TSA_STATE_WORDS, STATE_BYTES = TSA_STATE_WORDS * 4;
constexpr int TEAM = W * 32;
constexpr int kIT[NT] = {TSA_IT};
constexpr int kRND[NT] = {TSA_RND};
constexpr u64 kObsLo = TSA_OBSMASK_LO, kObsHi = TSA_OBSMASK_HI;
constexpr u32 kOnes = 0x01010101u, kTwos = 0x02020202u;

__host__ __device__ constexpr int groups(int j) { return (kIT[j] + 3) / 4; }
__host__ __device__ constexpr int wbase(int j) { int s = 0; for (int i = 0; i < j; ++i) s += groups(i); return s; }
__host__ __device__ constexpr int obase(int j) { int s = 0; for (int i = 0; i < j; ++i) s += (kIT[i] + 1) / 2; return s; }
__host__ __device__ constexpr int tier_bytes(int j) { int s = 0; for (int i = 0; i < j; ++i) s += W * groups(i) * 128; return s; }
constexpr int NWREG = wbase(NT), NOREG = obase(NT);
constexpr bool kByteMism = NOBS * ((TSA_STATE_WORDS + TSA_W * 128 - 1) / (TSA_W * 128)) <= 255;   // mismatch counters stay in byte lanes
constexpr int kTUnroll = TSA_TUNROLL;
constexpr int kScoreIters = (STATE_WORDS + TEAM * 4 - 1) / (TEAM * 4);

template <int N> struct VecT;
template <> struct VecT<1> { typedef u32 type; };
template <> struct VecT<2> { typedef uint2 type; };
template <> struct VecT<4> { typedef uint4 type; };
typedef VecT<CG>::type V;

__device__ __forceinline__ void unpack(const u32& v, u32 (&s)[1]) { s[0] = v; }
__device__ __forceinline__ void unpack(const uint2& v, u32 (&s)[2]) { s[0] = v.x; s[1] = v.y; }
__device__ __forceinline__ void unpack(const uint4& v, u32 (&s)[4]) { s[0] = v.x; s[1] = v.y; s[2] = v.z; s[3] = v.w; }
__device__ __forceinline__ u32 pack(const u32 (&s)[1]) { return s[0]; }
__device__ __forceinline__ uint2 pack(const u32 (&s)[2]) { return make_uint2(s[0], s[1]); }
__device__ __forceinline__ uint4 pack(const u32 (&s)[4]) { return make_uint4(s[0], s[1], s[2], s[3]); }

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

// sign-extended byte U of a weight word in one PRMT (selector nibble U picks the byte, U|8 its sign)
template <int U>
__device__ __forceinline__ int weight_of(u32 wword) {
  constexpr u32 sel = (u32)(U | ((U | 8) << 4) | ((U | 8) << 8) | ((U | 8) << 12));
  u32 r;
  asm("prmt.b32 %0, %1, 0, %2;" : "=r"(r) : "r"(wword), "n"(sel));
  return (int)r;
}
// 0xFF in every byte whose bit 7 is set, else 0x00
__device__ __forceinline__ u32 sign_mask(u32 x) {
  u32 r;
  asm("prmt.b32 %0, %1, 0, 0xBA98;" : "=r"(r) : "r"(x));
  return r;
}

__device__ __forceinline__ void team_sync() {
  if (W == 1) __syncwarp(); else __syncthreads();
}

// Debug build (-DTSA_BOUNDS=1, set by TSA_BOUNDS_CHECK=1 under TSA_TUNING=1): every shared-memory access made
// through the helpers below is checked against the CTA's dynamic shared-memory window and its own
// alignment, and traps if it falls outside (compute-sanitizer is not available on the GPU pool).
#ifdef TSA_BOUNDS
__device__ __forceinline__ void smem_check(u32 a, u32 bytes) {
  u32 total, base;
  asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(total));
  { extern __shared__ __align__(16) unsigned char tsa_smem_window[]; base = (u32)__cvta_generic_to_shared(tsa_smem_window); }
  if (a < base || a + bytes > base + total || (a & (bytes - 1u)) != 0u) __trap();
}
#else
__device__ __forceinline__ void smem_check(u32, u32) {}
#endif
// shared memory through 32-bit shared-window addresses
__device__ __forceinline__ void lds(u32 a, u32 (&s)[1]) { smem_check(a, 4); asm volatile("ld.shared.u32 %0, [%1];" : "=r"(s[0]) : "r"(a) : "memory"); }
__device__ __forceinline__ void lds(u32 a, u32 (&s)[2]) { smem_check(a, 8); asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(s[0]), "=r"(s[1]) : "r"(a) : "memory"); }
__device__ __forceinline__ void lds(u32 a, u32 (&s)[4]) {
  smem_check(a, 16);
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(s[0]), "=r"(s[1]), "=r"(s[2]), "=r"(s[3]) : "r"(a) : "memory");
}
__device__ __forceinline__ void sts(u32 a, const u32 (&s)[1]) { smem_check(a, 4); asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(s[0]) : "memory"); }
__device__ __forceinline__ void sts(u32 a, const u32 (&s)[2]) { smem_check(a, 8); asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(a), "r"(s[0]), "r"(s[1]) : "memory"); }
__device__ __forceinline__ void sts(u32 a, const u32 (&s)[4]) {
  smem_check(a, 16);
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(s[0]), "r"(s[1]), "r"(s[2]), "r"(s[3]) : "memory");
}

// Everything a thread keeps in registers for the whole launch.
struct Regs {
  u32 off2[NOREG];      // two 16-bit source-entry byte offsets per word
  u32 w[NWREG];         // four int8 weights per word
  u32 row[NT];          // byte offset of the entry this lane stores to (a private scratch entry if it finalises nothing)
  u32 take[NT];         // bit q: in combine round q add the partial sum of lane + 2^q
  u32 A[NT][CG];        // accumulator start per byte: 0x80 - t_lo (finalising lane; clamped bytes: 64 or 192), else 0
  u32 D[NT][CG];        // minus, per byte: t_hi - t_lo + 1 (clamped bytes: 0 or 128)
  int thq[NT];          // threshold-pair index of the row this lane finalises, -1 if none
};

// Threshold words of tier j for pair q.  Byte b of A + sum has bit 7 = [sum >= t_lo]; adding D gives
// bit 7 = [sum > t_hi].  A clamped condition keeps its initial value v for every sum (|sum| <= 62,
// checked by the host): v = 0: A = 64, D = 0; v = 2: A = 192, D = 0; v = 1: A = 192, D = -128.
__device__ __forceinline__ void set_threshold(const Params& p, Regs& r, int j, int q) {
  r.thq[j] = q;
  if (q < 0) return;                       // not a finalising lane: A stays 0
  const u32 an = (u32)(0x80 + (int)p.tha[q]) * kOnes, dn = (u32)((int)p.tha[q] - (int)p.thb[q]) * kOnes;
#pragma unroll
  for (int c = 0; c < CG; ++c) {
    const u32 cm = __ldg(p.lane_clamp + (j * 3 * CG + c) * TEAM + threadIdx.x);
    const u32 ca = __ldg(p.lane_clamp + (j * 3 * CG + CG + c) * TEAM + threadIdx.x);
    const u32 cd = __ldg(p.lane_clamp + (j * 3 * CG + 2 * CG + c) * TEAM + threadIdx.x);
    r.A[j][c] = (an & ~cm) | ca;
    r.D[j][c] = 0u - ((dn & ~cm) | cd);
  }
}

// a3 for one tier: accumulate the lane's edge slots, combine split rows, threshold, store.
// cur / nxt = shared addresses of the buffers holding the states at t-1 / receiving those at t.
template <int J>
__device__ __forceinline__ void tier(const Regs& r, u32 cur, u32 nxt) {
  constexpr int IT = kIT[J], RND = kRND[J], OB = obase(J), WB = wbase(J), B = TSA_BATCH;
  u32 acc[CG];
#pragma unroll
  for (int c = 0; c < CG; ++c) acc[c] = r.A[J][c];
#pragma unroll
  for (int k0 = 0; k0 < IT; k0 += B) {
    u32 s[B][CG];
#pragma unroll
    for (int b = 0; b < B; ++b) {
      const int k = k0 + b;
      if (k < IT) {
        const u32 o2 = r.off2[OB + k / 2];
        lds(cur + ((k & 1) ? (o2 >> 16) : (o2 & 0xFFFFu)), s[b]);
      }
    }
#pragma unroll
    for (int b = 0; b < B; ++b) {
      const int k = k0 + b;
      if (k < IT) {
        const u32 ww = r.w[WB + k / 4];
        const int wv = (k & 3) == 0 ? weight_of<0>(ww) : (k & 3) == 1 ? weight_of<1>(ww) : (k & 3) == 2 ? weight_of<2>(ww) : weight_of<3>(ww);
#pragma unroll
        for (int c = 0; c < CG; ++c) acc[c] += (u32)(wv * (int)s[b][c]);
      }
    }
  }
  // split rows: partial sums of consecutive lanes are added up a binary tree (partials start at 0)
#pragma unroll
  for (int q = 0; q < RND; ++q) {
    const u32 mask = ((r.take[J] >> q) & 1u) ? 0xFFFFFFFFu : 0u;
#pragma unroll
    for (int c = 0; c < CG; ++c) acc[c] += __shfl_down_sync(0xffffffffu, acc[c], 1u << q) & mask;
  }
  u32 ns[CG];
#pragma unroll
  for (int c = 0; c < CG; ++c) {
    const u32 ge = sign_mask(acc[c]);
    const u32 gt = sign_mask(acc[c] + r.D[J][c]);
    ns[c] = ((ge ^ gt) & kOnes) | (gt & kTwos);          // 0 / 1 / 2 per byte
  }
  sts(nxt + r.row[J], ns);
}

template <int J>
struct Tiers {
  static __device__ __forceinline__ void run(const Regs& r, u32 cur, u32 nxt) {
    tier<J>(r, cur, nxt);
    Tiers<J + 1>::run(r, cur, nxt);
  }
};
template <>
struct Tiers<NT> {
  static __device__ __forceinline__ void run(const Regs&, u32, u32) {}
};

// a4: mismatches of the whole state buffer at observation index oj (dummy entries, holes, unobserved
// and clamped lanes have a zero mask)
__device__ __forceinline__ void score(const Params& p, u32 buf, int oj, u32 (&mis)[4]) {
  const uint4* ow = (const uint4*)(p.obsw + (size_t)oj * STATE_WORDS);
  const uint4* om = (const uint4*)(p.obsm + (size_t)oj * STATE_WORDS);
#pragma unroll
  for (int x = 0; x < kScoreIters; ++x) {
    const int i = x * TEAM + (int)threadIdx.x;      // uint4 index
    if (STATE_WORDS % (TEAM * 4) == 0 || i * 4 < STATE_WORDS) {
      u32 s[4], v[4], m[4];
      lds(buf + (u32)i * 16u, s);
      unpack(__ldg(ow + i), v);
      unpack(__ldg(om + i), m);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const u32 d = s[c] ^ v[c];
        const u32 z = (d | (d >> 1)) & m[c];
        if (kByteMism) mis[c] += z; else mis[c] += (u32)__popc(z);
      }
    }
  }
}

// a3 + a4: returns the team's mismatch count of the parameters now in registers.  sbase = shared
// address of this team's three state buffers: [0] the t = 0 states (never written), [1], [2].
__device__ __forceinline__ u32 simulate(const Params& p, const Regs& r, u32 sbase, u32* red) {
  u32 mis[4] = {0u, 0u, 0u, 0u};
  int oj = 0;
  u32 cur = sbase, nxt = sbase + STATE_BYTES;
#pragma unroll (kTUnroll)
  for (int t = 1; t <= T; ++t) {
    Tiers<0>::run(r, cur, nxt);
    team_sync();
    const bool is_obs = t < 64 ? ((kObsLo >> t) & 1ull) : ((kObsHi >> (t - 64)) & 1ull);
    if (is_obs) { score(p, nxt, oj, mis); ++oj; }
    cur = nxt;
    nxt = (nxt == sbase + STATE_BYTES) ? sbase + 2 * STATE_BYTES : sbase + STATE_BYTES;
  }
  u32 m = 0;
#pragma unroll
  for (int c = 0; c < 4; ++c) m += kByteMism ? __dp4a(mis[c], kOnes, 0u) : mis[c];
  m = __reduce_add_sync(0xffffffffu, m);
  if (W > 1) {
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    m = 0;
#pragma unroll
    for (int i = 0; i < W; ++i) m += red[i];
    __syncthreads();
  }
  return m + p.fit_const;
}

template <int J>
__device__ __forceinline__ u32 tier_w_addr(int g, int warp, int lane) {
  constexpr int TB = tier_bytes(J), G = groups(J);
  return (u32)(TB + (warp * G + g) * 128 + lane * 4);
}

// weights and thresholds of this thread <-> one chain's rows in HBM
template <int J>
struct RowIO {
  static __device__ __forceinline__ void load(const Params& p, Regs& r, const i8* wrow, const i8* throw_, int warp, int lane) {
    constexpr int G = groups(J), WB = wbase(J);
#pragma unroll
    for (int g = 0; g < G; ++g) r.w[WB + g] = *(const u32*)(wrow + tier_w_addr<J>(g, warp, lane));
#pragma unroll
    for (int c = 0; c < CG; ++c) { r.A[J][c] = 0u; r.D[J][c] = 0u; }
    set_threshold(p, r, J, r.thq[J] >= 0 ? (int)throw_[r.row[J] / (CG * 4)] : -1);
    RowIO<J + 1>::load(p, r, wrow, throw_, warp, lane);
  }
  static __device__ __forceinline__ void store(const Regs& r, i8* wrow, i8* throw_, int warp, int lane) {
    constexpr int G = groups(J), WB = wbase(J);
#pragma unroll
    for (int g = 0; g < G; ++g) *(u32*)(wrow + tier_w_addr<J>(g, warp, lane)) = r.w[WB + g];
    if (r.thq[J] >= 0) throw_[r.row[J] / (CG * 4)] = (i8)r.thq[J];
    RowIO<J + 1>::store(r, wrow, throw_, warp, lane);
  }
};
template <>
struct RowIO<NT> {
  static __device__ __forceinline__ void load(const Params&, Regs&, const i8*, const i8*, int, int) {}
  static __device__ __forceinline__ void store(const Regs&, i8*, i8*, int, int) {}
};

extern "C" __global__ void __launch_bounds__(TEAM, TSA_MINBLOCKS) tsa_run_static(const __grid_constant__ Params p) {
  extern __shared__ __align__(16) u32 smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const u32 chain = blockIdx.x;
  const u32 gchain = p.chain_id_base + chain;

  Regs r;
#pragma unroll
  for (int i = 0; i < NOREG; ++i) r.off2[i] = __ldg(p.lane_off2 + i * TEAM + threadIdx.x);
#pragma unroll
  for (int j = 0; j < NT; ++j) {
    const u32 meta = __ldg(p.lane_meta + j * TEAM + threadIdx.x);
    r.row[j] = meta & kMetaOffMask;
    r.take[j] = meta >> kMetaCombineShift;
    r.thq[j] = (meta & kMetaHead) ? 0 : -1;
  }
  i8* const cur_w = p.cur_w + (size_t)chain * TSA_EPADA;
  i8* const cur_th = p.cur_th + (size_t)chain * TSA_NPADA;
  i8* const best_w = p.best_w + (size_t)chain * TSA_EPADA;
  i8* const best_th = p.best_th + (size_t)chain * TSA_NPADA;
  RowIO<0>::load(p, r, cur_w, cur_th, warp, lane);
  // three state buffers: t = 0 states (read only), then the two that alternate; dummies / holes stay 0
  for (int x = threadIdx.x; x < STATE_WORDS; x += TEAM) {
    smem[x] = __ldg(p.initw + x);
    smem[STATE_WORDS + x] = 0u;
    smem[2 * STATE_WORDS + x] = 0u;
  }
  const u32 sbase = (u32)__cvta_generic_to_shared(smem);
  u32* const red = smem + 3 * STATE_WORDS;
  // structural constraints (readings C1, C2): per node the number of non-zero in-edges,
  // non-zero out-edges and +1 in-edges of the chain's current vector, kept in shared memory behind the reduction
  // words; only the thread that holds the proposed weight reads or writes them, between two team barriers
  // (16-bit counters: a node's out-degree is bounded by N - 1 < 65 536 only, a hub may feed more than 255 nodes)
  unsigned short* const cin = (unsigned short*)(red + W);
  unsigned short* const cout = cin + TSA_NN;
  unsigned short* const cact = cout + TSA_NN;
  if (TSA_CONSTRAINED) {
    for (int i = threadIdx.x; i < TSA_NN; i += TEAM) {
      int a = 0, b = 0, c = 0;
      for (int x = __ldg(p.con_in_ptr + i); x < __ldg(p.con_in_ptr + i + 1); ++x) {
        const int v = cur_w[__ldg(p.con_in_slot + x)];
        a += v != 0; c += v == 1;
      }
      for (int x = __ldg(p.con_out_ptr + i); x < __ldg(p.con_out_ptr + i + 1); ++x) b += cur_w[__ldg(p.con_out_slot + x)] != 0;
      cin[i] = (unsigned short)a; cout[i] = (unsigned short)b; cact[i] = (unsigned short)c;
    }
  }

  u32 fcur = p.fit_cur[chain], fbest = p.fit_best[chain];
  const int trow = p.trace_row ? p.trace_row[chain] : -1;
  u64 level = p.g0 / (u64)p.steps_per_level;
  i64 left_in_level = p.steps_per_level - (i64)(p.g0 % (u64)p.steps_per_level);
  u64 st_steps = 0, st_acc = 0, st_worse = 0, st_best = 0;    // acceptance statistics of the level being run
  team_sync();

#pragma unroll 1
  for (i64 it = 0; it < p.steps; ++it) {
    const u64 g = p.g0 + (u64)it;
    u32 x[4];
    philox4x32_10((u32)g, (u32)(g >> 32), gchain, 0u, p.key0, p.key1, x);
    // a1 / a2: propose and apply in the registers of the one thread that holds the parameter
    const u32 pidx = __umulhi(x[0], (u32)TSA_NP);
    const bool is_w = pidx < (u32)TSA_NE;
    const u32 loc = is_w ? __ldg(p.wloc + pidx) : __ldg(p.thloc + (pidx - (u32)TSA_NE));
    const bool mine = (loc >> 16) == threadIdx.x;
    const int sel = mine ? (int)(loc & 0xFFu) : -1;
    u32 saved = 0u, code = 0u;
    bool moved = true;
    int dnz = 0, dact = 0, csrc = 0, cdst = 0;                          // constraint-counter changes if the move is accepted
    if (is_w) {
      const int sh = (int)((loc >> 8) & 3u) * 8;
#pragma unroll
      for (int i = 0; i < NWREG; ++i) if (i == sel) saved = r.w[i];
      const int oldv = (int)(saved << (24 - sh)) >> 24;
      int newv = (oldv + 2 + (int)__umulhi(x[1], 2u)) % 3 - 1;         // (code + 1 + r) mod 3 - 1, code = old + 1
      if (TSA_CONSTRAINED && mine) {
        // the two other values, listed cyclically after the old one; strike "to 0" if the edge is the target's only
        // non-zero in-edge or the source's only non-zero out-edge, "away from +1" if it is the target's only
        // activator; take entry mulhi(x1, length) of what is left; nothing left = null move
        const u32 en = __ldg(p.edge_nodes + pidx);
        csrc = (int)(en & 0xFFFFu); cdst = (int)(en >> 16);
        const bool bar_zero = oldv != 0 && (cin[cdst] == 1 || cout[csrc] == 1);
        const bool bar_nonplus = oldv == 1 && cact[cdst] == 1;
        int first = 2, second = 2;
#pragma unroll
        for (int k = 1; k <= 2; ++k) {
          const int v = (oldv + 1 + k) % 3 - 1;
          if (!((v == 0 && bar_zero) || (v != 1 && bar_nonplus))) { if (first == 2) first = v; else second = v; }
        }
        moved = first != 2;
        newv = !moved ? oldv : (second != 2 && __umulhi(x[1], 2u) != 0u) ? second : first;
        dnz = (newv != 0) - (oldv != 0); dact = (newv == 1) - (oldv == 1);
      }
      const u32 neww = (saved & ~(0xFFu << sh)) | (((u32)newv & 0xFFu) << sh);
#pragma unroll
      for (int i = 0; i < NWREG; ++i) if (i == sel) r.w[i] = neww;
      code = (u32)(newv + 1);
    } else {
#pragma unroll
      for (int j = 0; j < NT; ++j) if (j == sel) saved = (u32)r.thq[j];
      const int newq = ((int)saved + 1 + (int)__umulhi(x[1], (u32)(TSA_NPAIRS - 1))) % TSA_NPAIRS;
#pragma unroll
      for (int j = 0; j < NT; ++j) if (j == sel) set_threshold(p, r, j, newq);
      code = (u32)newq;
    }
    // a3 / a4
    const u32 fcand = simulate(p, r, sbase, red);
    // a5
    const u64 lv = level < (u64)(p.n_levels - 1) ? level : (u64)(p.n_levels - 1);
    const i64 d = (i64)fcand - (i64)fcur;
    bool acc = d <= 0;
    if (!acc && d <= (i64)p.dmax) acc = x[2] < __ldg(p.accept + lv * (u64)p.dmax + (u64)(d - 1));
    bool new_best = false;
    // a6
    if (acc) {
      fcur = fcand;
      if (TSA_CONSTRAINED && mine && is_w) {
        cin[cdst] = (unsigned short)(cin[cdst] + dnz); cout[csrc] = (unsigned short)(cout[csrc] + dnz);
        cact[cdst] = (unsigned short)(cact[cdst] + dact);
      }
      if (fcand < fbest) {
        fbest = fcand;
        new_best = true;
        RowIO<0>::store(r, best_w, best_th, warp, lane);
      }
    } else if (is_w) {
#pragma unroll
      for (int i = 0; i < NWREG; ++i) if (i == sel) r.w[i] = saved;
    } else {
#pragma unroll
      for (int j = 0; j < NT; ++j) if (j == sel) set_threshold(p, r, j, (int)saved);
    }
    if (trow >= 0 && mine) {
      const u64 idx = g - p.trace_g0;
      if (g >= p.trace_g0 && idx < (u64)p.trace_max)
        p.trace_rec[(size_t)trow * (size_t)p.trace_max + idx] =
            (u64)fcand | ((u64)pidx << 32) | ((u64)code << 56) | ((u64)(acc ? 1 : 0) << 60) | ((u64)(new_best ? 1 : 0) << 61) |
            ((u64)(moved ? 0 : 1) << 62);
    }
    if (p.level_stats) { st_steps += 1; st_acc += acc; st_worse += acc && d > 0; st_best += new_best; }
    if (--left_in_level == 0) {
      if (p.level_stats && level < (u64)(p.n_levels - 1)) {            // the last row absorbs the steps past the schedule
        if (threadIdx.x == 0) {
          atomicAdd(p.level_stats + lv * 4 + 0, st_steps); atomicAdd(p.level_stats + lv * 4 + 1, st_acc);
          atomicAdd(p.level_stats + lv * 4 + 2, st_worse); atomicAdd(p.level_stats + lv * 4 + 3, st_best);
        }
        st_steps = st_acc = st_worse = st_best = 0;
      }
      ++level; left_in_level = p.steps_per_level;
    }
  }
  if (p.level_stats && threadIdx.x == 0 && st_steps) {
    const u64 lv = level < (u64)(p.n_levels - 1) ? level : (u64)(p.n_levels - 1);
    atomicAdd(p.level_stats + lv * 4 + 0, st_steps); atomicAdd(p.level_stats + lv * 4 + 1, st_acc);
    atomicAdd(p.level_stats + lv * 4 + 2, st_worse); atomicAdd(p.level_stats + lv * 4 + 3, st_best);
  }
  // a7
  RowIO<0>::store(r, cur_w, cur_th, warp, lane);
  if (threadIdx.x == 0) { p.fit_cur[chain] = fcur; p.fit_best[chain] = fbest; }
}

}  // namespace tsa_static
