// sa_run kernel v4 / v5 (sm_100a), for networks of at most 128 nodes and 8 conditions: the node update
// of one time step is ONE dense int8 product on the tensor pipe instead of E shared-memory gathers,
//
//     sum[i][k] = SUM_j  W[i][j] * s[j][k]      (PAPER.md :66-70: the image of node i is a sum over its sources)
//
// with W the chain's N x N weight matrix (w_e at [dst(e)][src(e)], structural zeros elsewhere, padded
// to 16*MT x 32*KS) and s the N x K state matrix of all conditions at t-1.  One chain = one team of
// TW warps = one CTA; warp ww owns the row tiles of its NW/TW result words.  The team keeps the WHOLE
// of W in registers as mma.sync m16n8k32 A fragments (up to 2*NW/TW*KS*4 registers per thread) for
// the entire sa_run, every warp the states of t-1 as KS B fragments, and the team issues MT*KS IMMAs
// per time step (v5: the 2:4-sparse form, mma.sp m16n8k64 -- half the registers and half the IMMAs; the
// host permutes the nodes so that every row has at most two candidate edges per four columns).
// Two row tiles share one accumulator (v7): the states travel as the bytes 64*s (0x00 / 0x40 / 0x80, an
// unsigned B operand); the even tile of a pair multiplies s = (64*s) >> 6 by weights +-1, the odd tile
// multiplies 64*s by weights +-4, so its sums arrive 256-fold: one s32 holds two sums a byte apart,
// a word of four is ONE multiply-add of two accumulators, and only 2*MT accumulator registers are live.
// The words are thresholded with the same biased-byte trick as the gather kernel (bit 7 of word + A is
// [sum >= t_lo], bit 7 of word + A + D is [sum > t_hi]; three logic operations turn the two bits into
// the byte 64*s') and go through a 1-2 KB shared-memory buffer laid out so that every lane writes its
// result words with one vector store and reads its next B fragments with two vector loads (row <->
// column numbering chosen by the host, sa_dense_plan.cpp).
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
#define TSD_W 1
#define TSD_PH 1
#define TSD_CPB 8
#define TSD_REDERIVE 1
#define TSD_SP 1
#define TSD_SWZ 1
#define TSD_OBSW 2
#define TSD_TUNROLL 1
#define TSD_MOVM 1
#define TSD_FIXW_MASK 1
#endif
#ifndef TSD_MOVM
#define TSD_MOVM 0
#endif
#ifndef TSD_OBSW
#define TSD_OBSW TSD_KS
#endif
#ifndef TSD_CFOLD
#define TSD_CFOLD 0
#endif
#ifndef TSD_SPEC
#define TSD_SPEC 1
#endif
#ifndef TSD_SKIP
#define TSD_SKIP 0
#endif

#ifndef TSD_FIXW_MASK
#define TSD_FIXW_MASK 0
#endif
#ifndef TSD_IMMA_ORDER
#define TSD_IMMA_ORDER 0
#endif
#ifndef TSD_IMMA_VOLATILE
#define TSD_IMMA_VOLATILE 1
#endif
#if TSD_IMMA_VOLATILE
#define TSD_ASM_VOLATILE volatile
#else
#define TSD_ASM_VOLATILE
#endif
#ifndef TSD_CONSTRAINED
#define TSD_CONSTRAINED 0
#endif

namespace tsa_dense {

constexpr int MT = TSD_MT, KS = TSD_KS, NW = TSD_KS, T = TSD_T, NOBS = TSD_NOBS;
constexpr int CS = TSD_CS, TS = TSD_TS, NFIX = TSD_NFIX;
constexpr int TW = TSD_W, TEAM = TW * 32;       // warps / threads per chain
constexpr bool REDERIVE = TSD_REDERIVE != 0;    // tight register budget: derive the proposal twice rather than hold it over the time loop
// TSD_CFOLD: the biased thresholds 0x80 - t_lo enter as the C operand of the first IMMA of every accumulator (a quad
// of registers per result word, the two halves of the word TA twice), so the packed word already is x and the add
// of TA goes away.  An IMMA that reads a C quad instead of RZ costs more issue time than the add it saves on
// Mtb-shaped (149 against 164 M chain-steps/s); it gains 2 % where a chain has two IMMAs per step (HPG-shaped).
constexpr bool CFOLD = TSD_CFOLD != 0;
// bit (row tile * column steps + column step): that block of the weight matrix holds no candidate edge, so its IMMA
// is left out (the host numbers the nodes so that the few nodes of the last row tile take all their sources from one
// half of the columns: 13 instead of 14 IMMAs per time step on Mtb-shaped)
constexpr u32 kSkip = CFOLD ? 0u : (u32)TSD_SKIP;
constexpr int CPB = TSD_CPB;                    // chains per CTA (one-warp chains only), independent of one another: a CTA of
                                                // 4k warps puts k chains on every SM sub-partition, which 4k one-warp CTAs do not
constexpr int WPW = NW / TW;                    // result words per condition a lane produces
constexpr int MTW = 2 * WPW;                    // row tiles per warp (the last warp's may lie beyond MT)
constexpr int PH = TSD_PH, WPP = WPW / PH;       // phases of a time step, result words per phase
constexpr bool SP = TSD_SP != 0;                // 2:4-sparse A operand: mma.sp m16n8k64 (host guarantees <= 2 candidate edges per 4 columns)
constexpr int KSP = KS / 2;                     // sparse steps of 64 columns
constexpr int NA = SP ? MTW * KSP * 4 : MTW * KS * 4;   // A-fragment registers per thread
constexpr int NM = SP ? MTW * KSP : 1;          // selector (metadata) registers per thread
constexpr int kTUnroll = TSD_TUNROLL;           // unroll factor of the time loop
constexpr bool SWZ = TSD_SWZ != 0;              // swizzled exchange buffer (KS = 4, one warp per chain): conflict-free stores AND loads
// Register exchange (v8): the result words reach the next step's B fragments through MOVM (movmatrix, an 8 x 8
// transpose of 16-bit elements across the warp) instead of shared memory: no store, no barrier, no load.
constexpr bool MOVM = TSD_MOVM != 0;
constexpr u32 kFixW = TSD_FIXW_MASK;               // result words w that hold a clamped (condition, node) entry
__host__ __device__ constexpr int popc_below(u32 m, int w) { int n = 0; for (int i = 0; i < w; ++i) n += (int)((m >> i) & 1u); return n; }
constexpr int NFW = popc_below(kFixW, 32) > 0 ? popc_below(kFixW, 32) : 1;
constexpr int STATE_BYTES = MOVM ? 0 : SWZ ? 1024 : 8 * CS;   // one exchange buffer: 8 condition rows
constexpr int NBUF = TW > 1 ? 2 : 1;            // teams alternate between two exchange buffers: one barrier per time step
// Speculative look-ahead (TSD_SPEC = D > 1, one-warp chains): D warps hold the same chain and evaluate the proposals
// of the SA steps g .. g+D-1 against the same current vector at the same time; the steps up to and including the
// first accepted one are what the serial chain would have done (a rejected step leaves the vector unchanged, and
// proposal, level and random numbers of a step depend on (seed, chain, g) alone), so they are consumed and the rest
// is thrown away: bit-exact, 1 + r + r^2 + ... steps per pass at rejection rate r.  It pays where the chains
// are too few to fill the GPU (HPG-shaped: 1024 chains, 7 warps per SM); see run_spec below.
constexpr int SPEC = TSD_SPEC;
static_assert(SPEC >= 1 && SPEC <= 4 && (SPEC == 1 || TSD_W == 1), "look-ahead depth 1 .. 4, one-warp chains");
constexpr int RES_WORDS = SPEC > 1 ? 2 * SPEC : 0;      // per warp of a chain: its step's flags and candidate fitness
constexpr int XBYTES = NBUF * STATE_BYTES;              // exchange buffer(s) of one warp team
constexpr int CHAIN_SMEM = (SPEC * XBYTES + TSD_EPADA + TSD_NPADA + (2 * TW + 8 + RES_WORDS) * 4 + 15) / 16 * 16;   // bytes per chain
// The host numbers the observed nodes first, so only the result words w < OBSW hold scored entries; the observation
// words of a lane and time are stored w-major ([w][c]) and fetched with vector loads.
constexpr int OBSW = TSD_OBSW;
static_assert(OBSW >= 0 && OBSW <= NW, "scored words");
constexpr u64 kObsLo = TSD_OBSMASK_LO, kObsHi = TSD_OBSMASK_HI;
constexpr u32 kOnes = 0x01010101u, kTops = 0x80808080u;
constexpr int kImmaOrder = TSD_IMMA_ORDER;     // issue order of a phase's IMMAs: 0 word by word, 1 two words interleaved, 2 all words interleaved
constexpr int RPT = SP ? (KS / 2) * 4 : KS * 4; // A-fragment registers per row tile
constexpr bool kByteMism = NOBS * 2 * (OBSW > 0 ? OBSW : 1) <= 255;   // mismatch counters stay in byte lanes
// is time step t (1 .. T) scored?
__host__ __device__ constexpr bool obs_at(int t) { return t < 64 ? ((kObsLo >> t) & 1ull) != 0ull : ((kObsHi >> (t - 64)) & 1ull) != 0ull; }
// scored steps among 1 .. j-1
__host__ __device__ constexpr int obs_before(int j) { int n = 0; for (int t = 1; t < j; ++t) n += obs_at(t) ? 1 : 0; return n; }
__host__ __device__ constexpr bool obs_periodic() {
  if (T % kTUnroll != 0) return false;
  for (int t = 1; t + kTUnroll <= T; ++t) if (obs_at(t) != obs_at(t + kTUnroll)) return false;
  return true;
}
constexpr bool kObsPeriodic = obs_periodic();
static_assert(KS == 1 || KS == 2 || KS == 4, "KS must be 1, 2 or 4");
static_assert(!SP || KS % 2 == 0, "the sparse layout needs whole 64-column steps");
static_assert(!SWZ || (KS == 4 && TSD_W == 1), "the swizzled exchange buffer is for 16-byte units of one warp");
static_assert(2 * KS >= MT && MT >= 1, "row <-> column numbering needs MT <= 2*KS");
static_assert(!MOVM || TSD_W == 1, "the register exchange is for one warp per chain");
static_assert(WPW >= 1 && WPW * TW == NW, "team width must divide the words per condition");
static_assert(WPP >= 1 && WPP * PH == WPW, "phases must divide the words of a warp");
static_assert(CPB == 1 || (TW == 1 && CPB <= 16), "several chains per CTA: one-warp chains");
static_assert(TSD_SPEC == 1 || (TSD_CPB <= 15 && TSD_CPB * TSD_SPEC <= 32), "look-ahead: one named barrier per chain, at most 32 warps per CTA");
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

// (a >> 1) + b as one multiply-add (IMAD.HI: the FMA pipe has room, the ALU pipe does the logic operations)
__device__ __forceinline__ u32 half_plus(u32 a, u32 b) {
  u32 r;
  asm("mad.hi.u32 %0, %1, 0x80000000, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
// 8 x 8 transpose of 16-bit elements across the warp: lane (g, t) gives the elements (g, 2t), (g, 2t+1) and gets
// (2t, g), (2t+1, g) (SASS MOVM.16.MT88)
__device__ __forceinline__ u32 movm(u32 x) {
  u32 r;
  asm("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(r) : "r"(x));
  return r;
}

// D (16 x 8, s32) += A (16 x 32, s8, row) * B (32 x 8, u8, col)
__device__ __forceinline__ void imma(int (&c)[4], const u32* a, u32 b0, u32 b1) {
  asm TSD_ASM_VOLATILE("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// D (16 x 8, s32) += A (16 x 64, s8, 2:4 sparse: 16 x 32 stored + selectors e) * B (64 x 8, u8, col)
__device__ __forceinline__ void imma_sp(int (&c)[4], const u32* a, u32 b0, u32 b1, u32 b2, u32 b3, u32 e) {
  asm TSD_ASM_VOLATILE("mma.sp::ordered_metadata.sync.aligned.m16n8k64.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9,%10,%11}, {%0,%1,%2,%3}, %12, 0x0;"
               : "+r"(c[0]), "+r"(c[1]), "+r"(c[2]), "+r"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1), "r"(b2), "r"(b3), "r"(e));
}

// the same with a separate C operand (the first IMMA of an accumulator chain under CFOLD)
__device__ __forceinline__ void imma_c(int (&c)[4], const u32* a, u32 b0, u32 b1, const u32 (&ci)[4]) {
  asm TSD_ASM_VOLATILE("mma.sync.aligned.m16n8k32.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%11,%12,%13};"
               : "=r"(c[0]), "=r"(c[1]), "=r"(c[2]), "=r"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1), "r"(ci[0]), "r"(ci[1]), "r"(ci[2]), "r"(ci[3]));
}
__device__ __forceinline__ void imma_sp_c(int (&c)[4], const u32* a, u32 b0, u32 b1, u32 b2, u32 b3, u32 e, const u32 (&ci)[4]) {
  asm TSD_ASM_VOLATILE("mma.sp::ordered_metadata.sync.aligned.m16n8k64.row.col.s32.s8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9,%10,%11}, {%13,%14,%15,%16}, %12, 0x0;"
               : "=r"(c[0]), "=r"(c[1]), "=r"(c[2]), "=r"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1), "r"(b2), "r"(b3), "r"(e), "r"(ci[0]), "r"(ci[1]), "r"(ci[2]), "r"(ci[3]));
}

__device__ __forceinline__ void team_sync() {
  if (TW == 1) __syncwarp(); else __syncthreads();
}

// the SPEC warps that hold chain slot wc of the CTA (named barrier 1 + wc); one team otherwise
__device__ __forceinline__ void group_sync(int wc) {
  if (SPEC == 1) team_sync();
  else asm volatile("bar.sync %0, %1;" ::"r"(1 + wc), "n"(32 * TSD_SPEC) : "memory");
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
// shared memory through 32-bit shared-window addresses, up to four words at a time
__device__ __forceinline__ void lds_vec(u32 a, u32 (&s)[1]) { smem_check(a, 4); asm volatile("ld.shared.u32 %0, [%1];" : "=r"(s[0]) : "r"(a) : "memory"); }
__device__ __forceinline__ void lds_vec(u32 a, u32 (&s)[2]) { smem_check(a, 8); asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(s[0]), "=r"(s[1]) : "r"(a) : "memory"); }
__device__ __forceinline__ void lds_vec(u32 a, u32 (&s)[4]) {
  smem_check(a, 16);
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(s[0]), "=r"(s[1]), "=r"(s[2]), "=r"(s[3]) : "r"(a) : "memory");
}
__device__ __forceinline__ void sts_vec(u32 a, const u32 (&s)[1]) { smem_check(a, 4); asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(s[0]) : "memory"); }
__device__ __forceinline__ void sts_vec(u32 a, const u32 (&s)[2]) { smem_check(a, 8); asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(a), "r"(s[0]), "r"(s[1]) : "memory"); }
__device__ __forceinline__ void sts_vec(u32 a, const u32 (&s)[4]) {
  smem_check(a, 16);
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(s[0]), "r"(s[1]), "r"(s[2]), "r"(s[3]) : "memory");
}
__device__ __forceinline__ void sts_u8(u32 a, u32 v) { smem_check(a, 1); asm volatile("st.shared.u8 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }

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
  u32 M[NM];        // sparse layout: selector words of the warp's tiles (the same for every chain)
  u32 TA[CFOLD ? 1 : WPW];      // per byte (one row of this thread group): 0x80 - t_lo, padding rows 0
  u32 TB[WPW];      // TA minus, per byte: t_hi - t_lo + 1 (padding rows 0); CFOLD: only that difference
  u32 CI[CFOLD ? WPW : 1][4];   // CFOLD: TA & 0xFFFF twice, TA >> 16 twice
  u32 fix[MOVM ? 2 * NFW : NFIX];    // clamp fix-ups of this lane (entries of the warp's own rows): bit 31 valid, 0-23 shared address of the byte
  u32 fixv[MOVM ? 2 * NFW : NFIX];   // the byte to store there, 64 * value
                    // register exchange: fix[2f + c] = bytes to keep, fixv[2f + c] = bytes 64 * value to set, of result word
                    // (c, w) for the f-th w in kFixW
};

// One phase of a time step: the IMMAs of the row-tile pairs behind result words [P*WPP, (P+1)*WPP) of this
// warp -- word w is the pair (2w, 2w+1): the even tile takes the states s and weights +-1, the odd tile the
// bytes 64*s and weights +-4, both into ONE accumulator, so that accumulator register c holds
// sum(tile 2w, row g) + 256 * sum(tile 2w+1, row g) and register 2+c the same for row g+8 -- then the word
// acc[c] + 65536 * acc[2+c] on top of the biased thresholds, the two sign tests, the byte 64*s' per row,
// the score against the observation words (a4) and the store.  Phases run one after the other.
template <int P>
struct Phases {
  // IMMA number `step` (0 .. 2*KK-1) of word w's accumulator chain: KK sparse / dense column steps of the even
  // tile on the plain states, then KK of the odd tile on the 64-fold states
  template <int KK>
  static __device__ __forceinline__ void one(const Regs& r, const u32 (&bh)[2 * KS], const u32 (&bl)[2 * KS], int n_tiles,
                                             int (&acc)[4], int w, int step) {
    // (with an even number of row tiles the odd tile of a pair goes first: it takes the exchanged bytes as they are,
    // and the shift that makes the even tile's operand is off the chain's critical path)
    constexpr bool kOddFirst = MT % 2 == 0 && TSD_W == 1;
    const int odd = kOddFirst ? 1 - step / KK : step / KK;
    const int tile = 2 * (P * WPP + w) + odd, s = step % KK;
    if (!(TW * MTW <= MT || tile < n_tiles)) return;
    if ((kSkip >> (tile * KK + s)) & 1u) return;
    const u32* bb = odd ? bh : bl;
    if (CFOLD && step == 0) {
      if (SP) imma_sp_c(acc, &r.A[(tile * KSP + s) * 4], bb[4 * s], bb[4 * s + 1], bb[4 * s + 2], bb[4 * s + 3], r.M[SP ? tile * KSP + s : 0], r.CI[CFOLD ? P * WPP + w : 0]);
      else imma_c(acc, &r.A[(tile * KS + s) * 4], bb[2 * s], bb[2 * s + 1], r.CI[CFOLD ? P * WPP + w : 0]);
      return;
    }
    if (SP) imma_sp(acc, &r.A[(tile * KSP + s) * 4], bb[4 * s], bb[4 * s + 1], bb[4 * s + 2], bb[4 * s + 3], r.M[SP ? tile * KSP + s : 0]);
    else imma(acc, &r.A[(tile * KS + s) * 4], bb[2 * s], bb[2 * s + 1]);
  }
  static __device__ __forceinline__ void run(const Regs& r, const u32 (&bh)[2 * KS], const u32 (&bl)[2 * KS], int n_tiles, bool is_obs,
                                             const u32 (&ov)[2 * WPW], int ww, u32& cnt, bool store, u32 st, u32 st1, u32 (&nb)[2 * KS]) {
    constexpr int W0 = P * WPP, KK = SP ? KSP : KS, NSTEP = 2 * KK;
    int acc[WPP][4];
#pragma unroll
    for (int w = 0; w < WPP; ++w) { acc[w][0] = 0; acc[w][1] = 0; acc[w][2] = 0; acc[w][3] = 0; }
    constexpr int GRP = kImmaOrder == 0 ? 1 : kImmaOrder == 1 ? 2 : WPP;     // words whose chains are interleaved
#pragma unroll
    for (int w0 = 0; w0 < WPP; w0 += GRP)
#pragma unroll
      for (int step = 0; step < NSTEP; ++step)
#pragma unroll
        for (int w = w0; w < w0 + GRP && w < WPP; ++w) one<KK>(r, bh, bl, n_tiles, acc[w], w, step);
    u32 ns[2][WPP];
#pragma unroll
    for (int w = 0; w < WPP; ++w)
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const u32 pk = (u32)acc[w][c] + ((u32)acc[w][2 + c] << 16);
        const u32 x = CFOLD ? pk : pk + r.TA[CFOLD ? 0 : W0 + w], y = pk + r.TB[W0 + w];      // bit 7 of a byte: [sum >= t_lo], [sum > t_hi]
        ns[c][w] = half_plus((x ^ y) & kTops, y & kTops);            // 0x40 = exactly one of them (the first), 0x80 = both
      }
    if (is_obs) {
#pragma unroll
      for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int w = 0; w < WPP; ++w) {
          if (TW == 1 ? W0 + w >= OBSW : ww * WPW + W0 + w >= OBSW) continue;      // no scored entry in this word
          const u32 z = ns[c][w] ^ ov[2 * (W0 + w) + c];                             // bits 6 and 7 of every byte
          cnt = __umulhi((z | (z + z)) & kTops, 1u << 25) + cnt;                     // + [byte != 0] = (bit 7 | bit 6) >> 7
        }
    }
    if (MOVM) {
      // Word (c, w) of lane (g, t) holds rows g, g+8 of the tiles 2w, 2w+1 (bytes: 2w/g, 2w+1/g, 2w/g+8, 2w+1/g+8)
      // under condition 2t + c.  The low halves of the words c = 0, 1 side by side are the elements (g, 2t), (g, 2t+1)
      // of an 8 x 8 matrix [thread group][condition] of row pairs; its transpose gives lane (g', t') the pairs of
      // the thread groups 2t', 2t'+1 under condition g': B-fragment word 2w of that lane (the high halves: word
      // 2w+1) in the column numbering of sa_dense_plan.cpp.  Clamped entries are set before they travel.
#pragma unroll
      for (int w = 0; w < WPP; ++w) {
        u32 n0 = ns[0][w], n1 = ns[1][w];
        if ((kFixW >> (W0 + w)) & 1u) {
          const int f = popc_below(kFixW, W0 + w);
          n0 = (n0 & r.fix[2 * f]) | r.fixv[2 * f];
          n1 = (n1 & r.fix[2 * f + 1]) | r.fixv[2 * f + 1];
        }
        nb[2 * (W0 + w)] = movm(__byte_perm(n0, n1, 0x5410));
        nb[2 * (W0 + w) + 1] = movm(__byte_perm(n0, n1, 0x7632));
      }
    } else if (store) {
      sts_vec(st + W0 * 4, ns[0]);
      sts_vec(st1 + W0 * 4, ns[1]);
    }
    Phases<P + 1>::run(r, bh, bl, n_tiles, is_obs, ov, ww, cnt, store, st, st1, nb);
  }
};
template <>
struct Phases<PH> {
  static __device__ __forceinline__ void run(const Regs&, const u32 (&)[2 * KS], const u32 (&)[2 * KS], int, bool, const u32 (&)[2 * WPW], int, u32&,
                                             bool, u32, u32, u32 (&)[2 * KS]) {}
};

// a3 + a4 for the parameters now in registers: returns the team's mismatch count.
// sbuf = shared address of the exchange buffer(s), red = the team's reduction words [2][TW].
__device__ __forceinline__ u32 simulate(const Params& p, const Regs& r, u32 sbuf, volatile u32* red, int parity, int lane, int ww) {
  const int g = lane >> 2, t4 = lane & 3;
  // Exchange buffer.  Plain layout: condition rows of CS bytes, thread chunks of TS bytes (strides from
  // the host's conflict search).  Swizzled layout (16-byte units, unit (c, t', half) = the words
  // 4*half .. 4*half+3 of chunk t' of condition c): 128-byte row 4*half + c/2, 16-byte column
  // 4*(t'&1) + (c/2 + 2*(t'/2) + (c&1)) mod 4 -- a Latin square, so that the eight lanes of a quarter
  // warp hit eight different columns both when they store (c/2 and t'&1 vary) and when they load
  // (c&1, t'/2 and t'&1 vary).
  u32 st_addr = 0u, st_delta = 0u, ld_addr = 0u;
  if (MOVM) {
  } else if (SWZ) {
    const int tq = g & 3, half = g >> 2;
    const int q0 = 4 * (tq & 1) + ((t4 + 2 * (tq >> 1)) & 3), q1 = 4 * (tq & 1) + ((t4 + 2 * (tq >> 1) + 1) & 3);
    st_addr = sbuf + (u32)((4 * half + t4) * 128 + q0 * 16);
    st_delta = (u32)((q1 - q0) * 16);
    ld_addr = sbuf + (u32)((g >> 1) * 128 + (4 * (t4 & 1) + (((g >> 1) + 2 * (t4 >> 1) + (g & 1)) & 3)) * 16);
  } else {
    st_addr = sbuf + (u32)((2 * t4) * CS + (g & 3) * TS + ((g >> 2) * NW + ww * WPW) * 4);
    st_delta = (u32)CS;
    ld_addr = sbuf + (u32)(g * CS + t4 * TS);
  }
  if (!MOVM) asm volatile("" : "+r"(st_addr), "+r"(ld_addr));      // keep them in registers (no S2R in the loop)
  if (!MOVM && SWZ) asm volatile("" : "+r"(st_delta));
  const int n_tiles = MT - ww * MTW;                      // row tiles of this warp that exist (warp-uniform)
  u32 b[2 * KS];
  {
    const u32* src = p.init_frag + lane * 2 * KS;
#pragma unroll
    for (int i = 0; i < 2 * KS; ++i) b[i] = __ldg(src + i);
  }
  u32 mis = 0u;
  int oj_run = 0;
  // blocks of kTUnroll time steps; when the observation times repeat with that period, which steps of a
  // block are scored (and the index of their observation words) is known at compile time
#pragma unroll 1
  for (int tb = 0; tb < T; tb += kTUnroll)
#pragma unroll
  for (int j = 1; j <= kTUnroll; ++j) {
    const int t = tb + j;
    if (T % kTUnroll != 0 && t > T) break;
    const bool is_obs = kObsPeriodic ? obs_at(j) : obs_at(t);
    const int oj = kObsPeriodic ? tb / kTUnroll * obs_before(kTUnroll + 1) + obs_before(j) : oj_run;
    // observation words of this lane and time: [w][c], this warp's words first at 2 * ww * WPW
    const u32* ow = p.obs_word + ((size_t)oj * 32 + lane) * (2 * NW) + 2 * ww * WPW;
    u32 ov[2 * WPW];
    if (is_obs) {
      if (TW == 1) {
        constexpr int VW = 2 * NW >= 4 ? 4 : 2;                 // words per vector load (a lane's 2 * NW words are that aligned)
#pragma unroll
        for (int v = 0; v * VW < 2 * OBSW; ++v) {
          if (VW == 4) {
            const uint4 q = __ldg((const uint4*)ow + v);
            ov[4 * v] = q.x; ov[4 * v + 1] = q.y; ov[4 * v + 2] = q.z; ov[4 * v + 3] = q.w;
          } else {
            const uint2 q = __ldg((const uint2*)ow + v);
            ov[2 * v] = q.x; ov[2 * v + 1] = q.y;
          }
        }
      } else {
#pragma unroll
        for (int i = 0; i < 2 * WPW; ++i) if (ww * WPW + i / 2 < OBSW) ov[i] = __ldg(ow + i);
      }
    }
    const u32 boff = NBUF == 2 ? (u32)((kTUnroll % 2 == 0 ? j : t) & 1) * STATE_BYTES : 0u;
    u32 cnt = 0u;                                         // per byte at most 2*WPW <= 8
    if (TW == 1 && !MOVM) __syncwarp();   // every lane has its B fragments out of the single buffer
    u32 bl[2 * KS];                       // the plain states 0 / 1 / 2 for the even tiles
#pragma unroll
    for (int i = 0; i < 2 * KS; ++i) bl[i] = b[i] >> 6;
    // (the last step's states are exchanged like all others although nobody reads them: no test in the loop)
    u32 nb[2 * KS];
    Phases<0>::run(r, b, bl, n_tiles, is_obs, ov, ww, cnt, true, st_addr + boff, st_addr + st_delta + boff, nb);
    if (is_obs) {
      if (kByteMism) mis += cnt; else mis += __dp4a(cnt, kOnes, 0u);
      ++oj_run;
    }
    if (MOVM) {
#pragma unroll
      for (int i = 0; i < 2 * KS; ++i) b[i] = nb[i];
      continue;
    }
    __syncwarp();
#pragma unroll
    for (int f = 0; f < NFIX; ++f)
      if (r.fix[f] >> 31) sts_u8((r.fix[f] & 0xFFFFFFu) + boff, r.fixv[f]);
    team_sync();
    u32 lo[NW], hi[NW];
    lds_vec(ld_addr + boff, lo);
    lds_vec(ld_addr + boff + (SWZ ? 512 : NW * 4), hi);
#pragma unroll
    for (int i = 0; i < NW; ++i) { b[i] = lo[i]; b[NW + i] = hi[i]; }
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

// a1: the proposal of step gs, as seen by this thread.
struct Proposal {
  u32 x2, pidx, loc, slot, wx;
  int oldv, newv, wsel;
  bool is_w, mine, moved;
};

// GetCandidate for a weight under the structural constraints (readings C1, C2), by
// the lane that holds the weight: the two other values are listed cyclically after the old one; "to 0" is struck
// if the edge is the target's only non-zero in-edge or the source's only non-zero out-edge, "away from +1" if it
// is the target's only activator; the new value is entry mulhi(x1, length) of what is left; nothing left = null
// move (the old value).  cw = the chain's canonical weight row.
__device__ __noinline__ int constrained_weight(const Params& p, const i8* cw, u32 pidx, int oldv, u32 x1, bool* moved) {
  bool bar_zero = false, bar_nonplus = false;
  if (oldv != 0) {
    const u32 en = __ldg(p.edge_nodes + pidx);
    const int src = (int)(en & 0xFFFFu), dst = (int)(en >> 16);
    int in_nz = 0, act = 0, out_nz = 0;
    for (int x = __ldg(p.con_in_ptr + dst); x < __ldg(p.con_in_ptr + dst + 1); ++x) {
      const int v = cw[__ldg(p.con_in_slot + x)];
      in_nz += v != 0; act += v == 1;
    }
    for (int x = __ldg(p.con_out_ptr + src); x < __ldg(p.con_out_ptr + src + 1); ++x) out_nz += cw[__ldg(p.con_out_slot + x)] != 0;
    bar_zero = in_nz == 1 || out_nz == 1;
    bar_nonplus = oldv == 1 && act == 1;
  }
  int first = 2, second = 2;                             // 2 = struck
#pragma unroll
  for (int k = 1; k <= 2; ++k) {
    const int v = (oldv + 1 + k) % 3 - 1;
    if (!((v == 0 && bar_zero) || (v != 1 && bar_nonplus))) { if (first == 2) first = v; else second = v; }
  }
  *moved = first != 2;
  if (first == 2) return oldv;
  return (second != 2 && __umulhi(x1, 2u) != 0u) ? second : first;
}

__device__ __forceinline__ Proposal propose(const Params& p, u64 gs, u32 gchain, int lane, int ww, int g, const i8* cw, const i8* cth) {
  Proposal q;
  u32 x[4];
  philox4x32_10((u32)gs, (u32)(gs >> 32), gchain, 0u, p.key0, p.key1, x);
  q.x2 = x[2];
  q.pidx = __umulhi(x[0], (u32)TSD_NP);
  q.is_w = q.pidx < (u32)TSD_NE;
  q.loc = q.is_w ? __ldg(p.wloc + q.pidx) : __ldg(p.thloc + (q.pidx - (u32)TSD_NE));
  q.slot = q.loc >> 16;
  q.oldv = 0; q.newv = 0; q.wsel = -1; q.wx = 0u; q.moved = true;
  if (q.is_w) {
    q.mine = ((q.loc >> 9) & 31u) == (u32)lane && ((q.loc >> 14) & 3u) == (u32)ww;
    if (q.mine) {
      q.oldv = cw[q.slot];
      if (TSD_CONSTRAINED) q.newv = constrained_weight(p, cw, q.pidx, q.oldv, x[1], &q.moved);
      else q.newv = (q.oldv + 2 + (int)__umulhi(x[1], 2u)) % 3 - 1;      // (code + 1 + r) mod 3 - 1, code = old + 1
      q.wsel = (int)(q.loc & 0x7Fu);
      // the byte holds w (even row tiles) or 4w (odd ones)
      q.wx = (((u32)(q.oldv ^ q.newv) << (((u32)q.wsel / (u32)RPT & 1u) * 2u)) & 0xFFu) << (8 * ((q.loc >> 7) & 3u));
    }
  } else {
    q.mine = (q.loc & 7u) == (u32)g && (int)((q.loc >> 3) & 3u) / WPW == ww;
    if (q.mine) {
      q.oldv = cth[q.slot];
      q.newv = (q.oldv + 1 + (int)__umulhi(x[1], (u32)(TSD_NPAIRS - 1))) % TSD_NPAIRS;
    }
  }
  return q;
}

// threshold bytes of the row at `loc` go from pair `from` to pair `to`
__device__ __forceinline__ void shift_threshold(const Params& p, Regs& r, u32 loc, int from, int to) {
  const int w = (int)((loc >> 3) & 3u) % WPW, sh = 8 * (int)((loc >> 5) & 3u);
  const u32 da = (u32)((int)p.tha[to] - (int)p.tha[from]) << sh;
  const u32 dd = (u32)(((int)p.tha[from] - (int)p.thb[from]) - ((int)p.tha[to] - (int)p.thb[to])) << sh;
#pragma unroll
  for (int i = 0; i < WPW; ++i)
    if (i == w) {
      if (CFOLD) {
        const u32 ta = r.CI[CFOLD ? i : 0][0] + (r.CI[CFOLD ? i : 0][2] << 16) + da;
        r.CI[CFOLD ? i : 0][0] = ta & 0xFFFFu; r.CI[CFOLD ? i : 0][1] = ta & 0xFFFFu;
        r.CI[CFOLD ? i : 0][2] = ta >> 16; r.CI[CFOLD ? i : 0][3] = ta >> 16;
        r.TB[i] += dd;
      } else {
        r.TA[CFOLD ? 0 : i] += da; r.TB[i] += da + dd;
      }
    }
}

__device__ __forceinline__ void run_piece(const Params& p, u32 chain, i64 s0, i64 s1, u32* smem, int tix, int wc, int sd);


// add the piece's counts of level ctl[6] to the handle's table and clear them (one thread per chain)
__device__ __noinline__ void flush_stats(const Params& p, volatile u32* ctl) {
  if (ctl[2] != 0u) {
#pragma unroll
    for (int k = 0; k < 4; ++k) atomicAdd(p.level_stats + (size_t)ctl[6] * 4 + k, (u64)ctl[2 + k]);
  }
  ctl[2] = 0u; ctl[3] = 0u; ctl[4] = 0u; ctl[5] = 0u;
}

extern "C" __global__ void __launch_bounds__(TEAM * CPB * SPEC, TSD_MINBLOCKS) tsa_run_dense(const __grid_constant__ Params p) {
  extern __shared__ __align__(16) u32 smem_all[];
  const int tix = threadIdx.x % TEAM;                                 // thread within the chain's team
  const int wc = threadIdx.x / (TEAM * SPEC), sd = threadIdx.x / TEAM % SPEC;   // chain slot within the CTA, look-ahead position
  const u32 chain = blockIdx.x * CPB + wc;
  if (p.slot_steps == 0 && chain >= (u32)p.R) return;
  u32* const smem = smem_all + (size_t)wc * (CHAIN_SMEM / 4);
  // one chain per slot (slot_steps == 0), or balanced slots: this slot owns [lo, hi) of the line of
  // R*steps chain-steps and visits the chains ca .. cb it touches, one piece each
  // (the slot's bounds are derived again for every piece, from an opaque copy of the slot index, so
  // that they do not occupy registers across the time loop)
#pragma unroll 1
  for (int n = 0;; ++n) {
    u32 slot = chain;
    asm volatile("" : "+r"(slot));
    const i64 S = p.steps, total = (i64)p.R * S;
    const i64 lo = p.slot_steps == 0 ? (i64)slot * S : (i64)slot * p.slot_steps;
    const i64 hi = p.slot_steps == 0 ? lo + S : (lo + p.slot_steps < total ? lo + p.slot_steps : total);
    if (lo >= total) return;
    const i64 ca = lo / S, cb = (hi - 1) / S;
    const int count = (int)(cb - ca) + 1;
    if (n >= count) return;
    const bool head_first = cb > ca && hi < (cb + 1) * S;
    const i64 c = n == count - 1 ? ca : head_first ? (n == 0 ? cb : ca + n) : ca + 1 + n;
    const i64 b0 = c * S;
    run_piece(p, (u32)c, (lo > b0 ? lo : b0) - b0, (hi < b0 + S ? hi : b0 + S) - b0, smem, tix, wc, sd);
  }
}


// temperature level of SA step gs (reading 20)
__device__ __forceinline__ u64 level_of(const Params& p, u64 gs) {
  u64 level = ((gs | (u64)p.steps_per_level) >> 32) == 0 ? (u64)((u32)gs / (u32)p.steps_per_level) : gs / (u64)p.steps_per_level;
  if (level > (u64)(p.n_levels - 1)) level = (u64)(p.n_levels - 1);
  return level;
}

// The SA steps [s0, s1) of one chain with look-ahead (SPEC warps per chain, this one at position sd).  One pass:
// warp sd proposes and scores step it + sd against the current vector and posts (live, accepted, fitness); after the
// first barrier every warp knows the first accepted position a and the number of steps consumed (a + 1, or all live
// ones); warps other than a take their own change back and, if there is an a, apply step it + a's change to their
// registers (derived again from the canonical rows, which are still the old ones); after the second barrier warp a
// commits to the canonical rows and control words; the consumed warps write their trace records, warp 0 keeps the
// level statistics; the third barrier ends the pass.
__device__ __forceinline__ void run_spec(const Params& p, Regs& r, u32 chain, u32 gchain, i64 s0, i64 s1, u32 sbuf, i8* cw, i8* cth,
                                         volatile u32* red, volatile u32* ctl, int lane, int wc, int sd) {
  const int g = lane >> 2, t4 = lane & 3;
  volatile u32* const res = ctl + 8;                     // [2 * position] bit 1 live, bit 0 accepted; [2 * position + 1] candidate fitness
  const int trow = p.trace_row ? __ldg(p.trace_row + chain) : -1;
#pragma unroll 1
  for (i64 it = s0; it < s1;) {
    const i64 my = it + sd;
    const bool live = my < s1;                           // warp-uniform
    const u32 fcur = ctl[0], fbest = ctl[1];
    Proposal q;
    u32 fcand = 0u;
    bool acc = false;
    i64 d = 0;
    if (live) {
      q = propose(p, p.g0 + (u64)my, gchain, lane, 0, g, cw, cth);
      if (q.is_w) xor_reg(r.A, q.wsel, q.wx);
      else if (q.mine) shift_threshold(p, r, q.loc, q.oldv, q.newv);
      fcand = simulate(p, r, sbuf, red, 0, lane, 0);
      d = (i64)fcand - (i64)fcur;
      acc = d <= 0;
      if (!acc && d <= (i64)p.dmax) acc = q.x2 < __ldg(p.accept + level_of(p, p.g0 + (u64)my) * (u64)p.dmax + (u64)(d - 1));
    }
    if (lane == 0) { res[2 * sd] = live ? (acc ? 3u : 2u) : 0u; res[2 * sd + 1] = fcand; }
    group_sync(wc);
    int a = -1, consumed = 0;
#pragma unroll
    for (int j = 0; j < SPEC; ++j) {
      const u32 f = res[2 * j];
      if (a < 0 && consumed == j && (f & 2u)) { consumed = j + 1; if (f & 1u) a = j; }
    }
    if (live && sd != a) {                               // not the accepted step: the change is taken back
      if (q.is_w) xor_reg(r.A, q.wsel, q.wx);
      else if (q.mine) shift_threshold(p, r, q.loc, q.newv, q.oldv);
    }
    if (a >= 0 && sd != a) {                             // the accepted step's change, from the still unchanged canonical rows
      const Proposal qa = propose(p, p.g0 + (u64)(it + a), gchain, lane, 0, g, cw, cth);
      if (qa.is_w) xor_reg(r.A, qa.wsel, qa.wx);
      else if (qa.mine) shift_threshold(p, r, qa.loc, qa.oldv, qa.newv);
    }
    if (p.level_stats && sd == 0 && lane == 0) {
      for (int j = 0; j < consumed; ++j) {
        const u32 lv = (u32)level_of(p, p.g0 + (u64)(it + j)), fj = res[2 * j + 1];
        if (lv != ctl[6]) { flush_stats(p, ctl); ctl[6] = lv; }
        ctl[2] += 1u;
        if (j == a) { ctl[3] += 1u; ctl[4] += fj > fcur ? 1u : 0u; ctl[5] += fj < fbest ? 1u : 0u; }
      }
    }
    group_sync(wc);                                      // everyone has read the canonical rows and the control words
    const bool new_best = sd == a && fcand < fbest;
    if (sd == a) {
      if (lane == 0) { ctl[0] = fcand; if (new_best) ctl[1] = fcand; }
      if (q.mine) {
        if (q.is_w) cw[q.slot] = (i8)q.newv;
        else if (t4 == 0) cth[q.slot] = (i8)q.newv;
      }
      if (new_best) {
        __syncwarp();
        u32* const best_w = (u32*)(p.best_w + (size_t)chain * TSD_EPADA);
        u32* const best_th = (u32*)(p.best_th + (size_t)chain * TSD_NPADA);
        for (int i = lane; i < TSD_EPADA / 4; i += 32) best_w[i] = ((const u32*)cw)[i];
        for (int i = lane; i < TSD_NPADA / 4; i += 32) best_th[i] = ((const u32*)cth)[i];
      }
    }
    if (trow >= 0 && sd < consumed && q.mine && (q.is_w || t4 == 0)) {
      const u64 gs = p.g0 + (u64)my, idx = gs - p.trace_g0;
      const u32 code = q.is_w ? (u32)(q.newv + 1) : (u32)q.newv;
      if (gs >= p.trace_g0 && idx < (u64)p.trace_max)
        p.trace_rec[(size_t)trow * (size_t)p.trace_max + idx] =
            (u64)fcand | ((u64)q.pidx << 32) | ((u64)code << 56) | ((u64)(sd == a ? 1 : 0) << 60) | ((u64)(new_best ? 1 : 0) << 61) |
            ((u64)(q.moved ? 0 : 1) << 62);
    }
    group_sync(wc);                                      // the commit is visible
    it += consumed;
  }
}

// One piece of one chain's run: stage the chain (a0), advance it through steps [s0, s1) of this
// launch, write it back (a7).  A launch normally gives every chain one piece, [0, steps); when there
// are more chains than resident slots the host splits the (chain, step) line evenly over the slots
// (slot_steps > 0), and a chain that straddles two slots is handed over through HBM: the slot that
// runs its head does so FIRST and raises flags[chain]; the next slot runs the tail LAST.
__device__ __forceinline__ void run_piece(const Params& p, u32 chain, i64 s0, i64 s1, u32* smem, int tix, int wc, int sd) {
  const int lane = tix & 31, ww = tix >> 5, g = lane >> 2, t4 = lane & 3;
  const u32 gchain = p.chain_id_base + chain;
  // shared memory of this chain: exchange buffer(s) (one set per look-ahead warp), canonical weight and threshold rows,
  // reduction and control words, look-ahead results
  i8* const cw = (i8*)smem + SPEC * XBYTES;
  i8* const cth = cw + TSD_EPADA;
  volatile u32* const red = (volatile u32*)(cth + TSD_NPADA);
  u32* const xbuf = smem + (SPEC > 1 ? sd * (XBYTES / 4) : 0);
  const u32 sbuf = (u32)__cvta_generic_to_shared(xbuf);
  // (row addresses are formed where they are used, never held across the time loop)

  if (s0 > 0) {                              // the head of this chain is another slot's first piece
    if (tix == 0) {
      // the launch is cooperative (every slot is resident) and a head piece never waits, so this wait ends;
      // it is bounded all the same (about 2^26 x 200 ns) and reports instead of hanging the device
      u32 spins = 0u;
      while (*(volatile u32*)(p.flags + chain) == 0u) {
        __nanosleep(200);
        if (++spins > (1u << 26)) { atomicExch(p.err, 1u); break; }
      }
      __threadfence();
    }
    team_sync();
  }
  // a0: stage the chain
  for (int x = tix; x < XBYTES / 4; x += TEAM) xbuf[x] = 0u;
  if (SPEC == 1 || sd == 0) {
    for (int x = tix; x < TSD_EPADA / 4; x += TEAM) ((u32*)cw)[x] = __ldcg((const u32*)(p.cur_w + (size_t)chain * TSD_EPADA) + x);
    for (int x = tix; x < TSD_NPADA / 4; x += TEAM) ((u32*)cth)[x] = __ldcg((const u32*)(p.cur_th + (size_t)chain * TSD_NPADA) + x);
  }
  group_sync(wc);
  Regs r;
#pragma unroll
  for (int i = 0; i < NA; ++i) {
    const uint2 fs = __ldg((const uint2*)p.frag_slot + (ww * NA + i) * 32 + lane);
    const u32 o0 = fs.x & 0xFFFFu, o1 = fs.x >> 16, o2 = fs.y & 0xFFFFu, o3 = fs.y >> 16;
    const u32 b0 = o0 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o0];
    const u32 b1 = o1 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o1];
    const u32 b2 = o2 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o2];
    const u32 b3 = o3 == 0xFFFFu ? 0u : (u32)(unsigned char)cw[o3];
    const u32 wv = b0 | (b1 << 8) | (b2 << 16) | (b3 << 24);
    r.A[i] = (i / RPT) & 1 ? (wv << 2) & 0xFCFCFCFCu : wv;       // odd row tiles hold 4w
  }
#pragma unroll
  for (int i = 0; i < NM; ++i) r.M[i] = SP ? __ldg(p.meta + (ww * NM + i) * 32 + lane) : 0u;
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
    if (CFOLD) {
      r.CI[CFOLD ? w : 0][0] = ta & 0xFFFFu; r.CI[CFOLD ? w : 0][1] = ta & 0xFFFFu;
      r.CI[CFOLD ? w : 0][2] = ta >> 16; r.CI[CFOLD ? w : 0][3] = ta >> 16;
      asm volatile("" : "+r"(r.CI[CFOLD ? w : 0][0]), "+r"(r.CI[CFOLD ? w : 0][1]), "+r"(r.CI[CFOLD ? w : 0][2]), "+r"(r.CI[CFOLD ? w : 0][3]));
      r.TB[w] = td;
    } else {
      r.TA[CFOLD ? 0 : w] = ta; r.TB[w] = ta + td;
    }
  }
  if (MOVM) {
#pragma unroll
    for (int f = 0; f < 2 * NFW; ++f) {
      r.fix[f] = __ldg(p.fix + (2 * f) * 32 + lane);
      r.fixv[f] = __ldg(p.fix + (2 * f + 1) * 32 + lane);
    }
  } else {
#pragma unroll
    for (int f = 0; f < NFIX; ++f) {
      const u32 raw = __ldg(p.fix + (ww * NFIX + f) * 32 + lane);
      r.fix[f] = (raw & 0x80000000u) | (sbuf + (raw & 0xFFFFu));
      r.fixv[f] = ((raw >> 16) & 3u) << 6;
    }
  }

  // Chain control words live in shared memory and the proposal is derived a second time after the
  // simulation (from the step counter alone), so that nothing but the loop counter stays in
  // registers across the time loop: the register budget there decides warps per SM.
  volatile u32* const ctl = red + 2 * TW;               // [0] d_cur, [1] d_best, [2..5] steps / accepted / accepted worse / new best
                                                        // of the level [6] this piece is running, thread 0 only
  if (tix == 0 && (SPEC == 1 || sd == 0)) { ctl[0] = __ldcg(p.fit_cur + chain); ctl[1] = __ldcg(p.fit_best + chain); ctl[2] = 0u; ctl[6] = 0xFFFFFFFFu; }
  group_sync(wc);

  if (SPEC > 1) run_spec(p, r, chain, gchain, s0, s1, sbuf, cw, cth, red, ctl, lane, wc, sd);
#pragma unroll 1
  for (i64 it = s0; SPEC == 1 && it < s1; ++it) {
    // a1 / a2: propose; the threads that hold the parameter apply it in their registers.  Only they
    // read or write its byte in the canonical row, so the row needs no barrier of its own.
    const Proposal q1 = propose(p, p.g0 + (u64)it, gchain, lane, ww, g, cw, cth);
    if (q1.is_w) xor_reg(r.A, q1.wsel, q1.wx);
    else if (q1.mine) shift_threshold(p, r, q1.loc, q1.oldv, q1.newv);
    // a3 / a4
    const u32 fcand = simulate(p, r, sbuf, red, (int)(it & 1), lane, ww);
    // a5
    u64 gs = p.g0 + (u64)it;
    if (REDERIVE) asm volatile("" : "+l"(gs));           // opaque: derive the proposal again instead of keeping it live
    const Proposal q = REDERIVE ? propose(p, gs, gchain, lane, ww, g, cw, cth) : q1;
    const u32 fcur = ctl[0], fbest = ctl[1];
    u64 level = ((gs | (u64)p.steps_per_level) >> 32) == 0 ? (u64)((u32)gs / (u32)p.steps_per_level) : gs / (u64)p.steps_per_level;
    if (level > (u64)(p.n_levels - 1)) level = (u64)(p.n_levels - 1);
    const i64 d = (i64)fcand - (i64)fcur;
    bool acc = d <= 0;
    if (!acc && d <= (i64)p.dmax) acc = q.x2 < __ldg(p.accept + level * (u64)p.dmax + (u64)(d - 1));
    const bool new_best = acc && fcand < fbest;
    if (p.level_stats && tix == 0) {
      if ((u32)level != ctl[6]) { flush_stats(p, ctl); ctl[6] = (u32)level; }
      ctl[2] += 1u; ctl[3] += acc ? 1u : 0u; ctl[4] += (acc && d > 0) ? 1u : 0u; ctl[5] += new_best ? 1u : 0u;
    }
    team_sync();                                         // everyone has read the control words
    // a6
    if (acc) {
      if (tix == 0) { ctl[0] = fcand; if (new_best) ctl[1] = fcand; }
      if (q.mine) {
        if (q.is_w) cw[q.slot] = (i8)q.newv;
        else if (t4 == 0) cth[q.slot] = (i8)q.newv;
      }
      if (new_best) {
        team_sync();
        u32* const best_w = (u32*)(p.best_w + (size_t)chain * TSD_EPADA);
        u32* const best_th = (u32*)(p.best_th + (size_t)chain * TSD_NPADA);
        for (int i = tix; i < TSD_EPADA / 4; i += TEAM) best_w[i] = ((const u32*)cw)[i];
        for (int i = tix; i < TSD_NPADA / 4; i += TEAM) best_th[i] = ((const u32*)cth)[i];
      }
    } else if (q.is_w) {
      xor_reg(r.A, q.wsel, q.wx);
    } else if (q.mine) {
      shift_threshold(p, r, q.loc, q.newv, q.oldv);
    }
    team_sync();
    const int trow = p.trace_row ? __ldg(p.trace_row + chain) : -1;
    if (trow >= 0 && q.mine && (q.is_w || t4 == 0)) {
      const u64 idx = gs - p.trace_g0;
      const u32 code = q.is_w ? (u32)(q.newv + 1) : (u32)q.newv;
      if (gs >= p.trace_g0 && idx < (u64)p.trace_max)
        p.trace_rec[(size_t)trow * (size_t)p.trace_max + idx] =
            (u64)fcand | ((u64)q.pidx << 32) | ((u64)code << 56) | ((u64)(acc ? 1 : 0) << 60) | ((u64)(new_best ? 1 : 0) << 61) |
            ((u64)(q.moved ? 0 : 1) << 62);
    }
  }
  // a7
  group_sync(wc);
  if (SPEC == 1 || sd == 0) {
    for (int i = tix; i < TSD_EPADA / 4; i += TEAM) ((u32*)(p.cur_w + (size_t)chain * TSD_EPADA))[i] = ((const u32*)cw)[i];
    for (int i = tix; i < TSD_NPADA / 4; i += TEAM) ((u32*)(p.cur_th + (size_t)chain * TSD_NPADA))[i] = ((const u32*)cth)[i];
    if (tix == 0) { p.fit_cur[chain] = ctl[0]; p.fit_best[chain] = ctl[1]; if (p.level_stats) flush_stats(p, ctl); }
    if (s1 < p.steps) {                        // hand the chain over
      __threadfence();
      team_sync();
      if (tix == 0) { __threadfence(); atomicExch(p.flags + chain, 1u); }
    }
  }
  group_sync(wc);                            // the shared memory is free for the next piece
}

}  // namespace tsa_dense
