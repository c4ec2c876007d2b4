// CUDA kernels of libternary_sa.so (sm_100a).  Lanes over rows (a node's in-edges, long rows
// split over consecutive lanes), 4 conditions per 32-bit word in biased byte lanes, chain state
// (weights, thresholds, double-buffered node states) resident in shared memory for the whole
// sa_run, state gathers bank-conflict free by the host's edge schedule (sa_plan.cpp).
//
// Two launch shapes share every device function:
//   CtaTeam  — one chain per CTA, its passes spread over the CTA's warps, __syncthreads per step;
//              schedule tables read through L1 (__ldg).  Any network that fits shared memory.
//   WarpTeam — one chain per WARP, several chains per CTA, __syncwarp only; the schedule tables are
//              staged once per CTA in shared memory.  Small / medium networks with many chains.
// Shares nothing with oracle/.
#include "sa_kernels.h"

#include <mutex>

#include "../../include/ternary_sa.h"

namespace tsa {

// ------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11), this library's own implementation.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&out)[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ------------------------------------------------------------------------------------------
// Teams: the threads that cooperate on one chain.
// ------------------------------------------------------------------------------------------
struct CtaTeam {
  static constexpr bool kIsWarp = false;
  __device__ static __forceinline__ int tid() { return threadIdx.x; }
  __device__ static __forceinline__ int nthr() { return blockDim.x; }
  __device__ static __forceinline__ void sync() { __syncthreads(); }
};
struct WarpTeam {
  static constexpr bool kIsWarp = true;
  __device__ static __forceinline__ int tid() { return threadIdx.x & 31; }
  __device__ static __forceinline__ int nthr() { return 32; }
  __device__ static __forceinline__ void sync() { __syncwarp(); }
};

// Schedule tables: device-global pointers (CtaTeam) or their shared-memory copies (WarpTeam).
struct Tables {
  const int4* pass_info;
  const uint32_t* row_meta;
  const uint16_t* slot_off;
  const uint32_t* fix;
  const int8_t* obs_idx_of_t;
};
template <bool SM, typename T>
__device__ __forceinline__ T tab_ld(const T* p) {
  if (SM) return *p;
  return __ldg(p);
}

// ------------------------------------------------------------------------------------------
// Shared-memory carve-up of one chain.
// ------------------------------------------------------------------------------------------
struct Smem {
  int8_t* w;        // [EpadA] weights in slot order
  int8_t* th;       // [NpadA] threshold-pair index per entry
  char2* ab;        // [NpadA] (-t_lo, -t_hi-1) per entry
  uint32_t* S0;     // [state_words] node states, byte lanes; the first 32 words are the zero dummies
  uint32_t* S1;
  uint32_t* red;    // [32] cross-warp reduction scratch (CtaTeam)
};

__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

__host__ __device__ inline size_t smem_layout(const DevProblem& P, size_t* off_th, size_t* off_ab, size_t* off_s0,
                                              size_t* off_s1, size_t* off_red) {
  size_t o = 0;
  o += P.EpadA;                   *off_th = o;
  o += P.NpadA;                   *off_ab = o;
  o += (size_t)P.NpadA * 2;       *off_s0 = align16(o);
  o = *off_s0 + align16((size_t)P.state_words * 4);   *off_s1 = o;
  o += align16((size_t)P.state_words * 4);            *off_red = o;
  o += 32 * 4;
  return o;
}

__host__ __device__ inline size_t chain_smem_bytes(const DevProblem& P) {
  size_t a, b, c, d, e;
  return smem_layout(P, &a, &b, &c, &d, &e);
}

size_t smem_bytes(const DevProblem& P) { return chain_smem_bytes(P); }

// shared copy of the schedule tables (WarpTeam kernels), placed before the per-chain regions
__host__ __device__ inline size_t table_layout(const DevProblem& P, size_t* off_info, size_t* off_meta, size_t* off_fix,
                                               size_t* off_obs) {
  size_t o = align16((size_t)P.Epad * 2);                         *off_info = o;
  o += (size_t)P.n_chunks * P.n_pass * 16;                        *off_meta = o;
  o += (size_t)P.n_pass * 32 * 4;                                 *off_fix = o;
  o += align16((size_t)P.n_fix * 4);                              *off_obs = o;
  o += align16((size_t)P.T + 1);
  return o;
}

size_t table_bytes(const DevProblem& P) {
  size_t a, b, c, d;
  return table_layout(P, &a, &b, &c, &d);
}

__device__ __forceinline__ Smem carve(const DevProblem& P, unsigned char* base) {
  size_t o_th, o_ab, o_s0, o_s1, o_red;
  smem_layout(P, &o_th, &o_ab, &o_s0, &o_s1, &o_red);
  Smem s;
  s.w = (int8_t*)base;
  s.th = (int8_t*)(base + o_th);
  s.ab = (char2*)(base + o_ab);
  s.S0 = (uint32_t*)(base + o_s0);
  s.S1 = (uint32_t*)(base + o_s1);
  s.red = (uint32_t*)(base + o_red);
  return s;
}

// 16-byte vector copy by one team, n16 = number of int4
template <typename Team>
__device__ __forceinline__ void copy16(void* dst, const void* src, int n16) {
  for (int i = Team::tid(); i < n16; i += Team::nthr()) ((int4*)dst)[i] = ((const int4*)src)[i];
}

template <typename Team>
__device__ __forceinline__ void build_ab(const DevProblem& P, const Smem& sm) {
  for (int r = Team::tid(); r < P.n_entries; r += Team::nthr()) {
    const int q = sm.th[r];
    sm.ab[r] = make_char2(P.tha[q], P.thb[q]);
  }
}

template <typename Team>
__device__ __forceinline__ uint32_t team_sum(uint32_t v, uint32_t* red) {
  v = __reduce_add_sync(0xffffffffu, v);
  if (Team::kIsWarp || blockDim.x == 32) return v;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (lane == 0) red[warp] = v;
  __syncthreads();
  uint32_t tot = 0;
  for (int i = 0; i < nw; ++i) tot += red[i];
  __syncthreads();
  return tot;
}

template <int CG> struct Vec;
template <> struct Vec<1> { using T = uint32_t; };
template <> struct Vec<2> { using T = uint2; };
template <> struct Vec<4> { using T = uint4; };

template <int CG>
__device__ __forceinline__ void unpack(const typename Vec<CG>::T& v, uint32_t (&s)[CG]);
template <> __device__ __forceinline__ void unpack<1>(const uint32_t& v, uint32_t (&s)[1]) { s[0] = v; }
template <> __device__ __forceinline__ void unpack<2>(const uint2& v, uint32_t (&s)[2]) { s[0] = v.x; s[1] = v.y; }
template <> __device__ __forceinline__ void unpack<4>(const uint4& v, uint32_t (&s)[4]) { s[0] = v.x; s[1] = v.y; s[2] = v.z; s[3] = v.w; }

template <int CG>
__device__ __forceinline__ typename Vec<CG>::T pack(const uint32_t (&s)[CG]);
template <> __device__ __forceinline__ uint32_t pack<1>(const uint32_t (&s)[1]) { return s[0]; }
template <> __device__ __forceinline__ uint2 pack<2>(const uint32_t (&s)[2]) { return make_uint2(s[0], s[1]); }
template <> __device__ __forceinline__ uint4 pack<4>(const uint32_t (&s)[4]) { return make_uint4(s[0], s[1], s[2], s[3]); }

// ------------------------------------------------------------------------------------------
// a3 + a4: simulate every condition for T synchronous steps from shared-memory weights and
// thresholds, count mismatches at the observation times.
// Returns this thread's partial mismatch count (clamped entries are in P.fit_const).  All
// threads of the team must call it.
//
// Arithmetic per node word (4 conditions): acc = 0x80808080 + SUM w*s (one IMAD per edge, w a
// sign-extended int8, s in {0,1,2} per byte); because 128 + sum - threshold stays in [0,255]
// every byte is a valid base-256 digit, so
//   [sum >= t_lo] = bit 7 of (acc - t_lo),  [sum > t_hi] = bit 7 of (acc - t_hi - 1)
// per byte, and the new state is their sum: 0 if sum < t_lo, 2 if sum > t_hi, else 1.
// ------------------------------------------------------------------------------------------
template <int U>
__device__ __forceinline__ int weight_of(uint32_t wword) {
  // sign-extended byte U in one PRMT: selector nibble U picks the byte, nibble U|8 replicates its
  // sign bit (PTX prmt default mode; __byte_perm would mask bit 3 of the nibbles away)
  constexpr uint32_t sel = (uint32_t)(U | ((U | 8) << 4) | ((U | 8) << 8) | ((U | 8) << 12));
  uint32_t r;
  asm("prmt.b32 %0, %1, 0, %2;" : "=r"(r) : "r"(wword), "n"(sel));
  return (int)r;
}

template <int CG, int U>
__device__ __forceinline__ void edge_slot(const unsigned char* curb, uint32_t wword, const uint2& offs, uint32_t (&acc)[CG]) {
  using V = typename Vec<CG>::T;
  const int wv = weight_of<U>(wword);
  const uint32_t o2 = (U < 2) ? offs.x : offs.y;
  const uint32_t off = (U & 1) ? (o2 >> 16) : (o2 & 0xFFFFu);
  uint32_t s[CG];
  unpack<CG>(*(const V*)(curb + off), s);
#pragma unroll
  for (int c = 0; c < CG; ++c) acc[c] += (uint32_t)(wv * (int)s[c]);
}

template <int CG, bool DUMP, typename Team, bool SMTAB>
__device__ __forceinline__ uint32_t simulate(const DevProblem& P, const Tables& tab, const Smem& sm, uint8_t* dump) {
  using V = typename Vec<CG>::T;
  constexpr int kEntryShift = (CG == 1) ? 2 : (CG == 2) ? 3 : 4;   // log2(CG*4)
  const int tid = Team::tid(), nthr = Team::nthr(), lane = tid & 31, warp = tid >> 5, nwarps = nthr >> 5;
  const int NW = P.state_words;
  uint32_t mism = 0;
  for (int ch = 0; ch < P.n_chunks; ++ch) {
    const uint32_t* initw = P.initw + (size_t)ch * NW;
    for (int x = tid; x < NW; x += nthr) {
      sm.S0[x] = __ldg(initw + x);
      if (x < 32) sm.S1[x] = 0u;              // the dummy entries of the other buffer
    }
    Team::sync();
    uint32_t* cur = sm.S0;
    uint32_t* nxt = sm.S1;
    for (int t = 1; t <= P.T; ++t) {
      const int oj = tab_ld<SMTAB>(tab.obs_idx_of_t + t);
      const unsigned char* curb = (const unsigned char*)cur;
      for (int ps = warp; ps < P.n_pass; ps += nwarps) {
        // x = first slot, y = iterations | combine rounds << 16, z / w = fix-up list start / count
        const int4 info = tab_ld<SMTAB>(tab.pass_info + ch * P.n_pass + ps);
        const uint32_t meta = tab_ld<SMTAB>(tab.row_meta + ps * 32 + lane);
        const int iters = info.y & 0xFFFF, rounds = info.y >> 16;
        uint32_t acc[CG];
#pragma unroll
        for (int c = 0; c < CG; ++c) acc[c] = kBias;
        const unsigned char* wp = (const unsigned char*)sm.w + info.x + lane * 4;
        const unsigned char* op = (const unsigned char*)tab.slot_off + 2 * (info.x + lane * 4);
#pragma unroll 1
        for (int full = iters >> 2; full > 0; --full, wp += 128, op += 256) {
          const uint32_t wword = *(const uint32_t*)wp;
          const uint2 offs = tab_ld<SMTAB>((const uint2*)op);
          edge_slot<CG, 0>(curb, wword, offs, acc);
          edge_slot<CG, 1>(curb, wword, offs, acc);
          edge_slot<CG, 2>(curb, wword, offs, acc);
          edge_slot<CG, 3>(curb, wword, offs, acc);
        }
        const int rem = iters & 3;
        if (rem) {
          const uint32_t wword = *(const uint32_t*)wp;
          const uint2 offs = tab_ld<SMTAB>((const uint2*)op);
          edge_slot<CG, 0>(curb, wword, offs, acc);
          if (rem > 1) edge_slot<CG, 1>(curb, wword, offs, acc);
          if (rem > 2) edge_slot<CG, 2>(curb, wword, offs, acc);
        }
        // split rows: partial sums of consecutive lanes are added up a binary tree
#pragma unroll 1
        for (int q = 0; q < rounds; ++q) {
          const bool take = (meta >> (kMetaCombineShift + q)) & 1u;
#pragma unroll
          for (int c = 0; c < CG; ++c) {
            const uint32_t other = __shfl_down_sync(0xffffffffu, acc[c], 1u << q);
            if (take) acc[c] += other - kBias;
          }
        }
        if (meta & kMetaHead) {
          const uint32_t off = meta & kMetaOffMask;
          const char2 ab = sm.ab[off >> kEntryShift];
          uint32_t ns[CG];
#pragma unroll
          for (int c = 0; c < CG; ++c) {
            const uint32_t ge = ((acc[c] + (uint32_t)((int)ab.x * (int)kOnes)) >> 7) & kOnes;
            const uint32_t gt = ((acc[c] + (uint32_t)((int)ab.y * (int)kOnes)) >> 7) & kOnes;
            ns[c] = ge + gt;
          }
          *(V*)((unsigned char*)nxt + off) = pack<CG>(ns);
          if (oj >= 0) {
            const size_t ob = ((size_t)ch * P.n_obs + oj) * (size_t)NW * 4 + off;
            uint32_t ov[CG], om[CG];
            unpack<CG>(__ldg((const V*)((const unsigned char*)P.obsw + ob)), ov);
            unpack<CG>(__ldg((const V*)((const unsigned char*)P.obsm + ob)), om);
#pragma unroll
            for (int c = 0; c < CG; ++c) {
              const uint32_t x = ns[c] ^ ov[c];
              mism += __popc((x | (x >> 1)) & om[c]);
            }
          }
        }
        // clamped entries keep their initial value: byte stores after the pass's own stores
        if (info.w > 0) {
          __syncwarp();
          for (int i = lane; i < info.w; i += 32) {
            const uint32_t fx = tab_ld<SMTAB>(tab.fix + info.z + i);
            ((unsigned char*)nxt)[fx & 0xFFFFu] = (unsigned char)(fx >> 16);
          }
        }
      }
      Team::sync();
      if (DUMP && oj >= 0) {
        for (int i = tid; i < P.N; i += nthr) {
          const uint32_t* e = nxt + (size_t)__ldg(P.entry_of_node + i) * CG;
#pragma unroll
          for (int c = 0; c < CG; ++c)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
              const int k = ch * 4 * CG + c * 4 + b;
              if (k < P.K) dump[((size_t)k * P.n_obs + oj) * P.N + i] = (uint8_t)((e[c] >> (8 * b)) & 0xFFu);
            }
        }
      }
      uint32_t* tmp = cur; cur = nxt; nxt = tmp;
    }
  }
  return mism;
}

__device__ __forceinline__ Tables global_tables(const DevProblem& P) {
  Tables t;
  t.pass_info = P.pass_info; t.row_meta = P.row_meta; t.slot_off = P.slot_off; t.fix = P.fix;
  t.obs_idx_of_t = P.obs_idx_of_t;
  return t;
}

// ------------------------------------------------------------------------------------------
// sa_eval / sa_simulate: one CTA per parameter set (internal order).
// ------------------------------------------------------------------------------------------
template <int CG, bool DUMP>
__global__ void eval_kernel(const DevProblem P, const int8_t* __restrict__ w, const int8_t* __restrict__ th,
                            uint32_t* __restrict__ fit, uint8_t* dump) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Smem sm = carve(P, smem_raw);
  const Tables tab = global_tables(P);
  const size_t b = blockIdx.x;
  copy16<CtaTeam>(sm.w, w + b * P.EpadA, P.EpadA / 16);
  copy16<CtaTeam>(sm.th, th + b * P.NpadA, P.NpadA / 16);
  __syncthreads();
  build_ab<CtaTeam>(P, sm);
  __syncthreads();
  const uint32_t f = team_sum<CtaTeam>(simulate<CG, DUMP, CtaTeam, false>(P, tab, sm, dump), sm.red) + P.fit_const;
  if (threadIdx.x == 0) fit[b] = f;
}

// ------------------------------------------------------------------------------------------
// Chain initialisation: block q of four parameters takes
// Philox(ctr = (q, 0, chain, 1), key = seed); weight = mulhi(y,3)-1, pair = mulhi(y, n_pairs).
// ------------------------------------------------------------------------------------------
template <int CG>
__global__ void init_kernel(const DevProblem P, const DevChains C, const DevSched S) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Smem sm = carve(P, smem_raw);
  const Tables tab = global_tables(P);
  const size_t chain = blockIdx.x;
  const uint32_t gchain = S.chain_id_base + (uint32_t)chain;
  for (int i = threadIdx.x; i < P.EpadA; i += blockDim.x) sm.w[i] = 0;
  for (int i = threadIdx.x; i < P.NpadA; i += blockDim.x) sm.th[i] = 0;
  __syncthreads();
  for (int q = threadIdx.x; 4 * q < P.P; q += blockDim.x) {
    uint32_t y[4];
    philox4x32_10((uint32_t)q, 0u, gchain, 1u, S.key0, S.key1, y);
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const int p = 4 * q + m;
      if (p < P.E) sm.w[__ldg(P.slot_of_param + p)] = (int8_t)((int)__umulhi(y[m], 3u) - 1);
      else if (p < P.P) sm.th[__ldg(P.entry_of_node + (p - P.E))] = (int8_t)__umulhi(y[m], (uint32_t)P.n_pairs);
    }
  }
  __syncthreads();
  if (S.constrained && threadIdx.x == 0) {
    // repair pass (reading C3): every node gets an activating in-edge, then a non-zero out-edge
    for (int i = 0; i < P.N; ++i) {
      const int a = __ldg(P.con_in_ptr + i), b = __ldg(P.con_in_ptr + i + 1);
      bool act = false;
      for (int x = a; x < b; ++x) act = act || sm.w[__ldg(P.con_in_slot + x)] == 1;
      if (act) continue;
      uint32_t y[4];
      philox4x32_10((uint32_t)i, 0u, gchain, 2u, S.key0, S.key1, y);
      sm.w[__ldg(P.con_in_slot + a + (int)__umulhi(y[0], (uint32_t)(b - a)))] = 1;
    }
    for (int i = 0; i < P.N; ++i) {
      const int a = __ldg(P.con_out_ptr + i), b = __ldg(P.con_out_ptr + i + 1);
      bool nz = false;
      for (int x = a; x < b; ++x) nz = nz || sm.w[__ldg(P.con_out_slot + x)] != 0;
      if (nz) continue;
      uint32_t y[4];
      philox4x32_10((uint32_t)i, 0u, gchain, 2u, S.key0, S.key1, y);
      sm.w[__ldg(P.con_out_slot + a + (int)__umulhi(y[2], (uint32_t)(b - a)))] = (int8_t)(2 * (int)__umulhi(y[3], 2u) - 1);
    }
  }
  __syncthreads();
  build_ab<CtaTeam>(P, sm);
  __syncthreads();
  const uint32_t f = team_sum<CtaTeam>(simulate<CG, false, CtaTeam, false>(P, tab, sm, nullptr), sm.red) + P.fit_const;
  copy16<CtaTeam>(C.cur_w + chain * P.EpadA, sm.w, P.EpadA / 16);
  copy16<CtaTeam>(C.best_w + chain * P.EpadA, sm.w, P.EpadA / 16);
  copy16<CtaTeam>(C.cur_th + chain * P.NpadA, sm.th, P.NpadA / 16);
  copy16<CtaTeam>(C.best_th + chain * P.NpadA, sm.th, P.NpadA / 16);
  if (threadIdx.x == 0) { C.fit_cur[chain] = f; C.fit_best[chain] = f; }
}

// ------------------------------------------------------------------------------------------
// sa_run: `steps` chain-steps of one chain, everything on chip (Table 1 :130-149;
// SURVEY.md §8(c)-3).  Thread 0 of the team applies / reverts the one-byte mutation; every thread
// computes the Philox block and the accept decision redundantly so no broadcast is needed.
// ------------------------------------------------------------------------------------------
// GetCandidate for a weight under the structural constraints (readings C1, C2): the
// two other values are listed cyclically after the old one; "to 0" is struck if the edge is the target's
// only non-zero in-edge or the source's only non-zero out-edge, "away from +1" if it is the target's only
// activator; the new value is entry mulhi(x1, length) of what is left; nothing left = null move (old value).
// w = the chain's canonical weight row (slot order).  Executed by one thread.
__device__ __forceinline__ int constrained_weight(const DevProblem& P, const int8_t* w, int p, int oldv, uint32_t x1, bool* moved) {
  bool bar_zero = false, bar_nonplus = false;
  if (oldv != 0) {
    const uint32_t en = __ldg(P.edge_nodes + p);
    const int src = (int)(en & 0xFFFFu), dst = (int)(en >> 16);
    int in_nz = 0, act = 0, out_nz = 0;
    for (int x = __ldg(P.con_in_ptr + dst); x < __ldg(P.con_in_ptr + dst + 1); ++x) {
      const int v = w[__ldg(P.con_in_slot + x)];
      in_nz += v != 0; act += v == 1;
    }
    for (int x = __ldg(P.con_out_ptr + src); x < __ldg(P.con_out_ptr + src + 1); ++x) out_nz += w[__ldg(P.con_out_slot + x)] != 0;
    bar_zero = in_nz == 1 || out_nz == 1;
    bar_nonplus = oldv == 1 && act == 1;
  }
  int list[2], len = 0;
#pragma unroll
  for (int k = 1; k <= 2; ++k) {
    const int v = (oldv + 1 + k) % 3 - 1;
    if (!((v == 0 && bar_zero) || (v != 1 && bar_nonplus))) list[len++] = v;
  }
  *moved = len > 0;
  if (len == 0) return oldv;
  return list[len == 2 ? (int)__umulhi(x1, 2u) : 0];
}

// Acceptance statistics of one chain over the level it is running; added to the handle's [L][4] table
// when the level ends and when the launch ends.
struct LevelStats {
  unsigned long long steps = 0, accepted = 0, worse = 0, best = 0;
  __device__ __forceinline__ void count(bool acc, bool is_worse, bool new_best) {
    steps += 1; accepted += acc; worse += acc && is_worse; best += new_best;
  }
  __device__ __forceinline__ void flush(unsigned long long* table, uint64_t lv) {
    if (steps == 0) return;
    atomicAdd(table + lv * 4 + 0, steps); atomicAdd(table + lv * 4 + 1, accepted);
    atomicAdd(table + lv * 4 + 2, worse); atomicAdd(table + lv * 4 + 3, best);
    steps = accepted = worse = best = 0;
  }
};

template <int CG, typename Team, bool SMTAB>
__device__ __forceinline__ void run_chain(const DevProblem& P, const Tables& tab, const Smem& sm, const DevChains& C,
                                          const DevSched& S, const DevTrace& Tr, const size_t chain,
                                          const uint64_t g0, const int64_t steps) {
  const uint32_t gchain = S.chain_id_base + (uint32_t)chain;
  const bool leader = Team::tid() == 0;
  copy16<Team>(sm.w, C.cur_w + chain * P.EpadA, P.EpadA / 16);
  copy16<Team>(sm.th, C.cur_th + chain * P.NpadA, P.NpadA / 16);
  Team::sync();
  build_ab<Team>(P, sm);
  uint32_t fcur = C.fit_cur[chain], fbest = C.fit_best[chain];
  const int trow = Tr.row_of_chain ? Tr.row_of_chain[chain] : -1;

  uint64_t level = g0 / (uint64_t)S.steps_per_level;
  int64_t left_in_level = S.steps_per_level - (int64_t)(g0 % (uint64_t)S.steps_per_level);
  LevelStats stats;                 // acceptance statistics of the level being run, kept by the leader
  Team::sync();

  for (int64_t it = 0; it < steps; ++it) {
    const uint64_t g = g0 + (uint64_t)it;
    uint32_t x[4];
    philox4x32_10((uint32_t)g, (uint32_t)(g >> 32), gchain, 0u, S.key0, S.key1, x);
    const int p = (int)__umulhi(x[0], (uint32_t)P.P);
    // a1/a2: the leader proposes and applies; (loc, old) let it revert
    int loc = 0, oldv = 0, newv = 0;
    bool moved = true;
    if (leader) {
      if (p < P.E) {
        loc = __ldg(P.slot_of_param + p);
        oldv = sm.w[loc];
        if (S.constrained) newv = constrained_weight(P, sm.w, p, oldv, x[1], &moved);
        else newv = (oldv + 2 + (int)__umulhi(x[1], 2u)) % 3 - 1;     // (code + 1 + r) mod 3 - 1, code = old + 1
        sm.w[loc] = (int8_t)newv;
      } else {
        loc = __ldg(P.entry_of_node + (p - P.E));
        oldv = sm.th[loc];
        newv = (oldv + 1 + (int)__umulhi(x[1], (uint32_t)(P.n_pairs - 1))) % P.n_pairs;
        sm.th[loc] = (int8_t)newv;
        sm.ab[loc] = make_char2(P.tha[newv], P.thb[newv]);
      }
    }
    Team::sync();
    // a3/a4
    const uint32_t fcand = team_sum<Team>(simulate<CG, false, Team, SMTAB>(P, tab, sm, nullptr), sm.red) + P.fit_const;
    // a5
    const uint64_t lv = level < (uint64_t)(S.n_levels - 1) ? level : (uint64_t)(S.n_levels - 1);
    const int64_t d = (int64_t)fcand - (int64_t)fcur;
    bool acc = d <= 0;
    if (!acc && d <= (int64_t)S.dmax) acc = x[2] < __ldg(S.accept + lv * (uint64_t)S.dmax + (uint64_t)(d - 1));
    bool new_best = false;
    // a6
    if (acc) {
      fcur = fcand;
      if (fcand < fbest) {
        fbest = fcand;
        new_best = true;
        copy16<Team>(C.best_w + chain * P.EpadA, sm.w, P.EpadA / 16);
        copy16<Team>(C.best_th + chain * P.NpadA, sm.th, P.NpadA / 16);
        Team::sync();               // the copy reads sm.w/th; the next mutation writes them
      }
    } else if (leader) {
      if (p < P.E) sm.w[loc] = (int8_t)oldv;
      else { sm.th[loc] = (int8_t)oldv; sm.ab[loc] = make_char2(P.tha[oldv], P.thb[oldv]); }
    }
    if (trow >= 0 && leader) {
      const uint64_t idx = g - Tr.g_start;
      if (g >= Tr.g_start && idx < (uint64_t)Tr.max_steps) {
        const uint64_t code = (p < P.E) ? (uint64_t)(newv + 1) : (uint64_t)newv;
        Tr.records[(size_t)trow * Tr.max_steps + idx] =
            (uint64_t)fcand | ((uint64_t)p << 32) | (code << 56) | ((uint64_t)(acc ? 1 : 0) << 60) |
            ((uint64_t)(new_best ? 1 : 0) << 61) | ((uint64_t)(moved ? 0 : 1) << 62);
      }
    }
    if (S.level_stats && leader) stats.count(acc, d > 0, new_best);
    if (--left_in_level == 0) {
      if (S.level_stats && leader && level < (uint64_t)(S.n_levels - 1)) stats.flush(S.level_stats, lv);   // the last row absorbs the rest
      ++level; left_in_level = S.steps_per_level;
    }
  }
  if (S.level_stats && leader) stats.flush(S.level_stats, level < (uint64_t)(S.n_levels - 1) ? level : (uint64_t)(S.n_levels - 1));
  Team::sync();
  // a7
  copy16<Team>(C.cur_w + chain * P.EpadA, sm.w, P.EpadA / 16);
  copy16<Team>(C.cur_th + chain * P.NpadA, sm.th, P.NpadA / 16);
  if (leader) { C.fit_cur[chain] = fcur; C.fit_best[chain] = fbest; }
}

template <int CG>
__global__ void run_kernel(const DevProblem P, const DevChains C, const DevSched S, const DevTrace Tr,
                           const uint64_t g0, const int64_t steps) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Smem sm = carve(P, smem_raw);
  run_chain<CG, CtaTeam, false>(P, global_tables(P), sm, C, S, Tr, blockIdx.x, g0, steps);
}

// One chain per warp; the CTA first stages the schedule tables in shared memory.
template <int CG>
__global__ void __launch_bounds__(256) run_warp_kernel(const DevProblem P, const DevChains C, const DevSched S,
                                                       const DevTrace Tr, const uint64_t g0, const int64_t steps) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  size_t o_info, o_meta, o_fix, o_obs;
  const size_t tbytes = table_layout(P, &o_info, &o_meta, &o_fix, &o_obs);
  {
    const int n = threadIdx.x, step = blockDim.x;
    for (int i = n; i < (P.Epad * 2 + 15) / 16; i += step) ((int4*)smem_raw)[i] = __ldg((const int4*)P.slot_off + i);
    for (int i = n; i < P.n_chunks * P.n_pass; i += step) ((int4*)(smem_raw + o_info))[i] = __ldg(P.pass_info + i);
    for (int i = n; i < P.n_pass * 32; i += step) ((uint32_t*)(smem_raw + o_meta))[i] = __ldg(P.row_meta + i);
    for (int i = n; i < P.n_fix; i += step) ((uint32_t*)(smem_raw + o_fix))[i] = __ldg(P.fix + i);
    for (int i = n; i <= P.T; i += step) ((int8_t*)(smem_raw + o_obs))[i] = P.obs_idx_of_t[i];
  }
  __syncthreads();
  Tables tab;
  tab.slot_off = (const uint16_t*)smem_raw;
  tab.pass_info = (const int4*)(smem_raw + o_info);
  tab.row_meta = (const uint32_t*)(smem_raw + o_meta);
  tab.fix = (const uint32_t*)(smem_raw + o_fix);
  tab.obs_idx_of_t = (const int8_t*)(smem_raw + o_obs);
  const int warp = threadIdx.x >> 5, cpb = blockDim.x >> 5;
  const size_t chain = (size_t)blockIdx.x * cpb + warp;
  if (chain >= (size_t)C.R) return;             // no CTA-wide barrier after this point
  const Smem sm = carve(P, smem_raw + tbytes + (size_t)warp * align16(chain_smem_bytes(P)));
  run_chain<CG, WarpTeam, true>(P, tab, sm, C, S, Tr, chain, g0, steps);
}

__global__ void argmin_kernel(const uint32_t* __restrict__ fit, int R, unsigned long long* out) {
  __shared__ unsigned long long red[32];
  unsigned long long best = ~0ull;
  for (int i = threadIdx.x; i < R; i += blockDim.x) {
    const unsigned long long v = ((unsigned long long)fit[i] << 32) | (unsigned)i;
    best = v < best ? v : best;
  }
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long v = __shfl_xor_sync(0xffffffffu, best, o);
    best = v < best ? v : best;
  }
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < (int)(blockDim.x >> 5); ++i) best = red[i] < best ? red[i] : best;
    out[0] = best;
  }
}

// ------------------------------------------------------------------------------------------
// launch wrappers
// ------------------------------------------------------------------------------------------
template <typename K>
static cudaError_t set_smem(K kernel, size_t bytes) {
  if (bytes <= 48 * 1024) return cudaSuccess;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

#define TSA_DISPATCH_CG(P, ...)                            \
  switch ((P).CG) {                                        \
    case 1: { constexpr int CG = 1; __VA_ARGS__; } break;  \
    case 2: { constexpr int CG = 2; __VA_ARGS__; } break;  \
    default: { constexpr int CG = 4; __VA_ARGS__; } break; \
  }

cudaError_t launch_init(const DevProblem& P, const DevChains& C, const DevSched& S, int threads, cudaStream_t st) {
  const size_t sb = smem_bytes(P);
  cudaError_t e = cudaSuccess;
  TSA_DISPATCH_CG(P, {
    e = set_smem(init_kernel<CG>, sb);
    if (e == cudaSuccess) init_kernel<CG><<<C.R, threads, sb, st>>>(P, C, S);
  });
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_run(const DevProblem& P, const DevChains& C, const DevSched& S, const DevTrace& Tr,
                       uint64_t g0, int64_t steps, int threads, cudaStream_t st) {
  const size_t sb = smem_bytes(P);
  cudaError_t e = cudaSuccess;
  TSA_DISPATCH_CG(P, {
    e = set_smem(run_kernel<CG>, sb);
    if (e == cudaSuccess) run_kernel<CG><<<C.R, threads, sb, st>>>(P, C, S, Tr, g0, steps);
  });
  return e != cudaSuccess ? e : cudaGetLastError();
}

size_t warp_kernel_smem(const DevProblem& P, int chains_per_cta) {
  return table_bytes(P) + (size_t)chains_per_cta * align16(smem_bytes(P));
}

cudaError_t launch_run_warp(const DevProblem& P, const DevChains& C, const DevSched& S, const DevTrace& Tr,
                            uint64_t g0, int64_t steps, int chains_per_cta, cudaStream_t st) {
  const size_t sb = warp_kernel_smem(P, chains_per_cta);
  const unsigned grid = (unsigned)((C.R + chains_per_cta - 1) / chains_per_cta);
  cudaError_t e = cudaSuccess;
  TSA_DISPATCH_CG(P, {
    e = set_smem(run_warp_kernel<CG>, sb);
    if (e == cudaSuccess) run_warp_kernel<CG><<<grid, 32 * chains_per_cta, sb, st>>>(P, C, S, Tr, g0, steps);
  });
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_eval(const DevProblem& P, const int8_t* w, const int8_t* th, int64_t n, uint32_t* fit,
                        uint8_t* dump, int threads, cudaStream_t st) {
  const size_t sb = smem_bytes(P);
  cudaError_t e = cudaSuccess;
  TSA_DISPATCH_CG(P, {
    if (dump) {
      e = set_smem(eval_kernel<CG, true>, sb);
      if (e == cudaSuccess) eval_kernel<CG, true><<<(unsigned)n, threads, sb, st>>>(P, w, th, fit, dump);
    } else {
      e = set_smem(eval_kernel<CG, false>, sb);
      if (e == cudaSuccess) eval_kernel<CG, false><<<(unsigned)n, threads, sb, st>>>(P, w, th, fit, dump);
    }
  });
  return e != cudaSuccess ? e : cudaGetLastError();
}

// Level synchronisation of PAPER.md Table 1 (:150-155), on the device: per group of `group`
// consecutive chains, the smallest d_best (ties: smallest chain) ...
__global__ void group_argmin_kernel(const uint32_t* __restrict__ fit, int R, int group, unsigned long long* out) {
  const int first = blockIdx.x * group, last = min(R, first + group);
  unsigned long long best = ~0ull;
  for (int c = first + (int)threadIdx.x; c < last; c += (int)blockDim.x)
    best = min(best, ((unsigned long long)fit[c] << 32) | (unsigned)c);
  __shared__ unsigned long long sm[32];
  for (int o = 16; o > 0; o >>= 1) best = min(best, __shfl_down_sync(0xffffffffu, best, o));
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x < 32) {
    best = threadIdx.x < (blockDim.x + 31) / 32 ? sm[threadIdx.x] : ~0ull;
    for (int o = 16; o > 0; o >>= 1) best = min(best, __shfl_down_sync(0xffffffffu, best, o));
    if (threadIdx.x == 0) out[blockIdx.x] = best;
  }
}

// ... and its best vector becomes every member's best AND current vector ("use overall best
// solution to re-initialize all threads"; x_current = x_best at the top of the next level).
__global__ void level_broadcast_kernel(DevChains C, int EpadA, int NpadA, int group, const unsigned long long* __restrict__ win) {
  const int c = blockIdx.x;
  const unsigned long long w = win[c / group];
  const int src = (int)(w & 0xFFFFFFFFull);
  const uint32_t f = (uint32_t)(w >> 32);
  const uint32_t* sw = (const uint32_t*)(C.best_w + (size_t)src * EpadA);
  const uint32_t* sth = (const uint32_t*)(C.best_th + (size_t)src * NpadA);
  uint32_t* cw = (uint32_t*)(C.cur_w + (size_t)c * EpadA);
  uint32_t* cth = (uint32_t*)(C.cur_th + (size_t)c * NpadA);
  uint32_t* bw = (uint32_t*)(C.best_w + (size_t)c * EpadA);
  uint32_t* bth = (uint32_t*)(C.best_th + (size_t)c * NpadA);
  for (int i = threadIdx.x; i < EpadA / 4; i += blockDim.x) { const uint32_t v = sw[i]; cw[i] = v; if (c != src) bw[i] = v; }
  for (int i = threadIdx.x; i < NpadA / 4; i += blockDim.x) { const uint32_t v = sth[i]; cth[i] = v; if (c != src) bth[i] = v; }
  if (threadIdx.x == 0) { C.fit_cur[c] = f; C.fit_best[c] = f; }
}

cudaError_t launch_level_sync(const DevProblem& P, const DevChains& C, int group, unsigned long long* win, cudaStream_t st) {
  const int n_groups = (C.R + group - 1) / group;
  group_argmin_kernel<<<n_groups, group >= 256 ? 256 : 32, 0, st>>>(C.fit_best, C.R, group, win);
  level_broadcast_kernel<<<C.R, 128, 0, st>>>(C, P.EpadA, P.NpadA, group, win);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Level synchronisation for callers that cannot allocate (sa_level_sync_static).
//
// The winners of the groups go to this array, part of the library image, instead of a buffer from cudaMalloc: every
// GPU that loads the library carries its 512 KiB until the process ends.  All handles and threads share it and it
// keeps the last call's winners; group_argmin_kernel rewrites entries 0..n_groups-1 before level_broadcast_kernel
// reads them, both on the same stream, so nothing needs clearing.  Calls that overlap on the GPU race on it.
//
// On the host the name g_static_win is only a stand-in for the symbol, not an address a kernel could use: the device
// address comes from cudaGetSymbolAddress, asked once per device with that device current, and is what the kernels get.
// ------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned long long g_static_win[SA_LEVEL_SYNC_STATIC_MAX_GROUPS];

constexpr int kMaxDevices = 64;
static std::mutex g_static_win_mu;
static unsigned long long* g_static_win_addr[kMaxDevices] = {};   // per device ordinal, filled on first use

cudaError_t launch_level_sync_static(const DevProblem& P, const DevChains& C, int group, cudaStream_t st, const char** why) {
  *why = nullptr;
  const int n_groups = (C.R + group - 1) / group;
  if (n_groups > SA_LEVEL_SYNC_STATIC_MAX_GROUPS) {
    *why = "more groups than the fixed winner table holds";
    return cudaErrorInvalidValue;
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  cudaPointerAttributes attr;
  e = cudaPointerGetAttributes(&attr, C.fit_best);
  if (e != cudaSuccess) return e;
  if (attr.type != cudaMemoryTypeDevice || attr.device != dev || dev < 0 || dev >= kMaxDevices) {
    *why = "the device that owns the handle's chain store is not the current device";
    return cudaErrorInvalidValue;
  }
  unsigned long long* win = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_static_win_mu);
    if (!g_static_win_addr[dev]) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_static_win);     // device `dev` is current: this is ITS copy of the array
      if (e != cudaSuccess) return e;
      g_static_win_addr[dev] = (unsigned long long*)p;
    }
    win = g_static_win_addr[dev];
  }
  group_argmin_kernel<<<n_groups, group >= 256 ? 256 : 32, 0, st>>>(C.fit_best, C.R, group, win);
  level_broadcast_kernel<<<C.R, 128, 0, st>>>(C, P.EpadA, P.NpadA, group, win);
  return cudaGetLastError();
}

cudaError_t launch_argmin(const uint32_t* fit, int R, unsigned long long* out, cudaStream_t st) {
  argmin_kernel<<<1, 1024, 0, st>>>(fit, R, out);
  return cudaGetLastError();
}

}  // namespace tsa
