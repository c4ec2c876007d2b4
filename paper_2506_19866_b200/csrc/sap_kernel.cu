// Kernels of the paper's OWN model (sm_100a): parallel simulated annealing over x = [w, p, t, u, m, d]
// (§2.1-2.3, Table 1, §2.5.3).
//
// Mapping.  One chain = a group of LPC lanes of a warp (8, 16 or 32; a warp carries G = 32 / LPC chains),
// one lane = NS nodes ("node slots") and the in-edges of those nodes ("edge slots", a fixed number per
// node slot: the host sorts the nodes by in-degree so that slot n holds nodes of similar degree).  The
// chain never leaves the chip during a launch:
//   * per edge slot the lane keeps, in a register, a three-entry table of what the edge contributes to
//     its target's image for source state 0 / 1 / 2:  4 + (s // t) * w * p  in bytes 1 / 2 / 3 (byte 0 = 0)
//     (PAPER.md:66-68); the source publishes its state as the one-byte PRMT selector 0x41 + s in a
//     double-buffered shared array of at most 128 bytes per warp (no bank conflicts), so one edge costs
//     LDS.U8 + PRMT + IADD;
//   * per node slot: clip the image to [0,2], eligibility from the memory count, priority = u x age,
//     REDUX.MAX over the chain's lanes, bounded move, score against the
//     reference with the gradient weight, publish the new state;
//   * the canonical vector (caller's parameter order), the constraint counters (non-zero in / out
//     edges and activating in-edges per node) and the chain's fitness live in shared
//     memory; GetCandidate, the accept test and the commit are computed redundantly by every lane of
//     the chain, so they need no communication.
// Compiled at run time by NVRTC (sa_jit.cpp) with the network's shape as -D constants, and ahead of
// time with the defaults below (build check).  It includes nothing: sap_params.h is prepended by
// whoever compiles it.  Shares nothing with oracle/.
#ifndef TSP_N
#define TSP_N 63
#define TSP_E 178
#define TSP_K 1
#define TSP_T 19
#define TSP_LPC 32
#define TSP_NS 2
#define TSP_ESL 8, 3
#define TSP_WPB 4
#define TSP_MINBLOCKS 4
#endif

namespace tsa_paper {

constexpr int N = TSP_N, E = TSP_E, NP = 3 * TSP_E + 3 * TSP_N, NPPAD = (NP + 15) / 16 * 16, K = TSP_K, T = TSP_T;
constexpr int LPC = TSP_LPC, NS = TSP_NS, G = 32 / LPC, WPB = TSP_WPB;
constexpr int kESL[NS] = {TSP_ESL};                       // edge slots of node slot n
__host__ __device__ constexpr int es_off(int n) { int s = 0; for (int i = 0; i < n; ++i) s += kESL[i]; return s; }
constexpr int ES = es_off(NS);
constexpr int NSP = NS <= 1 ? 1 : NS <= 2 ? 2 : NS <= 4 ? 4 : 8;   // node slots padded to a vector load
constexpr int NPOS = NS * LPC;                            // node positions of a chain (>= N; the rest is padding)
constexpr int STATE_B = NPOS;                             // one state buffer of one chain: a one-byte selector per position
constexpr int BUF_B = G * STATE_B;                        // one state buffer of a warp's chains
constexpr int NCPAD = (N + 3) / 4 * 4;
constexpr int CHAIN_B = (NPPAD + 3 * NCPAD + 8 * 4 + 15) / 16 * 16;   // canonical vector, 3 counter rows, control words
constexpr int WARP_B = (2 * BUF_B + 15) / 16 * 16 + G * CHAIN_B;
constexpr u32 kEmptyLut = 0x04040400u;                    // an empty edge slot contributes 4 (= 0 after the bias) for every state
constexpr u32 kSel0 = 0x41u;                              // selector of state s = kSel0 + s: byte s+1 of the table, then zeros
static_assert(LPC == 8 || LPC == 16 || LPC == 32, "lanes per chain");
static_assert(NS >= 1 && NS <= 8 && NPOS >= N, "node slots");
static_assert(N <= 256 && ES <= 256, "ploc fields are 8 bits wide");

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
// shared memory through 32-bit shared-window addresses with a compile-time byte offset (which state buffer)
template <int OFF>
__device__ __forceinline__ u32 lds_u8(u32 a) { u32 v; smem_check(a + OFF, 1); asm volatile("ld.shared.u8 %0, [%1+%2];" : "=r"(v) : "r"(a), "n"(OFF) : "memory"); return v; }
template <int OFF>
__device__ __forceinline__ void sts_u8(u32 a, u32 v) { smem_check(a + OFF, 1); asm volatile("st.shared.u8 [%0+%1], %2;" ::"r"(a), "n"(OFF), "r"(v) : "memory"); }
// byte look-up: result byte 0 = byte (sel & 7) of {table, 0}, byte 1 = byte 4 (zero), bytes 2-3 = byte 0 of the
// table (kept zero).  Every selector here is 0x41 + state: no nibble has its replicate-sign bit set (the
// __byte_perm intrinsic would spend an instruction masking them)
__device__ __forceinline__ u32 prmt(u32 table, u32 sel) { u32 r; asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(table), "r"(0u), "r"(sel)); return r; }

// reductions over the LPC lanes of a chain (aligned lane groups of a full warp)
__device__ __forceinline__ u32 group_max(u32 v) {
  if constexpr (LPC == 32) {
    return __reduce_max_sync(0xffffffffu, v);
  } else {
#pragma unroll
    for (int o = LPC / 2; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
  }
}
__device__ __forceinline__ u32 group_sum(u32 v) {
  if constexpr (LPC == 32) {
    return __reduce_add_sync(0xffffffffu, v);
  } else {
#pragma unroll
    for (int o = LPC / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
  }
}

// value ranges, in increasing order: size and smallest value of a class
__device__ __forceinline__ int dom_size(int cls, bool fast) { return (cls == kT || cls == kD) ? 2 : cls == kU ? (fast ? 3 : 6) : 3; }
__device__ __forceinline__ int dom_base(int cls, bool fast) { return cls == kP ? -1 : (cls == kT || cls == kD) ? 1 : cls == kU ? (fast ? 10 : 1) : 0; }
__device__ __forceinline__ int class_of(int q) { return q < E ? kW : q < 2 * E ? kP : q < 3 * E ? kT : q < 3 * E + N ? kU : q < 3 * E + 2 * N ? kM : kD; }

// contribution table of an edge: byte s+1 = 4 + (s // t) * w * p, byte 0 = 0  (floor division, reading 16)
__device__ __forceinline__ u32 make_lut(int w, int p, int t) {
  const int c = w * p;
  const int v1 = t == 1 ? c : 0, v2 = t == 1 ? 2 * c : c;
  return (4u << 8) | ((u32)(v1 + 4) << 16) | ((u32)(v2 + 4) << 24);
}

// What a lane keeps in registers for its chain.
struct Lane {
  u32 lut[ES];     // contribution table of each edge slot
  u32 addr[ES];    // shared address of the source's selector (state buffer 0)
  u32 u[NS];       // node slot: speed u_i ...
  u32 m[NS];       // ... memory m_i ...
  int d[NS];       // ... step size d_i
  u32 self[NS];    // shared address of this lane's own selectors (state buffer 0)
  int node[NS];    // node id or -1
};

// Build the lane's registers from the chain's canonical vector in shared memory.
__device__ __forceinline__ void build_lane(const Params& p, const i8* canon, u32 sstate, int lig, Lane& L) {
#pragma unroll
  for (int e = 0; e < ES; ++e) {
    const int ed = __ldg(p.slot_edge + e * LPC + lig);
    L.lut[e] = ed < 0 ? kEmptyLut : make_lut(canon[ed], canon[E + ed], canon[2 * E + ed]);
    L.addr[e] = sstate + (u32)__ldg(p.slot_src + e * LPC + lig);
  }
#pragma unroll
  for (int n = 0; n < NS; ++n) {
    const int i = __ldg(p.pos_node + n * LPC + lig);
    L.node[n] = i;
    L.u[n] = i < 0 ? 1u : (u32)canon[3 * E + i];
    L.m[n] = i < 0 ? 0u : (u32)canon[3 * E + N + i];
    L.d[n] = i < 0 ? 1 : (int)canon[3 * E + 2 * N + i];
    L.self[n] = sstate + (u32)(n * LPC + lig);
  }
}

// First half of a transition, node slot NI (a template so that the slot's edge-slot count is a constant
// expression), reading state buffer RB: the image from the published states of t-1, eligibility, priority.
template <int NI, int RB>
struct Images {
  static __device__ __forceinline__ void run(const Lane& L, u32 t, const u32 (&s)[NS], const u32 (&last)[NS], const u32 (&cnt)[NS],
                                             u32 (&tg)[NS], u32 (&pr)[NS], u32& top) {
    constexpr int EO = es_off(NI), EN = kESL[NI];
    u32 acc = 0u;
#pragma unroll
    for (int j = 0; j < EN; ++j) acc += prmt(L.lut[EO + j], lds_u8<RB * BUF_B>(L.addr[EO + j]));   // 4 + (s_j // t_ji) * w_ji * p_ji
    const int img = (int)acc - 4 * EN;                                  // the image K_i (:66-68)
    tg[NI] = (u32)min(max(img, 0), 2);                                  // as far as the allowable states go (:70)
    const bool eligible = tg[NI] != s[NI] && cnt[NI] >= L.m[NI];        // told to update, memory criterion met (:79, :82)
    pr[NI] = eligible ? last[NI] : 0u;                                  // speed x time steps since last updated (:82), kept as a running product
    top = max(top, pr[NI]);
    Images<NI + 1, RB>::run(L, t, s, last, cnt, tg, pr, top);
  }
};
template <int RB>
struct Images<NS, RB> {
  static __device__ __forceinline__ void run(const Lane&, u32, const u32 (&)[NS], const u32 (&)[NS], const u32 (&)[NS], u32 (&)[NS],
                                             u32 (&)[NS], u32&) {}
};

// the lane's cost tables of one time point: byte s+1 of word n = |s - r| * (|g| + 1) for its node slot n
__device__ __forceinline__ void load_cost(const u32* row, u32 (&c)[NSP]) {
  if constexpr (NSP == 1) { c[0] = __ldg(row); }
  else if constexpr (NSP == 2) { const uint2 v = __ldg((const uint2*)row); c[0] = v.x; c[1] = v.y; }
  else {
#pragma unroll
    for (int i = 0; i < NSP; i += 4) { const uint4 v = __ldg((const uint4*)(row + i)); c[i] = v.x; c[i + 1] = v.y; c[i + 2] = v.z; c[i + 3] = v.w; }
  }
}

// One transition t-1 -> t reading state buffer RB and publishing into the other one,
// and row t of the objective (:104-111).
template <int RB, bool DUMP>
__device__ __forceinline__ void transition(const Lane& L, u32 t, const u32* cost_row, u32 (&s)[NS], u32 (&last)[NS], u32 (&cnt)[NS],
                                           u32& y, u8* dump_row) {
  u32 cost[NSP];
  load_cost(cost_row, cost);
  u32 tg[NS], pr[NS];
  u32 top = 0u;
  Images<0, RB>::run(L, t, s, last, cnt, tg, pr, top);
  top = group_max(top);
  top = top != 0u ? top : 0xFFFFFFFFu;                                // nobody eligible: no priority equals it
#pragma unroll
  for (int n = 0; n < NS; ++n) {
    const int delta = (int)tg[n] - (int)s[n];
    const bool mv = pr[n] == top;                                     // the nodes sharing the highest priority (:82)
    const int step = min(max(delta, -L.d[n]), L.d[n]);                // at most d_i levels toward K_i (:80)
    s[n] = (u32)((int)s[n] + (mv ? step : 0));
    last[n] = mv ? L.u[n] : last[n] + L.u[n];                         // u x (t + 1 - time of the last change): u after a move, + u otherwise
    cnt[n] = (delta != 0 && !mv) ? cnt[n] + 1u : 0u;                  // consecutive time steps told to update without moving
    const u32 sel = kSel0 + s[n];
    sts_u8<(1 - RB) * BUF_B>(L.self[n], sel);
    y += prmt(cost[n], sel);                                          // |S - R| (.) (|G| + 1)  (:104-111)
    if (DUMP && dump_row != nullptr && L.node[n] >= 0) dump_row[L.node[n]] = (u8)s[n];
  }
  __syncwarp();
}

// Simulate(x) (§2.1-2.3): the objective of the vector now in the lanes' registers.
template <bool DUMP>
__device__ __forceinline__ u32 simulate(const Params& p, const Lane& L, int lig, u8* dump) {
  u32 y = 0;
#pragma unroll 1
  for (int k = 0; k < K; ++k) {
    u32 s[NS], last[NS], cnt[NS];
    const u32 iw = __ldg(p.init_lane + k * LPC + lig);
    const u32* cost_row = p.cost_lane + ((size_t)(k * (T + 1)) * LPC + lig) * NSP;
    u8* dump_row = (DUMP && dump != nullptr) ? dump + (size_t)(k * (T + 1)) * N : nullptr;
    {
      u32 cost[NSP];
      load_cost(cost_row, cost);
#pragma unroll
      for (int n = 0; n < NS; ++n) {
        s[n] = (iw >> (2 * n)) & 3u; last[n] = L.u[n]; cnt[n] = 0u;     // age 1 at the first transition (reading P3)
        const u32 sel = kSel0 + s[n];
        sts_u8<0>(L.self[n], sel);
        y += prmt(cost[n], sel);                                      // row t0 of S, R and G (:92-100)
        if (DUMP && dump_row != nullptr && L.node[n] >= 0) dump_row[L.node[n]] = (u8)s[n];
      }
    }
    __syncwarp();
    u32 t = 1u;
#pragma unroll 1
    for (; t + 1u <= (u32)T; t += 2u) {                               // two transitions per trip: the buffer roles are constants
      transition<0, DUMP>(L, t, cost_row + (size_t)t * LPC * NSP, s, last, cnt, y, DUMP && dump_row ? dump_row + (size_t)t * N : nullptr);
      transition<1, DUMP>(L, t + 1u, cost_row + (size_t)(t + 1u) * LPC * NSP, s, last, cnt, y,
                          DUMP && dump_row ? dump_row + (size_t)(t + 1u) * N : nullptr);
    }
    if (T & 1) transition<0, DUMP>(L, (u32)T, cost_row + (size_t)T * LPC * NSP, s, last, cnt, y, DUMP && dump_row ? dump_row + (size_t)T * N : nullptr);
  }
  return group_sum(y);
}

// One chain's shared memory.
struct ChainMem {
  i8* canon;            // [NPPAD] canonical vector, caller's parameter order
  u8* cin;              // [N] in-edges of non-zero weight
  u8* cout;             // [N] out-edges of non-zero weight
  u8* cact;             // [N] in-edges with p = +1 and w != 0
  volatile u32* ctl;    // [0] d_cur, [1] d_best
  u32 sstate;           // shared address of the chain's state buffer 0
};

__device__ __forceinline__ ChainMem chain_mem(u8* smem_warp, int grp) {
  ChainMem m;
  u8* base = smem_warp + (2 * BUF_B + 15) / 16 * 16 + grp * CHAIN_B;
  m.canon = (i8*)base;
  m.cin = base + NPPAD; m.cout = m.cin + NCPAD; m.cact = m.cout + NCPAD;
  m.ctl = (volatile u32*)(base + NPPAD + 3 * NCPAD);
  m.sstate = (u32)__cvta_generic_to_shared(smem_warp) + (u32)(grp * STATE_B);
  return m;
}

// constraint counters of the canonical vector, one node per lane at a time
__device__ __forceinline__ void count_constraints(const Params& p, const ChainMem& m, int lig) {
  for (int i = lig; i < N; i += LPC) {
    int a = 0, b = 0, c = 0;
    for (int x = __ldg(p.in_ptr + i); x < __ldg(p.in_ptr + i + 1); ++x) {
      const int e = __ldg(p.in_edge + x);
      a += m.canon[e] != 0;
      c += m.canon[e] != 0 && m.canon[E + e] == 1;
    }
    for (int x = __ldg(p.out_ptr + i); x < __ldg(p.out_ptr + i + 1); ++x) b += m.canon[__ldg(p.out_edge + x)] != 0;
    m.cin[i] = (u8)a; m.cout[i] = (u8)b; m.cact[i] = (u8)c;
  }
}

// A proposal as every lane of the chain sees it.
struct Proposal {
  u32 x2, loc;
  int q, cls, oldv, newv;
  bool moved;
};

// GetCandidate (readings 7, P5): q = mulhi(x0, NP); the other values of the
// parameter are listed cyclically after the old one; with constraints on, those that would leave a
// node without a non-zero in- or out-edge or without an activating in-edge are struck; the new value
// is entry mulhi(x1, length) of the list; an empty list gives a null move.
__device__ __forceinline__ Proposal propose(const Params& p, const ChainMem& m, u64 gs, u32 gchain) {
  Proposal r;
  u32 x[4];
  philox4x32_10((u32)gs, (u32)(gs >> 32), gchain, 0u, p.key0, p.key1, x);
  r.x2 = x[2];
  r.q = (int)__umulhi(x[0], (u32)NP);
  r.loc = __ldg(p.ploc + r.q);
  r.cls = (int)(r.loc & 7u);
  r.oldv = m.canon[r.q];
  const int src = (int)((r.loc >> 16) & 255u), dst = (int)(r.loc >> 24);
  const bool fast = r.cls == kU && __ldg(p.fast + src) != 0;
  const int n = dom_size(r.cls, fast), base = dom_base(r.cls, fast), oi = r.oldv - base;
  // which other values are barred: only "weight to 0" and "polarity away from +1" can break a constraint
  bool bar_zero = false, bar_all = false;
  if (p.constrained && r.cls <= kP) {
    const int e = r.q - r.cls * E;
    const int w = m.canon[e], pol = m.canon[E + e];
    const bool last_act = pol == 1 && w != 0 && m.cact[dst] == 1;
    if (r.cls == kW) bar_zero = w != 0 && (m.cin[dst] == 1 || m.cout[src] == 1 || last_act);
    else bar_all = last_act;
  }
  int len = 0;
#pragma unroll
  for (int k = 1; k < 6; ++k)
    if (k < n) {
      const int v = base + (oi + k) % n;
      len += !(bar_all || (bar_zero && v == 0));
    }
  r.moved = len > 0;
  r.newv = r.oldv;
  if (r.moved) {
    int pick = (int)__umulhi(x[1], (u32)len);
#pragma unroll
    for (int k = 1; k < 6; ++k)
      if (k < n) {
        const int v = base + (oi + k) % n;
        if (!(bar_all || (bar_zero && v == 0))) {
          if (pick == 0) r.newv = v;
          --pick;
        }
      }
  }
  return r;
}

// Put value v of parameter q (class cls, location loc) into the owning lane's registers; the other
// parameters of the same edge / node are read from the canonical vector.
__device__ __forceinline__ void set_param(Lane& L, const ChainMem& m, const Proposal& r, int v, int lig) {
  const bool mine = (int)((r.loc >> 3) & 31u) == lig;
  const int sel = (int)((r.loc >> 8) & 255u);
  if (r.cls <= kT) {
    const int e = r.q - r.cls * E;
    const int w = r.cls == kW ? v : m.canon[e], pol = r.cls == kP ? v : m.canon[E + e], t = r.cls == kT ? v : m.canon[2 * E + e];
    const u32 lut = make_lut(w, pol, t);
#pragma unroll
    for (int k = 0; k < ES; ++k) if (mine && k == sel) L.lut[k] = lut;
  } else {
    const int i = r.q - 3 * E - (r.cls - kU) * N;
    const int u = r.cls == kU ? v : m.canon[3 * E + i], mm = r.cls == kM ? v : m.canon[3 * E + N + i], d = r.cls == kD ? v : m.canon[3 * E + 2 * N + i];
#pragma unroll
    for (int n = 0; n < NS; ++n)
      if (mine && n == sel) { L.u[n] = (u32)u; L.m[n] = (u32)mm; L.d[n] = d; }
  }
}

// commit an accepted move to the canonical vector and the constraint counters (one lane of the chain)
__device__ __forceinline__ void commit(const ChainMem& m, const Proposal& r) {
  if (r.cls <= kP) {
    const int e = r.q - r.cls * E;
    const int src = (int)((r.loc >> 16) & 255u), dst = (int)(r.loc >> 24);
    const int w0 = m.canon[e], p0 = m.canon[E + e];
    const int w1 = r.cls == kW ? r.newv : w0, p1 = r.cls == kP ? r.newv : p0;
    const int dnz = (w1 != 0) - (w0 != 0), dact = (w1 != 0 && p1 == 1) - (w0 != 0 && p0 == 1);
    m.cin[dst] = (u8)(m.cin[dst] + dnz); m.cout[src] = (u8)(m.cout[src] + dnz); m.cact[dst] = (u8)(m.cact[dst] + dact);
  }
  m.canon[r.q] = (i8)r.newv;
}

extern "C" __global__ void __launch_bounds__(32 * WPB, TSP_MINBLOCKS) tsp_run(const __grid_constant__ Params p) {
  extern __shared__ __align__(16) u8 smem_all[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, grp = lane / LPC, lig = lane % LPC;
  const u32 slot = (blockIdx.x * WPB + warp) * G + grp;
  const bool live = slot < (u32)p.R;                    // a warp's spare groups shadow the last chain and write nothing
  const u32 chain = live ? slot : (u32)(p.R - 1);
  const u32 gchain = p.chain_id_base + chain;
  const ChainMem m = chain_mem(smem_all + (size_t)warp * WARP_B, grp);

  // a0: stage the chain
  for (int x = lig; x < NPPAD / 4; x += LPC) ((u32*)m.canon)[x] = __ldcg((const u32*)(p.cur + (size_t)chain * NPPAD) + x);
  if (lig == 0) { m.ctl[0] = __ldcg(p.fit_cur + chain); m.ctl[1] = __ldcg(p.fit_best + chain); }
  __syncwarp();
  if (p.constrained) count_constraints(p, m, lig);
  Lane L;
  build_lane(p, m.canon, m.sstate, lig, L);
  __syncwarp();

  u64 st_steps = 0, st_acc = 0, st_worse = 0, st_best = 0;   // acceptance statistics of the level being run
  u64 st_level = ~0ull;
#pragma unroll 1
  for (i64 it = 0; it < p.steps; ++it) {
    const u64 gs = p.g0 + (u64)it;
    // a1 / a2: propose and apply
    const Proposal r = propose(p, m, gs, gchain);
    if (r.moved) set_param(L, m, r, r.newv, lig);
    // a3 / a4
    const u32 fcand = simulate<false>(p, L, lig, nullptr);
    // a5
    const u32 fcur = m.ctl[0], fbest = m.ctl[1];
    u64 level = ((gs | (u64)p.steps_per_level) >> 32) == 0 ? (u64)((u32)gs / (u32)p.steps_per_level) : gs / (u64)p.steps_per_level;
    if (level > (u64)(p.n_levels - 1)) level = (u64)(p.n_levels - 1);
    const i64 d = (i64)fcand - (i64)fcur;
    bool acc = d <= 0;
    if (!acc && d <= (i64)p.dmax) acc = r.x2 < __ldg(p.accept + level * (u64)p.dmax + (u64)(d - 1));
    const bool new_best = acc && fcand < fbest;
    __syncwarp();                                          // every lane has read the canonical vector and the control words
    // a6 (no barrier sits inside a branch: with several chains per warp the branches differ between lane groups)
    if (acc && lig == 0) {
      if (r.moved) commit(m, r);
      m.ctl[0] = fcand;
      if (new_best) m.ctl[1] = fcand;
    }
    __syncwarp();
    if (acc) {
      if (new_best && live)
        for (int x = lig; x < NPPAD / 4; x += LPC) ((u32*)(p.best + (size_t)chain * NPPAD))[x] = ((const u32*)m.canon)[x];
    } else if (r.moved) {
      set_param(L, m, r, r.oldv, lig);
    }
    if (p.level_stats) {
      if (level != st_level) {
        if (live && lig == 0 && st_steps) {
          atomicAdd(p.level_stats + st_level * 4 + 0, st_steps); atomicAdd(p.level_stats + st_level * 4 + 1, st_acc);
          atomicAdd(p.level_stats + st_level * 4 + 2, st_worse); atomicAdd(p.level_stats + st_level * 4 + 3, st_best);
        }
        st_level = level; st_steps = st_acc = st_worse = st_best = 0;
      }
      st_steps += 1; st_acc += acc; st_worse += acc && d > 0; st_best += new_best;
    }
    const int trow = (p.trace_row && live) ? __ldg(p.trace_row + chain) : -1;
    if (trow >= 0 && lig == 0 && gs >= p.trace_g0 && gs - p.trace_g0 < (u64)p.trace_max) {
      const bool fast = r.cls == kU && __ldg(p.fast + ((r.loc >> 16) & 255u)) != 0;
      const u32 code = (u32)(r.newv - dom_base(r.cls, fast));
      p.trace_rec[(size_t)trow * (size_t)p.trace_max + (gs - p.trace_g0)] =
          (u64)fcand | ((u64)r.q << 32) | ((u64)code << 56) | ((u64)(acc ? 1 : 0) << 60) | ((u64)(new_best ? 1 : 0) << 61) |
          ((u64)(r.moved ? 0 : 1) << 62);
    }
  }
  if (p.level_stats && live && lig == 0 && st_steps) {
    atomicAdd(p.level_stats + st_level * 4 + 0, st_steps); atomicAdd(p.level_stats + st_level * 4 + 1, st_acc);
    atomicAdd(p.level_stats + st_level * 4 + 2, st_worse); atomicAdd(p.level_stats + st_level * 4 + 3, st_best);
  }
  // a7: write back
  __syncwarp();
  if (live) {
    for (int x = lig; x < NPPAD / 4; x += LPC) ((u32*)(p.cur + (size_t)chain * NPPAD))[x] = ((const u32*)m.canon)[x];
    if (lig == 0) { p.fit_cur[chain] = m.ctl[0]; p.fit_best[chain] = m.ctl[1]; }
  }
}

// Objective of eval_n given vectors (sap_eval, sap_simulate): same staging, same Simulate.
extern "C" __global__ void __launch_bounds__(32 * WPB, TSP_MINBLOCKS) tsp_eval(const __grid_constant__ Params p) {
  extern __shared__ __align__(16) u8 smem_all[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, grp = lane / LPC, lig = lane % LPC;
  const i64 slot = ((i64)blockIdx.x * WPB + warp) * G + grp;
  const bool live = slot < p.eval_n;
  const i64 v = live ? slot : p.eval_n - 1;
  const ChainMem m = chain_mem(smem_all + (size_t)warp * WARP_B, grp);
  for (int x = lig; x < NP; x += LPC) m.canon[x] = p.eval_params[(size_t)v * NP + x];
  __syncwarp();
  Lane L;
  build_lane(p, m.canon, m.sstate, lig, L);
  __syncwarp();
  u32 y;
  if (p.eval_dump != nullptr) y = simulate<true>(p, L, lig, slot == 0 ? p.eval_dump : nullptr);   // the states of vector 0
  else y = simulate<false>(p, L, lig, nullptr);
  if (live && lig == 0 && p.eval_fit) p.eval_fit[v] = y;
}

// Initial vectors (readings 8, P6) and their objective: block b of four
// parameters takes Philox(ctr = (b, 0, chain, 1)); with constraints on, the repair pass of DESIGN.md
// reading P6 follows with Philox(ctr = (node, 0, chain, 2)).
extern "C" __global__ void __launch_bounds__(32 * WPB, TSP_MINBLOCKS) tsp_init(const __grid_constant__ Params p) {
  extern __shared__ __align__(16) u8 smem_all[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, grp = lane / LPC, lig = lane % LPC;
  const u32 slot = (blockIdx.x * WPB + warp) * G + grp;
  const bool live = slot < (u32)p.R;
  const u32 chain = live ? slot : (u32)(p.R - 1);
  const u32 gchain = p.chain_id_base + chain;
  const ChainMem m = chain_mem(smem_all + (size_t)warp * WARP_B, grp);
  for (int x = lig; x < NPPAD / 4; x += LPC) ((u32*)m.canon)[x] = 0u;
  __syncwarp();
  for (int b = lig; 4 * b < NP; b += LPC) {
    u32 y[4];
    philox4x32_10((u32)b, 0u, gchain, 1u, p.key0, p.key1, y);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int q = 4 * b + j;
      if (q < NP) {
        const int cls = class_of(q);
        const bool fast = cls == kU && __ldg(p.fast + (q - 3 * E)) != 0;
        m.canon[q] = (i8)(dom_base(cls, fast) + (int)__umulhi(y[j], (u32)dom_size(cls, fast)));
      }
    }
  }
  __syncwarp();
  if (p.constrained && lig == 0) {
    for (int i = 0; i < N; ++i) {                          // every node gets an activating in-edge ...
      const int a = __ldg(p.in_ptr + i), b = __ldg(p.in_ptr + i + 1);
      bool act = false;
      for (int x = a; x < b; ++x) { const int e = __ldg(p.in_edge + x); act = act || (m.canon[E + e] == 1 && m.canon[e] != 0); }
      if (act) continue;
      u32 y[4];
      philox4x32_10((u32)i, 0u, gchain, 2u, p.key0, p.key1, y);
      const int e = __ldg(p.in_edge + a + (int)__umulhi(y[0], (u32)(b - a)));
      m.canon[E + e] = 1;
      if (m.canon[e] == 0) m.canon[e] = (i8)(1 + (int)__umulhi(y[1], 2u));
    }
    for (int i = 0; i < N; ++i) {                          // ... and then an out-edge of non-zero weight
      const int a = __ldg(p.out_ptr + i), b = __ldg(p.out_ptr + i + 1);
      bool nz = false;
      for (int x = a; x < b; ++x) nz = nz || m.canon[__ldg(p.out_edge + x)] != 0;
      if (nz) continue;
      u32 y[4];
      philox4x32_10((u32)i, 0u, gchain, 2u, p.key0, p.key1, y);
      const int e = __ldg(p.out_edge + a + (int)__umulhi(y[2], (u32)(b - a)));
      m.canon[e] = (i8)(1 + (int)__umulhi(y[3], 2u));
    }
  }
  __syncwarp();
  Lane L;
  build_lane(p, m.canon, m.sstate, lig, L);
  __syncwarp();
  const u32 y = simulate<false>(p, L, lig, nullptr);
  if (live) {
    for (int x = lig; x < NPPAD / 4; x += LPC) {
      const u32 v = ((const u32*)m.canon)[x];
      ((u32*)(p.cur + (size_t)chain * NPPAD))[x] = v;
      ((u32*)(p.best + (size_t)chain * NPPAD))[x] = v;
    }
    if (lig == 0) { p.fit_cur[chain] = y; p.fit_best[chain] = y; }
  }
}

}  // namespace tsa_paper
