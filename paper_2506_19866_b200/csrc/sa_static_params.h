// Kernel argument block of the statically scheduled sa_run kernel (sa_static_kernel.cu).
// Included by the host code AND prepended to the kernel source that NVRTC compiles, so it uses
// only built-in types (NVRTC has no <cstdint>).  Plain data, device pointers.
#ifndef TSA_STATIC_PARAMS_H
#define TSA_STATIC_PARAMS_H

namespace tsa_static {

typedef unsigned int u32;
typedef unsigned long long u64;
typedef long long i64;
typedef signed char i8;

// meta word of one (tier, thread): bits 0-15 byte offset of the state entry the lane stores to (its
// private scratch entry if it finalises nothing), bit 16 = this lane finalises a node,
// bit 17+q = in combine round q add the partial sum of lane + 2^q.
constexpr u32 kMetaOffMask = 0xFFFFu;
constexpr u32 kMetaHead = 1u << 16;
constexpr int kMetaCombineShift = 17;

struct Params {
  // schedule of the problem, one column per thread of the team (W warps x 32 lanes)
  const u32* lane_off2;   // [NOREG][W*32]   two 16-bit source-entry byte offsets per word
  const u32* lane_meta;   // [NT][W*32]
  const u32* lane_clamp;  // [NT][3*CG][W*32] per word: 0xFF mask of clamped byte lanes, their A bytes, their D bytes
  const u32* initw;       // [STATE_WORDS]    state at t = 0, byte lanes
  const u32* obsw;        // [NOBS][STATE_WORDS] observed values (0 where unscored)
  const u32* obsm;        // [NOBS][STATE_WORDS] 0x01 in scored byte lanes
  const u32* wloc;        // [E]  weight register | byte << 8 | thread << 16 holding edge e
  const u32* thloc;       // [N]  tier | thread << 16 of the lane that finalises node i
  // structural constraints (kernels built with TSA_CONSTRAINED=1): CSR over the nodes' in- / out-edges holding each
  // edge's offset in the canonical weight row, and the end points of every caller edge (src | dst << 16)
  const int* con_in_ptr;  // [N+1]
  const int* con_in_slot; // [E]
  const int* con_out_ptr; // [N+1]
  const int* con_out_slot;// [E]
  const u32* edge_nodes;  // [E]
  i8 tha[16];             // -t_lo     per threshold pair
  i8 thb[16];             // -t_hi - 1 per threshold pair
  u32 fit_const;          // mismatches of clamped observed entries
  // chain store (HBM, SoA)
  int R;
  i8* cur_w;              // [R][EPADA]
  i8* cur_th;             // [R][NPADA]
  i8* best_w;
  i8* best_th;
  u32* fit_cur;           // [R]
  u32* fit_best;
  // annealing schedule
  u32 key0, key1, chain_id_base;
  int n_levels, dmax;
  i64 steps_per_level;
  const u32* accept;      // [L][D]
  // trace (row == nullptr: off)
  const int* trace_row;   // [R]
  u64* trace_rec;         // [n][trace_max]
  i64 trace_max;
  u64 trace_g0;
  // acceptance statistics per temperature level (nullptr: off): [L][4] = steps, accepted, accepted worse, new best
  u64* level_stats;
  // this launch
  u64 g0;
  i64 steps;
};

}  // namespace tsa_static
#endif
