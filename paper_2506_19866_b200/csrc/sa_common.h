// Internal structures shared by the host code and the kernels of libternary_sa.so.
// Not part of the ABI (include/ternary_sa.h is) and not shared with oracle/.
#pragma once
#include <cstdint>

#include <vector_types.h>

namespace tsa {

constexpr int kMaxPairs = 16;
constexpr int kWarp = 32;
constexpr uint32_t kBias = 0x80808080u;   // byte-lane accumulator bias
constexpr uint32_t kOnes = 0x01010101u;

// row_meta bits (one u32 per (pass, lane))
constexpr uint32_t kMetaOffMask = 0xFFFFu;     // byte offset of the node's state words
constexpr uint32_t kMetaHead = 1u << 16;       // this lane finalises a node in this pass
constexpr int kMetaCombineShift = 17;          // bit (17 + r): in combine round r add lane + 2^r

// Read-only problem description in device memory, identical for every chain.
//
// State layout: every node owns one "entry" of CG 32-bit words (4 conditions per word, byte
// lanes); entry e lives at byte offset e*CG*4, so its shared-memory bank unit is e mod nb,
// nb = 32/CG.  Entries 0..nb-1 are all-zero dummies, one per bank unit.
//
// Edge layout: a node's in-edges form one row, or several sub-rows in consecutive lanes when it
// is split; pass p = 32 rows handled by one warp, slot (p, k, lane) = edge k of that lane's row,
// stored as [pass][k/4][lane][k%4] (a lane's four consecutive weights are one 32-bit word, its
// four source offsets one 64-bit word).  The host orders every row's edges so that in each
// iteration k the nb lanes of a conflict group (half-warp for 64-bit loads) read nb distinct bank
// units: the state gathers are bank-conflict free by construction.  Empty cells read a dummy.
struct DevProblem {
  int N, E, P, K, T, n_obs, n_pairs;
  int CG;          // 32-bit state words per node (1, 2 or 4)
  int n_chunks;    // condition chunks of 4*CG conditions (K > 16 -> several)
  int n_pass;
  int n_entries;   // state entries incl. dummies and holes
  int Epad;        // number of slots
  int EpadA;       // Epad rounded up to 16 (row pitch of the weight store, bytes)
  int NpadA;       // n_entries rounded up to 16 (row pitch of the threshold store, bytes)
  int state_words; // n_entries*CG: words of one state buffer
  int n_fix;       // entries of `fix`
  uint32_t fit_const;            // mismatches of clamped observed entries (constant per problem)
  const int4*     pass_info;     // [n_chunks][n_pass]: x = first slot, y = iterations | combine rounds << 16,
                                 //   z, w = start / count of the (chunk, pass) clamp fix-up list in `fix`
  const uint32_t* row_meta;      // [n_pass*32]
  const uint16_t* slot_off;      // [Epad] byte offset of the source entry
  const int32_t*  slot_of_param; // [E] caller edge id -> slot
  const int32_t*  entry_of_node; // [N]
  const uint32_t* initw;         // [n_chunks][n_entries][CG] initial state, byte lanes
  const uint32_t* obsw;          // [n_chunks][n_obs][n_entries][CG] observed values (0 where unscored)
  const uint32_t* obsm;          // [n_chunks][n_obs][n_entries][CG] 0x01 in scored byte lanes
  const uint32_t* fix;           // entries: bits 0-15 byte offset in the state buffer, 16-23 value
  const int8_t*   obs_idx_of_t;  // [T+1] observation index of time t or -1
  // structural constraints (only filled when the handle was created with SA_CONSTRAINED):
  // CSR over the nodes' in- / out-edges in ascending caller edge order, holding each edge's SLOT in the
  // canonical weight row, and the end points of every caller edge
  const int32_t*  con_in_ptr;    // [N+1]
  const int32_t*  con_in_slot;   // [E]
  const int32_t*  con_out_ptr;   // [N+1]
  const int32_t*  con_out_slot;  // [E]
  const uint32_t* edge_nodes;    // [E] src | dst << 16
  int8_t tha[kMaxPairs];         // -t_lo      per pair
  int8_t thb[kMaxPairs];         // -t_hi - 1  per pair
};

// Chain-state store in HBM: structure of arrays, int8 rows in slot / entry order, 16-byte pitch.
struct DevChains {
  int R;
  int8_t *cur_w, *cur_th, *best_w, *best_th;   // [R][EpadA], [R][NpadA]
  uint32_t *fit_cur, *fit_best;                // [R]
};

struct DevSched {
  uint32_t key0, key1;           // Philox key = seed
  uint32_t chain_id_base;
  int n_levels, dmax;
  int64_t steps_per_level;
  const uint32_t* accept;        // device [L][D]
  unsigned long long* level_stats;   // device [L][4] steps, accepted, accepted worse, new best; nullptr = off
  uint32_t constrained;          // 1 = constrained GetCandidate / initialisation
};

struct DevTrace {
  const int32_t* row_of_chain;   // device [R]: trace row or -1; nullptr = tracing off
  uint64_t* records;             // device [n][max_steps]
  int64_t max_steps;
  uint64_t g_start;              // step counter when tracing was armed
};

}  // namespace tsa
