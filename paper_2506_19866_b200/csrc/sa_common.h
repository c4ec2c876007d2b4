// Internal structures shared by the host code and the kernels of libternary_sa.so.
// Not part of the ABI (include/ternary_sa.h is) and not shared with oracle/.
#pragma once
#include <cstdint>

namespace tsa {

constexpr int kMaxPairs = 16;
constexpr int kWarp = 32;
constexpr uint32_t kBias = 0x80808080u;   // byte-lane accumulator bias
constexpr uint32_t kOnes = 0x01010101u;

// Read-only problem description in device memory, identical for every chain.  Nodes are
// renumbered ("rows") by descending in-degree; edges live in "slots" of an ELL-by-pass layout:
// pass p = rows 32p..32p+31 handled by one warp, slot (p, k, lane) = in-edge k of row 32p+lane.
// Slots are stored as [pass][k/4][lane][k%4] so that one lane's four consecutive weights are one
// 32-bit word and its four source offsets one 64-bit word.
struct DevProblem {
  int N, E, P, K, T, n_obs, n_pairs;
  int CG;          // 32-bit state words per node: 4 conditions per word in byte lanes (1, 2 or 4)
  int n_chunks;    // condition chunks of 4*CG conditions (K > 16 -> several)
  int n_pass;      // ceil(rows / 32)
  int Epad;        // number of slots (multiple of 128 per pass-iteration group)
  int EpadA;       // Epad rounded up to 16 (row pitch of the weight store, bytes)
  int NpadA;       // N rounded up to 16 (row pitch of the threshold store, bytes)
  int state_words; // (N+1)*CG: words of one state buffer incl. the all-zero dummy node N
  const int32_t*  pass_base;     // [n_pass] first slot of the pass
  const int32_t*  pass_deg;      // [n_pass] real iterations of the pass (max in-degree of its rows)
  const uint16_t* slot_off;      // [Epad] byte offset of the source row's state words (row*CG*4); padding -> dummy
  const int32_t*  slot_of_param; // [E] caller edge id -> slot
  const int32_t*  row_of_node;   // [N]
  const int32_t*  node_of_row;   // [N]
  const uint32_t* initw;         // [n_chunks][N][CG] initial state, byte lanes
  const uint32_t* clampm;        // [n_chunks][N][CG] 0xFF in clamped byte lanes
  const uint32_t* obsw;          // [n_chunks][n_obs][N][CG] observed values (0 where unobserved)
  const uint32_t* obsm;          // [n_chunks][n_obs][N][CG] 0x01 in observed byte lanes
  const int8_t*   obs_idx_of_t;  // [T+1] observation index of time t or -1
  int8_t tha[kMaxPairs];         // -t_lo      per pair
  int8_t thb[kMaxPairs];         // -t_hi - 1  per pair
};

// Chain-state store in HBM: structure of arrays, int8 rows in slot / row order, 16-byte pitch.
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
};

struct DevTrace {
  const int32_t* row_of_chain;   // device [R]: trace row or -1; nullptr = tracing off
  uint64_t* records;             // device [n][max_steps]
  int64_t max_steps;
  uint64_t g_start;              // step counter when tracing was armed
};

}  // namespace tsa
