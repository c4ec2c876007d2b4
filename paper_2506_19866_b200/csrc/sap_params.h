// Kernel argument block of the paper-model kernels (sap_kernel.cu).  Included by the host code AND
// prepended to the kernel source that NVRTC compiles, so it uses only built-in types.  Plain data,
// device pointers.
#ifndef TSA_PAPER_PARAMS_H
#define TSA_PAPER_PARAMS_H

namespace tsa_paper {

typedef unsigned int u32;
typedef unsigned short u16;
typedef unsigned char u8;
typedef unsigned long long u64;
typedef long long i64;
typedef signed char i8;

// Parameter classes in the order of the vector x = [w, p, t, u, m, d].
enum { kW = 0, kP = 1, kT = 2, kU = 3, kM = 4, kD = 5 };

// ploc word of parameter q: bits 0-2 class, 3-7 owning lane (within the chain's lane group), 8-15 edge
// slot (w, p, t) or node slot (u, m, d) of that lane, 16-23 source node (edges) or the node itself,
// 24-31 destination node (edges).
struct Params {
  // problem tables, identical for every chain
  const u32* ploc;        // [NP]
  const u16* slot_src;    // [ES][LPC] byte offset (= position), in a chain's state buffer, of the source node's selector
  const int* slot_edge;   // [ES][LPC] caller edge id of the lane's edge slot, -1 = empty slot
  const int* pos_node;    // [NS][LPC] node id of the lane's node slot, -1 = padding
  const u32* init_lane;   // [K][LPC]  initial states of the lane's nodes, 2 bits per node slot
  const u32* cost_lane;   // [K][T+1][LPC][NSP] per node slot (padded to 1, 2, 4 or 8): byte s+1 = |s - r| * (|g| + 1), 0 if not measured
  const u8* fast;         // [N] 1 = speed range {10,11,12}
  const int* in_ptr;      // [N+1] CSR by destination over caller edge ids (ascending)
  const int* in_edge;     // [E]
  const int* out_ptr;     // [N+1] CSR by source
  const int* out_edge;    // [E]
  // chain store (HBM): canonical vectors in the caller's parameter order, values themselves
  int R;
  i8* cur;                // [R][NPPAD]
  i8* best;               // [R][NPPAD]
  u32* fit_cur;           // [R]
  u32* fit_best;          // [R]
  // annealing schedule
  u32 key0, key1, chain_id_base;
  int n_levels, dmax;
  i64 steps_per_level;
  const u32* accept;      // [L][D]
  u32 constrained;        // 1 = structural constraints in GetCandidate
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
  // evaluation / initialisation entry points
  const i8* eval_params;  // [eval_n][NP] caller layout, unpadded
  i64 eval_n;
  u32* eval_fit;          // [eval_n]
  u8* eval_dump;          // [K][T+1][N] states of vector 0, or nullptr
};

}  // namespace tsa_paper
#endif
