// Host-side plan of the paper-model kernels (sap_kernel.cu): which lane of a chain's lane group owns
// which nodes and in-edges, and the per-lane tables the kernels read.  Not shared with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/ternary_sa.h"

namespace tsa {

struct PaperPlan {
  int N = 0, E = 0, NP = 0, NPPAD = 0, K = 0, T = 0;
  int LPC = 32;                       // lanes per chain (8, 16 or 32)
  int NS = 1;                         // node slots per lane
  int ES = 0;                         // edge slots per lane
  std::vector<int32_t> esl;           // [NS] edge slots of node slot n = largest in-degree among the slot's nodes
  std::vector<int32_t> node_lane, node_slot;   // [N]
  std::vector<uint32_t> ploc;         // [NP]
  std::vector<uint16_t> slot_src;     // [ES][LPC]
  std::vector<int32_t> slot_edge;     // [ES][LPC]
  std::vector<int32_t> pos_node;      // [NS][LPC]
  std::vector<uint32_t> init_lane;    // [K][LPC]
  int NSP = 1;                        // NS padded to 1, 2, 4 or 8 (vector loads of the cost tables)
  std::vector<uint32_t> cost_lane;    // [K][T+1][LPC][NSP]: byte s+1 of a word = |s - r| * (|g| + 1)
  std::vector<uint8_t> fast;          // [N]
  std::vector<int32_t> in_ptr, in_edge, out_ptr, out_edge;
  std::vector<int32_t> src, dst;      // [E]
  int max_in_degree = 0;
  uint32_t max_objective = 0;         // 6 per measured entry
};

// Validates like sap_create (SA_EINVAL with the reason in *err) and builds the plan.  need_ref = false:
// obs->ref may be NULL (sap_simulate).  constrained: every node must have an in- and an out-edge.
// n_chains (0 = unknown) picks the lanes per chain for 33..64 nodes: 16 (two chains per warp, 5 % faster when
// the GPU is full) once R / 2 warps fill every SM's resident slots, else 32.
int build_paper_plan(const sap_network* net, const sap_observations* obs, bool need_ref, bool constrained, int64_t n_chains,
                     int sm_count, PaperPlan* out, std::string* err);

// every value of n vectors [n][NP] lies in its parameter's range
bool paper_params_valid(const PaperPlan& pl, const int8_t* params, int64_t n);

}  // namespace tsa
