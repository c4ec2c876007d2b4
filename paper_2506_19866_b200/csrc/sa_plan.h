// Host-side plan: turns the caller's network + observations into the device layout of
// sa_common.h — node entries and their bank classes, rows / split rows packed into passes, a
// bank-conflict-free edge schedule (bipartite edge colouring per conflict group), byte-lane
// packed conditions, clamp fix-up lists.  Pure host C++; deterministic.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/ternary_sa.h"

namespace tsa {

struct PlanOptions {
  bool split_rows = true;     // split long rows over consecutive lanes (TSA_NO_SPLIT=1 disables)
  bool bank_opt = true;       // optimise bank classes by hill climbing (TSA_NO_BANKOPT=1 disables)
  static PlanOptions from_env();
};

struct Plan {
  int N = 0, E = 0, P = 0, K = 0, T = 0, n_obs = 0, n_pairs = 0;
  int CG = 1, nb = 32, n_chunks = 1, n_pass = 0, n_entries = 0;
  int Epad = 0, EpadA = 0, NpadA = 0, state_words = 0;
  int max_in_degree = 0;
  uint32_t fit_const = 0;
  std::vector<int32_t> entry_of_node;                     // [N]
  std::vector<int32_t> pass_base, pass_iters, pass_rounds;   // [n_pass]
  std::vector<uint32_t> row_meta;                         // [n_pass*32]
  std::vector<uint16_t> slot_off;                         // [Epad]
  std::vector<int32_t> slot_of_param;                     // [E]
  std::vector<int32_t> param_of_slot;                     // [Epad], -1 = dummy cell
  std::vector<uint32_t> initw;                            // [n_chunks][n_entries][CG]
  std::vector<uint32_t> obsw, obsm;                       // [n_chunks][n_obs][n_entries][CG]
  std::vector<int32_t> fix_ptr;                           // [n_chunks*n_pass + 1]
  std::vector<uint32_t> fix;
  std::vector<int8_t> obs_idx_of_t;                       // [T+1]
  int8_t tha[16] = {0}, thb[16] = {0};
  // statistics for sa_get_info / DESIGN.md
  int total_iters = 0, n_rows = 0, n_split_nodes = 0;

  // caller order (int8 [E+N]) <-> internal rows (w [EpadA], th [NpadA])
  void to_internal(const int8_t* params, int8_t* w, int8_t* th) const;
  void to_caller(const int8_t* w, const int8_t* th, int8_t* params) const;
};

// Validates (SURVEY.md §8(b) "Validation in sa_create") and builds.  need_obs = false lets
// obs->obs be NULL (sa_simulate).  Returns SA_OK or SA_EINVAL with a message in err.
int build_plan(const sa_network* net, const sa_observations* obs, bool need_obs, const PlanOptions& opt,
               Plan* plan, std::string* err);

// Range checks of parameter vectors: weights in {-1,0,1}, pair index in [0, n_pairs).
bool params_valid(const Plan& plan, const int8_t* params, int64_t n);

}  // namespace tsa
