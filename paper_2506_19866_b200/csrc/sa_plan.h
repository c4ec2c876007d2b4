// Host-side plan: turns the caller's network + observations into the device layout of
// sa_common.h (row order, ELL-by-pass slots, byte-lane packed conditions).  Pure host C++.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/ternary_sa.h"

namespace tsa {

struct Plan {
  int N = 0, E = 0, P = 0, K = 0, T = 0, n_obs = 0, n_pairs = 0;
  int CG = 1, n_chunks = 1, n_pass = 0, Epad = 0, EpadA = 0, NpadA = 0, state_words = 0;
  int max_in_degree = 0;
  std::vector<int32_t> node_of_row, row_of_node;          // [N]
  std::vector<int32_t> pass_base, pass_deg;               // [n_pass]
  std::vector<uint16_t> slot_off;                         // [Epad]
  std::vector<int32_t> slot_of_param;                     // [E]
  std::vector<int32_t> param_of_slot;                     // [Epad], -1 = padding
  std::vector<uint32_t> initw, clampm;                    // [n_chunks][N][CG]
  std::vector<uint32_t> obsw, obsm;                       // [n_chunks][n_obs][N][CG]
  std::vector<int8_t> obs_idx_of_t;                       // [T+1]
  int8_t tha[16] = {0}, thb[16] = {0};

  // caller order (int8 [E+N]) <-> internal rows (w [EpadA], th [NpadA])
  void to_internal(const int8_t* params, int8_t* w, int8_t* th) const;
  void to_caller(const int8_t* w, const int8_t* th, int8_t* params) const;
};

// Validates (SURVEY.md §8(b) "Validation in sa_create") and builds.  need_obs = false lets
// obs->obs be NULL (sa_simulate).  Returns SA_OK or SA_EINVAL with a message in err.
int build_plan(const sa_network* net, const sa_observations* obs, bool need_obs, Plan* plan, std::string* err);

// Range checks of parameter vectors: weights in {-1,0,1}, pair index in [0, n_pairs).
bool params_valid(const Plan& plan, const int8_t* params, int64_t n);

}  // namespace tsa
