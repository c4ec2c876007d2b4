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
  bool store_opt = true;      // ... counting the conflicts of the result stores too (TSA_NO_STOREOPT=1: gathers only)
  bool tiers = true;          // group the passes into tiers for the statically scheduled kernel (TSA_NO_TIERS=1 disables)
  int min_team_warps = 1;     // lower bound of warps per chain (few chains: spread each over more warps)
  int max_lane_slots = 0;     // edge slots one thread may hold in registers; 0 = default for the CG
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

  // Static schedule (sa_static_kernel.cu).  team_warps = W > 0: the passes are ordered tier-major
  // (pass = tier*W + warp), all passes of a tier have the tier's iteration count, and the tables
  // below hold one column per thread of the team.  W = 0: not applicable, static_why says why.
  int team_warps = 0, n_tiers = 0, scratch_entry0 = 0;
  std::string static_why;
  std::vector<int32_t> tier_iters, tier_rounds;           // [n_tiers]
  std::vector<uint32_t> lane_off2;                        // [sum ceil(it/2)][W*32]
  std::vector<uint32_t> lane_meta;                        // [n_tiers][W*32]
  std::vector<uint32_t> lane_clamp;                       // [n_tiers][3*CG][W*32]: mask, A bytes, D bytes of clamped lanes
  std::vector<uint32_t> wloc;                             // [E]
  std::vector<uint32_t> thloc;                            // [N]

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
