// Host-side tables of the dense (tensor-pipe) sa_run kernel, sa_dense_kernel.cu: where every
// candidate edge sits in the mma.sync A fragments, the row <-> column numbering that makes the
// C -> B fragment exchange two vector stores and two vector loads, the observation words in the
// layout of a lane's result words, clamp fix-ups.  Pure host C++; deterministic.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "sa_plan.h"

namespace tsa {

struct DensePlan {
  bool ok = false;
  std::string why;          // reason when !ok
  int MT = 0, KS = 0;       // 16-row tiles, 32-column steps (KS = result words per condition and thread group)
  bool swizzle = false;     // swizzled exchange buffer (KS = 4, one warp per chain): 16 instead of 24 wavefronts per exchange
  bool movm = false;        // register exchange (movmatrix) instead of the shared-memory buffer (one warp per chain)
  uint32_t fix_words = 0;   // register exchange: result words w (bit w) that hold a clamped (condition, node) entry
  bool sparse = false;      // 2:4-sparse A operand (mma.sp m16n8k64): nodes permuted so that every row has <= 2 candidates per 4 columns
  int W = 1;                // warps per chain; warp ww owns result words ww*KS/W .. and their row tiles
  int CS = 0, TS = 0;       // byte strides of the exchange buffer: per condition, per B-fragment thread chunk
  int exchange_wavefronts = 0;   // shared-memory wavefronts of one exchange (2 stores + 2 loads)
  uint32_t skip_blocks = 0; // bit (row tile * column steps + column step): no candidate edge in that block of the matrix
  int obs_words = 0;        // result words w < obs_words hold the scored entries (observed nodes are numbered first)
  int n_fix_rounds = 1;
  int fit_const = 0;
  std::vector<uint16_t> frag_slot;   // [2*KS * (sparse ? KS/2 : KS) * 4][32][4] (row tiles padded to 2*KS)
  std::vector<uint32_t> meta;        // sparse: [2*KS * KS/2][32] selector words, one per tile and lane
  std::vector<uint16_t> th_entry;    // [8][KS][4]
  std::vector<uint32_t> init_frag;   // [32][2*KS]
  std::vector<uint32_t> obs_word;    // [n_obs][32][KS][2]
  std::vector<uint32_t> fix;         // [W][n_fix_rounds][32]; register exchange: [n_fix_rounds][2][2][32] keep / value masks
  std::vector<uint32_t> wloc;        // [E]
  std::vector<uint32_t> thloc;       // [N]
  size_t smem_bytes(const Plan& pl, int spec = 1) const {   // per chain, as CHAIN_SMEM in the kernel (spec = look-ahead warps)
    const size_t xbytes = (size_t)(W > 1 ? 2 : 1) * (movm ? 0 : swizzle ? 1024 : 8 * CS);
    return ((size_t)spec * xbytes + (size_t)pl.EpadA + (size_t)pl.NpadA + (size_t)(2 * W + 8 + (spec > 1 ? 2 * spec : 0)) * 4 + 15) / 16 * 16;
  }
};

// Applies when N <= 128 and K <= 8.  team_warps = warps per chain (1, 2 or 4; reduced until it
// divides KS).  Always returns; check dp->ok / dp->why.
void build_dense_plan(const sa_network* net, const sa_observations* obs, const Plan& plan, int team_warps, bool want_sparse,
                      bool want_swizzle, bool want_movm, DensePlan* dp);

}  // namespace tsa
