#include "sa_dense_plan.h"

#include <algorithm>
#include <map>

namespace tsa {

namespace {

// Shared-memory wavefronts of one warp-wide vector access (hardware serves 128 bytes per wavefront:
// a quarter-warp of 16-byte accesses, a half-warp of 8-byte ones, the whole warp of 4-byte ones).
int wavefronts(const int (&addr)[32], int vec_bytes) {
  const int per = vec_bytes == 16 ? 8 : vec_bytes == 8 ? 16 : 32;
  int total = 0;
  for (int p = 0; p < 32; p += per) {
    int words[32][4], cnt[32] = {0};
    for (int l = p; l < p + per; ++l)
      for (int b = addr[l] / 4; b < (addr[l] + vec_bytes) / 4; ++b) {
        const int bank = b % 32;
        bool seen = false;
        for (int x = 0; x < cnt[bank]; ++x) seen |= (words[bank][x] == b);
        if (!seen && cnt[bank] < 4) words[bank][cnt[bank]++] = b;
      }
    int worst = 1;
    for (int b = 0; b < 32; ++b) worst = std::max(worst, cnt[b]);
    total += worst;
  }
  return total;
}

// Strides (CS per condition, TS per B-thread chunk) of the exchange buffer with the fewest
// wavefronts for the kernel's two stores and two loads.
void pick_strides(int KS, int W, int* CS, int* TS, int* wf) {
  const int NW = KS, vec = NW * 4, WPW = NW / W, svec = WPW * 4;
  int best = 1 << 30;
  for (int ts = 2 * KS * 4; ts <= 2 * KS * 4 + 128; ts += 4) {
    if (ts % vec) continue;
    for (int cs = 4 * ts; cs <= 4 * ts + 256; cs += 4) {
      if (cs % vec || (8 * cs) % 16) continue;
      int w = 0, addr[32];
      for (int c = 0; c < 2; ++c)
        for (int ww = 0; ww < W; ++ww) {
          for (int l = 0; l < 32; ++l)
            addr[l] = (2 * (l % 4) + c) * cs + ((l / 4) % 4) * ts + (((l / 4) / 4) * NW + ww * WPW) * 4;
          w += wavefronts(addr, svec);
        }
      for (int half = 0; half < 2; ++half) {
        for (int l = 0; l < 32; ++l) addr[l] = (l / 4) * cs + (l % 4) * ts + half * NW * 4;
        w += W * wavefronts(addr, vec);
      }
      if (w < best) { best = w; *CS = cs; *TS = ts; }
    }
  }
  *wf = best;
}

}  // namespace

void build_dense_plan(const sa_network* net, const sa_observations* obs, const Plan& pl, int team_warps, DensePlan* dp) {
  *dp = DensePlan();
  const int N = pl.N, E = pl.E, K = pl.K, NO = pl.n_obs;
  if (N > 128) { dp->why = "more than 128 nodes"; return; }
  if (K > 8) { dp->why = "more than 8 conditions"; return; }
  if (pl.EpadA > 65534 || pl.NpadA > 65534) { dp->why = "canonical rows exceed 16-bit offsets"; return; }
  const int MT = (N + 15) / 16;
  int KS = (MT + 1) / 2;
  if (KS == 3) KS = 4;
  const int NW = KS;
  int W = team_warps >= 4 ? 4 : team_warps >= 2 ? 2 : 1;
  while (W > KS) W /= 2;
  const int WPW = NW / W, MTW = 2 * WPW;
  dp->MT = MT; dp->KS = KS; dp->W = W;
  pick_strides(KS, W, &dp->CS, &dp->TS, &dp->exchange_wavefronts);
  const int CS = dp->CS, TS = dp->TS;

  // Row r = 16m + 8h + g is produced by thread group g as byte j of its word w, q = 2m + h = 4w + j.
  // That byte is stored at chunk t' = g % 4, word pos = (g / 4) * NW + w, which B-fragment thread t'
  // reads as column k = 32*(pos/2) + 16*(pos%2) + 4t' + j.  Node i sits at row i.
  auto col_of_row = [&](int r) {
    const int m = r / 16, h = (r % 16) / 8, g = r % 8, q = 2 * m + h, w = q / 4, j = q % 4;
    const int pos = (g / 4) * NW + w;
    return 32 * (pos / 2) + 16 * (pos % 2) + 4 * (g % 4) + j;
  };
  auto state_offset = [&](int cond, int node) {     // byte of (cond, node) in the exchange buffer
    const int k = col_of_row(node), s = k / 32, hf = (k % 32) / 16, tq = (k % 16) / 4, j = k % 4;
    return cond * CS + tq * TS + (2 * s + hf) * 4 + j;
  };
  std::vector<int> node_of_col(32 * KS, -1);
  for (int i = 0; i < N; ++i) node_of_col[col_of_row(i)] = i;

  // A fragments: register (m, s, a) of lane (g, t) holds row 16m + g + 8(a&1), columns 32s + 16(a>>1) + 4t + 0..3;
  // row tile m belongs to warp m / MTW as its tile m % MTW
  std::map<std::pair<int, int>, int> edge_at;       // (dst, src) -> edge
  for (int e = 0; e < E; ++e) edge_at[{net->edge_dst[e], net->edge_src[e]}] = e;
  const int NA = 2 * NW * KS * 4;
  dp->frag_slot.assign((size_t)NA * 32 * 4, 0xFFFFu);
  dp->wloc.assign(E, 0u);
  for (int m = 0; m < 2 * NW; ++m)
    for (int s = 0; s < KS; ++s)
      for (int a = 0; a < 4; ++a)
        for (int lane = 0; lane < 32; ++lane)
          for (int b = 0; b < 4; ++b) {
            const int g = lane / 4, t = lane % 4, reg = (m * KS + s) * 4 + a;
            const int row = 16 * m + g + 8 * (a & 1), col = 32 * s + 16 * (a >> 1) + 4 * t + b;
            if (row >= N || node_of_col[col] < 0) continue;
            auto it = edge_at.find({row, node_of_col[col]});
            if (it == edge_at.end()) continue;
            const int e = it->second, slot = pl.slot_of_param[e];
            dp->frag_slot[((size_t)reg * 32 + lane) * 4 + b] = (uint16_t)slot;
            const int ww = m / MTW, wreg = ((m % MTW) * KS + s) * 4 + a;
            dp->wloc[e] = (uint32_t)wreg | ((uint32_t)b << 7) | ((uint32_t)lane << 9) | ((uint32_t)ww << 14) | ((uint32_t)slot << 16);
          }
  // thresholds: byte j of word w of thread group g <-> row
  dp->th_entry.assign((size_t)8 * NW * 4, 0xFFFFu);
  dp->thloc.assign(N, 0u);
  for (int g = 0; g < 8; ++g)
    for (int w = 0; w < NW; ++w)
      for (int j = 0; j < 4; ++j) {
        const int q = 4 * w + j, row = 16 * (q / 2) + 8 * (q % 2) + g;
        if (row >= N || q / 2 >= MT) continue;
        const int entry = pl.entry_of_node[row];
        dp->th_entry[((size_t)g * NW + w) * 4 + j] = (uint16_t)entry;
        dp->thloc[row] = (uint32_t)g | ((uint32_t)w << 3) | ((uint32_t)j << 5) | ((uint32_t)entry << 16);
      }
  // t = 0 states as B fragments: lane (g', t') word 2s + hf = columns 32s + 16hf + 4t' + 0..3 of condition g'
  dp->init_frag.assign((size_t)32 * 2 * KS, 0u);
  for (int lane = 0; lane < 32; ++lane)
    for (int x = 0; x < 2 * KS; ++x)
      for (int j = 0; j < 4; ++j) {
        const int cond = lane / 4, col = 32 * (x / 2) + 16 * (x % 2) + 4 * (lane % 4) + j;
        if (cond >= K || node_of_col[col] < 0) continue;
        dp->init_frag[(size_t)lane * 2 * KS + x] |= (uint32_t)obs->init_state[(size_t)cond * N + node_of_col[col]] << (8 * j);
      }
  // clamped (condition, node): restored by a byte store after every exchange; scored once, here
  // (the warp that owns the row's result word stores it, right after its own vector stores)
  std::vector<std::vector<uint32_t>> fixes(W);
  for (int k = 0; k < K; ++k)
    for (int i = 0; i < N; ++i)
      if (obs->clamp[(size_t)k * N + i]) {
        const int q = 2 * (i / 16) + (i % 16) / 8, ww = (q / 4) / WPW;
        fixes[ww].push_back((uint32_t)state_offset(k, i) | ((uint32_t)obs->init_state[(size_t)k * N + i] << 16) | 0x80000000u);
      }
  dp->n_fix_rounds = 1;
  for (int ww = 0; ww < W; ++ww) dp->n_fix_rounds = std::max(dp->n_fix_rounds, (int)(fixes[ww].size() + 31) / 32);
  dp->fix.assign((size_t)W * dp->n_fix_rounds * 32, 0u);
  for (int ww = 0; ww < W; ++ww) std::copy(fixes[ww].begin(), fixes[ww].end(), dp->fix.begin() + (size_t)ww * dp->n_fix_rounds * 32);
  // observations in the layout of a lane's result words; 3 = never equal to a state, so such an
  // entry always counts one mismatch, which fit_const takes back
  dp->obs_word.assign((size_t)NO * 32 * 2 * NW, 0x03030303u);
  long always = (long)NO * 32 * 2 * NW * 4, clamped_mis = 0;
  if (obs->obs) {
    for (int oj = 0; oj < NO; ++oj)
      for (int lane = 0; lane < 32; ++lane)
        for (int c = 0; c < 2; ++c)
          for (int w = 0; w < NW; ++w)
            for (int j = 0; j < 4; ++j) {
              const int g = lane / 4, t = lane % 4, cond = 2 * t + c, q = 4 * w + j, row = 16 * (q / 2) + 8 * (q % 2) + g;
              if (row >= N || q / 2 >= MT || cond >= K) continue;
              const uint8_t o = obs->obs[((size_t)cond * NO + oj) * N + row];
              if (o == SA_UNOBSERVED) continue;
              if (obs->clamp[(size_t)cond * N + row]) {
                if (o != obs->init_state[(size_t)cond * N + row]) ++clamped_mis;
                continue;
              }
              uint32_t& word = dp->obs_word[((size_t)oj * 32 + lane) * 2 * NW + c * NW + w];
              word = (word & ~(0xFFu << (8 * j))) | ((uint32_t)o << (8 * j));
              --always;
            }
  }
  dp->fit_const = (int)(clamped_mis - always);
  dp->ok = true;
}

}  // namespace tsa
