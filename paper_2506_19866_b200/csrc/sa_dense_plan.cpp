#include "sa_dense_plan.h"

#include <algorithm>
#include <map>

namespace tsa {

namespace {

constexpr uint32_t kStateScale = 64;   // the dense kernel exchanges a state s as the byte 64 * s (sa_dense_kernel.cu)

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

// Node -> row assignment for the 2:4-sparse layout.  Four consecutive matrix columns are the four rows
// that make up one result word of one thread group, {32w + g + 8x : x = 0..3} (see col_of_row below); a
// row of W may hold at most two candidate
// edges in any such group.  Local search over swaps and moves (deterministic), starting from the
// identity; returns false if some violation is left.
// movm: the register exchange's column numbering (a group = the rows 32w + 8h + 2t + {0, 1, 16, 17}).  A node of
// zone z stays in the rows below zone_end[z] (clamped and observed nodes are kept in the first result words).
// Optional pins (empty vectors = none): tile_req[node] >= 0 keeps the node in that row tile, reserved[tile] keeps every
// other node out of it; half_req[node] >= 0 keeps the node in rows whose column lies in that half (half_of_row).
bool assign_rows_2of4(const std::vector<std::vector<int>>& in_src, const std::vector<std::vector<int>>& out_dst,
                      int n_rows, bool movm, const std::vector<int>& zone, const int (&zone_end)[3],
                      const std::vector<int>& tile_req, const std::vector<int>& half_req, const std::vector<int>& half_of_row,
                      const std::vector<char>& reserved, std::vector<int>* row_of_node) {
  const int N = (int)in_src.size();
  std::vector<int>& row = *row_of_node;
  std::vector<int> node_at(n_rows, -1);
  for (int i = 0; i < N; ++i) node_at[row[i]] = i;
  auto group_of = [&](int r) { return movm ? (r / 32) * 8 + ((r % 16) / 8) * 4 + (r % 8) / 2 : (r / 32) * 8 + r % 8; };
  auto row_cost = [&](int i) {
    int cnt[64] = {0}, c = 0;
    for (int s : in_src[i]) if (++cnt[group_of(row[s])] > 2) ++c;
    return c;
  };
  long cost = 0;
  for (int i = 0; i < N; ++i) cost += row_cost(i);
  uint64_t st = 0x9E3779B97F4A7C15ull;
  auto rnd = [&](int n) {
    st ^= st >> 12; st ^= st << 25; st ^= st >> 27;
    return (int)((((st * 0x2545F4914F6CDD1Dull) >> 32) * (uint64_t)n) >> 32);
  };
  for (long it = 0; cost > 0 && it < 400000; ++it) {
    const int a = rnd(N), r2 = rnd(n_rows), b = node_at[r2];
    if (r2 == row[a] || (b >= 0 && group_of(row[b]) == group_of(row[a]))) continue;
    if (r2 >= zone_end[zone[a]] || (b >= 0 && row[a] >= zone_end[zone[b]])) continue;
    if (!reserved.empty()) {
      auto ok = [&](int node, int r) {
        if (tile_req[node] >= 0 ? r / 16 != tile_req[node] : reserved[r / 16] != 0) return false;
        return half_req[node] < 0 || half_of_row[r] == half_req[node];
      };
      if (!ok(a, r2) || (b >= 0 && !ok(b, row[a]))) continue;
    }
    long before = 0, after = 0;
    for (int i : out_dst[a]) before += row_cost(i);
    if (b >= 0) for (int i : out_dst[b]) before += row_cost(i);
    const int ra = row[a];
    row[a] = r2; if (b >= 0) row[b] = ra;
    for (int i : out_dst[a]) after += row_cost(i);
    if (b >= 0) for (int i : out_dst[b]) after += row_cost(i);
    if (after <= before) {                 // rows fed by both a and b are counted twice on both sides
      node_at[r2] = a; node_at[ra] = b;
      cost = 0;
      for (int i = 0; i < N; ++i) cost += row_cost(i);
    } else {
      row[a] = ra; if (b >= 0) row[b] = r2;
    }
  }
  return cost == 0;
}

}  // namespace

void build_dense_plan(const sa_network* net, const sa_observations* obs, const Plan& pl, int team_warps, bool want_sparse,
                      bool want_swizzle, bool want_movm, DensePlan* dp) {
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
  dp->movm = want_movm && W == 1;
  dp->swizzle = want_swizzle && KS == 4 && W == 1 && !dp->movm;
  if (dp->swizzle) dp->exchange_wavefronts = 16;
  if (dp->movm) dp->exchange_wavefronts = 0;

  // Row r = 16m + 8h + g (row tile m, half h) is produced by thread group g.  The tiles 2w and 2w+1 share one
  // accumulator (the odd tile's sums arrive 256-fold), whose registers c / 2+c are the halves h = 0 / 1, and the
  // word is acc[c] + 65536 * acc[2+c]: so the row is byte j = 2h + (m & 1) of word w = m / 2.
  // That byte is stored at chunk t' = g % 4, word pos = (g / 4) * NW + w, which B-fragment thread t'
  // reads as column k = 16*pos + 4t' + j.
  // Register exchange (movm): the low (h = 0) / high (h = 1) halves of the words (0, w), (1, w) travel through one
  // 8 x 8 transpose each and arrive as B-fragment word 2w + h of lane (g', t'), whose bytes are the rows
  // 16(2w + (j & 1)) + 8h + 2t' + (j >> 1): column k = 16(2w + h) + 4t' + j.
  auto col_of_row = [&](int r) {
    const int m = r / 16, h = (r % 16) / 8, g = r % 8, w = m / 2, j = 2 * h + (m & 1);
    if (dp->movm) return 16 * (2 * w + h) + 4 * (g / 2) + (m & 1) + 2 * (g & 1);
    const int pos = (g / 4) * NW + w;
    return 16 * pos + 4 * (g % 4) + j;
  };
  auto row_of_byte = [&](int g, int w, int j) { return 16 * (2 * w + (j & 1)) + 8 * (j >> 1) + g; };
  // node -> row: the identity, or (sparse layout) a permutation that puts at most two of any node's
  // sources into the same group of four columns
  std::vector<int> row_of_node(N);
  for (int i = 0; i < N; ++i) row_of_node[i] = i;
  // Zones: clamped nodes first (register exchange only: the result words that need a fix-up are then few), then the
  // other observed nodes (only the first result words are scored), then the rest; 32 rows per result word.
  std::vector<int> zone(N, 2);
  int zone_end[3] = {0, 0, 16 * MT};
  {
    int n0 = 0, n1 = 0;
    for (int i = 0; i < N; ++i) {
      bool clamped = false, observed = false;
      for (int k = 0; k < K; ++k) {
        if (obs->clamp[(size_t)k * N + i]) { clamped = true; continue; }
        if (obs->obs)
          for (int oj = 0; oj < NO; ++oj) observed |= obs->obs[((size_t)k * NO + oj) * N + i] != SA_UNOBSERVED;
      }
      zone[i] = (clamped && dp->movm) ? 0 : observed ? 1 : 2;
      n0 += zone[i] == 0; n1 += zone[i] == 1;
    }
    zone_end[0] = std::min(16 * MT, (n0 + 31) / 32 * 32);
    zone_end[1] = std::min(16 * MT, (n0 + n1 + 31) / 32 * 32);
    int next[3] = {0, n0, n0 + n1};
    for (int i = 0; i < N; ++i) row_of_node[i] = next[zone[i]]++;
  }
  if (want_sparse && KS % 2 == 0) {
    std::vector<std::vector<int>> in_src(N), out_dst(N);
    for (int e = 0; e < E; ++e) { in_src[net->edge_dst[e]].push_back(net->edge_src[e]); out_dst[net->edge_src[e]].push_back(net->edge_dst[e]); }
    // Empty blocks (see skip_blocks below): a row tile whose nodes take ALL their sources from one half of the columns
    // leaves its other block of the weight matrix without a candidate edge, and that block's IMMA is left out.
    // T = the few nodes of the last row tile (unobserved ones of small in-degree), X = a whole tile of 16 more nodes,
    // both chosen greedily so that the union S of their sources stays small; T and X are pinned to their tiles, S to
    // one half of the columns, and the 2:4 search runs under those pins.  Attempts: T and X (two blocks), T alone
    // (one), then the plain search.
    bool done = false;
    const int n_last = N - 16 * (MT - 1);
    const bool small_last = n_last >= 1 && n_last <= 8;       // else: X alone (one block)
    if (KS == 4 && !dp->movm && MT >= 3) {
      const int n_rows = 16 * MT;
      std::vector<int> half_of_row(n_rows);
      for (int r = 0; r < n_rows; ++r) half_of_row[r] = col_of_row(r) / 64;
      std::vector<std::vector<char>> src_of(N, std::vector<char>(N, 0));
      for (int i = 0; i < N; ++i) for (int sidx : in_src[i]) src_of[i][sidx] = 1;
      // greedy: add the node that enlarges the union of sources least (ties: smaller in-degree, lower index)
      auto grow = [&](std::vector<char>& chosen, std::vector<char>& uni, int count, bool zone2_only) {
        for (int k = 0; k < count; ++k) {
          int best = -1, best_u = 1 << 30;
          for (int i = 0; i < N; ++i) {
            if (chosen[i] || (zone2_only && zone[i] != 2)) continue;
            int u = 0;
            for (int j = 0; j < N; ++j) u += (uni[j] || src_of[i][j]) ? 1 : 0;
            if (u < best_u || (u == best_u && in_src[i].size() < in_src[best].size())) { best_u = u; best = i; }
          }
          if (best < 0) return false;
          chosen[best] = 1;
          for (int j = 0; j < N; ++j) uni[j] = uni[j] || src_of[best][j];
        }
        return true;
      };
      auto attempt = [&](const std::vector<int>& tile_req, const std::vector<int>& half_req, const std::vector<char>& reserved) {
        // constructive start: zone by zone, the pinned nodes first, the free ones preferably in the other half
        std::vector<int> trial(N, -1), node_at(n_rows, -1);
        auto put = [&](int node, int want_half, bool strict) {
          for (int r = 0; r < n_rows; ++r) {
            if (node_at[r] >= 0 || r >= zone_end[zone[node]]) continue;
            if (tile_req[node] >= 0 ? r / 16 != tile_req[node] : reserved[r / 16] != 0) continue;
            if (strict && want_half >= 0 && half_of_row[r] != want_half) continue;
            node_at[r] = node; trial[node] = r;
            return true;
          }
          return false;
        };
        int hs = -1;
        for (int i = 0; i < N; ++i) if (half_req[i] >= 0) hs = half_req[i];
        for (int z = 0; z < 3; ++z) {
          for (int i = 0; i < N; ++i) if (zone[i] == z && tile_req[i] >= 0 && !put(i, half_req[i], true)) return false;
          for (int i = 0; i < N; ++i) if (zone[i] == z && tile_req[i] < 0 && half_req[i] >= 0 && !put(i, half_req[i], true)) return false;
          for (int i = 0; i < N; ++i)
            if (zone[i] == z && tile_req[i] < 0 && half_req[i] < 0 && !put(i, 1 - hs, hs >= 0) && !put(i, -1, false)) return false;
        }
        if (!assign_rows_2of4(in_src, out_dst, n_rows, dp->movm, zone, zone_end, tile_req, half_req, half_of_row, reserved, &trial)) return false;
        row_of_node = trial;
        return true;
      };
      std::vector<char> in_t(N, 0), uni_t(N, 0);
      const bool have_t = !small_last || grow(in_t, uni_t, n_last, true);
      for (int variant = 0; variant < (small_last ? 2 : 1) && have_t && !done; ++variant) {   // 0: T and X (or X alone), 1: T alone
        std::vector<char> chosen = in_t, uni = uni_t;
        int x_tile = -1;
        if (variant == 0) {
          if (!grow(chosen, uni, 16, false)) continue;
          bool x_observed = false;
          for (int i = 0; i < N; ++i) x_observed = x_observed || (chosen[i] && !in_t[i] && zone[i] != 2);
          x_tile = x_observed ? zone_end[1] / 16 - 1 : small_last ? MT - 2 : MT - 1;
          if (x_tile < 0 || x_tile >= (small_last ? MT - 1 : MT)) continue;
        }
        for (int hs = 0; hs < 2 && !done; ++hs) {
          std::vector<int> tile_req(N, -1), half_req(N, -1);
          std::vector<char> reserved(MT, 0);
          if (small_last) reserved[MT - 1] = 1;
          if (x_tile >= 0) reserved[x_tile] = 1;
          for (int i = 0; i < N; ++i) {
            if (in_t[i]) tile_req[i] = MT - 1;
            else if (chosen[i]) tile_req[i] = x_tile;
            if (uni[i]) half_req[i] = hs;
          }
          done = attempt(tile_req, half_req, reserved);
        }
      }
      if (done) dp->sparse = true;
    }
    if (!done) {
      std::vector<int> trial = row_of_node;
      const std::vector<int> none;
      if (assign_rows_2of4(in_src, out_dst, 16 * MT, dp->movm, zone, zone_end, none, none, none, std::vector<char>(), &trial)) { row_of_node = trial; dp->sparse = true; }
    }
  }
  const int KSP = KS / 2;                            // sparse steps of 64 columns
  std::vector<int> node_of_row(32 * KS, -1), node_of_col(32 * KS, -1);
  for (int i = 0; i < N; ++i) { node_of_row[row_of_node[i]] = i; node_of_col[col_of_row(row_of_node[i])] = i; }
  auto state_offset = [&](int cond, int node) {     // byte of (cond, node) in the exchange buffer (shared-memory exchange only)
    const int k = col_of_row(row_of_node[node]), pos = k / 16, tq = (k % 16) / 4, j = k % 4;
    if (dp->swizzle)                                 // see the kernel: row 4*half + c/2, column from a Latin square
      return (4 * (pos / 4) + cond / 2) * 128 + (4 * (tq & 1) + ((cond / 2 + 2 * (tq / 2) + (cond & 1)) & 3)) * 16 + (pos % 4) * 4 + j;
    return cond * CS + tq * TS + pos * 4 + j;
  };
  std::map<std::pair<int, int>, int> edge_at;       // (dst, src) -> edge
  for (int e = 0; e < E; ++e) edge_at[{net->edge_dst[e], net->edge_src[e]}] = e;
  auto edge_of = [&](int row, int col) {            // candidate edge at matrix position (row, col) or -1
    if (node_of_row[row] < 0 || node_of_col[col] < 0) return -1;
    auto it = edge_at.find({node_of_row[row], node_of_col[col]});
    return it == edge_at.end() ? -1 : it->second;
  };
  dp->wloc.assign(E, 0u);
  auto place = [&](int e, int m, int wreg, int lane, int b, int global_reg) {
    const int slot = pl.slot_of_param[e];
    dp->frag_slot[((size_t)global_reg * 32 + lane) * 4 + b] = (uint16_t)slot;
    dp->wloc[e] = (uint32_t)wreg | ((uint32_t)b << 7) | ((uint32_t)lane << 9) | ((uint32_t)(m / MTW) << 14) | ((uint32_t)slot << 16);
  };
  const int tiles = 2 * NW;                          // row tiles padded to whole warps
  if (!dp->sparse) {
    // dense A fragments: register (m, s, a) of lane (g, t) holds row 16m + g + 8(a&1), columns 32s + 16(a>>1) + 4t + 0..3;
    // row tile m belongs to warp m / MTW as its tile m % MTW
    dp->frag_slot.assign((size_t)tiles * KS * 4 * 32 * 4, 0xFFFFu);
    for (int m = 0; m < tiles; ++m)
      for (int s = 0; s < KS; ++s)
        for (int a = 0; a < 4; ++a)
          for (int lane = 0; lane < 32; ++lane)
            for (int b = 0; b < 4; ++b) {
              const int g = lane / 4, t = lane % 4;
              const int e = edge_of(16 * m + g + 8 * (a & 1), 32 * s + 16 * (a >> 1) + 4 * t + b);
              if (e >= 0) place(e, m, ((m % MTW) * KS + s) * 4 + a, lane, b, (m * KS + s) * 4 + a);
            }
    dp->meta.assign(32, 0u);
  } else {
    // 2:4-sparse A (mma.sp m16n8k64, layout measured on sm_100a): tile (m, sp) covers columns 64sp .. 64sp+63
    // in 16 groups of four.  Per row and group two slots are stored: byte 2*(G%2) + slot of register
    // a = 2*(G/8) + half in lane 4g + (G%8)/2, and a 4-bit selector (position of slot 0, position of
    // slot 1 << 2, ascending) in nibble G%8 of the metadata word of lane 4g + 2*(G/8) + half.
    dp->frag_slot.assign((size_t)tiles * KSP * 4 * 32 * 4, 0xFFFFu);
    dp->meta.assign((size_t)tiles * KSP * 32, 0u);
    for (int m = 0; m < tiles; ++m)
      for (int sp = 0; sp < KSP; ++sp)
        for (int g = 0; g < 8; ++g)
          for (int half = 0; half < 2; ++half)
            for (int G = 0; G < 16; ++G) {
              int pos[4], edges[4], n = 0;
              for (int pp = 0; pp < 4; ++pp) {
                const int e = edge_of(16 * m + g + 8 * half, 64 * sp + 4 * G + pp);
                if (e >= 0) { pos[n] = pp; edges[n] = e; ++n; }
              }
              if (n > 2) { dp->why = "internal error: more than two candidate edges in a 2:4 group"; return; }
              int idx0 = 0, idx1 = 1, e0 = -1, e1 = -1;
              if (n == 2) { idx0 = pos[0]; idx1 = pos[1]; e0 = edges[0]; e1 = edges[1]; }
              else if (n == 1 && pos[0] < 3) { idx0 = pos[0]; idx1 = pos[0] + 1; e0 = edges[0]; }
              else if (n == 1) { idx0 = 2; idx1 = 3; e1 = edges[0]; }
              const int tile = m * KSP + sp, a = 2 * (G / 8) + half, lane = 4 * g + (G % 8) / 2;
              dp->meta[(size_t)tile * 32 + 4 * g + 2 * (G / 8) + half] |= (uint32_t)(idx0 | (idx1 << 2)) << (4 * (G % 8));
              const int wreg = ((m % MTW) * KSP + sp) * 4 + a;
              if (e0 >= 0) place(e0, m, wreg, lane, 2 * (G % 2), tile * 4 + a);
              if (e1 >= 0) place(e1, m, wreg, lane, 2 * (G % 2) + 1, tile * 4 + a);
            }
  }
  // blocks of the matrix (row tile x column step of the MMA) without any candidate edge: their IMMA is left out
  {
    const int KK = dp->sparse ? KSP : KS, cols = dp->sparse ? 64 : 32;
    std::vector<char> used((size_t)MT * KK, 0);
    for (int e = 0; e < E; ++e) {
      const int r = row_of_node[net->edge_dst[e]], c = col_of_row(row_of_node[net->edge_src[e]]);
      used[(size_t)(r / 16) * KK + c / cols] = 1;
    }
    dp->skip_blocks = 0;
    for (int m = 0; m < MT; ++m)
      for (int k = 0; k < KK; ++k)
        if (!used[(size_t)m * KK + k] && m * KK + k < 32) dp->skip_blocks |= 1u << (m * KK + k);
  }
  // thresholds: byte j of word w of thread group g <-> row_of_byte(g, w, j)
  dp->th_entry.assign((size_t)8 * NW * 4, 0xFFFFu);
  dp->thloc.assign(N, 0u);
  for (int g = 0; g < 8; ++g)
    for (int w = 0; w < NW; ++w)
      for (int j = 0; j < 4; ++j) {
        const int row = row_of_byte(g, w, j);
        if (row >= 16 * MT || node_of_row[row] < 0) continue;
        const int node = node_of_row[row], entry = pl.entry_of_node[node];
        dp->th_entry[((size_t)g * NW + w) * 4 + j] = (uint16_t)entry;
        dp->thloc[node] = (uint32_t)g | ((uint32_t)w << 3) | ((uint32_t)j << 5) | ((uint32_t)entry << 16);
      }
  // t = 0 states (as the bytes 64 * s, like every state the kernel exchanges) as B fragments: lane (g', t') word
  // pos = columns 16 pos + 4t' + 0..3 of condition g'
  dp->init_frag.assign((size_t)32 * 2 * KS, 0u);
  for (int lane = 0; lane < 32; ++lane)
    for (int x = 0; x < 2 * KS; ++x)
      for (int j = 0; j < 4; ++j) {
        const int cond = lane / 4, col = 16 * x + 4 * (lane % 4) + j;
        if (cond >= K || node_of_col[col] < 0) continue;
        dp->init_frag[(size_t)lane * 2 * KS + x] |= ((uint32_t)obs->init_state[(size_t)cond * N + node_of_col[col]] * kStateScale) << (8 * j);
      }
  // clamped (condition, node): restored by a byte store after every exchange; scored once, here
  // (the warp that owns the row's result word stores it, right after its own vector stores)
  if (dp->movm) {
    // register exchange: per result word w that holds a clamped entry (bit w of fix_words), per c = 0, 1 and lane:
    // the bytes to keep and the bytes 64 * value to set, [(2f + c) * 2 + {keep, value}][32]
    dp->fix_words = 0;
    for (int k = 0; k < K; ++k)
      for (int i = 0; i < N; ++i)
        if (obs->clamp[(size_t)k * N + i]) dp->fix_words |= 1u << (row_of_node[i] / 32);
    int fidx[8], nf = 0;
    for (int w = 0; w < NW; ++w) fidx[w] = ((dp->fix_words >> w) & 1u) ? nf++ : -1;
    dp->n_fix_rounds = std::max(1, nf);
    dp->fix.assign((size_t)dp->n_fix_rounds * 4 * 32, 0u);
    for (int f = 0; f < dp->n_fix_rounds; ++f)
      for (int c = 0; c < 2; ++c)
        for (int lane = 0; lane < 32; ++lane) dp->fix[((size_t)(2 * f + c) * 2) * 32 + lane] = 0xFFFFFFFFu;
    for (int k = 0; k < K; ++k)
      for (int i = 0; i < N; ++i)
        if (obs->clamp[(size_t)k * N + i]) {
          const int r = row_of_node[i], m = r / 16, w = m / 2, j = 2 * ((r % 16) / 8) + (m & 1), g = r % 8;
          const int lane = 4 * g + k / 2, c = k & 1, f = fidx[w];
          dp->fix[((size_t)(2 * f + c) * 2) * 32 + lane] &= ~(0xFFu << (8 * j));
          dp->fix[((size_t)(2 * f + c) * 2 + 1) * 32 + lane] |= ((uint32_t)obs->init_state[(size_t)k * N + i] * kStateScale) << (8 * j);
        }
  } else {
    std::vector<std::vector<uint32_t>> fixes(W);
    for (int k = 0; k < K; ++k)
      for (int i = 0; i < N; ++i)
        if (obs->clamp[(size_t)k * N + i]) {
          const int ww = (row_of_node[i] / 32) / WPW;
          fixes[ww].push_back((uint32_t)state_offset(k, i) | ((uint32_t)obs->init_state[(size_t)k * N + i] << 16) | 0x80000000u);
        }
    dp->n_fix_rounds = 1;
    for (int ww = 0; ww < W; ++ww) dp->n_fix_rounds = std::max(dp->n_fix_rounds, (int)(fixes[ww].size() + 31) / 32);
    dp->fix.assign((size_t)W * dp->n_fix_rounds * 32, 0u);
    for (int ww = 0; ww < W; ++ww) std::copy(fixes[ww].begin(), fixes[ww].end(), dp->fix.begin() + (size_t)ww * dp->n_fix_rounds * 32);
  }
  // observations in the layout of a lane's result words ([w][c] per lane and time), as the bytes 64 * value; 3 = never
  // equal to a state, so such an entry always counts one mismatch, which fit_const takes back.  Only the words
  // w < obs_words hold a scored entry; the kernel looks at no other.
  dp->obs_words = 0;
  if (obs->obs)
    for (int i = 0; i < N; ++i) {
      bool scored = false;
      for (int k = 0; k < K; ++k)
        for (int oj = 0; oj < NO; ++oj)
          scored |= !obs->clamp[(size_t)k * N + i] && obs->obs[((size_t)k * NO + oj) * N + i] != SA_UNOBSERVED;
      if (scored) dp->obs_words = std::max(dp->obs_words, row_of_node[i] / 32 + 1);
    }
  dp->obs_word.assign((size_t)NO * 32 * 2 * NW, 0x01010101u * (3u * kStateScale));
  long always = (long)NO * 32 * 2 * dp->obs_words * 4, clamped_mis = 0;
  if (obs->obs) {
    for (int oj = 0; oj < NO; ++oj)
      for (int lane = 0; lane < 32; ++lane)
        for (int c = 0; c < 2; ++c)
          for (int w = 0; w < NW; ++w)
            for (int j = 0; j < 4; ++j) {
              const int g = lane / 4, t = lane % 4, cond = 2 * t + c, row = row_of_byte(g, w, j);
              if (row >= 16 * MT || node_of_row[row] < 0 || cond >= K) continue;
              const int node = node_of_row[row];
              const uint8_t o = obs->obs[((size_t)cond * NO + oj) * N + node];
              if (o == SA_UNOBSERVED) continue;
              if (obs->clamp[(size_t)cond * N + node]) {
                if (o != obs->init_state[(size_t)cond * N + node]) ++clamped_mis;
                continue;
              }
              uint32_t& word = dp->obs_word[((size_t)oj * 32 + lane) * 2 * NW + 2 * w + c];
              word = (word & ~(0xFFu << (8 * j))) | (((uint32_t)o * kStateScale) << (8 * j));
              --always;
            }
  }
  dp->fit_const = (int)(clamped_mis - always);
  {                                                  // self-check: every edge sits in exactly one fragment byte
    std::vector<int> seen(pl.EpadA, 0);
    for (uint16_t s : dp->frag_slot) if (s != 0xFFFFu) ++seen[s];
    for (int e = 0; e < E; ++e)
      if (seen[pl.slot_of_param[e]] != 1) { dp->why = "internal error: edge not placed exactly once"; return; }
  }
  dp->ok = true;
}

}  // namespace tsa
