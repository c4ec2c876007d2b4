#include "sa_tuning.h"
#include "sa_plan.h"

#include "sa_common.h"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <numeric>
#include <queue>
#include <unordered_set>

namespace tsa {

namespace {

int fail(std::string* err, const std::string& msg) {
  if (err) *err = msg;
  return SA_EINVAL;
}

struct Rng {   // xorshift64*, fixed seed: plans are reproducible
  uint64_t s = 0x9E3779B97F4A7C15ull;
  uint32_t next() {
    s ^= s >> 12; s ^= s << 25; s ^= s >> 27;
    return (uint32_t)((s * 0x2545F4914F6CDD1Dull) >> 32);
  }
  int below(int n) { return (int)(((uint64_t)next() * (uint64_t)n) >> 32); }
};

struct Row {
  int node = -1;            // -1 = idle lane
  std::vector<int> edges;   // caller edge ids
  bool head = false;
  int part = 0, parts = 1;
};

// One candidate layout: rows packed into passes (32 lanes each), lanes in final order.
struct Layout {
  std::vector<std::vector<Row>> passes;
  std::vector<int> rounds;   // combine rounds per pass
};

// Step A + B: split long rows until the row budget is used, pack blocks into passes.
Layout make_layout(const std::vector<std::vector<int>>& in_edges, int budget_rows, bool split) {
  const int N = (int)in_edges.size();
  std::vector<int> parts(N, 1);
  if (split) {
    auto len = [&](int i) { return ((int)in_edges[i].size() + parts[i] - 1) / parts[i]; };
    std::priority_queue<std::pair<int, int>> heap;   // (sub-row length, -node)
    for (int i = 0; i < N; ++i) heap.push({len(i), -i});
    int total = N;
    while (total < budget_rows && !heap.empty()) {
      auto [l, negi] = heap.top();
      heap.pop();
      const int i = -negi;
      if (l <= 2) break;                       // nothing worth splitting is left
      if (parts[i] >= 32) continue;
      ++parts[i];
      ++total;
      heap.push({len(i), -i});
    }
  }
  struct Block { int node, len; };
  std::vector<Block> blocks(N);
  for (int i = 0; i < N; ++i) blocks[i] = {i, ((int)in_edges[i].size() + parts[i] - 1) / parts[i]};
  std::stable_sort(blocks.begin(), blocks.end(), [](const Block& a, const Block& b) { return a.len > b.len; });

  Layout lay;
  std::vector<char> placed(N, 0);
  int remaining = N;
  while (remaining > 0) {
    std::vector<Row> rows;
    int maxparts = 1;
    for (const Block& b : blocks) {
      if (placed[b.node]) continue;
      const int m = parts[b.node];
      if ((int)rows.size() + m > 32) continue;
      const auto& ed = in_edges[b.node];
      const int d = (int)ed.size(), q = d / m, r = d % m;   // first r parts get q+1 edges
      int pos = 0;
      for (int a = 0; a < m; ++a) {
        Row row;
        row.node = b.node; row.head = (a == 0); row.part = a; row.parts = m;
        const int cnt = q + (a < r ? 1 : 0);
        row.edges.assign(ed.begin() + pos, ed.begin() + pos + cnt);
        pos += cnt;
        rows.push_back(std::move(row));
      }
      maxparts = std::max(maxparts, m);
      placed[b.node] = 1;
      --remaining;
      if ((int)rows.size() == 32) break;
    }
    rows.resize(32);
    int rounds = 0;
    while ((1 << rounds) < maxparts) ++rounds;
    lay.passes.push_back(std::move(rows));
    lay.rounds.push_back(rounds);
  }
  return lay;
}

// Step C: bank classes.  cls[v] in [0, nb) for v < Nv (real nodes first, then virtual fillers so
// that every class has exactly Nv/nb members).  Minimises the shared-memory wavefronts of a time step: per pass CG x
// (max over its groups of max(longest row, heaviest bank)) for the gathers plus, per group, the largest number of its
// lanes that store to the same class (every lane stores one entry per pass: its node's, or its private scratch
// entry); ties broken by sum of squared loads.
struct BankOpt {
  int nb, CG, n_groups;
  std::vector<int> rowmax;                          // [group]
  std::vector<std::vector<std::pair<int, int>>> feeds;   // node -> (group, #edges into it)
  std::vector<int> load;                            // [group][nb]
  std::vector<int> gcost;                           // [group]
  std::vector<int> sgroup;                          // node -> group of the lane that stores its entry (-1: virtual filler)
  std::vector<int> scount;                          // [group][nb] lanes of the group that store to the class
  std::vector<int> smax;                            // [group]
  long long sumsq = 0;

  int store_cost(int g) const {
    int m = 0;
    for (int c = 0; c < nb; ++c) m = std::max(m, scount[(size_t)g * nb + c]);
    return m;
  }

  int group_cost(int g) const {
    int m = rowmax[g];
    for (int c = 0; c < nb; ++c) m = std::max(m, load[(size_t)g * nb + c]);
    return m;
  }
  long long primary() const {
    long long t = 0;
    for (int p = 0; p * CG < n_groups; ++p) {
      int m = 0;
      for (int g = p * CG; g < (p + 1) * CG; ++g) m = std::max(m, gcost[g]);
      t += (long long)CG * m;
      for (int g = p * CG; g < (p + 1) * CG; ++g) t += smax[g];
    }
    return t;
  }
  void move(int v, int from, int to) {
    if (sgroup[v] >= 0) { --scount[(size_t)sgroup[v] * nb + from]; ++scount[(size_t)sgroup[v] * nb + to]; }
    for (auto [g, cnt] : feeds[v]) {
      int& a = load[(size_t)g * nb + from];
      int& b = load[(size_t)g * nb + to];
      sumsq -= (long long)a * a + (long long)b * b;
      a -= cnt; b += cnt;
      sumsq += (long long)a * a + (long long)b * b;
    }
  }
};

std::vector<int> assign_classes(const Layout& lay, const int32_t* edge_src, int N, int CG, bool optimise, bool count_stores,
                                std::vector<int>* pass_iters) {
  const int nb = 32 / CG;
  const int n_pass = (int)lay.passes.size();
  BankOpt bo;
  bo.nb = nb; bo.CG = CG; bo.n_groups = n_pass * CG;
  bo.rowmax.assign(bo.n_groups, 0);
  const int per_class = (N + nb - 1) / nb, Nv = per_class * nb;
  bo.feeds.assign(Nv, {});
  bo.sgroup.assign(Nv, -1);
  bo.scount.assign((size_t)bo.n_groups * nb, 0);
  for (int p = 0; p < n_pass; ++p)
    for (int l = 0; l < 32; ++l) {
      const Row& r = lay.passes[p][l];
      const int g = p * CG + l / nb;
      if (!count_stores) continue;
      if (r.node >= 0 && r.head) bo.sgroup[r.node] = g;
      else ++bo.scount[(size_t)g * nb + l % nb];      // scratch entry of lane l: class l mod nb
    }
  std::vector<int> outdeg(N, 0);
  {
    std::vector<std::vector<int>> cnt(bo.n_groups);   // sources feeding each group
    for (int p = 0; p < n_pass; ++p)
      for (int l = 0; l < 32; ++l) {
        const Row& r = lay.passes[p][l];
        const int g = p * CG + l / nb;
        bo.rowmax[g] = std::max(bo.rowmax[g], (int)r.edges.size());
        for (int e : r.edges) { cnt[g].push_back(edge_src[e]); ++outdeg[edge_src[e]]; }
      }
    for (int g = 0; g < bo.n_groups; ++g) {
      std::sort(cnt[g].begin(), cnt[g].end());
      for (size_t a = 0; a < cnt[g].size();) {
        size_t b = a;
        while (b < cnt[g].size() && cnt[g][b] == cnt[g][a]) ++b;
        bo.feeds[cnt[g][a]].push_back({g, (int)(b - a)});
        a = b;
      }
    }
  }
  // initial classes: nodes by descending out-degree dealt round-robin (balances the total load)
  std::vector<int> order(Nv);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
    return (a < N ? outdeg[a] : -1) > (b < N ? outdeg[b] : -1);
  });
  std::vector<int> cls(Nv);
  for (int k = 0; k < Nv; ++k) cls[order[k]] = k % nb;
  bo.load.assign((size_t)bo.n_groups * nb, 0);
  for (int v = 0; v < N; ++v)
    for (auto [g, cnt] : bo.feeds[v]) bo.load[(size_t)g * nb + cls[v]] += cnt;
  for (int v = 0; v < N; ++v)
    if (bo.sgroup[v] >= 0) ++bo.scount[(size_t)bo.sgroup[v] * nb + cls[v]];
  bo.smax.resize(bo.n_groups);
  for (int g = 0; g < bo.n_groups; ++g) bo.smax[g] = bo.store_cost(g);
  bo.sumsq = 0;
  for (int x : bo.load) bo.sumsq += (long long)x * x;
  bo.gcost.resize(bo.n_groups);
  for (int g = 0; g < bo.n_groups; ++g) bo.gcost[g] = bo.group_cost(g);

  if (optimise && nb > 1 && Nv > 1) {
    Rng rng;
    long long best_p = bo.primary(), best_s = bo.sumsq;
    const long long budget = std::min<long long>(300000, 600LL * Nv);
    std::vector<int> touched, old;
    for (long long it = 0; it < budget; ++it) {
      const int a = rng.below(Nv), b = rng.below(Nv);
      if (cls[a] == cls[b] || (a >= N && b >= N)) continue;
      const int ca = cls[a], cb = cls[b];
      bo.move(a, ca, cb);
      bo.move(b, cb, ca);
      touched.clear();
      for (auto [g, c] : bo.feeds[a]) touched.push_back(g);
      for (auto [g, c] : bo.feeds[b]) touched.push_back(g);
      old.resize(touched.size());
      for (size_t k = 0; k < touched.size(); ++k) old[k] = bo.gcost[touched[k]];
      for (size_t k = 0; k < touched.size(); ++k) bo.gcost[touched[k]] = bo.group_cost(touched[k]);
      const int sga = bo.sgroup[a], sgb = bo.sgroup[b];
      const int olda = sga >= 0 ? bo.smax[sga] : 0, oldb = sgb >= 0 ? bo.smax[sgb] : 0;
      if (sga >= 0) bo.smax[sga] = bo.store_cost(sga);
      if (sgb >= 0) bo.smax[sgb] = bo.store_cost(sgb);
      const long long p = bo.primary();
      if (p < best_p || (p == best_p && bo.sumsq <= best_s)) {
        best_p = p; best_s = bo.sumsq;
        cls[a] = cb; cls[b] = ca;
      } else {
        bo.move(a, cb, ca);
        bo.move(b, ca, cb);
        for (size_t k = touched.size(); k-- > 0;) bo.gcost[touched[k]] = old[k];
        if (sga >= 0) bo.smax[sga] = olda;
        if (sgb >= 0) bo.smax[sgb] = oldb;
      }
    }
  }
  pass_iters->assign(n_pass, 0);
  for (int p = 0; p < n_pass; ++p)
    for (int g = p * CG; g < (p + 1) * CG; ++g) (*pass_iters)[p] = std::max((*pass_iters)[p], bo.gcost[g]);
  cls.resize(N);
  return cls;
}

double layout_cost(const Layout& lay, const std::vector<int>& iters) {
  // one iteration = 1; a pass costs about 3.5 iterations of node work, a combine round 0.6
  double c = 0;
  for (size_t p = 0; p < iters.size(); ++p) c += iters[p] + 3.5 + 0.6 * lay.rounds[p];
  return c;
}

// Step D: proper edge colouring of the bipartite multigraph (lanes x bank classes) of one group
// with `colors` >= max degree colours (Koenig): lane_colour[l][c] = index into the lane's edge
// list or -1.  Alternating-path recolouring.
void colour_group(const std::vector<std::vector<int>>& lane_banks, int nb, int colors,
                  std::vector<std::vector<int>>* lane_colour) {
  const int L = (int)lane_banks.size();
  std::vector<std::vector<int>> atL(L, std::vector<int>(colors, -1));    // edge id at (lane, colour)
  std::vector<std::vector<int>> atB(nb, std::vector<int>(colors, -1));   // edge id at (bank, colour)
  struct Edge { int l, b, k, col; };
  std::vector<Edge> edges;
  for (int l = 0; l < L; ++l)
    for (int k = 0; k < (int)lane_banks[l].size(); ++k) edges.push_back({l, lane_banks[l][k], k, -1});
  for (int id = 0; id < (int)edges.size(); ++id) {
    Edge& e = edges[id];
    int a = -1, b = -1;
    for (int c = 0; c < colors; ++c) if (atL[e.l][c] < 0) { a = c; break; }
    for (int c = 0; c < colors; ++c) if (atB[e.b][c] < 0) { b = c; break; }
    if (atB[e.b][a] >= 0) {
      // a is free at the lane but taken at the bank; b is free at the bank.  Flip a <-> b along the
      // alternating path that starts at the bank with colour a (it cannot come back to e.l).
      std::vector<int> path;
      bool at_bank = true;
      int vert = e.b, col = a;
      while (true) {
        const int pe = at_bank ? atB[vert][col] : atL[vert][col];
        if (pe < 0) break;
        path.push_back(pe);
        vert = at_bank ? edges[pe].l : edges[pe].b;
        at_bank = !at_bank;
        col = (col == a) ? b : a;
      }
      for (int pe : path) { atL[edges[pe].l][edges[pe].col] = -1; atB[edges[pe].b][edges[pe].col] = -1; }
      for (int pe : path) {
        edges[pe].col = (edges[pe].col == a) ? b : a;
        atL[edges[pe].l][edges[pe].col] = pe;
        atB[edges[pe].b][edges[pe].col] = pe;
      }
    }
    e.col = a;
    atL[e.l][a] = id;
    atB[e.b][a] = id;
  }
  lane_colour->assign(L, std::vector<int>(colors, -1));
  for (const Edge& e : edges) (*lane_colour)[e.l][e.col] = e.k;
}

}  // namespace

PlanOptions PlanOptions::from_env() {
  PlanOptions o;
  if (const char* e = tsa::tune_env("TSA_NO_SPLIT")) o.split_rows = !(e[0] == '1');
  if (const char* e = tsa::tune_env("TSA_NO_BANKOPT")) o.bank_opt = !(e[0] == '1');
  if (const char* e = tsa::tune_env("TSA_NO_STOREOPT")) o.store_opt = !(e[0] == '1');
  if (const char* e = tsa::tune_env("TSA_NO_TIERS")) o.tiers = !(e[0] == '1');
  if (const char* e = tsa::tune_env("TSA_TEAM_MIN")) o.min_team_warps = std::max(1, std::atoi(e));
  if (const char* e = tsa::tune_env("TSA_MAX_SLOTS")) o.max_lane_slots = std::max(0, std::atoi(e));
  return o;
}

int build_plan(const sa_network* net, const sa_observations* obs, bool need_obs, const PlanOptions& opt,
               Plan* pl, std::string* err) {
  if (!net || !obs || !pl) return fail(err, "null argument");
  const int N = net->n_nodes, E = net->n_edges, NP = net->n_pairs;
  const int K = obs->n_cond, T = obs->n_steps, NO = obs->n_obs;
  if (N <= 0 || E <= 0 || NP <= 0 || K <= 0 || T <= 0 || NO <= 0) return fail(err, "all counts must be > 0");
  if (NP > 16) return fail(err, "n_pairs must be <= 16");
  if (NP < 2) return fail(err, "n_pairs must be >= 2 (a threshold mutation needs another pair)");
  if (T > 127 || NO > 127) return fail(err, "n_steps and n_obs must be <= 127");
  if (E > (1 << 24) - 1) return fail(err, "n_edges must fit 24 bits (trace record)");
  if (!net->edge_src || !net->edge_dst || !net->th_lo || !net->th_hi) return fail(err, "null network array");
  if (!obs->obs_times || !obs->init_state || !obs->clamp) return fail(err, "null observation array");
  if (need_obs && !obs->obs) return fail(err, "obs is NULL");

  for (int q = 0; q < NP; ++q)
    if (net->th_lo[q] >= net->th_hi[q]) return fail(err, "th_lo must be < th_hi");
  std::vector<int> indeg(N, 0);
  {
    std::unordered_set<uint64_t> seen;
    seen.reserve((size_t)E * 2);
    for (int e = 0; e < E; ++e) {
      int s = net->edge_src[e], d = net->edge_dst[e];
      if (s < 0 || s >= N || d < 0 || d >= N) return fail(err, "edge endpoint out of range");
      if (s == d) return fail(err, "self-loops are not allowed");
      if (!seen.insert(((uint64_t)(uint32_t)s << 32) | (uint32_t)d).second) return fail(err, "duplicate edge");
      ++indeg[d];
    }
  }
  const int maxdeg = *std::max_element(indeg.begin(), indeg.end());
  // byte-lane accumulator: 128 + sum - t_lo and 128 + sum - t_hi - 1 must stay base-256 digits for
  // every |sum| <= 2*max_in_degree (reading 24)
  for (int q = 0; q < NP; ++q) {
    const int lo = net->th_lo[q], hi = net->th_hi[q];
    if (128 - 2 * maxdeg - lo < 0 || 128 + 2 * maxdeg - lo > 255 || 128 - 2 * maxdeg - hi - 1 < 0 ||
        128 + 2 * maxdeg - hi - 1 > 255)
      return fail(err, "max in-degree exceeds the byte-lane accumulator range (|sum| <= 2*deg must keep 128+sum-t in [0,255])");
  }
  for (int j = 0; j < NO; ++j) {
    int t = obs->obs_times[j];
    if (t < 1 || t > T || (j > 0 && t <= obs->obs_times[j - 1]))
      return fail(err, "obs_times must be strictly increasing in [1, T]");
  }
  for (size_t x = 0; x < (size_t)K * N; ++x) {
    if (obs->init_state[x] > 2) return fail(err, "init_state must be in {0,1,2}");
    if (obs->clamp[x] > 1) return fail(err, "clamp must be 0 or 1");
  }
  if (need_obs)
    for (size_t x = 0; x < (size_t)K * NO * N; ++x)
      if (obs->obs[x] > 2 && obs->obs[x] != SA_UNOBSERVED) return fail(err, "obs must be in {0,1,2,255}");

  Plan& p = *pl;
  p = Plan();
  p.N = N; p.E = E; p.P = E + N; p.K = K; p.T = T; p.n_obs = NO; p.n_pairs = NP;
  p.max_in_degree = maxdeg;
  const int kc = std::min(K, 16);
  p.CG = kc <= 4 ? 1 : kc <= 8 ? 2 : 4;
  p.nb = 32 / p.CG;
  p.n_chunks = (K + 4 * p.CG - 1) / (4 * p.CG);
  const int CG = p.CG, nb = p.nb;
  const int per_class = (N + nb - 1) / nb;
  // nb zero dummies first, then per_class entries per class, then one scratch entry per lane (the
  // static kernel lets lanes that finalise no node store there instead of predicating the store)
  p.scratch_entry0 = nb * (1 + per_class);
  p.n_entries = p.scratch_entry0 + 32;
  p.state_words = p.n_entries * CG;
  if ((size_t)p.state_words * 4 > 65535) return fail(err, "network too large for 16-bit state offsets (n_entries*CG*4 <= 65535)");
  for (int q = 0; q < NP; ++q) { p.tha[q] = (int8_t)(-net->th_lo[q]); p.thb[q] = (int8_t)(-net->th_hi[q] - 1); }

  std::vector<std::vector<int>> in_edges(N);
  for (int e = 0; e < E; ++e) in_edges[net->edge_dst[e]].push_back(e);

  // candidate pass counts; keep the cheapest layout under the cost model
  const int P0 = (N + 31) / 32;
  std::vector<int> cand = {P0};
  if (opt.split_rows) {
    for (int c : {P0 + 1, P0 + 2, P0 + (P0 + 3) / 4, P0 + (P0 + 1) / 2})
      if (std::find(cand.begin(), cand.end(), c) == cand.end()) cand.push_back(c);
  }
  Layout best_lay;
  std::vector<int> best_cls, best_iters;
  double best_cost = 1e300;
  for (int c : cand) {
    Layout lay = make_layout(in_edges, 32 * c, opt.split_rows);
    std::vector<int> iters;
    std::vector<int> cls = assign_classes(lay, net->edge_src, N, CG, opt.bank_opt, opt.store_opt, &iters);
    const double cost = layout_cost(lay, iters);
    if (cost < best_cost) { best_cost = cost; best_lay = std::move(lay); best_cls = std::move(cls); best_iters = std::move(iters); }
  }
  // Tiers: order the passes by iteration count, give each of W warps one pass per tier, pad every
  // pass to its tier's count.  One thread then holds sum(tier iterations) edge slots in registers.
  int W = 0, NT = 0;
  if (!opt.tiers) p.static_why = "tiers disabled";
  else if (p.n_chunks != 1) p.static_why = "more than 16 conditions";
  else {
    for (int k = 0; k < K && p.static_why.empty(); ++k)
      for (int i = 0; i < N; ++i)
        if (obs->clamp[(size_t)k * N + i] && indeg[i] > 31) { p.static_why = "a clamped node has in-degree > 31"; break; }
  }
  if (p.static_why.empty()) {
    const int np0 = (int)best_lay.passes.size();
    std::vector<int> order(np0);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return best_iters[a] > best_iters[b]; });
    const int max_slots = opt.max_lane_slots > 0 ? opt.max_lane_slots : (CG == 4 ? 64 : 48);   // Large: 64 -> 8 warps per chain, 3.47 M (40: 16 warps, 3.30 M)
    // W is a power of two (a 128-register budget then fills an SM's 512 threads with whole teams)
    int w_lo = 1;
    while (w_lo < std::min(opt.min_team_warps, 32) && 2 * w_lo <= np0) w_lo *= 2;
    long best_cost = -1;
    for (int w = w_lo; w <= 32 && (w == w_lo || w <= np0); w *= 2) {
      const int nt = (np0 + w - 1) / w;
      int slots = 0;
      for (int j = 0; j < nt; ++j) slots += std::max(best_iters[order[j * w]], 1);
      if (slots > max_slots) continue;
      const long cost = (long)(slots + 4 * nt) * w;
      if (best_cost < 0 || cost < best_cost) { best_cost = cost; W = w; NT = nt; }
    }
    if (W == 0) p.static_why = "too many edge slots per thread";
    else {
      Layout sorted;
      std::vector<int> it2;
      for (int x = 0; x < NT * W; ++x) {
        if (x < np0) {
          sorted.passes.push_back(std::move(best_lay.passes[order[x]]));
          sorted.rounds.push_back(best_lay.rounds[order[x]]);
        } else {
          sorted.passes.push_back(std::vector<Row>(32));
          sorted.rounds.push_back(0);
        }
        it2.push_back(std::max(best_iters[order[(x / W) * W]], 1));
      }
      best_lay = std::move(sorted);
      best_iters = std::move(it2);
    }
  }
  const Layout& lay = best_lay;
  p.n_pass = (int)lay.passes.size();

  // entries: dummies 0..nb-1 (class = index), then the j-th node of class c at nb + j*nb + c
  p.entry_of_node.assign(N, -1);
  {
    std::vector<int> fill(nb, 0);
    for (int i = 0; i < N; ++i) {
      const int c = best_cls[i];
      p.entry_of_node[i] = nb + fill[c] * nb + c;
      ++fill[c];
    }
  }

  p.pass_base.resize(p.n_pass);
  p.pass_iters = best_iters;
  p.pass_rounds = lay.rounds;
  int slots = 0;
  for (int ps = 0; ps < p.n_pass; ++ps) {
    p.pass_base[ps] = slots;
    slots += ((p.pass_iters[ps] + 3) / 4) * 128;
    p.total_iters += p.pass_iters[ps];
  }
  p.Epad = std::max(slots, 128);
  p.EpadA = (p.Epad + 15) & ~15;
  p.NpadA = (p.n_entries + 15) & ~15;
  p.slot_off.assign(p.Epad, 0);
  p.param_of_slot.assign(p.Epad, -1);
  p.slot_of_param.assign(E, -1);
  p.row_meta.assign((size_t)p.n_pass * 32, 0u);

  for (int ps = 0; ps < p.n_pass; ++ps) {
    const int iters = p.pass_iters[ps];
    for (int g = 0; g < CG; ++g) {
      std::vector<std::vector<int>> lane_banks(nb);
      for (int l = 0; l < nb; ++l)
        for (int e : lay.passes[ps][g * nb + l].edges) lane_banks[l].push_back(best_cls[net->edge_src[e]]);
      std::vector<std::vector<int>> colour;
      colour_group(lane_banks, nb, std::max(iters, 1), &colour);
      for (int k = 0; k < iters; ++k) {
        std::vector<char> bank_used(nb, 0);
        for (int l = 0; l < nb; ++l)
          if (colour[l][k] >= 0) bank_used[lane_banks[l][colour[l][k]]] = 1;
        int free_bank = 0;
        for (int l = 0; l < nb; ++l) {
          const int lane = g * nb + l;
          const int slot = p.pass_base[ps] + (k / 4) * 128 + lane * 4 + (k % 4);
          if (colour[l][k] >= 0) {
            const int e = lay.passes[ps][lane].edges[colour[l][k]];
            p.slot_off[slot] = (uint16_t)(p.entry_of_node[net->edge_src[e]] * CG * 4);
            p.param_of_slot[slot] = e;
            p.slot_of_param[e] = slot;
          } else {
            while (bank_used[free_bank]) ++free_bank;        // an unused bank unit: its dummy entry
            bank_used[free_bank] = 1;
            p.slot_off[slot] = (uint16_t)(free_bank * CG * 4);
          }
        }
      }
    }
    for (int lane = 0; lane < 32; ++lane) {
      const Row& r = lay.passes[ps][lane];
      if (r.node < 0) continue;
      ++p.n_rows;
      uint32_t meta = (uint32_t)(p.entry_of_node[r.node] * CG * 4);
      if (r.head) { meta |= kMetaHead; if (r.parts > 1) ++p.n_split_nodes; }
      // combine tree over the block's consecutive lanes: in round q part a (a % 2^(q+1) == 0)
      // adds part a + 2^q if it exists
      for (int q = 0; q < lay.rounds[ps]; ++q)
        if (r.part % (2 << q) == 0 && r.part + (1 << q) < r.parts) meta |= 1u << (kMetaCombineShift + q);
      p.row_meta[(size_t)ps * 32 + lane] = meta;
    }
  }
  for (int e = 0; e < E; ++e)
    if (p.slot_of_param[e] < 0) return fail(err, "internal error: edge without a slot");
  // self-check: in every iteration the nb lanes of a conflict group read nb distinct bank units
  for (int ps = 0; ps < p.n_pass; ++ps)
    for (int k = 0; k < p.pass_iters[ps]; ++k)
      for (int g = 0; g < CG; ++g) {
        uint32_t seen = 0;
        for (int l = 0; l < nb; ++l) {
          const int slot = p.pass_base[ps] + (k / 4) * 128 + (g * nb + l) * 4 + (k % 4);
          const uint32_t bit = 1u << ((p.slot_off[slot] / (CG * 4)) % nb);
          if (seen & bit) return fail(err, "internal error: edge schedule has a bank conflict");
          seen |= bit;
        }
      }

  // conditions packed 4 per 32-bit word (byte lanes), CG words per entry, chunks of 4*CG conditions.
  // A clamped (k, i) never changes, so it is scored once here (fit_const), masked out of the
  // observation words and restored by a byte store after each step (fix-up list of its pass).
  std::vector<int> pass_of_node(N, 0);
  for (int ps = 0; ps < p.n_pass; ++ps)
    for (const Row& r : lay.passes[ps])
      if (r.node >= 0 && r.head) pass_of_node[r.node] = ps;
  const int per_chunk = 4 * CG, NE = p.n_entries;
  p.initw.assign((size_t)p.n_chunks * NE * CG, 0u);
  p.obsw.assign((size_t)p.n_chunks * NO * NE * CG, 0u);
  p.obsm.assign((size_t)p.n_chunks * NO * NE * CG, 0u);
  std::vector<std::vector<uint32_t>> fixes((size_t)p.n_chunks * p.n_pass);
  for (int k = 0; k < K; ++k) {
    const int ch = k / per_chunk, c = k % per_chunk, cg = c / 4, b = c % 4, sh = 8 * b;
    for (int i = 0; i < N; ++i) {
      const int en = p.entry_of_node[i];
      const uint8_t iv = obs->init_state[(size_t)k * N + i];
      const bool clamped = obs->clamp[(size_t)k * N + i] != 0;
      p.initw[((size_t)ch * NE + en) * CG + cg] |= (uint32_t)iv << sh;
      if (clamped)
        fixes[(size_t)ch * p.n_pass + pass_of_node[i]].push_back((uint32_t)(en * CG * 4 + cg * 4 + b) | ((uint32_t)iv << 16));
      if (!need_obs) continue;
      for (int j = 0; j < NO; ++j) {
        const uint8_t o = obs->obs[((size_t)k * NO + j) * N + i];
        if (o == SA_UNOBSERVED) continue;
        if (clamped) { if (o != iv) ++p.fit_const; continue; }
        const size_t ow = (((size_t)ch * NO + j) * NE + en) * CG + cg;
        p.obsw[ow] |= (uint32_t)o << sh;
        p.obsm[ow] |= 1u << sh;
      }
    }
  }
  p.fix_ptr.assign((size_t)p.n_chunks * p.n_pass + 1, 0);
  for (size_t x = 0; x < fixes.size(); ++x) {
    p.fix_ptr[x] = (int32_t)p.fix.size();
    p.fix.insert(p.fix.end(), fixes[x].begin(), fixes[x].end());
  }
  p.fix_ptr[fixes.size()] = (int32_t)p.fix.size();
  if (p.fix.empty()) p.fix.push_back(0u);
  p.obs_idx_of_t.assign(T + 1, -1);
  for (int j = 0; j < NO; ++j) p.obs_idx_of_t[obs->obs_times[j]] = (int8_t)j;

  // tables of the statically scheduled kernel: one column per thread (warp, lane) of the team
  if (W > 0) {
    p.team_warps = W;
    p.n_tiers = NT;
    const int TEAM = W * 32, EB = CG * 4;
    for (int j = 0; j < NT; ++j) {
      p.tier_iters.push_back(p.pass_iters[j * W]);
      int r = 0;
      for (int w = 0; w < W; ++w) r = std::max(r, lay.rounds[j * W + w]);
      p.tier_rounds.push_back(r);
    }
    std::vector<int> wbase(NT + 1, 0);
    for (int j = 0; j < NT; ++j) wbase[j + 1] = wbase[j] + (p.tier_iters[j] + 3) / 4;
    auto slot_of = [&](int ps, int k, int lane) { return p.pass_base[ps] + (k / 4) * 128 + lane * 4 + (k % 4); };
    for (int j = 0; j < NT; ++j) {
      const int it = p.tier_iters[j];
      for (int r = 0; r < (it + 1) / 2; ++r)
        for (int th = 0; th < TEAM; ++th) {
          const int ps = j * W + th / 32, lane = th % 32;
          const uint32_t lo = p.slot_off[slot_of(ps, 2 * r, lane)];
          const uint32_t hi = (2 * r + 1 < it) ? p.slot_off[slot_of(ps, 2 * r + 1, lane)] : 0u;
          p.lane_off2.push_back(lo | (hi << 16));
        }
    }
    p.lane_meta.assign((size_t)NT * TEAM, 0u);
    p.lane_clamp.assign((size_t)NT * 3 * CG * TEAM, 0u);
    p.thloc.assign(N, 0u);
    for (int j = 0; j < NT; ++j)
      for (int th = 0; th < TEAM; ++th) {
        const int ps = j * W + th / 32, lane = th % 32;
        const Row& r = lay.passes[ps][lane];
        const uint32_t rm = p.row_meta[(size_t)ps * 32 + lane];
        uint32_t meta = (uint32_t)((p.scratch_entry0 + lane) * EB);
        if (r.node >= 0 && r.head) {
          meta = (uint32_t)(p.entry_of_node[r.node] * EB) | kMetaHead;
          p.thloc[r.node] = (uint32_t)j | ((uint32_t)th << 16);
          for (int k = 0; k < K; ++k) {
            if (!obs->clamp[(size_t)k * N + r.node]) continue;
            const uint32_t v = obs->init_state[(size_t)k * N + r.node];
            const int cg = k / 4, sh = 8 * (k % 4);
            p.lane_clamp[((size_t)j * 3 * CG + cg) * TEAM + th] |= 0xFFu << sh;
            p.lane_clamp[((size_t)j * 3 * CG + CG + cg) * TEAM + th] |= (v == 0 ? 64u : 192u) << sh;
            p.lane_clamp[((size_t)j * 3 * CG + 2 * CG + cg) * TEAM + th] |= (v == 1 ? 128u : 0u) << sh;
          }
        }
        meta |= rm & ~(kMetaOffMask | kMetaHead);          // the combine bits
        p.lane_meta[(size_t)j * TEAM + th] = meta;
      }
    p.wloc.assign(E, 0u);
    for (int e = 0; e < E; ++e) {
      const int s = p.slot_of_param[e];
      int ps = p.n_pass - 1;
      while (p.pass_base[ps] > s) --ps;
      const int rel = s - p.pass_base[ps], g = rel / 128, lane = (rel % 128) / 4, byte = rel % 4;
      const int j = ps / W, th = (ps % W) * 32 + lane;
      p.wloc[e] = (uint32_t)(wbase[j] + g) | ((uint32_t)byte << 8) | ((uint32_t)th << 16);
    }
  }
  return SA_OK;
}

void Plan::to_internal(const int8_t* params, int8_t* w, int8_t* th) const {
  std::fill(w, w + EpadA, (int8_t)0);
  std::fill(th, th + NpadA, (int8_t)0);
  for (int e = 0; e < E; ++e) w[slot_of_param[e]] = params[e];
  for (int i = 0; i < N; ++i) th[entry_of_node[i]] = params[E + i];
}

void Plan::to_caller(const int8_t* w, const int8_t* th, int8_t* params) const {
  for (int e = 0; e < E; ++e) params[e] = w[slot_of_param[e]];
  for (int i = 0; i < N; ++i) params[E + i] = th[entry_of_node[i]];
}

bool params_valid(const Plan& plan, const int8_t* params, int64_t n) {
  for (int64_t r = 0; r < n; ++r) {
    const int8_t* x = params + r * plan.P;
    for (int e = 0; e < plan.E; ++e)
      if (x[e] < -1 || x[e] > 1) return false;
    for (int i = 0; i < plan.N; ++i)
      if (x[plan.E + i] < 0 || x[plan.E + i] >= plan.n_pairs) return false;
  }
  return true;
}

}  // namespace tsa
