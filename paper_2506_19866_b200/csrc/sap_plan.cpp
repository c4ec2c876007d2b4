#include "sa_tuning.h"
#include "sap_plan.h"

#include <algorithm>
#include <cstdlib>
#include <numeric>
#include <set>
#include <utility>

namespace tsa {

int build_paper_plan(const sap_network* net, const sap_observations* obs, bool need_ref, bool constrained, int64_t n_chains,
                     int sm_count, PaperPlan* out, std::string* err) {
  auto fail = [&](const std::string& m) { *err = m; return SA_EINVAL; };
  if (!net || !obs) return fail("null argument");
  const int N = net->n_nodes, E = net->n_edges, K = obs->n_cond, T = obs->n_steps;
  if (N <= 0 || E <= 0 || K <= 0 || T <= 0) return fail("counts must be positive");
  if (N > 256) return fail("the paper-model kernel handles at most 256 nodes");
  if (T > 4095) return fail("at most 4095 transitions");
  if (!net->edge_src || !net->edge_dst || !net->fast || !obs->init_state) return fail("null array");
  if (need_ref && !obs->ref) return fail("reference matrix is NULL");
  PaperPlan& pl = *out;
  pl = PaperPlan();
  pl.N = N; pl.E = E; pl.NP = 3 * E + 3 * N; pl.NPPAD = (pl.NP + 15) / 16 * 16; pl.K = K; pl.T = T;
  pl.src.assign(net->edge_src, net->edge_src + E);
  pl.dst.assign(net->edge_dst, net->edge_dst + E);
  std::set<std::pair<int, int>> seen;
  for (int e = 0; e < E; ++e) {
    const int s = pl.src[e], d = pl.dst[e];
    if (s < 0 || s >= N || d < 0 || d >= N) return fail("edge endpoint out of range");
    // s == d is allowed: autoregulation is an edge like any other in PAPER.md:55-70, and the oracle takes it too
    if (!seen.insert({s, d}).second) return fail("duplicate edge");
  }
  pl.fast.assign(net->fast, net->fast + N);
  for (int i = 0; i < N; ++i)
    if (pl.fast[i] > 1) return fail("fast flags must be 0 or 1");
  for (size_t x = 0; x < (size_t)K * N; ++x)
    if (obs->init_state[x] > 2) return fail("initial state outside {0,1,2}");
  if (obs->ref)
    for (size_t x = 0; x < (size_t)K * (T + 1) * N; ++x)
      if (obs->ref[x] > 2 && obs->ref[x] != SA_UNOBSERVED) return fail("reference entry outside {0,1,2,255}");

  // CSR by destination / source over caller edge ids, ascending
  pl.in_ptr.assign(N + 1, 0); pl.out_ptr.assign(N + 1, 0);
  for (int e = 0; e < E; ++e) { ++pl.in_ptr[pl.dst[e] + 1]; ++pl.out_ptr[pl.src[e] + 1]; }
  for (int i = 0; i < N; ++i) { pl.in_ptr[i + 1] += pl.in_ptr[i]; pl.out_ptr[i + 1] += pl.out_ptr[i]; }
  pl.in_edge.assign(E, 0); pl.out_edge.assign(E, 0);
  {
    std::vector<int> a(pl.in_ptr.begin(), pl.in_ptr.end() - 1), b(pl.out_ptr.begin(), pl.out_ptr.end() - 1);
    for (int e = 0; e < E; ++e) { pl.in_edge[a[pl.dst[e]]++] = e; pl.out_edge[b[pl.src[e]]++] = e; }
  }
  for (int i = 0; i < N; ++i) {
    const int din = pl.in_ptr[i + 1] - pl.in_ptr[i], dout = pl.out_ptr[i + 1] - pl.out_ptr[i];
    pl.max_in_degree = std::max(pl.max_in_degree, din);
    if (constrained && (din == 0 || dout == 0))
      return fail("with constraints on every node needs an in-edge and an out-edge (PAPER.md:187-191)");
  }

  // lanes per chain, node slots; nodes sorted by in-degree so that a node slot holds nodes of similar degree
  pl.LPC = N <= 16 ? 8 : N <= 32 ? 16 : 32;
  // measured on paper_mtb (63 nodes), R = 10 240: 32 lanes 407 M, 16 lanes 428 M, 8 lanes 290 M chain-steps/s
  if (N > 32 && N <= 64 && n_chains / 2 >= 16LL * std::max(sm_count, 1)) pl.LPC = 16;
  if (const char* e = tsa::tune_env("TSA_PAPER_LPC")) {
    const int v = std::atoi(e);
    if ((v == 8 || v == 16 || v == 32) && 8 * v >= N) pl.LPC = v;
  }
  pl.NS = (N + pl.LPC - 1) / pl.LPC;
  std::vector<int> order(N);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
    return pl.in_ptr[a + 1] - pl.in_ptr[a] > pl.in_ptr[b + 1] - pl.in_ptr[b];
  });
  pl.node_lane.assign(N, 0); pl.node_slot.assign(N, 0);
  pl.pos_node.assign((size_t)pl.NS * pl.LPC, -1);
  pl.esl.assign(pl.NS, 0);
  for (int r = 0; r < N; ++r) {
    const int i = order[r], n = r / pl.LPC, l = r % pl.LPC;
    pl.node_lane[i] = l; pl.node_slot[i] = n;
    pl.pos_node[(size_t)n * pl.LPC + l] = i;
    pl.esl[n] = std::max(pl.esl[n], pl.in_ptr[i + 1] - pl.in_ptr[i]);
  }
  std::vector<int> eoff(pl.NS + 1, 0);
  for (int n = 0; n < pl.NS; ++n) eoff[n + 1] = eoff[n] + pl.esl[n];
  pl.ES = eoff[pl.NS];
  if (pl.ES > 256) return fail("too many edge slots per lane for the paper-model kernel (in-degrees too large)");

  pl.slot_src.assign((size_t)std::max(pl.ES, 1) * pl.LPC, 0);
  pl.slot_edge.assign((size_t)std::max(pl.ES, 1) * pl.LPC, -1);
  pl.ploc.assign(pl.NP, 0);
  for (int i = 0; i < N; ++i) {
    const int l = pl.node_lane[i], n = pl.node_slot[i];
    for (int x = pl.in_ptr[i]; x < pl.in_ptr[i + 1]; ++x) {
      const int e = pl.in_edge[x], k = eoff[n] + (x - pl.in_ptr[i]), s = pl.src[e];
      pl.slot_edge[(size_t)k * pl.LPC + l] = e;
      pl.slot_src[(size_t)k * pl.LPC + l] = (uint16_t)(pl.node_slot[s] * pl.LPC + pl.node_lane[s]);
      for (int cls = 0; cls < 3; ++cls)
        pl.ploc[(size_t)cls * E + e] = (uint32_t)cls | ((uint32_t)l << 3) | ((uint32_t)k << 8) | ((uint32_t)s << 16) | ((uint32_t)i << 24);
    }
    for (int cls = 3; cls < 6; ++cls)
      pl.ploc[(size_t)3 * E + (size_t)(cls - 3) * N + i] = (uint32_t)cls | ((uint32_t)l << 3) | ((uint32_t)n << 8) | ((uint32_t)i << 16);
  }

  pl.init_lane.assign((size_t)K * pl.LPC, 0);
  for (int k = 0; k < K; ++k)
    for (int i = 0; i < N; ++i)
      pl.init_lane[(size_t)k * pl.LPC + pl.node_lane[i]] |= (uint32_t)obs->init_state[(size_t)k * N + i] << (2 * pl.node_slot[i]);
  pl.NSP = pl.NS <= 1 ? 1 : pl.NS <= 2 ? 2 : pl.NS <= 4 ? 4 : 8;
  pl.cost_lane.assign((size_t)K * (T + 1) * pl.LPC * pl.NSP, 0);
  if (obs->ref) {
    uint64_t scored = 0;
    for (int k = 0; k < K; ++k)
      for (int t = 0; t <= T; ++t)
        for (int i = 0; i < N; ++i) {
          const uint8_t r = obs->ref[((size_t)k * (T + 1) + t) * N + i];
          if (r == SA_UNOBSERVED) continue;
          int g = 0;                                         // gradient row t of G: 0 for t0
          if (t > 0) {
            const uint8_t rp = obs->ref[((size_t)k * (T + 1) + t - 1) * N + i];
            if (rp != SA_UNOBSERVED) g = (int)r - (int)rp;
          }
          uint32_t word = 0;                                 // byte s+1: |s - r| * (|g| + 1); byte 0 stays 0
          for (int s = 0; s < 3; ++s) word |= (uint32_t)(std::abs(s - (int)r) * (std::abs(g) + 1)) << (8 * (s + 1));
          pl.cost_lane[(((size_t)k * (T + 1) + t) * pl.LPC + pl.node_lane[i]) * pl.NSP + pl.node_slot[i]] = word;
          ++scored;
        }
    pl.max_objective = (uint32_t)std::min<uint64_t>(6 * scored, 0xFFFFFFFFull);
  }
  return SA_OK;
}

bool paper_params_valid(const PaperPlan& pl, const int8_t* params, int64_t n) {
  const int E = pl.E, N = pl.N;
  for (int64_t r = 0; r < n; ++r) {
    const int8_t* x = params + r * pl.NP;
    for (int e = 0; e < E; ++e) {
      if (x[e] < 0 || x[e] > 2) return false;
      if (x[E + e] < -1 || x[E + e] > 1) return false;
      if (x[2 * E + e] < 1 || x[2 * E + e] > 2) return false;
    }
    for (int i = 0; i < N; ++i) {
      const int u = x[3 * E + i], m = x[3 * E + N + i], d = x[3 * E + 2 * N + i];
      if (pl.fast[i] ? (u < 10 || u > 12) : (u < 1 || u > 6)) return false;
      if (m < 0 || m > 2 || d < 1 || d > 2) return false;
    }
  }
  return true;
}

}  // namespace tsa
