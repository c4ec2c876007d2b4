#include "sa_plan.h"

#include "sa_common.h"

#include <algorithm>
#include <cstdlib>
#include <numeric>
#include <unordered_set>

namespace tsa {

namespace {
int fail(std::string* err, const std::string& msg) {
  if (err) *err = msg;
  return SA_EINVAL;
}
}  // namespace

int build_plan(const sa_network* net, const sa_observations* obs, bool need_obs, Plan* pl, std::string* err) {
  if (!net || !obs || !pl) return fail(err, "null argument");
  const int N = net->n_nodes, E = net->n_edges, NP = net->n_pairs;
  const int K = obs->n_cond, T = obs->n_steps, NO = obs->n_obs;
  if (N <= 0 || E <= 0 || NP <= 0 || K <= 0 || T <= 0 || NO <= 0) return fail(err, "all counts must be > 0");
  if (NP > 16) return fail(err, "n_pairs must be <= 16");
  if (NP < 2) return fail(err, "n_pairs must be >= 2 (a threshold mutation needs another pair)");
  if (T > 127 || NO > 127) return fail(err, "n_steps and n_obs must be <= 127");
  if (N > 65534) return fail(err, "n_nodes must be <= 65534");
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
  int maxdeg = *std::max_element(indeg.begin(), indeg.end());
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
  p.n_chunks = (K + 4 * p.CG - 1) / (4 * p.CG);
  p.state_words = (N + 1) * p.CG;
  if ((size_t)p.state_words * 4 > 65535) return fail(err, "network too large for 16-bit state offsets ((N+1)*CG*4 <= 65535)");
  for (int q = 0; q < NP; ++q) { p.tha[q] = (int8_t)(-net->th_lo[q]); p.thb[q] = (int8_t)(-net->th_hi[q] - 1); }

  // rows: nodes by descending in-degree (stable), so the 32 rows of a pass have similar lengths
  p.node_of_row.resize(N);
  std::iota(p.node_of_row.begin(), p.node_of_row.end(), 0);
  std::stable_sort(p.node_of_row.begin(), p.node_of_row.end(), [&](int a, int b) { return indeg[a] > indeg[b]; });
  p.row_of_node.resize(N);
  for (int r = 0; r < N; ++r) p.row_of_node[p.node_of_row[r]] = r;

  // in-edges per row, in caller edge order
  std::vector<std::vector<int>> in_edges(N);
  for (int e = 0; e < E; ++e) in_edges[p.row_of_node[net->edge_dst[e]]].push_back(e);

  p.n_pass = (N + kWarp - 1) / kWarp;
  p.pass_base.resize(p.n_pass);
  p.pass_deg.resize(p.n_pass);
  int slots = 0;
  for (int ps = 0; ps < p.n_pass; ++ps) {
    int deg = 0;
    for (int l = 0; l < 32 && ps * 32 + l < N; ++l) deg = std::max(deg, (int)in_edges[ps * 32 + l].size());
    p.pass_base[ps] = slots;
    p.pass_deg[ps] = deg;
    slots += ((deg + 3) / 4) * 128;
  }
  p.Epad = std::max(slots, 128);
  p.EpadA = (p.Epad + 15) & ~15;
  p.NpadA = (N + 15) & ~15;
  const uint16_t dummy = (uint16_t)(N * p.CG * 4);
  p.slot_off.assign(p.Epad, dummy);
  p.param_of_slot.assign(p.Epad, -1);
  p.slot_of_param.assign(E, -1);
  for (int r = 0; r < N; ++r) {
    int ps = r / 32, l = r % 32;
    for (int k = 0; k < (int)in_edges[r].size(); ++k) {
      int e = in_edges[r][k];
      int slot = p.pass_base[ps] + (k / 4) * 128 + l * 4 + (k % 4);
      p.slot_off[slot] = (uint16_t)(p.row_of_node[net->edge_src[e]] * p.CG * 4);
      p.param_of_slot[slot] = e;
      p.slot_of_param[e] = slot;
    }
  }

  // conditions packed 4 per 32-bit word (byte lanes), CG words per node, chunks of 4*CG conditions
  const int CG = p.CG, per_chunk = 4 * CG;
  p.initw.assign((size_t)p.n_chunks * N * CG, 0u);
  p.clampm.assign((size_t)p.n_chunks * N * CG, 0u);
  p.obsw.assign((size_t)p.n_chunks * NO * N * CG, 0u);
  p.obsm.assign((size_t)p.n_chunks * NO * N * CG, 0u);
  for (int k = 0; k < K; ++k) {
    int ch = k / per_chunk, c = k % per_chunk, cg = c / 4, sh = 8 * (c % 4);
    for (int i = 0; i < N; ++i) {
      int r = p.row_of_node[i];
      size_t w = ((size_t)ch * N + r) * CG + cg;
      p.initw[w] |= (uint32_t)obs->init_state[(size_t)k * N + i] << sh;
      if (obs->clamp[(size_t)k * N + i]) p.clampm[w] |= 0xFFu << sh;
      if (need_obs)
        for (int j = 0; j < NO; ++j) {
          uint8_t o = obs->obs[((size_t)k * NO + j) * N + i];
          if (o == SA_UNOBSERVED) continue;
          size_t ow = (((size_t)ch * NO + j) * N + r) * CG + cg;
          p.obsw[ow] |= (uint32_t)o << sh;
          p.obsm[ow] |= 1u << sh;
        }
    }
  }
  p.obs_idx_of_t.assign(T + 1, -1);
  for (int j = 0; j < NO; ++j) p.obs_idx_of_t[obs->obs_times[j]] = (int8_t)j;
  return SA_OK;
}

void Plan::to_internal(const int8_t* params, int8_t* w, int8_t* th) const {
  std::fill(w, w + EpadA, (int8_t)0);
  std::fill(th, th + NpadA, (int8_t)0);
  for (int e = 0; e < E; ++e) w[slot_of_param[e]] = params[e];
  for (int i = 0; i < N; ++i) th[row_of_node[i]] = params[E + i];
}

void Plan::to_caller(const int8_t* w, const int8_t* th, int8_t* params) const {
  for (int e = 0; e < E; ++e) params[e] = w[slot_of_param[e]];
  for (int i = 0; i < N; ++i) params[E + i] = th[row_of_node[i]];
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
