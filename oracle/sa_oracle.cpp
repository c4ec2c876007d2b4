// CPU ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded, obviously-correct restatement of the hot path of
// arxiv 2506.19866 ("GPU-accelerated modeling of biological regulatory networks") in the
// simplified ternary model that BASELINE.json pins.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call it.  It shares no code, header, table or helper with the CUDA path under
// paper_2506_19866_b200/csrc and neither includes the other.
//
// Style rules kept on purpose: one byte per node state, a per-node list of in-edges in the
// caller's edge order, no bit tricks, no blocking, no incremental evaluation, every SA step
// re-simulates everything.  A reader can check each function against the cited passage by eye.
//
// Parity pins (tests/test_oracle_*.py, -m "not gpu"): hand-worked Examples A and B, the
// proposal/accept mapping arithmetic, the acceptance-table closed form, the all-zero-weights
// closed form, invariants (i)-(viii), brute force over a 4-node / 6-edge network, and Philox
// against ATen's independent implementation.  Nothing on the hot path is "parity unpinned".
//
// Round 2 adds, without touching any of the above, the structural constraints of PAPER.md §2.5.3 for this
// model (orc_valid, orc_init_chain_c, orc_propose_c, orc_run_chain_c at the end of the file; DESIGN.md
// readings C1-C3), pinned by tests/test_oracle_constraints.py.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct Problem {
  int N = 0, E = 0, n_pairs = 0, K = 0, T = 0, n_obs = 0;
  std::vector<int> src, dst;              // caller's edge order
  std::vector<std::vector<int>> in_edges; // in_edges[i] = edge ids e with dst[e] == i, ascending
  std::vector<int> th_lo, th_hi;          // [n_pairs]
  std::vector<int> obs_times;             // [n_obs], strictly increasing, in [1, T]
  std::vector<uint8_t> init, clamp;       // [K][N]
  std::vector<uint8_t> obs;               // [K][n_obs][N], 255 = unobserved
};

// a node's input is the cumulative effect of its source nodes; the config model
// (BASELINE.json configs[0]) makes it  sum_i = SUM_{e: dst(e)=i} w_e * s_src(e)  and
//   s'_i = 0 if sum < t_lo,  2 if sum > t_hi,  else 1      (both compares strict),
// all nodes updated synchronously (PAPER.md:74 names the synchronous scheme); a clamped node
// keeps its initial value (reading 9).  One step: s (time t-1) -> s2 (time t).
void step_once(const Problem& P, const int8_t* x, int k, const uint8_t* s, uint8_t* s2) {
  for (int i = 0; i < P.N; ++i) {
    if (P.clamp[(size_t)k * P.N + i]) {
      s2[i] = P.init[(size_t)k * P.N + i];
      continue;
    }
    int sum = 0;                                   // a node with no in-edges has sum = 0
    for (int e : P.in_edges[i]) sum += (int)x[e] * (int)s[P.src[e]];   // uses s, never s2
    int q = x[P.E + i];
    int lo = P.th_lo[q], hi = P.th_hi[q];
    s2[i] = (sum < lo) ? 0 : (sum > hi) ? 2 : 1;
  }
}

// SURVEY.md §8(c)-1.  Fitness(x) = number of observed (k, j, i) entries whose simulated state at
// observation time obs_times[j] differs from obs[k][j][i] (distance between the
// simulated matrix S and the reference R over the measured entities; reading 14: 0/1 per entry).
// traj, when given, receives every state: [K][T+1][N], t = 0 is the initial state (not scored).
uint32_t fitness(const Problem& P, const int8_t* x, uint8_t* traj) {
  uint32_t f = 0;
  std::vector<uint8_t> s(P.N), s2(P.N);
  for (int k = 0; k < P.K; ++k) {
    for (int i = 0; i < P.N; ++i) s[i] = P.init[(size_t)k * P.N + i];
    if (traj) std::memcpy(traj + ((size_t)k * (P.T + 1)) * P.N, s.data(), P.N);
    for (int t = 1; t <= P.T; ++t) {
      step_once(P, x, k, s.data(), s2.data());
      s.swap(s2);
      if (traj) std::memcpy(traj + ((size_t)k * (P.T + 1) + t) * P.N, s.data(), P.N);
      for (int j = 0; j < P.n_obs; ++j) {
        if (P.obs_times[j] != t) continue;
        const uint8_t* o = &P.obs[((size_t)k * P.n_obs + j) * P.N];
        for (int i = 0; i < P.N; ++i)
          if (o[i] != 255 && o[i] != s[i]) ++f;
      }
    }
  }
  return f;
}

// Philox4x32-10 (Salmon et al., SC'11), written from the published
// description: 10 rounds; per round (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2 as 64-bit products,
// (c0,c1,c2,c3) <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0); the key is bumped by the Weyl constants
// between rounds (9 bumps).
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    uint64_t p0 = M0 * (uint64_t)c0, p1 = M1 * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// mulhi(a, b) = floor(a*b / 2^32): maps a uniform u32 to [0, b)
uint32_t mulhi(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * (uint64_t)b) >> 32); }

// SURVEY.md §8(c)-2 ("a randomized parameter vector" per thread): block q of four
// parameters takes Philox(ctr = (q, 0, chain, 1), key = seed).
void init_chain(const Problem& P, uint64_t seed, uint32_t chain, int8_t* x) {
  const int NP = P.E + P.N;
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  for (int q = 0; 4 * q < NP; ++q) {
    uint32_t ctr[4] = {(uint32_t)q, 0u, chain, 1u}, y[4];
    philox4x32_10(ctr, key, y);
    for (int m = 0; m < 4; ++m) {
      int p = 4 * q + m;
      if (p >= NP) break;
      x[p] = (p < P.E) ? (int8_t)((int)mulhi(y[m], 3u) - 1) : (int8_t)mulhi(y[m], (uint32_t)P.n_pairs);
    }
  }
}

// SURVEY.md §8(c)-3, GetCandidate ("random single-element change"; reading 7):
// index uniform over all parameters, new value uniform over the OTHER values (never a no-op).
void propose(uint32_t x0, uint32_t x1, int NP, int E, int n_pairs, const int8_t* cur, int* p_out, int* new_out) {
  int p = (int)mulhi(x0, (uint32_t)NP);
  int nv;
  if (p < E) {
    int code = cur[p] + 1;                                   // 0,1,2
    nv = (code + 1 + (int)mulhi(x1, 2u)) % 3 - 1;            // one of the two other weights
  } else {
    int old = cur[p];
    nv = (old + 1 + (int)mulhi(x1, (uint32_t)(n_pairs - 1))) % n_pairs;   // any other pair
  }
  *p_out = p; *new_out = nv;
}

// SURVEY.md §8(c)-3, accept rule (readings 1-4): Metropolis in integer form,
// accept iff d <= 0 or (d <= D and x2 < floor(2^32 * exp(-d/T_level))), strict <.
bool accept_move(int64_t d, uint32_t x2, const uint32_t* row, int D) {
  if (d <= 0) return true;
  if (d > D) return false;
  return x2 < row[d - 1];
}

} // namespace

extern "C" {

void* orc_problem_create(int N, int E, const int32_t* src, const int32_t* dst, int n_pairs,
                         const int8_t* th_lo, const int8_t* th_hi, int K, int T, int n_obs,
                         const int32_t* obs_times, const uint8_t* init, const uint8_t* clamp,
                         const uint8_t* obs) {
  Problem* P = new Problem();
  P->N = N; P->E = E; P->n_pairs = n_pairs; P->K = K; P->T = T; P->n_obs = n_obs;
  P->src.assign(src, src + E); P->dst.assign(dst, dst + E);
  P->in_edges.assign(N, {});
  for (int e = 0; e < E; ++e) P->in_edges[dst[e]].push_back(e);
  for (int q = 0; q < n_pairs; ++q) { P->th_lo.push_back(th_lo[q]); P->th_hi.push_back(th_hi[q]); }
  P->obs_times.assign(obs_times, obs_times + n_obs);
  P->init.assign(init, init + (size_t)K * N);
  P->clamp.assign(clamp, clamp + (size_t)K * N);
  P->obs.assign(obs, obs + (size_t)K * n_obs * N);
  return P;
}

void orc_problem_destroy(void* h) { delete (Problem*)h; }

uint32_t orc_fitness(const void* h, const int8_t* params) { return fitness(*(const Problem*)h, params, nullptr); }

// full trajectory [K][T+1][N]; returns the fitness
uint32_t orc_simulate(const void* h, const int8_t* params, uint8_t* traj) {
  return fitness(*(const Problem*)h, params, traj);
}

void orc_fitness_batch(const void* h, const int8_t* params, int64_t n, uint32_t* out) {
  const Problem& P = *(const Problem*)h;
  for (int64_t r = 0; r < n; ++r) out[r] = fitness(P, params + r * (P.E + P.N), nullptr);
}

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

uint32_t orc_mulhi(uint32_t a, uint32_t b) { return mulhi(a, b); }

void orc_init_chain(const void* h, uint64_t seed, uint32_t chain, int8_t* params) {
  init_chain(*(const Problem*)h, seed, chain, params);
}

void orc_propose(uint32_t x0, uint32_t x1, int n_params, int n_edges, int n_pairs, const int8_t* cur,
                 int32_t* p_out, int32_t* new_out) {
  int p, nv;
  propose(x0, x1, n_params, n_edges, n_pairs, cur, &p, &nv);
  *p_out = p; *new_out = nv;
}

int orc_accept(int64_t d, uint32_t x2, const uint32_t* row, int D) { return accept_move(d, x2, row, D) ? 1 : 0; }

// SA steps g0 .. g0+n_steps-1 of one chain (Table 1, :130-149).
// cur/best and their fitnesses are updated in place.  trace (optional) gets one u64 per step:
// bits 0-31 delta_cand, 32-55 parameter index, 56-59 new value code (weight+1 or pair index),
// bit 60 accepted, bit 61 new best.
void orc_run_chain(const void* h, uint64_t seed, uint32_t chain, uint64_t g0, int64_t n_steps,
                   int n_levels, int64_t steps_per_level, int D, const uint32_t* table,
                   int8_t* cur, int8_t* best, uint32_t* fit_cur, uint32_t* fit_best, uint64_t* trace) {
  const Problem& P = *(const Problem*)h;
  const int NP = P.E + P.N;
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  std::vector<int8_t> cand(NP);
  for (int64_t it = 0; it < n_steps; ++it) {
    uint64_t g = g0 + (uint64_t)it;
    uint32_t ctr[4] = {(uint32_t)g, (uint32_t)(g >> 32), chain, 0u}, x[4];
    philox4x32_10(ctr, key, x);                       // x[3] is reserved (unused)
    int p, nv;
    propose(x[0], x[1], NP, P.E, P.n_pairs, cur, &p, &nv);
    std::memcpy(cand.data(), cur, NP);
    cand[p] = (int8_t)nv;
    uint32_t f_cand = fitness(P, cand.data(), nullptr);   // every step evaluates a candidate
    int64_t d = (int64_t)f_cand - (int64_t)*fit_cur;
    uint64_t level = g / (uint64_t)steps_per_level;        // reading 20: saturates at L-1
    if (level > (uint64_t)(n_levels - 1)) level = (uint64_t)(n_levels - 1);
    bool acc = accept_move(d, x[2], table + level * (uint64_t)D, D);
    bool new_best = false;
    if (acc) {
      std::memcpy(cur, cand.data(), NP);
      *fit_cur = f_cand;
      if (f_cand < *fit_best) {                             // strict <
        std::memcpy(best, cand.data(), NP);
        *fit_best = f_cand;
        new_best = true;
      }
    }
    if (trace) {
      uint64_t code = (p < P.E) ? (uint64_t)(nv + 1) : (uint64_t)nv;
      trace[it] = (uint64_t)f_cand | ((uint64_t)p << 32) | (code << 56) |
                  ((uint64_t)(acc ? 1 : 0) << 60) | ((uint64_t)(new_best ? 1 : 0) << 61);
    }
  }
}

// T_l = t0 * (t_end/t0)^(l/(L-1)) (T_0 = t0 if L == 1);
// accept[l][d-1] = floor(2^32 * exp(-d / T_l)), d = 1..D, clamped to 2^32 - 1.
void orc_geometric_table(double t0, double t_end, int L, int D, uint32_t* out) {
  for (int l = 0; l < L; ++l) {
    double temp = (L == 1) ? t0 : t0 * std::pow(t_end / t0, (double)l / (double)(L - 1));
    for (int d = 1; d <= D; ++d) {
      double v = std::floor(4294967296.0 * std::exp(-(double)d / temp));
      out[(size_t)l * D + (d - 1)] = (v >= 4294967295.0) ? 0xFFFFFFFFu : (uint32_t)v;
    }
  }
}


// ---------------------------------------------------------------------------------------------------
// Structural constraints in the config model, where one signed weight stands for the
// paper's weight and polarity (w = +1 is an active activator, w = -1 an active inhibitor, 0 no edge):
//   (a) every node has an in-edge and an out-edge of non-zero weight  (:187-191),
//   (b) every node has an in-edge with w = +1                         (:193-199).
// Checked by scanning the whole vector (reading C1).  Threshold parameters are unconstrained.
int orc_valid(const void* h, const int8_t* x) {
  const Problem& P = *(const Problem*)h;
  std::vector<int> in_nz(P.N, 0), out_nz(P.N, 0), act(P.N, 0);
  for (int e = 0; e < P.E; ++e) {
    if (x[e] != 0) { in_nz[P.dst[e]] += 1; out_nz[P.src[e]] += 1; }
    if (x[e] == 1) act[P.dst[e]] += 1;
  }
  for (int i = 0; i < P.N; ++i)
    if (in_nz[i] == 0 || out_nz[i] == 0 || act[i] == 0) return 0;
  return 1;
}

// Initial vector under constraints (:201 "each thread is given a valid solution vector"; reading C3): the
// unconstrained vector of init_chain, then a repair pass "by conditionals" with Philox(ctr = (i, 0, chain, 2))
// = (y0..y3) for node i: first, for i = 0..N-1, a node without a +1 in-edge gets w = +1 on its
// mulhi(y0, indeg)-th in-edge (caller's edge order); then, for i = 0..N-1, a node without a non-zero
// out-edge gets w = 2 * mulhi(y3, 2) - 1 on its mulhi(y2, outdeg)-th out-edge.
void orc_init_chain_c(const void* h, uint64_t seed, uint32_t chain, int8_t* x) {
  const Problem& P = *(const Problem*)h;
  init_chain(P, seed, chain, x);
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  std::vector<std::vector<int>> out_edges(P.N);
  for (int e = 0; e < P.E; ++e) out_edges[P.src[e]].push_back(e);
  for (int i = 0; i < P.N; ++i) {
    bool act = false;
    for (int e : P.in_edges[i]) act = act || x[e] == 1;
    if (act) continue;
    uint32_t ctr[4] = {(uint32_t)i, 0u, chain, 2u}, y[4];
    philox4x32_10(ctr, key, y);
    x[P.in_edges[i][mulhi(y[0], (uint32_t)P.in_edges[i].size())]] = 1;
  }
  for (int i = 0; i < P.N; ++i) {
    bool nz = false;
    for (int e : out_edges[i]) nz = nz || x[e] != 0;
    if (nz) continue;
    uint32_t ctr[4] = {(uint32_t)i, 0u, chain, 2u}, y[4];
    philox4x32_10(ctr, key, y);
    x[out_edges[i][mulhi(y[2], (uint32_t)out_edges[i].size())]] = (int8_t)(2 * (int)mulhi(y[3], 2u) - 1);
  }
}

// GetCandidate under constraints (:201 "by using conditionals when perturbing the weight or polarity
// components"; reading C2): index as in propose(); for a weight the two other values are listed
// cyclically after the old one (code+1, code+2 mod 3), those whose vector would break (a) or (b) are
// struck, the new value is entry mulhi(x1, length) of the list; an empty list gives a null move
// (*new_out = old value, returns 0).  With both values allowed this is propose().  Thresholds as in propose().
int orc_propose_c(const void* h, uint32_t x0, uint32_t x1, const int8_t* cur, int32_t* p_out, int32_t* new_out) {
  const Problem& P = *(const Problem*)h;
  const int NP = P.E + P.N;
  const int p = (int)mulhi(x0, (uint32_t)NP);
  *p_out = p;
  if (p >= P.E) {
    int q, nv;
    propose(x0, x1, NP, P.E, P.n_pairs, cur, &q, &nv);
    *new_out = nv;
    return 1;
  }
  const int code = cur[p] + 1;
  std::vector<int8_t> cand(cur, cur + NP);
  int list[2], len = 0;
  for (int k = 1; k <= 2; ++k) {
    const int v = (code + k) % 3 - 1;
    cand[p] = (int8_t)v;
    if (orc_valid(h, cand.data())) list[len++] = v;
  }
  if (len == 0) { *new_out = cur[p]; return 0; }
  *new_out = list[mulhi(x1, (uint32_t)len)];
  return 1;
}

// orc_run_chain with the constrained GetCandidate; trace bit 62 = null move.  Everything else (Philox
// counter layout, roles of x0 / x1 / x2, level rule, accept test, strict-improvement best) as above.
void orc_run_chain_c(const void* h, uint64_t seed, uint32_t chain, uint64_t g0, int64_t n_steps,
                     int n_levels, int64_t steps_per_level, int D, const uint32_t* table,
                     int8_t* cur, int8_t* best, uint32_t* fit_cur, uint32_t* fit_best, uint64_t* trace) {
  const Problem& P = *(const Problem*)h;
  const int NP = P.E + P.N;
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  std::vector<int8_t> cand(NP);
  for (int64_t it = 0; it < n_steps; ++it) {
    uint64_t g = g0 + (uint64_t)it;
    uint32_t ctr[4] = {(uint32_t)g, (uint32_t)(g >> 32), chain, 0u}, x[4];
    philox4x32_10(ctr, key, x);
    int32_t p, nv;
    const int moved = orc_propose_c(h, x[0], x[1], cur, &p, &nv);
    std::memcpy(cand.data(), cur, NP);
    cand[p] = (int8_t)nv;
    uint32_t f_cand = fitness(P, cand.data(), nullptr);
    int64_t d = (int64_t)f_cand - (int64_t)*fit_cur;
    uint64_t level = g / (uint64_t)steps_per_level;
    if (level > (uint64_t)(n_levels - 1)) level = (uint64_t)(n_levels - 1);
    bool acc = accept_move(d, x[2], table + level * (uint64_t)D, D);
    bool new_best = false;
    if (acc) {
      std::memcpy(cur, cand.data(), NP);
      *fit_cur = f_cand;
      if (f_cand < *fit_best) {
        std::memcpy(best, cand.data(), NP);
        *fit_best = f_cand;
        new_best = true;
      }
    }
    if (trace) {
      uint64_t code = (p < P.E) ? (uint64_t)(nv + 1) : (uint64_t)nv;
      trace[it] = (uint64_t)f_cand | ((uint64_t)p << 32) | (code << 56) | ((uint64_t)(acc ? 1 : 0) << 60) |
                  ((uint64_t)(new_best ? 1 : 0) << 61) | ((uint64_t)(moved ? 0 : 1) << 62);
    }
  }
}

} // extern "C"

