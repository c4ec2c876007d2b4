// CPU ORACLE, PAPER MODEL — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded restatement of the paper's OWN model (arxiv 2506.19866 §2.1-2.3,
// §2.5.3): three parameters per edge (weight w, polarity p,
// activation threshold t), three per node (speed u, memory m, step size d), the priority update
// scheme, the gradient-weighted Manhattan objective, the structural constraints in GetCandidate and at
// initialisation, inside the chain step of Table 1.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code with the CUDA path
// under paper_2506_19866_b200/csrc; within oracle/ it links the Philox4x32-10, mulhi and accept
// functions of sa_oracle.cpp (pinned there) instead of repeating them.
//
// Style rules as in sa_oracle.cpp: one byte per state, per-node edge lists in the caller's edge
// order, no bit tricks, no incremental evaluation, constraints checked by scanning the whole vector.
//
// Pins (tests/test_oracle_paper_pins.py, -m "not gpu"): hand-worked Example C (priority update, every
// rule exercised) and Example D (objective) under tests/golden/, parameter counts 102 / 723, y = 0 on
// self-generated data, the first transition against the synchronous oracle where the two models
// coincide, value-domain mappings at the mulhi boundaries, brute force over every neighbour of every
// valid vector of a 3-node network for the constraints, the wiring of the chain step recomputed
// outside this file from ATen's Philox.
// PARITY UNPINNED (ref [9] of the paper, which defines the priority scheme in full, is not in the
// container): the readings P1-P6 of DESIGN.md §3 that ref [9] would have settled — clipping the image
// to [0,2] before comparing it with the state, the memory counter's reset rule, the age of a node at
// t = 1, "priority class" = equal priority value.  The hand-worked example pins the code to these
// readings, not the readings to the paper.

#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

extern "C" {
void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out);   // sa_oracle.cpp
uint32_t orc_mulhi(uint32_t a, uint32_t b);
int orc_accept(int64_t d, uint32_t x2, const uint32_t* row, int D);
}

namespace {

struct PProblem {
  int N = 0, E = 0, K = 0, T = 0;
  std::vector<int> src, dst;
  std::vector<std::vector<int>> in_edges, out_edges;   // edge ids, ascending (caller's order)
  std::vector<uint8_t> fast;                           // [N] 1 = speed range {10,11,12}, 0 = {1..6}
  std::vector<uint8_t> init;                           // [K][N]
  std::vector<uint8_t> ref;                            // [K][T+1][N] reference matrix R, 255 = not measured
  int NP() const { return 3 * E + 3 * N; }
};

// Parameter vector x = [w(E), p(E), t(E), u(N), m(N), d(N)], values themselves:
// w in {0,1,2}, p in {-1,0,1}, t in {1,2} (:61-64); u in {1..6} or {10,11,12}, m in {0,1,2}, d in {1,2} (:78-80).
struct View {
  const int8_t *w, *p, *t, *u, *m, *d;
  View(const PProblem& P, const int8_t* x) : w(x), p(x + P.E), t(x + 2 * P.E), u(x + 3 * P.E), m(x + 3 * P.E + P.N), d(x + 3 * P.E + 2 * P.N) {}
};

// Number of values of parameter index q and the i-th of them, in increasing order.
int domain_size(const PProblem& P, int q) {
  if (q < 2 * P.E) return 3;                         // w, p
  if (q < 3 * P.E) return 2;                         // t
  q -= 3 * P.E;
  if (q < P.N) return P.fast[q] ? 3 : 6;             // u
  if (q < 2 * P.N) return 3;                         // m
  return 2;                                          // d
}
int domain_value(const PProblem& P, int q, int i) {
  if (q < P.E) return i;                             // w: 0,1,2
  if (q < 2 * P.E) return i - 1;                     // p: -1,0,1
  if (q < 3 * P.E) return i + 1;                     // t: 1,2
  q -= 3 * P.E;
  if (q < P.N) return P.fast[q] ? 10 + i : 1 + i;    // u
  if (q < 2 * P.N) return i;                         // m
  return i + 1;                                      // d
}
int domain_index(const PProblem& P, int q, int v) {
  for (int i = 0; i < domain_size(P, q); ++i)
    if (domain_value(P, q, i) == v) return i;
  return -1;
}

// One transition t-1 -> t of the priority update scheme (readings P1-P4).
// s: states at t-1 (in), states at t (out).  last[i]: time of node i's last state change (0 at the
// start).  told[i]: consecutive time steps up to t-1 at which node i was told to update but did not.
void priority_step(const PProblem& P, const View& x, int t, uint8_t* s, int* last, int* told_run) {
  const int N = P.N;
  std::vector<int> target(N), prio(N);
  std::vector<char> told(N), eligible(N);
  int top = 0;
  for (int i = 0; i < N; ++i) {
    // image (:66-68, reading 16): K_i = SUM over sources j of (s_j // t_ji) * w_ji * p_ji, floor division
    int K = 0;
    for (int e : P.in_edges[i]) K += ((int)s[P.src[e]] / (int)x.t[e]) * (int)x.w[e] * (int)x.p[e];
    // :70, :82: the image pushes s_i toward K_i as far as the allowable states go (P1)
    target[i] = K < 0 ? 0 : K > 2 ? 2 : K;
    told[i] = target[i] != (int)s[i];                  // image differs from the state and there is room to move
    eligible[i] = told[i] && told_run[i] >= (int)x.m[i];   // memory criterion (:79, P2)
    prio[i] = eligible[i] ? (int)x.u[i] * (t - last[i]) : 0;   // :82: speed x time steps since last updated (P3)
    if (prio[i] > top) top = prio[i];
  }
  for (int i = 0; i < N; ++i) {
    if (eligible[i] && prio[i] == top) {               // the nodes sharing the highest priority (P4) move ...
      int dist = target[i] > (int)s[i] ? target[i] - (int)s[i] : (int)s[i] - target[i];
      int step = dist < (int)x.d[i] ? dist : (int)x.d[i];   // ... at most d_i levels toward K_i (:80, :82)
      s[i] = (uint8_t)(target[i] > (int)s[i] ? (int)s[i] + step : (int)s[i] - step);
      last[i] = t;
      told_run[i] = 0;
    } else if (told[i]) {
      told_run[i] += 1;
    } else {
      told_run[i] = 0;
    }
  }
  // (the loop above reads s[i] and target[i] of node i only, so updating s in place is still the
  // synchronous "updated at the end of the current time step" of :82: every image was formed before it)
}

// Objective (:88-111, readings 15, 17): y = SUM over time courses, t = 0..T and measured i of
// |s_{t,i} - r_{t,i}| * (|g_{t,i}| + 1), g_{0,i} = 0, g_{t,i} = r_{t,i} - r_{t-1,i} (0 where either is
// not measured).  traj (optional): [K][T+1][N].
uint32_t objective(const PProblem& P, const int8_t* params, uint8_t* traj) {
  const View x(P, params);
  const int N = P.N;
  uint32_t y = 0;
  std::vector<uint8_t> s(N);
  std::vector<int> last(N), told_run(N);
  for (int k = 0; k < P.K; ++k) {
    for (int i = 0; i < N; ++i) { s[i] = P.init[(size_t)k * N + i]; last[i] = 0; told_run[i] = 0; }
    for (int t = 0; t <= P.T; ++t) {
      if (t > 0) priority_step(P, x, t, s.data(), last.data(), told_run.data());
      if (traj) std::memcpy(traj + ((size_t)k * (P.T + 1) + t) * N, s.data(), N);
      const uint8_t* r = &P.ref[((size_t)k * (P.T + 1) + t) * N];
      const uint8_t* rp = t > 0 ? r - N : nullptr;
      for (int i = 0; i < N; ++i) {
        if (r[i] == 255) continue;
        int g = (rp && rp[i] != 255) ? (int)r[i] - (int)rp[i] : 0;
        y += (uint32_t)(std::abs((int)s[i] - (int)r[i]) * (std::abs(g) + 1));
      }
    }
  }
  return y;
}

// Structural constraints (:186-199, reading 18): (a) every node has an in-edge and an out-edge of
// non-zero weight; (b) every node has an in-edge with p = +1 and w != 0.
bool valid(const PProblem& P, const int8_t* params) {
  const View x(P, params);
  for (int i = 0; i < P.N; ++i) {
    int in_w = 0, out_w = 0, act = 0;
    for (int e : P.in_edges[i]) { in_w += x.w[e]; if (x.p[e] == 1 && x.w[e] != 0) act += 1; }
    for (int e : P.out_edges[i]) out_w += x.w[e];
    if (in_w == 0 || out_w == 0 || act < 1) return false;
  }
  return true;
}

void philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint64_t seed, uint32_t out[4]) {
  uint32_t ctr[4] = {c0, c1, c2, c3}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  orc_philox4x32_10(ctr, key, out);
}

// Initial vector (:124 "a randomized parameter vector"; :201 "each thread is given a valid solution
// vector"; readings 8, P6).  Block b of four parameters takes Philox(ctr = (b, 0, chain, 1)): value
// index = mulhi(y, domain size).  With constraints on, a repair pass follows (the paper uses a
// solver; here conditionals, as in GetCandidate): node i takes Philox(ctr = (i, 0, chain, 2)) = (y0..y3);
// first, for i = 0..N-1: if node i has no in-edge with p = +1 and w != 0, its mulhi(y0, indeg)-th
// in-edge gets p = +1 and, if its weight is 0, w = 1 + mulhi(y1, 2); then, for i = 0..N-1: if node i
// has no out-edge with w != 0, its mulhi(y2, outdeg)-th out-edge gets w = 1 + mulhi(y3, 2).
void init_chain(const PProblem& P, uint64_t seed, uint32_t chain, int constrained, int8_t* x) {
  const int NP = P.NP();
  for (int b = 0; 4 * b < NP; ++b) {
    uint32_t y[4];
    philox((uint32_t)b, 0u, chain, 1u, seed, y);
    for (int j = 0; j < 4 && 4 * b + j < NP; ++j) {
      int q = 4 * b + j;
      x[q] = (int8_t)domain_value(P, q, (int)orc_mulhi(y[j], (uint32_t)domain_size(P, q)));
    }
  }
  if (!constrained) return;
  int8_t *w = x, *p = x + P.E;
  for (int i = 0; i < P.N; ++i) {
    int act = 0;
    for (int e : P.in_edges[i]) if (p[e] == 1 && w[e] != 0) act += 1;
    if (act >= 1) continue;
    uint32_t y[4];
    philox((uint32_t)i, 0u, chain, 2u, seed, y);
    int e = P.in_edges[i][orc_mulhi(y[0], (uint32_t)P.in_edges[i].size())];
    p[e] = 1;
    if (w[e] == 0) w[e] = (int8_t)(1 + (int)orc_mulhi(y[1], 2u));
  }
  for (int i = 0; i < P.N; ++i) {
    int out_w = 0;
    for (int e : P.out_edges[i]) out_w += w[e];
    if (out_w != 0) continue;
    uint32_t y[4];
    philox((uint32_t)i, 0u, chain, 2u, seed, y);
    int e = P.out_edges[i][orc_mulhi(y[2], (uint32_t)P.out_edges[i].size())];
    w[e] = (int8_t)(1 + (int)orc_mulhi(y[3], 2u));
  }
}

// GetCandidate (:131-133 "random single-element change"; :201 constraints "by using conditionals when
// perturbing the weight or polarity components"; readings 7, P5).  q = mulhi(x0, 3E+3N).  The other
// values of parameter q are listed cyclically after the old one (old+1, old+2, ... in domain order);
// with constraints on, those that would break (a) or (b) are struck from the list; the new value is
// entry mulhi(x1, length) of the list.  An empty list gives a null move: candidate = current,
// *new_out = old value, returns 0 (else 1).
int propose(const PProblem& P, uint32_t x0, uint32_t x1, const int8_t* cur, int constrained, int* q_out, int* new_out) {
  const int NP = P.NP();
  const int q = (int)orc_mulhi(x0, (uint32_t)NP);
  const int n = domain_size(P, q), old_i = domain_index(P, q, cur[q]);
  std::vector<int> list;
  std::vector<int8_t> cand(cur, cur + NP);
  for (int k = 1; k < n; ++k) {
    int v = domain_value(P, q, (old_i + k) % n);
    if (constrained) {
      cand[q] = (int8_t)v;
      if (!valid(P, cand.data())) continue;
    }
    list.push_back(v);
  }
  *q_out = q;
  if (list.empty()) { *new_out = cur[q]; return 0; }
  *new_out = list[orc_mulhi(x1, (uint32_t)list.size())];
  return 1;
}

}  // namespace

extern "C" {

void* orcp_problem_create(int N, int E, const int32_t* src, const int32_t* dst, const uint8_t* fast, int K, int T,
                          const uint8_t* init, const uint8_t* ref) {
  PProblem* P = new PProblem();
  P->N = N; P->E = E; P->K = K; P->T = T;
  P->src.assign(src, src + E); P->dst.assign(dst, dst + E);
  P->in_edges.assign(N, {}); P->out_edges.assign(N, {});
  for (int e = 0; e < E; ++e) { P->in_edges[dst[e]].push_back(e); P->out_edges[src[e]].push_back(e); }
  P->fast.assign(fast, fast + N);
  P->init.assign(init, init + (size_t)K * N);
  P->ref.assign(ref, ref + (size_t)K * (T + 1) * N);
  return P;
}

void orcp_problem_destroy(void* h) { delete (PProblem*)h; }

uint32_t orcp_objective(const void* h, const int8_t* params) { return objective(*(const PProblem*)h, params, nullptr); }

uint32_t orcp_simulate(const void* h, const int8_t* params, uint8_t* traj) { return objective(*(const PProblem*)h, params, traj); }

void orcp_objective_batch(const void* h, const int8_t* params, int64_t n, uint32_t* out) {
  const PProblem& P = *(const PProblem*)h;
  for (int64_t r = 0; r < n; ++r) out[r] = objective(P, params + r * P.NP(), nullptr);
}

int orcp_valid(const void* h, const int8_t* params) { return valid(*(const PProblem*)h, params) ? 1 : 0; }

void orcp_init_chain(const void* h, uint64_t seed, uint32_t chain, int constrained, int8_t* params) {
  init_chain(*(const PProblem*)h, seed, chain, constrained, params);
}

int orcp_propose(const void* h, uint32_t x0, uint32_t x1, const int8_t* cur, int constrained, int32_t* q_out, int32_t* new_out) {
  int q, nv;
  int moved = propose(*(const PProblem*)h, x0, x1, cur, constrained, &q, &nv);
  *q_out = q; *new_out = nv;
  return moved;
}

int orcp_domain_size(const void* h, int q) { return domain_size(*(const PProblem*)h, q); }
int orcp_domain_value(const void* h, int q, int i) { return domain_value(*(const PProblem*)h, q, i); }

// SA steps g0 .. g0+n_steps-1 of one chain (Table 1 :130-149), as orc_run_chain of
// sa_oracle.cpp (same Philox counter layout, same roles of x0 / x1 / x2, same level
// rule, same integer accept test) around this model's GetCandidate and Simulate.  Trace record: bits
// 0-31 delta_cand, 32-55 parameter index, 56-59 index of the new value in the parameter's domain,
// bit 60 accepted, bit 61 new best, bit 62 null move (no feasible value; the candidate is the current vector).
void orcp_run_chain(const void* h, uint64_t seed, uint32_t chain, uint64_t g0, int64_t n_steps, int n_levels,
                    int64_t steps_per_level, int D, const uint32_t* table, int constrained, int8_t* cur, int8_t* best,
                    uint32_t* fit_cur, uint32_t* fit_best, uint64_t* trace) {
  const PProblem& P = *(const PProblem*)h;
  const int NP = P.NP();
  std::vector<int8_t> cand(NP);
  for (int64_t it = 0; it < n_steps; ++it) {
    uint64_t g = g0 + (uint64_t)it;
    uint32_t x[4];
    philox((uint32_t)g, (uint32_t)(g >> 32), chain, 0u, seed, x);
    int q, nv;
    int moved = propose(P, x[0], x[1], cur, constrained, &q, &nv);
    std::memcpy(cand.data(), cur, NP);
    cand[q] = (int8_t)nv;
    uint32_t f_cand = objective(P, cand.data(), nullptr);      // every step evaluates a candidate
    int64_t d = (int64_t)f_cand - (int64_t)*fit_cur;
    uint64_t level = g / (uint64_t)steps_per_level;
    if (level > (uint64_t)(n_levels - 1)) level = (uint64_t)(n_levels - 1);
    bool acc = orc_accept(d, x[2], table + level * (uint64_t)D, D) != 0;
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
      uint64_t code = (uint64_t)domain_index(P, q, nv);
      trace[it] = (uint64_t)f_cand | ((uint64_t)q << 32) | (code << 56) | ((uint64_t)(acc ? 1 : 0) << 60) |
                  ((uint64_t)(new_best ? 1 : 0) << 61) | ((uint64_t)(moved ? 0 : 1) << 62);
    }
  }
}

}  // extern "C"
