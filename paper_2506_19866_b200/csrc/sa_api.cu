// C ABI of libternary_sa.so (include/ternary_sa.h): argument checking, device memory, launches.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <memory>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "sa_tuning.h"
#include "../../include/ternary_sa.h"
#include "sa_common.h"
#include "sa_host.h"
#include "sa_jit.h"
#include "sa_kernels.h"
#include "sa_plan.h"

namespace {

using tsa::cuda_err;
using tsa::DevPool;
using tsa::g_alloc;
using tsa::g_err;
using tsa::g_free;
using tsa::set_err;

int upload_problem(const tsa::Plan& pl, DevPool& pool, tsa::DevProblem* P, cudaStream_t st) {
  tsa::DevProblem& d = *P;
  std::memset(&d, 0, sizeof(d));
  d.N = pl.N; d.E = pl.E; d.P = pl.P; d.K = pl.K; d.T = pl.T; d.n_obs = pl.n_obs; d.n_pairs = pl.n_pairs;
  d.CG = pl.CG; d.n_chunks = pl.n_chunks; d.n_pass = pl.n_pass; d.n_entries = pl.n_entries;
  d.Epad = pl.Epad; d.EpadA = pl.EpadA; d.NpadA = pl.NpadA; d.state_words = pl.state_words;
  d.fit_const = pl.fit_const;
  d.n_fix = (int)pl.fix.size();
  std::memcpy(d.tha, pl.tha, sizeof(d.tha));
  std::memcpy(d.thb, pl.thb, sizeof(d.thb));
  std::vector<int4> info((size_t)pl.n_chunks * pl.n_pass);
  for (int ch = 0; ch < pl.n_chunks; ++ch)
    for (int ps = 0; ps < pl.n_pass; ++ps) {
      const size_t x = (size_t)ch * pl.n_pass + ps;
      info[x] = make_int4(pl.pass_base[ps], pl.pass_iters[ps] | (pl.pass_rounds[ps] << 16), pl.fix_ptr[x],
                          pl.fix_ptr[x + 1] - pl.fix_ptr[x]);
    }
  int rc;
  if ((rc = pool.upload(info, &d.pass_info, st))) return rc;
  if ((rc = pool.upload(pl.row_meta, &d.row_meta, st))) return rc;
  if ((rc = pool.upload(pl.slot_off, &d.slot_off, st))) return rc;
  if ((rc = pool.upload(pl.slot_of_param, &d.slot_of_param, st))) return rc;
  if ((rc = pool.upload(pl.entry_of_node, &d.entry_of_node, st))) return rc;
  if ((rc = pool.upload(pl.initw, &d.initw, st))) return rc;
  if ((rc = pool.upload(pl.obsw, &d.obsw, st))) return rc;
  if ((rc = pool.upload(pl.obsm, &d.obsm, st))) return rc;
  if ((rc = pool.upload(pl.fix, &d.fix, st))) return rc;
  if ((rc = pool.upload(pl.obs_idx_of_t, &d.obs_idx_of_t, st))) return rc;
  // the host vector `info` must outlive the async copy
  if (cudaStreamSynchronize(st) != cudaSuccess) return set_err(SA_ECUDA, "upload failed");
  return SA_OK;
}

int pick_threads(const tsa::DevProblem& P, int64_t n_ctas, int sm_count) {
  if (const char* env = tsa::tune_env("TSA_TEAM_WARPS")) {
    int w = std::atoi(env);
    if (w >= 1 && w <= 32) return 32 * w;
  }
  // aim at ~32 resident warps per SM: CTAs per SM are bounded by shared memory, the 32-CTA limit
  // and the grid itself; the rest comes from warps per chain (at most one per pass, at most 8)
  const size_t sb = tsa::smem_bytes(P) + 1024;
  int64_t per_sm = std::min<int64_t>(32, (int64_t)(227 * 1024 / sb));
  per_sm = std::max<int64_t>(1, std::min<int64_t>(per_sm, (n_ctas + sm_count - 1) / sm_count));
  int warps = (int)std::max<int64_t>(1, 32 / per_sm);
  warps = std::min(warps, std::min(P.n_pass, 8));
  return 32 * warps;
}

// WarpTeam launch shape: chains per CTA that minimises the busiest SM's chain count (all chains run
// the same number of steps, so the makespan is set by the fullest SM), larger CTAs on ties.
// Returns 0 when the warp-per-chain kernel does not apply.
int pick_warp_cpb(const tsa::DevProblem& P, int64_t R, int sm_count) {
  if (const char* env = std::getenv("TSA_KERNEL")) {
    if (std::string(env) == "cta") return 0;
    if (std::string(env) == "warp" && P.n_pass <= 32) {
      int cpb = 8;
      if (const char* c = tsa::tune_env("TSA_CPB")) cpb = std::max(1, std::min(8, std::atoi(c)));
      return tsa::warp_kernel_smem(P, cpb) <= 227 * 1024 ? cpb : 0;
    }
  }
  if (P.n_pass > 8) return 0;                                   // one warp per chain would be too slow
  if (P.n_pass > 1 && R < 16LL * sm_count) return 0;            // few chains: spread each over a CTA
  int best = 0;
  int64_t best_load = 0;
  for (int cpb = 8; cpb >= 1; --cpb) {
    const size_t sb = tsa::warp_kernel_smem(P, cpb);
    if (sb > 227 * 1024) continue;
    const int64_t ctas = (R + cpb - 1) / cpb;
    const int64_t fit = std::min<int64_t>(32, (int64_t)((228 * 1024) / (sb + 1024)));
    if (fit < 1) continue;
    const int64_t per_sm = (ctas + sm_count - 1) / sm_count;
    const int64_t load = (per_sm <= fit) ? per_sm * cpb                      // single wave: static imbalance
                                         : (R + sm_count - 1) / sm_count + cpb;   // several waves: dynamic, ~even
    const int64_t resident = std::min(per_sm, fit) * cpb;
    if (resident < std::min<int64_t>(16, (R + sm_count - 1) / sm_count)) continue;   // keep >= 16 warps per SM if possible
    if (best == 0 || load < best_load) { best = cpb; best_load = load; }
  }
  return best;
}

}  // namespace

struct sa_handle {
  tsa::Plan plan;
  tsa::DevProblem P;
  tsa::DevChains C;
  tsa::DevSched S;
  tsa::DevTrace Tr;
  DevPool pool;         // problem + chain store
  DevPool trace_pool;   // trace buffers (re-armed by sa_set_trace)
  cudaStream_t stream = 0;
  uint64_t g = 0;       // global step counter
  int threads = 32;
  int warp_cpb = 0;     // > 0: sa_run uses the warp-per-chain kernel with this many chains per CTA
  int sm_count = 148;
  int64_t launches = 0;
  int32_t n_traced = 0;
  int64_t trace_steps = 0;
  // statically scheduled kernel (sa_jit.h): device tables, the compiled kernel, the family choice
  const uint32_t *d_lane_off2 = nullptr, *d_lane_meta = nullptr, *d_lane_clamp = nullptr, *d_wloc = nullptr, *d_thloc = nullptr;
  const tsa::StaticKernel* sk = nullptr;
  bool sk_tried = false;
  // dense (tensor-pipe) kernel (sa_dense_plan.h): host tables, device tables, the compiled kernel
  tsa::DensePlan dplan;
  const uint16_t *d_frag_slot = nullptr, *d_th_entry = nullptr;
  const uint32_t *d_meta = nullptr, *d_init_frag = nullptr, *d_obs_word = nullptr, *d_fix = nullptr, *d_dwloc = nullptr, *d_dthloc = nullptr;
  const tsa::StaticKernel* dk = nullptr;
  bool dk_tried = false;
  uint32_t* d_flags = nullptr;      // [R] hand-over flags of the balanced launch
  uint32_t* d_err = nullptr;        // [1] raised by a kernel whose hand-over wait gave up
  unsigned long long* d_win = nullptr;   // [R] winners of the level synchronisation (sa_run_levels)
  int64_t last_slot_steps = 0;
  std::string dense_why;
  int family = SA_KERNEL_AUTO;
  std::string static_why;
};

namespace {

int env_family(int family) {
  if (const char* env = std::getenv("TSA_KERNEL")) {
    const std::string e(env);
    if (e == "generic" || e == "cta" || e == "warp") return SA_KERNEL_GENERIC;
    if (e == "static") return SA_KERNEL_STATIC;
    if (e == "dense") return SA_KERNEL_DENSE;
  }
  return family;
}

// Decide (once) whether sa_run uses the dense kernel; compiles it on first use.
bool use_dense(sa_handle* h) {
  const int fam = env_family(h->family);
  if (fam != SA_KERNEL_AUTO && fam != SA_KERNEL_DENSE) return false;
  if (!h->dk_tried) {
    h->dk_tried = true;
    tsa::StaticTuning tune = tsa::StaticTuning::from_env();
    // chains per SM the registers allow;
    // fewer chains than that: do not squeeze the registers for an occupancy the grid cannot reach
    const int per_sm = (int)((h->C.R + h->sm_count - 1) / std::max(h->sm_count, 1));
    // small networks (at most 16 weight registers per thread): 16 chains per SM; else 12 at 168 registers, which also
    // measures 1 % faster than 16 at 128 with the sparse operand (183.0 against 180.8 M on Mtb-shaped)
    const bool light = h->dplan.MT * h->dplan.KS * 4 <= 64;
    const int resident = std::max(1, std::min(light ? 16 : 12, per_sm));
    if (!tsa::tune_env("TSA_DENSE_BLOCKS")) tune.dense_blocks = resident;
    // one-warp chains: all of an SM's chains in ONE CTA, whose warps the hardware spreads evenly over the four
    // sub-partitions (one-warp CTAs land unevenly: measured 155 against 163 M chain-steps/s on Mtb-shaped)
    if (tune.dense_cpb == 0) tune.dense_cpb = h->dplan.W == 1 ? (tune.dense_blocks > 0 && tsa::tune_env("TSA_DENSE_BLOCKS") ? 1 : resident) : 1;
    tune.constrained = h->S.constrained ? 1 : 0;
    h->dk = tsa::dense_kernel_get(h->plan, h->dplan, tune, &h->dense_why);
  }
  return h->dk != nullptr;
}

tsa_dense::Params dense_params(const sa_handle* h, int64_t steps) {
  tsa_dense::Params q;
  std::memset(&q, 0, sizeof(q));
  q.frag_slot = h->d_frag_slot; q.meta = h->d_meta; q.th_entry = h->d_th_entry; q.init_frag = h->d_init_frag;
  q.obs_word = h->d_obs_word; q.fix = h->d_fix; q.wloc = h->d_dwloc; q.thloc = h->d_dthloc;
  q.con_in_ptr = h->P.con_in_ptr; q.con_in_slot = h->P.con_in_slot; q.con_out_ptr = h->P.con_out_ptr;
  q.con_out_slot = h->P.con_out_slot; q.edge_nodes = h->P.edge_nodes;
  std::memcpy(q.tha, h->P.tha, 16);
  std::memcpy(q.thb, h->P.thb, 16);
  q.fit_const = h->dplan.fit_const;
  q.R = h->C.R;
  q.cur_w = h->C.cur_w; q.cur_th = h->C.cur_th; q.best_w = h->C.best_w; q.best_th = h->C.best_th;
  q.fit_cur = h->C.fit_cur; q.fit_best = h->C.fit_best;
  q.key0 = h->S.key0; q.key1 = h->S.key1; q.chain_id_base = h->S.chain_id_base;
  q.n_levels = h->S.n_levels; q.dmax = h->S.dmax; q.steps_per_level = h->S.steps_per_level;
  q.accept = h->S.accept;
  q.level_stats = h->S.level_stats;
  q.trace_row = h->Tr.row_of_chain; q.trace_rec = (tsa_dense::u64*)h->Tr.records;
  q.trace_max = h->Tr.max_steps; q.trace_g0 = h->Tr.g_start;
  q.g0 = h->g; q.steps = steps;
  q.err = h->d_err;
  return q;
}

// Decide (once) whether sa_run uses the static kernel; compiles it on first use.
bool use_static(sa_handle* h) {
  const int fam = env_family(h->family);
  if (fam == SA_KERNEL_GENERIC || fam == SA_KERNEL_DENSE) return false;
  if (!h->sk_tried) {
    h->sk_tried = true;
    tsa::StaticTuning tune = tsa::StaticTuning::from_env();
    tune.constrained = h->S.constrained ? 1 : 0;
    h->sk = tsa::static_kernel_get(h->plan, tune, &h->static_why);
  }
  return h->sk != nullptr;
}

tsa_static::Params static_params(const sa_handle* h, int64_t steps) {
  tsa_static::Params q;
  std::memset(&q, 0, sizeof(q));
  q.lane_off2 = h->d_lane_off2; q.lane_meta = h->d_lane_meta; q.lane_clamp = h->d_lane_clamp;
  q.initw = h->P.initw; q.obsw = h->P.obsw; q.obsm = h->P.obsm;
  q.wloc = h->d_wloc; q.thloc = h->d_thloc;
  q.con_in_ptr = h->P.con_in_ptr; q.con_in_slot = h->P.con_in_slot; q.con_out_ptr = h->P.con_out_ptr;
  q.con_out_slot = h->P.con_out_slot; q.edge_nodes = h->P.edge_nodes;
  std::memcpy(q.tha, h->P.tha, 16);
  std::memcpy(q.thb, h->P.thb, 16);
  q.fit_const = h->P.fit_const;
  q.R = h->C.R;
  q.cur_w = h->C.cur_w; q.cur_th = h->C.cur_th; q.best_w = h->C.best_w; q.best_th = h->C.best_th;
  q.fit_cur = h->C.fit_cur; q.fit_best = h->C.fit_best;
  q.key0 = h->S.key0; q.key1 = h->S.key1; q.chain_id_base = h->S.chain_id_base;
  q.n_levels = h->S.n_levels; q.dmax = h->S.dmax; q.steps_per_level = h->S.steps_per_level;
  q.accept = h->S.accept;
  q.level_stats = h->S.level_stats;
  q.trace_row = h->Tr.row_of_chain; q.trace_rec = (tsa_static::u64*)h->Tr.records;
  q.trace_max = h->Tr.max_steps; q.trace_g0 = h->Tr.g_start;
  q.g0 = h->g; q.steps = steps;
  return q;
}

tsa::PlanOptions plan_options(int64_t n_chains, int sm_count) {
  tsa::PlanOptions o = tsa::PlanOptions::from_env();
  if (!tsa::tune_env("TSA_TEAM_MIN")) {
    // few chains: spread each over more warps so that an SM still sees ~16 resident warps
    const int64_t want = (16LL * sm_count + n_chains - 1) / std::max<int64_t>(n_chains, 1);
    o.min_team_warps = (int)std::max<int64_t>(1, std::min<int64_t>(32, want));
  }
  return o;
}

// Host plans (edge schedule, bank classes, 2:4 row search, fragment tables) are a pure function of the problem and
// the options, and take tens of milliseconds: sa_create keeps the last few, keyed by the problem's bytes, so that a
// second handle on the same problem (another chain range, another schedule, a restart) only pays for the device side.
struct CachedPlans { tsa::Plan plan; tsa::DensePlan dplan; uint64_t born = 0; };
constexpr size_t kCachedPlans = 8;
uint64_t g_plans_clock = 0;
std::mutex g_plans_mu;
std::map<std::string, std::shared_ptr<const CachedPlans>> g_plans;

bool plan_key(const sa_network* net, const sa_observations* obs, const tsa::PlanOptions& o, const tsa::StaticTuning& t, std::string* key) {
  if (net->n_nodes <= 0 || net->n_edges <= 0 || net->n_pairs <= 0 || net->n_pairs > 16 || !net->edge_src || !net->edge_dst ||
      !net->th_lo || !net->th_hi || obs->n_cond <= 0 || obs->n_steps <= 0 || obs->n_obs <= 0 || !obs->obs_times ||
      !obs->init_state || !obs->clamp || !obs->obs)
    return false;                                        // let build_plan say what is wrong
  const size_t N = (size_t)net->n_nodes, E = (size_t)net->n_edges, K = (size_t)obs->n_cond, NO = (size_t)obs->n_obs;
  if (N > 100000 || E > 10000000 || K > 1024 || NO > 100000) return false;
  auto put = [&](const void* ptr, size_t n) { key->append((const char*)ptr, n); };
  const int32_t head[] = {net->n_nodes, net->n_edges, net->n_pairs, obs->n_cond, obs->n_steps, obs->n_obs, (int32_t)o.split_rows,
                          (int32_t)o.bank_opt, (int32_t)o.store_opt, (int32_t)o.tiers, o.min_team_warps, o.max_lane_slots, t.dense_warps, t.dense_sparse,
                          t.dense_swizzle, t.dense_movm};
  put(head, sizeof(head));
  put(net->edge_src, E * 4); put(net->edge_dst, E * 4); put(net->th_lo, (size_t)net->n_pairs); put(net->th_hi, (size_t)net->n_pairs);
  put(obs->obs_times, NO * 4); put(obs->init_state, K * N); put(obs->clamp, K * N); put(obs->obs, K * NO * N);
  return true;
}

}  // namespace

extern "C" {

const char* sa_last_error(void) { return g_err.c_str(); }

int sa_set_allocator(sa_alloc_fn alloc, sa_free_fn release) {
  if ((alloc == nullptr) != (release == nullptr)) return set_err(SA_EINVAL, "give both hooks or neither");
  g_alloc = alloc;
  g_free = release;
  return SA_OK;
}

int sa_geometric_table(double t0, double t_end, int32_t L, int32_t D, uint32_t* out) {
  if (!out || L <= 0 || D <= 0 || !(t0 > 0.0) || !(t_end > 0.0)) return set_err(SA_EINVAL, "bad table arguments");
  for (int l = 0; l < L; ++l) {
    const double temp = (L == 1) ? t0 : t0 * std::pow(t_end / t0, (double)l / (double)(L - 1));
    for (int d = 1; d <= D; ++d) {
      const double v = std::floor(4294967296.0 * std::exp(-(double)d / temp));
      out[(size_t)l * D + (d - 1)] = v >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)v;
    }
  }
  return SA_OK;
}

int sa_clear_plan_cache(void) {
  std::lock_guard<std::mutex> lock(g_plans_mu);
  g_plans.clear();
  return SA_OK;
}

int sa_create(const sa_network* net, const sa_observations* obs, const sa_schedule* sched, sa_handle** out) {
  if (!out) return set_err(SA_EINVAL, "out is NULL");
  *out = nullptr;
  if (!net || !obs || !sched) return set_err(SA_EINVAL, "null argument");
  if (sched->n_chains <= 0 || sched->n_levels <= 0 || sched->steps_per_level <= 0 || sched->dmax <= 0 || !sched->accept)
    return set_err(SA_EINVAL, "bad schedule");
  std::unique_ptr<sa_handle> h(new (std::nothrow) sa_handle());
  if (!h) return set_err(SA_ENOMEM, "host allocation failed");
  std::string err;
  // argument errors are reported before device errors, so validation works without a GPU
  int dev = 0;
  cudaError_t dev_err = cudaGetDevice(&dev);
  if (dev_err == cudaSuccess) dev_err = cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
  int rc = SA_OK;
  {
    const tsa::PlanOptions popt = plan_options(sched->n_chains, h->sm_count);
    const tsa::StaticTuning tune = tsa::StaticTuning::from_env();
    std::string key;
    const bool keyed = plan_key(net, obs, popt, tune, &key);
    std::shared_ptr<const CachedPlans> hit;
    if (keyed) {
      std::lock_guard<std::mutex> lock(g_plans_mu);
      auto it = g_plans.find(key);
      if (it != g_plans.end()) hit = it->second;
    }
    if (hit) {
      h->plan = hit->plan; h->dplan = hit->dplan;
    } else {
      rc = tsa::build_plan(net, obs, true, popt, &h->plan, &err);
      if (rc != SA_OK) return set_err(rc, err);
      tsa::build_dense_plan(net, obs, h->plan, tune.dense_warps, tune.dense_sparse != 0, tune.dense_swizzle != 0, tune.dense_movm != 0, &h->dplan);
      if (keyed) {
        auto entry = std::make_shared<CachedPlans>();
        entry->plan = h->plan; entry->dplan = h->dplan;
        std::lock_guard<std::mutex> lock(g_plans_mu);
        if (g_plans.size() >= kCachedPlans && !g_plans.count(key)) {          // full: the oldest entry makes room
          auto oldest = g_plans.begin();
          for (auto it = g_plans.begin(); it != g_plans.end(); ++it)
            if (it->second->born < oldest->second->born) oldest = it;
          g_plans.erase(oldest);
        }
        entry->born = ++g_plans_clock;
        g_plans[key] = entry;
      }
    }
  }
  if (sched->flags & ~(SA_LEVEL_STATS | SA_CONSTRAINED)) return set_err(SA_EINVAL, "unknown schedule flag");
  if (sched->flags & SA_CONSTRAINED) {
    std::vector<char> has_in(net->n_nodes, 0), has_out(net->n_nodes, 0);
    for (int e = 0; e < net->n_edges; ++e) { has_in[net->edge_dst[e]] = 1; has_out[net->edge_src[e]] = 1; }
    for (int i = 0; i < net->n_nodes; ++i)
      if (!has_in[i] || !has_out[i])
        return set_err(SA_EINVAL, "with constraints on every node needs an in-edge and an out-edge (PAPER.md:187-191)");
  }
  if (dev_err != cudaSuccess) return cuda_err(dev_err, "cudaGetDevice");
  cudaStream_t st = h->stream;
  if ((rc = upload_problem(h->plan, h->pool, &h->P, st))) return rc;
  if (h->plan.team_warps > 0) {
    if ((rc = h->pool.upload(h->plan.lane_off2, &h->d_lane_off2, st))) return rc;
    if ((rc = h->pool.upload(h->plan.lane_meta, &h->d_lane_meta, st))) return rc;
    if ((rc = h->pool.upload(h->plan.lane_clamp, &h->d_lane_clamp, st))) return rc;
    if ((rc = h->pool.upload(h->plan.wloc, &h->d_wloc, st))) return rc;
    if ((rc = h->pool.upload(h->plan.thloc, &h->d_thloc, st))) return rc;
  }
  if (h->dplan.ok) {
    if ((rc = h->pool.upload(h->dplan.frag_slot, &h->d_frag_slot, st))) return rc;
    if ((rc = h->pool.upload(h->dplan.th_entry, &h->d_th_entry, st))) return rc;
    if ((rc = h->pool.upload(h->dplan.meta, &h->d_meta, st))) return rc;
    if ((rc = h->pool.upload(h->dplan.init_frag, &h->d_init_frag, st))) return rc;
    if ((rc = h->pool.upload(h->dplan.obs_word, &h->d_obs_word, st))) return rc;
    if ((rc = h->pool.upload(h->dplan.fix, &h->d_fix, st))) return rc;
    if ((rc = h->pool.upload(h->dplan.wloc, &h->d_dwloc, st))) return rc;
    if ((rc = h->pool.upload(h->dplan.thloc, &h->d_dthloc, st))) return rc;
    h->d_flags = (uint32_t*)h->pool.alloc((size_t)sched->n_chains * 4, st);
    h->d_err = (uint32_t*)h->pool.alloc(4, st);
    if (!h->d_flags || !h->d_err) return set_err(SA_ENOMEM, "device allocation failed (flags)");
    TSA_CUDA(cudaMemsetAsync(h->d_err, 0, 4, st));
  }

  const int R = sched->n_chains;
  tsa::DevChains& C = h->C;
  C.R = R;
  C.cur_w = (int8_t*)h->pool.alloc((size_t)R * h->P.EpadA, st);
  C.best_w = (int8_t*)h->pool.alloc((size_t)R * h->P.EpadA, st);
  C.cur_th = (int8_t*)h->pool.alloc((size_t)R * h->P.NpadA, st);
  C.best_th = (int8_t*)h->pool.alloc((size_t)R * h->P.NpadA, st);
  C.fit_cur = (uint32_t*)h->pool.alloc((size_t)R * 4, st);
  C.fit_best = (uint32_t*)h->pool.alloc((size_t)R * 4, st);
  if (!C.cur_w || !C.best_w || !C.cur_th || !C.best_th || !C.fit_cur || !C.fit_best)
    return set_err(SA_ENOMEM, "device allocation failed (chain store)");

  tsa::DevSched& S = h->S;
  S.key0 = (uint32_t)sched->seed; S.key1 = (uint32_t)(sched->seed >> 32);
  S.chain_id_base = sched->chain_id_base;
  S.n_levels = sched->n_levels; S.dmax = sched->dmax; S.steps_per_level = sched->steps_per_level;
  {
    std::vector<uint32_t> tab(sched->accept, sched->accept + (size_t)sched->n_levels * sched->dmax);
    if ((rc = h->pool.upload(tab, &S.accept, st))) return rc;
  }
  S.level_stats = nullptr;
  S.constrained = (sched->flags & SA_CONSTRAINED) ? 1u : 0u;
  if (S.constrained) {
    // CSR over in- / out-edges in ascending caller edge order, as slots of the canonical weight row
    const int N = net->n_nodes, E = net->n_edges;
    std::vector<int32_t> in_ptr(N + 1, 0), out_ptr(N + 1, 0), in_slot(E), out_slot(E);
    std::vector<uint32_t> nodes(E);
    for (int e = 0; e < E; ++e) { ++in_ptr[net->edge_dst[e] + 1]; ++out_ptr[net->edge_src[e] + 1]; }
    for (int i = 0; i < N; ++i) { in_ptr[i + 1] += in_ptr[i]; out_ptr[i + 1] += out_ptr[i]; }
    std::vector<int32_t> a(in_ptr.begin(), in_ptr.end() - 1), b(out_ptr.begin(), out_ptr.end() - 1);
    for (int e = 0; e < E; ++e) {
      in_slot[a[net->edge_dst[e]]++] = h->plan.slot_of_param[e];
      out_slot[b[net->edge_src[e]]++] = h->plan.slot_of_param[e];
      nodes[e] = (uint32_t)net->edge_src[e] | ((uint32_t)net->edge_dst[e] << 16);
    }
    if ((rc = h->pool.upload(in_ptr, &h->P.con_in_ptr, st))) return rc;
    if ((rc = h->pool.upload(in_slot, &h->P.con_in_slot, st))) return rc;
    if ((rc = h->pool.upload(out_ptr, &h->P.con_out_ptr, st))) return rc;
    if ((rc = h->pool.upload(out_slot, &h->P.con_out_slot, st))) return rc;
    if ((rc = h->pool.upload(nodes, &h->P.edge_nodes, st))) return rc;
    TSA_CUDA(cudaStreamSynchronize(st));                 // the host vectors die with this block
  }
  if (sched->flags & SA_LEVEL_STATS) {
    S.level_stats = (unsigned long long*)h->pool.alloc((size_t)sched->n_levels * 4 * 8, st);
    if (!S.level_stats) return set_err(SA_ENOMEM, "device allocation failed (level statistics)");
    TSA_CUDA(cudaMemsetAsync(S.level_stats, 0, (size_t)sched->n_levels * 4 * 8, st));
  }
  std::memset(&h->Tr, 0, sizeof(h->Tr));

  const size_t sb = tsa::smem_bytes(h->P);
  if (sb > 227 * 1024) return set_err(SA_EINVAL, "chain state does not fit shared memory (N, E too large for this kernel family)");
  h->threads = pick_threads(h->P, R, h->sm_count);
  h->warp_cpb = pick_warp_cpb(h->P, R, h->sm_count);
  TSA_CUDA(tsa::launch_init(h->P, h->C, h->S, h->threads, st));
  ++h->launches;
  TSA_CUDA(cudaStreamSynchronize(st));   // host vectors used by the async uploads die with this frame
  *out = h.release();
  return SA_OK;
}

void sa_destroy(sa_handle* h) {
  if (!h) return;
  cudaStreamSynchronize(h->stream);
  delete h;
}

int sa_set_stream(sa_handle* h, void* cuda_stream) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  h->stream = (cudaStream_t)cuda_stream;
  return SA_OK;
}

int sa_run(sa_handle* h, int64_t steps) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (steps < 0) return set_err(SA_EINVAL, "steps < 0");
  if (steps == 0) return SA_OK;
  if (use_dense(h)) {
    std::string why;
    tsa_dense::Params q = dense_params(h, steps);
    unsigned grid = (unsigned)((h->C.R + h->dk->chains_per_cta - 1) / h->dk->chains_per_cta);
    // More chains than resident slots: split the line of R*steps chain-steps evenly over the slots
    // (DESIGN.md §6 "balanced slots") instead of running ceil(R / slots) uneven waves.
    const int cpb = h->dk->chains_per_cta;
    const int64_t slots = (int64_t)h->dk->blocks_per_sm * h->sm_count * cpb;
    h->last_slot_steps = 0;
    if (slots > 0 && h->C.R > slots && !tsa::tune_env("TSA_DENSE_NO_BALANCE")) {
      const int64_t total = (int64_t)h->C.R * steps;
      q.slot_steps = std::max<int64_t>((total + slots - 1) / slots, steps);
      q.flags = h->d_flags;
      TSA_CUDA(cudaMemsetAsync(h->d_flags, 0, (size_t)h->C.R * 4, h->stream));
      grid = (unsigned)(((total + q.slot_steps - 1) / q.slot_steps + cpb - 1) / cpb);
      h->last_slot_steps = q.slot_steps;
    }
    // A slot that holds the tail of a chain waits for the slot that holds its head, so every slot must
    // be resident at once: the balanced launch is cooperative.  If the device cannot take the whole
    // grid right now (another context holds SMs), fall back to the plain launch, one chain per CTA.
    bool launched = false;
    if (q.slot_steps > 0) {
      launched = tsa::dense_kernel_launch(h->dk, grid, (void*)h->stream, q, &why, true) == 0;
      if (!launched) {
        q.slot_steps = 0; q.flags = nullptr;
        h->last_slot_steps = 0;
        grid = (unsigned)((h->C.R + cpb - 1) / cpb);
      }
    }
    if (!launched && tsa::dense_kernel_launch(h->dk, grid, (void*)h->stream, q, &why) != 0) return set_err(SA_ECUDA, why);
    ++h->launches;
    h->g += (uint64_t)steps;
    return SA_OK;
  }
  if (env_family(h->family) == SA_KERNEL_DENSE)
    return set_err(h->dplan.ok ? SA_ECUDA : SA_EINVAL, "dense kernel unavailable: " + h->dense_why);
  if (use_static(h)) {
    const tsa_static::Params q = static_params(h, steps);
    std::string why;
    if (tsa::static_kernel_launch(h->sk, (unsigned)h->C.R, (void*)h->stream, q, &why) != 0) return set_err(SA_ECUDA, why);
    ++h->launches;
    h->g += (uint64_t)steps;
    return SA_OK;
  }
  if (env_family(h->family) == SA_KERNEL_STATIC)
    return set_err(h->plan.team_warps > 0 ? SA_ECUDA : SA_EINVAL, "static kernel unavailable: " + h->static_why);
  if (h->warp_cpb > 0)
    TSA_CUDA(tsa::launch_run_warp(h->P, h->C, h->S, h->Tr, h->g, steps, h->warp_cpb, h->stream));
  else
    TSA_CUDA(tsa::launch_run(h->P, h->C, h->S, h->Tr, h->g, steps, h->threads, h->stream));
  ++h->launches;
  h->g += (uint64_t)steps;
  return SA_OK;
}

int sa_run_levels(sa_handle* h, int64_t n_levels, int32_t group_size) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (n_levels < 0) return set_err(SA_EINVAL, "n_levels < 0");
  if (group_size < 0) return set_err(SA_EINVAL, "group_size < 0");
  if (h->g % (uint64_t)h->S.steps_per_level != 0)
    return set_err(SA_EINVAL, "sa_run_levels must start at a level boundary (step counter % steps_per_level == 0)");
  const int group = (group_size == 0 || group_size > h->C.R) ? h->C.R : group_size;
  const int n_groups = (h->C.R + group - 1) / group;
  if (!h->d_win) {
    h->d_win = (unsigned long long*)h->pool.alloc((size_t)h->C.R * 8, h->stream);   // enough for any group size
    if (!h->d_win) return set_err(SA_ENOMEM, "device allocation failed (level winners)");
  }
  (void)n_groups;
  for (int64_t l = 0; l < n_levels; ++l) {
    const int rc = sa_run(h, h->S.steps_per_level);
    if (rc != SA_OK) return rc;
    TSA_CUDA(tsa::launch_level_sync(h->P, h->C, group, h->d_win, h->stream));
    h->launches += 2;
  }
  return SA_OK;
}

int sa_level_sync_static(sa_handle* h, int32_t group_size) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (group_size < 0) return set_err(SA_EINVAL, "group_size < 0");
  const int group = (group_size == 0 || group_size > h->C.R) ? h->C.R : group_size;
  const int64_t n_groups = ((int64_t)h->C.R + group - 1) / group;
  if (n_groups > SA_LEVEL_SYNC_STATIC_MAX_GROUPS)
    return set_err(SA_EINVAL, "sa_level_sync_static: " + std::to_string(n_groups) + " groups (" + std::to_string(h->C.R) +
                                  " chains in groups of " + std::to_string(group) + ") exceed the fixed winner table of " +
                                  std::to_string(SA_LEVEL_SYNC_STATIC_MAX_GROUPS) + " groups; use larger groups or sa_run_levels");
  const char* why = nullptr;
  const cudaError_t e = tsa::launch_level_sync_static(h->P, h->C, group, h->stream, &why);
  if (e != cudaSuccess) {
    if (why) return set_err(SA_EINVAL, std::string("sa_level_sync_static: ") + why);
    return cuda_err(e, "sa_level_sync_static");
  }
  h->launches += 2;
  return SA_OK;
}

// after a stream synchronisation: did a kernel of this handle give up a hand-over wait?
static int check_device_error(sa_handle* h) {
  if (!h->d_err) return SA_OK;
  uint32_t e = 0;
  TSA_CUDA(cudaMemcpyAsync(&e, h->d_err, 4, cudaMemcpyDeviceToHost, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  if (e) return set_err(SA_ECUDA, "a balanced-slot hand-over wait timed out; the chains of this handle are invalid");
  return SA_OK;
}

int sa_get_fitness(sa_handle* h, uint32_t* cur_fit, uint32_t* best_fit) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  const size_t bytes = (size_t)h->C.R * 4;
  if (cur_fit) TSA_CUDA(cudaMemcpyAsync(cur_fit, h->C.fit_cur, bytes, cudaMemcpyDeviceToHost, h->stream));
  if (best_fit) TSA_CUDA(cudaMemcpyAsync(best_fit, h->C.fit_best, bytes, cudaMemcpyDeviceToHost, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  return check_device_error(h);
}

int sa_get_level_stats(sa_handle* h, uint64_t* stats) {
  if (!h || !stats) return set_err(SA_EINVAL, "null argument");
  if (!h->S.level_stats) return set_err(SA_EINVAL, "the handle was created without SA_LEVEL_STATS");
  TSA_CUDA(cudaMemcpyAsync(stats, h->S.level_stats, (size_t)h->S.n_levels * 4 * 8, cudaMemcpyDeviceToHost, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  return check_device_error(h);
}

int sa_get_chain(sa_handle* h, int32_t chain, int8_t* cur, uint32_t* cur_fit, int8_t* best, uint32_t* best_fit) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (chain < 0 || chain >= h->C.R) return set_err(SA_EINVAL, "chain out of range");
  const tsa::DevProblem& P = h->P;
  std::vector<int8_t> w(P.EpadA), th(P.NpadA);
  cudaStream_t st = h->stream;
  if (cur) {
    TSA_CUDA(cudaMemcpyAsync(w.data(), h->C.cur_w + (size_t)chain * P.EpadA, P.EpadA, cudaMemcpyDeviceToHost, st));
    TSA_CUDA(cudaMemcpyAsync(th.data(), h->C.cur_th + (size_t)chain * P.NpadA, P.NpadA, cudaMemcpyDeviceToHost, st));
    TSA_CUDA(cudaStreamSynchronize(st));
    h->plan.to_caller(w.data(), th.data(), cur);
  }
  if (best) {
    TSA_CUDA(cudaMemcpyAsync(w.data(), h->C.best_w + (size_t)chain * P.EpadA, P.EpadA, cudaMemcpyDeviceToHost, st));
    TSA_CUDA(cudaMemcpyAsync(th.data(), h->C.best_th + (size_t)chain * P.NpadA, P.NpadA, cudaMemcpyDeviceToHost, st));
    TSA_CUDA(cudaStreamSynchronize(st));
    h->plan.to_caller(w.data(), th.data(), best);
  }
  if (cur_fit) TSA_CUDA(cudaMemcpyAsync(cur_fit, h->C.fit_cur + chain, 4, cudaMemcpyDeviceToHost, st));
  if (best_fit) TSA_CUDA(cudaMemcpyAsync(best_fit, h->C.fit_best + chain, 4, cudaMemcpyDeviceToHost, st));
  TSA_CUDA(cudaStreamSynchronize(st));
  return check_device_error(h);
}

int sa_best(sa_handle* h, uint32_t* fitness, int32_t* chain, int8_t* params) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  DevPool tmp;
  unsigned long long* d = (unsigned long long*)tmp.alloc(8, h->stream);
  if (!d) return set_err(SA_ENOMEM, "device allocation failed");
  TSA_CUDA(tsa::launch_argmin(h->C.fit_best, h->C.R, d, h->stream));
  ++h->launches;
  unsigned long long packed = 0;
  TSA_CUDA(cudaMemcpyAsync(&packed, d, 8, cudaMemcpyDeviceToHost, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  const int32_t c = (int32_t)(packed & 0xFFFFFFFFull);
  if (fitness) *fitness = (uint32_t)(packed >> 32);
  if (chain) *chain = c;
  if (params) return sa_get_chain(h, c, nullptr, nullptr, params, nullptr);
  return SA_OK;
}

static int eval_sets(const tsa::Plan& pl, const tsa::DevProblem& P, const int8_t* params, int64_t n, uint32_t* fitness,
                     uint8_t* dump_dev, int threads, cudaStream_t st, int64_t* launches) {
  const int64_t kBatch = 65536;
  DevPool tmp;
  const int64_t cap = std::min(n, kBatch);
  int8_t* dw = (int8_t*)tmp.alloc((size_t)cap * P.EpadA, st);
  int8_t* dth = (int8_t*)tmp.alloc((size_t)cap * P.NpadA, st);
  uint32_t* dfit = (uint32_t*)tmp.alloc((size_t)cap * 4, st);
  if (!dw || !dth || !dfit) return set_err(SA_ENOMEM, "device allocation failed (eval)");
  std::vector<int8_t> hw((size_t)cap * P.EpadA), hth((size_t)cap * P.NpadA);
  for (int64_t a = 0; a < n; a += kBatch) {
    const int64_t m = std::min(kBatch, n - a);
    for (int64_t r = 0; r < m; ++r)
      pl.to_internal(params + (a + r) * pl.P, hw.data() + r * P.EpadA, hth.data() + r * P.NpadA);
    TSA_CUDA(cudaMemcpyAsync(dw, hw.data(), (size_t)m * P.EpadA, cudaMemcpyHostToDevice, st));
    TSA_CUDA(cudaMemcpyAsync(dth, hth.data(), (size_t)m * P.NpadA, cudaMemcpyHostToDevice, st));
    TSA_CUDA(tsa::launch_eval(P, dw, dth, m, dfit, dump_dev, threads, st));
    if (launches) ++*launches;
    if (fitness) TSA_CUDA(cudaMemcpyAsync(fitness + a, dfit, (size_t)m * 4, cudaMemcpyDeviceToHost, st));
    TSA_CUDA(cudaStreamSynchronize(st));
  }
  return SA_OK;
}

int sa_eval(sa_handle* h, const int8_t* params, int64_t n, uint32_t* fitness) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (!params || !fitness || n < 0) return set_err(SA_EINVAL, "bad sa_eval arguments");
  if (n == 0) return SA_OK;
  if (!tsa::params_valid(h->plan, params, n)) return set_err(SA_EINVAL, "parameter value out of range");
  return eval_sets(h->plan, h->P, params, n, fitness, nullptr, h->threads, h->stream, &h->launches);
}

int sa_simulate(const sa_network* net, const sa_observations* obs, const int8_t* params, uint8_t* states) {
  if (!net || !obs || !params || !states) return set_err(SA_EINVAL, "null argument");
  tsa::Plan pl;
  std::string err;
  int rc = tsa::build_plan(net, obs, false, tsa::PlanOptions::from_env(), &pl, &err);
  if (rc != SA_OK) return set_err(rc, err);
  if (!tsa::params_valid(pl, params, 1)) return set_err(SA_EINVAL, "parameter value out of range");
  int dev = 0, sms = 148;
  TSA_CUDA(cudaGetDevice(&dev));
  TSA_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  DevPool pool;
  tsa::DevProblem P;
  cudaStream_t st = 0;
  if ((rc = upload_problem(pl, pool, &P, st))) return rc;
  if (tsa::smem_bytes(P) > 227 * 1024) return set_err(SA_EINVAL, "chain state does not fit shared memory");
  const size_t out_bytes = (size_t)pl.K * pl.n_obs * pl.N;
  uint8_t* d_out = (uint8_t*)pool.alloc(out_bytes, st);
  if (!d_out) return set_err(SA_ENOMEM, "device allocation failed");
  TSA_CUDA(cudaMemsetAsync(d_out, 0, out_bytes, st));
  rc = eval_sets(pl, P, params, 1, nullptr, d_out, pick_threads(P, 1, sms), st, nullptr);
  if (rc != SA_OK) return rc;
  TSA_CUDA(cudaMemcpy(states, d_out, out_bytes, cudaMemcpyDeviceToHost));
  return SA_OK;
}

int sa_set_trace(sa_handle* h, const int32_t* chains, int32_t n, int64_t max_steps) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  h->trace_pool.clear();
  std::memset(&h->Tr, 0, sizeof(h->Tr));
  h->n_traced = 0;
  h->trace_steps = 0;
  if (n == 0) return SA_OK;
  if (n < 0 || !chains || max_steps <= 0) return set_err(SA_EINVAL, "bad sa_set_trace arguments");
  std::vector<int32_t> row(h->C.R, -1);
  for (int32_t i = 0; i < n; ++i) {
    if (chains[i] < 0 || chains[i] >= h->C.R) return set_err(SA_EINVAL, "traced chain out of range");
    if (row[chains[i]] != -1) return set_err(SA_EINVAL, "traced chain listed twice");
    row[chains[i]] = i;
  }
  const int32_t* d_row = nullptr;
  int rc = h->trace_pool.upload(row, &d_row, h->stream);
  if (rc) return rc;
  // n * max_steps records of 8 bytes: refuse what cannot be a device buffer before the product can wrap
  if (max_steps > tsa::kMaxTraceRecords || (int64_t)n * max_steps > tsa::kMaxTraceRecords) {
    h->trace_pool.clear();
    return set_err(SA_EINVAL, "sa_set_trace: more than 2^34 trace records (128 GiB) asked for");
  }
  const size_t bytes = (size_t)n * (size_t)max_steps * 8;
  uint64_t* rec = (uint64_t*)h->trace_pool.alloc(bytes, h->stream);
  if (!rec) { h->trace_pool.clear(); return set_err(SA_ENOMEM, "device allocation failed (trace)"); }
  TSA_CUDA(cudaMemsetAsync(rec, 0, bytes, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  h->Tr.row_of_chain = d_row;
  h->Tr.records = rec;
  h->Tr.max_steps = max_steps;
  h->Tr.g_start = h->g;
  h->n_traced = n;
  h->trace_steps = max_steps;
  return SA_OK;
}

int sa_get_trace(sa_handle* h, uint64_t* records) {
  if (!h || !records) return set_err(SA_EINVAL, "null argument");
  if (h->n_traced == 0) return set_err(SA_EINVAL, "tracing is off");
  const size_t bytes = (size_t)h->n_traced * (size_t)h->trace_steps * 8;
  TSA_CUDA(cudaMemcpyAsync(records, h->Tr.records, bytes, cudaMemcpyDeviceToHost, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  return SA_OK;
}

int sa_select_kernel(sa_handle* h, int family) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (family != SA_KERNEL_AUTO && family != SA_KERNEL_GENERIC && family != SA_KERNEL_STATIC && family != SA_KERNEL_DENSE)
    return set_err(SA_EINVAL, "unknown kernel family");
  h->family = family;
  return SA_OK;
}

int sa_jit_check(const sa_network* net, const sa_observations* obs, int32_t n_chains, int64_t info[8], char* log,
                 size_t log_bytes) {
  if (!net || !obs || !info || n_chains <= 0) return set_err(SA_EINVAL, "bad sa_jit_check arguments");
  for (int i = 0; i < 8; ++i) info[i] = 0;
  if (log && log_bytes) log[0] = 0;
  auto put_log = [&](const std::string& s) {
    if (log && log_bytes) { std::strncpy(log, s.c_str(), log_bytes - 1); log[log_bytes - 1] = 0; }
  };
  tsa::Plan pl;
  std::string err, dense_note;
  const int rc = tsa::build_plan(net, obs, obs->obs != nullptr, plan_options(n_chains, 148), &pl, &err);
  if (rc != SA_OK) return set_err(rc, err);
  {
    tsa::DensePlan dp;
    tsa::build_dense_plan(net, obs, pl, tsa::StaticTuning::from_env().dense_warps, tsa::StaticTuning::from_env().dense_sparse != 0,
                          tsa::StaticTuning::from_env().dense_swizzle != 0, tsa::StaticTuning::from_env().dense_movm != 0, &dp);
    if (dp.ok) {
      info[6] = 1;
      std::string cubin, clog;
      if (!tsa::dense_kernel_compile(tsa::dense_kernel_defines(pl, dp, tsa::StaticTuning::from_env()), &cubin, &clog)) {
        put_log(clog);
        return set_err(SA_ECUDA, "dense kernel did not compile: " + clog.substr(0, 400));
      }
      info[7] = (int64_t)cubin.size();
      const int blocks = dp.MT * (dp.sparse ? dp.KS / 2 : dp.KS);
      int skipped = 0;
      for (int b = 0; b < blocks && b < 32; ++b) skipped += (int)((dp.skip_blocks >> b) & 1u);
      dense_note = "dense plan: sparse=" + std::to_string(dp.sparse ? 1 : 0) + " immas_per_step=" + std::to_string(blocks - skipped) +
                   " obs_words=" + std::to_string(dp.obs_words);
      put_log(dense_note);
    }
  }
  if (pl.team_warps <= 0) { put_log(dense_note.empty() ? pl.static_why : dense_note + "; static kernel: " + pl.static_why); return SA_OK; }
  info[0] = 1;
  info[1] = pl.team_warps;
  info[2] = pl.n_tiers;
  for (int v : pl.tier_iters) info[3] += v;
  info[5] = (int64_t)(((size_t)3 * pl.state_words * 4 + (size_t)pl.team_warps * 4 + 15) & ~(size_t)15);
  std::string cubin, clog;
  if (!tsa::static_kernel_compile(tsa::static_kernel_defines(pl, tsa::StaticTuning::from_env()), &cubin, &clog)) {
    put_log(clog);
    return set_err(SA_ECUDA, "static kernel did not compile: " + clog.substr(0, 400));
  }
  info[4] = (int64_t)cubin.size();
  return SA_OK;
}

int sa_kernel_source_id(int32_t family, uint64_t* id) {
  if (!id) return set_err(SA_EINVAL, "id is NULL");
  if (!tsa::kernel_source_id(family, id)) return set_err(SA_EINVAL, "family must be SA_KERNEL_STATIC, SA_KERNEL_DENSE or SA_KERNEL_PAPER");
  return SA_OK;
}

int sa_plan_info(const sa_network* net, const sa_observations* obs, int64_t info[16]) {
  if (!net || !obs || !info) return set_err(SA_EINVAL, "null argument");
  tsa::Plan pl;
  std::string err;
  const int rc = tsa::build_plan(net, obs, obs->obs != nullptr, tsa::PlanOptions::from_env(), &pl, &err);
  if (rc != SA_OK) return set_err(rc, err);
  for (int i = 0; i < 16; ++i) info[i] = 0;
  info[0] = 2;
  info[5] = pl.Epad;
  info[8] = pl.n_pass;
  info[9] = pl.total_iters;
  info[10] = pl.n_rows;
  info[11] = pl.n_split_nodes;
  info[12] = pl.CG;
  info[13] = pl.n_entries;
  info[14] = pl.max_in_degree;
  info[15] = pl.fit_const;
  return SA_OK;
}

int sa_get_dense_info(sa_handle* h, int64_t info[8]) {
  if (!h || !info) return set_err(SA_EINVAL, "null argument");
  for (int i = 0; i < 8; ++i) info[i] = 0;
  if (!h->dplan.ok) return SA_OK;
  info[0] = 1;
  info[1] = h->dplan.MT;
  info[2] = h->dplan.KS;
  info[3] = h->dplan.sparse ? 1 : 0;
  info[4] = h->dplan.W;
  info[5] = h->dk ? h->dk->blocks_per_sm : 0;
  info[6] = h->last_slot_steps;
  {
    const int blocks = h->dplan.MT * (h->dplan.sparse ? h->dplan.KS / 2 : h->dplan.KS);
    int skipped = 0;
    for (int b = 0; b < blocks && b < 32; ++b) skipped += (int)((h->dplan.skip_blocks >> b) & 1u);
    info[7] = blocks - skipped;
  }
  return SA_OK;
}

int sa_get_info(sa_handle* h, int64_t info[16]) {
  if (!h || !info) return set_err(SA_EINVAL, "null argument");
  for (int i = 0; i < 16; ++i) info[i] = 0;
  const bool wk = h->warp_cpb > 0;
  info[0] = wk ? 3 : 2;                          // sa_run kernel: 2 = CTA per chain, 3 = warp per chain
  info[1] = wk ? 32 * h->warp_cpb : h->threads;
  info[2] = wk ? h->warp_cpb : 1;
  info[3] = wk ? (int64_t)tsa::warp_kernel_smem(h->P, h->warp_cpb) : (int64_t)tsa::smem_bytes(h->P);
  info[4] = wk ? (h->C.R + h->warp_cpb - 1) / h->warp_cpb : h->C.R;
  if (h->sk && env_family(h->family) != SA_KERNEL_GENERIC) {
    info[0] = 4;                                 // statically scheduled kernel: one team of W warps per chain
    info[1] = h->sk->threads;
    info[2] = 1;
    info[3] = (int64_t)h->sk->smem_bytes;
    info[4] = h->C.R;
    info[14] = h->sk->regs;
  }
  info[15] = h->plan.team_warps;
  if (h->dk && (env_family(h->family) == SA_KERNEL_AUTO || env_family(h->family) == SA_KERNEL_DENSE)) {
    info[0] = 5;                                 // dense kernel: one warp per chain, W in mma.sync A fragments
    info[1] = h->dk->threads;
    info[2] = h->dk->chains_per_cta;
    info[3] = (int64_t)h->dk->smem_bytes;
    info[4] = (h->C.R + h->dk->chains_per_cta - 1) / h->dk->chains_per_cta;
    if (h->last_slot_steps > 0) info[4] = (int64_t)h->dk->blocks_per_sm * h->sm_count;   // balanced slots
    info[14] = h->dk->regs;
    info[15] = h->dplan.W;
  }
  info[5] = h->P.Epad;
  info[6] = h->sm_count;
  info[7] = h->launches;
  info[8] = h->plan.n_pass;
  info[9] = h->plan.total_iters;
  info[10] = h->plan.n_rows;
  info[11] = h->plan.n_split_nodes;
  info[12] = h->plan.CG;
  info[13] = h->plan.n_entries;
  return SA_OK;
}

}  // extern "C"
