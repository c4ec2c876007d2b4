// C ABI of the paper-model half of libternary_sa.so (include/ternary_sa.h, "The paper's OWN model"):
// argument checking, device memory, launches of the NVRTC-compiled kernels of sap_kernel.cu, and the
// small ahead-of-time kernels of the level synchronisation (Table 1 :150-155).
#include <cuda_runtime.h>

#include <cstring>
#include <memory>
#include <new>
#include <string>
#include <vector>

#include "../../include/ternary_sa.h"
#include "sa_host.h"
#include "sa_jit.h"
#include "sa_kernels.h"
#include "sap_params.h"
#include "sap_plan.h"

using tsa::cuda_err;
using tsa::DevPool;
using tsa::set_err;

struct sap_handle {
  tsa::PaperPlan plan;
  tsa_paper::Params q;              // device pointers and the schedule; per-launch fields filled at launch
  const tsa::PaperKernels* k = nullptr;
  DevPool pool, trace_pool;
  cudaStream_t stream = 0;
  uint64_t g = 0;                   // global step counter
  int R = 0, sm_count = 148;
  uint32_t flags = 0;
  int n_levels = 0;
  int64_t launches = 0;
  int32_t n_traced = 0;
  int64_t trace_steps = 0;
  unsigned long long* d_win = nullptr;
};

namespace {

int upload_plan(const tsa::PaperPlan& pl, DevPool& pool, tsa_paper::Params* q, cudaStream_t st) {
  int rc;
  if ((rc = pool.upload(pl.ploc, &q->ploc, st))) return rc;
  if ((rc = pool.upload(pl.slot_src, &q->slot_src, st))) return rc;
  if ((rc = pool.upload(pl.slot_edge, &q->slot_edge, st))) return rc;
  if ((rc = pool.upload(pl.pos_node, &q->pos_node, st))) return rc;
  if ((rc = pool.upload(pl.init_lane, &q->init_lane, st))) return rc;
  if ((rc = pool.upload(pl.cost_lane, &q->cost_lane, st))) return rc;
  if ((rc = pool.upload(pl.fast, &q->fast, st))) return rc;
  if ((rc = pool.upload(pl.in_ptr, &q->in_ptr, st))) return rc;
  if ((rc = pool.upload(pl.in_edge, &q->in_edge, st))) return rc;
  if ((rc = pool.upload(pl.out_ptr, &q->out_ptr, st))) return rc;
  if ((rc = pool.upload(pl.out_edge, &q->out_edge, st))) return rc;
  return SA_OK;
}

unsigned grid_for(const tsa::StaticKernel& k, int64_t n) { return (unsigned)((n + k.chains_per_cta - 1) / k.chains_per_cta); }

// Level synchronisation of PAPER.md Table 1 (:150-155) on the device: per group of `group` consecutive
// chains the smallest d_best (ties: smallest chain) ...
__global__ void sap_group_argmin(const uint32_t* __restrict__ fit, int R, int group, unsigned long long* out) {
  const int first = blockIdx.x * group, last = min(R, first + group);
  unsigned long long best = ~0ull;
  for (int c = first + (int)threadIdx.x; c < last; c += (int)blockDim.x)
    best = min(best, ((unsigned long long)fit[c] << 32) | (unsigned)c);
  __shared__ unsigned long long sm[32];
  for (int o = 16; o > 0; o >>= 1) best = min(best, __shfl_down_sync(0xffffffffu, best, o));
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x < 32) {
    best = threadIdx.x < (blockDim.x + 31) / 32 ? sm[threadIdx.x] : ~0ull;
    for (int o = 16; o > 0; o >>= 1) best = min(best, __shfl_down_sync(0xffffffffu, best, o));
    if (threadIdx.x == 0) out[blockIdx.x] = best;
  }
}

// ... and its best vector becomes every member's best AND current vector (x_current = x_best, :129).
__global__ void sap_level_broadcast(int8_t* cur, int8_t* best, uint32_t* fit_cur, uint32_t* fit_best, int pitch, int group,
                                    const unsigned long long* __restrict__ win) {
  const int c = blockIdx.x;
  const unsigned long long w = win[c / group];
  const int src = (int)(w & 0xFFFFFFFFull);
  const uint32_t f = (uint32_t)(w >> 32);
  const uint32_t* s = (const uint32_t*)(best + (size_t)src * pitch);
  uint32_t* cc = (uint32_t*)(cur + (size_t)c * pitch);
  uint32_t* cb = (uint32_t*)(best + (size_t)c * pitch);
  for (int i = threadIdx.x; i < pitch / 4; i += blockDim.x) { const uint32_t v = s[i]; cc[i] = v; if (c != src) cb[i] = v; }
  if (threadIdx.x == 0) { fit_cur[c] = f; fit_best[c] = f; }
}

}  // namespace

extern "C" {

int sap_create(const sap_network* net, const sap_observations* obs, const sa_schedule* sched, uint32_t flags, sap_handle** out) {
  if (!out) return set_err(SA_EINVAL, "out is NULL");
  *out = nullptr;
  if (!net || !obs || !sched) return set_err(SA_EINVAL, "null argument");
  if (sched->n_chains <= 0 || sched->n_levels <= 0 || sched->steps_per_level <= 0 || sched->dmax <= 0 || !sched->accept)
    return set_err(SA_EINVAL, "bad schedule");
  if (flags & ~(SAP_CONSTRAINED | SAP_LEVEL_STATS)) return set_err(SA_EINVAL, "unknown flag");
  std::unique_ptr<sap_handle> h(new (std::nothrow) sap_handle());
  if (!h) return set_err(SA_ENOMEM, "host allocation failed");
  std::string err;
  int dev = 0;
  cudaError_t dev_err = cudaGetDevice(&dev);
  if (dev_err == cudaSuccess) dev_err = cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
  int rc = tsa::build_paper_plan(net, obs, true, (flags & SAP_CONSTRAINED) != 0, sched->n_chains, h->sm_count, &h->plan, &err);
  if (rc != SA_OK) return set_err(rc, err);          // argument errors first, so validation works without a GPU
  if (dev_err != cudaSuccess) return cuda_err(dev_err, "cudaGetDevice");
  h->flags = flags;
  h->R = sched->n_chains;
  h->n_levels = sched->n_levels;
  std::string why;
  h->k = tsa::paper_kernels_get(h->plan, &why);
  if (!h->k) return set_err(SA_ECUDA, "paper-model kernels unavailable: " + why);
  cudaStream_t st = h->stream;
  tsa_paper::Params& q = h->q;
  std::memset(&q, 0, sizeof(q));
  if ((rc = upload_plan(h->plan, h->pool, &q, st))) return rc;
  const size_t pitch = (size_t)h->plan.NPPAD;
  q.R = h->R;
  q.cur = (int8_t*)h->pool.alloc((size_t)h->R * pitch, st);
  q.best = (int8_t*)h->pool.alloc((size_t)h->R * pitch, st);
  q.fit_cur = (uint32_t*)h->pool.alloc((size_t)h->R * 4, st);
  q.fit_best = (uint32_t*)h->pool.alloc((size_t)h->R * 4, st);
  if (!q.cur || !q.best || !q.fit_cur || !q.fit_best) return set_err(SA_ENOMEM, "device allocation failed (chain store)");
  q.key0 = (uint32_t)sched->seed; q.key1 = (uint32_t)(sched->seed >> 32);
  q.chain_id_base = sched->chain_id_base;
  q.n_levels = sched->n_levels; q.dmax = sched->dmax; q.steps_per_level = sched->steps_per_level;
  {
    std::vector<uint32_t> tab(sched->accept, sched->accept + (size_t)sched->n_levels * sched->dmax);
    if ((rc = h->pool.upload(tab, &q.accept, st))) return rc;
    TSA_CUDA(cudaStreamSynchronize(st));               // `tab` dies with this block
  }
  q.constrained = (flags & SAP_CONSTRAINED) ? 1u : 0u;
  if (flags & SAP_LEVEL_STATS) {
    q.level_stats = (unsigned long long*)h->pool.alloc((size_t)sched->n_levels * 4 * 8, st);
    if (!q.level_stats) return set_err(SA_ENOMEM, "device allocation failed (level statistics)");
    TSA_CUDA(cudaMemsetAsync(q.level_stats, 0, (size_t)sched->n_levels * 4 * 8, st));
  }
  if (tsa::paper_kernel_launch(&h->k->init, grid_for(h->k->init, h->R), (void*)st, q, &why) != 0) return set_err(SA_ECUDA, why);
  ++h->launches;
  TSA_CUDA(cudaStreamSynchronize(st));                 // host vectors used by the async uploads die with this frame
  *out = h.release();
  return SA_OK;
}

void sap_destroy(sap_handle* h) {
  if (!h) return;
  cudaStreamSynchronize(h->stream);
  delete h;
}

int sap_set_stream(sap_handle* h, void* cuda_stream) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  h->stream = (cudaStream_t)cuda_stream;
  return SA_OK;
}

int sap_run(sap_handle* h, int64_t steps) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (steps < 0) return set_err(SA_EINVAL, "steps < 0");
  if (steps == 0) return SA_OK;
  tsa_paper::Params q = h->q;
  q.g0 = h->g; q.steps = steps;
  std::string why;
  if (tsa::paper_kernel_launch(&h->k->run, grid_for(h->k->run, h->R), (void*)h->stream, q, &why) != 0) return set_err(SA_ECUDA, why);
  ++h->launches;
  h->g += (uint64_t)steps;
  return SA_OK;
}

int sap_run_levels(sap_handle* h, int64_t n_levels, int32_t group_size) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (n_levels < 0) return set_err(SA_EINVAL, "n_levels < 0");
  if (group_size < 0) return set_err(SA_EINVAL, "group_size < 0");
  if (h->g % (uint64_t)h->q.steps_per_level != 0)
    return set_err(SA_EINVAL, "sap_run_levels must start at a level boundary (step counter % steps_per_level == 0)");
  const int group = (group_size == 0 || group_size > h->R) ? h->R : group_size;
  const int n_groups = (h->R + group - 1) / group;
  if (!h->d_win) {
    h->d_win = (unsigned long long*)h->pool.alloc((size_t)h->R * 8, h->stream);
    if (!h->d_win) return set_err(SA_ENOMEM, "device allocation failed (level winners)");
  }
  for (int64_t l = 0; l < n_levels; ++l) {
    const int rc = sap_run(h, h->q.steps_per_level);
    if (rc != SA_OK) return rc;
    sap_group_argmin<<<n_groups, group >= 256 ? 256 : 32, 0, h->stream>>>(h->q.fit_best, h->R, group, h->d_win);
    sap_level_broadcast<<<h->R, 128, 0, h->stream>>>(h->q.cur, h->q.best, h->q.fit_cur, h->q.fit_best, h->plan.NPPAD, group, h->d_win);
    TSA_CUDA(cudaGetLastError());
    h->launches += 2;
  }
  return SA_OK;
}

int sap_get_fitness(sap_handle* h, uint32_t* cur_fit, uint32_t* best_fit) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  const size_t bytes = (size_t)h->R * 4;
  if (cur_fit) TSA_CUDA(cudaMemcpyAsync(cur_fit, h->q.fit_cur, bytes, cudaMemcpyDeviceToHost, h->stream));
  if (best_fit) TSA_CUDA(cudaMemcpyAsync(best_fit, h->q.fit_best, bytes, cudaMemcpyDeviceToHost, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  return SA_OK;
}

int sap_get_chain(sap_handle* h, int32_t chain, int8_t* cur, uint32_t* cur_fit, int8_t* best, uint32_t* best_fit) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (chain < 0 || chain >= h->R) return set_err(SA_EINVAL, "chain out of range");
  const size_t pitch = (size_t)h->plan.NPPAD, np = (size_t)h->plan.NP;
  cudaStream_t st = h->stream;
  if (cur) TSA_CUDA(cudaMemcpyAsync(cur, h->q.cur + (size_t)chain * pitch, np, cudaMemcpyDeviceToHost, st));
  if (best) TSA_CUDA(cudaMemcpyAsync(best, h->q.best + (size_t)chain * pitch, np, cudaMemcpyDeviceToHost, st));
  if (cur_fit) TSA_CUDA(cudaMemcpyAsync(cur_fit, h->q.fit_cur + chain, 4, cudaMemcpyDeviceToHost, st));
  if (best_fit) TSA_CUDA(cudaMemcpyAsync(best_fit, h->q.fit_best + chain, 4, cudaMemcpyDeviceToHost, st));
  TSA_CUDA(cudaStreamSynchronize(st));
  return SA_OK;
}

int sap_best(sap_handle* h, uint32_t* fitness, int32_t* chain, int8_t* params) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  DevPool tmp;
  unsigned long long* d = (unsigned long long*)tmp.alloc(8, h->stream);
  if (!d) return set_err(SA_ENOMEM, "device allocation failed");
  TSA_CUDA(tsa::launch_argmin(h->q.fit_best, h->R, d, h->stream));
  ++h->launches;
  unsigned long long packed = 0;
  TSA_CUDA(cudaMemcpyAsync(&packed, d, 8, cudaMemcpyDeviceToHost, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  const int32_t c = (int32_t)(packed & 0xFFFFFFFFull);
  if (fitness) *fitness = (uint32_t)(packed >> 32);
  if (chain) *chain = c;
  if (params) return sap_get_chain(h, c, nullptr, nullptr, params, nullptr);
  return SA_OK;
}

static int eval_vectors(const tsa::PaperPlan& pl, const tsa::PaperKernels* k, tsa_paper::Params q, const int8_t* params, int64_t n,
                        uint32_t* fitness, uint8_t* dump_dev, cudaStream_t st, int64_t* launches) {
  const int64_t kBatch = 1 << 18;
  DevPool tmp;
  const int64_t cap = std::min(n, kBatch);
  int8_t* dp = (int8_t*)tmp.alloc((size_t)cap * pl.NP, st);
  uint32_t* dfit = (uint32_t*)tmp.alloc((size_t)cap * 4, st);
  if (!dp || !dfit) return set_err(SA_ENOMEM, "device allocation failed (eval)");
  for (int64_t a = 0; a < n; a += kBatch) {
    const int64_t m = std::min(kBatch, n - a);
    TSA_CUDA(cudaMemcpyAsync(dp, params + a * pl.NP, (size_t)m * pl.NP, cudaMemcpyHostToDevice, st));
    q.eval_params = dp; q.eval_n = m; q.eval_fit = dfit; q.eval_dump = dump_dev;
    std::string why;
    if (tsa::paper_kernel_launch(&k->eval, grid_for(k->eval, m), (void*)st, q, &why) != 0) return set_err(SA_ECUDA, why);
    if (launches) ++*launches;
    if (fitness) TSA_CUDA(cudaMemcpyAsync(fitness + a, dfit, (size_t)m * 4, cudaMemcpyDeviceToHost, st));
    TSA_CUDA(cudaStreamSynchronize(st));
  }
  return SA_OK;
}

int sap_eval(sap_handle* h, const int8_t* params, int64_t n, uint32_t* fitness) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  if (!params || !fitness || n < 0) return set_err(SA_EINVAL, "bad sap_eval arguments");
  if (n == 0) return SA_OK;
  if (!tsa::paper_params_valid(h->plan, params, n)) return set_err(SA_EINVAL, "parameter value out of range");
  return eval_vectors(h->plan, h->k, h->q, params, n, fitness, nullptr, h->stream, &h->launches);
}

int sap_simulate(const sap_network* net, const sap_observations* obs, const int8_t* params, uint8_t* states) {
  if (!net || !obs || !params || !states) return set_err(SA_EINVAL, "null argument");
  tsa::PaperPlan pl;
  std::string err;
  int rc = tsa::build_paper_plan(net, obs, false, false, 0, 148, &pl, &err);
  if (rc != SA_OK) return set_err(rc, err);
  if (!tsa::paper_params_valid(pl, params, 1)) return set_err(SA_EINVAL, "parameter value out of range");
  std::string why;
  const tsa::PaperKernels* k = tsa::paper_kernels_get(pl, &why);
  if (!k) return set_err(SA_ECUDA, "paper-model kernels unavailable: " + why);
  DevPool pool;
  tsa_paper::Params q;
  std::memset(&q, 0, sizeof(q));
  cudaStream_t st = 0;
  if ((rc = upload_plan(pl, pool, &q, st))) return rc;
  const size_t out_bytes = (size_t)pl.K * (pl.T + 1) * pl.N;
  uint8_t* d_out = (uint8_t*)pool.alloc(out_bytes, st);
  if (!d_out) return set_err(SA_ENOMEM, "device allocation failed");
  TSA_CUDA(cudaMemsetAsync(d_out, 0, out_bytes, st));
  rc = eval_vectors(pl, k, q, params, 1, nullptr, d_out, st, nullptr);
  if (rc != SA_OK) return rc;
  TSA_CUDA(cudaMemcpy(states, d_out, out_bytes, cudaMemcpyDeviceToHost));
  return SA_OK;
}

int sap_set_trace(sap_handle* h, const int32_t* chains, int32_t n, int64_t max_steps) {
  if (!h) return set_err(SA_EINVAL, "null handle");
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  h->trace_pool.clear();
  h->q.trace_row = nullptr; h->q.trace_rec = nullptr; h->q.trace_max = 0; h->q.trace_g0 = 0;
  h->n_traced = 0;
  h->trace_steps = 0;
  if (n == 0) return SA_OK;
  if (n < 0 || !chains || max_steps <= 0) return set_err(SA_EINVAL, "bad sap_set_trace arguments");
  std::vector<int32_t> row(h->R, -1);
  for (int32_t i = 0; i < n; ++i) {
    if (chains[i] < 0 || chains[i] >= h->R) return set_err(SA_EINVAL, "traced chain out of range");
    if (row[chains[i]] != -1) return set_err(SA_EINVAL, "traced chain listed twice");
    row[chains[i]] = i;
  }
  const int32_t* d_row = nullptr;
  int rc = h->trace_pool.upload(row, &d_row, h->stream);
  if (rc) return rc;
  // n * max_steps records of 8 bytes: refuse what cannot be a device buffer before the product can wrap
  if (max_steps > tsa::kMaxTraceRecords || (int64_t)n * max_steps > tsa::kMaxTraceRecords) {
    h->trace_pool.clear();
    return set_err(SA_EINVAL, "sap_set_trace: more than 2^34 trace records (128 GiB) asked for");
  }
  const size_t bytes = (size_t)n * (size_t)max_steps * 8;
  unsigned long long* rec = (unsigned long long*)h->trace_pool.alloc(bytes, h->stream);
  if (!rec) { h->trace_pool.clear(); return set_err(SA_ENOMEM, "device allocation failed (trace)"); }
  TSA_CUDA(cudaMemsetAsync(rec, 0, bytes, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  h->q.trace_row = d_row;
  h->q.trace_rec = rec;
  h->q.trace_max = max_steps;
  h->q.trace_g0 = h->g;
  h->n_traced = n;
  h->trace_steps = max_steps;
  return SA_OK;
}

int sap_get_trace(sap_handle* h, uint64_t* records) {
  if (!h || !records) return set_err(SA_EINVAL, "null argument");
  if (h->n_traced == 0) return set_err(SA_EINVAL, "tracing is off");
  const size_t bytes = (size_t)h->n_traced * (size_t)h->trace_steps * 8;
  TSA_CUDA(cudaMemcpyAsync(records, h->q.trace_rec, bytes, cudaMemcpyDeviceToHost, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  return SA_OK;
}

int sap_get_level_stats(sap_handle* h, uint64_t* stats) {
  if (!h || !stats) return set_err(SA_EINVAL, "null argument");
  if (!h->q.level_stats) return set_err(SA_EINVAL, "the handle was created without SAP_LEVEL_STATS");
  TSA_CUDA(cudaMemcpyAsync(stats, h->q.level_stats, (size_t)h->n_levels * 4 * 8, cudaMemcpyDeviceToHost, h->stream));
  TSA_CUDA(cudaStreamSynchronize(h->stream));
  return SA_OK;
}

int sap_get_info(sap_handle* h, int64_t info[12]) {
  if (!h || !info) return set_err(SA_EINVAL, "null argument");
  info[0] = h->plan.LPC; info[1] = h->plan.NS; info[2] = h->plan.ES;
  info[3] = h->k->run.threads; info[4] = h->k->run.chains_per_cta; info[5] = (int64_t)h->k->run.smem_bytes;
  info[6] = grid_for(h->k->run, h->R); info[7] = h->k->run.regs; info[8] = h->k->run.blocks_per_sm;
  info[9] = h->sm_count; info[10] = h->launches; info[11] = h->plan.max_objective;
  return SA_OK;
}

int sap_jit_check(const sap_network* net, const sap_observations* obs, int64_t info[4], char* log, size_t log_bytes) {
  if (!net || !obs || !info) return set_err(SA_EINVAL, "bad sap_jit_check arguments");
  for (int i = 0; i < 4; ++i) info[i] = 0;
  if (log && log_bytes) log[0] = 0;
  tsa::PaperPlan pl;
  std::string err;
  const int rc = tsa::build_paper_plan(net, obs, obs->ref != nullptr, false, 0, 148, &pl, &err);
  if (rc != SA_OK) return set_err(rc, err);
  info[0] = pl.LPC; info[1] = pl.NS; info[2] = pl.ES;
  std::string cubin, clog;
  if (!tsa::paper_kernel_compile(tsa::paper_kernel_defines(pl, 4, 4), &cubin, &clog)) {
    if (log && log_bytes) { std::strncpy(log, clog.c_str(), log_bytes - 1); log[log_bytes - 1] = 0; }
    return set_err(SA_ECUDA, "paper-model kernels did not compile: " + clog.substr(0, 400));
  }
  info[3] = (int64_t)cubin.size();
  return SA_OK;
}

}  // extern "C"
