/* ternary_sa.h — C ABI of the B200-native parallel simulated-annealing library for ternary
 * (Low/Medium/High) discrete logic regulatory networks.
 *
 * Method: arxiv 2506.19866, "GPU-accelerated modeling of biological regulatory networks"
 * (PAPER.md under /root/reference): Table 1 is the chain step, §2.1
 * the node update, §2.3 the objective.  The model is the
 * simplified "config model" that BASELINE.json pins (DESIGN.md §1/§3).
 *
 * All pointers in this header are HOST pointers unless a comment says "device".  The caller owns
 * every input array; the library copies what it needs during the call and keeps no caller
 * pointer.  Outputs go to caller-allocated host buffers of the documented size.
 *
 * Every function that returns int returns SA_OK (0) or a negative code; sa_last_error() then
 * holds a message (thread-local).  Nothing throws or exits across this boundary.  A handle is not
 * thread-safe.  There is no CPU fallback: without a CUDA device sa_create fails with SA_ECUDA.
 */
#ifndef TERNARY_SA_H
#define TERNARY_SA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SA_OK      0
#define SA_EINVAL -1   /* bad sizes / values / ordering / NULL pointer */
#define SA_ENOMEM -2   /* host or device allocation failed */
#define SA_ECUDA  -3   /* CUDA runtime error; text in sa_last_error() */

#define SA_UNOBSERVED 255u

typedef struct sa_handle sa_handle;              /* opaque, owned by the library */

/* Candidate structure: nodes and directed candidate edges whose weight may become 0
 * (Fig.1 caption :176).  No self-loops, no duplicate (src,dst). */
typedef struct {
  int32_t n_nodes, n_edges;                      /* N, E */
  const int32_t *edge_src, *edge_dst;            /* [E], in [0,N) */
  int32_t n_pairs;                               /* number of (t_lo,t_hi) pairs, 6 in all configs; <= 16 */
  const int8_t *th_lo, *th_hi;                   /* [n_pairs], th_lo[q] < th_hi[q] */
} sa_network;

/* Experimental conditions and discretised time-course observations (the
 * reference matrix R; here one [n_obs][N] block per condition, 255 = entity not measured). */
typedef struct {
  int32_t n_cond, n_steps, n_obs;                /* K, T, n_obs */
  const int32_t *obs_times;                      /* [n_obs], strictly increasing, in [1,T] */
  const uint8_t *init_state;                     /* [K][N] in {0,1,2}: state at t = 0 (never scored) */
  const uint8_t *clamp;                          /* [K][N] 0/1: a clamped node keeps init_state for all t */
  const uint8_t *obs;                            /* [K][n_obs][N] in {0,1,2} or SA_UNOBSERVED; may be NULL
                                                    for sa_simulate only */
} sa_observations;

/* Annealing schedule (temperature levels, iterations per level). */
typedef struct {
  int32_t  n_chains;                             /* R chains held by this handle */
  uint64_t seed;                                 /* Philox key */
  int32_t  n_levels, steps_per_level, dmax;      /* L, S_l, D */
  const uint32_t *accept;                        /* [L][D]: floor(2^32 * exp(-d/T_l)), d = 1..D */
  uint32_t chain_id_base;                        /* global id of chain 0 (chain-range partition over
                                                    GPUs, reading 25); usually 0 */
  uint32_t flags;                                /* SA_CONSTRAINED | SA_LEVEL_STATS or 0 (sa_create); sap_create takes its flags
                                                    as an argument and ignores this field */
} sa_schedule;

#define SA_CONSTRAINED  1u   /* structural constraints of PAPER.md:186-201 in GetCandidate and at initialisation, in this
                                model's terms (readings C1-C3): every node keeps an in- and an out-edge of
                                non-zero weight and an in-edge of weight +1; a weight proposal chooses among the values
                                that keep them (a null move if none does, trace bit 62); every chain starts from a
                                valid vector.  Needs an in- and an out-edge at every node (SA_EINVAL otherwise).
                                Every kernel family implements it. */
#define SA_LEVEL_STATS 2u   /* count accepted / accepted-worse / new-best moves per temperature level */

/* Parameter vector layout everywhere in this ABI: int8 params[E+N];
 *   params[e]     = weight of edge e (caller's edge order), in {-1,0,+1};
 *   params[E + i] = threshold-pair index of node i, in [0, n_pairs). */

/* Build the device-resident problem, allocate the chain store (SoA int8 in HBM), initialise
 * every chain from Philox domain 1 and evaluate its fitness.
 * Validation (SA_EINVAL): counts > 0, endpoints in range, no self-loop / duplicate edge,
 * th_lo < th_hi, states in {0,1,2}, obs in {0,1,2,255}, obs_times strictly increasing in [1,T],
 * accumulator range: 128 + s - th_lo[q] and 128 + s - th_hi[q] - 1 in [0,255] for all |s| <=
 * 2*max_in_degree (in-degree <= 62 with thresholds in [-3,3]); kernel limits: n_pairs in [2,16],
 * n_steps <= 127, n_obs <= 127, E < 2^24, state entries x words per entry x 4 <= 65535 bytes (about
 * 16 000 nodes at K <= 4, 4 000 at K <= 16).  On failure *out = NULL.
 * The host-side plans of a problem (tens of milliseconds) are kept, keyed by the problem's bytes, for the next
 * sa_create on the same problem (the last eight problems, the oldest making room for a ninth; thread safe). */
int sa_create(const sa_network *net, const sa_observations *obs, const sa_schedule *sched, sa_handle **out);

/* Forget the kept host plans: the next sa_create on any problem plans from scratch (host only; what a
 * measurement of the cold path calls between handles, bench.py's e2e.cold_plan).  Always SA_OK. */
int sa_clear_plan_cache(void);

/* Advance every chain by `steps` SA steps (Table 1 inner loop :130-149; SURVEY.md
 * §8(c)-3): propose, simulate all K conditions for T steps, score, accept/reject, commit.
 * Asynchronous on the handle's stream.  The global step counter persists across calls;
 * level(g) = min(g / steps_per_level, L-1).  sa_run(a); sa_run(b) == sa_run(a+b). */
int sa_run(sa_handle *h, int64_t steps);

/* Chain with the smallest best fitness (ties: smallest chain index).  Any output may be NULL.
 * params receives E+N bytes.  Synchronises the stream.  (min over threads.) */
int sa_best(sa_handle *h, uint32_t *fitness, int32_t *chain, int8_t *params);

void sa_destroy(sa_handle *h);                   /* NULL is a no-op */

/* ---- diagnostics (parity and tests) ---- */

/* Fitness (PAPER.md:104-111 as the 0/1 mismatch count) of n given parameter
 * sets, params [n][E+N] -> fitness [n].  Same simulate/score code as sa_run. */
int sa_eval(sa_handle *h, const int8_t *params, int64_t n, uint32_t *fitness);

/* Simulate one parameter set and return the states at the observation times,
 * states [K][n_obs][N] in {0,1,2} (Simulate() generates pseudo-experimental time
 * series).  Needs no handle; obs->obs is ignored and may be NULL. */
int sa_simulate(const sa_network *net, const sa_observations *obs, const int8_t *params, uint8_t *states);

/* The level structure of PAPER.md Table 1 (:125-155) with the synchronisation done on the device:
 * n_levels times { sa_run(steps_per_level); then, per group of group_size consecutive chains, the
 * member with the smallest best fitness (ties: smallest chain) gives its best vector to every member
 * as best AND current vector, fitness included }.  group_size = 0: all chains form one group (the
 * paper's algorithm); 32 is the group-wise variant of its future work (:321).  The step counter must
 * be at a level boundary.  Asynchronous like sa_run; the synchronisation is not traced. */
int sa_run_levels(sa_handle *h, int64_t n_levels, int32_t group_size);

/* One level synchronisation (the second half of a sa_run_levels level, Table 1 :150-155) for
 * callers that may not allocate device memory once set-up is over.
 *
 * Who that is: sa_run_levels takes its winner table (one u64 per group) from cudaMalloc, or from the
 * sa_set_allocator hooks, the first time a handle calls it.  That is no use to a program that shares
 * the GPU with a framework which has already reserved all of its memory (the request would fail, or
 * make that framework flush its cache), to one whose own arena is frozen after start-up, or to a
 * service loop that cannot afford the device-wide stall cudaMalloc and cudaFree imply.  Such a
 * caller creates its handles up front, then drives Table 1 itself:
 *     for each level { sa_run(h, steps_per_level); sa_level_sync_static(h, group_size); }
 * which leaves the chain store exactly as sa_run_levels(h, 1, group_size) per level would.
 *
 * Inputs and outputs are the handle's chain store (best / current vectors and fitnesses in device
 * memory, allocated by sa_create).  The winner table lives in a fixed array inside the library image:
 * SA_LEVEL_SYNC_STATIC_MAX_GROUPS u64 = 512 KiB of device memory on every GPU that loads the library,
 * held until the process exits.  The call makes no cudaMalloc / cudaFree and uses no allocating
 * library routine; it launches two kernels on the handle's stream and returns without waiting.
 *
 * - ceil(n_chains / group_size) must not exceed SA_LEVEL_SYNC_STATIC_MAX_GROUPS (group_size = 0: one
 *   group, always fits); otherwise SA_EINVAL and nothing is launched.
 * - The device that owns the handle must be current (SA_EINVAL otherwise).
 * - The first call on each device looks up the array's device address (cudaGetSymbolAddress) and
 *   keeps it; make that first call before any stream capture begins.
 * - The array is shared by every handle and every thread of the process and keeps what the last call
 *   left in it.  Nothing in it has to start at zero: a call writes every entry it later reads.  Two
 *   calls whose kernels can overlap on the GPU (different streams, no dependency between them) race
 *   on it; order them with an event or use one stream.
 * - Unlike sa_run_levels the step counter need not sit on a level boundary. */
#define SA_LEVEL_SYNC_STATIC_MAX_GROUPS 65536
int sa_level_sync_static(sa_handle *h, int32_t group_size);

/* One chain's current and best vectors ([E+N] each) and fitnesses.  Any output may be NULL. */
int sa_get_chain(sa_handle *h, int32_t chain, int8_t *cur, uint32_t *cur_fit, int8_t *best, uint32_t *best_fit);

/* Acceptance statistics kept on the device by every kernel family (needs SA_LEVEL_STATS in sched->flags):
 * stats [L][4] = per level of the schedule (the last one absorbing steps past it), summed over all chains
 * since sa_create: steps, accepted moves, accepted moves with delta_cand > delta_cur ("worse solutions
 * that are temporarily accepted"), new bests.  Synchronises the stream. */
int sa_get_level_stats(sa_handle *h, uint64_t *stats);

/* All chains' current / best fitness, [R] each.  Either may be NULL. */
int sa_get_fitness(sa_handle *h, uint32_t *cur_fit, uint32_t *best_fit);

/* Trace the next sa_run calls for `n` chains (local indices): one u64 record per traced chain
 * per step, up to max_steps steps counted from the step counter at the time of this call.
 * Record: bits 0-31 delta_cand, 32-55 parameter index p, 56-59 new value code (weight+1 or pair
 * index), bit 60 accepted, bit 61 new best, bit 62 null move (SA_CONSTRAINED: no value of the weight keeps the
 * constraints; the candidate is the current vector).  n = 0 switches tracing off. */
int sa_set_trace(sa_handle *h, const int32_t *chains, int32_t n, int64_t max_steps);

/* records [n][max_steps] (row order = order given to sa_set_trace); steps not yet run are 0. */
int sa_get_trace(sa_handle *h, uint64_t *records);

/* Host helper, double precision: T_l = t0*(t_end/t0)^(l/(L-1)), T_0 = t0 if
 * L == 1; out[l*D + d-1] = floor(2^32 * exp(-d/T_l)) clamped to 2^32-1. */
int sa_geometric_table(double t0, double t_end, int32_t n_levels, int32_t dmax, uint32_t *out);

/* Which kernel family a handle uses and how it was launched (for bench.py / DESIGN.md):
 * info[0] = sa_run kernel variant (2 = generic, CTA per chain; 3 = generic, warp per chain;
 * 4 = statically scheduled, 5 = dense / tensor pipe), [1] = threads per CTA, [2] = chains per CTA, [3] = dynamic shared
 * memory bytes per CTA, [4] = CTAs in the sa_run grid, [5] = edge slots per chain (padded),
 * [6] = SM count, [7] = kernels launched so far by this handle, [8] = passes per time step,
 * [9] = edge iterations per time step (sum over passes), [10] = rows, [11] = split nodes,
 * [12] = state words per node, [13] = state entries, [14] = registers per thread of the static /
 * dense kernel (0 if not loaded), [15] = warps per chain of the static schedule or the dense team
 * (0 = not applicable).  For the dense kernel [4] is the number of resident slots when the last
 * sa_run used balanced slots (more chains than slots).
 * The variant is decided at the first sa_run; before it, info[0] reports the generic choice. */
int sa_get_info(sa_handle *h, int64_t info[16]);

/* Shape of the dense kernel for this handle: info[0] = 1 if it applies (else all zero), [1] = 16-row
 * tiles MT, [2] = 32-column steps KS, [3] = 1 if the 2:4-sparse A operand is used (mma.sp m16n8k64:
 * MT * KS/2 IMMAs per time step instead of MT * KS), [4] = warps per chain, [5] = resident CTAs per
 * SM of the loaded kernel (0 before the first sa_run), [6] = chain-steps per slot of the last sa_run
 * if it used balanced slots (else 0), [7] = IMMAs per simulated time step (the blocks of the matrix that hold a
 * candidate edge: MT * KS/2 or MT * KS minus the empty ones). */
int sa_get_dense_info(sa_handle *h, int64_t info[8]);

/* Kernel family of sa_run.  AUTO (default): the dense kernel — the node update as an int8 product
 * on the tensor pipe with the chain's weight matrix in mma.sync fragments — when the
 * network has at most 128 nodes and 8 conditions; else the statically scheduled gather kernel —
 * edge schedule, weights and thresholds in registers — when it applies; both are compiled for the
 * problem at hand by NVRTC at the first sa_run.  Else the generic one.  GENERIC: the ahead-of-time
 * compiled table-driven kernels.  STATIC / DENSE: that family only; sa_run fails with SA_EINVAL /
 * SA_ECUDA (reason in sa_last_error) instead of falling back.  All families produce identical
 * results.
 *
 * Environment.  Always read: TSA_KERNEL=generic|static|dense overrides sa_select_kernel (also cta|warp:
 * the generic family with one CTA / one warp per chain); TSA_NVRTC_LIB=<path> names the libnvrtc to load.
 * Read ONLY when TSA_TUNING=1 (measurements and the parity tests, which show that none of them changes
 * a result): TSA_TEAM_WARPS, TSA_TEAM_MIN, TSA_CPB, TSA_NO_SPLIT, TSA_NO_BANKOPT, TSA_NO_STOREOPT,
 * TSA_NO_TIERS, TSA_MAX_SLOTS (generic / static launch shape and host schedule); TSA_JIT_REGS,
 * TSA_JIT_BATCH, TSA_JIT_TUNROLL (static kernel); TSA_DENSE_BLOCKS, TSA_DENSE_PH, TSA_DENSE_CPB,
 * TSA_DENSE_SWZ, TSA_DENSE_SP, TSA_DENSE_MOVM, TSA_DENSE_W, TSA_DENSE_REDERIVE, TSA_DENSE_TUNROLL, TSA_DENSE_CFOLD, TSA_DENSE_SPEC,
 * TSA_DENSE_NO_BALANCE (dense kernel); TSA_PAPER_LPC, TSA_PAPER_WPB, TSA_PAPER_BLOCKS (paper model);
 * TSA_BOUNDS_CHECK=1 compiles the run-time kernels with shared-memory bounds checks that trap (debug);
 * TSA_JIT_DUMP=<dir> keeps every run-time compiled cubin and its option list there (for cuobjdump). */
#define SA_KERNEL_AUTO    0
#define SA_KERNEL_GENERIC 1
#define SA_KERNEL_STATIC  2
#define SA_KERNEL_DENSE   3
int sa_select_kernel(sa_handle *h, int family);

/* Host only: a 64-bit FNV-1a of the run-time compiled source text this library carries for one kernel family
 * (SA_KERNEL_STATIC, SA_KERNEL_DENSE, or SA_KERNEL_PAPER for the sap_* kernels).  profiles/inst_counts.json stores it
 * beside every instruction count taken with ncu; bench.py reports no issue-slot fraction when the loaded library's
 * differs (the count belongs to another kernel text), and a CPU test compares both with the sources in the tree. */
#define SA_KERNEL_PAPER   4
int sa_kernel_source_id(int32_t family, uint64_t *id);

/* Host only (no GPU needed): build the plan of a problem for n_chains chains and compile the
 * statically scheduled kernel for it.  info[0] = 1 if the static kernel applies, [1] = warps per
 * chain, [2] = tiers, [3] = edge slots per thread, [4] = cubin bytes, [5] = shared memory bytes per
 * CTA, [6] = 1 if the dense kernel applies, [7] = its cubin bytes; log (may be NULL) receives the reason / NVRTC log, truncated to log_bytes,
 * or on success a line "dense plan: sparse=S immas_per_step=I obs_words=W" for the dense kernel.  Returns SA_OK
 * also when the kernel does not apply (info[0] = 0); SA_ECUDA when NVRTC is missing or fails. */
int sa_jit_check(const sa_network *net, const sa_observations *obs, int32_t n_chains, int64_t info[8],
                 char *log, size_t log_bytes);

/* Host only (no GPU needed): build the execution plan of a problem and report its shape in the
 * same slots as sa_get_info ([0], [5], [8]-[13]), plus [14] = max in-degree, [15] = number of
 * mismatches contributed by clamped observed entries (constant over all parameter sets).
 * obs->obs may be NULL.  Fails like sa_create on invalid input. */
int sa_plan_info(const sa_network *net, const sa_observations *obs, int64_t info[16]);

/* ==================================================================================================
 * The paper's OWN model: three parameters
 * per edge and per node, the priority update scheme, the gradient-weighted objective, the structural
 * constraints, acceptance statistics per temperature level.  Same chain step (Table 1), same
 * Philox counter layout, same integer accept test and same trace records as above.
 *
 * Parameter vector everywhere below: int8 params[3E+3N] = [w(E), p(E), t(E), u(N), m(N), d(N)]
 * (PAPER.md:106-108), the values themselves: w in {0,1,2} weight, p in {-1,0,1} polarity, t in {1,2}
 * activation threshold of edge e in the caller's edge order (:61-64); u speed in {1..6} (slow node) or
 * {10,11,12} (fast node), m memory in {0,1,2}, d step size in {1,2} of node i (:78-80).
 * ================================================================================================== */

typedef struct sap_handle sap_handle;            /* opaque, owned by the library */

typedef struct {
  int32_t n_nodes, n_edges;                      /* N <= 256, E */
  const int32_t *edge_src, *edge_dst;            /* [E], no duplicate (src,dst); src == dst (autoregulation) allowed */
  const uint8_t *fast;                           /* [N] 1 = speed range {10,11,12}, 0 = {1..6} */
} sap_network;

/* Time courses: K independent courses (the paper has one), each T transitions =
 * T+1 time points including t0. */
typedef struct {
  int32_t n_cond, n_steps;                       /* K, T (T <= 4095) */
  const uint8_t *init_state;                     /* [K][N] in {0,1,2}: state at t0 */
  const uint8_t *ref;                            /* [K][T+1][N] reference matrix R in {0,1,2}, SA_UNOBSERVED = entity
                                                    not measured; may be NULL for sap_simulate only */
} sap_observations;

#define SAP_CONSTRAINED 1u   /* structural constraints of PAPER.md:186-201 in GetCandidate and at initialisation */
#define SAP_LEVEL_STATS 2u   /* count accepted / accepted-worse / new-best moves per temperature level */

/* Build the device-resident problem, allocate the chain store ([R][pitch] int8 in HBM, caller's parameter
 * order), give every chain its initial vector (Philox domain 1; with SAP_CONSTRAINED followed by the
 * repair pass of DESIGN.md reading P6, Philox domain 2, so that every chain starts from a valid
 * vector) and evaluate it.  sched is the same structure as for sa_create; dmax should be
 * at least the largest objective (6 per measured entry) if no worse move is to be rejected outright.
 * Validation (SA_EINVAL): counts > 0, N <= 256, T <= 4095, endpoints in range, no duplicate edge
 * (a self-loop is an edge like any other here, unlike in the config model), fast in {0,1}, states in {0,1,2}, ref in {0,1,2,255}, at most 256 edge slots per lane
 * (in-degrees), and with SAP_CONSTRAINED an in-edge and an out-edge at every node. */
int sap_create(const sap_network *net, const sap_observations *obs, const sa_schedule *sched, uint32_t flags,
               sap_handle **out);

/* Advance every chain by `steps` SA steps (Table 1 :130-149): GetCandidate (uniform
 * parameter index; new value uniform over the parameter's other values, with SAP_CONSTRAINED over
 * those that keep constraints (a) and (b), a null move if there is none), Simulate (priority update
 * scheme §2.2, objective §2.3), integer Metropolis test, commit.  Asynchronous on the handle's stream. */
int sap_run(sap_handle *h, int64_t steps);

/* Table 1 with its level synchronisation on the device, as sa_run_levels. */
int sap_run_levels(sap_handle *h, int64_t n_levels, int32_t group_size);

int sap_best(sap_handle *h, uint32_t *fitness, int32_t *chain, int8_t *params /* [3E+3N] */);
void sap_destroy(sap_handle *h);

/* Objective y = SUM |S - R| (.) (|G| + 1) of n given vectors, params [n][3E+3N]. */
int sap_eval(sap_handle *h, const int8_t *params, int64_t n, uint32_t *fitness);

/* Simulate one vector: states [K][T+1][N], t0 included.  Needs no handle. */
int sap_simulate(const sap_network *net, const sap_observations *obs, const int8_t *params, uint8_t *states);

int sap_get_chain(sap_handle *h, int32_t chain, int8_t *cur, uint32_t *cur_fit, int8_t *best, uint32_t *best_fit);
int sap_get_fitness(sap_handle *h, uint32_t *cur_fit, uint32_t *best_fit);

/* Trace as sa_set_trace / sa_get_trace.  Record: bits 0-31 delta_cand, 32-55 parameter index, 56-59 index
 * of the new value in the parameter's range (increasing order), bit 60 accepted, bit 61 new best, bit 62
 * null move (no value of the parameter keeps the constraints; the candidate is the current vector). */
int sap_set_trace(sap_handle *h, const int32_t *chains, int32_t n, int64_t max_steps);
int sap_get_trace(sap_handle *h, uint64_t *records);

/* Acceptance statistics kept on the device (needs SAP_LEVEL_STATS): stats [L][4] = per level of the
 * schedule (the last one absorbing steps past it), summed over all chains since sap_create: steps,
 * accepted moves, accepted moves with delta_cand > delta_cur ("worse solutions that are temporarily
 * accepted"), new bests.  Synchronises the stream. */
int sap_get_level_stats(sap_handle *h, uint64_t *stats);

/* info[0] = lanes per chain, [1] = node slots per lane, [2] = edge slots per lane, [3] = threads per CTA,
 * [4] = chains per CTA, [5] = dynamic shared memory bytes per CTA, [6] = CTAs of the sap_run grid,
 * [7] = registers per thread of the run kernel, [8] = resident CTAs per SM, [9] = SM count,
 * [10] = kernels launched so far by this handle, [11] = largest objective (6 per measured entry). */
int sap_get_info(sap_handle *h, int64_t info[12]);

int sap_set_stream(sap_handle *h, void *cuda_stream);

/* Host only (no GPU needed): plan + NVRTC compile of the paper-model kernels for this network.
 * info[0] = lanes per chain, [1] = node slots, [2] = edge slots, [3] = cubin bytes. */
int sap_jit_check(const sap_network *net, const sap_observations *obs, int64_t info[4], char *log, size_t log_bytes);

/* ---- plumbing ---- */

/* CUDA stream (cudaStream_t as void*) the handle's kernels and copies run on; default stream 0. */
int sa_set_stream(sa_handle *h, void *cuda_stream);

/* Process-wide device allocator hooks (e.g. PyTorch's caching allocator); NULL, NULL restores
 * cudaMalloc / cudaFree.  alloc returns a DEVICE pointer or NULL.  Set before sa_create. */
typedef void *(*sa_alloc_fn)(size_t bytes, void *cuda_stream);
typedef void (*sa_free_fn)(void *device_ptr);
int sa_set_allocator(sa_alloc_fn alloc, sa_free_fn release);

/* Roofline denominator, measured: issue rates of independent integer instruction streams on
 * the current device.  out[0] = IADD3, [1] = LOP3, [2] = IMAD, [3] = mixed IADD3+IMAD,
 * in warp-instructions per second (whole GPU); out[4] = SM count, out[5] = SM clock in Hz as
 * observed through clock64 over the run.  (SURVEY.md §8(d) "Which roofline".) */
int sa_int32_peak(double out[6]);

/* Second ceiling of the dense kernel, measured: issue rates of the legacy int8 tensor path on the current
 * device, in MMA instructions per second (whole GPU): out[0] = mma.sync m16n8k32 s8 (SASS IMMA.16832.S8),
 * out[1] = mma.sp m16n8k64 s8 (IMMA.SP.16864.S8), out[2] = SM count, out[3] = SM clock in Hz observed. */
int sa_imma_peak(double out[4]);

const char *sa_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TERNARY_SA_H */
