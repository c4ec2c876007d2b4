// Run-time compilation of sa_static_kernel.cu for one problem's schedule (NVRTC, loaded with
// dlopen) and its launch through the driver API (entry points from cudaGetDriverEntryPoint, so
// libternary_sa.so links neither libnvrtc nor libcuda and still loads on a box without a GPU).
#pragma once
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "sa_dense_params.h"
#include "sa_dense_plan.h"
#include "sa_plan.h"
#include "sa_static_params.h"
#include "sap_params.h"
#include "sap_plan.h"

namespace tsa {

struct StaticTuning {
  int max_regs = 0;       // static kernel: register budget per thread -> __launch_bounds__ min blocks; 0 = from the edge
                          // slots a thread holds (measured on a B200: < 24 slots 128, 24 .. 43 slots 168 -- Mtb-shaped 70.9
                          // -> 75.9 M chain-steps/s --, more 255 with 12 gathers in flight -- Large 3.50 -> 3.73 M)
  int batch = 0;          // state gathers issued back to back before their IMADs; 0 = 8, or 12 at 255 registers
  int t_unroll = 1;       // unroll factor of the time loop
  int dense_blocks = 0;   // dense kernel: resident chains (CTAs) per SM the register allocation aims at; 0 = 16 (128
                          // registers) with the sparse A operand, 12 (168 registers) with the dense one
  int dense_phases = 1;   // dense kernel: phases of a time step (accumulator tiles live at a time = row tiles / phases)
  int dense_cpb = 0;      // dense kernel: one-warp chains per CTA (1 .. 16, independent of one another); 0 = chosen from
                          // the chain count: a CTA of 4k warps puts k chains on every SM sub-partition
  int dense_swizzle = 1;  // dense kernel: swizzled exchange buffer when it applies
  int dense_spec = 1;     // dense kernel: look-ahead depth (warps per one-warp chain that score consecutive SA steps at once)
  int dense_movm = 0;     // dense kernel: exchange the states through registers (movmatrix) when one warp runs a chain;
                          // measured slower than the shared-memory exchange (143 against 148 M on Mtb-shaped), kept as an option
  int dense_sparse = 1;   // dense kernel: use the 2:4-sparse A operand (mma.sp) when the network allows it
  int dense_warps = 1;    // dense kernel: warps per chain (1, 2 or 4); 1 measured fastest at every R
  int constrained = 0;    // static / dense kernel: build the constrained GetCandidate in (handles created with SA_CONSTRAINED)
  static StaticTuning from_env();
};

// -D options of the kernel for this plan (the cache key of a compiled kernel).
std::vector<std::string> static_kernel_defines(const Plan& plan, const StaticTuning& tune);

// Compile only (no GPU needed).  Returns false with the NVRTC log / reason in *log.
bool static_kernel_compile(const std::vector<std::string>& defines, std::string* cubin, std::string* log);

struct StaticKernel {
  int chains_per_cta = 1;
  int blocks_per_sm = 0;      // resident CTAs per SM at this kernel's registers and shared memory (occupancy query)
  void* module = nullptr;     // CUmodule
  void* function = nullptr;   // CUfunction
  int threads = 0;
  size_t smem_bytes = 0;
  int regs = 0;
};

// Compile (cached per process by the define list), load into the current context, and size the
// dynamic shared memory.  Returns nullptr with the reason in *why.
const StaticKernel* static_kernel_get(const Plan& plan, const StaticTuning& tune, std::string* why);

// cuLaunchKernel on `stream`; returns a CUresult (0 = success) and the error text in *why.
int static_kernel_launch(const StaticKernel* k, unsigned grid, void* stream, const tsa_static::Params& params, std::string* why);

// The dense (tensor-pipe) kernel, sa_dense_kernel.cu: same cache, loader and launch path.
std::vector<std::string> dense_kernel_defines(const Plan& plan, const DensePlan& dp, const StaticTuning& tune);
bool dense_kernel_compile(const std::vector<std::string>& defines, std::string* cubin, std::string* log);
// chains per CTA the kernel will be built for (1 unless the plan has one-warp chains)
int dense_chains_per_cta(const DensePlan& dp, const StaticTuning& tune);
// look-ahead depth the kernel will be built with (1 unless the plan has one-warp chains)
int dense_look_ahead(const DensePlan& dp, const StaticTuning& tune);
const StaticKernel* dense_kernel_get(const Plan& plan, const DensePlan& dp, const StaticTuning& tune, std::string* why);
// cooperative = true: cuLaunchCooperativeKernel (every CTA of the grid resident at once, or the launch fails)
int dense_kernel_launch(const StaticKernel* k, unsigned grid, void* stream, const tsa_dense::Params& params, std::string* why,
                        bool cooperative = false);

// The paper-model kernels, sap_kernel.cu: one module with three entry points (tsp_run, tsp_eval, tsp_init).
struct PaperKernels {
  StaticKernel run, eval, init;
};
std::vector<std::string> paper_kernel_defines(const PaperPlan& plan, int warps_per_cta, int min_blocks);
bool paper_kernel_compile(const std::vector<std::string>& defines, std::string* cubin, std::string* log);
const PaperKernels* paper_kernels_get(const PaperPlan& plan, std::string* why);
int paper_kernel_launch(const StaticKernel* k, unsigned grid, void* stream, const tsa_paper::Params& params, std::string* why);

// FNV-1a-64 of the NVRTC source text this library was built with: which = 2 statically scheduled kernel, 3 dense
// kernel, 4 paper-model kernels.  false for any other value.
bool kernel_source_id(int which, uint64_t* id);

}  // namespace tsa
