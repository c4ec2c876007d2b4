// Launch wrappers of the CUDA kernels (sa_kernels.cu).  Internal to libternary_sa.so.
#pragma once
#include <cuda_runtime.h>

#include "sa_common.h"

namespace tsa {

size_t smem_bytes(const DevProblem& P);

// one CTA of `threads` threads per chain / parameter set
cudaError_t launch_init(const DevProblem& P, const DevChains& C, const DevSched& S, int threads, cudaStream_t st);
cudaError_t launch_run(const DevProblem& P, const DevChains& C, const DevSched& S, const DevTrace& Tr,
                       uint64_t g0, int64_t steps, int threads, cudaStream_t st);
// one chain per warp, chains_per_cta warps per CTA, schedule tables staged in shared memory
size_t warp_kernel_smem(const DevProblem& P, int chains_per_cta);
cudaError_t launch_run_warp(const DevProblem& P, const DevChains& C, const DevSched& S, const DevTrace& Tr,
                            uint64_t g0, int64_t steps, int chains_per_cta, cudaStream_t st);
cudaError_t launch_eval(const DevProblem& P, const int8_t* w, const int8_t* th, int64_t n, uint32_t* fit,
                        uint8_t* dump, int threads, cudaStream_t st);
// PAPER.md Table 1 :150-155: per group of `group` consecutive chains, the member with the smallest
// d_best (ties: smallest chain) gives its best vector to every member as best and current vector.
// win = device scratch, one u64 per group.
cudaError_t launch_level_sync(const DevProblem& P, const DevChains& C, int group, unsigned long long* win, cudaStream_t st);
// The same synchronisation with the winners kept in a fixed device array of this library instead of a buffer the
// caller allocated (sa_level_sync_static in include/ternary_sa.h): nothing is allocated.  Returns cudaErrorInvalidValue
// with *why set when there are more groups than the array holds or the chain store is not on the current device.
cudaError_t launch_level_sync_static(const DevProblem& P, const DevChains& C, int group, cudaStream_t st, const char** why);
// out[0] = (fitness << 32) | chain of the best chain (smallest fitness, then smallest index)
cudaError_t launch_argmin(const uint32_t* fit, int R, unsigned long long* out, cudaStream_t st);

}  // namespace tsa
