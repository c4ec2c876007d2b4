// Host-side helpers shared by the translation units that implement the C ABI (sa_api.cu, sap_api.cu):
// the thread-local error text, the process-wide device allocator hooks and a pool of device buffers.
// Not part of the ABI and not shared with oracle/.
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "../../include/ternary_sa.h"

namespace tsa {

constexpr int64_t kMaxTraceRecords = (int64_t)1 << 34;   // *_set_trace: chains x steps, 8 bytes each

inline thread_local std::string g_err;
inline sa_alloc_fn g_alloc = nullptr;
inline sa_free_fn g_free = nullptr;

inline int set_err(int code, const std::string& msg) {
  g_err = msg;
  return code;
}

inline int cuda_err(cudaError_t e, const char* what) {
  return set_err(SA_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define TSA_CUDA(call)                                        \
  do {                                                        \
    cudaError_t e__ = (call);                                 \
    if (e__ != cudaSuccess) return tsa::cuda_err(e__, #call); \
  } while (0)

// Device buffers owned by a handle; released through the hooks they were allocated with.
struct DevPool {
  std::vector<void*> ptrs;
  sa_free_fn release = nullptr;
  bool hooked = false;
  ~DevPool() { clear(); }
  void clear() {
    for (void* p : ptrs) {
      if (!p) continue;
      if (hooked) release(p); else cudaFree(p);
    }
    ptrs.clear();
  }
  void* alloc(size_t bytes, cudaStream_t st) {
    if (bytes == 0) bytes = 16;
    void* p = nullptr;
    if (ptrs.empty()) { hooked = (g_alloc && g_free); release = g_free; }
    if (hooked) p = g_alloc(bytes, (void*)st);
    else if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); p = nullptr; }
    if (p) ptrs.push_back(p);
    return p;
  }
  template <typename T>
  int upload(const std::vector<T>& v, const T** out, cudaStream_t st) {
    T* d = (T*)alloc(v.size() * sizeof(T), st);
    if (!d) return set_err(SA_ENOMEM, "device allocation failed");
    if (!v.empty()) TSA_CUDA(cudaMemcpyAsync(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st));
    *out = d;
    return SA_OK;
  }
};

}  // namespace tsa
