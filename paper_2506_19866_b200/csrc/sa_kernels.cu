// CUDA kernels of libternary_sa.so (sm_100a).  Generic "one CTA per chain" family:
// lanes over rows (nodes sorted by in-degree), 4 conditions per 32-bit word in biased byte lanes,
// chain state (weights, thresholds, double-buffered node states) resident in shared memory for
// the whole sa_run.  See DESIGN.md §5-§6.  Shares nothing with oracle/.
#include "sa_kernels.h"

namespace tsa {

// ------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11), this library's own implementation.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&out)[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ------------------------------------------------------------------------------------------
// Shared-memory carve-up of one chain.
// ------------------------------------------------------------------------------------------
struct Smem {
  int8_t* w;        // [EpadA] weights in slot order
  int8_t* th;       // [NpadA] threshold-pair index per row
  char2* ab;        // [NpadA] (-t_lo, -t_hi-1) per row
  uint32_t* S0;     // [state_words] node states, byte lanes; word (N*CG ..) = dummy zero node
  uint32_t* S1;
  uint32_t* red;    // [32] cross-warp reduction scratch
};

__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

__host__ __device__ inline size_t smem_layout(const DevProblem& P, size_t* off_th, size_t* off_ab, size_t* off_s0,
                                              size_t* off_s1, size_t* off_red) {
  size_t o = 0;
  o += P.EpadA;                   *off_th = o;
  o += P.NpadA;                   *off_ab = o;
  o += (size_t)P.NpadA * 2;       *off_s0 = align16(o);
  o = *off_s0 + align16((size_t)P.state_words * 4);   *off_s1 = o;
  o += align16((size_t)P.state_words * 4);            *off_red = o;
  o += 32 * 4;
  return o;
}

size_t smem_bytes(const DevProblem& P) {
  size_t a, b, c, d, e;
  return smem_layout(P, &a, &b, &c, &d, &e);
}

__device__ __forceinline__ Smem carve(const DevProblem& P, unsigned char* base) {
  size_t o_th, o_ab, o_s0, o_s1, o_red;
  smem_layout(P, &o_th, &o_ab, &o_s0, &o_s1, &o_red);
  Smem s;
  s.w = (int8_t*)base;
  s.th = (int8_t*)(base + o_th);
  s.ab = (char2*)(base + o_ab);
  s.S0 = (uint32_t*)(base + o_s0);
  s.S1 = (uint32_t*)(base + o_s1);
  s.red = (uint32_t*)(base + o_red);
  return s;
}

// 16-byte vector copy, n16 = number of int4
__device__ __forceinline__ void copy16(void* dst, const void* src, int n16) {
  for (int i = threadIdx.x; i < n16; i += blockDim.x) ((int4*)dst)[i] = ((const int4*)src)[i];
}

__device__ __forceinline__ void build_ab(const DevProblem& P, const Smem& sm) {
  for (int r = threadIdx.x; r < P.N; r += blockDim.x) {
    const int q = sm.th[r];
    sm.ab[r] = make_char2(P.tha[q], P.thb[q]);
  }
}

__device__ __forceinline__ uint32_t block_sum(uint32_t v, uint32_t* red) {
  v = __reduce_add_sync(0xffffffffu, v);
  if (blockDim.x == 32) return v;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (lane == 0) red[warp] = v;
  __syncthreads();
  uint32_t tot = 0;
  for (int i = 0; i < nw; ++i) tot += red[i];
  __syncthreads();
  return tot;
}

template <int CG> struct Vec;
template <> struct Vec<1> { using T = uint32_t; };
template <> struct Vec<2> { using T = uint2; };
template <> struct Vec<4> { using T = uint4; };

template <int CG>
__device__ __forceinline__ void unpack(const typename Vec<CG>::T& v, uint32_t (&s)[CG]);
template <> __device__ __forceinline__ void unpack<1>(const uint32_t& v, uint32_t (&s)[1]) { s[0] = v; }
template <> __device__ __forceinline__ void unpack<2>(const uint2& v, uint32_t (&s)[2]) { s[0] = v.x; s[1] = v.y; }
template <> __device__ __forceinline__ void unpack<4>(const uint4& v, uint32_t (&s)[4]) { s[0] = v.x; s[1] = v.y; s[2] = v.z; s[3] = v.w; }

template <int CG>
__device__ __forceinline__ typename Vec<CG>::T pack(const uint32_t (&s)[CG]);
template <> __device__ __forceinline__ uint32_t pack<1>(const uint32_t (&s)[1]) { return s[0]; }
template <> __device__ __forceinline__ uint2 pack<2>(const uint32_t (&s)[2]) { return make_uint2(s[0], s[1]); }
template <> __device__ __forceinline__ uint4 pack<4>(const uint32_t (&s)[4]) { return make_uint4(s[0], s[1], s[2], s[3]); }

// ------------------------------------------------------------------------------------------
// a3 + a4: simulate every condition for T synchronous steps from shared-memory weights and
// thresholds, count mismatches at the observation times.
// Returns this thread's partial mismatch count.  All threads of the CTA must call it.
//
// Arithmetic per node word (4 conditions): acc = 0x80808080 + SUM w*s (one IMAD per edge, w a
// sign-extended int8, s in {0,1,2} per byte); because |sum| + |threshold| <= 127 every byte
// stays a valid base-256 digit, so
//   [sum >= t_lo] = bit 7 of (acc - t_lo),  [sum > t_hi] = bit 7 of (acc - t_hi - 1)
// per byte, and the new state is their sum: 0 if sum < t_lo, 2 if sum > t_hi, else 1.
// ------------------------------------------------------------------------------------------
template <int CG, bool DUMP>
__device__ __forceinline__ uint32_t simulate(const DevProblem& P, const Smem& sm, uint8_t* dump) {
  using V = typename Vec<CG>::T;
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nthr >> 5;
  const int NW = P.N * CG;
  uint32_t mism = 0;
  for (int ch = 0; ch < P.n_chunks; ++ch) {
    const uint32_t* initw = P.initw + (size_t)ch * NW;
    const uint32_t* clampm = P.clampm + (size_t)ch * NW;
    for (int x = tid; x < P.state_words; x += nthr) {
      sm.S0[x] = (x < NW) ? __ldg(initw + x) : 0u;
      if (x >= NW) sm.S1[x] = 0u;
    }
    __syncthreads();
    uint32_t* cur = sm.S0;
    uint32_t* nxt = sm.S1;
    for (int t = 1; t <= P.T; ++t) {
      const int oj = P.obs_idx_of_t[t];
      const unsigned char* curb = (const unsigned char*)cur;
      for (int ps = warp; ps < P.n_pass; ps += nwarps) {
        const int base = __ldg(P.pass_base + ps), deg = __ldg(P.pass_deg + ps);
        uint32_t acc[CG];
#pragma unroll
        for (int c = 0; c < CG; ++c) acc[c] = kBias;
        for (int k4 = 0; k4 * 4 < deg; ++k4) {
          const int s0 = base + k4 * 128 + lane * 4;
          const uint32_t wword = *(const uint32_t*)(sm.w + s0);
          const uint2 offs = __ldg((const uint2*)(P.slot_off + s0));
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            if (k4 * 4 + u < deg) {
              const int wv = (int)(int8_t)(wword >> (8 * u));
              const uint32_t o2 = (u < 2) ? offs.x : offs.y;
              const uint32_t off = (u & 1) ? (o2 >> 16) : (o2 & 0xFFFFu);
              uint32_t s[CG];
              unpack<CG>(*(const V*)(curb + off), s);
#pragma unroll
              for (int c = 0; c < CG; ++c) acc[c] += (uint32_t)(wv * (int)s[c]);
            }
          }
        }
        const int row = ps * 32 + lane;
        if (row < P.N) {
          const char2 ab = sm.ab[row];
          uint32_t cm[CG], iv[CG], ns[CG];
          unpack<CG>(__ldg((const V*)(clampm + row * CG)), cm);
          unpack<CG>(__ldg((const V*)(initw + row * CG)), iv);
#pragma unroll
          for (int c = 0; c < CG; ++c) {
            const uint32_t ge = ((acc[c] + (uint32_t)((int)ab.x * (int)kOnes)) >> 7) & kOnes;
            const uint32_t gt = ((acc[c] + (uint32_t)((int)ab.y * (int)kOnes)) >> 7) & kOnes;
            ns[c] = ((ge + gt) & ~cm[c]) | (iv[c] & cm[c]);
          }
          *(V*)(nxt + row * CG) = pack<CG>(ns);
          if (oj >= 0) {
            const size_t ow = (((size_t)ch * P.n_obs + oj) * P.N + row) * CG;
            uint32_t ov[CG], om[CG];
            unpack<CG>(__ldg((const V*)(P.obsw + ow)), ov);
            unpack<CG>(__ldg((const V*)(P.obsm + ow)), om);
#pragma unroll
            for (int c = 0; c < CG; ++c) {
              const uint32_t x = ns[c] ^ ov[c];
              mism += __popc((x | (x >> 1)) & om[c]);
            }
            if (DUMP) {
              const int node = P.node_of_row[row];
#pragma unroll
              for (int c = 0; c < CG; ++c)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                  const int k = ch * 4 * CG + c * 4 + b;
                  if (k < P.K) dump[((size_t)k * P.n_obs + oj) * P.N + node] = (uint8_t)((ns[c] >> (8 * b)) & 0xFFu);
                }
            }
          }
        }
      }
      __syncthreads();
      uint32_t* tmp = cur; cur = nxt; nxt = tmp;
    }
  }
  return mism;
}

// ------------------------------------------------------------------------------------------
// sa_eval / sa_simulate: one CTA per parameter set (internal order).
// ------------------------------------------------------------------------------------------
template <int CG, bool DUMP>
__global__ void eval_kernel(const DevProblem P, const int8_t* __restrict__ w, const int8_t* __restrict__ th,
                            uint32_t* __restrict__ fit, uint8_t* dump) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Smem sm = carve(P, smem_raw);
  const size_t b = blockIdx.x;
  copy16(sm.w, w + b * P.EpadA, P.EpadA / 16);
  copy16(sm.th, th + b * P.NpadA, P.NpadA / 16);
  __syncthreads();
  build_ab(P, sm);
  __syncthreads();
  const uint32_t f = block_sum(simulate<CG, DUMP>(P, sm, dump), sm.red);
  if (threadIdx.x == 0) fit[b] = f;
}

// ------------------------------------------------------------------------------------------
// Chain initialisation: block q of four parameters takes
// Philox(ctr = (q, 0, chain, 1), key = seed); weight = mulhi(y,3)-1, pair = mulhi(y, n_pairs).
// ------------------------------------------------------------------------------------------
template <int CG>
__global__ void init_kernel(const DevProblem P, const DevChains C, const DevSched S) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Smem sm = carve(P, smem_raw);
  const size_t chain = blockIdx.x;
  const uint32_t gchain = S.chain_id_base + (uint32_t)chain;
  for (int i = threadIdx.x; i < P.EpadA; i += blockDim.x) sm.w[i] = 0;
  for (int i = threadIdx.x; i < P.NpadA; i += blockDim.x) sm.th[i] = 0;
  __syncthreads();
  for (int q = threadIdx.x; 4 * q < P.P; q += blockDim.x) {
    uint32_t y[4];
    philox4x32_10((uint32_t)q, 0u, gchain, 1u, S.key0, S.key1, y);
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const int p = 4 * q + m;
      if (p < P.E) sm.w[__ldg(P.slot_of_param + p)] = (int8_t)((int)__umulhi(y[m], 3u) - 1);
      else if (p < P.P) sm.th[__ldg(P.row_of_node + (p - P.E))] = (int8_t)__umulhi(y[m], (uint32_t)P.n_pairs);
    }
  }
  __syncthreads();
  build_ab(P, sm);
  __syncthreads();
  const uint32_t f = block_sum(simulate<CG, false>(P, sm, nullptr), sm.red);
  copy16(C.cur_w + chain * P.EpadA, sm.w, P.EpadA / 16);
  copy16(C.best_w + chain * P.EpadA, sm.w, P.EpadA / 16);
  copy16(C.cur_th + chain * P.NpadA, sm.th, P.NpadA / 16);
  copy16(C.best_th + chain * P.NpadA, sm.th, P.NpadA / 16);
  if (threadIdx.x == 0) { C.fit_cur[chain] = f; C.fit_best[chain] = f; }
}

// ------------------------------------------------------------------------------------------
// sa_run: `steps` chain-steps of one chain, everything on chip (Table 1 :130-149;
// SURVEY.md §8(c)-3).  Thread 0 applies / reverts the one-byte mutation; every thread computes
// the Philox block and the accept decision redundantly so no broadcast is needed.
// ------------------------------------------------------------------------------------------
template <int CG>
__global__ void run_kernel(const DevProblem P, const DevChains C, const DevSched S, const DevTrace Tr,
                           const uint64_t g0, const int64_t steps) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Smem sm = carve(P, smem_raw);
  const size_t chain = blockIdx.x;
  const uint32_t gchain = S.chain_id_base + (uint32_t)chain;
  copy16(sm.w, C.cur_w + chain * P.EpadA, P.EpadA / 16);
  copy16(sm.th, C.cur_th + chain * P.NpadA, P.NpadA / 16);
  __syncthreads();
  build_ab(P, sm);
  uint32_t fcur = C.fit_cur[chain], fbest = C.fit_best[chain];
  const int trow = Tr.row_of_chain ? Tr.row_of_chain[chain] : -1;

  uint64_t level = g0 / (uint64_t)S.steps_per_level;
  int64_t left_in_level = S.steps_per_level - (int64_t)(g0 % (uint64_t)S.steps_per_level);
  __syncthreads();

  for (int64_t it = 0; it < steps; ++it) {
    const uint64_t g = g0 + (uint64_t)it;
    uint32_t x[4];
    philox4x32_10((uint32_t)g, (uint32_t)(g >> 32), gchain, 0u, S.key0, S.key1, x);
    const int p = (int)__umulhi(x[0], (uint32_t)P.P);
    // a1/a2: thread 0 proposes and applies; (loc, old) let it revert
    int loc = 0, oldv = 0, newv = 0;
    if (threadIdx.x == 0) {
      if (p < P.E) {
        loc = __ldg(P.slot_of_param + p);
        oldv = sm.w[loc];
        newv = (oldv + 2 + (int)__umulhi(x[1], 2u)) % 3 - 1;          // (code + 1 + r) mod 3 - 1, code = old + 1
        sm.w[loc] = (int8_t)newv;
      } else {
        loc = __ldg(P.row_of_node + (p - P.E));
        oldv = sm.th[loc];
        newv = (oldv + 1 + (int)__umulhi(x[1], (uint32_t)(P.n_pairs - 1))) % P.n_pairs;
        sm.th[loc] = (int8_t)newv;
        sm.ab[loc] = make_char2(P.tha[newv], P.thb[newv]);
      }
    }
    __syncthreads();
    // a3/a4
    const uint32_t fcand = block_sum(simulate<CG, false>(P, sm, nullptr), sm.red);
    // a5
    const uint64_t lv = level < (uint64_t)(S.n_levels - 1) ? level : (uint64_t)(S.n_levels - 1);
    const int64_t d = (int64_t)fcand - (int64_t)fcur;
    bool acc = d <= 0;
    if (!acc && d <= (int64_t)S.dmax) acc = x[2] < __ldg(S.accept + lv * (uint64_t)S.dmax + (uint64_t)(d - 1));
    bool new_best = false;
    // a6
    if (acc) {
      fcur = fcand;
      if (fcand < fbest) {
        fbest = fcand;
        new_best = true;
        copy16(C.best_w + chain * P.EpadA, sm.w, P.EpadA / 16);
        copy16(C.best_th + chain * P.NpadA, sm.th, P.NpadA / 16);
        __syncthreads();            // the copy reads sm.w/th; the next mutation writes them
      }
    } else if (threadIdx.x == 0) {
      if (p < P.E) sm.w[loc] = (int8_t)oldv;
      else { sm.th[loc] = (int8_t)oldv; sm.ab[loc] = make_char2(P.tha[oldv], P.thb[oldv]); }
    }
    if (trow >= 0 && threadIdx.x == 0) {
      const uint64_t idx = g - Tr.g_start;
      if (g >= Tr.g_start && idx < (uint64_t)Tr.max_steps) {
        const uint64_t code = (p < P.E) ? (uint64_t)(newv + 1) : (uint64_t)newv;
        Tr.records[(size_t)trow * Tr.max_steps + idx] =
            (uint64_t)fcand | ((uint64_t)p << 32) | (code << 56) | ((uint64_t)(acc ? 1 : 0) << 60) |
            ((uint64_t)(new_best ? 1 : 0) << 61);
      }
    }
    if (--left_in_level == 0) { ++level; left_in_level = S.steps_per_level; }
  }
  __syncthreads();
  // a7
  copy16(C.cur_w + chain * P.EpadA, sm.w, P.EpadA / 16);
  copy16(C.cur_th + chain * P.NpadA, sm.th, P.NpadA / 16);
  if (threadIdx.x == 0) { C.fit_cur[chain] = fcur; C.fit_best[chain] = fbest; }
}

__global__ void argmin_kernel(const uint32_t* __restrict__ fit, int R, unsigned long long* out) {
  __shared__ unsigned long long red[32];
  unsigned long long best = ~0ull;
  for (int i = threadIdx.x; i < R; i += blockDim.x) {
    const unsigned long long v = ((unsigned long long)fit[i] << 32) | (unsigned)i;
    best = v < best ? v : best;
  }
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long v = __shfl_xor_sync(0xffffffffu, best, o);
    best = v < best ? v : best;
  }
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < (int)(blockDim.x >> 5); ++i) best = red[i] < best ? red[i] : best;
    out[0] = best;
  }
}

// ------------------------------------------------------------------------------------------
// launch wrappers
// ------------------------------------------------------------------------------------------
template <typename K>
static cudaError_t set_smem(K kernel, size_t bytes) {
  if (bytes <= 48 * 1024) return cudaSuccess;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

#define TSA_DISPATCH_CG(P, ...)                            \
  switch ((P).CG) {                                        \
    case 1: { constexpr int CG = 1; __VA_ARGS__; } break;  \
    case 2: { constexpr int CG = 2; __VA_ARGS__; } break;  \
    default: { constexpr int CG = 4; __VA_ARGS__; } break; \
  }

cudaError_t launch_init(const DevProblem& P, const DevChains& C, const DevSched& S, int threads, cudaStream_t st) {
  const size_t sb = smem_bytes(P);
  cudaError_t e = cudaSuccess;
  TSA_DISPATCH_CG(P, {
    e = set_smem(init_kernel<CG>, sb);
    if (e == cudaSuccess) init_kernel<CG><<<C.R, threads, sb, st>>>(P, C, S);
  });
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_run(const DevProblem& P, const DevChains& C, const DevSched& S, const DevTrace& Tr,
                       uint64_t g0, int64_t steps, int threads, cudaStream_t st) {
  const size_t sb = smem_bytes(P);
  cudaError_t e = cudaSuccess;
  TSA_DISPATCH_CG(P, {
    e = set_smem(run_kernel<CG>, sb);
    if (e == cudaSuccess) run_kernel<CG><<<C.R, threads, sb, st>>>(P, C, S, Tr, g0, steps);
  });
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_eval(const DevProblem& P, const int8_t* w, const int8_t* th, int64_t n, uint32_t* fit,
                        uint8_t* dump, int threads, cudaStream_t st) {
  const size_t sb = smem_bytes(P);
  cudaError_t e = cudaSuccess;
  TSA_DISPATCH_CG(P, {
    if (dump) {
      e = set_smem(eval_kernel<CG, true>, sb);
      if (e == cudaSuccess) eval_kernel<CG, true><<<(unsigned)n, threads, sb, st>>>(P, w, th, fit, dump);
    } else {
      e = set_smem(eval_kernel<CG, false>, sb);
      if (e == cudaSuccess) eval_kernel<CG, false><<<(unsigned)n, threads, sb, st>>>(P, w, th, fit, dump);
    }
  });
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_argmin(const uint32_t* fit, int R, unsigned long long* out, cudaStream_t st) {
  argmin_kernel<<<1, 1024, 0, st>>>(fit, R, out);
  return cudaGetLastError();
}

}  // namespace tsa
