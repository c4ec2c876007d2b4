// Tuning knobs.  Launch geometry and host-schedule options (TSA_DENSE_*, TSA_JIT_*, TSA_TEAM_*, TSA_NO_*,
// TSA_CPB, TSA_MAX_SLOTS, TSA_PAPER_*) are read from the environment ONLY when TSA_TUNING=1 is set: they
// exist for the parity tests (every setting must give the same results) and for measurements, are
// listed in include/ternary_sa.h, and none of them changes a result.  TSA_KERNEL and TSA_NVRTC_LIB
// are always read.
#pragma once
#include <cstdlib>

namespace tsa {

inline const char* tune_env(const char* name) {
  const char* on = std::getenv("TSA_TUNING");
  if (!on || on[0] != '1') return nullptr;
  return std::getenv(name);
}

}  // namespace tsa
