// Ahead-of-time build of the statically scheduled kernel with its default (Mtb-shaped) schedule:
// the build check of sa_static_kernel.cu and the copy cuobjdump shows.  sa_run never launches this
// copy; it launches the one NVRTC compiles for the problem at hand (sa_jit.cpp).
#include "sa_static_params.h"
#include "sa_static_kernel.cu"
