// Ahead-of-time build of the paper-model kernels with their default (paper_mtb) shape: the build check
// of sap_kernel.cu and the copy cuobjdump shows.  sap_run never launches this copy; it launches the
// one NVRTC compiles for the network at hand (sa_jit.cpp).
#include "sap_params.h"
#include "sap_kernel.cu"
