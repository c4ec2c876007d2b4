// Ahead-of-time build of the dense (tensor-pipe) kernel with its default (Mtb-shaped) shape: the
// build check of sa_dense_kernel.cu and the copy cuobjdump shows.  sa_run never launches this copy;
// it launches the one NVRTC compiles for the problem at hand (sa_jit.cpp).
#include "sa_dense_params.h"
#include "sa_dense_kernel.cu"
