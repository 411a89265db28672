// temporary stubs until the remaining tcgen05 kernels land (the driver keeps these sub-steps on the SIMT kernels)
#include "pf_internal.h"
namespace pf {
int launch_tri_einsum_tc(TmaCtx*, const bf16*, const bf16*, float*, int, int, int, int, cudaStream_t) {
  tc_set_error("triangle einsum tcgen05 kernel not built");
  return -1;
}
}
