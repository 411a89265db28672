// temporary stubs until the tcgen05 kernels land
#include "pf_internal.h"
namespace pf {
struct TmaCtx { int dummy; };
static const char* g_tc_err = "tcgen05 kernels not built";
TmaCtx* tma_ctx_create() { return new TmaCtx(); }
void tma_ctx_destroy(TmaCtx* c) { delete c; }
const char* tc_last_error() { return g_tc_err; }
int launch_gemm_tc(TmaCtx*, const bf16*, int, const bf16*, long, int, int, const Epi&, int, cudaStream_t) { return -1; }
int launch_attn_tc(TmaCtx*, const bf16*, const bf16*, const bf16*, const float*, bf16*, int, int, int, int, int, int, cudaStream_t) { return -1; }
int launch_tri_einsum_tc(TmaCtx*, const bf16*, const bf16*, float*, int, int, int, int, cudaStream_t) { return -1; }
}
