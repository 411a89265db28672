// Host side of TMA for all tensor-core kernels: the cuTensorMapEncodeTiled driver entry point (taken at run time through
// cudaGetDriverEntryPoint, so the library needs no libcuda at link time), the thread-local error string of the tcgen05
// launchers, and the two tensor-map encoders (bf16 rank <= 3 with element strides; general rank <= 4 with byte strides).
#include "pf_internal.h"

#include <cudaTypedefs.h>
#include <string>

namespace pf {

// ------------------------------------------------------------------------------------------------
// host: TMA descriptor encoding through the driver entry point (no link-time libcuda dependency)
// ------------------------------------------------------------------------------------------------
struct TmaCtx {
  PFN_cuTensorMapEncodeTiled_v12000 encode = nullptr;
};

static thread_local std::string g_tc_err;
const char* tc_last_error() { return g_tc_err.c_str(); }
void tc_set_error(const std::string& s) { g_tc_err = s; }

TmaCtx* tma_ctx_create() {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
  if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn) {
    g_tc_err = std::string("cudaGetDriverEntryPoint(cuTensorMapEncodeTiled): ") + cudaGetErrorString(e);
    cudaGetLastError();
    return nullptr;
  }
  TmaCtx* c = new TmaCtx();
  c->encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
  return c;
}
void tma_ctx_destroy(TmaCtx* c) { delete c; }

// bf16 tensor of rank 2 or 3, innermost extent d0 contiguous; strides in ELEMENTS for dims 1.. ; box in elements.
int tma_encode_bf16(TmaCtx* ctx, CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                    const uint64_t* strides_elems, const uint32_t* box, int swizzle_bytes) {
  cuuint64_t gd[3];
  cuuint64_t gs[2];
  cuuint32_t bx[3], es[3];
  for (int i = 0; i < rank; ++i) {
    gd[i] = dims[i];
    bx[i] = box[i];
    es[i] = 1;
  }
  for (int i = 0; i + 1 < rank; ++i) gs[i] = strides_elems[i] * 2;
  CUtensorMapSwizzle sw = swizzle_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                          : swizzle_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
                                                : CU_TENSOR_MAP_SWIZZLE_NONE;
  CUresult r = ctx->encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, const_cast<void*>(base), gd, gs, bx,
                           es, CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    g_tc_err = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r);
    return -1;
  }
  return 0;
}

// General form: elem_kind 0 = bf16, 1 = fp16, 2 = fp32; rank <= 4; strides in BYTES for dims 1.. (multiples of 16).
int tma_encode(TmaCtx* ctx, CUtensorMap* out, const void* base, int elem_kind, int rank, const uint64_t* dims,
               const uint64_t* strides_bytes, const uint32_t* box, int swizzle_bytes) {
  cuuint64_t gd[4];
  cuuint64_t gs[3];
  cuuint32_t bx[4], es[4];
  for (int i = 0; i < rank; ++i) {
    gd[i] = dims[i];
    bx[i] = box[i];
    es[i] = 1;
  }
  for (int i = 0; i + 1 < rank; ++i) gs[i] = strides_bytes[i];
  CUtensorMapDataType dt = elem_kind == 2 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                           : elem_kind == 1 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16
                                            : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  CUtensorMapSwizzle sw = swizzle_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                          : swizzle_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
                                                : CU_TENSOR_MAP_SWIZZLE_NONE;
  CUresult r = ctx->encode(out, dt, (cuuint32_t)rank, const_cast<void*>(base), gd, gs, bx, es,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    g_tc_err = "cuTensorMapEncodeTiled (rank " + std::to_string(rank) + ") failed with CUresult " + std::to_string((int)r);
    return -1;
  }
  return 0;
}

}  // namespace pf
