// Projection GEMM on tcgen05 tensor cores (sm_100a):  acc[r, n] = sum_k A[r, k] Wt[n, k]
//   A  bf16 [R, K] row-major (K contiguous), Wt bf16 [Nw, K] (K contiguous)  ->  fp32 accumulator in TMEM
//   -> fused epilogue (struct Epi: bias / scale / sigmoid / ReLU / masks / gating / residual add / layout changes).
// Structure: one 128 x BN output tile per CTA, BLOCK_K = 64 (one 128-byte swizzle atom), TMA -> shared memory ring
// (mbarrier full/empty) -> one elected thread issues tcgen05.mma (M=128, N=BN, K=16) -> tcgen05.commit ->
// four epilogue warps read their TMEM lane quarter with tcgen05.ld and write the result.  Two CTAs are resident
// per SM (<= 96 KB of shared memory, <= 256 TMEM columns each) so one CTA's epilogue overlaps the other's main loop.
// Used by every Linear of SURVEY.md App. A on the PF_BF16 path (north_star: "LayerNorm fused into the ... projections",
// "transitions fused with their residual adds" — here: projections with fused epilogues; LN is a separate kernel).
#include "pf_internal.h"
#include "pf_device.cuh"
#include "pf_tc.cuh"

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

// ------------------------------------------------------------------------------------------------
// epilogue: 32 consecutive output columns [n0, n0+32) of one row, values in registers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float fast_sigmoid(float x) { return __fdividef(1.0f, 1.0f + __expf(-x)); }

__device__ __forceinline__ void epilogue_chunk32(const Epi& e, const RowInfo& ri, long r, int n0, int Nout,
                                                 const uint32_t (&acc)[32], const uint32_t (&acc2)[32]) {
  if (e.kind == EPI_STORE) {
    float v[32];
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      int n = n0 + j;
      float x = __uint_as_float(acc[j]);
      if (n < e.scale_cols) x *= e.scale;
      if (e.bias) x += __ldg(e.bias + min(n, Nout - 1));
      if (n >= e.act_lo && n < e.act_hi) x = (e.act == ACT_SIGMOID) ? fast_sigmoid(x) : fmaxf(x, 0.f);
      v[j] = x * ri.mask;
    }
    if (n0 + 32 <= e.vt_from && n0 + 32 <= Nout) {
      bf16* dst = reinterpret_cast<bf16*>(e.out) + r * e.ldo + n0;
#pragma unroll
      for (int j = 0; j < 32; j += 8) {
        uint4 u;
        __nv_bfloat162 p0 = __floats2bfloat162_rn(v[j], v[j + 1]), p1 = __floats2bfloat162_rn(v[j + 2], v[j + 3]);
        __nv_bfloat162 p2 = __floats2bfloat162_rn(v[j + 4], v[j + 5]), p3 = __floats2bfloat162_rn(v[j + 6], v[j + 7]);
        u.x = *reinterpret_cast<uint32_t*>(&p0);
        u.y = *reinterpret_cast<uint32_t*>(&p1);
        u.z = *reinterpret_cast<uint32_t*>(&p2);
        u.w = *reinterpret_cast<uint32_t*>(&p3);
        *reinterpret_cast<uint4*>(dst + j) = u;
      }
    } else {
      long br = r / e.geom.D2;
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        int n = n0 + j;
        if (n >= Nout) break;
        if (n < e.vt_from)
          reinterpret_cast<bf16*>(e.out)[r * e.ldo + n] = __float2bfloat16_rn(v[j]);
        else   // transposed columns: consecutive rows (lanes) are contiguous
          reinterpret_cast<bf16*>(e.vt)[(br * (Nout - e.vt_from) + (n - e.vt_from)) * e.Lpad + ri.y] =
              __float2bfloat16_rn(v[j]);
      }
    }
  } else if (e.kind == EPI_GATED_CM) {
    bf16* base = reinterpret_cast<bf16*>(e.out) + (((long)ri.b * Nout) * e.geom.D1 + ri.x) * e.Lpad + ri.y;
    long cstride = (long)e.geom.D1 * e.Lpad;
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      int n = n0 + j;
      if (n >= Nout) break;
      float p = __uint_as_float(acc[j]) + __ldg(e.bias + n);
      float g = fast_sigmoid(__uint_as_float(acc2[j]) + __ldg(e.bias2 + n));
      base[n * cstride] = __float2bfloat16_rn(ri.mask * g * p);
    }
  } else if (e.kind == EPI_RESID) {
    float* dst = e.resid + ri.dst * e.ldr + n0;
    const bf16* gp = e.gate ? reinterpret_cast<const bf16*>(e.gate) + r * e.ldg + n0 : nullptr;
#pragma unroll
    for (int j = 0; j < 32; j += 4) {
      if (n0 + j >= Nout) break;
      float4 o = *reinterpret_cast<float4*>(dst + j);
      float x0 = __uint_as_float(acc[j]) + __ldg(e.bias + n0 + j);
      float x1 = __uint_as_float(acc[j + 1]) + __ldg(e.bias + n0 + j + 1);
      float x2 = __uint_as_float(acc[j + 2]) + __ldg(e.bias + n0 + j + 2);
      float x3 = __uint_as_float(acc[j + 3]) + __ldg(e.bias + n0 + j + 3);
      if (gp) {
        uint2 gu = *reinterpret_cast<const uint2*>(gp + j);
        __nv_bfloat162 g01 = *reinterpret_cast<__nv_bfloat162*>(&gu.x), g23 = *reinterpret_cast<__nv_bfloat162*>(&gu.y);
        x0 *= __low2float(g01);
        x1 *= __high2float(g01);
        x2 *= __low2float(g23);
        x3 *= __high2float(g23);
      }
      o.x += x0;
      o.y += x1;
      o.z += x2;
      o.w += x3;
      *reinterpret_cast<float4*>(dst + j) = o;
    }
  } else {   // EPI_HEADS
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      int n = n0 + j;
      if (n >= Nout) break;
      reinterpret_cast<bf16*>(e.out)[(((long)ri.b * Nout + n) * e.geom.D1 + ri.x) * e.Lpad + ri.y] =
          __float2bfloat16_rn(__uint_as_float(acc[j]) * e.scale);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// kernel
// ------------------------------------------------------------------------------------------------
constexpr int GEMM_BM = 128;
constexpr int GEMM_BK = 64;
constexpr int GEMM_THREADS = 192;

template <int BN, int STAGES>
struct GemmSmem {
  static constexpr int A_BYTES = GEMM_BM * GEMM_BK * 2;
  static constexpr int B_BYTES = BN * GEMM_BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int BAR_OFFSET = STAGES * STAGE_BYTES;
  static constexpr int TOTAL = BAR_OFFSET + 256 + 1024;   // barriers + tmem slot + alignment slack
};

template <int BN, int STAGES, bool DUAL>
__global__ void __launch_bounds__(GEMM_THREADS, 2)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, long R, int K, int Nout,
               Epi epi) {
  using L = GemmSmem<BN, STAGES>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = tc::align_smem_1024(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + L::BAR_OFFSET);
  uint64_t* empty = full + STAGES;
  uint64_t* tmem_full = empty + STAGES;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tmem_full + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m0 = blockIdx.x * GEMM_BM;
  const int nw0 = blockIdx.y * BN;   // first weight row of this tile
  const int num_kb = K / GEMM_BK;

  if (warp == 0 && lane == 0) {
    tc::prefetch_tmap(&tmA);
    tc::prefetch_tmap(&tmB);
    for (int s = 0; s < STAGES; ++s) {
      tc::mbar_init(&full[s], 1);
      tc::mbar_init(&empty[s], 1);
    }
    tc::mbar_init(tmem_full, 1);
    tc::fence_barrier_init();
  }
  if (warp == 1) tc::tmem_alloc<BN>(tmem_slot);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (tc::elect_one()) {
      for (int kb = 0; kb < num_kb; ++kb) {
        int s = kb % STAGES;
        uint32_t ph = (kb / STAGES) & 1;
        tc::mbar_wait(&empty[s], ph ^ 1);
        tc::mbar_arrive_expect_tx(&full[s], L::STAGE_BYTES);
        uint8_t* a = smem + s * L::STAGE_BYTES;
        tc::tma_load_2d(a, &tmA, &full[s], kb * GEMM_BK, m0);
        tc::tma_load_2d(a + L::A_BYTES, &tmB, &full[s], kb * GEMM_BK, nw0);
      }
    }
  } else if (warp == 1) {
    if (tc::elect_one()) {
      constexpr uint32_t idesc = tc::idesc_bf16_f32(GEMM_BM, BN);
      for (int kb = 0; kb < num_kb; ++kb) {
        int s = kb % STAGES;
        uint32_t ph = (kb / STAGES) & 1;
        tc::mbar_wait(&full[s], ph);
        tc::tc_fence_after();
        uint32_t a_addr = tc::smem_u32(smem + s * L::STAGE_BYTES);
        uint64_t a_desc = tc::smem_desc_kmajor<128>(a_addr);
        uint64_t b_desc = tc::smem_desc_kmajor<128>(a_addr + L::A_BYTES);
#pragma unroll
        for (int k = 0; k < GEMM_BK / 16; ++k)   // 16 bf16 = 32 bytes = 2 descriptor address units per MMA K-step
          tc::mma_bf16(tmem_base, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | k) != 0);
        tc::mma_commit(&empty[s]);
      }
      tc::mma_commit(tmem_full);
    }
  } else {
    const int quarter = warp & 3;   // TMEM lane quarter this warp may read
    const int row = quarter * 32 + lane;
    const long r = (long)m0 + row;
    const bool valid = r < R;
    RowInfo ri;
    ri.b = ri.x = ri.y = 0;
    ri.mask = 0.f;
    ri.dst = 0;
    if (valid) ri = row_info(r, epi);
    tc::mbar_wait(tmem_full, 0);
    tc::tc_fence_after();
    const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
    constexpr int NCOLS = DUAL ? BN / 2 : BN;
#pragma unroll 1
    for (int c0 = 0; c0 < NCOLS; c0 += 32) {
      int n0 = (DUAL ? 0 : nw0) + c0;
      if (n0 >= Nout) break;
      uint32_t v[32], v2[32];
      tc::tmem_ld32(lane_addr + c0, v);
      if (DUAL) tc::tmem_ld32(lane_addr + NCOLS + c0, v2);
      tc::tmem_ld_wait();
      if (valid) epilogue_chunk32(epi, ri, r, n0, Nout, v, DUAL ? v2 : v);
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 1) tc::tmem_dealloc<BN>(tmem_base);
}

template <int BN, int STAGES, bool DUAL>
static int launch_variant(const CUtensorMap& tmA, const CUtensorMap& tmB, long R, int K, int Nout, int Nw, const Epi& epi,
                          cudaStream_t st) {
  using L = GemmSmem<BN, STAGES>;
  auto kern = gemm_tc_kernel<BN, STAGES, DUAL>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, L::TOTAL);
    if (e != cudaSuccess) {
      tc_set_error(std::string("cudaFuncSetAttribute(gemm_tc): ") + cudaGetErrorString(e));
      return -1;
    }
    configured = true;
  }
  dim3 grid((unsigned)((R + GEMM_BM - 1) / GEMM_BM), (unsigned)((Nw + BN - 1) / BN));
  kern<<<grid, GEMM_THREADS, L::TOTAL, st>>>(tmA, tmB, R, K, Nout, epi);
  return 0;
}

int launch_gemm_tc(TmaCtx* ctx, const bf16* A, int lda, const bf16* Wt, long R, int K, int Nout, const Epi& epi,
                   int num_sms, cudaStream_t st) {
  (void)num_sms;
  if (K % GEMM_BK != 0 || lda % 8 != 0) {
    tc_set_error("gemm_tc: K must be a multiple of 64 and lda a multiple of 8");
    return -1;
  }
  const bool dual = epi.kind == EPI_GATED_CM;
  const int Nw = dual ? 2 * Nout : Nout;
  if (dual && Nout != 128) {
    tc_set_error("gemm_tc: gated projection expects 128 output channels");
    return -1;
  }
  const int BN = dual ? 256 : (Nw >= 256 ? 256 : (Nw > 64 ? 128 : 64));
  CUtensorMap tmA, tmB;
  uint64_t dA[2] = {(uint64_t)K, (uint64_t)R}, sA[1] = {(uint64_t)lda};
  uint32_t bA[2] = {GEMM_BK, GEMM_BM};
  uint64_t dB[2] = {(uint64_t)K, (uint64_t)Nw}, sB[1] = {(uint64_t)K};
  uint32_t bB[2] = {GEMM_BK, (uint32_t)BN};
  if (tma_encode_bf16(ctx, &tmA, A, 2, dA, sA, bA, 128) != 0) return -1;
  if (tma_encode_bf16(ctx, &tmB, Wt, 2, dB, sB, bB, 128) != 0) return -1;
  if (dual) return launch_variant<256, 2, true>(tmA, tmB, R, K, Nout, Nw, epi, st);
  if (BN == 256) return launch_variant<256, 2, false>(tmA, tmB, R, K, Nout, Nw, epi, st);
  if (BN == 128) return launch_variant<128, 3, false>(tmA, tmB, R, K, Nout, Nw, epi, st);
  return launch_variant<64, 4, false>(tmA, tmB, R, K, Nout, Nw, epi, st);
}

}  // namespace pf
