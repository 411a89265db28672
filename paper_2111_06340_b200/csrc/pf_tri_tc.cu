// Triangle multiplicative update, the contraction itself (A.5; A.6 through the driver's transposition identity):
//     t[bc, i, j] = sum_k a[bc, i, k] * b[bc, j, k]        bc = (batch, channel), a/b channel-major bf16 [B*C, N, Npad]
// = one N x N x N "NT" GEMM per (batch, channel) on tcgen05 tensor cores (north_star: "channel-batched GEMMs").
// One CTA = one 128 x 128 tile of one channel: 3-D TMA tiles (k, row, bc) with out-of-range k / rows zero-filled,
// 3-stage ring, fp32 accumulator in TMEM, epilogue stores bf16 rows (64 B per thread per chunk) for the
// LayerNorm-across-channels kernel that follows (bf16 like the other inter-kernel intermediates: halves this tensor's traffic).
#include "pf_internal.h"
#include "pf_device.cuh"
#include "pf_tc.cuh"

namespace pf {

int tma_encode_bf16(TmaCtx* ctx, CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                    const uint64_t* strides_elems, const uint32_t* box, int swizzle_bytes);

constexpr int TRI_BM = 128, TRI_BN = 128, TRI_BK = 64, TRI_STAGES = 3, TRI_THREADS = 192;
constexpr int TRI_STAGE_BYTES = (TRI_BM + TRI_BN) * TRI_BK * 2;
constexpr int TRI_BAR_OFF = TRI_STAGES * TRI_STAGE_BYTES;
constexpr int TRI_SMEM = TRI_BAR_OFF + 256 + 1024;

__global__ void __launch_bounds__(TRI_THREADS, 2)
tri_einsum_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                     bf16* __restrict__ t, int N, int Npad, const int* __restrict__ key_tiles, int channels) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = tc::align_smem_1024(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + TRI_BAR_OFF);
  uint64_t* empty = full + TRI_STAGES;
  uint64_t* tmem_full = empty + TRI_STAGES;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tmem_full + 1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int j0 = blockIdx.x * TRI_BN, i0 = blockIdx.y * TRI_BM, bc = blockIdx.z;
  int num_kb = (N + TRI_BK - 1) / TRI_BK;
  if (key_tiles) num_kb = min(num_kb, key_tiles[bc / channels]);   // operands are exactly zero at masked residues k

  if (warp == 0 && lane == 0) {
    tc::prefetch_tmap(&tmA);
    tc::prefetch_tmap(&tmB);
    for (int s = 0; s < TRI_STAGES; ++s) {
      tc::mbar_init(&full[s], 1);
      tc::mbar_init(&empty[s], 1);
    }
    tc::mbar_init(tmem_full, 1);
    tc::fence_barrier_init();
  }
  if (warp == 1) tc::tmem_alloc<TRI_BN>(tmem_slot);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (tc::elect_one()) {
      for (int kb = 0; kb < num_kb; ++kb) {
        int s = kb % TRI_STAGES;
        tc::mbar_wait(&empty[s], ((kb / TRI_STAGES) & 1) ^ 1);
        tc::mbar_arrive_expect_tx(&full[s], TRI_STAGE_BYTES);
        uint8_t* a = smem + s * TRI_STAGE_BYTES;
        tc::tma_load_3d(a, &tmA, &full[s], kb * TRI_BK, i0, bc);
        tc::tma_load_3d(a + TRI_BM * TRI_BK * 2, &tmB, &full[s], kb * TRI_BK, j0, bc);
      }
    }
  } else if (warp == 1) {
    if (tc::elect_one()) {
      constexpr uint32_t idesc = tc::idesc_f16_f32(TRI_BM, TRI_BN);   // operands and result fp16 (R17, round 2)
      for (int kb = 0; kb < num_kb; ++kb) {
        int s = kb % TRI_STAGES;
        tc::mbar_wait(&full[s], (kb / TRI_STAGES) & 1);
        tc::tc_fence_after();
        uint32_t a_addr = tc::smem_u32(smem + s * TRI_STAGE_BYTES);
        uint64_t a_desc = tc::smem_desc_kmajor<128>(a_addr);
        uint64_t b_desc = tc::smem_desc_kmajor<128>(a_addr + TRI_BM * TRI_BK * 2);
#pragma unroll
        for (int k = 0; k < TRI_BK / 16; ++k) tc::mma_bf16(tmem_base, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | k) != 0);
        tc::mma_commit(&empty[s]);
      }
      tc::mma_commit(tmem_full);
    }
  } else {
    const int quarter = warp & 3;
    const int i = i0 + quarter * 32 + lane;
    tc::mbar_wait(tmem_full, 0);
    tc::tc_fence_after();
    const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
    bf16* dst = t + ((long)bc * N + i) * Npad + j0;
#pragma unroll 1
    for (int c0 = 0; c0 < TRI_BN; c0 += 32) {
      if (j0 + c0 >= N) break;
      uint32_t v[32];
      tc::tmem_ld32(lane_addr + c0, v);
      tc::tmem_ld_wait();
      if (i < N) {
#pragma unroll
        for (int j = 0; j < 32; j += 8)   // Npad is a multiple of 8: whole 16-byte groups stay inside the padded row
          if (j0 + c0 + j < Npad) {
            uint32_t pk[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              __half2 h = __floats2half2_rn(__uint_as_float(v[j + 2 * e]), __uint_as_float(v[j + 2 * e + 1]));
              pk[e] = *reinterpret_cast<uint32_t*>(&h);
            }
            *reinterpret_cast<uint4*>(dst + c0 + j) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
          }
      }
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 1) tc::tmem_dealloc<TRI_BN>(tmem_base);
}

bool configure_tri_kernel() {
  cudaError_t e = cudaFuncSetAttribute(tri_einsum_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TRI_SMEM);
  if (e != cudaSuccess) tc_set_error(std::string("cudaFuncSetAttribute(tri_einsum_tc): ") + cudaGetErrorString(e));
  return e == cudaSuccess;
}

int launch_tri_einsum_tc(TmaCtx* ctx, const bf16* a_cm, const bf16* b_cm, bf16* t_cm, int batch, int N, int Npad,
                         const int* key_tiles, int channels, int num_sms, cudaStream_t st) {
  (void)num_sms;
  CUtensorMap tmA, tmB;
  uint64_t d[3] = {(uint64_t)N, (uint64_t)N, (uint64_t)batch}, s[2] = {(uint64_t)Npad, (uint64_t)N * Npad};
  uint32_t bx[3] = {TRI_BK, TRI_BM, 1};
  if (tma_encode_bf16(ctx, &tmA, a_cm, 3, d, s, bx, 128) != 0) return -1;
  if (tma_encode_bf16(ctx, &tmB, b_cm, 3, d, s, bx, 128) != 0) return -1;
  dim3 grid((N + TRI_BN - 1) / TRI_BN, (N + TRI_BM - 1) / TRI_BM, batch);
  tri_einsum_tc_kernel<<<grid, TRI_THREADS, TRI_SMEM, st>>>(tmA, tmB, t_cm, N, Npad, key_tiles, channels);
  return 0;
}

}  // namespace pf
