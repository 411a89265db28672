// Gated attention core on tcgen05 tensor cores (sm_100a), shared by MSA row attention with pair bias (A.1), MSA
// column attention (A.2) and triangle attention around the starting / ending node (A.7 / A.8) after the driver's row
// permutation:  for every (b, r, h) and query i
//     o[i, :] = gate[i, :] * sum_j softmax_j( q[i].k[j] + bias[b, h, i, j] + NEG(keymask[b, j]) ) v[j, :]
// (q already carries 1/sqrt(d), R12).  Flash-style: logits never leave the SM (north_star: "no materialised N^3
// logits").  One CTA = one (b*r, h, 128-query tile); key tiles of 64:
//   TMA -> smem {Q 128x32, K 64x32 (64B swizzle), V^T 32x64, bias 128x64 (128B swizzle)}      [control thread]
//   S = Q K^T        tcgen05.mma M=128 N=64 K=2x16  -> TMEM cols [0,64)                         [control thread]
//   thread-per-row online softmax in fp32 from tcgen05.ld, P (bf16) -> smem in the UMMA 128B-swizzle layout
//   O_tile = P V     tcgen05.mma M=128 N=32 K=4x16  -> TMEM cols [64,96)                        [control thread]
//   o_acc = o_acc * alpha + O_tile in registers; gate and 1/l applied at the end, 64-byte row stores.
// ~77 KB of shared memory and 128 TMEM columns per CTA -> 2 CTAs per SM hide each other's MMA / barrier latency.
#include "pf_internal.h"
#include "pf_device.cuh"
#include "pf_tc.cuh"

namespace pf {

int tma_encode_bf16(TmaCtx* ctx, CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                    const uint64_t* strides_elems, const uint32_t* box, int swizzle_bytes);

constexpr int AT_BQ = 128;        // queries per CTA
constexpr int AT_BK = 64;         // keys per tile
constexpr int AT_THREADS = 160;   // 4 softmax warps + 1 control warp
constexpr int AT_STAGES = 2;
constexpr int AT_MAXKEYS = 1024;  // mask terms kept in shared memory

struct AttnSmem {
  static constexpr int Q_OFF = 0;                                  // 128 x 32 bf16, 64B swizzle: 8 KB
  static constexpr int P_OFF = Q_OFF + AT_BQ * 64;                 // 128 x 64 bf16, 128B swizzle: 16 KB
  static constexpr int STAGE_OFF = P_OFF + AT_BQ * 128;
  static constexpr int K_BYTES = AT_BK * 64;                       // 64 x 32 bf16: 4 KB
  static constexpr int V_BYTES = 32 * 128;                         // 32 x 64 bf16: 4 KB
  static constexpr int B_BYTES = AT_BQ * 128;                      // 128 x 64 bf16: 16 KB
  static constexpr int STAGE_BYTES = K_BYTES + V_BYTES + B_BYTES;  // 24 KB
  static constexpr int MASK_OFF = STAGE_OFF + AT_STAGES * STAGE_BYTES;
  static constexpr int BAR_OFF = MASK_OFF + AT_MAXKEYS * 4;
  static constexpr int TOTAL = BAR_OFF + 128 + 1024;
};

__global__ void __launch_bounds__(AT_THREADS, 2)
attn_tc_kernel(const __grid_constant__ CUtensorMap tmQK, const __grid_constant__ CUtensorMap tmV,
               const __grid_constant__ CUtensorMap tmBias, const bf16* __restrict__ qkg, const float* __restrict__ keymask,
               bf16* __restrict__ o, int R, int L, int H, int has_bias) {
  using SM = AttnSmem;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = tc::align_smem_1024(smem_raw);
  float* mterm = reinterpret_cast<float*>(smem + SM::MASK_OFF);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::BAR_OFF);
  uint64_t* q_full = bars;                 // 1
  uint64_t* kv_full = bars + 1;            // [AT_STAGES]
  uint64_t* kv_empty = kv_full + AT_STAGES;
  uint64_t* s_full = kv_empty + AT_STAGES;
  uint64_t* p_full = s_full + 1;
  uint64_t* o_full = p_full + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(o_full + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i0 = blockIdx.x * AT_BQ;
  const int h = blockIdx.y;
  const int br = blockIdx.z;
  const int b = br / R;
  const int C = H * 32;
  const int n_kt = (L + AT_BK - 1) / AT_BK;

  if (warp == 4) {
    if (lane == 0) {
      tc::prefetch_tmap(&tmQK);
      tc::prefetch_tmap(&tmV);
      if (has_bias) tc::prefetch_tmap(&tmBias);
      tc::mbar_init(q_full, 1);
      for (int s = 0; s < AT_STAGES; ++s) {
        tc::mbar_init(&kv_full[s], 1);
        tc::mbar_init(&kv_empty[s], 1);
      }
      tc::mbar_init(s_full, 1);
      tc::mbar_init(p_full, 128);
      tc::mbar_init(o_full, 1);
      tc::fence_barrier_init();
    }
    __syncwarp();
    tc::tmem_alloc<128>(tmem_slot);
  } else {
    // additive key mask in the exp2 domain: 0 for an unmasked key, -inf for a masked or out-of-range key (R3)
    for (int j = threadIdx.x; j < n_kt * AT_BK; j += 128)
      mterm[j] = (j < L && keymask[(long)b * L + j] > 0.5f) ? 0.f : -INFINITY;
  }
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const uint32_t tmem_S = tmem_base, tmem_O = tmem_base + 64;

  if (warp == 4) {
    if (tc::elect_one()) {
      const uint32_t stage_tx = SM::K_BYTES + SM::V_BYTES + (has_bias ? SM::B_BYTES : 0);
      auto load_tile = [&](int kt) {
        int s = kt % AT_STAGES;
        uint8_t* st = smem + SM::STAGE_OFF + s * SM::STAGE_BYTES;
        tc::mbar_arrive_expect_tx(&kv_full[s], stage_tx);
        tc::tma_load_3d(st, &tmQK, &kv_full[s], C + h * 32, kt * AT_BK, br);
        tc::tma_load_2d(st + SM::K_BYTES, &tmV, &kv_full[s], kt * AT_BK, (br * H + h) * 32);
        if (has_bias) tc::tma_load_3d(st + SM::K_BYTES + SM::V_BYTES, &tmBias, &kv_full[s], kt * AT_BK, i0, b * H + h);
      };
      tc::mbar_arrive_expect_tx(q_full, AT_BQ * 64);
      tc::tma_load_3d(smem + SM::Q_OFF, &tmQK, q_full, h * 32, i0, br);     // box {32, 64, 1} twice: rows i0.., i0+64..
      tc::tma_load_3d(smem + SM::Q_OFF + 64 * 64, &tmQK, q_full, h * 32, i0 + 64, br);
      load_tile(0);
      constexpr uint32_t idesc_s = tc::idesc_bf16_f32(AT_BQ, AT_BK);
      constexpr uint32_t idesc_o = tc::idesc_bf16_f32(AT_BQ, 32);
      const uint64_t q_desc = tc::smem_desc_kmajor<64>(tc::smem_u32(smem + SM::Q_OFF));
      const uint64_t p_desc = tc::smem_desc_kmajor<128>(tc::smem_u32(smem + SM::P_OFF));
      tc::mbar_wait(q_full, 0);
      for (int kt = 0; kt < n_kt; ++kt) {
        int s = kt % AT_STAGES;
        if (kt + 1 < n_kt) {
          int s2 = (kt + 1) % AT_STAGES;
          tc::mbar_wait(&kv_empty[s2], (((kt + 1) / AT_STAGES) & 1) ^ 1);
          load_tile(kt + 1);
        }
        tc::mbar_wait(&kv_full[s], (kt / AT_STAGES) & 1);
        tc::tc_fence_after();
        uint32_t st_addr = tc::smem_u32(smem + SM::STAGE_OFF + s * SM::STAGE_BYTES);
        uint64_t k_desc = tc::smem_desc_kmajor<64>(st_addr);
        uint64_t v_desc = tc::smem_desc_kmajor<128>(st_addr + SM::K_BYTES);
        tc::mma_bf16(tmem_S, q_desc, k_desc, idesc_s, false);
        tc::mma_bf16(tmem_S, q_desc + 2, k_desc + 2, idesc_s, true);
        tc::mma_commit(s_full);
        tc::mbar_wait(p_full, kt & 1);
        tc::tc_fence_after();
#pragma unroll
        for (int k = 0; k < AT_BK / 16; ++k) tc::mma_bf16(tmem_O, p_desc + 2 * k, v_desc + 2 * k, idesc_o, k != 0);
        tc::mma_commit(o_full);
        tc::mma_commit(&kv_empty[s]);
      }
    }
  } else {
    const int row = warp * 32 + lane;            // warp w reads TMEM lanes [32w, 32w+32)
    const int i = i0 + row;
    const uint32_t lane_addr = (uint32_t)(warp * 32) << 16;
    const float LOG2E = 1.4426950408889634f;
    float m_run = -INFINITY, l_run = 0.f;
    float oacc[32];
#pragma unroll
    for (int d = 0; d < 32; ++d) oacc[d] = 0.f;
    for (int kt = 0; kt < n_kt; ++kt) {
      int s = kt % AT_STAGES;
      const uint8_t* bias_t = smem + SM::STAGE_OFF + s * SM::STAGE_BYTES + SM::K_BYTES + SM::V_BYTES;
      if (has_bias) tc::mbar_wait(&kv_full[s], (kt / AT_STAGES) & 1);
      tc::mbar_wait(s_full, kt & 1);
      tc::tc_fence_after();
      uint32_t sv[2][32];
      tc::tmem_ld32(tmem_S + lane_addr, sv[0]);
      tc::tmem_ld32(tmem_S + lane_addr + 32, sv[1]);
      tc::tmem_ld_wait();
      float x[64];
      float mx = -INFINITY;
#pragma unroll
      for (int c = 0; c < 8; ++c) {   // 8 keys per 16-byte bias chunk
        float bf[8];
        if (has_bias) {
          uint4 u = *reinterpret_cast<const uint4*>(bias_t + tc::swz_offset<128>(row, c));
          const __nv_bfloat162* p2 = reinterpret_cast<const __nv_bfloat162*>(&u);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            bf[2 * e] = __low2float(p2[e]);
            bf[2 * e + 1] = __high2float(p2[e]);
          }
        } else {
#pragma unroll
          for (int e = 0; e < 8; ++e) bf[e] = 0.f;
        }
        float4 m0 = *reinterpret_cast<const float4*>(mterm + kt * AT_BK + c * 8);
        float4 m1 = *reinterpret_cast<const float4*>(mterm + kt * AT_BK + c * 8 + 4);
        float mt[8] = {m0.x, m0.y, m0.z, m0.w, m1.x, m1.y, m1.z, m1.w};
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          int j = c * 8 + e;
          float sj = __uint_as_float(sv[j >> 5][j & 31]) + bf[e];
          float xv = fmaf(sj, LOG2E, mt[e]);
          x[j] = xv;
          mx = fmaxf(mx, xv);
        }
      }
      float m_new = fmaxf(m_run, mx);
      float m_use = (m_new == -INFINITY) ? 0.f : m_new;
      float alpha = exp2f(m_run - m_use);
      float sum = 0.f;
      uint8_t* prow = smem + SM::P_OFF;
      // PV(kt-1) must have finished reading P before it is overwritten
      if (kt > 0) {
        tc::mbar_wait(o_full, (kt - 1) & 1);
        tc::tc_fence_after();
        uint32_t ov[32];
        tc::tmem_ld32(tmem_O + lane_addr, ov);
        tc::tmem_ld_wait();
#pragma unroll
        for (int d = 0; d < 32; ++d) oacc[d] += __uint_as_float(ov[d]);
      }
#pragma unroll
      for (int d = 0; d < 32; ++d) oacc[d] *= alpha;
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        uint32_t pk[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          float p0 = exp2f(x[c * 8 + 2 * e] - m_use), p1 = exp2f(x[c * 8 + 2 * e + 1] - m_use);
          sum += p0 + p1;
          __nv_bfloat162 pp = __floats2bfloat162_rn(p0, p1);
          pk[e] = *reinterpret_cast<uint32_t*>(&pp);
        }
        *reinterpret_cast<uint4*>(prow + tc::swz_offset<128>(row, c)) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
      }
      l_run = l_run * alpha + sum;
      m_run = m_new;
      tc::fence_proxy_async_smem();
      tc::tc_fence_before();
      tc::mbar_arrive(p_full);
    }
    // last tile's PV
    tc::mbar_wait(o_full, (n_kt - 1) & 1);
    tc::tc_fence_after();
    {
      uint32_t ov[32];
      tc::tmem_ld32(tmem_O + lane_addr, ov);
      tc::tmem_ld_wait();
#pragma unroll
      for (int d = 0; d < 32; ++d) oacc[d] += __uint_as_float(ov[d]);
    }
    if (i < L) {
      float inv = l_run > 0.f ? 1.0f / l_run : 0.f;
      const bf16* gp = qkg + ((long)br * L + i) * (3 * C) + 2 * C + h * 32;
      bf16* op = o + ((long)br * L + i) * C + h * 32;
#pragma unroll
      for (int d = 0; d < 32; d += 8) {
        uint4 gu = *reinterpret_cast<const uint4*>(gp + d);   // the gate is stored as fp16 (bounded in [0,1], not an MMA operand)
        const __half2* g2 = reinterpret_cast<const __half2*>(&gu);
        uint32_t pk[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          __nv_bfloat162 pp = __floats2bfloat162_rn(oacc[d + 2 * e] * inv * __low2float(g2[e]),
                                                    oacc[d + 2 * e + 1] * inv * __high2float(g2[e]));
          pk[e] = *reinterpret_cast<uint32_t*>(&pp);
        }
        *reinterpret_cast<uint4*>(op + d) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
      }
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 4) tc::tmem_dealloc<128>(tmem_base);
}

int launch_attn_tc(TmaCtx* ctx, const bf16* qkg, const bf16* vt, const bf16* bias, const float* keymask, bf16* o, int B,
                   int R, int L, int Lpad, int H, int num_sms, cudaStream_t st) {
  (void)num_sms;
  if (L > AT_MAXKEYS) {
    tc_set_error("attn_tc: key length above 1024 not supported");
    return -1;
  }
  const int C = H * 32;
  CUtensorMap tmQK, tmV, tmB;
  {
    uint64_t d[3] = {(uint64_t)3 * C, (uint64_t)L, (uint64_t)B * R}, s[2] = {(uint64_t)3 * C, (uint64_t)L * 3 * C};
    uint32_t bx[3] = {32, 64, 1};
    if (tma_encode_bf16(ctx, &tmQK, qkg, 3, d, s, bx, 64) != 0) return -1;
  }
  {
    uint64_t d[2] = {(uint64_t)L, (uint64_t)B * R * H * 32}, s[1] = {(uint64_t)Lpad};
    uint32_t bx[2] = {64, 32};
    if (tma_encode_bf16(ctx, &tmV, vt, 2, d, s, bx, 128) != 0) return -1;
  }
  if (bias) {
    uint64_t d[3] = {(uint64_t)L, (uint64_t)L, (uint64_t)B * H}, s[2] = {(uint64_t)Lpad, (uint64_t)L * Lpad};
    uint32_t bx[3] = {64, 128, 1};
    if (tma_encode_bf16(ctx, &tmB, bias, 3, d, s, bx, 128) != 0) return -1;
  } else {
    tmB = tmV;
  }
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem::TOTAL);
    if (e != cudaSuccess) {
      tc_set_error(std::string("cudaFuncSetAttribute(attn_tc): ") + cudaGetErrorString(e));
      return -1;
    }
    configured = true;
  }
  dim3 grid((L + AT_BQ - 1) / AT_BQ, H, B * R);
  attn_tc_kernel<<<grid, AT_THREADS, AttnSmem::TOTAL, st>>>(tmQK, tmV, tmB, qkg, keymask, o, R, L, H, bias ? 1 : 0);
  return 0;
}

}  // namespace pf
