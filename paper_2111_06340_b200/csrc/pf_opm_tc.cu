// Outer-product-mean core on tcgen05 tensor cores (A.4, reading R5/R6):
//     z[b,i,j,:] += ( vec_{c1,c2}( sum_s a[s,i,c1] b[s,j,c2] ) / (1e-3 + n_ij) ) W_out + b_out,   n_ij = sum_s mu_si mu_sj
// a, b arrive masked and transposed from the projection epilogue as ab_t[(b,i), ch, Spad] (ch 0..31 = a, 32..63 = b;
// s contiguous), so both operands of the first contraction are K-major tiles TMA can fetch directly.
// One CTA = 128 residues i x 2 residues j of one protein.  For c1 = 0..31 (software-pipelined over two TMEM buffers):
//   GEMM1  D1[i, (j,c2)] = sum_s a[s,i,c1] b[s,j,c2]        M=128, N=64,  K=S     (a streamed per c1, b resident)
//   epilogue warps: D1 fp32 (TMEM) -> fp16 pairs written back over the same TMEM columns (j at 32-bit columns 32 j + [0, 16))
//   GEMM2  acc_j[i, e] += sum_c2 D1[i,(j,c2)] W_out[c1*32+c2, e]   M=128, N=128, K=32  per j, accumulated over c1 in TMEM,
//          its A operand read from tensor memory: the kernel is paced by shared-memory bandwidth (GEMM1 alone asks for
//          192 B/clk at M=128, N=64), so the outer product makes no trip through shared memory
// so the 32x32 outer product per pair never reaches HBM (north_star bullet 3).  Final: acc_j / (1e-3 + n_ij) + b_out
// added to the fp32 pair stream, 512 contiguous bytes per thread.
#include "pf_internal.h"
#include "pf_device.cuh"
#include "pf_tc.cuh"

namespace pf {

int tma_encode_bf16(TmaCtx* ctx, CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                    const uint64_t* strides_elems, const uint32_t* box, int swizzle_bytes);

constexpr int OP_BI = 128, OP_BJ = 2, OP_C = 32, OP_CZ = 128, OP_BK = 64;
constexpr int OP_MAX_KB = 8;       // S <= 512
constexpr int OP_A_STAGES = 12;    // upper bound; the launch uses as many 16 KB stages as fit beside the resident b operand
constexpr int OP_THREADS = 192;
constexpr int OP_NB = 4;           // at most 4 outer-product tiles in flight between the two contractions (TMEM: 4 x 64 columns)
// Per launch: nb = 4 tiles in flight and GEMM2 lagging GEMM1 by 2 when the contraction is short (N_seq <= 256: GEMM1 is too short
// to hide the relayout of the previous tile behind it), nb = 2 / lag 1 otherwise (the shared memory goes to a deeper a ring,
// which is what bounds the long contractions).

// Shared memory: W_out tiles and the barriers at fixed offsets, then the resident b operand
// (n_kb x 8 KB, n_kb = k-blocks of this launch) and behind it the ring of a tiles: as many 16 KB stages as fit.  The a stream
// is fetched from L2 with a latency of ~1 us, so its rate is ring bytes / latency (measured: 64 KB in flight gave ~71 GB/s per
// SM and bounded the kernel; the multicast variant, which cuts L2 traffic instead, was slower).
struct OpmSmem {
  static constexpr int B_KB_BYTES = OP_BJ * OP_C * 128;                  // 8 KB
  static constexpr int A_BYTES = OP_BI * 128;                            // 16 KB
  static constexpr int W_OFF = 0;
  static constexpr int W_BYTES = OP_CZ * 64;                             // 128 e x 32 c2 bf16 = 8 KB
  static constexpr int BAR_OFF = 0;
  static constexpr int TOTAL = 227 * 1024;
  static __host__ __device__ int b_off(int nb) { return 1024 + nb * W_BYTES; }                  // W ring first, at 1024
  static __host__ __device__ int ring_bytes(int nb) { return TOTAL - 1024 - b_off(nb); }        // b operand + a ring
};

__global__ void __launch_bounds__(OP_THREADS, 1)
opm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
              const __grid_constant__ CUtensorMap tmW, const float* __restrict__ bout, const float* __restrict__ seq_mask,
              const float* __restrict__ msa_mask, float* __restrict__ z, int S, int N, int s0, int Sc, int add_bias,
              int a_stages, int nb_shift) {
  using SM = OpmSmem;
  {
    // both residues j of this CTA padded: every output is at a masked position (uniform over the CTA: exit before any setup)
    const int jj = blockIdx.x * OP_BJ, bb = blockIdx.z;
    bool any = false;
    for (int e = 0; e < OP_BJ; ++e) any = any || (jj + e < N && seq_mask[(long)bb * N + jj + e] > 0.5f);
    if (!any) return;
  }
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = tc::align_smem_1024(smem_raw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::BAR_OFF);
  uint64_t* b_full = bars;
  uint64_t* a_full = bars + 1;                    // [OP_A_STAGES]
  uint64_t* a_empty = a_full + OP_A_STAGES;       // [OP_A_STAGES]
  uint64_t* w_full = a_empty + OP_A_STAGES;       // [OP_NB]
  uint64_t* w_empty = w_full + OP_NB;             // [OP_NB]
  uint64_t* d1_full = w_empty + OP_NB;            // [OP_NB]
  uint64_t* ov_full = d1_full + OP_NB;            // [OP_NB]
  uint64_t* acc_full = ov_full + OP_NB;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_full + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int j0 = blockIdx.x * OP_BJ, i0 = blockIdx.y * OP_BI, b = blockIdx.z;
  // this launch contracts the sequences [s0, s0 + Sc) (Sc <= 512: the b operand of the chunk stays resident in shared memory);
  // the normaliser counts all S sequences, and the chunks add up because the projection is linear (bias with the first chunk)
  const int n_kb = (Sc + OP_BK - 1) / OP_BK;
  const int nb = 1 << nb_shift, lag = nb >> 1;
  const int W_OFF = 1024, B_OFF = SM::b_off(nb);
  const int A_OFF = B_OFF + n_kb * SM::B_KB_BYTES;

  if (warp == 0 && lane == 0) {
    tc::prefetch_tmap(&tmA);
    tc::prefetch_tmap(&tmB);
    tc::prefetch_tmap(&tmW);
    tc::mbar_init(b_full, 1);
    for (int s = 0; s < OP_A_STAGES; ++s) {
      tc::mbar_init(&a_full[s], 1);
      tc::mbar_init(&a_empty[s], 1);
    }
    for (int s = 0; s < OP_NB; ++s) {
      tc::mbar_init(&w_full[s], 1);
      tc::mbar_init(&w_empty[s], 1);
      tc::mbar_init(&d1_full[s], 1);
      tc::mbar_init(&ov_full[s], 128);
    }
    tc::mbar_init(acc_full, 1);
    tc::fence_barrier_init();
  }
  if (warp == 1) tc::tmem_alloc<512>(tmem_slot);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const uint32_t tmem_acc = tmem_base;            // 2 x 128 columns
  const uint32_t tmem_d1 = tmem_base + 256;       // OP_NB x 64 columns

  if (warp == 0) {
    if (tc::elect_one()) {
      tc::mbar_arrive_expect_tx(b_full, (uint32_t)n_kb * SM::B_KB_BYTES);
      for (int kb = 0; kb < n_kb; ++kb)
        tc::tma_load_3d(smem + B_OFF + kb * SM::B_KB_BYTES, &tmB, b_full, s0 + kb * OP_BK, OP_C, b * N + j0);
      int s = 0;
      uint32_t ph = 0;                               // ring position and its phase (no divisions on this path)
      for (int c1 = 0; c1 < OP_C; ++c1) {
        for (int kb = 0; kb < n_kb; ++kb) {
          tc::mbar_wait(&a_empty[s], ph ^ 1);
          tc::mbar_arrive_expect_tx(&a_full[s], SM::A_BYTES);
          tc::tma_load_3d(smem + A_OFF + s * SM::A_BYTES, &tmA, &a_full[s], s0 + kb * OP_BK, c1, b * N + i0);
          if (++s == a_stages) { s = 0; ph ^= 1; }
        }
        int ws = c1 & (nb - 1);
        tc::mbar_wait(&w_empty[ws], ((c1 >> nb_shift) & 1) ^ 1);
        tc::mbar_arrive_expect_tx(&w_full[ws], SM::W_BYTES);
        tc::tma_load_2d(smem + W_OFF + ws * SM::W_BYTES, &tmW, &w_full[ws], c1 * OP_C, 0);
      }
    }
  } else if (warp == 1) {
    if (tc::elect_one()) {
      // a, b, the outer product and W_out are fp16 (R17 round 2: 8x finer rounding than bf16 at the same rate)
      constexpr uint32_t idesc1 = tc::idesc_f16_f32(OP_BI, OP_BJ * OP_C);
      constexpr uint32_t idesc2 = tc::idesc_f16_f32(OP_BI, OP_CZ);
      tc::mbar_wait(b_full, 0);
      int s = 0;
      uint32_t ph = 0;
      for (int c1 = 0; c1 < OP_C + lag; ++c1) {
        if (c1 < OP_C) {
          // No wait for the buffer: its previous content (tile c1 - nb, converted in place) was the A operand of GEMM2(c1 - nb),
          // issued by this thread lag = nb / 2 iterations ago, and tcgen05.mma operations of one thread execute in issue order.
          int buf = c1 & (nb - 1);
          for (int kb = 0; kb < n_kb; ++kb) {
            tc::mbar_wait(&a_full[s], ph);
            tc::tc_fence_after();
            uint64_t a_desc = tc::smem_desc_kmajor<128>(tc::smem_u32(smem + A_OFF + s * SM::A_BYTES));
            uint64_t b_desc = tc::smem_desc_kmajor<128>(tc::smem_u32(smem + B_OFF + kb * SM::B_KB_BYTES));
#pragma unroll
            for (int k = 0; k < OP_BK / 16; ++k)
              tc::mma_bf16(tmem_d1 + buf * 64, a_desc + 2 * k, b_desc + 2 * k, idesc1, (kb | k) != 0);
            tc::mma_commit(&a_empty[s]);
            if (++s == a_stages) { s = 0; ph ^= 1; }
          }
          tc::mma_commit(&d1_full[buf]);
        }
        if (c1 >= lag) {
          int p = c1 - lag, pb = p & (nb - 1);
          tc::mbar_wait(&ov_full[pb], (p >> nb_shift) & 1);
          tc::mbar_wait(&w_full[pb], (p >> nb_shift) & 1);
          tc::tc_fence_after();
          uint64_t w_desc = tc::smem_desc_kmajor<64>(tc::smem_u32(smem + W_OFF + pb * SM::W_BYTES));
#pragma unroll
          for (int j = 0; j < OP_BJ; ++j) {
            const uint32_t o_t = tmem_d1 + pb * 64 + j * 32;   // fp16 pairs: 8 columns per K = 16 step
            tc::mma_bf16_ts(tmem_acc + j * OP_CZ, o_t, w_desc, idesc2, p != 0);
            tc::mma_bf16_ts(tmem_acc + j * OP_CZ, o_t + 8, w_desc + 2, idesc2, true);
          }
          tc::mma_commit(&w_empty[pb]);
        }
      }
      tc::mma_commit(acc_full);
    }
  } else {
    const int quarter = warp & 3;
    const int row = quarter * 32 + lane;
    const int i = i0 + row;
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    for (int c1 = 0; c1 < OP_C; ++c1) {
      int buf = c1 & (nb - 1);
      tc::mbar_wait(&d1_full[buf], (c1 >> nb_shift) & 1);
      tc::tc_fence_after();
      uint32_t v[2][32];
      tc::tmem_ld32(tmem_d1 + buf * 64 + lane_addr, v[0]);
      tc::tmem_ld32(tmem_d1 + buf * 64 + lane_addr + 32, v[1]);
      tc::tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < OP_BJ; ++j) {
        uint32_t pk[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
          __half2 pp = __floats2half2_rn(__uint_as_float(v[j][2 * e]), __uint_as_float(v[j][2 * e + 1]));
          pk[e] = *reinterpret_cast<uint32_t*>(&pp);
        }
        tc::tmem_st16(tmem_d1 + buf * 64 + lane_addr + j * 32, pk);   // over this thread's own (already loaded) columns
      }
      tc::tmem_st_wait();
      tc::tc_fence_before();
      tc::mbar_arrive(&ov_full[buf]);
    }
    // n_ij = (sum_s rho_s) sigma_i sigma_j   (R5)
    float cnt = 0.f;
    for (int s = lane; s < S; s += 32) cnt += msa_mask[(long)b * S + s];
    cnt = warp_sum(cnt);
    tc::mbar_wait(acc_full, 0);
    tc::tc_fence_after();
    const float si = (i < N) ? seq_mask[(long)b * N + i] : 0.f;
#pragma unroll 1
    for (int j = 0; j < OP_BJ; ++j) {
      const int jj = j0 + j;
      const bool ok = (i < N) && (jj < N);
      const float inv = ok ? 1.0f / (1e-3f + cnt * si * seq_mask[(long)b * N + jj]) : 0.f;
      float* dst = z + (((long)b * N + i) * N + jj) * OP_CZ;
#pragma unroll 1
      for (int c0 = 0; c0 < OP_CZ; c0 += 32) {
        uint32_t v[32];
        tc::tmem_ld32(tmem_acc + j * OP_CZ + lane_addr + c0, v);
        tc::tmem_ld_wait();
        if (ok) {
#pragma unroll
          for (int e = 0; e < 32; e += 4) {
            float4 o = *reinterpret_cast<float4*>(dst + c0 + e);
            float4 bo = add_bias ? __ldg(reinterpret_cast<const float4*>(bout + c0 + e)) : make_float4(0.f, 0.f, 0.f, 0.f);
            o.x += __uint_as_float(v[e]) * inv + bo.x;
            o.y += __uint_as_float(v[e + 1]) * inv + bo.y;
            o.z += __uint_as_float(v[e + 2]) * inv + bo.z;
            o.w += __uint_as_float(v[e + 3]) * inv + bo.w;
            *reinterpret_cast<float4*>(dst + c0 + e) = o;
          }
        }
      }
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 1) tc::tmem_dealloc<512>(tmem_base);
}

bool configure_opm_kernel() {
  cudaError_t e = cudaFuncSetAttribute(opm_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, OpmSmem::TOTAL);
  if (e != cudaSuccess) tc_set_error(std::string("cudaFuncSetAttribute(opm_tc): ") + cudaGetErrorString(e));
  return e == cudaSuccess;
}

int launch_opm_tc(TmaCtx* ctx, const bf16* ab_t, const bf16* wout_t, const float* bout, const float* seq_mask,
                  const float* msa_mask, float* z, int B, int S, int Spad, int N, cudaStream_t st) {
  CUtensorMap tmA, tmB, tmW;
  uint64_t d[3] = {(uint64_t)S, 2 * OP_C, (uint64_t)B * N}, s[2] = {(uint64_t)Spad, (uint64_t)2 * OP_C * Spad};
  uint32_t bxA[3] = {OP_BK, 1, OP_BI}, bxB[3] = {OP_BK, OP_C, OP_BJ};
  if (tma_encode_bf16(ctx, &tmA, ab_t, 3, d, s, bxA, 128) != 0) return -1;
  if (tma_encode_bf16(ctx, &tmB, ab_t, 3, d, s, bxB, 128) != 0) return -1;
  uint64_t dw[2] = {(uint64_t)OP_C * OP_C, OP_CZ}, sw[1] = {(uint64_t)OP_C * OP_C};
  uint32_t bxW[2] = {OP_C, OP_CZ};
  if (tma_encode_bf16(ctx, &tmW, wout_t, 2, dw, sw, bxW, 64) != 0) return -1;
  dim3 grid((N + OP_BJ - 1) / OP_BJ, (N + OP_BI - 1) / OP_BI, B);
  const int chunk = OP_MAX_KB * OP_BK;   // 512 sequences per launch; the extra-MSA stack (S in the thousands) takes several
  for (int s0 = 0; s0 < S; s0 += chunk) {
    const int Sc = S - s0 < chunk ? S - s0 : chunk, n_kb = (Sc + OP_BK - 1) / OP_BK;
    const int nb_shift = Sc <= 256 ? 2 : 1;
    int stages = (OpmSmem::ring_bytes(1 << nb_shift) - n_kb * OpmSmem::B_KB_BYTES) / OpmSmem::A_BYTES;
    stages = stages > OP_A_STAGES ? OP_A_STAGES : stages;
    opm_tc_kernel<<<grid, OP_THREADS, OpmSmem::TOTAL, st>>>(tmA, tmB, tmW, bout, seq_mask, msa_mask, z, S, N, s0, Sc,
                                                            s0 == 0 ? 1 : 0, stages, nb_shift);
  }
  return 0;
}

}  // namespace pf
