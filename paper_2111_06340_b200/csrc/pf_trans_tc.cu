// Fused transition on tcgen05 tensor cores (sm_100a) — SURVEY.md App. A.3 (MSA, C = 256) and A.9 (pair, C = 128):
//     res[r, :] += relu(LayerNorm(res[r, :]) W1 + b1) W2 + b2,      W1: C -> 4C,  W2: 4C -> C
// (north_star: "MSA and pair transitions fused with their residual adds"; §8(a) rows 3 / 9: "hidden stays on-chip").
// The 4C-wide hidden activation never reaches HBM and, since round 2, not even shared memory: per 128-row tile it is produced
// 128 columns at a time into TMEM (GEMM1), rectified by the epilogue warps IN PLACE (tcgen05.ld -> +b1, relu, bf16 pairs ->
// tcgen05.st over the thread's own fp32 columns) and consumed from tensor memory as the A operand of GEMM2 (tcgen05.mma with a
// TMEM A operand), which accumulates the C output columns in TMEM over the 4C/128 chunks.  HBM traffic per row is one fp32 read
// and one fp32 reduce-add of C values (the algorithmic minimum 8C bytes + the L2-resident weights).  The kernel is paced by
// shared-memory bandwidth (128 B/clk: both operands of a 128 x 128 x 16 MMA from shared memory already take all of it, and the
// weight tiles arriving by TMA and the staging traffic come on top), so every byte kept out of shared memory is time.
//
// One persistent CTA per SM, 18 working warps (20 launched: register re-allocation is per warpgroup of four):
//   warps 0-7   epilogue, two teams of four warps.  E1(chunk): team t rectifies columns [64t, 64t+64) of the hidden chunk into
//               32-bit columns [64t, 64t+32) of the same accumulator buffer.  E2(tile): the C output columns + b2 in 32-column
//               fp32 boxes through staging tiles -> TMA reduce-add into the residual (the add happens at L2).  At C = 256 the
//               staging tiles are the tile's own A1 buffer (idle after its last GEMM1); the team leaders hand it back to the
//               producers once the reduce-adds have read it.
//   warps 8-15  LayerNorm producers: warp-per-row, 128-bit loads, warp-shuffle statistics, fp16 result straight into the
//               UMMA K-major 128B-swizzle layout (A1, double buffered: the LayerNorm of tile t+1 runs under the GEMMs of tile
//               t); the next rows are pulled into L2 by a bulk prefetch.
//   warp 16     TMA: [128 x 64] weight tiles of W1^T / W2^T through one ring, in the order the MMA thread consumes them
//   warp 17     TMEM allocation + the single MMA-issuing thread.  Issue order per tile: G1(0), G1(1), G2(0), G1(2), G2(1),
//               ... so the rectification of chunk c overlaps GEMM1 of chunk c+1 (hidden accumulator double-buffered in TMEM).
//               GEMM1(c+2) overwrites the buffer GEMM2(c) reads its A operand from: both are issued by this one thread, in
//               that order, and tcgen05.mma operations of one thread execute in issue order (no barrier in between).
#include "pf_internal.h"
#include "pf_device.cuh"
#include "pf_tc.cuh"
#include "pf_lnprod.cuh"

#include <cuda_fp16.h>
#include <string>

namespace pf {

int tma_encode(TmaCtx* ctx, CUtensorMap* out, const void* base, int elem_kind, int rank, const uint64_t* dims,
               const uint64_t* strides_bytes, const uint32_t* box, int swizzle_bytes);

constexpr int TR_THREADS = 20 * 32;      // warps 18, 19 only complete the fourth warpgroup (setmaxnreg is per warpgroup)
constexpr int TR_EPI_WARPS = 8;
constexpr int TR_PROD_WARPS = 8;
constexpr int TR_HC = 128;              // hidden columns per chunk

template <int C>
struct TrSmem {
  static constexpr int KB1 = C / 64;                       // k-blocks of GEMM1 (K = C)
  static constexpr int NH = C / 128;                       // 128-column halves of the output
  static constexpr int A1_BUFS = 2;
  static constexpr int A1_BYTES = 128 * C * 2;
  static constexpr int KB_BYTES = 128 * 128;               // one [128 x 64] 16-bit k-block = one [128 x 32] fp32 output box
  static constexpr int ST_BYTES = 4 * KB_BYTES;            // output staging: two teams x two boxes
  // C = 256: the staging boxes of tile t live in the A1 buffer of tile t (idle once its last GEMM1 has retired; handed back
  // to the LayerNorm producers when the reduce-adds have read it); C = 128 has room for a region of its own
  static constexpr bool ST_ALIAS = (C == 256);
  static constexpr int W_STAGE = KB_BYTES;                 // [128 rows x 64 k] 16-bit
  static constexpr int W_STAGES = 5;
  static constexpr int A1_OFF = 0;
  static constexpr int ST_OFF = A1_OFF + A1_BUFS * A1_BYTES;
  static constexpr int W_OFF = ST_OFF + (ST_ALIAS ? 0 : ST_BYTES);
  static constexpr int B1_OFF = W_OFF + W_STAGES * W_STAGE;   // fp32 b1 [4C]
  static constexpr int B2_OFF = B1_OFF + 4 * C * 4;           // fp32 b2 [C]
  static constexpr int BAR_OFF = B2_OFF + C * 4;
  static constexpr int TOTAL = BAR_OFF + 256 + 1024;
  static constexpr int TMEM_ACC2 = 256;                    // acc1[2] at columns 0 / 128, acc2 at [256, 256 + C)
  static_assert(!ST_ALIAS || A1_BYTES == ST_BYTES, "aliased staging must fit the A1 buffer");
  static_assert(TOTAL <= 227 * 1024, "shared memory budget");
};

struct TrParams {
  const float* res;       // [R, C] fp32 residual (read for the LayerNorm; updated through the tensor map)
  const float* gamma;
  const float* beta;
  const float* b1;        // [4C]
  const float* b2;        // [C]
  long R;
  long num_tiles;
  const unsigned char* tile_active;   // optional: 0 = every row of the 128-row tile is masked, skip it
};

__device__ __forceinline__ bool tr_tile_on(long t, const TrParams& p) { return !p.tile_active || p.tile_active[t] != 0; }

__device__ __forceinline__ uint32_t tr_pack_bf16(float a, float b) {
  __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&h);
}
__device__ __forceinline__ uint32_t tr_pack_f16(float a, float b) {
  __half2 h = __floats2half2_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&h);
}

template <int C>
__global__ void __launch_bounds__(TR_THREADS, 1)
transition_kernel(const __grid_constant__ CUtensorMap tmW1, const __grid_constant__ CUtensorMap tmW2,
                  const __grid_constant__ CUtensorMap tmR, const __grid_constant__ TrParams p) {
  using SM = TrSmem<C>;
  constexpr int KB1 = SM::KB1, NH = SM::NH, WS = SM::W_STAGES, A1B = SM::A1_BUFS;
  constexpr int NC = 4 * C / TR_HC;                        // hidden chunks per tile
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = tc::align_smem_1024(smem_raw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::BAR_OFF);
  uint64_t* a1_full = bars;                // [2]
  uint64_t* a1_empty = bars + 2;           // [2]
  uint64_t* w_full = bars + 4;             // [WS]
  uint64_t* w_empty = w_full + WS;         // [WS]
  uint64_t* acc1_full = w_empty + WS;      // [2]
  uint64_t* a2_full = acc1_full + 2;       // [2]
  uint64_t* acc2_full = a2_full + 2;       // 1
  uint64_t* acc2_empty = acc2_full + 1;    // 1
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc2_empty + 1);
  float* sb1 = reinterpret_cast<float*>(smem + SM::B1_OFF);
  float* sb2 = reinterpret_cast<float*>(smem + SM::B2_OFF);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 16 && lane == 0) {
    tc::prefetch_tmap(&tmW1);
    tc::prefetch_tmap(&tmW2);
    tc::prefetch_tmap(&tmR);
    for (int i = 0; i < 2; ++i) {
      tc::mbar_init(&a1_full[i], TR_PROD_WARPS * 32);
      tc::mbar_init(&a1_empty[i], SM::ST_ALIAS ? 2 : 1);   // aliased staging: one arrival per team leader
      tc::mbar_init(&acc1_full[i], 1);
      tc::mbar_init(&a2_full[i], TR_EPI_WARPS * 32);
    }
    for (int i = 0; i < WS; ++i) {
      tc::mbar_init(&w_full[i], 1);
      tc::mbar_init(&w_empty[i], 1);
    }
    tc::mbar_init(acc2_full, 1);
    tc::mbar_init(acc2_empty, TR_EPI_WARPS * 32);
    tc::fence_barrier_init();
  }
  if (warp == 17) tc::tmem_alloc<512>(tmem_slot);
  for (int i = threadIdx.x; i < 4 * C; i += TR_THREADS) sb1[i] = __ldg(p.b1 + i);
  for (int i = threadIdx.x; i < C; i += TR_THREADS) sb2[i] = __ldg(p.b2 + i);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  // 20 x 96 registers at launch = the CTA's pool: warps 16-19 drop to 40, the epilogue warps grow to 120
  if (warp >= 16) tc::reg_dealloc<40>();
  if (warp < TR_EPI_WARPS) {
    tc::reg_alloc<120>();
    // =========================================================== epilogue (two teams of four warps)
    const int team = warp >> 2, quarter = warp & 3;
    const int lr = quarter * 32 + lane;                // tile row = TMEM lane
    const bool leader = (threadIdx.x & 127) == 0;
    const int bar_id = 1 + team;
    const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
    const uint32_t sw = (uint32_t)(lr & 7);
    uint32_t cc = 0;                                   // hidden chunks consumed so far (all tiles)
    uint32_t it = 0;
    for (long tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
      if (!tr_tile_on(tile, p)) continue;
#pragma unroll 1
      for (int c = 0; c < NC; ++c, ++cc) {
        const uint32_t buf = cc & 1, ph = (cc >> 1) & 1;
        if (SM::ST_ALIAS && c == 1 && it > 0 && leader) {
          // the previous tile's reduce-adds have read their staging boxes (its A1 buffer): hand it to the producers
          tc::bulk_wait_read<0>();
          tc::mbar_arrive(&a1_empty[(it - 1) % A1B]);
        }
        tc::mbar_wait(&acc1_full[buf], ph);
        tc::tc_fence_after();
        const float* bb = sb1 + c * TR_HC + team * 64;
        const uint32_t ta = lane_addr + buf * TR_HC + team * 64;
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
          uint32_t v[32];
          float b1r[32];
          tc::tmem_ld32(ta + hf * 32, v);
#pragma unroll
          for (int q = 0; q < 8; ++q) {   // bias to registers first: a shared load between the stores below could not move
            const float4 t = *reinterpret_cast<const float4*>(bb + hf * 32 + q * 4);
            b1r[q * 4 + 0] = t.x;
            b1r[q * 4 + 1] = t.y;
            b1r[q * 4 + 2] = t.z;
            b1r[q * 4 + 3] = t.w;
          }
          tc::tmem_ld_wait();
          uint32_t pk[16];
#pragma unroll
          for (int e = 0; e < 32; e += 2)
            pk[e >> 1] = tr_pack_bf16(fmaxf(__uint_as_float(v[e]) + b1r[e], 0.f), fmaxf(__uint_as_float(v[e + 1]) + b1r[e + 1], 0.f));
          // bf16 pairs back into tensor memory, over this thread's own (already loaded) fp32 input columns: hidden columns
          // 64 team + 32 hf + [0, 32) -> 32-bit columns 64 team + 16 hf + [0, 16) of the chunk's accumulator buffer
          tc::tmem_st16(ta + hf * 16, pk);
        }
        tc::tmem_st_wait();
        tc::tc_fence_before();
        tc::mbar_arrive(&a2_full[buf]);
      }
      // ---- E2: output columns + b2 -> fp32 staging (two 16 KB boxes per team) -> TMA reduce-add
      tc::mbar_wait(acc2_full, it & 1);                // all GEMM2 of this tile complete: acc2 final
      tc::tc_fence_after();
      // staging boxes: two per team, written only by that team, so the team leader's own bulk-group bookkeeping covers every reuse
      uint8_t* stage = smem + (SM::ST_ALIAS ? SM::A1_OFF + (int)(it % A1B) * SM::A1_BYTES : SM::ST_OFF) + team * 2 * SM::KB_BYTES;
      if (!SM::ST_ALIAS) {
        if (leader) tc::bulk_wait_read<0>();           // the previous tile's reduce-adds have read their staging boxes
        tc::named_bar_sync(bar_id, 128);
      }
      // One box: registers + b2 -> swizzled fp32 staging tile -> TMA reduce-add into the residual
      auto emit = [&](int bx, const uint32_t (&v)[32], uint8_t* sb) {
        const float* bb = sb2 + bx * 32;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const float4 t = *reinterpret_cast<const float4*>(bb + q * 4);
          *reinterpret_cast<float4*>(sb + lr * 128 + (((uint32_t)q ^ sw) << 4)) =
              make_float4(__uint_as_float(v[q * 4 + 0]) + t.x, __uint_as_float(v[q * 4 + 1]) + t.y,
                          __uint_as_float(v[q * 4 + 2]) + t.z, __uint_as_float(v[q * 4 + 3]) + t.w);
        }
        tc::fence_proxy_async_smem();
        tc::named_bar_sync(bar_id, 128);
        if (leader) {
          tc::tma_reduce_add_2d(&tmR, sb, bx * 32, (int)(tile * 128));
          tc::bulk_commit();
        }
      };
      // This team's boxes are bx = team, team + 2, ... (2 at C = 128, 4 at C = 256), two at a time through registers; the
      // accumulator is handed back to the MMA thread as soon as its last columns are in registers, before they are staged.
      constexpr int NBOX = C / 64;
      uint32_t va[32], vb[32];
      tc::tmem_ld32(lane_addr + SM::TMEM_ACC2 + team * 32, va);
      tc::tmem_ld32(lane_addr + SM::TMEM_ACC2 + (team + 2) * 32, vb);
      tc::tmem_ld_wait();
      if (NBOX == 2) {
        tc::tc_fence_before();
        tc::mbar_arrive(acc2_empty);
      }
      emit(team, va, stage);
      emit(team + 2, vb, stage + SM::KB_BYTES);
      if (NBOX == 4) {
        tc::tmem_ld32(lane_addr + SM::TMEM_ACC2 + (team + 4) * 32, va);
        tc::tmem_ld32(lane_addr + SM::TMEM_ACC2 + (team + 6) * 32, vb);
        tc::tmem_ld_wait();
        tc::tc_fence_before();
        tc::mbar_arrive(acc2_empty);
        if (leader) tc::bulk_wait_read<1>();           // the first box has been read by its reduce-add
        tc::named_bar_sync(bar_id, 128);
        emit(team + 4, va, stage);
        if (leader) tc::bulk_wait_read<1>();
        tc::named_bar_sync(bar_id, 128);
        emit(team + 6, vb, stage + SM::KB_BYTES);
      }
      ++it;
    }
    if (leader) tc::bulk_wait<0>();
  } else if (warp < 16) {
    // ============================================================= A1 producers: LayerNorm of fp32 rows
    using LN = LnProd<C>;
    constexpr int RU = LN::ROWS;                       // rows per batch of this warp (4 at C = 256, 8 at C = 128)
    const int pw = warp - 8;
    LN ln;
    ln.init(p.gamma, p.beta, lane);
    uint32_t it = 0;
    for (long tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
      if (!tr_tile_on(tile, p)) continue;
      const uint32_t abuf = it % A1B;
      const long nxt = tile + gridDim.x;
      const bool nxt_on = nxt < p.num_tiles && tr_tile_on(nxt, p);
      tc::mbar_wait(&a1_empty[abuf], ((it / A1B) & 1) ^ 1);
      uint8_t* abase = smem + SM::A1_OFF + abuf * SM::A1_BYTES;
#pragma unroll 1
      for (int r0 = 0; r0 < 16; r0 += RU) {
        // short-distance L2 prefetch of this warp's next batch of rows (first batch of the next active tile after the last)
        if (lane == 0 && (r0 + RU < 16 || nxt_on)) {
          const long r = (r0 + RU < 16 ? tile : nxt) * 128 + pw * 16 + (r0 + RU < 16 ? r0 + RU : 0);
          if (r < p.R) {
            const long n = p.R - r < RU ? p.R - r : RU;
            tc::prefetch_l2_bulk(p.res + r * C, (uint32_t)(n * C * 4));
          }
        }
        const float* rp[LN::PASSES];
        int lr[LN::PASSES];
#pragma unroll
        for (int ps = 0; ps < LN::PASSES; ++ps) {
          lr[ps] = pw * 16 + ln.row_of(r0, ps);
          const long r = tile * 128 + lr[ps];
          rp[ps] = r < p.R ? p.res + r * C : nullptr;
        }
        ln.run(rp, lr, abase);
      }
      tc::fence_proxy_async_smem();
      tc::mbar_arrive(&a1_full[abuf]);
      ++it;
    }
  } else if (warp == 16) {
    // ============================================================= weight tiles, in the MMA thread's consumption order
    if (tc::elect_one()) {
      uint32_t wc = 0;
      auto load = [&](const CUtensorMap* m, int k0, int row0) {
        const uint32_t s = wc % WS;
        tc::mbar_wait(&w_empty[s], ((wc / WS) & 1) ^ 1);
        tc::mbar_arrive_expect_tx(&w_full[s], SM::W_STAGE);
        tc::tma_load_2d(smem + SM::W_OFF + s * SM::W_STAGE, m, &w_full[s], k0, row0);
        ++wc;
      };
      auto g1 = [&](int c) {   // W1^T [4C, C]: rows = hidden columns of the chunk
        for (int kb = 0; kb < KB1; ++kb) load(&tmW1, kb * 64, c * TR_HC);
      };
      auto g2 = [&](int c) {   // W2^T [C, 4C]: rows = output columns, k = hidden columns of the chunk
        for (int kb = 0; kb < 2; ++kb)
          for (int nh = 0; nh < NH; ++nh) load(&tmW2, c * TR_HC + kb * 64, nh * 128);
      };
      for (long tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
        if (!tr_tile_on(tile, p)) continue;
        g1(0);
        for (int c = 1; c < NC; ++c) {
          g1(c);
          g2(c - 1);
        }
        g2(NC - 1);
      }
    }
  } else if (warp == 17) {
    // ============================================================= MMA issue
    if (tc::elect_one()) {
      constexpr uint32_t idesc1 = tc::idesc_f16_f32(128, 128);    // GEMM1: fp16 LayerNorm output x fp16 W1
      constexpr uint32_t idesc2 = tc::idesc_bf16_f32(128, 128);   // GEMM2: bf16 hidden x bf16 W2
      uint32_t wc = 0, c1 = 0, c2 = 0, it = 0;
      const uint32_t acc2 = tmem_base + SM::TMEM_ACC2;
      for (long tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
      if (!tr_tile_on(tile, p)) continue;
        const uint32_t abuf = it % A1B;
        const uint32_t a1_addr = tc::smem_u32(smem + SM::A1_OFF + abuf * SM::A1_BYTES);
        auto gemm1 = [&](int c) {
          // No wait for the buffer: its previous content (chunk c - 2, rectified in place) was the A operand of GEMM2(c - 2),
          // issued by this thread before this GEMM1, and tcgen05.mma operations of one thread execute in issue order.
          const uint32_t buf = c1 & 1;
          const uint32_t d = tmem_base + buf * TR_HC;
#pragma unroll 1
          for (int kb = 0; kb < KB1; ++kb, ++wc) {
            const uint32_t s = wc % WS;
            tc::mbar_wait(&w_full[s], (wc / WS) & 1);
            tc::tc_fence_after();
            const uint64_t a_desc = tc::smem_desc_kmajor<128>(a1_addr + kb * SM::KB_BYTES);
            const uint64_t b_desc = tc::smem_desc_kmajor<128>(tc::smem_u32(smem + SM::W_OFF + s * SM::W_STAGE));
#pragma unroll
            for (int k = 0; k < 4; ++k) tc::mma_bf16(d, a_desc + 2 * k, b_desc + 2 * k, idesc1, (kb | k) != 0);
            tc::mma_commit(&w_empty[s]);
          }
          tc::mma_commit(&acc1_full[buf]);
          ++c1;
          (void)c;
        };
        auto gemm2 = [&](int c) {
          const uint32_t buf = c2 & 1;
          tc::mbar_wait(&a2_full[buf], (c2 >> 1) & 1);
          tc::tc_fence_after();
          const uint32_t a2_t = tmem_base + buf * TR_HC;   // rectified chunk, bf16 pairs: k-block kb at columns 64 kb + [0, 32)
#pragma unroll 1
          for (int kb = 0; kb < 2; ++kb) {
#pragma unroll 1
            for (int nh = 0; nh < NH; ++nh, ++wc) {
              const uint32_t s = wc % WS;
              tc::mbar_wait(&w_full[s], (wc / WS) & 1);
              tc::tc_fence_after();
              const uint64_t b_desc = tc::smem_desc_kmajor<128>(tc::smem_u32(smem + SM::W_OFF + s * SM::W_STAGE));
#pragma unroll
              for (int k = 0; k < 4; ++k)
                tc::mma_bf16_ts(acc2 + nh * 128, a2_t + kb * 64 + k * 8, b_desc + 2 * k, idesc2, (c | kb | k) != 0);
              tc::mma_commit(&w_empty[s]);
            }
          }
          ++c2;
        };
        tc::mbar_wait(&a1_full[abuf], (it / A1B) & 1);
        tc::tc_fence_after();
        gemm1(0);
        for (int c = 1; c < NC; ++c) {
          gemm1(c);
          if (!SM::ST_ALIAS && c == NC - 1) tc::mma_commit(&a1_empty[abuf]);   // every GEMM1 of this tile has been issued: A1 is free when they finish
          if (c == 1) {
            // acc2 of the previous tile must have been drained by E2 before the first GEMM2 overwrites it
            tc::mbar_wait(acc2_empty, (it & 1) ^ 1);
            tc::tc_fence_after();
          }
          gemm2(c - 1);
        }
        gemm2(NC - 1);
        tc::mma_commit(acc2_full);
        ++it;
      }
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 17) tc::tmem_dealloc<512>(tmem_base);
}

// ------------------------------------------------------------------------------------------------
// host
// ------------------------------------------------------------------------------------------------
template <int C>
static int launch_tr(const CUtensorMap& tmW1, const CUtensorMap& tmW2, const CUtensorMap& tmR, const TrParams& p, int num_sms,
                     cudaStream_t st) {
  auto kern = transition_kernel<C>;
  unsigned grid = (unsigned)(p.num_tiles < (long)num_sms ? p.num_tiles : (long)num_sms);
  kern<<<grid, TR_THREADS, TrSmem<C>::TOTAL, st>>>(tmW1, tmW2, tmR, p);
  return 0;
}

template <int C>
static bool configure_tr() {
  cudaError_t e = cudaFuncSetAttribute(transition_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, TrSmem<C>::TOTAL);
  if (e != cudaSuccess) tc_set_error(std::string("cudaFuncSetAttribute(transition): ") + cudaGetErrorString(e));
  return e == cudaSuccess;
}
bool configure_transition_kernels() { return configure_tr<128>() && configure_tr<256>(); }

// w1t: fp16 [4C, C] (K = C contiguous); w2t: bf16 [C, 4C] (K = 4C contiguous); res: fp32 [R, C] updated in place.
int launch_transition_tc(TmaCtx* ctx, float* res, long R, int C, const float* gamma, const float* beta, const void* w1t,
                         const float* b1, const void* w2t, const float* b2, const unsigned char* tile_active, int num_sms,
                         cudaStream_t st) {
  if (C != 128 && C != 256) {
    tc_set_error("transition_tc: C must be 128 or 256");
    return -1;
  }
  TrParams p;
  p.res = res; p.gamma = gamma; p.beta = beta; p.b1 = b1; p.b2 = b2;
  p.R = R;
  p.num_tiles = (R + 127) / 128;
  p.tile_active = tile_active;
  CUtensorMap tmW1, tmW2, tmR;
  {
    uint64_t dims[2] = {(uint64_t)C, (uint64_t)4 * C}, str[1] = {(uint64_t)C * 2};
    uint32_t box[2] = {64, 128};
    if (tma_encode(ctx, &tmW1, w1t, 1, 2, dims, str, box, 128) != 0) return -1;
  }
  {
    uint64_t dims[2] = {(uint64_t)4 * C, (uint64_t)C}, str[1] = {(uint64_t)4 * C * 2};
    uint32_t box[2] = {64, 128};
    if (tma_encode(ctx, &tmW2, w2t, 0, 2, dims, str, box, 128) != 0) return -1;
  }
  {
    uint64_t dims[2] = {(uint64_t)C, (uint64_t)R}, str[1] = {(uint64_t)C * 4};
    uint32_t box[2] = {32, 128};
    if (tma_encode(ctx, &tmR, res, 2, 2, dims, str, box, 128) != 0) return -1;
  }
  return C == 128 ? launch_tr<128>(tmW1, tmW2, tmR, p, num_sms, st) : launch_tr<256>(tmW1, tmW2, tmR, p, num_sms, st);
}

}  // namespace pf
