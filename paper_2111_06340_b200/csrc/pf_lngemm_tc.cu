// Persistent LayerNorm-fused projection GEMM on tcgen05 tensor cores (sm_100a) — every Linear of SURVEY.md App. A whose
// reduction length is one channel dimension (K = c_z = 128 or K = c_m = 256):
//     acc[r, n] = sum_k A[r, k] Wt[n, k],      r = (b, x, y) rows of a [B, D1, D2] grid,
//     A = LayerNorm(fp32 residual rows)  (R4; north_star: "LayerNorm fused into the q/k/v/gate/bias projections")
//         or a 16-bit activation [R, K] fetched by TMA (out-projections, LN_out(t) W_z),
// followed by per-64-column epilogue groups (G2Op): scaled / biased / activated 16-bit row-major stores, gated channel-major
// triangle operands, pair-bias heads, transposed V / outer-product operands, or "residual += (acc + bias) * gate".
//
// One persistent CTA per SM, 18 working warps (20 launched: register re-allocation is per warpgroup of four):
//   warps 0-7   epilogue, two teams of four warps (team t takes the 64-column groups j with j % 2 == t, so one team's TMEM
//               loads / barriers hide behind the other's arithmetic): tcgen05.ld their TMEM lane quarter -> registers ->
//               shared-memory staging tile (one per team) -> ONE TMA store per group: row-major 16-bit (128B swizzle),
//               transposed 16-bit (V^T / outer-product operands, channel-major triangle operands, pair-bias heads: the
//               tile is written to shared memory already transposed, the box is {y, ...}) or a TMA reduce-add into the fp32
//               residual (the add happens at L2)
//   warps 8-15  A producers (a_mode 0): warp-per-row LayerNorm with 128-bit loads and warp-shuffle statistics, several rows in
//               flight per warp, result written as fp16/bf16 straight into the UMMA K-major 128B-swizzle layout
//   warp 16     TMA: weight tiles [256 x 64] through a ring (and the A tile itself in a_mode 1, issued by warp 8)
//   warp 17     TMEM allocation + the single MMA-issuing thread
// The A tile (128 rows x K) stays resident while all N tiles are swept, A is double buffered (the LayerNorm of tile t+1
// overlaps the MMAs / epilogue of tile t) and so is the 128 x 256 fp32 accumulator in TMEM (2 x 256 columns).
// A tile covers XT x YT rows so that every output — also a transposed residual — is one 4-D TMA box {cols, YT, XT, 1}.
#include "pf_internal.h"
#include "pf_device.cuh"
#include "pf_tc.cuh"
#include "pf_lnprod.cuh"

#include <cuda_fp16.h>
#include <string>

namespace pf {

int tma_encode(TmaCtx* ctx, CUtensorMap* out, const void* base, int elem_kind, int rank, const uint64_t* dims,
               const uint64_t* strides_bytes, const uint32_t* box, int swizzle_bytes);

#ifdef PF_G2_TRACE
// Timeline tracing of CTA 0 (experiments only; never defined in the product build): per traced thread a private slot of
// (tag, clock64) pairs written with plain stores (no atomics: ~10 ns per event).
__device__ unsigned long long g2_trace_buf[4 * 8192];
__device__ int g2_trace_nw = 0;   // trace only the launches with this many weight rows (0 = all launches)
#define G2_TRACE_DECL unsigned g2_trc = 0;
#define G2_TRACE(slot, tag)                                                         \
  do {                                                                              \
    if (blockIdx.x == 0 && g2_trc < 4000 && (g2_trace_nw == 0 || g2_trace_nw == p.Nw)) { \
      g2_trace_buf[(slot) * 8192 + 2 * g2_trc] = (tag);                             \
      g2_trace_buf[(slot) * 8192 + 2 * g2_trc + 1] = (unsigned long long)clock64(); \
      ++g2_trc;                                                                     \
    }                                                                               \
  } while (0)
#else
#define G2_TRACE_DECL
#define G2_TRACE(slot, tag)
#endif

#ifdef PF_G2_ABLATE
// Timing experiments only (never defined in the product build; results are wrong while a bit is set):
// 1 no TMA stores / staging waits in the epilogue, 2 epilogue groups skipped entirely, 4 LayerNorm producers read no global memory
__device__ int g2_ablate = 0;
extern "C" void pf_debug_g2_ablate(int v) { cudaMemcpyToSymbol(g2_ablate, &v, sizeof(int)); }
#define G2_ABL(bit) (g2_ablate & (bit))
#else
#define G2_ABL(bit) 0
#endif

constexpr int G2_BN = 256;
constexpr int G2_THREADS = 20 * 32;   // warps 18, 19 only complete the fourth warpgroup (register re-allocation is per warpgroup)
constexpr int G2_EPI_WARPS = 8;
// 20 warps x 96 registers at launch = the CTA's register pool (61440); setmaxnreg moves registers between whole warpgroups
// inside that pool.  LayerNorm-fed kernels: warps 16-19 drop to 40, which lets the eight epilogue warps grow to 120 (the
// LayerNorm producers keep 96: 8 x 32 x (120 + 96) + 4 x 32 x 40 = 60416).  TMA-fed kernels: warps 8-19 drop to 40, the
// epilogue warps grow to 128.  Measured: the epilogue at 96 registers spilled its staging loop (out-projection with gate
// 300 -> 213 us at cfg2 once it had 128).
#ifndef PF_G2_EPI_REGS
#define PF_G2_EPI_REGS 120
#define PF_G2_MISC_REGS 40
#endif
constexpr int G2_EPI_REGS = PF_G2_EPI_REGS, G2_MISC_REGS = PF_G2_MISC_REGS, G2_EPI_REGS_TMA = 128, G2_IDLE_REGS = 40;
constexpr int G2_PROD_WARPS = 8;

struct G2Params {
  int B, D1, D2, XT, YT, yt_shift, ytw_shift, tiles_x_per_b, tiles_y;
  long num_tiles;
  int Nw, n_tiles;
  const float* src;
  int src_transposed;
  const float* gamma;
  const float* beta;
  int op_fmt;
  const float* bias;
  int rowmask;
  const float* seq_mask;
  const float* msa_mask;
  int mask_transposed;
  const __half* gate;
  int ldg;
  bf16* cm_out[2];
  int cm_channels;
  bf16* heads_out;
  int n_heads;
  bf16* vt_out;
  int vt_cols;
  int Lpad;
  const unsigned char* tile_active;
  unsigned swap_mask;
  int has_cms;            // some group is G2_CMS: the epilogue warps publish the tile's row masks once per tile
  int bias_lo, bias_n;    // the bias table holds columns [bias_lo, bias_lo + bias_n); all other columns have zero bias
  G2Op ops[G2_MAX_OPS];
};

template <int K>
struct G2Smem {
  static constexpr int KB = K / 64;
  static constexpr int A_BYTES = 128 * K * 2;
  static constexpr int KB_BYTES = 128 * 128;            // one 64-wide k-block of the A tile
  static constexpr int W_STAGE = G2_BN * 64 * 2;        // 32 KB
  static constexpr int W_STAGES = 2;
  static constexpr int ST_PER_TEAM = (K == 256) ? 1 : 2;   // staging tiles per epilogue team (K = 256 has no room for two)
  static constexpr int A_OFF = 0;
  static constexpr int W_OFF = 2 * A_BYTES;
  static constexpr int ST_OFF = W_OFF + W_STAGES * W_STAGE;
  static constexpr int ST_BYTES = 128 * 128;            // per team of four warps; each warp owns a quarter (32 rows x 128 B)
  static constexpr int STW_BYTES = 32 * 128;
  // fp32 bias table, staged ONCE per CTA: columns [bias_lo, bias_lo + BIAS_FLOATS) of the bias vector, followed by 64 zeros
  // that stand in for every 64-column group outside the table (q, k, v of the attention projections carry no bias)
  static constexpr int BIAS_FLOATS = (K == 256) ? 256 : 768;
  static constexpr int BIAS_OFF = ST_OFF + 2 * ST_PER_TEAM * ST_BYTES;
  static constexpr int RM_OFF = BIAS_OFF + (BIAS_FLOATS + 64) * 4;   // row masks of the current tile, two buffers (G2_CMS)
  static constexpr int RM_BYTES = (K == 128) ? 2 * 128 * 4 : 0;     // only the K = 128 kernels have operand-swapped gated groups
  static constexpr int BAR_OFF = RM_OFF + RM_BYTES;
  static constexpr int TOTAL = BAR_OFF + 192 + 1024;
};

struct TileCoord {
  int b, x0, y0;
};
__device__ __forceinline__ bool tile_on(long t, const G2Params& p) { return !p.tile_active || p.tile_active[t] != 0; }
__device__ __forceinline__ TileCoord tile_coord(long t, const G2Params& p) {
  TileCoord c;
  int ty = (int)(t % p.tiles_y);
  long tx = t / p.tiles_y;
  c.b = (int)(tx / p.tiles_x_per_b);
  c.x0 = (int)(tx - (long)c.b * p.tiles_x_per_b) * p.XT;
  c.y0 = ty * p.YT;
  return c;
}

// sigmoid(x) = 0.5 + 0.5 tanh(x / 2) with the MUFU tanh approximation: one MUFU and two FMA-pipe instructions per value
// (the ex2 + rcp form costs two MUFU; the epilogue warps are the critical path of this kernel).  tanh.approx has a
// relative error of ~2^-11, i.e. <= 2.5e-4 absolute on the gate, which is stored as fp16 (2^-11 relative) anyway.
__device__ __forceinline__ float fast_sigmoid2(float x) {
  float t;
  asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(x * 0.5f));
  return fmaf(t, 0.5f, 0.5f);
}
// 32 consecutive fp32 values from shared memory into registers (eight 128-bit loads).  Epilogue groups fetch their bias this
// way BEFORE the arithmetic: a shared-memory load placed between the staging stores could not be moved across them.
__device__ __forceinline__ void lds32(const float* src, float (&dst)[32]) {
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    const float4 t = *reinterpret_cast<const float4*>(src + q * 4);
    dst[q * 4 + 0] = t.x;
    dst[q * 4 + 1] = t.y;
    dst[q * 4 + 2] = t.z;
    dst[q * 4 + 3] = t.w;
  }
}

__device__ __forceinline__ uint32_t pack16(float a, float b, int fmt) {
  if (fmt) {
    __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&h);
  }
  __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&h);
}


// One 64-column row-major 16-bit output group of one tile row: TMEM -> (scale, bias, activation) -> 128B-swizzled staging row.
template <int ACT, int FMT>
__device__ __forceinline__ void g2_row16_group(uint32_t taddr, uint8_t* srow, const float* bias64, float scale, uint32_t sw) {
#pragma unroll
  for (int hf = 0; hf < 2; ++hf) {
    uint32_t v[32];
    float bb[32];
    tc::tmem_ld32(taddr + hf * 32, v);
    lds32(bias64 + hf * 32, bb);
    tc::tmem_ld_wait();
    uint32_t pk[16];
#pragma unroll
    for (int e = 0; e < 32; e += 2) {
      float x0 = fmaf(__uint_as_float(v[e]), scale, bb[e]), x1 = fmaf(__uint_as_float(v[e + 1]), scale, bb[e + 1]);
      if (ACT == ACT_SIGMOID) {
        x0 = fast_sigmoid2(x0);
        x1 = fast_sigmoid2(x1);
      } else if (ACT == ACT_RELU) {
        x0 = fmaxf(x0, 0.f);
        x1 = fmaxf(x1, 0.f);
      }
      pk[e >> 1] = pack16(x0, x1, FMT);
    }
#pragma unroll
    for (int c = 0; c < 4; ++c)
      *reinterpret_cast<uint4*>(srow + (((uint32_t)(hf * 4 + c) ^ sw) << 4)) =
          make_uint4(pk[c * 4], pk[c * 4 + 1], pk[c * 4 + 2], pk[c * 4 + 3]);
  }
}

// The same for a group without bias and activation (q, k of the attention projections): both TMEM loads are issued before
// the single wait, and the arithmetic is one multiply (q: log2(e)/sqrt(d)) or nothing (k) per value before the conversion.
template <int FMT>
__device__ __forceinline__ void g2_row16_plain(uint32_t taddr, uint8_t* srow, float scale, uint32_t sw) {
  uint32_t v[2][32];
  tc::tmem_ld32(taddr, v[0]);
  tc::tmem_ld32(taddr + 32, v[1]);
  tc::tmem_ld_wait();
  const bool scaled = scale != 1.0f;
#pragma unroll
  for (int hf = 0; hf < 2; ++hf) {
    uint32_t pk[16];
#pragma unroll
    for (int e = 0; e < 32; e += 2) {
      float x0 = __uint_as_float(v[hf][e]), x1 = __uint_as_float(v[hf][e + 1]);
      if (scaled) {
        x0 *= scale;
        x1 *= scale;
      }
      pk[e >> 1] = pack16(x0, x1, FMT);
    }
#pragma unroll
    for (int c = 0; c < 4; ++c)
      *reinterpret_cast<uint4*>(srow + (((uint32_t)(hf * 4 + c) ^ sw) << 4)) =
          make_uint4(pk[c * 4], pk[c * 4 + 1], pk[c * 4 + 2], pk[c * 4 + 3]);
  }
}

// Sigmoid gate stored as fp16: the pre-activation is rounded to fp16 pairs first and the sigmoid is evaluated on the
// pair, sigmoid(x) = 0.5 + 0.5 tanh(x / 2) with tanh.approx.f16x2 — one MUFU per TWO values and the result is already the
// packed fp16 pair that is stored (per value: 1 FFMA + 2.5 half-rate-free packed ops instead of 4.5 fp32 ops + 1 MUFU).
// The gate is a number in [0, 1] kept in fp16 anyway; the extra error of the fp16 evaluation is ~5e-4 absolute.
template <int FMT>
__device__ __forceinline__ void g2_row16_gate(uint32_t taddr, uint8_t* srow, const float* bias64, float scale, uint32_t sw) {
  static_assert(FMT == 1, "the packed gate path stores fp16");
  const __half2 half_h = __floats2half2_rn(0.5f, 0.5f);
#pragma unroll
  for (int hf = 0; hf < 2; ++hf) {
    uint32_t v[32];
    float bb[32];
    tc::tmem_ld32(taddr + hf * 32, v);
    lds32(bias64 + hf * 32, bb);
    tc::tmem_ld_wait();
    uint32_t pk[16];
#pragma unroll
    for (int e = 0; e < 32; e += 2) {
      const float x0 = fmaf(__uint_as_float(v[e]), scale, bb[e]), x1 = fmaf(__uint_as_float(v[e + 1]), scale, bb[e + 1]);
      __half2 h = __hmul2(__floats2half2_rn(x0, x1), half_h);
      uint32_t hu = *reinterpret_cast<uint32_t*>(&h), tu;
      asm("tanh.approx.f16x2 %0, %1;" : "=r"(tu) : "r"(hu));
      __half2 r = __hfma2(*reinterpret_cast<__half2*>(&tu), half_h, half_h);
      pk[e >> 1] = *reinterpret_cast<uint32_t*>(&r);
    }
#pragma unroll
    for (int c = 0; c < 4; ++c)
      *reinterpret_cast<uint4*>(srow + (((uint32_t)(hf * 4 + c) ^ sw) << 4)) =
          make_uint4(pk[c * 4], pk[c * 4 + 1], pk[c * 4 + 2], pk[c * 4 + 3]);
  }
}

template <int K, int AMODE>
__global__ void __launch_bounds__(G2_THREADS, 1)
gemm2_kernel(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmA,
             const __grid_constant__ CUtensorMap tmO0, const __grid_constant__ CUtensorMap tmT0,
             const __grid_constant__ CUtensorMap tmT1, const __grid_constant__ CUtensorMap tmH,
             const __grid_constant__ CUtensorMap tmR, const __grid_constant__ CUtensorMap tmVS,
             const __grid_constant__ G2Params p) {
  using SM = G2Smem<K>;
  constexpr int KB = SM::KB;
  constexpr int WS = SM::W_STAGES;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = tc::align_smem_1024(smem_raw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::BAR_OFF);
  uint64_t* a_full = bars;             // [2]
  uint64_t* a_empty = bars + 2;        // [2]
  uint64_t* w_full = bars + 4;         // [WS]
  uint64_t* w_empty = w_full + WS;     // [WS]
  uint64_t* acc_full = w_empty + WS;   // [2]
  uint64_t* acc_empty = acc_full + 2;  // [2]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  G2_TRACE_DECL

  if (warp == 16 && lane == 0) {
    tc::prefetch_tmap(&tmW);
    if (AMODE == 1) tc::prefetch_tmap(&tmA);
    tc::prefetch_tmap(&tmO0);
    tc::prefetch_tmap(&tmT0);
    tc::prefetch_tmap(&tmT1);
    tc::prefetch_tmap(&tmH);
    tc::prefetch_tmap(&tmR);
    tc::prefetch_tmap(&tmVS);
    for (int i = 0; i < 2; ++i) {
      tc::mbar_init(&a_full[i], AMODE == 0 ? G2_PROD_WARPS * 32 : 1);
      tc::mbar_init(&a_empty[i], 1);
      tc::mbar_init(&acc_full[i], 1);
      tc::mbar_init(&acc_empty[i], G2_EPI_WARPS * 32);
    }
    for (int i = 0; i < WS; ++i) {
      tc::mbar_init(&w_full[i], 1);
      tc::mbar_init(&w_empty[i], 1);
    }
    tc::fence_barrier_init();
  }
  if (warp == 17) tc::tmem_alloc<512>(tmem_slot);
  for (int i = threadIdx.x; i < SM::BIAS_FLOATS + 64; i += G2_THREADS)
    reinterpret_cast<float*>(smem + SM::BIAS_OFF)[i] = (p.bias && i < p.bias_n) ? __ldg(p.bias + p.bias_lo + i) : 0.f;
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp >= 16) {   // one site for the whole fourth warpgroup (warps 18, 19 have no other work)
    if (AMODE == 0) tc::reg_dealloc<G2_MISC_REGS>();
    else tc::reg_dealloc<G2_IDLE_REGS>();
  }
  if (warp < G2_EPI_WARPS) {
    if (AMODE == 0) tc::reg_alloc<G2_EPI_REGS>();
    else tc::reg_alloc<G2_EPI_REGS_TMA>();
    // =========================================================== epilogue: eight free-running warps.  Warp w owns the 32 tile
    // rows of TMEM lane quarter w % 4 and the 64-column groups j with j % 2 == w / 4; it stages its 32 x 128 B piece in its
    // own shared-memory tile and issues its own TMA store, so no barrier couples it to any other warp.
    const int team = warp >> 2, quarter = warp & 3;
    const int lr = quarter * 32 + lane;                // tile row = TMEM lane
    const bool leader = lane == 0;
    const int xl = lr >> p.yt_shift, yl = lr & (p.YT - 1);
    const int xw0 = (quarter * 32) >> p.yt_shift, yw0 = (quarter * 32) & (p.YT - 1);   // first row of this warp in the tile
    const int xlw = lane >> p.ytw_shift, ylw = lane & ((1 << p.ytw_shift) - 1);         // this row inside the warp's box
    const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
    constexpr int NST = SM::ST_PER_TEAM;
    uint8_t* const sb_team = smem + SM::ST_OFF + (team * 4 + quarter) * NST * SM::STW_BYTES;   // this warp's staging tile(s)
    uint32_t gcnt = 0;                                  // staging steps of this warp so far
    uint8_t* sb = sb_team;
    bf16* sb16 = reinterpret_cast<bf16*>(sb);
    const float* const sbias_tab = reinterpret_cast<const float*>(smem + SM::BIAS_OFF);
    const uint32_t sw = (uint32_t)(lr & 7);
    uint32_t ac = 0;                                   // accumulator buffers consumed so far
    uint32_t tcount = 0;                               // tiles processed so far
    for (long tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
      if (!tile_on(tile, p)) continue;
      const TileCoord tcd = tile_coord(tile, p);
      const int x = tcd.x0 + xl, y = tcd.y0 + yl;
      const bool valid = x < p.D1 && y < p.D2;
      float mask = 1.0f;
      if (valid && p.rowmask == RM_MSA) {
        mask = p.mask_transposed ? p.msa_mask[(long)tcd.b * p.D2 + y] * p.seq_mask[(long)tcd.b * p.D1 + x]
                                 : p.msa_mask[(long)tcd.b * p.D1 + x] * p.seq_mask[(long)tcd.b * p.D2 + y];
      } else if (valid && p.rowmask == RM_PAIR) {
        mask = p.seq_mask[(long)tcd.b * p.D1 + x] * p.seq_mask[(long)tcd.b * p.D2 + y];
      }
      const long grow = ((long)tcd.b * p.D1 + x) * p.D2 + y;   // GEMM row index (gate rows)
      float* rmask = reinterpret_cast<float*>(smem + SM::RM_OFF) + (tcount & 1) * 128;
      if (SM::RM_BYTES && p.has_cms) {
        // operand-swapped gated groups index the row mask by TMEM column: publish this tile's 128 masks (the buffer of two
        // tiles ago is free: every warp passed the previous tile's barrier after its last read of it)
        if (team == 0) rmask[lr] = valid ? mask : 0.f;
        tc::named_bar_sync(3, G2_EPI_WARPS * 32);
      }
      ++tcount;
      for (int nt = 0; nt < p.n_tiles; ++nt, ++ac) {
        const uint32_t buf = ac & 1;
        // this warp's two groups of the window: their descriptors are fetched (indexed constant loads) BEFORE waiting for the
        // accumulator, so that latency is off the critical path
        const G2Op op_a = p.ops[nt * 4 + team], op_b = p.ops[nt * 4 + team + 2];
        if (lane == 0 && quarter == 0) G2_TRACE(team, 0x100 + 0);
        tc::mbar_wait(&acc_full[buf], (ac >> 1) & 1);
        tc::tc_fence_after();
        if (lane == 0 && quarter == 0) G2_TRACE(team, 0x100 + 1);
        const uint32_t tacc = lane_addr + buf * G2_BN;
#pragma unroll 1
        for (int j = team; j < 4; j += 2) {
          const G2Op& op = (j == team) ? op_a : op_b;
          const int kind = op.kind;
          if (kind == G2_SKIP || G2_ABL(2)) continue;
          if (lane == 0 && quarter == 0) G2_TRACE(team, 0x100 + 3);
          // this group's 64 bias values: inside the table, or the zero pad behind it
          const int bcol = nt * G2_BN + j * 64 - p.bias_lo;
          const float* const sbias = sbias_tab + ((bcol >= 0 && bcol + 64 <= p.bias_n) ? bcol : SM::BIAS_FLOATS);
          const int bcol2 = bcol + 128;   // gate partner of a dual group
          const float* const sbias2 = sbias_tab + ((bcol2 >= 0 && bcol2 + 64 <= p.bias_n) ? bcol2 : SM::BIAS_FLOATS);
          if (kind == G2_ROW16) {
            sb = sb_team + (gcnt++ % NST) * SM::STW_BYTES;
            sb16 = reinterpret_cast<bf16*>(sb);
            if (leader && quarter == 0) G2_TRACE(team, 0x120);
            if (leader && !G2_ABL(1)) tc::bulk_wait_read<NST - 1>();
            __syncwarp();
            if (leader && quarter == 0) G2_TRACE(team, 0x121);
            {
              const float scale = op.scale;
              const uint32_t ta = tacc + j * 64;
              uint8_t* srow = sb + lane * 128;
              const float* b64 = sbias;
              if (op.act == ACT_SIGMOID) {
                if (op.fmt) g2_row16_gate<1>(ta, srow, b64, scale, sw);
                else g2_row16_group<ACT_SIGMOID, 0>(ta, srow, b64, scale, sw);
              } else if (op.act == ACT_RELU) {
                if (op.fmt) g2_row16_group<ACT_RELU, 1>(ta, srow, b64, scale, sw);
                else g2_row16_group<ACT_RELU, 0>(ta, srow, b64, scale, sw);
              } else if (b64 == sbias_tab + SM::BIAS_FLOATS) {   // no bias: the zero pad
                if (op.fmt) g2_row16_plain<1>(ta, srow, scale, sw);
                else g2_row16_plain<0>(ta, srow, scale, sw);
              } else {
                if (op.fmt) g2_row16_group<ACT_NONE, 1>(ta, srow, b64, scale, sw);
                else g2_row16_group<ACT_NONE, 0>(ta, srow, b64, scale, sw);
              }
            }
            if (leader && quarter == 0) G2_TRACE(team, 0x122);
            tc::fence_proxy_async_smem();
            __syncwarp();
            if (leader && quarter == 0) G2_TRACE(team, 0x123);
            if (leader && !G2_ABL(1)) {
              tc::tma_store_4d(&tmO0, sb, op.dst_col, tcd.y0 + yw0, tcd.x0 + xw0, tcd.b);
              tc::bulk_commit();
            }
            if (leader && quarter == 0) G2_TRACE(team, 0x124);
          } else if (kind == G2_RESID) {
#pragma unroll 1
            for (int hf = 0; hf < 2; ++hf) {
              sb = sb_team + (gcnt++ % NST) * SM::STW_BYTES;
            sb16 = reinterpret_cast<bf16*>(sb);
            if (leader && !G2_ABL(1)) tc::bulk_wait_read<NST - 1>();
              __syncwarp();
              uint32_t v[32];
              float bb[32];
              tc::tmem_ld32(tacc + j * 64 + hf * 32, v);
              lds32(sbias + hf * 32, bb);
              const __half* gp = (p.gate && valid) ? p.gate + grow * p.ldg + op.dst_col + hf * 32 : nullptr;
              uint4 gu[4];
              if (gp) {
#pragma unroll
                for (int c = 0; c < 4; ++c) gu[c] = *reinterpret_cast<const uint4*>(gp + c * 8);
              }
              tc::tmem_ld_wait();
              float f[32];
#pragma unroll
              for (int e = 0; e < 32; ++e) f[e] = __uint_as_float(v[e]) + bb[e];
              if (gp) {
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                  const uint32_t gw[4] = {gu[c].x, gu[c].y, gu[c].z, gu[c].w};
#pragma unroll
                  for (int e = 0; e < 4; ++e) {
                    const __half2 g2 = *reinterpret_cast<const __half2*>(&gw[e]);
                    f[c * 8 + 2 * e] *= __low2float(g2);
                    f[c * 8 + 2 * e + 1] *= __high2float(g2);
                  }
                }
              }
#pragma unroll
              for (int c = 0; c < 8; ++c)
                *reinterpret_cast<float4*>(sb + lane * 128 + (((uint32_t)c ^ sw) << 4)) =
                    make_float4(f[c * 4], f[c * 4 + 1], f[c * 4 + 2], f[c * 4 + 3]);
              tc::fence_proxy_async_smem();
              __syncwarp();
              if (leader && !G2_ABL(1)) {
                tc::tma_reduce_add_4d(&tmR, sb, op.dst_col + hf * 32, tcd.y0 + yw0, tcd.x0 + xw0, tcd.b);
                tc::bulk_commit();
              }
            }
          } else if (kind == G2_CM_DUAL) {
            // 64 channels of a gated, masked triangle operand, channel-major: staging tile [channel][x][y] (2-byte stores of
            // consecutive lanes are consecutive in shared memory), one TMA store with box {YT, XT, 64, 1}
            sb = sb_team + (gcnt++ % NST) * SM::STW_BYTES;
            sb16 = reinterpret_cast<bf16*>(sb);
            if (leader && !G2_ABL(1)) tc::bulk_wait_read<NST - 1>();
            __syncwarp();
#pragma unroll 1
            for (int hf = 0; hf < 2; ++hf) {
              uint32_t v[32], g[32];
              float bp[32], bg[32];
              tc::tmem_ld32(tacc + j * 64 + hf * 32, v);
              tc::tmem_ld32(tacc + 128 + j * 64 + hf * 32, g);
              lds32(sbias + hf * 32, bp);
              lds32(sbias2 + hf * 32, bg);
              tc::tmem_ld_wait();
              __half r[32];   // triangle operands are fp16 (R17, round 2)
#pragma unroll
              for (int e = 0; e < 32; ++e) {
                const float pv = __uint_as_float(v[e]) + bp[e];
                const float gv = fast_sigmoid2(__uint_as_float(g[e]) + bg[e]);
                r[e] = __float2half_rn(mask * gv * pv);
              }
#pragma unroll
              for (int e = 0; e < 32; ++e) reinterpret_cast<__half*>(sb16)[(hf * 32 + e) * 32 + lane] = r[e];
            }
            tc::fence_proxy_async_smem();
            __syncwarp();
            if (leader) {
              tc::tma_store_4d(op.map ? &tmT1 : &tmT0, sb, tcd.y0 + yw0, tcd.x0 + xw0, op.dst_col, tcd.b);
              tc::bulk_commit();
            }
          } else if (kind == G2_HEADS) {
            // pair-bias heads [b, head, x, y]: staging tile [head][x][y], box {YT, XT, n_heads, 1}
            sb = sb_team + (gcnt++ % NST) * SM::STW_BYTES;
            sb16 = reinterpret_cast<bf16*>(sb);
            if (leader && !G2_ABL(1)) tc::bulk_wait_read<NST - 1>();
            __syncwarp();
            uint32_t v[32];
            tc::tmem_ld32(tacc + j * 64, v);
            tc::tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 8; ++e)
              if (e < op.ncols) reinterpret_cast<__half*>(sb16)[e * 32 + lane] = __float2half_rn(__uint_as_float(v[e]) * op.scale);   // fp16 (R17)
            tc::fence_proxy_async_smem();
            __syncwarp();
            if (leader) {
              tc::tma_store_4d(&tmH, sb, tcd.y0 + yw0, tcd.x0 + xw0, op.dst_col, tcd.b);
              tc::bulk_commit();
            }
          } else if (kind == G2_CMS) {
            // gated, masked triangle operand out of two operand-swapped halves (p | gate): this thread owns channel
            // 32 quarter + lane and the 64 tile rows [64 j, +64) -> 128-byte staging row -> TMA store {64 y, 1 x, 32 channels}
            sb = sb_team + (gcnt++ % NST) * SM::STW_BYTES;
            const int ch = quarter * 32 + lane;
            const int wcol = nt * G2_BN - p.bias_lo;   // the whole window's bias is in the table (checked by the launcher)
            const float bpv = sbias_tab[wcol + ch], bgv = sbias_tab[wcol + 128 + ch];
            if (leader && !G2_ABL(1)) tc::bulk_wait_read<NST - 1>();
            __syncwarp();
#pragma unroll 1
            for (int hf = 0; hf < 2; ++hf) {
              uint32_t v[32], g[32];
              float mk[32];
              tc::tmem_ld32(tacc + j * 64 + hf * 32, v);
              tc::tmem_ld32(tacc + 128 + j * 64 + hf * 32, g);
              lds32(rmask + j * 64 + hf * 32, mk);
              tc::tmem_ld_wait();
              uint32_t pk[16];
#pragma unroll
              for (int e = 0; e < 32; e += 2) {
                const float o0 = mk[e] * fast_sigmoid2(__uint_as_float(g[e]) + bgv) * (__uint_as_float(v[e]) + bpv);
                const float o1 = mk[e + 1] * fast_sigmoid2(__uint_as_float(g[e + 1]) + bgv) * (__uint_as_float(v[e + 1]) + bpv);
                pk[e >> 1] = pack16(o0, o1, 1);   // triangle operands are fp16 (R17, round 2)
              }
#pragma unroll
              for (int c = 0; c < 4; ++c)
                *reinterpret_cast<uint4*>(sb + lane * 128 + (((uint32_t)(hf * 4 + c) ^ sw) << 4)) =
                    make_uint4(pk[c * 4], pk[c * 4 + 1], pk[c * 4 + 2], pk[c * 4 + 3]);
            }
            tc::fence_proxy_async_smem();
            __syncwarp();
            if (leader && !G2_ABL(1)) {
              const int r0 = j * 64;   // first tile row of this group
              tc::tma_store_4d(op.map ? &tmT1 : &tmT0, sb, tcd.y0 + (r0 & (p.YT - 1)), tcd.x0 + (r0 >> p.yt_shift),
                               op.dst_col + quarter * 32, tcd.b);
              tc::bulk_commit();
            }
          } else if (kind == G2_VTS) {
            // operand-swapped half-window: this thread owns output column (channel) 32 quarter + lane of the half and reads 64
            // consecutive tile rows from TMEM: convert, stage as a 128-byte row, one TMA store {64 y, 32 channels}
            sb = sb_team + (gcnt++ % NST) * SM::STW_BYTES;
            if (leader && !G2_ABL(1)) tc::bulk_wait_read<NST - 1>();
            __syncwarp();
            g2_row16_plain<0>(tacc + j * 64, sb + lane * 128, 1.0f, sw);
            tc::fence_proxy_async_smem();
            __syncwarp();
            if (leader && !G2_ABL(1)) {
              const int r0 = (j & 1) * 64;   // first tile row of this group
              tc::tma_store_4d(&tmVS, sb, tcd.y0 + (r0 & (p.YT - 1)), op.dst_col + quarter * 32, tcd.x0 + (r0 >> p.yt_shift), tcd.b);
              tc::bulk_commit();
            }
          } else {   // G2_VT
            // 64 columns written transposed, [(b, x), column, y]: staging tile [x][column][y], box {YT, 64, XT, 1}
            sb = sb_team + (gcnt++ % NST) * SM::STW_BYTES;
            sb16 = reinterpret_cast<bf16*>(sb);
            if (leader && !G2_ABL(1)) tc::bulk_wait_read<NST - 1>();
            __syncwarp();
            const float mk = op.masked ? mask : 1.0f;
            bf16* dst = sb16 + ((xlw * 64) << p.ytw_shift) + ylw;
            if (!op.masked && sbias == sbias_tab + SM::BIAS_FLOATS) {
              // V^T of the attention projections: no bias, no mask -> convert and store only
#pragma unroll 1
              for (int hf = 0; hf < 2; ++hf) {
                uint32_t v[32];
                tc::tmem_ld32(tacc + j * 64 + hf * 32, v);
                tc::tmem_ld_wait();
#pragma unroll
                for (int e = 0; e < 32; ++e) dst[(hf * 32 + e) << p.ytw_shift] = __float2bfloat16_rn(__uint_as_float(v[e]));
              }
            } else {
#pragma unroll 1
              for (int hf = 0; hf < 2; ++hf) {
                uint32_t v[32];
                float bb[32];
                tc::tmem_ld32(tacc + j * 64 + hf * 32, v);
                lds32(sbias + hf * 32, bb);
                tc::tmem_ld_wait();
                uint16_t r[32];   // op.fmt: 0 bf16, 1 fp16 (the outer-product operands, R17 round 2)
#pragma unroll
                for (int e = 0; e < 32; ++e) {
                  const float val = (__uint_as_float(v[e]) + bb[e]) * mk;
                  r[e] = op.fmt ? __half_as_ushort(__float2half_rn(val)) : __bfloat16_as_ushort(__float2bfloat16_rn(val));
                }
#pragma unroll
                for (int e = 0; e < 32; ++e) reinterpret_cast<uint16_t*>(dst)[(hf * 32 + e) << p.ytw_shift] = r[e];
              }
            }
            tc::fence_proxy_async_smem();
            __syncwarp();
            if (leader) {
              tc::tma_store_4d(&tmT0, sb, tcd.y0 + yw0, op.dst_col, tcd.x0 + xw0, tcd.b);
              tc::bulk_commit();
            }
          }
        }
        tc::tc_fence_before();
        tc::mbar_arrive(&acc_empty[buf]);
        if (lane == 0 && quarter == 0) G2_TRACE(team, 0x100 + 2);
      }
    }
    if (leader) tc::bulk_wait<0>();
  } else if (warp < 16) {
    if (AMODE == 0) {
      // ========================================================= A producers: LayerNorm of gathered fp32 rows
      using LN = LnProd<K>;
      constexpr int RU = LN::ROWS;                     // rows per batch of this warp (4 at K = 256, 8 at K = 128)
      const int pw = warp - 8;
      LN ln;
      ln.init(p.gamma, p.beta, lane);
      auto src_row = [&](const TileCoord& c, int lr) -> const float* {
        const int x = c.x0 + (lr >> p.yt_shift), y = c.y0 + (lr & (p.YT - 1));
        if (x >= p.D1 || y >= p.D2) return nullptr;
        const long srow = p.src_transposed ? ((long)c.b * p.D2 + y) * p.D1 + x : ((long)c.b * p.D1 + x) * p.D2 + y;
        return p.src + srow * K;
      };
      uint32_t it = 0;
      for (long tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
        if (!tile_on(tile, p)) continue;
        const uint32_t abuf = it & 1;
        // (A bulk L2 prefetch of the next batch of rows used to sit here; once the epilogue stopped spilling it measured as a
        // small loss — the 128 per-row prefetch operations per tile compete with the weight loads and the stores in the TMA queue.)
        if (lane == 0 && pw == 0) G2_TRACE(2, 0x200);
        tc::mbar_wait(&a_empty[abuf], ((it >> 1) & 1) ^ 1);
        if (lane == 0 && pw == 0) G2_TRACE(2, 0x201);
        const TileCoord tcd = tile_coord(tile, p);
        uint8_t* abase = smem + SM::A_OFF + abuf * SM::A_BYTES;
#pragma unroll 1
        for (int r0 = 0; r0 < 16; r0 += RU) {
          const float* rp[LN::PASSES];
          int lr[LN::PASSES];
#pragma unroll
          for (int ps = 0; ps < LN::PASSES; ++ps) {
            lr[ps] = pw * 16 + ln.row_of(r0, ps);
            rp[ps] = G2_ABL(4) ? nullptr : src_row(tcd, lr[ps]);
          }
          ln.run(rp, lr, abase);
        }
        tc::fence_proxy_async_smem();
        tc::mbar_arrive(&a_full[abuf]);
        if (lane == 0 && pw == 0) G2_TRACE(2, 0x202);
        ++it;
      }
    } else {
      tc::reg_dealloc<G2_IDLE_REGS>();
      // ========================================================= A by TMA (a_mode 1)
      if (warp == 8 && tc::elect_one()) {
        uint32_t it = 0;
        for (long tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
          if (!tile_on(tile, p)) continue;
          const uint32_t abuf = it & 1;
          tc::mbar_wait(&a_empty[abuf], ((it >> 1) & 1) ^ 1);
          const TileCoord tcd = tile_coord(tile, p);
          uint8_t* abase = smem + SM::A_OFF + abuf * SM::A_BYTES;
          tc::mbar_arrive_expect_tx(&a_full[abuf], SM::A_BYTES);
#pragma unroll
          for (int kb = 0; kb < KB; ++kb)
            tc::tma_load_4d(abase + kb * SM::KB_BYTES, &tmA, &a_full[abuf], kb * 64, tcd.y0, tcd.x0, tcd.b);
          ++it;
        }
      }
    }
  } else if (warp == 16) {
    // ============================================================= weight tiles
    if (tc::elect_one()) {
      uint32_t wc = 0;
      for (long tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
        if (!tile_on(tile, p)) continue;
        for (int nt = 0; nt < p.n_tiles; ++nt) {
#pragma unroll 1
          for (int kb = 0; kb < KB; ++kb, ++wc) {
            const uint32_t s = wc % WS;
            tc::mbar_wait(&w_empty[s], ((wc / WS) & 1) ^ 1);
            tc::mbar_arrive_expect_tx(&w_full[s], SM::W_STAGE);
            tc::tma_load_2d(smem + SM::W_OFF + s * SM::W_STAGE, &tmW, &w_full[s], kb * 64, nt * G2_BN);
          }
        }
      }
    }
  } else if (warp == 17) {
    // ============================================================= MMA issue
    if (tc::elect_one()) {
      uint32_t it = 0, wc = 0, ac = 0;
      for (long tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
        if (!tile_on(tile, p)) continue;
        const uint32_t abuf = it & 1;
        G2_TRACE(3, 0x300);
        tc::mbar_wait(&a_full[abuf], (it >> 1) & 1);
        tc::tc_fence_after();
        G2_TRACE(3, 0x301);
        const uint32_t a_addr = tc::smem_u32(smem + SM::A_OFF + abuf * SM::A_BYTES);
        for (int nt = 0; nt < p.n_tiles; ++nt, ++ac) {
          const uint32_t buf = ac & 1;
          G2_TRACE(3, 0x302);
          tc::mbar_wait(&acc_empty[buf], ((ac >> 1) & 1) ^ 1);
          tc::tc_fence_after();
          G2_TRACE(3, 0x303);
          int n_eff = p.Nw - nt * G2_BN;
          n_eff = n_eff >= G2_BN ? G2_BN : ((n_eff + 15) & ~15);
          const uint32_t idesc = p.op_fmt ? tc::idesc_f16_f32(128, n_eff) : tc::idesc_bf16_f32(128, n_eff);
          const uint32_t d_tmem = tmem_base + buf * G2_BN;
          const unsigned swp = (p.swap_mask >> (2 * nt)) & 3u;
          // per 128-column half when a half of this window is operand-swapped
          const int nh0 = n_eff < 128 ? n_eff : 128, nh1 = n_eff - 128;
          const uint32_t idesc_sw = p.op_fmt ? tc::idesc_f16_f32(128, 128) : tc::idesc_bf16_f32(128, 128);
#pragma unroll 1
          for (int kb = 0; kb < KB; ++kb, ++wc) {
            const uint32_t s = wc % WS;
            tc::mbar_wait(&w_full[s], (wc / WS) & 1);
            tc::tc_fence_after();
            const uint64_t a_desc = tc::smem_desc_kmajor<128>(a_addr + kb * SM::KB_BYTES);
            const uint32_t w_addr = tc::smem_u32(smem + SM::W_OFF + s * SM::W_STAGE);
            const uint64_t b_desc = tc::smem_desc_kmajor<128>(w_addr);
            if (swp == 0) {
#pragma unroll
              for (int k = 0; k < 4; ++k) tc::mma_bf16(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | k) != 0);
            } else {
#pragma unroll 1
              for (int hh = 0; hh < 2; ++hh) {
                const int nh = hh ? nh1 : nh0;
                if (nh <= 0) continue;
                const uint64_t wh_desc = tc::smem_desc_kmajor<128>(w_addr + hh * (128 * 128));   // weight rows [128 hh, +128)
                if ((swp >> hh) & 1) {   // D[out column, tile row] = W_half (M side) x A tile (N side)
#pragma unroll
                  for (int k = 0; k < 4; ++k)
                    tc::mma_bf16(d_tmem + hh * 128, wh_desc + 2 * k, a_desc + 2 * k, idesc_sw, (kb | k) != 0);
                } else {
                  const uint32_t idh = p.op_fmt ? tc::idesc_f16_f32(128, nh) : tc::idesc_bf16_f32(128, nh);
#pragma unroll
                  for (int k = 0; k < 4; ++k)
                    tc::mma_bf16(d_tmem + hh * 128, a_desc + 2 * k, wh_desc + 2 * k, idh, (kb | k) != 0);
                }
              }
            }
            tc::mma_commit(&w_empty[s]);
          }
          tc::mma_commit(&acc_full[buf]);
          G2_TRACE(3, 0x304);
        }
        tc::mma_commit(&a_empty[abuf]);
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
template <int K, int AMODE>
static int launch_g2(const CUtensorMap& tmW, const CUtensorMap& tmA, const CUtensorMap& tmO0, const CUtensorMap& tmT0,
                     const CUtensorMap& tmT1, const CUtensorMap& tmH, const CUtensorMap& tmR, const CUtensorMap& tmVS,
                     const G2Params& p, int num_sms, cudaStream_t st) {
  auto kern = gemm2_kernel<K, AMODE>;
  unsigned grid = (unsigned)(p.num_tiles < (long)num_sms ? p.num_tiles : (long)num_sms);
  kern<<<grid, G2_THREADS, G2Smem<K>::TOTAL, st>>>(tmW, tmA, tmO0, tmT0, tmT1, tmH, tmR, tmVS, p);
  return 0;
}

// Per-device kernel attributes (dynamic shared memory above 48 KB), set once per handle at create time on the handle's device.
template <int K, int AMODE>
static bool configure_g2() {
  cudaError_t e = cudaFuncSetAttribute(gemm2_kernel<K, AMODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, G2Smem<K>::TOTAL);
  if (e != cudaSuccess) tc_set_error(std::string("cudaFuncSetAttribute(gemm2): ") + cudaGetErrorString(e));
  return e == cudaSuccess;
}
bool configure_gemm2_kernels() {
  return configure_g2<128, 0>() && configure_g2<128, 1>() && configure_g2<256, 0>() && configure_g2<256, 1>() &&
         configure_g2<64, 0>();
}

#ifdef PF_G2_TRACE
extern "C" void pf_debug_g2_trace_select(int nw) { cudaMemcpyToSymbol(g2_trace_nw, &nw, sizeof(int)); }
extern "C" int pf_debug_g2_trace(unsigned long long* out, int reset) {
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(out, g2_trace_buf, sizeof(g2_trace_buf));
  if (reset) {
    static unsigned long long zeros[4 * 8192];
    cudaMemcpyToSymbol(g2_trace_buf, zeros, sizeof(zeros));
  }
  return 4 * 8192;
}
#endif

int launch_gemm2(TmaCtx* ctx, const G2Desc& d, int num_sms, cudaStream_t st) {
  if (d.K != 128 && d.K != 256 && !(d.K == 64 && d.a_mode == 0)) {
    tc_set_error("gemm2: K must be 128 or 256 (or 64 for a LayerNorm-fed GEMM: the extra-MSA stack)");
    return -1;
  }
  G2Params p;
  memset(&p, 0, sizeof(p));
  p.B = d.B; p.D1 = d.D1; p.D2 = d.D2;
  p.YT = g2_pick_yt(d.D2);
  p.XT = 128 / p.YT;
  p.yt_shift = 0;
  while ((1 << p.yt_shift) < p.YT) ++p.yt_shift;
  p.tiles_y = (d.D2 + p.YT - 1) / p.YT;
  p.tiles_x_per_b = (d.D1 + p.XT - 1) / p.XT;
  p.num_tiles = (long)d.B * p.tiles_x_per_b * p.tiles_y;
  p.Nw = d.Nw;
  p.n_tiles = (d.Nw + G2_BN - 1) / G2_BN;
  if (p.n_tiles * 4 > G2_MAX_OPS || d.n_ops > G2_MAX_OPS) {
    tc_set_error("gemm2: too many output columns");
    return -1;
  }
  p.src = d.src; p.src_transposed = d.src_transposed; p.gamma = d.gamma; p.beta = d.beta;
  p.op_fmt = d.op_fmt;
  p.bias = d.bias;
  p.rowmask = d.rowmask; p.seq_mask = d.seq_mask; p.msa_mask = d.msa_mask; p.mask_transposed = d.mask_transposed;
  p.gate = reinterpret_cast<const __half*>(d.gate); p.ldg = d.ldg;
  p.cm_out[0] = reinterpret_cast<bf16*>(d.cm_out[0]); p.cm_out[1] = reinterpret_cast<bf16*>(d.cm_out[1]);
  p.cm_channels = d.cm_channels;
  p.heads_out = reinterpret_cast<bf16*>(d.heads_out); p.n_heads = d.n_heads;
  p.vt_out = reinterpret_cast<bf16*>(d.vt_out); p.vt_cols = d.vt_cols;
  p.Lpad = d.Lpad;
  p.tile_active = d.tile_active;
  p.bias_lo = d.bias_lo;
  p.bias_n = d.bias ? (d.bias_n > 0 ? d.bias_n : d.Nw - d.bias_lo) : 0;
  {
    const int cap = d.K == 256 ? G2Smem<256>::BIAS_FLOATS : G2Smem<128>::BIAS_FLOATS;
    if (p.bias_n > cap || (p.bias_lo & 63) || p.bias_lo < 0) {
      tc_set_error("gemm2: bias range does not fit the shared-memory table (give bias_lo / bias_n, multiples of 64)");
      return -1;
    }
  }
  bool need_bias = false;
  p.has_cms = 0;
  for (int i = 0; i < G2_MAX_OPS; ++i) {
    if (i < d.n_ops) p.ops[i] = d.ops[i];
    else p.ops[i].kind = G2_SKIP;
    if (p.ops[i].kind == G2_CMS) p.has_cms = 1;
    if (p.ops[i].kind == G2_RESID || p.ops[i].kind == G2_CM_DUAL || p.ops[i].kind == G2_CMS) need_bias = true;
  }
  if (d.a_mode == 0 && d.op_fmt != 1) {
    tc_set_error("gemm2: LayerNorm-fed GEMMs use fp16 operands");
    return -1;
  }
  if (need_bias && !d.bias) {
    tc_set_error("gemm2: residual / gated groups need a bias vector");
    return -1;
  }

  CUtensorMap tmW, tmA, tmO0, tmT[2], tmH, tmR;
  const int ek = d.op_fmt ? 1 : 0;   // 0 bf16, 1 fp16, 2 fp32
  {
    uint64_t dims[2] = {(uint64_t)d.K, (uint64_t)d.Nw}, str[1] = {(uint64_t)d.K * 2};
    uint32_t box[2] = {64, G2_BN};
    if (tma_encode(ctx, &tmW, d.Wt, ek, 2, dims, str, box, 128) != 0) return -1;
  }
  const uint64_t D1 = d.D1, D2 = d.D2, Bn = d.B, Lp = d.Lpad;
  const uint32_t YT = (uint32_t)p.YT, XT = (uint32_t)p.XT;
  const uint32_t YTW = YT < 32 ? YT : 32, XTW = 32 / YTW;   // the 32 rows one epilogue warp stores: YTW consecutive y of XTW x
  p.ytw_shift = 0;
  while ((1u << p.ytw_shift) < YTW) ++p.ytw_shift;
  if (d.a_mode == 1) {
    uint64_t dims[4] = {(uint64_t)d.K, D2, D1, Bn};
    uint64_t str[3] = {(uint64_t)d.K * 2, D2 * d.K * 2, D1 * D2 * d.K * 2};
    uint32_t box[4] = {64, YT, XT, 1};
    if (tma_encode(ctx, &tmA, d.A, ek, 4, dims, str, box, 128) != 0) return -1;
  } else {
    tmA = tmW;
  }
  if (d.row_out[0]) {
    uint64_t ld = d.row_ld[0];
    uint64_t dims[4] = {ld, D2, D1, Bn};
    uint64_t str[3] = {ld * 2, D2 * ld * 2, D1 * D2 * ld * 2};
    uint32_t box[4] = {64, YTW, XTW, 1};
    if (tma_encode(ctx, &tmO0, d.row_out[0], 0, 4, dims, str, box, 128) != 0) return -1;
  } else {
    tmO0 = tmW;
  }
  CUtensorMap tmVS = tmW;
  tmT[0] = tmT[1] = tmH = tmW;
  if (d.vt_out && d.cm_out[0]) {
    tc_set_error("gemm2: transposed-column and channel-major outputs cannot be combined");
    return -1;
  }
  p.swap_mask = d.swap_mask;
  if (p.has_cms && (d.K != 128 || p.YT < 64 || !d.cm_out[0] || d.bias_lo != 0 || d.Nw > G2Smem<128>::BIAS_FLOATS)) {
    tc_set_error("gemm2: operand-swapped gated groups need K = 128, YT >= 64, cm_out and the whole bias in the table");
    return -1;
  }
  if (d.swap_mask && !p.has_cms) {
    if (!d.vt_out || p.YT < 64) {
      tc_set_error("gemm2: operand-swapped transposed outputs need vt_out and a tile of at least 64 consecutive y");
      return -1;
    }
    uint64_t vc = d.vt_cols;
    uint64_t dims[4] = {D2, vc, D1, Bn};
    uint64_t str[3] = {Lp * 2, vc * Lp * 2, D1 * vc * Lp * 2};
    uint32_t box[4] = {64, 32, 1, 1};
    if (tma_encode(ctx, &tmVS, d.vt_out, 0, 4, dims, str, box, 128) != 0) return -1;
  }
  if (d.vt_out) {   // [(b, x), column, y] with row pitch Lpad: dims {y, column, x, b}
    uint64_t vc = d.vt_cols;
    uint64_t dims[4] = {D2, vc, D1, Bn};
    uint64_t str[3] = {Lp * 2, vc * Lp * 2, D1 * vc * Lp * 2};
    uint32_t box[4] = {YTW, 64, XTW, 1};
    if (tma_encode(ctx, &tmT[0], d.vt_out, 0, 4, dims, str, box, 0) != 0) return -1;
  }
  for (int i = 0; i < 2; ++i) {
    if (!d.cm_out[i]) continue;   // [(b, channel), x, y] with row pitch Lpad: dims {y, x, channel, b}
    uint64_t ch = d.cm_channels;
    uint64_t dims[4] = {D2, D1, ch, Bn};
    uint64_t str[3] = {Lp * 2, D1 * Lp * 2, ch * D1 * Lp * 2};
    uint32_t box[4] = {YTW, XTW, 64, 1};
    uint32_t box_s[4] = {64, 1, 32, 1};   // operand-swapped groups: 128-byte rows of 64 y per channel, 128B swizzle
    if (tma_encode(ctx, &tmT[i], d.cm_out[i], 0, 4, dims, str, p.has_cms ? box_s : box, p.has_cms ? 128 : 0) != 0) return -1;
  }
  if (d.heads_out) {   // [(b, head), x, y] with row pitch Lpad
    uint64_t nh = d.n_heads;
    uint64_t dims[4] = {D2, D1, nh, Bn};
    uint64_t str[3] = {Lp * 2, D1 * Lp * 2, nh * D1 * Lp * 2};
    uint32_t box[4] = {YTW, XTW, (uint32_t)d.n_heads, 1};
    if (tma_encode(ctx, &tmH, d.heads_out, 0, 4, dims, str, box, 0) != 0) return -1;
  }
  if (d.resid) {
    uint64_t ld = d.resid_ld;
    uint64_t dims[4] = {ld, D2, D1, Bn};
    uint64_t str[3];
    if (d.resid_transposed) {   // destination array is [B, D2, D1, ld]: y is its second axis
      str[0] = D1 * ld * 4; str[1] = ld * 4; str[2] = D1 * D2 * ld * 4;
    } else {
      str[0] = ld * 4; str[1] = D2 * ld * 4; str[2] = D1 * D2 * ld * 4;
    }
    uint32_t box[4] = {32, YTW, XTW, 1};
    if (tma_encode(ctx, &tmR, d.resid, 2, 4, dims, str, box, 128) != 0) return -1;
  } else {
    tmR = tmW;
  }
  if (d.K == 64) return launch_g2<64, 0>(tmW, tmA, tmO0, tmT[0], tmT[1], tmH, tmR, tmVS, p, num_sms, st);
  if (d.K == 128) {
    return d.a_mode == 0 ? launch_g2<128, 0>(tmW, tmA, tmO0, tmT[0], tmT[1], tmH, tmR, tmVS, p, num_sms, st)
                         : launch_g2<128, 1>(tmW, tmA, tmO0, tmT[0], tmT[1], tmH, tmR, tmVS, p, num_sms, st);
  }
  return d.a_mode == 0 ? launch_g2<256, 0>(tmW, tmA, tmO0, tmT[0], tmT[1], tmH, tmR, tmVS, p, num_sms, st)
                       : launch_g2<256, 1>(tmW, tmA, tmO0, tmT[0], tmT[1], tmH, tmR, tmVS, p, num_sms, st);
}

}  // namespace pf
