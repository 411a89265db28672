// LayerNorm producer shared by the LN-fused projection GEMM and the fused transition (R4: biased variance, eps = 1e-5
// inside the sqrt, affine gamma / beta): fp32 rows from global memory -> fp16 A operand in the UMMA K-major 128B-swizzle
// layout.  A warp normalises several rows at once with LPR = K/16 lanes per row (16 lanes at K = 256, 8 at K = 128): every
// lane owns 16 columns (four float4, coalesced: the LPR lanes of a row read LPR consecutive float4 per load), the row
// statistics need log2(LPR) shuffle steps shared by all rows of the pass, and gamma / beta cost 32 registers per lane.
// Two passes (4 rows at K = 256, 8 rows at K = 128) are in flight per call.
#pragma once
#include "pf_device.cuh"

#include <cuda_fp16.h>

namespace pf {

template <int K>
struct LnProd {
  static constexpr int LPR = K / 16;          // lanes per row
  static constexpr int RPP = 32 / LPR;        // rows per pass
  static constexpr int PASSES = 2;
  static constexpr int ROWS = RPP * PASSES;   // rows per call
  float4 gm[4], bt[4];
  int sub, rsel;

  __device__ __forceinline__ void init(const float* gamma, const float* beta, int lane) {
    sub = lane % LPR;
    rsel = lane / LPR;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      gm[i] = __ldg(reinterpret_cast<const float4*>(gamma) + i * LPR + sub);
      bt[i] = __ldg(reinterpret_cast<const float4*>(beta) + i * LPR + sub);
    }
  }
  // tile row (0..127) this lane works on in pass `pass` of the batch starting at tile row r0
  __device__ __forceinline__ int row_of(int r0, int pass) const { return r0 + pass * RPP + rsel; }

  // rp[pass]: this lane's source row (nullptr = a row outside the tensor: normalises zeros, finite, never stored to HBM);
  // lr[pass]: its tile row; abase: the A tile ([K/64] k-blocks of 128 rows x 128 B)
  __device__ __forceinline__ void run(const float* const (&rp)[PASSES], const int (&lr)[PASSES], uint8_t* abase) const {
    float4 v[PASSES][4];
#pragma unroll
    for (int ps = 0; ps < PASSES; ++ps) {
      if (rp[ps]) {
        const float4* xp = reinterpret_cast<const float4*>(rp[ps]);
#pragma unroll
        for (int i = 0; i < 4; ++i) v[ps][i] = ld_nc_f4(xp + i * LPR + sub);
      } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) v[ps][i] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
#pragma unroll
    for (int ps = 0; ps < PASSES; ++ps) {
      float s = 0.f;
#pragma unroll
      for (int i = 0; i < 4; ++i) s += (v[ps][i].x + v[ps][i].y) + (v[ps][i].z + v[ps][i].w);
#pragma unroll
      for (int o = LPR / 2; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      const float mean = s * (1.0f / K);
      float q = 0.f;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float a = v[ps][i].x - mean, b = v[ps][i].y - mean, c = v[ps][i].z - mean, d = v[ps][i].w - mean;
        q += (a * a + b * b) + (c * c + d * d);
      }
#pragma unroll
      for (int o = LPR / 2; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
      const float rstd = rsqrtf(q * (1.0f / K) + 1e-5f);
      const float nm = -mean * rstd;
      uint8_t* arow = abase + lr[ps] * 128;
      const uint32_t sw = (uint32_t)(lr[ps] & 7);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float o0 = fmaf(v[ps][i].x, rstd, nm) * gm[i].x + bt[i].x;
        const float o1 = fmaf(v[ps][i].y, rstd, nm) * gm[i].y + bt[i].y;
        const float o2 = fmaf(v[ps][i].z, rstd, nm) * gm[i].z + bt[i].z;
        const float o3 = fmaf(v[ps][i].w, rstd, nm) * gm[i].w + bt[i].w;
        // columns (i * LPR + sub) * 4 .. +3  ->  k-block col / 64, 16-byte chunk (col % 64) / 8, half (col % 8) / 4
        const int col = (i * LPR + sub) * 4;
        const int kb = col >> 6;
        const uint32_t chunk = (uint32_t)((col & 63) >> 3);
        __half2 h01 = __floats2half2_rn(o0, o1), h23 = __floats2half2_rn(o2, o3);   // fp16 operand (R17)
        *reinterpret_cast<uint2*>(arow + kb * (128 * 128) + ((chunk ^ sw) << 4) + ((col >> 2) & 1) * 8) =
            make_uint2(*reinterpret_cast<uint32_t*>(&h01), *reinterpret_cast<uint32_t*>(&h23));
      }
    }
  }
};

}  // namespace pf
