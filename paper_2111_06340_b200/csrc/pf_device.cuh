// Device helpers shared by all kernels: type conversion, warp reductions, row geometry and the
// projection-GEMM epilogue (one definition, used element-wise by the SIMT GEMM and row-wise by the tcgen05 GEMM).
#pragma once
#include "pf_internal.h"

namespace pf {

__device__ __forceinline__ float to_f32(float v) { return v; }
__device__ __forceinline__ float to_f32(bf16 v) { return __bfloat162float(v); }
__device__ __forceinline__ float to_f32(__half v) { return __half2float(v); }
__device__ __forceinline__ void store1(__half* p, float v) { *p = __float2half_rn(v); }
__device__ __forceinline__ void store1(float* p, float v) { *p = v; }
__device__ __forceinline__ void store1(bf16* p, float v) { *p = __float2bfloat16_rn(v); }
__device__ __forceinline__ void store4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ void store4(bf16* p, float4 v) {
  __nv_bfloat162 lo = __floats2bfloat162_rn(v.x, v.y), hi = __floats2bfloat162_rn(v.z, v.w);
  uint2 u;
  u.x = *reinterpret_cast<uint32_t*>(&lo);
  u.y = *reinterpret_cast<uint32_t*>(&hi);
  *reinterpret_cast<uint2*>(p) = u;
}

__device__ __forceinline__ float4 ld_nc_f4(const float4* p) {
  float4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
  return r;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

__device__ __forceinline__ float sigmoidf_acc(float x) { return 1.0f / (1.0f + expf(-x)); }

// Row r = (b, x, y) of a [B, D1, D2] grid  ->  row (b, y, x) of the [B, D2, D1] grid.
__device__ __forceinline__ long transposed_row(long r, const RowGeom& g) {
  long per = (long)g.D1 * g.D2;
  long b = r / per;
  int rem = (int)(r - b * per);
  int x = rem / g.D2, y = rem - x * g.D2;
  return (b * g.D2 + y) * g.D1 + x;
}

struct RowInfo {
  int b, x, y;
  float mask;
  long dst;   // residual destination row (EPI_RESID)
};

__device__ __forceinline__ RowInfo row_info(long r, const Epi& e) {
  RowInfo ri;
  long per = (long)e.geom.D1 * e.geom.D2;
  ri.b = (int)(r / per);
  int rem = (int)(r - (long)ri.b * per);
  ri.x = rem / e.geom.D2;
  ri.y = rem - ri.x * e.geom.D2;
  ri.mask = 1.0f;
  if (e.rowmask == RM_MSA) {
    if (e.mask_transposed)
      ri.mask = e.msa_mask[(long)ri.b * e.geom.D2 + ri.y] * e.seq_mask[(long)ri.b * e.geom.D1 + ri.x];
    else
      ri.mask = e.msa_mask[(long)ri.b * e.geom.D1 + ri.x] * e.seq_mask[(long)ri.b * e.geom.D2 + ri.y];
  } else if (e.rowmask == RM_PAIR) {
    ri.mask = e.seq_mask[(long)ri.b * e.geom.D1 + ri.x] * e.seq_mask[(long)ri.b * e.geom.D2 + ri.y];
  }
  ri.dst = e.transposed ? ((long)ri.b * e.geom.D2 + ri.y) * e.geom.D1 + ri.x : r;
  return ri;
}

// One output element of a projection GEMM (see struct Epi for the four kinds).
template <typename T>
__device__ __forceinline__ void epilogue_elem(const Epi& e, const RowInfo& ri, long r, int n, int Nout, float acc,
                                              float acc2) {
  if (e.kind == EPI_STORE) {
    float v = acc * (n < e.scale_cols ? e.scale : 1.0f);
    if (e.bias) v += __ldg(e.bias + n);
    if (n >= e.act_lo && n < e.act_hi) {
      if (e.act == ACT_SIGMOID) v = sigmoidf_acc(v);
      else if (e.act == ACT_RELU) v = fmaxf(v, 0.f);
    }
    v *= ri.mask;
    if (n < e.vt_from) {
      store1(reinterpret_cast<T*>(e.out) + r * e.ldo + n, v);
    } else {
      long br = r / e.geom.D2;
      store1(reinterpret_cast<T*>(e.vt) + (br * (Nout - e.vt_from) + (n - e.vt_from)) * e.Lpad + ri.y, v);
    }
  } else if (e.kind == EPI_GATED_CM) {
    float v = ri.mask * sigmoidf_acc(acc2 + __ldg(e.bias2 + n)) * (acc + __ldg(e.bias + n));
    store1(reinterpret_cast<T*>(e.out) + (((long)ri.b * Nout + n) * e.geom.D1 + ri.x) * e.Lpad + ri.y, v);
  } else if (e.kind == EPI_RESID) {
    float v = acc + __ldg(e.bias + n);
    if (e.gate) v *= to_f32(reinterpret_cast<const T*>(e.gate)[r * e.ldg + n]);
    e.resid[ri.dst * e.ldr + n] += v;
  } else {  // EPI_HEADS
    store1(reinterpret_cast<T*>(e.out) + (((long)ri.b * Nout + n) * e.geom.D1 + ri.x) * e.Lpad + ri.y, acc * e.scale);
  }
}

}  // namespace pf
