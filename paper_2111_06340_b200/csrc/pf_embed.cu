// Input embedder, recycling embedder and the recycled trunk ("recycling", "three
// recycling procedures"; readings E.1-E.3 of DESIGN.md §2b):
//   E.1  z_ij = Lin_a(tf_i) + Lin_b(tf_j) + Lin_rel(onehot(clip(r_i - r_j, -R, R) + R)),   m_si = Lin_m(msa_feat_si) + Lin_t(tf_i)
//   E.2  z_ij += LN_z(zprev_ij) + Lin_d(onehot_bins(|xprev_i - xprev_j|)),                 m_0i += LN_m(mprev_0i)
//   E.3  n_cycles x (E.1, E.2 with the previous cycle's trunk output, trunk)
// All of it is HBM-bound elementwise work with reduction lengths of 15 .. 65, so it runs in fp32 on the SIMT pipes: one warp
// per output row, 128-bit loads / stores, warp-shuffle LayerNorm statistics; one-hot Linears are row gathers from tables in
// shared memory.  E.1 and E.2 are ONE pass over each stream and run IN PLACE: the row that holds the previous cycle's value
// is read by the warp that then overwrites it, so recycling costs no copy of m or z.
#include "pf_handle.h"
#include "pf_device.cuh"

#include <algorithm>
#include <cmath>
#include <string>
#include <vector>

using namespace pf;

struct pf_embedder {
  pf_embed_config cfg;
  float* w = nullptr;        // device fp32 blob (pf_embedder_floats layout)
  float* edges2 = nullptr;   // device [2 * n_dist_bins]: squared lower / upper bin edges (fp32, computed as the oracle does)
  float* ws = nullptr;       // [B, N, 2 c_z + c_m]: Lin_a(tf) | Lin_b(tf) | Lin_t(tf)
  size_t ws_floats = 0;
  long long launches = 0;
  int device = -1;
  struct Off { size_t w_a, b_a, w_b, b_b, w_rel, b_rel, w_m, b_m, w_t, b_t, ln_m_g, ln_m_b, ln_z_g, ln_z_b, w_d, b_d, w_e, b_e, total; } off;
};

namespace pf { void api_set_error(const std::string& s); }
static pf_status efail(pf_status s, const std::string& msg) {
  api_set_error(msg);
  return s;
}

static pf_embedder::Off embed_offsets(const pf_embed_config& c) {
  pf_embedder::Off o{};
  size_t at = 0;
  auto take = [&](size_t n) { size_t r = at; at += n; return r; };
  const size_t nrel = 2 * (size_t)c.max_relpos + 1;
  o.w_a = take((size_t)c.tf_dim * c.c_z); o.b_a = take(c.c_z);
  o.w_b = take((size_t)c.tf_dim * c.c_z); o.b_b = take(c.c_z);
  o.w_rel = take(nrel * c.c_z); o.b_rel = take(c.c_z);
  o.w_m = take((size_t)c.msa_dim * c.c_m); o.b_m = take(c.c_m);
  o.w_t = take((size_t)c.tf_dim * c.c_m); o.b_t = take(c.c_m);
  o.ln_m_g = take(c.c_m); o.ln_m_b = take(c.c_m);
  o.ln_z_g = take(c.c_z); o.ln_z_b = take(c.c_z);
  o.w_d = take((size_t)c.n_dist_bins * c.c_z); o.b_d = take(c.c_z);
  o.w_e = take((size_t)c.extra_dim * c.c_e); o.b_e = take(c.c_e);
  o.total = at;
  return o;
}

// ------------------------------------------------------------------------------------------------
// kernels
// ------------------------------------------------------------------------------------------------
// per residue (b, i): out[(b,i), :] = [ Lin_a(tf) | Lin_b(tf) | Lin_t(tf) ]  (2 c_z + c_m values), reduction length tf_dim
__global__ void embed_residue_kernel(const float* __restrict__ tf, const float* __restrict__ w, pf_embedder::Off o, int tf_dim,
                                     int c_z, int c_m, float* __restrict__ out) {
  extern __shared__ float f[];
  const long r = blockIdx.x;
  for (int k = threadIdx.x; k < tf_dim; k += blockDim.x) f[k] = tf[r * tf_dim + k];
  __syncthreads();
  const int width = 2 * c_z + c_m;
  for (int n = threadIdx.x; n < width; n += blockDim.x) {
    const float* W;
    float acc;
    int col, ld;
    if (n < c_z) { W = w + o.w_a; acc = w[o.b_a + n]; col = n; ld = c_z; }
    else if (n < 2 * c_z) { W = w + o.w_b; acc = w[o.b_b + n - c_z]; col = n - c_z; ld = c_z; }
    else { W = w + o.w_t; acc = w[o.b_t + n - 2 * c_z]; col = n - 2 * c_z; ld = c_m; }
    for (int k = 0; k < tf_dim; ++k) acc = fmaf(f[k], __ldg(W + (long)k * ld + col), acc);
    out[r * width + n] = acc;
  }
}

// warp-level LayerNorm of a row held as NV float4 per lane (R4), result added to acc
template <int NV>
__device__ __forceinline__ void warp_ln_add(const float4 (&v)[NV], const float4* gamma, const float4* beta, int lane, int C,
                                            float4 (&acc)[NV]) {
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) s += (v[i].x + v[i].y) + (v[i].z + v[i].w);
  s = warp_sum(s);
  const float mean = s / C;
  float q = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const float a = v[i].x - mean, b = v[i].y - mean, c = v[i].z - mean, d = v[i].w - mean;
    q += (a * a + b * b) + (c * c + d * d);
  }
  q = warp_sum(q);
  const float rstd = rsqrtf(q / C + 1e-5f);
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const float4 g = __ldg(gamma + lane * NV + i), be = __ldg(beta + lane * NV + i);
    acc[i].x += (v[i].x - mean) * rstd * g.x + be.x;
    acc[i].y += (v[i].y - mean) * rstd * g.y + be.y;
    acc[i].z += (v[i].z - mean) * rstd * g.z + be.z;
    acc[i].w += (v[i].w - mean) * rstd * g.w + be.w;
  }
}

// MSA rows (b, s, i), one warp per row, lane owns C/32 consecutive channels:
//   m[b,s,i,:] = msa_feat[b,s,i,:] W_m + b_m + Lin_t(tf_i)   (+ LN_m(m_old[b,0,i,:]) for s == 0, E.2; LN(0) = beta without a previous cycle)
template <int C>
__global__ void __launch_bounds__(256) embed_msa_kernel(const float* __restrict__ feat, const float* __restrict__ w,
                                                        pf_embedder::Off o, const float* __restrict__ res_lin, int res_ld,
                                                        int res_off, int msa_dim, int has_prev, float* __restrict__ m, int S,
                                                        int N, long rows) {
  constexpr int NV = C / 128;                       // float4 per lane
  extern __shared__ __align__(16) float wm[];       // W_m [msa_dim, C]
  for (int k = threadIdx.x; k < msa_dim * C / 4; k += blockDim.x)
    reinterpret_cast<float4*>(wm)[k] = __ldg(reinterpret_cast<const float4*>(w + o.w_m) + k);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const long warp = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), nwarps = (long)gridDim.x * (blockDim.x >> 5);
  for (long r = warp; r < rows; r += nwarps) {
    const long bs = r / N;
    const int i = (int)(r - bs * N), s = (int)(bs % S);
    const long b = bs / S;
    const float* fr = feat + r * msa_dim;
    const float f0 = lane < msa_dim ? __ldg(fr + lane) : 0.f;
    const float f1 = lane + 32 < msa_dim ? __ldg(fr + lane + 32) : 0.f;
    float4 acc[NV];
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      const float4 bm = __ldg(reinterpret_cast<const float4*>(w + o.b_m) + lane * NV + q);
      const float4 t = __ldg(reinterpret_cast<const float4*>(res_lin + (b * N + i) * res_ld + res_off) + lane * NV + q);
      acc[q] = make_float4(bm.x + t.x, bm.y + t.y, bm.z + t.z, bm.w + t.w);
    }
    for (int k = 0; k < msa_dim; ++k) {
      const float fk = __shfl_sync(0xffffffffu, k < 32 ? f0 : f1, k & 31);
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        const float4 wv = reinterpret_cast<const float4*>(wm + k * C)[lane * NV + q];
        acc[q].x = fmaf(fk, wv.x, acc[q].x);
        acc[q].y = fmaf(fk, wv.y, acc[q].y);
        acc[q].z = fmaf(fk, wv.z, acc[q].z);
        acc[q].w = fmaf(fk, wv.w, acc[q].w);
      }
    }
    float4* dst = reinterpret_cast<float4*>(m + r * C) + lane * NV;
    if (s == 0) {
      float4 v[NV];
#pragma unroll
      for (int q = 0; q < NV; ++q) v[q] = has_prev ? dst[q] : make_float4(0.f, 0.f, 0.f, 0.f);
      warp_ln_add<NV>(v, reinterpret_cast<const float4*>(w + o.ln_m_g), reinterpret_cast<const float4*>(w + o.ln_m_b), lane, C, acc);
    }
#pragma unroll
    for (int q = 0; q < NV; ++q) dst[q] = acc[q];
  }
}

// pair rows (b, i, j), one warp per row, lane owns C/32 consecutive channels:
//   z[b,i,j,:] = Lin_a(tf_i) + Lin_b(tf_j) + W_rel[clip(r_i - r_j) + R] + b_rel + LN_z(z_old[b,i,j,:]) + W_d[bin(|x_i - x_j|)] + b_d
template <int C>
__global__ void __launch_bounds__(256) embed_pair_kernel(const float* __restrict__ w, pf_embedder::Off o,
                                                         const float* __restrict__ res_lin, int res_ld,
                                                         const int* __restrict__ ridx, const float* __restrict__ xprev,
                                                         const float* __restrict__ edges2, int max_relpos, int n_bins,
                                                         int has_prev, float* __restrict__ z, int N, long rows) {
  constexpr int NV = C / 128;
  extern __shared__ __align__(16) float tab[];      // W_rel [2R+1, C] | W_d [n_bins, C] | edges2 [2 n_bins]
  const int nrel = 2 * max_relpos + 1;
  float* wrel = tab;
  float* wd = tab + nrel * C;
  float* ed = wd + n_bins * C;
  for (int k = threadIdx.x; k < nrel * C; k += blockDim.x) wrel[k] = __ldg(w + o.w_rel + k);
  for (int k = threadIdx.x; k < n_bins * C; k += blockDim.x) wd[k] = __ldg(w + o.w_d + k);
  for (int k = threadIdx.x; k < 2 * n_bins; k += blockDim.x) ed[k] = __ldg(edges2 + k);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const long warp = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), nwarps = (long)gridDim.x * (blockDim.x >> 5);
  for (long r = warp; r < rows; r += nwarps) {
    const long bi = r / N;
    const int j = (int)(r - bi * N);
    const long b = bi / N;
    const long bj = b * N + j;
    int rel = __ldg(ridx + bi) - __ldg(ridx + bj);
    rel = min(max(rel, -max_relpos), max_relpos) + max_relpos;
    int bin = -1;
    if (xprev) {
      // the comparison decides an integer: fp32, this operation order, no fused multiply-add (as the oracle does it)
      const float dx = __fsub_rn(__ldg(xprev + bi * 3 + 0), __ldg(xprev + bj * 3 + 0));
      const float dy = __fsub_rn(__ldg(xprev + bi * 3 + 1), __ldg(xprev + bj * 3 + 1));
      const float dz = __fsub_rn(__ldg(xprev + bi * 3 + 2), __ldg(xprev + bj * 3 + 2));
      const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
      for (int k = 0; k < n_bins; ++k)
        if (d2 > ed[k] && d2 < ed[n_bins + k]) bin = k;
    }
    float4* dst = reinterpret_cast<float4*>(z + r * C) + lane * NV;
    float4 acc[NV], v[NV];
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      v[q] = has_prev ? dst[q] : make_float4(0.f, 0.f, 0.f, 0.f);
      const float4 a = __ldg(reinterpret_cast<const float4*>(res_lin + bi * res_ld) + lane * NV + q);
      const float4 bb = __ldg(reinterpret_cast<const float4*>(res_lin + bj * res_ld + C) + lane * NV + q);
      const float4 wr = reinterpret_cast<const float4*>(wrel + rel * C)[lane * NV + q];
      const float4 br = __ldg(reinterpret_cast<const float4*>(w + o.b_rel) + lane * NV + q);
      const float4 bd = __ldg(reinterpret_cast<const float4*>(w + o.b_d) + lane * NV + q);
      acc[q] = make_float4(a.x + bb.x + wr.x + br.x + bd.x, a.y + bb.y + wr.y + br.y + bd.y, a.z + bb.z + wr.z + br.z + bd.z,
                           a.w + bb.w + wr.w + br.w + bd.w);
      if (bin >= 0) {
        const float4 wv = reinterpret_cast<const float4*>(wd + bin * C)[lane * NV + q];
        acc[q].x += wv.x; acc[q].y += wv.y; acc[q].z += wv.z; acc[q].w += wv.w;
      }
    }
    warp_ln_add<NV>(v, reinterpret_cast<const float4*>(w + o.ln_z_g), reinterpret_cast<const float4*>(w + o.ln_z_b), lane, C, acc);
#pragma unroll
    for (int q = 0; q < NV; ++q) dst[q] = acc[q];
  }
}

// E.4 extra-MSA rows (b, s, i), one warp per row, lane owns two of the c_e = 64 channels: e = extra_msa_feat W_e + b_e
__global__ void __launch_bounds__(256) embed_extra_kernel(const float* __restrict__ feat, const float* __restrict__ w,
                                                          pf_embedder::Off o, int extra_dim, float* __restrict__ out, long rows) {
  extern __shared__ __align__(16) float we[];       // W_e [extra_dim, 64]
  for (int k = threadIdx.x; k < extra_dim * 64; k += blockDim.x) we[k] = __ldg(w + o.w_e + k);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const long warp = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), nwarps = (long)gridDim.x * (blockDim.x >> 5);
  const float2 be = __ldg(reinterpret_cast<const float2*>(w + o.b_e) + lane);
  for (long r = warp; r < rows; r += nwarps) {
    const float f0 = lane < extra_dim ? __ldg(feat + r * extra_dim + lane) : 0.f;
    float a0 = be.x, a1 = be.y;
    for (int k = 0; k < extra_dim; ++k) {
      const float fk = __shfl_sync(0xffffffffu, f0, k);
      const float2 wv = reinterpret_cast<const float2*>(we + k * 64)[lane];
      a0 = fmaf(fk, wv.x, a0);
      a1 = fmaf(fk, wv.y, a1);
    }
    reinterpret_cast<float2*>(out + r * 64)[lane] = make_float2(a0, a1);
  }
}

// ------------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------------
static bool embed_cfg_ok(const pf_embed_config& c) {
  return c.extra_dim >= 1 && c.extra_dim <= 32 && c.c_e == 64 && (c.c_m == 128 || c.c_m == 256) && (c.c_z == 128 || c.c_z == 256) && c.tf_dim >= 1 && c.tf_dim <= 1024 &&
         c.msa_dim >= 1 && c.msa_dim <= 64 && c.max_relpos >= 0 && c.max_relpos <= 64 && c.n_dist_bins >= 1 &&
         c.n_dist_bins <= 64 && c.last_break > c.first_break && c.first_break >= 0.f;
}

extern "C" size_t pf_embedder_floats(const pf_embed_config* cfg) {
  if (!cfg || !embed_cfg_ok(*cfg)) return 0;
  return embed_offsets(*cfg).total;
}

extern "C" pf_status pf_embedder_create(pf_embedder_t** out, const float* weights_host, size_t n_floats,
                                        const pf_embed_config* cfg) {
  if (!out || !weights_host || !cfg) return efail(PF_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  if (!embed_cfg_ok(*cfg))
    return efail(PF_ERR_SHAPE, "embedder dims: c_m, c_z in {128, 256}, msa_dim <= 64, max_relpos <= 64, n_dist_bins <= 64");
  pf_embedder::Off off = embed_offsets(*cfg);
  if (n_floats != off.total) return efail(PF_ERR_SHAPE, "embedder weights blob length != pf_embedder_floats(cfg)");
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return efail(PF_ERR_CUDA, "cudaGetDevice");
  pf_embedder* e = new (std::nothrow) pf_embedder();
  if (!e) return efail(PF_ERR_ALLOC, "host alloc");
  e->cfg = *cfg;
  e->off = off;
  e->device = dev;
  // squared bin edges exactly as the oracle forms them: K lower edges evenly spaced (the last one = last_break), rounded to
  // fp32, squared in fp32; upper edge of bin k = lower edge of bin k + 1, infinity for the last bin
  const int nb = cfg->n_dist_bins;
  std::vector<float> ed(2 * (size_t)nb);
  for (int k = 0; k < nb; ++k) {
    const double step = nb > 1 ? ((double)cfg->last_break - (double)cfg->first_break) / (nb - 1) : 0.0;
    const float ek = (k == nb - 1 && nb > 1) ? cfg->last_break : (float)((double)cfg->first_break + k * step);
    ed[k] = ek * ek;
  }
  for (int k = 0; k < nb; ++k) ed[nb + k] = k + 1 < nb ? ed[k + 1] : INFINITY;
  if (cudaMalloc(&e->w, off.total * 4) != cudaSuccess || cudaMalloc(&e->edges2, ed.size() * 4) != cudaSuccess) {
    pf_embedder_destroy(e);
    return efail(PF_ERR_ALLOC, "cudaMalloc embedder weights");
  }
  if (cudaMemcpy(e->w, weights_host, off.total * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(e->edges2, ed.data(), ed.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
    pf_embedder_destroy(e);
    return efail(PF_ERR_CUDA, "embedder weights H2D");
  }
  // dynamic shared memory above 48 KB (the W_m table at c_m = 256), per device
  const int msa_smem = cfg->msa_dim * cfg->c_m * 4;
  cudaError_t ce = cfg->c_m == 256
                       ? cudaFuncSetAttribute(embed_msa_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, msa_smem)
                       : cudaFuncSetAttribute(embed_msa_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, msa_smem);
  const int pair_smem = ((2 * cfg->max_relpos + 1 + cfg->n_dist_bins) * cfg->c_z + 2 * cfg->n_dist_bins) * 4;
  if (ce == cudaSuccess)
    ce = cfg->c_z == 256
             ? cudaFuncSetAttribute(embed_pair_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, pair_smem)
             : cudaFuncSetAttribute(embed_pair_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, pair_smem);
  if (ce != cudaSuccess) {
    pf_embedder_destroy(e);
    return efail(PF_ERR_CUDA, std::string("cudaFuncSetAttribute(embedder): ") + cudaGetErrorString(ce));
  }
  *out = e;
  return PF_OK;
}

extern "C" void pf_embedder_destroy(pf_embedder_t* e) {
  if (!e) return;
  cudaFree(e->w);
  cudaFree(e->edges2);
  cudaFree(e->ws);
  delete e;
}

extern "C" long long pf_embedder_last_launch_count(const pf_embedder_t* e) { return e ? e->launches : 0; }

extern "C" pf_status pf_embedder_forward(pf_embedder_t* e, const float* target_feat, const int* residue_index,
                                         const float* msa_feat, const float* x_prev, int has_prev, float* msa, float* pair,
                                         int B, int S, int N, void* stream) {
  if (!e || !target_feat || !residue_index || !msa_feat || !msa || !pair) return efail(PF_ERR_INVALID_ARG, "null argument");
  if (B < 1 || S < 1 || N < 1) return efail(PF_ERR_SHAPE, "B, S, N must be >= 1");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != e->device)
    return efail(PF_ERR_INVALID_ARG, "the current device is not the one the embedder was created on");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const pf_embed_config& c = e->cfg;
  const int width = 2 * c.c_z + c.c_m;
  const size_t need = (size_t)B * N * width;
  if (need > e->ws_floats) {
    cudaDeviceSynchronize();
    cudaFree(e->ws);
    e->ws = nullptr;
    e->ws_floats = 0;
    if (cudaMalloc(&e->ws, need * 4) != cudaSuccess) {
      cudaGetLastError();
      return efail(PF_ERR_ALLOC, "cudaMalloc embedder workspace");
    }
    e->ws_floats = need;
  }
  e->launches = 0;
  embed_residue_kernel<<<(unsigned)((long)B * N), 128, c.tf_dim * 4, st>>>(target_feat, e->w, e->off, c.tf_dim, c.c_z, c.c_m, e->ws);
  const long mrows = (long)B * S * N, prows = (long)B * N * N;
  int sms = 148;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  auto grid_for = [&](long rows, int per_sm) { return (unsigned)std::max(1L, std::min((rows + 7) / 8, (long)sms * per_sm)); };
  const int msa_smem = c.msa_dim * c.c_m * 4;
  if (c.c_m == 256)
    embed_msa_kernel<256><<<grid_for(mrows, 4), 256, msa_smem, st>>>(msa_feat, e->w, e->off, e->ws, width, 2 * c.c_z, c.msa_dim,
                                                                      has_prev, msa, S, N, mrows);
  else
    embed_msa_kernel<128><<<grid_for(mrows, 4), 256, msa_smem, st>>>(msa_feat, e->w, e->off, e->ws, width, 2 * c.c_z, c.msa_dim,
                                                                      has_prev, msa, S, N, mrows);
  const int pair_smem = ((2 * c.max_relpos + 1 + c.n_dist_bins) * c.c_z + 2 * c.n_dist_bins) * 4;
  if (c.c_z == 256)
    embed_pair_kernel<256><<<grid_for(prows, 4), 256, pair_smem, st>>>(e->w, e->off, e->ws, width, residue_index, x_prev,
                                                                        e->edges2, c.max_relpos, c.n_dist_bins, has_prev, pair, N, prows);
  else
    embed_pair_kernel<128><<<grid_for(prows, 4), 256, pair_smem, st>>>(e->w, e->off, e->ws, width, residue_index, x_prev,
                                                                        e->edges2, c.max_relpos, c.n_dist_bins, has_prev, pair, N, prows);
  e->launches = 3;
  cudaError_t ce = cudaGetLastError();
  if (ce != cudaSuccess) return efail(PF_ERR_CUDA, std::string("embedder launch failed: ") + cudaGetErrorString(ce));
  return PF_OK;
}

extern "C" pf_status pf_embedder_forward_extra(pf_embedder_t* e, const float* extra_msa_feat, float* extra_msa, int B, int S_e,
                                               int N, void* stream) {
  if (!e || !extra_msa_feat || !extra_msa) return efail(PF_ERR_INVALID_ARG, "null argument");
  if (B < 1 || S_e < 1 || N < 1) return efail(PF_ERR_SHAPE, "B, S_e, N must be >= 1");
  int dev = -1, sms = 148;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != e->device)
    return efail(PF_ERR_INVALID_ARG, "the current device is not the one the embedder was created on");
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const long rows = (long)B * S_e * N;
  const unsigned grid = (unsigned)std::max(1L, std::min((rows + 7) / 8, (long)sms * 8));
  embed_extra_kernel<<<grid, 256, e->cfg.extra_dim * 64 * 4, reinterpret_cast<cudaStream_t>(stream)>>>(
      extra_msa_feat, e->w, e->off, e->cfg.extra_dim, extra_msa, rows);
  e->launches = 1;
  cudaError_t ce = cudaGetLastError();
  if (ce != cudaSuccess) return efail(PF_ERR_CUDA, std::string("extra-MSA embedder launch failed: ") + cudaGetErrorString(ce));
  return PF_OK;
}

extern "C" pf_status pf_evoformer_forward_recycled(pf_evoformer_t* h, pf_embedder_t* e, pf_extra_msa_t* x,
                                                   const float* target_feat, const int* residue_index, const float* msa_feat,
                                                   const float* x_prev, const float* extra_msa_feat, float* extra_msa,
                                                   const float* extra_msa_mask, float* msa, float* pair, const float* seq_mask,
                                                   const float* msa_mask, int B, int S, int S_e, int N, int n_blocks,
                                                   int n_extra_blocks, int n_cycles, void* stream) {
  if (!h || !e) return efail(PF_ERR_INVALID_ARG, "null handle");
  if (n_cycles < 1) return efail(PF_ERR_SHAPE, "n_cycles must be >= 1");
  if (e->cfg.c_m != h->cfg.c_m || e->cfg.c_z != h->cfg.c_z) return efail(PF_ERR_SHAPE, "embedder and trunk channel dims differ");
  if (x && (!extra_msa_feat || !extra_msa || !extra_msa_mask)) return efail(PF_ERR_INVALID_ARG, "extra-MSA stack given without its features / buffer / mask");
  long long launches = 0;
  for (int c = 0; c < n_cycles; ++c) {
    pf_status s = pf_embedder_forward(e, target_feat, residue_index, msa_feat, x_prev, c > 0 ? 1 : 0, msa, pair, B, S, N, stream);
    if (s != PF_OK) return s;
    launches += e->launches;
    if (x) {
      s = pf_embedder_forward_extra(e, extra_msa_feat, extra_msa, B, S_e, N, stream);
      if (s != PF_OK) return s;
      launches += e->launches;
      s = pf_extra_msa_forward(x, extra_msa, pair, seq_mask, extra_msa_mask, B, S_e, N, n_extra_blocks, stream);
      if (s != PF_OK) return s;
      launches += pf_extra_msa_last_launch_count(x);
    }
    s = pf_evoformer_forward(h, msa, pair, seq_mask, msa_mask, B, S, N, n_blocks, stream);
    if (s != PF_OK) return s;
    launches += h->launches;
  }
  h->launches = launches;
  return PF_OK;
}
