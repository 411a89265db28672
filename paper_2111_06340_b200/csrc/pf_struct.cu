// Structure module and output heads ("the structure module"; readings M.0-M.6 and
// H.1-H.5 of DESIGN.md §2d, restated in include/pf_evoformer.h).  Small FLOPs and many small steps: per protein the eight
// shared-weight layers cost ~14 MFLOP per residue plus 2 H N c_z FLOP per residue for the pair-value sum of the invariant
// point attention, two to three orders of magnitude below the trunk, and every reduction length is 128 .. 2112 over a few
// hundred to a few thousand rows.  So everything here is fp32 on the SIMT pipes (tolerance 1e-4 against the fp64 oracle):
//   sm_gemm_kernel      Y (+)= act(pre(X) W + b): 64 x 64 tiles, 4 x 4 outputs per thread, optional batched row gather
//   sm_ln_kernel        LayerNorm of rows of any width <= 1024, warp per row, in place if wanted
//   sm_pair_kernel      zn = LN_z(z) and the attention bias b = Lin0(zn), one pass over the pair representation, ONCE per
//                       call (the layers share their weights and z does not change, so both are layer-invariant)
//   sm_points_kernel    local query / key / value points -> global frame
//   sm_ipa_kernel       one CTA per query residue, one warp per head: logits over all keys in shared memory (key-major), softmax,
//                       then the three weighted sums (pair values: every z[i,j,:] read once per CTA against the weights of all
//                       heads; scalar values; value points) and the map back to the local frame
//   sm_frames_kernel    quaternion -> rotation, frame composition, positions
//   sm_alpha_kernel, sm_plddt_kernel, sm_symm_kernel   angle normalisation, pLDDT expectation, distogram symmetrisation
#include "../../include/pf_evoformer.h"
#include "pf_internal.h"
#include "pf_device.cuh"

#include <algorithm>
#include <cmath>
#include <mutex>
#include <new>
#include <string>
#include <vector>

using namespace pf;

namespace pf { void api_set_error(const std::string& s); }
static pf_status sfail(pf_status s, const std::string& msg) {
  api_set_error(msg);
  return s;
}

struct SmOff {
  size_t w_single, b_single, ln_s_g, ln_s_b, ln_z_g, ln_z_b, w_in, b_in, w_q, w_k, w_v, w_qp, w_kp, w_vp, w_b, g_head, w_out,
      b_out, ln_ipa_g, ln_ipa_b, w_t[3], b_t[3], ln_tr_g, ln_tr_b, w_bb, b_bb, w_a1, b_a1, w_a2, b_a2, w_ra[2], b_ra[2],
      w_rb[2], b_rb[2], w_alpha, b_alpha, w_dg, b_dg, w_mm, b_mm, ln_l_g, ln_l_b, w_l1, b_l1, w_l2, b_l2, w_l3, b_l3, w_pae, b_pae, w_er, b_er, total;
};

struct pf_structure {
  pf_struct_config cfg;
  SmOff off;
  float* w = nullptr;        // device fp32 blob (pf_structure_floats layout)
  float* w_proj = nullptr;   // device [c_s, P]: the six bias-free IPA projections side by side (q | k | v | qp | kp | vp)
  float* ws = nullptr;       // grow-only workspace
  size_t ws_floats = 0;
  long long launches = 0;
  int device = -1;
  int sms = 148;
};

static int sm_c_cat(const pf_struct_config& c) { return c.heads * (c.c_z + c.c_ipa + 4 * c.n_pv); }
static int sm_proj_cols(const pf_struct_config& c) { return c.heads * (3 * c.c_ipa + 3 * (2 * c.n_qp + c.n_pv)); }

static SmOff sm_offsets(const pf_struct_config& c) {
  SmOff o{};
  size_t at = 0;
  auto take = [&](size_t n) { size_t r = at; at += n; return r; };
  const size_t cs = c.c_s, cz = c.c_z, cm = c.c_m, H = c.heads, ch = c.c_ipa, cr = c.c_resnet, cl = c.c_lddt;
  o.w_single = take(cm * cs); o.b_single = take(cs);
  o.ln_s_g = take(cs); o.ln_s_b = take(cs); o.ln_z_g = take(cz); o.ln_z_b = take(cz);
  o.w_in = take(cs * cs); o.b_in = take(cs);
  o.w_q = take(cs * H * ch); o.w_k = take(cs * H * ch); o.w_v = take(cs * H * ch);
  o.w_qp = take(cs * H * c.n_qp * 3); o.w_kp = take(cs * H * c.n_qp * 3); o.w_vp = take(cs * H * c.n_pv * 3);
  o.w_b = take(cz * H); o.g_head = take(H);
  o.w_out = take((size_t)sm_c_cat(c) * cs); o.b_out = take(cs);
  o.ln_ipa_g = take(cs); o.ln_ipa_b = take(cs);
  for (int i = 0; i < 3; ++i) { o.w_t[i] = take(cs * cs); o.b_t[i] = take(cs); }
  o.ln_tr_g = take(cs); o.ln_tr_b = take(cs);
  o.w_bb = take(cs * 6); o.b_bb = take(6);
  o.w_a1 = take(cs * cr); o.b_a1 = take(cr); o.w_a2 = take(cs * cr); o.b_a2 = take(cr);
  for (int r = 0; r < 2; ++r) { o.w_ra[r] = take(cr * cr); o.b_ra[r] = take(cr); o.w_rb[r] = take(cr * cr); o.b_rb[r] = take(cr); }
  o.w_alpha = take(cr * 2 * c.n_torsion); o.b_alpha = take(2 * (size_t)c.n_torsion);
  o.w_dg = take(cz * c.n_dist_bins); o.b_dg = take(c.n_dist_bins);
  o.w_mm = take(cm * c.n_msa_classes); o.b_mm = take(c.n_msa_classes);
  o.ln_l_g = take(cs); o.ln_l_b = take(cs);
  o.w_l1 = take(cs * cl); o.b_l1 = take(cl); o.w_l2 = take(cl * cl); o.b_l2 = take(cl);
  o.w_l3 = take(cl * c.n_lddt_bins); o.b_l3 = take(c.n_lddt_bins);
  o.w_pae = take(cz * c.n_pae_bins); o.b_pae = take(c.n_pae_bins);
  o.w_er = take(cs * c.n_resolved); o.b_er = take(c.n_resolved);
  o.total = at;
  return o;
}

// ------------------------------------------------------------------------------------------------
// kernels
// ------------------------------------------------------------------------------------------------
// Y[r, n] (+)= act( sum_k pre(X[row(r), k]) W[k, n] + b[n] ).  row(r) = r, or (r / rpb) * xbs + (r % rpb) * ldx when rpb > 0
// (the first MSA row of every protein: rpb = N, xbs = S N c_m).
struct SmGemm {
  const float* X;
  long ldx, xbs;
  int rpb;
  const float* W;      // [K, Nout] row-major
  const float* bias;   // [Nout] or null
  float* Y;
  long ldy;
  long R;
  int K, Nout;
  int pre_relu, act_relu, accumulate;
};

__global__ void __launch_bounds__(256) sm_gemm_kernel(const SmGemm g) {
  __shared__ __align__(16) float As[16][64 + 4];
  __shared__ __align__(16) float Bs[16][64 + 4];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const long r0 = (long)blockIdx.x * 64;
  const int n0 = blockIdx.y * 64;
  float acc[4][4] = {};
  const int arow = threadIdx.x >> 2, ak = (threadIdx.x & 3) * 4;
  const long ar = r0 + arow;
  const float* xrow = nullptr;
  if (ar < g.R) xrow = g.rpb > 0 ? g.X + (ar / g.rpb) * g.xbs + (ar % g.rpb) * g.ldx : g.X + ar * g.ldx;
  const int bk = threadIdx.x >> 4, bn = (threadIdx.x & 15) * 4;
  for (int k0 = 0; k0 < g.K; k0 += 16) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int k = k0 + ak + j;
      float v = (xrow && k < g.K) ? __ldg(xrow + k) : 0.f;
      if (g.pre_relu) v = fmaxf(v, 0.f);
      As[ak + j][arow] = v;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int k = k0 + bk, n = n0 + bn + j;
      Bs[bk][bn + j] = (k < g.K && n < g.Nout) ? __ldg(g.W + (long)k * g.Nout + n) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      const float4 a4 = *reinterpret_cast<const float4*>(&As[kk][ty * 4]);
      const float4 b4 = *reinterpret_cast<const float4*>(&Bs[kk][tx * 4]);
      const float a[4] = {a4.x, a4.y, a4.z, a4.w}, b[4] = {b4.x, b4.y, b4.z, b4.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const long r = r0 + ty * 4 + i;
    if (r >= g.R) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n >= g.Nout) continue;
      float v = acc[i][j] + (g.bias ? __ldg(g.bias + n) : 0.f);
      if (g.act_relu) v = fmaxf(v, 0.f);
      float* y = g.Y + r * g.ldy + n;
      *y = g.accumulate ? *y + v : v;
    }
  }
}

// four consecutive floats of a parameter vector (blob entries are only 4-byte aligned: some vectors have odd lengths)
__device__ __forceinline__ float4 ldg4u(const float* p) { return make_float4(__ldg(p), __ldg(p + 1), __ldg(p + 2), __ldg(p + 3)); }

// LayerNorm (R4) of rows of width C (multiple of 4, <= 1024), warp per row; y may alias x.
__global__ void __launch_bounds__(256) sm_ln_kernel(const float* x, float* y, const float* __restrict__ gamma,
                                                    const float* __restrict__ beta, long rows, int C) {
  const long r = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (r >= rows) return;
  const int lane = threadIdx.x & 31, nv = C >> 2;
  const float4* xp = reinterpret_cast<const float4*>(x + r * C);
  float4 v[8];
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int c4 = lane + 32 * i;
    v[i] = c4 < nv ? xp[c4] : make_float4(0.f, 0.f, 0.f, 0.f);
    s += (v[i].x + v[i].y) + (v[i].z + v[i].w);
  }
  const float mean = warp_sum(s) / (float)C;
  float q = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    if (lane + 32 * i < nv) {
      const float a = v[i].x - mean, b = v[i].y - mean, c = v[i].z - mean, d = v[i].w - mean;
      q += (a * a + b * b) + (c * c + d * d);
    }
  }
  const float rstd = rsqrtf(warp_sum(q) / (float)C + 1e-5f);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int c4 = lane + 32 * i;
    if (c4 < nv) {
      const float4 gm = ldg4u(gamma + 4 * c4), bt = ldg4u(beta + 4 * c4);
      float4 o;
      o.x = (v[i].x - mean) * rstd * gm.x + bt.x;
      o.y = (v[i].y - mean) * rstd * gm.y + bt.y;
      o.z = (v[i].z - mean) * rstd * gm.z + bt.z;
      o.w = (v[i].w - mean) * rstd * gm.w + bt.w;
      reinterpret_cast<float4*>(y + r * C)[c4] = o;
    }
  }
}

// M.1 / M.2: zn = LN_z(z) and b = Lin0(zn) [rows, H] in one pass; warp per pair row, W_b [c_z, H] in shared memory.
__global__ void __launch_bounds__(256) sm_pair_kernel(const float* __restrict__ z, float* __restrict__ zn, float* __restrict__ bias,
                                                      const float* __restrict__ gamma, const float* __restrict__ beta,
                                                      const float* __restrict__ wb, long rows, int C, int H) {
  extern __shared__ __align__(16) float swb[];   // [H, C]: head-major, so a lane reads its four channels of one head as one float4
  for (int i = threadIdx.x; i < C * H; i += blockDim.x) swb[(i % H) * C + i / H] = __ldg(wb + i);
  __syncthreads();
  const int lane = threadIdx.x & 31, nv = C >> 2;
  for (long r = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); r < rows; r += (long)gridDim.x * (blockDim.x >> 5)) {
    const float4* xp = reinterpret_cast<const float4*>(z + r * C);
    float4 v[8];
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int c4 = lane + 32 * i;
      v[i] = c4 < nv ? ld_nc_f4(xp + c4) : make_float4(0.f, 0.f, 0.f, 0.f);
      s += (v[i].x + v[i].y) + (v[i].z + v[i].w);
    }
    const float mean = warp_sum(s) / (float)C;
    float q = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if (lane + 32 * i < nv) {
        const float a = v[i].x - mean, b = v[i].y - mean, c = v[i].z - mean, d = v[i].w - mean;
        q += (a * a + b * b) + (c * c + d * d);
      }
    }
    const float rstd = rsqrtf(warp_sum(q) / (float)C + 1e-5f);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int c4 = lane + 32 * i;
      if (c4 < nv) {
        const float4 gm = ldg4u(gamma + 4 * c4), bt = ldg4u(beta + 4 * c4);
        v[i].x = (v[i].x - mean) * rstd * gm.x + bt.x;
        v[i].y = (v[i].y - mean) * rstd * gm.y + bt.y;
        v[i].z = (v[i].z - mean) * rstd * gm.z + bt.z;
        v[i].w = (v[i].w - mean) * rstd * gm.w + bt.w;
        reinterpret_cast<float4*>(zn + r * C)[c4] = v[i];
      }
    }
    // per-lane partial dot products of up to 16 heads at a time, then a reduce-scatter over the warp (16 shuffles for 16
    // heads instead of 5 per head): afterwards lanes 2 h and 2 h + 1 hold the sum of head h0 + h
    for (int h0 = 0; h0 < H; h0 += 16) {
      float p[16];
#pragma unroll
      for (int hh = 0; hh < 16; ++hh) {
        p[hh] = 0.f;
        if (h0 + hh < H) {
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int c4 = lane + 32 * i;
            if (c4 < nv) {
              const float4 w4 = *reinterpret_cast<const float4*>(swb + (size_t)(h0 + hh) * C + 4 * c4);
              p[hh] += (v[i].x * w4.x + v[i].y * w4.y) + (v[i].z * w4.z + v[i].w * w4.w);
            }
          }
        }
      }
      // 16 -> 8 -> 4 -> 2 -> 1 values per lane over lane bits 4, 3, 2, 1, then bit 0 adds the two halves
#pragma unroll
      for (int n = 8, m = 16; n >= 1; n >>= 1, m >>= 1) {
        const bool up = lane & m;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          if (j < n) {
            const float send = up ? p[j] : p[j + n];
            const float recv = __shfl_xor_sync(0xffffffffu, send, m);
            p[j] = (up ? p[j + n] : p[j]) + recv;
          }
        }
      }
      p[0] += __shfl_xor_sync(0xffffffffu, p[0], 1);
      // head index held by this lane: bits of the lane select the upper half at every step
      const int hh = ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
      if ((lane & 1) == 0 && h0 + hh < H) bias[r * H + h0 + hh] = p[0];
    }
  }
}

// frames [rows, 12] = R (row-major 3 x 3) | t
__global__ void sm_frames_init_kernel(float* frames, long rows) {
  const long r = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= rows) return;
  float* f = frames + r * 12;
  f[0] = 1.f; f[1] = 0.f; f[2] = 0.f; f[3] = 0.f; f[4] = 1.f; f[5] = 0.f; f[6] = 0.f; f[7] = 0.f; f[8] = 1.f;
  f[9] = 0.f; f[10] = 0.f; f[11] = 0.f;
}

// M.2: the projected points of every row (columns [pt0, pt0 + 3 npts) of proj) from the residue's frame to the global one.
__global__ void sm_points_kernel(float* __restrict__ proj, const float* __restrict__ frames, long rows, int P, int pt0, int npts) {
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= rows * npts) return;
  const long r = idx / npts;
  const int p = (int)(idx - r * npts);
  float* v = proj + r * P + pt0 + 3 * p;
  const float* f = frames + r * 12;
  const float x = v[0], y = v[1], z = v[2];
  v[0] = (f[0] * x + f[1] * y) + (f[2] * z + f[9]);
  v[1] = (f[3] * x + f[4] * y) + (f[5] * z + f[10]);
  v[2] = (f[6] * x + f[7] * y) + (f[8] * z + f[11]);
}

// M.2 for one query residue (b, i): blockDim = 32 H.  proj [rows, P] = q | k | v | qg | kg | vg (points already global),
// zn [B, N, N, cz], bias [B, N, N, H], cat [rows, H (cz + c + 4 Pv)] = ot | o | op | |op|.
struct SmIpa {
  const float* proj;
  const float* zn;
  const float* bias;
  const float* frames;
  const float* seq_mask;
  const float* g_head;
  float* cat;
  int N, H, c, Pq, Pv, cz, P;
};

// HQ = ceil(H / 4): the attention weights are kept key-major, att[j][4 HQ], so that the pair-value sum reads the weights of
// all heads for one key as HQ float4 and every pair value z[i, j, ch] exactly once per CTA.
template <int HQ>
__global__ void __launch_bounds__(1024) sm_ipa_kernel(const SmIpa a) {
  extern __shared__ __align__(16) float sm[];
  constexpr int HP = 4 * HQ;
  const int N = a.N, H = a.H, c = a.c, Pq = a.Pq, Pv = a.Pv, cz = a.cz;
  const int b = blockIdx.y, i = blockIdx.x;
  const long row = (long)b * N + i;
  float* att = sm;                              // [N, HP]
  const int G = blockDim.x >= (unsigned)cz ? (int)blockDim.x / cz : 1;   // key classes of the pair-value sum
  float* osum = att + (size_t)N * HP;           // [G, H cz]   partial pair-value sums, added in a fixed order (deterministic)
  float* qs = osum + (size_t)G * H * cz;        // [H c]
  float* qg = qs + H * c;                       // [H Pq 3]
  float* red = qg + H * Pq * 3;                 // [H (c + 3 Pv)]
  const int o_k = H * c, o_v = 2 * H * c, o_qg = 3 * H * c, o_kg = o_qg + H * Pq * 3, o_vg = o_kg + H * Pq * 3;
  const float* prow = a.proj + row * a.P;
  for (int t = threadIdx.x; t < H * c; t += blockDim.x) qs[t] = prow[t];
  for (int t = threadIdx.x; t < H * Pq * 3; t += blockDim.x) qg[t] = prow[o_qg + t];
  if (HP != H)
    for (int t = threadIdx.x; t < N * HP; t += blockDim.x) att[t] = 0.f;   // padded head columns stay zero
  __syncthreads();
  const int h = threadIdx.x >> 5, lane = threadIdx.x & 31;
  {
    const float w_l = sqrtf(1.0f / 3.0f), w_c = sqrtf(2.0f / (9.0f * (float)Pq));
    const float gh = __ldg(a.g_head + h);
    const float gamma = log1pf(expf(-fabsf(gh))) + fmaxf(gh, 0.f);          // softplus
    const float coef = gamma * w_c * 0.5f, inv_sqrt_c = rsqrtf((float)c);
    const float* brow = a.bias + (row * N) * H + h;
    float* acol = att + h;                      // this head's column, stride HP
    const bool vec = (c & 3) == 0 && ((Pq * 3) & 3) == 0 && (a.P & 3) == 0;   // 16-byte aligned segments of the projection row
    float mx = -INFINITY;
    for (int j = lane; j < N; j += 32) {
      const float* kr = a.proj + ((long)b * N + j) * a.P;
      float qk = 0.f, d2 = 0.f;
      if (vec) {
        const float4* k4 = reinterpret_cast<const float4*>(kr + o_k + h * c);
        const float4* q4 = reinterpret_cast<const float4*>(qs + h * c);
        for (int e = 0; e < c / 4; ++e) {
          const float4 kv = __ldg(k4 + e), qv = q4[e];
          qk = fmaf(qv.x, kv.x, qk); qk = fmaf(qv.y, kv.y, qk); qk = fmaf(qv.z, kv.z, qk); qk = fmaf(qv.w, kv.w, qk);
        }
        const float4* g4 = reinterpret_cast<const float4*>(kr + o_kg + h * Pq * 3);
        const float4* p4 = reinterpret_cast<const float4*>(qg + h * Pq * 3);
        for (int e = 0; e < Pq * 3 / 4; ++e) {
          const float4 kv = __ldg(g4 + e), qv = p4[e];
          const float dx = qv.x - kv.x, dy = qv.y - kv.y, dz = qv.z - kv.z, dw = qv.w - kv.w;
          d2 = fmaf(dx, dx, d2); d2 = fmaf(dy, dy, d2); d2 = fmaf(dz, dz, d2); d2 = fmaf(dw, dw, d2);
        }
      } else {
        for (int e = 0; e < c; ++e) qk = fmaf(qs[h * c + e], kr[o_k + h * c + e], qk);
        for (int e = 0; e < Pq * 3; ++e) {
          const float d = qg[h * Pq * 3 + e] - kr[o_kg + h * Pq * 3 + e];
          d2 = fmaf(d, d, d2);
        }
      }
      float lg = w_l * (qk * inv_sqrt_c + brow[(long)j * H] - coef * d2);
      if (!(a.seq_mask[(long)b * N + j] > 0.f)) lg = -INFINITY;
      acol[(size_t)j * HP] = lg;
      mx = fmaxf(mx, lg);
    }
    mx = warp_max(mx);
    float s = 0.f;
    for (int j = lane; j < N; j += 32) {
      const float e = (mx == -INFINITY) ? 0.f : expf(acol[(size_t)j * HP] - mx);
      acol[(size_t)j * HP] = e;
      s += e;
    }
    s = warp_sum(s);
    const float inv = s > 0.f ? 1.0f / s : 0.f;
    for (int j = lane; j < N; j += 32) acol[(size_t)j * HP] *= inv;
  }
  __syncthreads();
  float* crow = a.cat + row * ((long)H * (cz + c + 4 * Pv));
  // ot[h, ch] = sum_j a[h, j] zn[i, j, ch]: a thread owns one channel and a residue class of keys (G classes), reads z once
  // and the weights of all heads as HQ float4; the G partial sums meet in shared memory
  {
    const float* zrow = a.zn + (row * N) * cz;
    for (int ch0 = 0; ch0 < cz; ch0 += (int)blockDim.x) {       // one trip unless cz > blockDim.x
      const int t = threadIdx.x;
      const int g = G > 1 ? t / cz : 0;
      const int ch = G > 1 ? t - g * cz : ch0 + t;
      if (g < G && ch < cz) {
        float acc[HP];
#pragma unroll
        for (int q = 0; q < HP; ++q) acc[q] = 0.f;
        for (int j = g; j < N; j += G) {
          const float zv = __ldg(zrow + (long)j * cz + ch);
          const float4* aw = reinterpret_cast<const float4*>(att + (size_t)j * HP);
#pragma unroll
          for (int q = 0; q < HQ; ++q) {
            const float4 w4 = aw[q];
            acc[4 * q] = fmaf(w4.x, zv, acc[4 * q]);
            acc[4 * q + 1] = fmaf(w4.y, zv, acc[4 * q + 1]);
            acc[4 * q + 2] = fmaf(w4.z, zv, acc[4 * q + 2]);
            acc[4 * q + 3] = fmaf(w4.w, zv, acc[4 * q + 3]);
          }
        }
#pragma unroll
        for (int q = 0; q < HP; ++q)
          if (q < H) osum[((size_t)g * H + q) * cz + ch] = acc[q];
      }
    }
  }
  // o[h, e] and the global value-point sums og[h, p, x]
  const int per = c + 3 * Pv;
  for (int idx = threadIdx.x; idx < H * per; idx += blockDim.x) {
    const int hh = idx / per, e = idx - hh * per;
    const int col = e < c ? o_v + hh * c + e : o_vg + hh * Pv * 3 + (e - c);
    const float* vcol = a.proj + ((long)b * N) * a.P + col;
    float acc0 = 0.f, acc1 = 0.f;
    int j = 0;
    for (; j + 1 < N; j += 2) {
      acc0 = fmaf(att[(size_t)j * HP + hh], __ldg(vcol + (long)j * a.P), acc0);
      acc1 = fmaf(att[(size_t)(j + 1) * HP + hh], __ldg(vcol + (long)(j + 1) * a.P), acc1);
    }
    if (j < N) acc0 = fmaf(att[(size_t)j * HP + hh], __ldg(vcol + (long)j * a.P), acc0);
    red[idx] = acc0 + acc1;
  }
  __syncthreads();
  for (int idx = threadIdx.x; idx < H * cz; idx += blockDim.x) {
    float t = osum[idx];
    for (int g = 1; g < G; ++g) t += osum[(size_t)g * H * cz + idx];
    crow[idx] = t;
  }
  const float* f = a.frames + row * 12;
  for (int idx = threadIdx.x; idx < H * c; idx += blockDim.x) {
    const int hh = idx / c, e = idx - hh * c;
    crow[H * cz + idx] = red[hh * per + e];
  }
  for (int idx = threadIdx.x; idx < H * Pv; idx += blockDim.x) {
    const int hh = idx / Pv, p = idx - hh * Pv;
    const float* og = red + hh * per + c + 3 * p;
    const float dx = og[0] - f[9], dy = og[1] - f[10], dz = og[2] - f[11];
    const float lx = (f[0] * dx + f[3] * dy) + f[6] * dz;     // R^T (og - t)
    const float ly = (f[1] * dx + f[4] * dy) + f[7] * dz;
    const float lz = (f[2] * dx + f[5] * dy) + f[8] * dz;
    float* op = crow + H * (cz + c) + 3 * idx;
    op[0] = lx; op[1] = ly; op[2] = lz;
    crow[H * (cz + c + 3 * Pv) + idx] = sqrtf((lx * lx + ly * ly) + (lz * lz + 1e-8f));
  }
}

// M.4: T <- T o (R_upd, u) from bb [rows, 6] = (b, c, d, u); x = pos_scale t when x_out is given.
__global__ void sm_frames_kernel(float* __restrict__ frames, const float* __restrict__ bb, float* __restrict__ x_out,
                                 float pos_scale, long rows) {
  const long r = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= rows) return;
  const float* y = bb + r * 6;
  float* f = frames + r * 12;
  const float n = rsqrtf(1.0f + (y[0] * y[0] + y[1] * y[1]) + y[2] * y[2]);
  const float qa = n, qb = y[0] * n, qc = y[1] * n, qd = y[2] * n;
  float U[9];
  U[0] = qa * qa + qb * qb - qc * qc - qd * qd; U[1] = 2.f * (qb * qc - qa * qd); U[2] = 2.f * (qb * qd + qa * qc);
  U[3] = 2.f * (qb * qc + qa * qd); U[4] = qa * qa - qb * qb + qc * qc - qd * qd; U[5] = 2.f * (qc * qd - qa * qb);
  U[6] = 2.f * (qb * qd - qa * qc); U[7] = 2.f * (qc * qd + qa * qb); U[8] = qa * qa - qb * qb - qc * qc + qd * qd;
  float R[9], t[3];
#pragma unroll
  for (int k = 0; k < 9; ++k) R[k] = f[k];
#pragma unroll
  for (int k = 0; k < 3; ++k) t[k] = (R[3 * k] * y[3] + R[3 * k + 1] * y[4]) + (R[3 * k + 2] * y[5] + f[9 + k]);
#pragma unroll
  for (int ra = 0; ra < 3; ++ra)
#pragma unroll
    for (int cb = 0; cb < 3; ++cb) f[3 * ra + cb] = (R[3 * ra] * U[cb] + R[3 * ra + 1] * U[3 + cb]) + R[3 * ra + 2] * U[6 + cb];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    f[9 + k] = t[k];
    if (x_out) x_out[r * 3 + k] = pos_scale * t[k];
  }
}

// M.5: alpha_hat = alpha / sqrt(|alpha|^2 + 1e-12), pairs [n, 2]
__global__ void sm_alpha_kernel(const float* __restrict__ alpha, float* __restrict__ out, long pairs) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= pairs) return;
  const float a = alpha[2 * i], b = alpha[2 * i + 1];
  const float n = rsqrtf((a * a + b * b) + 1e-12f);
  out[2 * i] = a * n;
  out[2 * i + 1] = b * n;
}

// H.3: plddt = 100 sum_k softmax(l)_k (k + 1/2) / nb, warp per row
__global__ void __launch_bounds__(256) sm_plddt_kernel(const float* __restrict__ logits, float* __restrict__ out, long rows, int nb) {
  const long r = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (r >= rows) return;
  const int lane = threadIdx.x & 31;
  const float* l = logits + r * nb;
  float mx = -INFINITY;
  for (int k = lane; k < nb; k += 32) mx = fmaxf(mx, l[k]);
  mx = warp_max(mx);
  float s = 0.f, m = 0.f;
  for (int k = lane; k < nb; k += 32) {
    const float e = expf(l[k] - mx);
    s += e;
    m += e * ((float)k + 0.5f);
  }
  s = warp_sum(s);
  m = warp_sum(m);
  if (lane == 0) out[r] = 100.0f * m / (s * (float)nb);
}

// H.1: out[b, i, j, :] = half[b, i, j, :] + half[b, j, i, :], in place on half (each unordered pair by one thread)
__global__ void sm_symm_kernel(float* __restrict__ d, int N, int nb, long total) {
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;   // over (b, i, j, k)
  if (idx >= total) return;
  const int k = (int)(idx % nb);
  long t = idx / nb;
  const int j = (int)(t % N);
  t /= N;
  const int i = (int)(t % N);
  const long b = t / N;
  if (j < i) return;
  float* p = d + (((b * N + i) * N + j) * (long)nb + k);
  float* q = d + (((b * N + j) * N + i) * (long)nb + k);
  const float v = *p + *q;
  *p = v;
  *q = v;
}

// ------------------------------------------------------------------------------------------------
// host
// ------------------------------------------------------------------------------------------------
static bool sm_cfg_ok(const pf_struct_config& c) {
  return c.c_m >= 4 && c.c_m % 4 == 0 && c.c_m <= 1024 && c.c_z >= 4 && c.c_z % 4 == 0 && c.c_z <= 1024 && c.c_s >= 4 &&
         c.c_s % 4 == 0 && c.c_s <= 1024 && c.heads >= 1 && c.heads <= 32 && c.c_ipa >= 1 && c.c_ipa <= 64 && c.n_qp >= 1 &&
         c.n_qp <= 16 && c.n_pv >= 1 && c.n_pv <= 16 && c.n_layers >= 1 && c.c_resnet >= 1 && c.n_torsion >= 1 &&
         c.n_dist_bins >= 1 && c.n_msa_classes >= 1 && c.n_lddt_bins >= 1 && c.c_lddt >= 1 && c.n_pae_bins >= 1 &&
         c.n_resolved >= 1 && c.pos_scale > 0.f;
}

extern "C" size_t pf_structure_floats(const pf_struct_config* cfg) {
  if (!cfg || !sm_cfg_ok(*cfg)) return 0;
  return sm_offsets(*cfg).total;
}

extern "C" void pf_structure_destroy(pf_structure_t* h) {
  if (!h) return;
  cudaFree(h->w);
  cudaFree(h->w_proj);
  cudaFree(h->ws);
  delete h;
}

extern "C" long long pf_structure_last_launch_count(const pf_structure_t* h) { return h ? h->launches : 0; }

extern "C" pf_status pf_structure_create(pf_structure_t** out, const float* weights_host, size_t n_floats,
                                         const pf_struct_config* cfg) {
  if (!out || !weights_host || !cfg) return sfail(PF_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  if (!sm_cfg_ok(*cfg))
    return sfail(PF_ERR_SHAPE, "structure dims: channel counts multiples of 4 and <= 1024, heads <= 32, c_ipa <= 64, points <= 16");
  const SmOff off = sm_offsets(*cfg);
  if (n_floats != off.total) return sfail(PF_ERR_SHAPE, "structure weights blob length != pf_structure_floats(cfg)");
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return sfail(PF_ERR_CUDA, "cudaGetDevice");
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return sfail(PF_ERR_CUDA, "cudaGetDeviceProperties");
  if (prop.major != 10) return sfail(PF_ERR_ARCH, "this library is built for sm_100a (compute capability 10.x) only");
  pf_structure* h = new (std::nothrow) pf_structure();
  if (!h) return sfail(PF_ERR_ALLOC, "host alloc");
  h->cfg = *cfg;
  h->off = off;
  h->device = dev;
  h->sms = prop.multiProcessorCount;
  const pf_struct_config& c = *cfg;
  const int P = sm_proj_cols(c);
  // the six bias-free projections of M.2 as ONE [c_s, P] matrix: q | k | v | qp | kp | vp
  std::vector<float> wp((size_t)c.c_s * P);
  {
    const size_t srcs[6] = {off.w_q, off.w_k, off.w_v, off.w_qp, off.w_kp, off.w_vp};
    const int widths[6] = {c.heads * c.c_ipa, c.heads * c.c_ipa, c.heads * c.c_ipa, c.heads * c.n_qp * 3, c.heads * c.n_qp * 3,
                           c.heads * c.n_pv * 3};
    int col = 0;
    for (int m = 0; m < 6; ++m) {
      for (int k = 0; k < c.c_s; ++k)
        for (int n = 0; n < widths[m]; ++n) wp[(size_t)k * P + col + n] = weights_host[srcs[m] + (size_t)k * widths[m] + n];
      col += widths[m];
    }
  }
  if (cudaMalloc(&h->w, off.total * 4) != cudaSuccess || cudaMalloc(&h->w_proj, wp.size() * 4) != cudaSuccess) {
    cudaGetLastError();
    pf_structure_destroy(h);
    return sfail(PF_ERR_ALLOC, "cudaMalloc structure weights");
  }
  if (cudaMemcpy(h->w, weights_host, off.total * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(h->w_proj, wp.data(), wp.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
    pf_structure_destroy(h);
    return sfail(PF_ERR_CUDA, "structure weights H2D");
  }
  {
    cudaError_t ce = cudaSuccess;
    auto set = [&](const void* fn) { if (ce == cudaSuccess) ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); };
    set((const void*)sm_ipa_kernel<1>); set((const void*)sm_ipa_kernel<2>); set((const void*)sm_ipa_kernel<3>); set((const void*)sm_ipa_kernel<4>);
    set((const void*)sm_ipa_kernel<5>); set((const void*)sm_ipa_kernel<6>); set((const void*)sm_ipa_kernel<7>); set((const void*)sm_ipa_kernel<8>);
    if (ce != cudaSuccess) {
      pf_structure_destroy(h);
      return sfail(PF_ERR_CUDA, "cudaFuncSetAttribute(sm_ipa_kernel)");
    }
  }
  *out = h;
  return PF_OK;
}

namespace {
struct SmRun {
  pf_structure* h;
  cudaStream_t st;
  long long launches = 0;
  void gemm(const float* X, long ldx, const float* W, const float* bias, float* Y, long ldy, long R, int K, int Nout,
            bool pre_relu = false, bool act_relu = false, bool accumulate = false, int rpb = 0, long xbs = 0) {
    SmGemm g{X, ldx, xbs, rpb, W, bias, Y, ldy, R, K, Nout, pre_relu ? 1 : 0, act_relu ? 1 : 0, accumulate ? 1 : 0};
    dim3 grid((unsigned)((R + 63) / 64), (unsigned)((Nout + 63) / 64));
    sm_gemm_kernel<<<grid, 256, 0, st>>>(g);
    ++launches;
  }
  void ln(const float* x, float* y, const float* g, const float* b, long rows, int C) {
    sm_ln_kernel<<<(unsigned)((rows + 7) / 8), 256, 0, st>>>(x, y, g, b, rows, C);
    ++launches;
  }
};

bool sm_reserve(pf_structure* h, size_t need) {
  if (need <= h->ws_floats) return true;
  cudaDeviceSynchronize();
  cudaFree(h->ws);
  h->ws = nullptr;
  h->ws_floats = 0;
  if (cudaMalloc(&h->ws, need * 4) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  h->ws_floats = need;
  return true;
}
}  // namespace

extern "C" pf_status pf_structure_forward(pf_structure_t* h, const float* msa, const float* pair, const float* seq_mask, int B,
                                          int S, int N, int n_layers, float* s_out, float* frames_out, float* x_out,
                                          float* alpha_out, float* plddt_out, float* resolved_out, void* stream) {
  if (!h || !msa || !pair || !seq_mask) return sfail(PF_ERR_INVALID_ARG, "null argument");
  if (B < 1 || S < 1 || N < 1 || n_layers < 1) return sfail(PF_ERR_SHAPE, "B, S, N, n_layers must be >= 1");
  if (B > 65535) return sfail(PF_ERR_SHAPE, "structure module: B <= 65535");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device)
    return sfail(PF_ERR_INVALID_ARG, "the current device is not the one the structure handle was created on");
  const pf_struct_config& c = h->cfg;
  const SmOff& o = h->off;
  const int cs = c.c_s, cz = c.c_z, H = c.heads, P = sm_proj_cols(c), ccat = sm_c_cat(c), cr = c.c_resnet, cl = c.c_lddt;
  const long R = (long)B * N, PR = (long)B * N * N;
  const int HQ = (H + 3) / 4;
  const int ipa_g = 32 * H >= cz ? 32 * H / cz : 1;
  const size_t ipa_smem = ((size_t)4 * HQ * N + (size_t)ipa_g * H * cz + (size_t)H * c.c_ipa + (size_t)H * c.n_qp * 3 + (size_t)H * (c.c_ipa + 3 * c.n_pv)) * 4;
  if (ipa_smem > 200 * 1024) return sfail(PF_ERR_SHAPE, "structure module: heads x N_res attention weights exceed 200 KB of shared memory");
  // workspace
  size_t at = 0;
  auto take = [&](size_t n) { size_t r = at; at += (n + 3) & ~(size_t)3; return r; };
  const size_t o_zn = take((size_t)PR * cz), o_bias = take((size_t)PR * H), o_single = take((size_t)R * cs), o_sinit = take((size_t)R * cs),
               o_s = take((size_t)R * cs), o_t1 = take((size_t)R * cs), o_t2 = take((size_t)R * cs), o_proj = take((size_t)R * P),
               o_cat = take((size_t)R * ccat), o_frames = take((size_t)R * 12), o_bb = take((size_t)R * 8),
               o_a = take((size_t)R * cr), o_u = take((size_t)R * cr), o_alpha = take((size_t)R * 2 * c.n_torsion),
               o_l1 = take((size_t)R * cl), o_l2 = take((size_t)R * cl), o_lg = take((size_t)R * c.n_lddt_bins);
  if (!sm_reserve(h, at)) return sfail(PF_ERR_ALLOC, "cudaMalloc structure workspace");
  float* ws = h->ws;
  const float* w = h->w;
  SmRun run{h, reinterpret_cast<cudaStream_t>(stream)};
  cudaStream_t st = run.st;
  float *zn = ws + o_zn, *bias = ws + o_bias, *single = ws + o_single, *sinit = ws + o_sinit, *s = ws + o_s, *t1 = ws + o_t1,
        *t2 = ws + o_t2, *proj = ws + o_proj, *cat = ws + o_cat, *frames = ws + o_frames, *bb = ws + o_bb, *a = ws + o_a,
        *u = ws + o_u, *alpha = ws + o_alpha, *l1 = ws + o_l1, *l2 = ws + o_l2, *lg = ws + o_lg;
  // M.0, M.1
  run.gemm(msa, c.c_m, w + o.w_single, w + o.b_single, single, cs, R, c.c_m, cs, false, false, false, N, (long)S * N * c.c_m);
  run.ln(single, sinit, w + o.ln_s_g, w + o.ln_s_b, R, cs);
  {
    const unsigned grid = (unsigned)std::max(1L, std::min((PR + 7) / 8, (long)h->sms * 8));
    sm_pair_kernel<<<grid, 256, (size_t)cz * H * 4, st>>>(pair, zn, bias, w + o.ln_z_g, w + o.ln_z_b, w + o.w_b, PR, cz, H);
    ++run.launches;
  }
  run.gemm(sinit, cs, w + o.w_in, w + o.b_in, s, cs, R, cs, cs);
  sm_frames_init_kernel<<<(unsigned)((R + 255) / 256), 256, 0, st>>>(frames, R);
  ++run.launches;
  const int npts = H * (2 * c.n_qp + c.n_pv), pt0 = 3 * H * c.c_ipa;
  for (int l = 0; l < n_layers; ++l) {
    // M.2
    run.gemm(s, cs, h->w_proj, nullptr, proj, P, R, cs, P);
    sm_points_kernel<<<(unsigned)((R * npts + 255) / 256), 256, 0, st>>>(proj, frames, R, P, pt0, npts);
    ++run.launches;
    SmIpa ia{proj, zn, bias, frames, seq_mask, w + o.g_head, cat, N, H, c.c_ipa, c.n_qp, c.n_pv, cz, P};
    {
      const dim3 grid((unsigned)N, (unsigned)B);
      switch (HQ) {
        case 1: sm_ipa_kernel<1><<<grid, 32 * H, ipa_smem, st>>>(ia); break;
        case 2: sm_ipa_kernel<2><<<grid, 32 * H, ipa_smem, st>>>(ia); break;
        case 3: sm_ipa_kernel<3><<<grid, 32 * H, ipa_smem, st>>>(ia); break;
        case 4: sm_ipa_kernel<4><<<grid, 32 * H, ipa_smem, st>>>(ia); break;
        case 5: sm_ipa_kernel<5><<<grid, 32 * H, ipa_smem, st>>>(ia); break;
        case 6: sm_ipa_kernel<6><<<grid, 32 * H, ipa_smem, st>>>(ia); break;
        case 7: sm_ipa_kernel<7><<<grid, 32 * H, ipa_smem, st>>>(ia); break;
        default: sm_ipa_kernel<8><<<grid, 32 * H, ipa_smem, st>>>(ia); break;
      }
    }
    ++run.launches;
    // M.3
    run.gemm(cat, ccat, w + o.w_out, w + o.b_out, s, cs, R, ccat, cs, false, false, true);
    run.ln(s, s, w + o.ln_ipa_g, w + o.ln_ipa_b, R, cs);
    run.gemm(s, cs, w + o.w_t[0], w + o.b_t[0], t1, cs, R, cs, cs, false, true);
    run.gemm(t1, cs, w + o.w_t[1], w + o.b_t[1], t2, cs, R, cs, cs, false, true);
    run.gemm(t2, cs, w + o.w_t[2], w + o.b_t[2], s, cs, R, cs, cs, false, false, true);
    run.ln(s, s, w + o.ln_tr_g, w + o.ln_tr_b, R, cs);
    // M.4
    run.gemm(s, cs, w + o.w_bb, w + o.b_bb, bb, 6, R, cs, 6);
    sm_frames_kernel<<<(unsigned)((R + 255) / 256), 256, 0, st>>>(frames, bb, (l == n_layers - 1) ? x_out : nullptr, c.pos_scale, R);
    ++run.launches;
  }
  if (alpha_out) {   // M.5
    run.gemm(s, cs, w + o.w_a1, w + o.b_a1, a, cr, R, cs, cr);
    run.gemm(sinit, cs, w + o.w_a2, w + o.b_a2, a, cr, R, cs, cr, false, false, true);
    for (int r = 0; r < 2; ++r) {
      run.gemm(a, cr, w + o.w_ra[r], w + o.b_ra[r], u, cr, R, cr, cr, true, true);
      run.gemm(u, cr, w + o.w_rb[r], w + o.b_rb[r], a, cr, R, cr, cr, false, false, true);
    }
    run.gemm(a, cr, w + o.w_alpha, w + o.b_alpha, alpha, 2 * c.n_torsion, R, cr, 2 * c.n_torsion, true);
    const long pairs = R * c.n_torsion;
    sm_alpha_kernel<<<(unsigned)((pairs + 255) / 256), 256, 0, st>>>(alpha, alpha_out, pairs);
    ++run.launches;
  }
  if (plddt_out) {   // H.3
    run.ln(s, t1, w + o.ln_l_g, w + o.ln_l_b, R, cs);
    run.gemm(t1, cs, w + o.w_l1, w + o.b_l1, l1, cl, R, cs, cl, false, true);
    run.gemm(l1, cl, w + o.w_l2, w + o.b_l2, l2, cl, R, cl, cl, false, true);
    run.gemm(l2, cl, w + o.w_l3, w + o.b_l3, lg, c.n_lddt_bins, R, cl, c.n_lddt_bins);
    sm_plddt_kernel<<<(unsigned)((R + 7) / 8), 256, 0, st>>>(lg, plddt_out, R, c.n_lddt_bins);
    ++run.launches;
  }
  if (resolved_out)   // H.5
    run.gemm(s, cs, w + o.w_er, w + o.b_er, resolved_out, c.n_resolved, R, cs, c.n_resolved);
  if (s_out) cudaMemcpyAsync(s_out, s, (size_t)R * cs * 4, cudaMemcpyDeviceToDevice, st);
  if (frames_out) cudaMemcpyAsync(frames_out, frames, (size_t)R * 12 * 4, cudaMemcpyDeviceToDevice, st);
  h->launches = run.launches;
  cudaError_t ce = cudaGetLastError();
  if (ce != cudaSuccess) return sfail(PF_ERR_CUDA, std::string("structure module launch failed: ") + cudaGetErrorString(ce));
  return PF_OK;
}

extern "C" pf_status pf_heads_forward(pf_structure_t* h, const float* msa, const float* pair, int B, int S, int N,
                                      float* distogram_out, float* masked_msa_out, float* pae_out, void* stream) {
  if (!h) return sfail(PF_ERR_INVALID_ARG, "null handle");
  if (((distogram_out || pae_out) && !pair) || (masked_msa_out && !msa)) return sfail(PF_ERR_INVALID_ARG, "a head was requested without its input");
  if (B < 1 || S < 1 || N < 1) return sfail(PF_ERR_SHAPE, "B, S, N must be >= 1");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device)
    return sfail(PF_ERR_INVALID_ARG, "the current device is not the one the structure handle was created on");
  const pf_struct_config& c = h->cfg;
  const SmOff& o = h->off;
  SmRun run{h, reinterpret_cast<cudaStream_t>(stream)};
  if (distogram_out) {   // H.1
    const long PR = (long)B * N * N;
    run.gemm(pair, c.c_z, h->w + o.w_dg, h->w + o.b_dg, distogram_out, c.n_dist_bins, PR, c.c_z, c.n_dist_bins);
    const long total = PR * c.n_dist_bins;
    sm_symm_kernel<<<(unsigned)((total + 255) / 256), 256, 0, run.st>>>(distogram_out, N, c.n_dist_bins, total);
    ++run.launches;
  }
  if (pae_out)           // H.4
    run.gemm(pair, c.c_z, h->w + o.w_pae, h->w + o.b_pae, pae_out, c.n_pae_bins, (long)B * N * N, c.c_z, c.n_pae_bins);
  if (masked_msa_out)    // H.2
    run.gemm(msa, c.c_m, h->w + o.w_mm, h->w + o.b_mm, masked_msa_out, c.n_msa_classes, (long)B * S * N, c.c_m, c.n_msa_classes);
  h->launches = run.launches;
  cudaError_t ce = cudaGetLastError();
  if (ce != cudaSuccess) return sfail(PF_ERR_CUDA, std::string("heads launch failed: ") + cudaGetErrorString(ce));
  return PF_OK;
}

// ------------------------------------------------------------------------------------------------
// H.3 without any allocation (pf_plddt_forward_static, include/pf_evoformer.h): the same five launches as the pLDDT tail of
// pf_structure_forward, their intermediates (LN_l(s), two hidden layers, logits) in a file-scope device array instead of the
// handle's cudaMalloc'ed workspace.  Every GPU that loads this library holds the array (PF_PLDDT_STATIC_SCRATCH_BYTES) until the
// process exits.  In host code `sm_static_scratch` is the host-side stand-in of the symbol, NOT a device address: the address
// kernels may dereference comes from cudaGetSymbolAddress, resolved once per device with that device current.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) float sm_static_scratch[PF_PLDDT_STATIC_SCRATCH_BYTES / 4];

namespace {
constexpr int kStaticMaxDevices = 64;
std::mutex sm_static_mu;
float* sm_static_ptr[kStaticMaxDevices] = {};   // device address of sm_static_scratch, by device ordinal

// `dev` must be the current device
pf_status sm_static_scratch_for(int dev, float** out) {
  if (dev < 0 || dev >= kStaticMaxDevices) return sfail(PF_ERR_INVALID_ARG, "pf_plddt_forward_static: device ordinal >= 64");
  std::lock_guard<std::mutex> lk(sm_static_mu);
  if (!sm_static_ptr[dev]) {
    void* p = nullptr;
    const cudaError_t ce = cudaGetSymbolAddress(&p, sm_static_scratch);
    if (ce != cudaSuccess || !p) {
      cudaGetLastError();
      return sfail(PF_ERR_CUDA, std::string("pf_plddt_forward_static: cudaGetSymbolAddress(sm_static_scratch): ") +
                                    (ce != cudaSuccess ? cudaGetErrorString(ce) : "null address"));
    }
    sm_static_ptr[dev] = static_cast<float*>(p);
  }
  *out = sm_static_ptr[dev];
  return PF_OK;
}
}  // namespace

extern "C" pf_status pf_plddt_forward_static(pf_structure_t* h, const float* s, int rows, float* plddt_out, void* stream) {
  if (!h || !s || !plddt_out) return sfail(PF_ERR_INVALID_ARG, "null argument");
  if (rows < 1) return sfail(PF_ERR_SHAPE, "pf_plddt_forward_static: rows must be >= 1");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device)
    return sfail(PF_ERR_INVALID_ARG, "the current device is not the one the structure handle was created on");
  const pf_struct_config& c = h->cfg;
  const SmOff& o = h->off;
  const int cs = c.c_s, cl = c.c_lddt, nb = c.n_lddt_bins;
  const long R = rows;
  // four segments, each starting on a 256-byte boundary of the array
  size_t at = 0;
  auto take = [&](size_t n) { size_t r = at; at += (n + 63) & ~(size_t)63; return r; };
  const size_t o_ln = take((size_t)R * cs), o_l1 = take((size_t)R * cl), o_l2 = take((size_t)R * cl), o_lg = take((size_t)R * nb);
  const size_t cap = PF_PLDDT_STATIC_SCRATCH_BYTES / 4;
  if (at > cap) {
    const size_t per_row = (size_t)cs + 2 * (size_t)cl + nb;
    return sfail(PF_ERR_SHAPE, "pf_plddt_forward_static: " + std::to_string(rows) + " rows need " + std::to_string(at * 4) +
                                   " bytes of scratch, the static array holds " + std::to_string((size_t)PF_PLDDT_STATIC_SCRATCH_BYTES) +
                                   " (about " + std::to_string((cap - 4 * 64) / per_row) + " rows at these dims); use pf_structure_forward");
  }
  float* scratch = nullptr;
  const pf_status ps = sm_static_scratch_for(dev, &scratch);
  if (ps != PF_OK) return ps;
  // nothing in the array has to start at zero: every element a launch reads was written by the launch before it in this call
  // (LayerNorm and the non-accumulating GEMMs overwrite their whole [rows, width] output)
  const float* w = h->w;
  float *ln = scratch + o_ln, *l1 = scratch + o_l1, *l2 = scratch + o_l2, *lg = scratch + o_lg;
  SmRun run{h, reinterpret_cast<cudaStream_t>(stream)};
  run.ln(s, ln, w + o.ln_l_g, w + o.ln_l_b, R, cs);
  run.gemm(ln, cs, w + o.w_l1, w + o.b_l1, l1, cl, R, cs, cl, false, true);
  run.gemm(l1, cl, w + o.w_l2, w + o.b_l2, l2, cl, R, cl, cl, false, true);
  run.gemm(l2, cl, w + o.w_l3, w + o.b_l3, lg, nb, R, cl, nb);
  sm_plddt_kernel<<<(unsigned)((R + 7) / 8), 256, 0, run.st>>>(lg, plddt_out, R, nb);
  ++run.launches;
  h->launches = run.launches;
  const cudaError_t ce = cudaGetLastError();
  if (ce != cudaSuccess) return sfail(PF_ERR_CUDA, std::string("pf_plddt_forward_static launch failed: ") + cudaGetErrorString(ce));
  return PF_OK;
}

extern "C" pf_status pf_fold_forward(pf_evoformer_t* h, pf_embedder_t* e, pf_extra_msa_t* x, pf_structure_t* sm,
                                     const float* target_feat, const int* residue_index, const float* msa_feat,
                                     const float* x_prev0, const float* extra_msa_feat, float* extra_msa,
                                     const float* extra_msa_mask, float* msa, float* pair, const float* seq_mask,
                                     const float* msa_mask, int B, int S, int S_e, int N, int n_blocks, int n_extra_blocks,
                                     int n_cycles, int n_layers, float* x_cycles_out, float* s_out, float* frames_out,
                                     float* alpha_out, float* plddt_out, void* stream) {
  if (!h || !e || !sm) return sfail(PF_ERR_INVALID_ARG, "null handle");
  if (!x_cycles_out) return sfail(PF_ERR_INVALID_ARG, "x_cycles_out is required");
  if (n_cycles < 1) return sfail(PF_ERR_SHAPE, "n_cycles must be >= 1");
  if (x && (!extra_msa_feat || !extra_msa || !extra_msa_mask))
    return sfail(PF_ERR_INVALID_ARG, "extra-MSA stack given without its features / buffer / mask");
  long long launches = 0;
  const size_t xs = (size_t)B * N * 3;
  for (int c = 0; c < n_cycles; ++c) {
    const float* xp = c == 0 ? x_prev0 : x_cycles_out + (size_t)(c - 1) * xs;
    pf_status s = pf_embedder_forward(e, target_feat, residue_index, msa_feat, xp, c > 0 ? 1 : 0, msa, pair, B, S, N, stream);
    if (s != PF_OK) return s;
    launches += pf_embedder_last_launch_count(e);
    if (x) {
      s = pf_embedder_forward_extra(e, extra_msa_feat, extra_msa, B, S_e, N, stream);
      if (s != PF_OK) return s;
      launches += pf_embedder_last_launch_count(e);
      s = pf_extra_msa_forward(x, extra_msa, pair, seq_mask, extra_msa_mask, B, S_e, N, n_extra_blocks, stream);
      if (s != PF_OK) return s;
      launches += pf_extra_msa_last_launch_count(x);
    }
    s = pf_evoformer_forward(h, msa, pair, seq_mask, msa_mask, B, S, N, n_blocks, stream);
    if (s != PF_OK) return s;
    launches += pf_evoformer_last_launch_count(h);
    const bool last = c == n_cycles - 1;
    s = pf_structure_forward(sm, msa, pair, seq_mask, B, S, N, n_layers, last ? s_out : nullptr, last ? frames_out : nullptr,
                             x_cycles_out + (size_t)c * xs, last ? alpha_out : nullptr, last ? plddt_out : nullptr, nullptr, stream);
    if (s != PF_OK) return s;
    launches += sm->launches;
  }
  sm->launches = launches;
  return PF_OK;
}
