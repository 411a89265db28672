// Extra-MSA stack (readings X.1-X.9 of DESIGN.md §2c): the Evoformer block at
// c_e = 64 MSA channels with GLOBAL column attention, N_seq in the thousands, over the same pair representation.
//   X.1 row attention with pair bias   tcgen05 path of the main block: LayerNorm-fused projection (K = 64), heads of dimension 8
//                                      zero-padded to the 32 the attention core is built for, out-projection + residual
//   X.2 global column attention        two fp32 SIMT kernels below (reduction lengths 8 .. 64: HBM-bound elementwise work)
//   X.3 transition                     LayerNorm-fused GEMM (K = 64) + ReLU, second GEMM reduce-added into e
//   X.4 outer-product-mean             projection GEMM (K = 64) + the main block's tensor-core core, contraction chunked over s
//   X.5-X.9 pair stack                 the main block's kernels, unchanged
// Implementation: the handle wraps an inner pf_evoformer (main dims) that owns the pair-stack weights of the extra blocks, the
// pair-bias projection of X.1, the outer-product output projection and the workspace arena; this file owns the MSA-side
// parameters, re-laid out for the kernels above.
#include "pf_handle.h"
#include "pf_device.cuh"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <string>
#include <vector>

using namespace pf;

namespace pf { void api_set_error(const std::string& s); }
static pf_status xfail(pf_status s, const std::string& msg) {
  api_set_error(msg);
  return s;
}

struct pf_extra_msa {
  pf_extra_config cfg;
  pf_evoformer* inner = nullptr;
  ExtraOff off;
  ExtraT xt;
  float* w32 = nullptr;
  uint16_t* w16 = nullptr;
  float* wf = nullptr;
  float* o_glob = nullptr;
  size_t o_glob_floats = 0;
  long long launches = 0;
};

// ------------------------------------------------------------------------------------------------
// X.2 global column attention
// ------------------------------------------------------------------------------------------------
constexpr int XG_C = 64;         // c_e
constexpr int XG_MAXD = 16;      // key + value dimensions together (2 x head dimension 8)

// Kernel A, one block per column (b, i): x_s = LN(e[s,i]) for all s; qbar = sum_s mu_s x_s / (sum_s mu_s + 1e-10);
// k_s | v_s = x_s [W_k | W_v] kept in shared memory; q = qbar W_q / sqrt(d); per head h (one warp each):
// o_h = sum_s softmax_s(q_h . k_s + NEG(mu_s)) v_s  ->  o_glob[b, i, h d .. h d + d)
__global__ void __launch_bounds__(256) extra_global_col_a_kernel(const float* __restrict__ e, const float* __restrict__ seq_mask,
                                                                 const float* __restrict__ msa_mask, const float* __restrict__ w,
                                                                 GlobalColW o, float* __restrict__ o_glob, int S, int N, int H) {
  extern __shared__ __align__(16) float sm[];
  const int d = XG_C / H;                     // head dimension
  float* kv = sm;                             // [S][2 d]
  float* wkv = kv + (size_t)S * 2 * d;        // [64][2 d]
  float* xrow = wkv + XG_C * 2 * d;           // [8 warps][64]
  float* qpart = xrow + 8 * XG_C;             // [8 warps][64]
  float* cpart = qpart + 8 * XG_C;            // [8]
  float* qv = cpart + 8;                      // [64]
  float* mus = qv + XG_C;                     // [S]
  const int i = blockIdx.x, b = blockIdx.y;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int t = threadIdx.x; t < XG_C * d; t += 256) {
    const int k = t / d, c = t % d;
    wkv[k * 2 * d + c] = __ldg(w + o.wk + k * d + c);
    wkv[k * 2 * d + d + c] = __ldg(w + o.wv + k * d + c);
  }
  const float sig = seq_mask[(long)b * N + i];
  for (int s = threadIdx.x; s < S; s += 256) mus[s] = msa_mask[(long)b * S + s] * sig;
  __syncthreads();
  const float2 g = __ldg(reinterpret_cast<const float2*>(w + o.ln_g) + lane), be = __ldg(reinterpret_cast<const float2*>(w + o.ln_b) + lane);
  float q0 = 0.f, q1 = 0.f, cnt = 0.f;
  for (int s = warp; s < S; s += 8) {
    const float2 v = __ldg(reinterpret_cast<const float2*>(e + (((long)b * S + s) * N + i) * XG_C) + lane);
    const float mean = warp_sum(v.x + v.y) * (1.0f / XG_C);
    const float a0 = v.x - mean, a1 = v.y - mean;
    const float rstd = rsqrtf(warp_sum(a0 * a0 + a1 * a1) * (1.0f / XG_C) + 1e-5f);
    const float x0 = a0 * rstd * g.x + be.x, x1 = a1 * rstd * g.y + be.y;
    const float mu = mus[s];
    q0 = fmaf(mu, x0, q0);
    q1 = fmaf(mu, x1, q1);
    cnt += mu;
    reinterpret_cast<float2*>(xrow + warp * XG_C)[lane] = make_float2(x0, x1);
    __syncwarp();
    // k_s | v_s: output c = lane % (2 d) from the half lane / (2 d) of the reduction (2 d = 16: two halves of 32 inputs)
    const int c = lane % (2 * d), half = lane / (2 * d), per = XG_C / (32 / (2 * d));
    float acc = 0.f;
    for (int k = half * per; k < (half + 1) * per; ++k) acc = fmaf(xrow[warp * XG_C + k], wkv[k * 2 * d + c], acc);
    for (int off = 2 * d; off < 32; off <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if (lane < 2 * d) kv[(size_t)s * 2 * d + lane] = acc;
    __syncwarp();
  }
  reinterpret_cast<float2*>(qpart + warp * XG_C)[lane] = make_float2(q0, q1);
  if (lane == 0) cpart[warp] = cnt;
  __syncthreads();
  if (threadIdx.x < XG_C) {
    float a = 0.f, n = 0.f;
    for (int wv = 0; wv < 8; ++wv) {
      a += qpart[wv * XG_C + threadIdx.x];
      n += cpart[wv];
    }
    xrow[threadIdx.x] = a / (n + 1e-10f);      // qbar (xrow is free now)
  }
  __syncthreads();
  if (threadIdx.x < XG_C) {
    float a = 0.f;
    for (int k = 0; k < XG_C; ++k) a = fmaf(xrow[k], __ldg(w + o.wq + k * XG_C + threadIdx.x), a);
    qv[threadIdx.x] = a * rsqrtf((float)d);
  }
  __syncthreads();
  for (int h = warp; h < H; h += 8) {
    float qh[XG_MAXD / 2];
    for (int c = 0; c < d; ++c) qh[c] = qv[h * d + c];
    float mx = -INFINITY;
    for (int s = lane; s < S; s += 32) {
      float l = 0.f;
      for (int c = 0; c < d; ++c) l = fmaf(qh[c], kv[(size_t)s * 2 * d + c], l);
      l += 1e9f * (mus[s] - 1.0f);
      mx = fmaxf(mx, l);
    }
    mx = warp_max(mx);
    float den = 0.f, acc[XG_MAXD / 2];
    for (int c = 0; c < d; ++c) acc[c] = 0.f;
    for (int s = lane; s < S; s += 32) {
      float l = 0.f;
      for (int c = 0; c < d; ++c) l = fmaf(qh[c], kv[(size_t)s * 2 * d + c], l);
      l += 1e9f * (mus[s] - 1.0f);
      const float p = expf(l - mx);
      den += p;
      for (int c = 0; c < d; ++c) acc[c] = fmaf(p, kv[(size_t)s * 2 * d + d + c], acc[c]);
    }
    den = warp_sum(den);
    for (int c = 0; c < d; ++c) acc[c] = warp_sum(acc[c]);
    if (lane < d) o_glob[((long)b * N + i) * XG_C + h * d + lane] = acc[lane] / den;
  }
}

// Kernel B, one warp per row (b, s, i): e[s,i] += Lin_o( sigmoid(Lin_g(LN(e[s,i]))) (.) o_glob[b,i] )
__global__ void __launch_bounds__(256) extra_global_col_b_kernel(float* __restrict__ e, const float* __restrict__ seq_mask,
                                                                 const float* __restrict__ msa_mask, const float* __restrict__ w,
                                                                 GlobalColW o, const float* __restrict__ o_glob, int S, int N,
                                                                 long rows) {
  __shared__ __align__(16) float wg[XG_C * XG_C], wo[XG_C * XG_C], rowbuf[8][XG_C];
  for (int t = threadIdx.x; t < XG_C * XG_C; t += 256) {
    wg[t] = __ldg(w + o.wg + t);
    wo[t] = __ldg(w + o.wo + t);
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const long warp = (long)blockIdx.x * 8 + wib, nwarps = (long)gridDim.x * 8;
  const float2 g = __ldg(reinterpret_cast<const float2*>(w + o.ln_g) + lane), be = __ldg(reinterpret_cast<const float2*>(w + o.ln_b) + lane);
  const float2 bg = __ldg(reinterpret_cast<const float2*>(w + o.bg) + lane), bo = __ldg(reinterpret_cast<const float2*>(w + o.bo) + lane);
  for (long r = warp; r < rows; r += nwarps) {
    const long bs = r / N;
    const int i = (int)(r - bs * N);
    const long b = bs / S;
    // rows at masked positions are skipped: their outputs are unspecified (R3) and stay what they were (finite)
    if (msa_mask[bs] * seq_mask[b * N + i] < 0.5f) continue;
    float2* ep = reinterpret_cast<float2*>(e + r * XG_C) + lane;
    const float2 v = *ep;
    const float mean = warp_sum(v.x + v.y) * (1.0f / XG_C);
    const float a0 = v.x - mean, a1 = v.y - mean;
    const float rstd = rsqrtf(warp_sum(a0 * a0 + a1 * a1) * (1.0f / XG_C) + 1e-5f);
    reinterpret_cast<float2*>(rowbuf[wib])[lane] = make_float2(a0 * rstd * g.x + be.x, a1 * rstd * g.y + be.y);
    __syncwarp();
    float g0 = bg.x, g1 = bg.y;
#pragma unroll 8
    for (int k = 0; k < XG_C; ++k) {
      const float xk = rowbuf[wib][k];
      const float2 wv = reinterpret_cast<const float2*>(wg + k * XG_C)[lane];
      g0 = fmaf(xk, wv.x, g0);
      g1 = fmaf(xk, wv.y, g1);
    }
    const float2 og = __ldg(reinterpret_cast<const float2*>(o_glob + (b * N + i) * XG_C) + lane);
    __syncwarp();
    reinterpret_cast<float2*>(rowbuf[wib])[lane] = make_float2(og.x * sigmoidf_acc(g0), og.y * sigmoidf_acc(g1));
    __syncwarp();
    float u0 = bo.x, u1 = bo.y;
#pragma unroll 8
    for (int k = 0; k < XG_C; ++k) {
      const float tk = rowbuf[wib][k];
      const float2 wv = reinterpret_cast<const float2*>(wo + k * XG_C)[lane];
      u0 = fmaf(tk, wv.x, u0);
      u1 = fmaf(tk, wv.y, u1);
    }
    __syncwarp();
    *ep = make_float2(v.x + u0, v.y + u1);
  }
}

static size_t global_a_smem(int S, int H) {
  const int d = XG_C / H;
  return ((size_t)S * 2 * d + XG_C * 2 * d + 8 * XG_C + 8 * XG_C + 8 + XG_C + (size_t)S) * sizeof(float);
}

void pf::launch_extra_global_col(float* e, const float* seq_mask, const float* msa_mask, const float* w32, const GlobalColW& o,
                                 float* o_glob, int B, int S, int N, int c_e, int heads, cudaStream_t st) {
  (void)c_e;
  extra_global_col_a_kernel<<<dim3((unsigned)N, (unsigned)B), 256, global_a_smem(S, heads), st>>>(e, seq_mask, msa_mask, w32, o,
                                                                                                 o_glob, S, N, heads);
  const long rows = (long)B * S * N;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const long blocks = std::max(1L, std::min((rows + 7) / 8, (long)sms * 8));
  extra_global_col_b_kernel<<<(unsigned)blocks, 256, 0, st>>>(e, seq_mask, msa_mask, w32, o, o_glob, S, N, rows);
}

// ------------------------------------------------------------------------------------------------
// weights
// ------------------------------------------------------------------------------------------------
static AttnW x_attn_offsets(size_t& o, int c, int heads, int bias_kind, int c_bias) {
  AttnW a{};
  auto take = [&](size_t n) { size_t r = o; o += n; return r; };
  a.ln_g = take(c); a.ln_b = take(c);
  if (bias_kind == 1) { a.ln_z_g = take(c_bias); a.ln_z_b = take(c_bias); }
  if (bias_kind) a.w_bias = take((size_t)c_bias * heads);
  a.wq = take((size_t)c * c); a.wk = take((size_t)c * c); a.wv = take((size_t)c * c);
  a.wg = take((size_t)c * c); a.bg = take(c);
  a.wo = take((size_t)c * c); a.bo = take(c);
  return a;
}
static TransW x_trans_offsets(size_t& o, int c, int n) {
  TransW t{};
  auto take = [&](size_t k) { size_t r = o; o += k; return r; };
  t.ln_g = take(c); t.ln_b = take(c);
  t.w1 = take((size_t)c * n * c); t.b1 = take((size_t)n * c);
  t.w2 = take((size_t)n * c * c); t.b2 = take(c);
  return t;
}
static TriMulW x_trimul_offsets(size_t& o, int cz, int ct) {
  TriMulW t{};
  auto take = [&](size_t k) { size_t r = o; o += k; return r; };
  t.ln_in_g = take(cz); t.ln_in_b = take(cz);
  t.w_ap = take((size_t)cz * ct); t.b_ap = take(ct);
  t.w_ag = take((size_t)cz * ct); t.b_ag = take(ct);
  t.w_bp = take((size_t)cz * ct); t.b_bp = take(ct);
  t.w_bg = take((size_t)cz * ct); t.b_bg = take(ct);
  t.w_g = take((size_t)cz * cz); t.b_g = take(cz);
  t.ln_out_g = take(ct); t.ln_out_b = take(ct);
  t.w_z = take((size_t)ct * cz); t.b_z = take(cz);
  return t;
}
static ExtraOff extra_offsets(const pf_extra_config& c) {
  ExtraOff x{};
  size_t o = 0;
  auto take = [&](size_t k) { size_t r = o; o += k; return r; };
  const int d = c.c_e / c.heads_msa;
  x.row = x_attn_offsets(o, c.c_e, c.heads_msa, 1, c.c_z);
  x.col.ln_g = take(c.c_e); x.col.ln_b = take(c.c_e);
  x.col.wq = take((size_t)c.c_e * c.c_e); x.col.wk = take((size_t)c.c_e * d); x.col.wv = take((size_t)c.c_e * d);
  x.col.wg = take((size_t)c.c_e * c.c_e); x.col.bg = take(c.c_e);
  x.col.wo = take((size_t)c.c_e * c.c_e); x.col.bo = take(c.c_e);
  x.msa_trans = x_trans_offsets(o, c.c_e, c.transition_n);
  x.opm.ln_g = take(c.c_e); x.opm.ln_b = take(c.c_e);
  x.opm.wa = take((size_t)c.c_e * c.c_opm); x.opm.ba = take(c.c_opm);
  x.opm.wb = take((size_t)c.c_e * c.c_opm); x.opm.bb = take(c.c_opm);
  x.opm.wout = take((size_t)c.c_opm * c.c_opm * c.c_z); x.opm.bout = take(c.c_z);
  x.tri_out = x_trimul_offsets(o, c.c_z, c.c_tri);
  x.tri_in = x_trimul_offsets(o, c.c_z, c.c_tri);
  x.tri_start = x_attn_offsets(o, c.c_z, c.heads_pair, 2, c.c_z);
  x.tri_end = x_attn_offsets(o, c.c_z, c.heads_pair, 2, c.c_z);
  x.pair_trans = x_trans_offsets(o, c.c_z, c.transition_n);
  x.total = o;
  return x;
}

static bool extra_cfg_ok(const pf_extra_config& c) {
  return c.c_e == 64 && c.c_z == 128 && c.heads_msa == 8 && c.heads_pair == 4 && c.head_dim_pair == 32 && c.c_opm == 32 &&
         c.c_tri == 128 && c.transition_n == 4 && c.n_blocks_max >= 1;
}

extern "C" size_t pf_extra_msa_block_floats(const pf_extra_config* cfg) {
  if (!cfg || !extra_cfg_ok(*cfg)) return 0;
  return extra_offsets(*cfg).total;
}

static uint16_t x_bf16(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  u += 0x7FFFu + ((u >> 16) & 1);
  return (uint16_t)(u >> 16);
}
static uint16_t x_f16(float f) {
  __half h = __float2half_rn(f);
  uint16_t b;
  memcpy(&b, &h, 2);
  return b;
}

extern "C" void pf_extra_msa_destroy(pf_extra_msa_t* x) {
  if (!x) return;
  pf_evoformer_destroy(x->inner);
  cudaFree(x->w32);
  cudaFree(x->w16);
  cudaFree(x->wf);
  cudaFree(x->o_glob);
  delete x;
}

extern "C" pf_status pf_extra_msa_create(pf_extra_msa_t** out, const float* weights_host, size_t n_floats,
                                         const pf_extra_config* cfg) {
  if (!out || !weights_host || !cfg) return xfail(PF_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  if (!extra_cfg_ok(*cfg))
    return xfail(PF_ERR_SHAPE, "only the AlphaFold extra-MSA dims are built: c_e=64 c_z=128 heads 8/4 head_dim_pair=32 c_opm=32 c_tri=128 n=4");
  const pf_extra_config& c = *cfg;
  const ExtraOff xo = extra_offsets(c);
  if (n_floats != xo.total * (size_t)c.n_blocks_max) return xfail(PF_ERR_SHAPE, "weights blob length != n_blocks_max * pf_extra_msa_block_floats(cfg)");
  // inner handle: main dims (c_m = 32 * heads = 256); per block it holds LN'(z) + pair-bias projection of X.1, the
  // outer-product output projection and the pair stack; its MSA-side entries stay zero and are never used
  pf_config ic{};
  ic.c_m = 32 * c.heads_msa; ic.c_z = c.c_z; ic.heads_msa = c.heads_msa; ic.heads_pair = c.heads_pair; ic.head_dim = 32;
  ic.c_opm = c.c_opm; ic.c_tri = c.c_tri; ic.transition_n = c.transition_n; ic.n_blocks_max = c.n_blocks_max; ic.dtype = PF_BF16;
  const BlockW mo = block_offsets(ic);
  std::vector<float> blob(mo.total * (size_t)c.n_blocks_max, 0.f);
  auto cp = [&](float* dst, const float* src, size_t n) { memcpy(dst, src, n * sizeof(float)); };
  for (int b = 0; b < c.n_blocks_max; ++b) {
    const float* s = weights_host + (size_t)b * xo.total;
    float* d = blob.data() + (size_t)b * mo.total;
    cp(d + mo.row.ln_z_g, s + xo.row.ln_z_g, c.c_z);
    cp(d + mo.row.ln_z_b, s + xo.row.ln_z_b, c.c_z);
    cp(d + mo.row.w_bias, s + xo.row.w_bias, (size_t)c.c_z * c.heads_msa);
    cp(d + mo.opm.wout, s + xo.opm.wout, (size_t)c.c_opm * c.c_opm * c.c_z);
    cp(d + mo.opm.bout, s + xo.opm.bout, c.c_z);
    cp(d + mo.tri_out.ln_in_g, s + xo.tri_out.ln_in_g, xo.tri_in.ln_in_g - xo.tri_out.ln_in_g);
    cp(d + mo.tri_in.ln_in_g, s + xo.tri_in.ln_in_g, xo.tri_start.ln_g - xo.tri_in.ln_in_g);
    cp(d + mo.tri_start.ln_g, s + xo.tri_start.ln_g, xo.tri_end.ln_g - xo.tri_start.ln_g);
    cp(d + mo.tri_end.ln_g, s + xo.tri_end.ln_g, xo.pair_trans.ln_g - xo.tri_end.ln_g);
    cp(d + mo.pair_trans.ln_g, s + xo.pair_trans.ln_g, xo.total - xo.pair_trans.ln_g);
  }
  pf_extra_msa* x = new (std::nothrow) pf_extra_msa();
  if (!x) return xfail(PF_ERR_ALLOC, "host alloc");
  x->cfg = c;
  x->off = xo;
  pf_status st = pf_evoformer_create(&x->inner, blob.data(), blob.size(), &ic);
  if (st != PF_OK) {
    delete x;
    return st;
  }
  // MSA-side matrices, re-laid out: [N_out, K] with K contiguous; head h of the row attention occupies rows / columns
  // [32 h, 32 h + d) of the padded 32 H-wide attention, the rest is zero
  const int ce = c.c_e, H = c.heads_msa, d = ce / H, C = 32 * H, n4 = c.transition_n * ce;
  ExtraT t{};
  {
    size_t o16 = 0, of = 0;
    auto take = [&](size_t k) { size_t r = o16; o16 += (k + 63) / 64 * 64; return r; };
    auto takef = [&](size_t k) { size_t r = of; of += (k + 31) / 32 * 32; return r; };
    t.row_w_in = take((size_t)4 * C * ce);
    t.row_wo = take((size_t)ce * C);
    t.tr_w1 = take((size_t)n4 * ce);
    t.tr_w2 = take((size_t)ce * n4);
    t.opm_wab = take((size_t)2 * c.c_opm * ce);
    t.total16 = o16;
    t.row_b_in = takef((size_t)4 * C);
    t.opm_bias_ab = takef((size_t)2 * c.c_opm);
    t.total_f32 = of;
  }
  x->xt = t;
  std::vector<uint16_t> w16(t.total16 * c.n_blocks_max, 0);
  std::vector<float> wf(t.total_f32 * c.n_blocks_max, 0.f);
  for (int b = 0; b < c.n_blocks_max; ++b) {
    const float* s = weights_host + (size_t)b * xo.total;
    uint16_t* d16 = w16.data() + (size_t)b * t.total16;
    float* df = wf.data() + (size_t)b * t.total_f32;
    const size_t segs[4] = {xo.row.wq, xo.row.wk, xo.row.wg, xo.row.wv};   // projection column order q | k | gate | v
    for (int seg = 0; seg < 4; ++seg)
      for (int h = 0; h < H; ++h)
        for (int cc = 0; cc < d; ++cc)
          for (int k = 0; k < ce; ++k)
            d16[t.row_w_in + ((size_t)seg * C + h * 32 + cc) * ce + k] = x_f16(s[segs[seg] + (size_t)k * ce + h * d + cc]);
    for (int h = 0; h < H; ++h)
      for (int cc = 0; cc < d; ++cc) df[t.row_b_in + 2 * C + h * 32 + cc] = s[xo.row.bg + h * d + cc];
    for (int n = 0; n < ce; ++n)
      for (int h = 0; h < H; ++h)
        for (int cc = 0; cc < d; ++cc) d16[t.row_wo + (size_t)n * C + h * 32 + cc] = x_bf16(s[xo.row.wo + (size_t)(h * d + cc) * ce + n]);
    for (int n = 0; n < n4; ++n)
      for (int k = 0; k < ce; ++k) d16[t.tr_w1 + (size_t)n * ce + k] = x_f16(s[xo.msa_trans.w1 + (size_t)k * n4 + n]);
    for (int n = 0; n < ce; ++n)
      for (int k = 0; k < n4; ++k) d16[t.tr_w2 + (size_t)n * n4 + k] = x_bf16(s[xo.msa_trans.w2 + (size_t)k * ce + n]);
    for (int n = 0; n < c.c_opm; ++n)
      for (int k = 0; k < ce; ++k) {
        d16[t.opm_wab + (size_t)n * ce + k] = x_f16(s[xo.opm.wa + (size_t)k * c.c_opm + n]);
        d16[t.opm_wab + (size_t)(c.c_opm + n) * ce + k] = x_f16(s[xo.opm.wb + (size_t)k * c.c_opm + n]);
      }
    for (int n = 0; n < c.c_opm; ++n) {
      df[t.opm_bias_ab + n] = s[xo.opm.ba + n];
      df[t.opm_bias_ab + c.c_opm + n] = s[xo.opm.bb + n];
    }
  }
  if (cudaMalloc(&x->w32, n_floats * 4) != cudaSuccess || cudaMalloc(&x->w16, w16.size() * 2) != cudaSuccess ||
      cudaMalloc(&x->wf, wf.size() * 4) != cudaSuccess) {
    pf_extra_msa_destroy(x);
    return xfail(PF_ERR_ALLOC, "cudaMalloc extra-MSA weights");
  }
  if (cudaMemcpy(x->w32, weights_host, n_floats * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(x->w16, w16.data(), w16.size() * 2, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(x->wf, wf.data(), wf.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
    pf_extra_msa_destroy(x);
    return xfail(PF_ERR_CUDA, "extra-MSA weights H2D");
  }
  cudaError_t ce_ = cudaFuncSetAttribute(extra_global_col_a_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  if (ce_ != cudaSuccess) {
    pf_extra_msa_destroy(x);
    return xfail(PF_ERR_CUDA, std::string("cudaFuncSetAttribute(global column attention): ") + cudaGetErrorString(ce_));
  }
  *out = x;
  return PF_OK;
}

extern "C" long long pf_extra_msa_last_launch_count(const pf_extra_msa_t* x) { return x ? x->launches : 0; }

static pf_status extra_dispatch(pf_extra_msa* x, float* e, float* pair, const float* sm, const float* mm, int B, int S, int N,
                                int block0, int block1, int step0, int step1, void* stream) {
  if (!x || !e || !pair || !sm || !mm) return xfail(PF_ERR_INVALID_ARG, "null argument");
  if (B < 1 || S < 1 || N < 1) return xfail(PF_ERR_SHAPE, "B, S, N must be >= 1");
  if (N > 1024) return xfail(PF_ERR_SHAPE, "N_res above 1024 not supported (keys per attention row)");
  if (global_a_smem(S, x->cfg.heads_msa) > 200 * 1024)
    return xfail(PF_ERR_SHAPE, "N_seq of the extra MSA above ~2900 not supported (keys / values of one column are kept in shared memory)");
  if ((long)B * x->cfg.c_tri > 65535) return xfail(PF_ERR_SHAPE, "batch above 511 not supported by the extra-MSA stack");
  pf_evoformer* h = x->inner;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device)
    return xfail(PF_ERR_INVALID_ARG, "the current device is not the one the handle was created on");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  std::string err;
  if (!ensure_workspace(h, B, S, N, st, err)) return xfail(PF_ERR_ALLOC, err);
  const size_t need = (size_t)B * N * x->cfg.c_e;
  if (need > x->o_glob_floats) {
    cudaDeviceSynchronize();
    cudaFree(x->o_glob);
    x->o_glob = nullptr;
    x->o_glob_floats = 0;
    if (cudaMalloc(&x->o_glob, need * 4) != cudaSuccess) {
      cudaGetLastError();
      return xfail(PF_ERR_ALLOC, "cudaMalloc extra-MSA scratch");
    }
    x->o_glob_floats = need;
  }
  h->launches = 0;
  if (block1 > block0 && !tc_prepare_flags(h, sm, mm, B, S, N, st)) return xfail(PF_ERR_CUDA, "mask flags launch failed");
  for (int blk = block0; blk < block1; ++blk) {
    ExtraBlockDev xb{x->w32 + (size_t)blk * x->off.total, x->w16 + (size_t)blk * x->xt.total16, x->wf + (size_t)blk * x->xt.total_f32,
                     x->o_glob, x->cfg.c_e, x->cfg.heads_msa, x->cfg.c_e / x->cfg.heads_msa};
    for (int step = step0; step <= step1; ++step) {
      if (!tc_run_extra_substep(h, x->off, x->xt, xb, e, pair, sm, mm, B, S, N, blk, step, st, err)) return xfail(PF_ERR_CUDA, err);
      cudaError_t ce = cudaGetLastError();
      if (ce != cudaSuccess)
        return xfail(PF_ERR_CUDA, std::string("launch failed in extra block ") + std::to_string(blk) + " substep " +
                                      std::to_string(step) + ": " + cudaGetErrorString(ce));
    }
  }
  x->launches = h->launches;
  return PF_OK;
}

extern "C" pf_status pf_extra_msa_forward(pf_extra_msa_t* x, float* extra_msa, float* pair, const float* seq_mask,
                                          const float* extra_msa_mask, int B, int S, int N, int n_blocks, void* stream) {
  if (!x) return xfail(PF_ERR_INVALID_ARG, "null handle");
  if (n_blocks < 0 || n_blocks > x->cfg.n_blocks_max) return xfail(PF_ERR_SHAPE, "n_blocks out of range");
  return extra_dispatch(x, extra_msa, pair, seq_mask, extra_msa_mask, B, S, N, 0, n_blocks, 1, 9, stream);
}

extern "C" pf_status pf_extra_msa_forward_substep(pf_extra_msa_t* x, float* extra_msa, float* pair, const float* seq_mask,
                                                  const float* extra_msa_mask, int B, int S, int N, int block, int substep,
                                                  void* stream) {
  if (!x) return xfail(PF_ERR_INVALID_ARG, "null handle");
  if (block < 0 || block >= x->cfg.n_blocks_max) return xfail(PF_ERR_SHAPE, "block out of range");
  if (substep < 1 || substep > 9) return xfail(PF_ERR_SHAPE, "substep not in 1..9");
  return extra_dispatch(x, extra_msa, pair, seq_mask, extra_msa_mask, B, S, N, block, block + 1, substep, substep, stream);
}

extern "C" pf_status pf_extra_msa_set_profiling(pf_extra_msa_t* x, int enable) {
  if (!x) return xfail(PF_ERR_INVALID_ARG, "null handle");
  return pf_evoformer_set_profiling(x->inner, enable);
}
extern "C" pf_status pf_extra_msa_get_profile(pf_extra_msa_t* x, int kind, long long* launches, double* ms, double* flops,
                                              double* bytes) {
  if (!x) return xfail(PF_ERR_INVALID_ARG, "null handle");
  return pf_evoformer_get_profile(x->inner, kind, launches, ms, flops, bytes);
}
