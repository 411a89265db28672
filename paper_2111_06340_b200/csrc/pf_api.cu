// C-ABI entry points and the block/trunk driver: sequences the nine sub-steps of SURVEY.md §8(a) over the
// kernels of pf_simt.cu (fp32 path) and, through pf_trunk_tc.cu, the tcgen05 kernels (bf16 path).  No arithmetic of the method lives here except the
// constant 1/sqrt(head_dim) handed to the q-projection epilogue (R12).
#include "pf_handle.h"


#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

using namespace pf;

static thread_local std::string g_err;
static pf_status fail(pf_status s, const std::string& msg) {
  g_err = msg;
  return s;
}
extern "C" const char* pf_last_error(void) { return g_err.c_str(); }
namespace pf {
void api_set_error(const std::string& s) { g_err = s; }   // other translation units of the C ABI (pf_embed.cu)
}

#define CUDA_TRY(expr)                                                                              \
  do {                                                                                              \
    cudaError_t _e = (expr);                                                                        \
    if (_e != cudaSuccess)                                                                          \
      return fail(PF_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(_e));                 \
  } while (0)

// ------------------------------------------------------------------------------------------------
// weight blob offsets (floats, within one block) — SURVEY.md Appendix B order
// ------------------------------------------------------------------------------------------------
static AttnW attn_offsets(size_t& o, int c, int heads, int bias_kind /*0 none,1 row,2 self*/, int c_bias) {
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
static TransW trans_offsets(size_t& o, int c, int n) {
  TransW t{};
  auto take = [&](size_t k) { size_t r = o; o += k; return r; };
  t.ln_g = take(c); t.ln_b = take(c);
  t.w1 = take((size_t)c * n * c); t.b1 = take((size_t)n * c);
  t.w2 = take((size_t)n * c * c); t.b2 = take(c);
  return t;
}
static TriMulW trimul_offsets(size_t& o, int cz, int ct) {
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
BlockW pf::block_offsets(const pf_config& c) {
  BlockW w{};
  size_t o = 0;
  w.row = attn_offsets(o, c.c_m, c.heads_msa, 1, c.c_z);
  w.col = attn_offsets(o, c.c_m, c.heads_msa, 0, 0);
  w.msa_trans = trans_offsets(o, c.c_m, c.transition_n);
  {
    auto take = [&](size_t k) { size_t r = o; o += k; return r; };
    w.opm.ln_g = take(c.c_m); w.opm.ln_b = take(c.c_m);
    w.opm.wa = take((size_t)c.c_m * c.c_opm); w.opm.ba = take(c.c_opm);
    w.opm.wb = take((size_t)c.c_m * c.c_opm); w.opm.bb = take(c.c_opm);
    w.opm.wout = take((size_t)c.c_opm * c.c_opm * c.c_z); w.opm.bout = take(c.c_z);
  }
  w.tri_out = trimul_offsets(o, c.c_z, c.c_tri);
  w.tri_in = trimul_offsets(o, c.c_z, c.c_tri);
  w.tri_start = attn_offsets(o, c.c_z, c.heads_pair, 2, c.c_z);
  w.tri_end = attn_offsets(o, c.c_z, c.heads_pair, 2, c.c_z);
  w.pair_trans = trans_offsets(o, c.c_z, c.transition_n);
  w.total = o;
  return w;
}

extern "C" size_t pf_evoformer_block_floats(const pf_config* cfg) {
  if (!cfg) return 0;
  return block_offsets(*cfg).total;
}

static const char* const kKindNames[KK_COUNT] = {"ln_rows", "gemm", "attn_core", "tri_einsum", "ln_channels", "opm_core", "ln_gemm", "transition", "mask_flags", "global_col_attn", "embedders", "pair_bias_heads", "opm_operands"};


Arena pf::arena_layout(const pf_config& c, int B, int S, int N) {
  size_t es = (c.dtype == PF_F32) ? 4 : 2;
  size_t M = (size_t)B * S * N, P = (size_t)B * N * N;
  int Np = pad8(N), Sp = pad8(S);
  size_t n = c.transition_n;
  auto mx = [](size_t a, size_t b) { return a > b ? a : b; };
  Arena a{};
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes, 1024); return r; };
  const bool f32 = c.dtype == PF_F32;   // x, oa, ob: LayerNorm output and row-major outer-product operands of the SIMT path only
  a.x = take(f32 ? mx(M * c.c_m, P * c.c_z) * es : 0);
  a.qkg = take(mx(M * mx(n, 3) * c.c_m, P * mx(n, 3) * c.c_z) * es);
  a.vt = take(mx(mx((size_t)B * S * c.c_m * Np, (size_t)B * N * c.c_m * Sp), (size_t)B * N * c.c_z * Np) * es);
  a.o = take(mx(M * c.c_m, P * c.c_z) * es);
  a.bias = take((size_t)B * mx(c.heads_msa, c.heads_pair) * N * Np * es);
  a.acm = take((size_t)B * c.c_tri * N * Np * es);
  a.bcm = take((size_t)B * c.c_tri * N * Np * es);
  a.g = take(P * c.c_z * es);
  a.tcm = take((size_t)B * c.c_tri * N * Np * 4);
  a.tn = take(P * c.c_tri * es);
  a.oa = take(f32 ? M * c.c_opm * es : 0);
  a.ob = take(f32 ? M * c.c_opm * es : 0);
  a.f_msa = take((size_t)g2_num_tiles(B, S, N));
  a.f_msat = take((size_t)g2_num_tiles(B, N, S));
  a.f_pair = take((size_t)g2_num_tiles(B, N, N));
  a.f_msa_lin = take((M + 127) / 128);
  a.f_pair_lin = take((P + 127) / 128);
  a.f_pair_x = take((size_t)g2_num_tiles(B, N, N));
  a.f_msat_x = take((size_t)g2_num_tiles(B, N, S));
  a.kt_seq = take((size_t)B * 4);
  a.kt_msa = take((size_t)B * 4);
  a.rl_row = take((size_t)B * S * 8);
  a.rl_col = take((size_t)B * N * 8);
  a.rl_tri = take((size_t)B * N * 8);
  a.rl_count = take(3 * 4);
  a.total = o;
  return a;
}

extern "C" size_t pf_evoformer_workspace_bytes(const pf_evoformer_t* h, int B, int S, int N) {
  if (!h || B < 1 || S < 1 || N < 1) return 0;
  return arena_layout(h->cfg, B, S, N).total;
}

extern "C" long long pf_evoformer_last_launch_count(const pf_evoformer_t* h) { return h ? h->launches : 0; }

extern "C" pf_status pf_evoformer_create(pf_evoformer_t** out, const float* weights_host, size_t n_weight_floats,
                                         const pf_config* cfg) {
  if (!out || !weights_host || !cfg) return fail(PF_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  const pf_config& c = *cfg;
  if (c.head_dim != 32) return fail(PF_ERR_SHAPE, "head_dim must be 32");
  if (c.c_m != 256 || c.c_z != 128 || c.heads_msa * c.head_dim != c.c_m || c.heads_pair * c.head_dim != c.c_z ||
      c.c_opm != 32 || c.c_tri != 128 || c.transition_n != 4)
    return fail(PF_ERR_SHAPE, "only the AlphaFold channel dims are built: c_m=256 c_z=128 heads 8/4 c_opm=32 c_tri=128 n=4");
  if (c.n_blocks_max < 1) return fail(PF_ERR_SHAPE, "n_blocks_max < 1");
  if (c.dtype != PF_F32 && c.dtype != PF_BF16) return fail(PF_ERR_INVALID_ARG, "bad dtype");
  BlockW off = block_offsets(c);
  if (n_weight_floats != off.total * (size_t)c.n_blocks_max)
    return fail(PF_ERR_SHAPE, "weights blob length != n_blocks_max * pf_evoformer_block_floats(cfg)");
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) return fail(PF_ERR_ARCH, "device is not compute capability 10.x (sm_100a build)");
  pf_evoformer* h = new (std::nothrow) pf_evoformer();
  if (!h) return fail(PF_ERR_ALLOC, "host alloc");
  h->cfg = c;
  h->off = off;
  h->num_sms = prop.multiProcessorCount;
  h->device = dev;
  size_t nbytes = n_weight_floats * sizeof(float);
  if (cudaMalloc(&h->w32, nbytes) != cudaSuccess) { delete h; return fail(PF_ERR_ALLOC, "cudaMalloc weights"); }
  if (cudaMemcpy(h->w32, weights_host, nbytes, cudaMemcpyHostToDevice) != cudaSuccess) {
    pf_evoformer_destroy(h);
    return fail(PF_ERR_CUDA, "weights H2D");
  }
  if (c.dtype == PF_BF16) {
    h->tc = tc_layout(c);
    std::vector<uint16_t> w16(h->tc.total16 * c.n_blocks_max, 0);
    std::vector<float> wf(h->tc.total_f32 * c.n_blocks_max, 0.f);
    F16Range range;
    for (int b = 0; b < c.n_blocks_max; ++b)
      build_tc_block(c, off, h->tc, weights_host + (size_t)b * off.total, w16, (size_t)b * h->tc.total16, wf,
                     (size_t)b * h->tc.total_f32, &range);
    if (range.overflow) {
      pf_evoformer_destroy(h);
      return fail(PF_ERR_SHAPE, std::to_string(range.overflow) + " weight(s) that multiply a LayerNorm output exceed the fp16 "
                                "range (|w| > 65504 or NaN); see the value-range precondition in pf_evoformer.h");
    }
    h->f16_below_normal = range.below_normal;
    if (cudaMalloc(&h->w16, w16.size() * 2) != cudaSuccess || cudaMalloc(&h->wf, wf.size() * 4) != cudaSuccess) {
      pf_evoformer_destroy(h);
      return fail(PF_ERR_ALLOC, "cudaMalloc bf16 weights");
    }
    if (cudaMemcpy(h->w16, w16.data(), w16.size() * 2, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(h->wf, wf.data(), wf.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
      pf_evoformer_destroy(h);
      return fail(PF_ERR_CUDA, "bf16 weights H2D");
    }
    h->tma = tma_ctx_create();
    if (!h->tma) {
      pf_evoformer_destroy(h);
      return fail(PF_ERR_CUDA, std::string("TMA driver entry point: ") + tc_last_error());
    }
    if (!configure_gemm2_kernels() || !configure_transition_kernels() || !configure_attn_kernel() ||
        !configure_opm_kernel() || !configure_tri_kernel()) {
      pf_evoformer_destroy(h);
      return fail(PF_ERR_CUDA, std::string("kernel attributes: ") + tc_last_error());
    }
  }
  *out = h;
  return PF_OK;
}

extern "C" void pf_evoformer_destroy(pf_evoformer_t* h) {
  if (!h) return;
  cudaFree(h->w32);
  cudaFree(h->w16);
  cudaFree(h->wf);
  cudaFree(h->ws);
  cudaFree(h->stage);
  if (h->h2d_stream) {
    cudaStreamDestroy(h->h2d_stream);
    cudaStreamDestroy(h->d2h_stream);
    for (cudaEvent_t e : h->host_ev) cudaEventDestroy(e);
  }
  if (h->tma) tma_ctx_destroy(h->tma);
  for (auto& g : h->graphs) cudaGraphExecDestroy(g.exec);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
  delete h;
}

extern "C" pf_status pf_evoformer_set_profiling(pf_evoformer_t* h, int enable) {
  if (!h) return fail(PF_ERR_INVALID_ARG, "null handle");
  h->prof_on = enable != 0;
  h->prof.clear();
  h->ev_used = 0;
  return PF_OK;
}

extern "C" int pf_evoformer_profile_kinds(void) { return KK_COUNT; }

extern "C" const char* pf_evoformer_profile_name(int kind) {
  return (kind >= 0 && kind < KK_COUNT) ? kKindNames[kind] : "";
}

extern "C" pf_status pf_evoformer_get_profile(pf_evoformer_t* h, int kind, long long* launches, double* ms,
                                              double* flops, double* bytes) {
  if (!h || !launches || !ms || !flops || !bytes) return fail(PF_ERR_INVALID_ARG, "null argument");
  if (kind < 0 || kind >= KK_COUNT) return fail(PF_ERR_INVALID_ARG, "kind out of range");
  *launches = 0; *ms = 0; *flops = 0; *bytes = 0;
  for (const auto& r : h->prof) {
    if (r.kind != kind) continue;
    cudaError_t e = cudaEventSynchronize(r.e1);
    float t = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&t, r.e0, r.e1);
    if (e != cudaSuccess) return fail(PF_ERR_CUDA, std::string("profile events: ") + cudaGetErrorString(e));
    *launches += 1; *ms += t; *flops += r.flops; *bytes += r.bytes;
  }
  return PF_OK;
}

extern "C" long long pf_evoformer_profile_records(const pf_evoformer_t* h) { return h ? (long long)h->prof.size() : 0; }

extern "C" pf_status pf_evoformer_get_profile_record(pf_evoformer_t* h, long long index, int* kind, double* ms, double* flops,
                                                     double* bytes) {
  if (!h || !kind || !ms || !flops || !bytes) return fail(PF_ERR_INVALID_ARG, "null argument");
  if (index < 0 || index >= (long long)h->prof.size()) return fail(PF_ERR_INVALID_ARG, "record index out of range");
  const auto& r = h->prof[(size_t)index];
  cudaError_t e = cudaEventSynchronize(r.e1);
  float t = 0.f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&t, r.e0, r.e1);
  if (e != cudaSuccess) return fail(PF_ERR_CUDA, std::string("profile events: ") + cudaGetErrorString(e));
  *kind = r.kind; *ms = t; *flops = r.flops; *bytes = r.bytes;
  return PF_OK;
}

// ------------------------------------------------------------------------------------------------
// sub-step drivers
// ------------------------------------------------------------------------------------------------
// fp32 SIMT path (PF_F32): LayerNorm kernel + SIMT GEMMs with fused epilogues + SIMT contractions.
struct Driver {
  typedef float T;
  pf_evoformer* h;
  cudaStream_t st;
  int B, S, N;
  float* msa;
  float* pair;
  const float* seq_mask;
  const float* msa_mask;
  Arena ar;
  const float* w;        // fp32 weights of the current block (device)
  std::string err;

  template <typename U>
  U* buf(size_t off) { return reinterpret_cast<U*>(h->ws + off); }
  void pb(int kind, double flops, double bytes) { h->prof_begin(kind, flops, bytes, st); }
  void pe() { h->prof_end(st); }

  static Epi epi_base(int kind, RowGeom g) {
    Epi e;
    memset(&e, 0, sizeof(e));
    e.kind = kind;
    e.scale = 1.0f;
    e.vt_from = 1 << 30;
    e.geom = g;
    return e;
  }

  // acc = A[R,K] W[K,Nout]; W (and W2) fp32 [K, ldw]
  void gemm(const T* A, int lda, const float* W, const float* W2, int ldw, long R, int K, int Nout, const Epi& e) {
    double nacc = (e.kind == EPI_GATED_CM) ? 2.0 : 1.0;
    double out_b = (e.kind == EPI_RESID) ? 8.0 + (e.gate ? 4.0 : 0.0) : 4.0;
    pb(KK_GEMM, 2.0 * R * K * Nout * nacc, (double)R * K * 4.0 + (double)R * Nout * out_b + nacc * K * Nout * 4.0);
    launch_gemm_simt<T>(A, lda, W, W2, ldw, R, K, Nout, e, st);
    pe();
  }
  void ln_rows(const float* x, T* y, const float* gamma, const float* beta, long rows, int C, RowGeom g, int transposed) {
    pb(KK_LN, 0.0, (double)rows * C * 8.0);
    launch_ln_rows<T>(x, y, gamma, beta, rows, C, g, transposed, st);
    pe();
  }
  void attention(const T* qkg, const T* vt, const T* bias, const float* keymask, T* o, int R, int L, int H) {
    double rows = (double)B * R * L, C = H * 32.0;
    pb(KK_ATTN, 4.0 * rows * L * C, 5.0 * rows * C * 4.0 + (bias ? (double)B * H * L * L * 4.0 : 0.0));
    launch_attn_simt<T>(qkg, vt, bias, keymask, o, B, R, L, pad8(L), H, st);
    pe();
  }

  // Gated attention sub-step on a residual stream `res` viewed as rows (b, x in D1, y in D2), attention along y.
  //   transposed: rows are gathered from / scattered to the (b, y, x) layout of `res`  (A.2, A.8 via their identities)
  void attn_substep(float* res, int C, int H, RowGeom g, bool transposed, const AttnW& a, const float* keymask,
                    const float* bias_src_ln_g, const float* bias_src_ln_b, bool self_bias) {
    long R = (long)g.B * g.D1 * g.D2;
    int L = g.D2, Lp = pad8(L);
    T* X = buf<T>(ar.x);
    T* QKG = buf<T>(ar.qkg);
    T* VT = buf<T>(ar.vt);
    T* O = buf<T>(ar.o);
    T* BIAS = nullptr;
    if (bias_src_ln_g) {   // A.1: bias from LN'(z), own LayerNorm; z rows (b, i, j)
      long P = (long)B * N * N;
      RowGeom gz{B, N, N};
      ln_rows(pair, X, bias_src_ln_g, bias_src_ln_b, P, h->cfg.c_z, gz, 0);
      BIAS = buf<T>(ar.bias);
      Epi e = epi_base(EPI_HEADS, gz);
      e.out = BIAS;
      e.Lpad = pad8(N);
      gemm(X, h->cfg.c_z, w + a.w_bias, nullptr, H, P, h->cfg.c_z, H, e);
    }
    ln_rows(res, X, w + a.ln_g, w + a.ln_b, R, C, g, transposed ? 1 : 0);
    if (self_bias) {       // A.7 / A.8: bias from the same LN(z) rows
      BIAS = buf<T>(ar.bias);
      Epi e = epi_base(EPI_HEADS, g);
      e.out = BIAS;
      e.Lpad = Lp;
      gemm(X, C, w + a.w_bias, nullptr, H, R, C, H, e);
    }
    const float scale = 0.17677669529663687f;   // 1/sqrt(32)  (R12)
    for (int part = 0; part < 4; ++part) {
      Epi e = epi_base(EPI_STORE, g);
      const float* W = w + (part == 0 ? a.wq : part == 1 ? a.wk : part == 2 ? a.wg : a.wv);
      if (part < 3) {
        e.out = QKG + part * C; e.ldo = 3 * C;
        if (part == 0) { e.scale = scale; e.scale_cols = C; }
        if (part == 2) { e.bias = w + a.bg; e.act = ACT_SIGMOID; e.act_lo = 0; e.act_hi = C; }
      } else {
        e.vt_from = 0; e.vt = VT; e.Lpad = Lp;
      }
      gemm(X, C, W, nullptr, C, R, C, C, e);
    }
    attention(QKG, VT, BIAS, keymask, O, g.D1, L, H);
    Epi e = epi_base(EPI_RESID, g);
    e.bias = w + a.bo;
    e.resid = res; e.ldr = C;
    e.transposed = transposed ? 1 : 0;
    gemm(O, C, w + a.wo, nullptr, C, R, C, C, e);
  }

  void transition_substep(float* res, long R, int C, const TransW& t) {
    int n = h->cfg.transition_n;
    RowGeom g{1, 1, (int)R};
    T* X = buf<T>(ar.x);
    T* Hb = buf<T>(ar.qkg);
    ln_rows(res, X, w + t.ln_g, w + t.ln_b, R, C, g, 0);
    Epi e1 = epi_base(EPI_STORE, g);
    e1.out = Hb; e1.ldo = n * C;
    e1.bias = w + t.b1;
    e1.act = ACT_RELU; e1.act_lo = 0; e1.act_hi = n * C;
    gemm(X, C, w + t.w1, nullptr, n * C, R, C, n * C, e1);
    Epi e2 = epi_base(EPI_RESID, g);
    e2.bias = w + t.b2;
    e2.resid = res; e2.ldr = C;
    gemm(Hb, n * C, w + t.w2, nullptr, C, R, n * C, C, e2);
  }

  void opm_substep() {
    const pf_config& c = h->cfg;
    const OpmW& o = h->off.opm;
    long M = (long)B * S * N;
    double P = (double)B * N * N, cc = (double)c.c_opm * c.c_opm;
    T* X = buf<T>(ar.x);
    RowGeom g{B, S, N};
    T* OA = buf<T>(ar.oa);
    T* OB = buf<T>(ar.ob);
    ln_rows(msa, X, w + o.ln_g, w + o.ln_b, M, c.c_m, g, 0);
    for (int part = 0; part < 2; ++part) {
      Epi e = epi_base(EPI_STORE, g);
      e.out = part ? OB : OA; e.ldo = c.c_opm;
      e.bias = w + (part ? o.bb : o.ba);
      e.rowmask = RM_MSA; e.seq_mask = seq_mask; e.msa_mask = msa_mask;
      gemm(X, c.c_m, w + (part ? o.wb : o.wa), nullptr, c.c_opm, M, c.c_m, c.c_opm, e);
    }
    pb(KK_OPM, 2.0 * P * cc * S + 2.0 * P * cc * c.c_z, 2.0 * M * c.c_opm * 4.0 + 8.0 * P * c.c_z);
    launch_opm_simt<T>(OA, OB, w + o.wout, w + o.bout, seq_mask, msa_mask, pair, B, S, N, c.c_opm, c.c_z, st);
    pe();
  }

  void trimul_substep(bool incoming) {
    const pf_config& c = h->cfg;
    const TriMulW& t = incoming ? h->off.tri_in : h->off.tri_out;
    long P = (long)B * N * N;
    int Np = pad8(N);
    RowGeom g{B, N, N};
    T* X = buf<T>(ar.x);
    T* ACM = buf<T>(ar.acm);
    T* BCM = buf<T>(ar.bcm);
    T* G = buf<T>(ar.g);
    float* TCM = buf<float>(ar.tcm);
    T* TN = buf<T>(ar.tn);
    ln_rows(pair, X, w + t.ln_in_g, w + t.ln_in_b, P, c.c_z, g, incoming ? 1 : 0);
    for (int part = 0; part < 2; ++part) {
      // incoming (A.6) = outgoing on the transposed rows with the a/b projections swapped (SURVEY.md §0 finding 1)
      bool use_b = (part == 1) != incoming;
      Epi e = epi_base(EPI_GATED_CM, g);
      e.out = part ? BCM : ACM;
      e.Lpad = Np;
      e.bias = w + (use_b ? t.b_bp : t.b_ap);
      e.bias2 = w + (use_b ? t.b_bg : t.b_ag);
      e.rowmask = RM_PAIR; e.seq_mask = seq_mask;
      gemm(X, c.c_z, w + (use_b ? t.w_bp : t.w_ap), w + (use_b ? t.w_bg : t.w_ag), c.c_tri, P, c.c_z, c.c_tri, e);
    }
    {
      Epi e = epi_base(EPI_STORE, g);
      e.out = G; e.ldo = c.c_z;
      e.bias = w + t.b_g;
      e.act = ACT_SIGMOID; e.act_lo = 0; e.act_hi = c.c_z;
      gemm(X, c.c_z, w + t.w_g, nullptr, c.c_z, P, c.c_z, c.c_z, e);
    }
    pb(KK_TRI, 2.0 * B * c.c_tri * (double)N * N * N, (double)B * c.c_tri * N * Np * 12.0);
    launch_tri_einsum_simt<T>(ACM, BCM, TCM, B * c.c_tri, N, Np, st);
    pe();
    pb(KK_LNC, 0.0, (double)P * c.c_tri * 8.0);
    launch_lnc<T>(TCM, TN, w + t.ln_out_g, w + t.ln_out_b, nullptr, B, c.c_tri, N, Np, st);
    pe();
    Epi e = epi_base(EPI_RESID, g);
    e.bias = w + t.b_z;
    e.resid = pair; e.ldr = c.c_z;
    e.gate = G; e.ldg = c.c_z;
    e.transposed = incoming ? 1 : 0;
    gemm(TN, c.c_tri, w + t.w_z, nullptr, c.c_z, P, c.c_tri, c.c_z, e);
  }

  bool run_substep(int block, int step) {
    const pf_config& c = h->cfg;
    w = h->w32 + (size_t)block * h->off.total;
    switch (step) {
      case 1: attn_substep(msa, c.c_m, c.heads_msa, RowGeom{B, S, N}, false, h->off.row, seq_mask,
                           w + h->off.row.ln_z_g, w + h->off.row.ln_z_b, false); return true;
      case 2: attn_substep(msa, c.c_m, c.heads_msa, RowGeom{B, N, S}, true, h->off.col, msa_mask, nullptr, nullptr, false);
              return true;
      case 3: transition_substep(msa, (long)B * S * N, c.c_m, h->off.msa_trans); return true;
      case 4: opm_substep(); return true;
      case 5: trimul_substep(false); return true;
      case 6: trimul_substep(true); return true;
      case 7: attn_substep(pair, c.c_z, c.heads_pair, RowGeom{B, N, N}, false, h->off.tri_start, seq_mask, nullptr,
                           nullptr, true); return true;
      case 8: attn_substep(pair, c.c_z, c.heads_pair, RowGeom{B, N, N}, true, h->off.tri_end, seq_mask, nullptr, nullptr,
                           true); return true;
      case 9: transition_substep(pair, (long)B * N * N, c.c_z, h->off.pair_trans); return true;
    }
    err = "substep not in 1..9";
    return false;
  }
};


static pf_status check_and_grow(pf_evoformer* h, int B, int S, int N, cudaStream_t st) {
  size_t need = arena_layout(h->cfg, B, S, N).total;
  if (need > h->ws_bytes) {
    cudaDeviceSynchronize();
    cudaFree(h->ws);
    h->ws = nullptr;
    h->ws_bytes = 0;
    h->ws_B = h->ws_S = h->ws_N = 0;
    if (cudaMalloc(&h->ws, need) != cudaSuccess) {
      cudaGetLastError();
      return fail(PF_ERR_ALLOC, "cudaMalloc workspace");
    }
    h->ws_bytes = need;
  }
  // Masked tiles are skipped (pf_flags.cu): what they would have written must still be finite when a partially masked tile
  // later reads it.  Within one arena layout every region keeps its element type from call to call, so stale contents are
  // finite outputs of earlier launches; the layout (offsets and types) is a function of (B, S, N), so the arena is zero-filled,
  // in stream order, whenever that shape differs from the previous call's (a slightly smaller tail batch on the same handle
  // would otherwise reinterpret fp32 bytes as 16-bit values).
  if (B != h->ws_B || S != h->ws_S || N != h->ws_N) {
    if (cudaMemsetAsync(h->ws, 0, need, st) != cudaSuccess) return fail(PF_ERR_CUDA, "cudaMemsetAsync workspace");
    h->ws_B = B; h->ws_S = S; h->ws_N = N;
  }
  return PF_OK;
}

bool pf::ensure_workspace(pf_evoformer* h, int B, int S, int N, cudaStream_t st, std::string& err) {
  if (check_and_grow(h, B, S, N, st) == PF_OK) return true;
  err = g_err;
  return false;
}

// Largest batch one launch sequence takes: gridDim.z of the per-(protein, channel) and per-(protein, row) kernels is capped
// at 65535.  Larger batches are cut into chunks of proteins (proteins are independent).
static int max_batch_per_pass(const pf_config& c, int S, int N) {
  const int lim = 65535;
  int cap = lim / c.c_tri;                                       // triangle einsum: grid.z = B * c_tri
  if (c.dtype == PF_F32) cap = std::min(cap, lim / std::max(S, N));   // SIMT attention: grid.z = B * rows
  return std::max(cap, 1);
}

static pf_status dispatch_pass(pf_evoformer* h, float* msa, float* pair, const float* sm, const float* mm, int B, int S,
                               int N, int block0, int block1, int step0, int step1, cudaStream_t st, long long& launches);

static pf_status dispatch(pf_evoformer* h, float* msa, float* pair, const float* sm, const float* mm, int B, int S,
                          int N, int block0, int block1, int step0, int step1, void* stream) {
  if (!h || !msa || !pair || !sm || !mm) return fail(PF_ERR_INVALID_ARG, "null argument");
  if (B < 1 || S < 1 || N < 1) return fail(PF_ERR_SHAPE, "B, S, N must be >= 1");
  if (S > 65535 || N > 65535) return fail(PF_ERR_SHAPE, "N_seq and N_res must be <= 65535");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device)
    return fail(PF_ERR_INVALID_ARG, "the current device is not the one the handle was created on");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int cap = max_batch_per_pass(h->cfg, S, N);
  const int passes = (B + cap - 1) / cap;
  long long launches = 0;
  int b0 = 0;
  for (int p = 0; p < passes; ++p) {
    const int bc = (B - b0 + (passes - p) - 1) / (passes - p);
    pf_status s = dispatch_pass(h, msa + (size_t)b0 * S * N * h->cfg.c_m, pair + (size_t)b0 * N * N * h->cfg.c_z,
                                sm + (size_t)b0 * N, mm + (size_t)b0 * S, bc, S, N, block0, block1, step0, step1, st, launches);
    if (s != PF_OK) return s;
    b0 += bc;
  }
  h->launches = launches;
  return PF_OK;
}

// the launch sequence of one pass (workspace already sized): mask flags, then the sub-steps
static pf_status pass_launches(pf_evoformer* h, float* msa, float* pair, const float* sm, const float* mm, int B, int S, int N,
                               int block0, int block1, int step0, int step1, cudaStream_t st) {
  Driver d;
  d.h = h; d.st = st; d.B = B; d.S = S; d.N = N;
  d.msa = msa; d.pair = pair; d.seq_mask = sm; d.msa_mask = mm;
  d.ar = arena_layout(h->cfg, B, S, N);
  h->launches = 0;
  if (h->cfg.dtype == PF_BF16 && block1 > block0 && !tc_prepare_flags(h, sm, mm, B, S, N, st))
    return fail(PF_ERR_CUDA, "mask flags launch failed");
  for (int blk = block0; blk < block1; ++blk)
    for (int step = step0; step <= step1; ++step) {
      bool ok = (h->cfg.dtype == PF_F32) ? d.run_substep(blk, step)
                                         : tc_run_substep(h, msa, pair, sm, mm, B, S, N, blk, step, st, d.err);
      if (!ok) return fail(PF_ERR_CUDA, d.err);
      cudaError_t e = cudaGetLastError();
      if (e != cudaSuccess)
        return fail(PF_ERR_CUDA, std::string("launch failed in block ") + std::to_string(blk) + " substep " +
                                     std::to_string(step) + ": " + cudaGetErrorString(e));
    }
  return PF_OK;
}

// Small problems are launch-bound: 25 launches per block with several tensor-map encodings each cost the host ~10-15 us per
// launch while the kernels of a single 64-residue protein take less.  Whole forward calls on such shapes are therefore
// captured once into a CUDA graph per (buffers, shape, block range) and replayed; tensor maps are by-value kernel parameters,
// so the graph holds them.  Not used while profiling (events per launch), for the fp32 path, or for single sub-steps.
static bool graph_wanted(const pf_evoformer* h, int B, int S, int N, int block0, int block1, int step0, int step1) {
  static const int env = getenv("PF_GRAPH") ? atoi(getenv("PF_GRAPH")) : 1;
  if (!env || h->prof_on || h->cfg.dtype != PF_BF16 || step0 != 1 || step1 != 9 || block1 - block0 < 2) return false;
  return env == 2 || (double)B * S * N <= 131072.0;
}

static pf_status dispatch_pass(pf_evoformer* h, float* msa, float* pair, const float* sm, const float* mm, int B, int S,
                               int N, int block0, int block1, int step0, int step1, cudaStream_t st, long long& launches) {
  char* const ws_before = h->ws;
  pf_status s = check_and_grow(h, B, S, N, st);
  if (s != PF_OK) return s;
  if (h->ws != ws_before) {   // the arena moved: every captured graph points into the old one
    for (auto& g : h->graphs) cudaGraphExecDestroy(g.exec);
    h->graphs.clear();
  }
  if (graph_wanted(h, B, S, N, block0, block1, step0, step1)) {
    for (auto& g : h->graphs)
      if (g.msa == msa && g.pair == pair && g.sm == sm && g.mm == mm && g.B == B && g.S == S && g.N == N && g.block0 == block0 &&
          g.block1 == block1) {
        if (cudaGraphLaunch(g.exec, st) != cudaSuccess) return fail(PF_ERR_CUDA, "cudaGraphLaunch");
        h->launches = g.launches;
        launches += g.launches;
        return PF_OK;
      }
    // captured on a stream of the handle's own (the caller's may be the legacy default stream, which cannot be captured;
    // nothing executes during capture) and replayed on the caller's stream
    if (!h->cap_stream && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
      h->cap_stream = nullptr;
      cudaGetLastError();
    }
    cudaStream_t cs = h->cap_stream;
    if (cs && cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      s = pass_launches(h, msa, pair, sm, mm, B, S, N, block0, block1, step0, step1, cs);
      cudaGraph_t graph = nullptr;
      cudaError_t ce = cudaStreamEndCapture(cs, &graph);
      cudaGraphExec_t exec = nullptr;
      if (s == PF_OK && ce == cudaSuccess && graph && cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess) {
        cudaGraphDestroy(graph);
        if (h->graphs.size() >= 16) {   // bounded cache: drop the oldest
          cudaGraphExecDestroy(h->graphs.front().exec);
          h->graphs.erase(h->graphs.begin());
        }
        h->graphs.push_back({msa, pair, sm, mm, B, S, N, block0, block1, exec, h->launches});
        if (cudaGraphLaunch(exec, st) != cudaSuccess) return fail(PF_ERR_CUDA, "cudaGraphLaunch");
        launches += h->launches;
        return PF_OK;
      }
      if (graph) cudaGraphDestroy(graph);
      cudaGetLastError();   // capture did not work out: fall through to plain launches
    } else {
      cudaGetLastError();
    }
  }
  s = pass_launches(h, msa, pair, sm, mm, B, S, N, block0, block1, step0, step1, st);
  if (s != PF_OK) return s;
  launches += h->launches;
  return PF_OK;
}

extern "C" pf_status pf_evoformer_forward(pf_evoformer_t* h, float* msa, float* pair, const float* seq_mask,
                                          const float* msa_mask, int B, int S, int N, int n_blocks, void* stream) {
  if (!h) return fail(PF_ERR_INVALID_ARG, "null handle");
  if (n_blocks < 0 || n_blocks > h->cfg.n_blocks_max) return fail(PF_ERR_SHAPE, "n_blocks out of range");
  return dispatch(h, msa, pair, seq_mask, msa_mask, B, S, N, 0, n_blocks, 1, 9, stream);
}

extern "C" pf_status pf_evoformer_forward_substep(pf_evoformer_t* h, float* msa, float* pair, const float* seq_mask,
                                                  const float* msa_mask, int B, int S, int N, int block, int substep,
                                                  void* stream) {
  if (!h) return fail(PF_ERR_INVALID_ARG, "null handle");
  if (block < 0 || block >= h->cfg.n_blocks_max) return fail(PF_ERR_SHAPE, "block out of range");
  if (substep < 1 || substep > 9) return fail(PF_ERR_SHAPE, "substep not in 1..9");
  return dispatch(h, msa, pair, seq_mask, msa_mask, B, S, N, block, block + 1, substep, substep, stream);
}

extern "C" pf_status pf_evoformer_forward_host(pf_evoformer_t* h, float* msa_host, float* pair_host,
                                               const float* seq_mask_host, const float* msa_mask_host, int B, int S,
                                               int N, int n_blocks, void* stream) {
  if (!h || !msa_host || !pair_host || !seq_mask_host || !msa_mask_host) return fail(PF_ERR_INVALID_ARG, "null argument");
  if (B < 1 || S < 1 || N < 1) return fail(PF_ERR_SHAPE, "B, S, N must be >= 1");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  size_t nm = (size_t)B * S * N * h->cfg.c_m * 4, nz = (size_t)B * N * N * h->cfg.c_z * 4;
  size_t ns = align_up((size_t)B * N * 4, 256), nr = align_up((size_t)B * S * 4, 256);
  size_t need = align_up(nm, 256) + align_up(nz, 256) + ns + nr;
  if (need > h->stage_bytes) {
    cudaDeviceSynchronize();
    cudaFree(h->stage);
    h->stage = nullptr;
    h->stage_bytes = 0;
    if (cudaMalloc(&h->stage, need) != cudaSuccess) {
      cudaGetLastError();
      return fail(PF_ERR_ALLOC, "cudaMalloc staging");
    }
    h->stage_bytes = need;
  }
  float* dm = reinterpret_cast<float*>(h->stage);
  float* dz = reinterpret_cast<float*>(h->stage + align_up(nm, 256));
  float* ds = reinterpret_cast<float*>(h->stage + align_up(nm, 256) + align_up(nz, 256));
  float* dr = reinterpret_cast<float*>(h->stage + align_up(nm, 256) + align_up(nz, 256) + ns);
  // Proteins are independent, so the batch is pipelined in chunks: while chunk c is computed on the caller's stream, chunk
  // c+1 is copied in and chunk c-1 is copied out on two copy streams (PCIe is full duplex).  Pageable host memory still
  // works (the copies then serialise inside the driver).
  if (!h->h2d_stream) {
    CUDA_TRY(cudaStreamCreateWithFlags(&h->h2d_stream, cudaStreamNonBlocking));
    CUDA_TRY(cudaStreamCreateWithFlags(&h->d2h_stream, cudaStreamNonBlocking));
    for (auto& e : h->host_ev) CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  }
  // Chunk sizes.  The copies are the longer leg (cfg2: 1.6 GB each way, 38-40 ms full duplex, against 36 ms of compute), so
  // compute follows the copy-in by one chunk and the call ends one chunk's compute + copy-out after the last byte has
  // landed: seven equal chunks of B/8 (equal, so that none of them stalls the ones behind it: at cfg2 a chunk of 8 proteins
  // is 6.9 waves of 128-row tiles, chunks of 13-14 were 1.3x slower per protein than their copy) between two half chunks at
  // the ends (the first copy-in and the last compute + copy-out are not overlapped with anything).  Measured at cfg2
  // (proteins/s): this plan 1391; 8 equal 1373; 16 equal 1234; 7 equal 1216; the former 4,8,14,13,13,8,4 plan 1295.
  // PF_HOST_CHUNKS=a,b,c,... (at most 16 sizes that add up to B) overrides the plan (tuning other shapes).
  int sizes[16];
  int n_chunks = 0;
  if (const char* plan = getenv("PF_HOST_CHUNKS")) {
    int sum = 0;
    for (const char* q = plan; *q && n_chunks < 16;) {
      sizes[n_chunks] = atoi(q);
      if (sizes[n_chunks] < 1) { sum = -1; break; }
      sum += sizes[n_chunks++];
      while (*q && *q != ',') ++q;
      if (*q == ',') ++q;
    }
    if (sum != B) n_chunks = 0;
  }
  if (n_chunks > 0) {
  } else if (B < 16) {
    n_chunks = B < 8 ? B : 8;
    for (int c = 0, b0 = 0; c < n_chunks; ++c) {
      sizes[c] = (B - b0 + (n_chunks - c) - 1) / (n_chunks - c);
      b0 += sizes[c];
    }
  } else {
    const int e1 = B / 16, mid = B - 2 * e1;
    const int n_mid = 7;
    sizes[n_chunks++] = e1;
    for (int c = 0, left = mid; c < n_mid; ++c) {
      sizes[n_chunks] = (left + (n_mid - c) - 1) / (n_mid - c);
      left -= sizes[n_chunks++];
    }
    sizes[n_chunks++] = e1;
  }
  const size_t pm = (size_t)S * N * h->cfg.c_m, pz = (size_t)N * N * h->cfg.c_z;   // floats per protein
  CUDA_TRY(cudaEventRecord(h->host_ev[32], st));                  // earlier work on the caller's stream comes first
  CUDA_TRY(cudaStreamWaitEvent(h->h2d_stream, h->host_ev[32], 0));
  CUDA_TRY(cudaStreamWaitEvent(h->d2h_stream, h->host_ev[32], 0));
  CUDA_TRY(cudaMemcpyAsync(ds, seq_mask_host, (size_t)B * N * 4, cudaMemcpyHostToDevice, h->h2d_stream));
  CUDA_TRY(cudaMemcpyAsync(dr, msa_mask_host, (size_t)B * S * 4, cudaMemcpyHostToDevice, h->h2d_stream));
  int b0 = 0;
  for (int c = 0; c < n_chunks; ++c) {
    const int bc = sizes[c];
    CUDA_TRY(cudaMemcpyAsync(dm + b0 * pm, msa_host + b0 * pm, bc * pm * 4, cudaMemcpyHostToDevice, h->h2d_stream));
    CUDA_TRY(cudaMemcpyAsync(dz + b0 * pz, pair_host + b0 * pz, bc * pz * 4, cudaMemcpyHostToDevice, h->h2d_stream));
    CUDA_TRY(cudaEventRecord(h->host_ev[c], h->h2d_stream));
    b0 += bc;
  }
  b0 = 0;
  for (int c = 0; c < n_chunks; ++c) {
    const int bc = sizes[c];
    CUDA_TRY(cudaStreamWaitEvent(st, h->host_ev[c], 0));
    pf_status s = pf_evoformer_forward(h, dm + b0 * pm, dz + b0 * pz, ds + (size_t)b0 * N, dr + (size_t)b0 * S, bc, S, N, n_blocks,
                                       stream);
    if (s != PF_OK) return s;
    CUDA_TRY(cudaEventRecord(h->host_ev[16 + c], st));
    CUDA_TRY(cudaStreamWaitEvent(h->d2h_stream, h->host_ev[16 + c], 0));
    CUDA_TRY(cudaMemcpyAsync(msa_host + b0 * pm, dm + b0 * pm, bc * pm * 4, cudaMemcpyDeviceToHost, h->d2h_stream));
    CUDA_TRY(cudaMemcpyAsync(pair_host + b0 * pz, dz + b0 * pz, bc * pz * 4, cudaMemcpyDeviceToHost, h->d2h_stream));
    b0 += bc;
  }
  CUDA_TRY(cudaStreamSynchronize(h->d2h_stream));
  CUDA_TRY(cudaStreamSynchronize(st));
  return PF_OK;
}
