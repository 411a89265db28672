// C-ABI entry points and the block/trunk driver: sequences the nine sub-steps of SURVEY.md §8(a) over the
// kernels of pf_simt.cu / pf_gemm_tc.cu / pf_attn_tc.cu.  No arithmetic of the method lives here except the
// constant 1/sqrt(head_dim) handed to the q-projection epilogue (R12).
#include "../../include/pf_evoformer.h"
#include "pf_internal.h"

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

#define CUDA_TRY(expr)                                                                              \
  do {                                                                                              \
    cudaError_t _e = (expr);                                                                        \
    if (_e != cudaSuccess)                                                                          \
      return fail(PF_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(_e));                 \
  } while (0)

// ------------------------------------------------------------------------------------------------
// weight blob offsets (floats, within one block) — SURVEY.md Appendix B order
// ------------------------------------------------------------------------------------------------
struct AttnW {
  size_t ln_g, ln_b, ln_z_g, ln_z_b, w_bias, wq, wk, wv, wg, bg, wo, bo;
};
struct TransW {
  size_t ln_g, ln_b, w1, b1, w2, b2;
};
struct OpmW {
  size_t ln_g, ln_b, wa, ba, wb, bb, wout, bout;
};
struct TriMulW {
  size_t ln_in_g, ln_in_b, w_ap, b_ap, w_ag, b_ag, w_bp, b_bp, w_bg, b_bg, w_g, b_g, ln_out_g, ln_out_b, w_z, b_z;
};
struct BlockW {
  AttnW row, col, tri_start, tri_end;
  TransW msa_trans, pair_trans;
  OpmW opm;
  TriMulW tri_out, tri_in;
  size_t total;
};

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
static BlockW block_offsets(const pf_config& c) {
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

// ------------------------------------------------------------------------------------------------
// tensor-core weight set (bf16, [Nout, K] with K contiguous), offsets in bf16 elements within one block
// ------------------------------------------------------------------------------------------------
struct AttnT { size_t wqkgv, wo, bias_qkgv /*float offset in fused-bias array*/; };
struct TcBlock {
  AttnT row, col, tri_start, tri_end;
  size_t mt_w1, mt_w2, pt_w1, pt_w2;
  size_t opm_wab, opm_bias_ab /*float*/, opm_wout;
  size_t to_wa, to_wb, to_wg, to_wz, ti_wa, ti_wb, ti_wg, ti_wz;
  size_t total_bf16, total_f32;
};

// ------------------------------------------------------------------------------------------------
// handle
// ------------------------------------------------------------------------------------------------
struct pf_evoformer {
  pf_config cfg;
  BlockW off;
  TcBlock tc;
  float* w32 = nullptr;      // device fp32 blob
  bf16* w16 = nullptr;       // device bf16 transposed matrices (PF_BF16 only)
  float* wf = nullptr;       // device fused fp32 bias vectors (PF_BF16 only)
  char* ws = nullptr;        // workspace arena
  size_t ws_bytes = 0;
  char* stage = nullptr;     // forward_host staging
  size_t stage_bytes = 0;
  int num_sms = 148;
  unsigned tc_mask = 0;      // bit0 gemm, bit1 attention, bit2 triangle einsum, bit3 opm
  long long launches = 0;
  TmaCtx* tma = nullptr;
  // per-launch CUDA-event profiling (pf_evoformer_set_profiling)
  bool prof_on = false;
  struct ProfRec { int kind; cudaEvent_t e0, e1; double flops, bytes; };
  std::vector<ProfRec> prof;
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_used = 0;
  cudaEvent_t next_event() {
    if (ev_used == ev_pool.size()) {
      cudaEvent_t e;
      cudaEventCreate(&e);
      ev_pool.push_back(e);
    }
    return ev_pool[ev_used++];
  }
};

enum KernelKind { KK_LN = 0, KK_GEMM, KK_ATTN, KK_TRI, KK_LNC, KK_OPM, KK_COUNT };
static const char* const kKindNames[KK_COUNT] = {"ln_rows", "gemm", "attn_core", "tri_einsum", "ln_channels", "opm_core"};

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
static int pad8(int v) { return (v + 7) / 8 * 8; }

struct Arena {
  size_t x, qkg, vt, o, bias, acm, bcm, g, tcm, tn, oa, ob, total;
};
static Arena arena_layout(const pf_config& c, int B, int S, int N) {
  size_t es = (c.dtype == PF_F32) ? 4 : 2;
  size_t M = (size_t)B * S * N, P = (size_t)B * N * N;
  int Np = pad8(N), Sp = pad8(S);
  size_t n = c.transition_n;
  auto mx = [](size_t a, size_t b) { return a > b ? a : b; };
  Arena a{};
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes, 1024); return r; };
  a.x = take(mx(M * c.c_m, P * c.c_z) * es);
  a.qkg = take(mx(M * mx(n, 3) * c.c_m, P * mx(n, 3) * c.c_z) * es);
  a.vt = take(mx(mx((size_t)B * S * c.c_m * Np, (size_t)B * N * c.c_m * Sp), (size_t)B * N * c.c_z * Np) * es);
  a.o = take(mx(M * c.c_m, P * c.c_z) * es);
  a.bias = take((size_t)B * mx(c.heads_msa, c.heads_pair) * N * Np * es);
  a.acm = take((size_t)B * c.c_tri * N * Np * es);
  a.bcm = take((size_t)B * c.c_tri * N * Np * es);
  a.g = take(P * c.c_z * es);
  a.tcm = take((size_t)B * c.c_tri * N * Np * 4);
  a.tn = take(P * c.c_tri * es);
  a.oa = take(M * c.c_opm * es);
  a.ob = take(M * c.c_opm * es);
  a.total = o;
  return a;
}

extern "C" size_t pf_evoformer_workspace_bytes(const pf_evoformer_t* h, int B, int S, int N) {
  if (!h || B < 1 || S < 1 || N < 1) return 0;
  return arena_layout(h->cfg, B, S, N).total;
}

extern "C" long long pf_evoformer_last_launch_count(const pf_evoformer_t* h) { return h ? h->launches : 0; }

static uint16_t f32_to_bf16_bits(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  uint32_t lsb = (u >> 16) & 1;
  u += 0x7FFFu + lsb;
  return (uint16_t)(u >> 16);
}

// dst[n, k] = src[k, n]  (src row-major [K, Nout]) as bf16
static void put_transposed(std::vector<uint16_t>& dst, size_t at, const float* src, int K, int Nout) {
  for (int n = 0; n < Nout; ++n)
    for (int k = 0; k < K; ++k) dst[at + (size_t)n * K + k] = f32_to_bf16_bits(src[(size_t)k * Nout + n]);
}

static TcBlock tc_layout(const pf_config& c) {
  TcBlock t{};
  size_t o = 0, f = 0;
  auto take = [&](size_t k) { size_t r = o; o += align_up(k, 64); return r; };
  auto takef = [&](size_t k) { size_t r = f; f += align_up(k, 32); return r; };
  auto attn = [&](int ch) {
    AttnT a{};
    a.wqkgv = take((size_t)4 * ch * ch);
    a.wo = take((size_t)ch * ch);
    a.bias_qkgv = takef((size_t)4 * ch);
    return a;
  };
  t.row = attn(c.c_m);
  t.col = attn(c.c_m);
  t.tri_start = attn(c.c_z);
  t.tri_end = attn(c.c_z);
  size_t n = c.transition_n;
  t.mt_w1 = take(n * c.c_m * c.c_m); t.mt_w2 = take(n * c.c_m * c.c_m);
  t.pt_w1 = take(n * c.c_z * c.c_z); t.pt_w2 = take(n * c.c_z * c.c_z);
  t.opm_wab = take((size_t)2 * c.c_opm * c.c_m);
  t.opm_bias_ab = takef((size_t)2 * c.c_opm);
  t.opm_wout = take((size_t)c.c_opm * c.c_opm * c.c_z);
  t.to_wa = take((size_t)2 * c.c_tri * c.c_z); t.to_wb = take((size_t)2 * c.c_tri * c.c_z);
  t.to_wg = take((size_t)c.c_z * c.c_z); t.to_wz = take((size_t)c.c_z * c.c_tri);
  t.ti_wa = take((size_t)2 * c.c_tri * c.c_z); t.ti_wb = take((size_t)2 * c.c_tri * c.c_z);
  t.ti_wg = take((size_t)c.c_z * c.c_z); t.ti_wz = take((size_t)c.c_z * c.c_tri);
  t.total_bf16 = o;
  t.total_f32 = f;
  return t;
}

static void build_tc_block(const pf_config& c, const BlockW& off, const TcBlock& t, const float* w,
                           std::vector<uint16_t>& w16, size_t base16, std::vector<float>& wf, size_t basef) {
  auto attn = [&](const AttnW& a, const AttnT& d, int ch) {
    // column order of the fused projection: [q | k | gate | v]
    put_transposed(w16, base16 + d.wqkgv + (size_t)0 * ch * ch, w + a.wq, ch, ch);
    put_transposed(w16, base16 + d.wqkgv + (size_t)1 * ch * ch, w + a.wk, ch, ch);
    put_transposed(w16, base16 + d.wqkgv + (size_t)2 * ch * ch, w + a.wg, ch, ch);
    put_transposed(w16, base16 + d.wqkgv + (size_t)3 * ch * ch, w + a.wv, ch, ch);
    put_transposed(w16, base16 + d.wo, w + a.wo, ch, ch);
    for (int i = 0; i < 4 * ch; ++i) wf[basef + d.bias_qkgv + i] = 0.f;
    for (int i = 0; i < ch; ++i) wf[basef + d.bias_qkgv + 2 * ch + i] = w[a.bg + i];
  };
  attn(off.row, t.row, c.c_m);
  attn(off.col, t.col, c.c_m);
  attn(off.tri_start, t.tri_start, c.c_z);
  attn(off.tri_end, t.tri_end, c.c_z);
  int n = c.transition_n;
  put_transposed(w16, base16 + t.mt_w1, w + off.msa_trans.w1, c.c_m, n * c.c_m);
  put_transposed(w16, base16 + t.mt_w2, w + off.msa_trans.w2, n * c.c_m, c.c_m);
  put_transposed(w16, base16 + t.pt_w1, w + off.pair_trans.w1, c.c_z, n * c.c_z);
  put_transposed(w16, base16 + t.pt_w2, w + off.pair_trans.w2, n * c.c_z, c.c_z);
  put_transposed(w16, base16 + t.opm_wab, w + off.opm.wa, c.c_m, c.c_opm);
  put_transposed(w16, base16 + t.opm_wab + (size_t)c.c_opm * c.c_m, w + off.opm.wb, c.c_m, c.c_opm);
  for (int i = 0; i < c.c_opm; ++i) {
    wf[basef + t.opm_bias_ab + i] = w[off.opm.ba + i];
    wf[basef + t.opm_bias_ab + c.c_opm + i] = w[off.opm.bb + i];
  }
  put_transposed(w16, base16 + t.opm_wout, w + off.opm.wout, c.c_opm * c.c_opm, c.c_z);
  auto tri = [&](const TriMulW& s, size_t wa, size_t wb, size_t wg, size_t wz) {
    put_transposed(w16, base16 + wa, w + s.w_ap, c.c_z, c.c_tri);
    put_transposed(w16, base16 + wa + (size_t)c.c_tri * c.c_z, w + s.w_ag, c.c_z, c.c_tri);
    put_transposed(w16, base16 + wb, w + s.w_bp, c.c_z, c.c_tri);
    put_transposed(w16, base16 + wb + (size_t)c.c_tri * c.c_z, w + s.w_bg, c.c_z, c.c_tri);
    put_transposed(w16, base16 + wg, w + s.w_g, c.c_z, c.c_z);
    put_transposed(w16, base16 + wz, w + s.w_z, c.c_tri, c.c_z);
  };
  tri(off.tri_out, t.to_wa, t.to_wb, t.to_wg, t.to_wz);
  tri(off.tri_in, t.ti_wa, t.ti_wb, t.ti_wg, t.ti_wz);
}

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
  if (c.dtype != PF_F32 && c.dtype != PF_BF16 && c.dtype != PF_BF16_SIMT) return fail(PF_ERR_INVALID_ARG, "bad dtype");
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
  size_t nbytes = n_weight_floats * sizeof(float);
  if (cudaMalloc(&h->w32, nbytes) != cudaSuccess) { delete h; return fail(PF_ERR_ALLOC, "cudaMalloc weights"); }
  if (cudaMemcpy(h->w32, weights_host, nbytes, cudaMemcpyHostToDevice) != cudaSuccess) {
    pf_evoformer_destroy(h);
    return fail(PF_ERR_CUDA, "weights H2D");
  }
  if (c.dtype == PF_BF16) {
    h->tc = tc_layout(c);
    std::vector<uint16_t> w16(h->tc.total_bf16 * c.n_blocks_max, 0);
    std::vector<float> wf(h->tc.total_f32 * c.n_blocks_max, 0.f);
    for (int b = 0; b < c.n_blocks_max; ++b)
      build_tc_block(c, off, h->tc, weights_host + (size_t)b * off.total, w16, (size_t)b * h->tc.total_bf16, wf,
                     (size_t)b * h->tc.total_f32);
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
    h->tc_mask = 0xF;   // bit0 projection GEMMs on tcgen05; attention / triangle einsum / OPM bits as kernels land
    if (const char* e = getenv("PF_TC_MASK")) h->tc_mask = (unsigned)strtoul(e, nullptr, 0);   // debug bisect only
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
  if (h->tma) tma_ctx_destroy(h->tma);
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

// ------------------------------------------------------------------------------------------------
// sub-step driver, templated on the storage type of intermediates
// ------------------------------------------------------------------------------------------------
template <typename T>
struct Driver {
  pf_evoformer* h;
  cudaStream_t st;
  int B, S, N;
  float* msa;
  float* pair;
  const float* seq_mask;
  const float* msa_mask;
  Arena ar;
  const float* w;        // fp32 weights of the current block (device)
  const bf16* w16;       // tc weights of the current block
  const float* wf;       // fused biases of the current block
  std::string err;

  template <typename U>
  U* buf(size_t off) { return reinterpret_cast<U*>(h->ws + off); }

  bool tc(unsigned bit) const { return (h->tc_mask >> bit) & 1u; }

  // one kernel launch: counts it and, when profiling, brackets it with events on the launch stream
  void pb(int kind, double flops, double bytes) {
    h->launches++;
    if (!h->prof_on) return;
    pf_evoformer::ProfRec r{kind, h->next_event(), h->next_event(), flops, bytes};
    cudaEventRecord(r.e0, st);
    h->prof.push_back(r);
  }
  void pe() {
    if (h->prof_on) cudaEventRecord(h->prof.back().e1, st);
  }
  static constexpr double es() { return (double)sizeof(T); }

  static Epi epi_base(int kind, RowGeom g) {
    Epi e;
    memset(&e, 0, sizeof(e));
    e.kind = kind;
    e.scale = 1.0f;
    e.vt_from = 1 << 30;
    e.geom = g;
    return e;
  }

  // acc = A[R,K] W[K,Nout]; W (and W2) fp32 [K, ldw] for SIMT; wt bf16 [Nout(*2), K] for tcgen05
  bool gemm(const T* A, int lda, const float* W, const float* W2, int ldw, const bf16* wt, long R, int K, int Nout,
            const Epi& e) {
    double nacc = (e.kind == EPI_GATED_CM) ? 2.0 : 1.0;
    double out_b = (e.kind == EPI_RESID) ? 8.0 + (e.gate ? es() : 0.0) : es();
    pb(KK_GEMM, 2.0 * R * K * Nout * nacc, (double)R * K * es() + (double)R * Nout * out_b + nacc * K * Nout * 2.0);
    if constexpr (std::is_same<T, bf16>::value) {
      if (tc(0) && wt) {
        if (launch_gemm_tc(h->tma, A, lda, wt, R, K, Nout, e, h->num_sms, st) != 0) {
          err = std::string("gemm_tc: ") + tc_last_error();
          return false;
        }
        pe();
        return true;
      }
    }
    launch_gemm_simt<T>(A, lda, W, W2, ldw, R, K, Nout, e, st);
    pe();
    return true;
  }

  void ln_rows(const float* x, T* y, const float* gamma, const float* beta, long rows, int C, RowGeom g, int transposed) {
    pb(KK_LN, 0.0, (double)rows * C * (4.0 + es()));
    launch_ln_rows<T>(x, y, gamma, beta, rows, C, g, transposed, st);
    pe();
  }

  bool attention(const T* qkg, const T* vt, const T* bias, const float* keymask, T* o, int R, int L, int H) {
    double rows = (double)B * R * L, C = H * 32.0;
    pb(KK_ATTN, 4.0 * rows * L * C, 5.0 * rows * C * es() + (bias ? (double)B * H * L * L * es() : 0.0));
    if constexpr (std::is_same<T, bf16>::value) {
      if (tc(1)) {
        if (launch_attn_tc(h->tma, qkg, vt, bias, keymask, o, B, R, L, pad8(L), H, h->num_sms, st) != 0) {
          err = std::string("attn_tc: ") + tc_last_error();
          return false;
        }
        pe();
        return true;
      }
    }
    launch_attn_simt<T>(qkg, vt, bias, keymask, o, B, R, L, pad8(L), H, st);
    pe();
    return true;
  }

  // Gated attention sub-step on a residual stream `res` viewed as rows (b, x in D1, y in D2), attention along y.
  //   transposed: rows are gathered from / scattered to the (b, y, x) layout of `res`  (A.2, A.8 via their identities)
  bool attn_substep(float* res, int C, int H, RowGeom g, bool transposed, const AttnW& a, const AttnT& at,
                    const float* keymask, const float* bias_src_ln_g, const float* bias_src_ln_b, bool self_bias) {
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
      if (!gemm(X, h->cfg.c_z, w + a.w_bias, nullptr, H, nullptr, P, h->cfg.c_z, H, e)) return false;
    }
    ln_rows(res, X, w + a.ln_g, w + a.ln_b, R, C, g, transposed ? 1 : 0);
    if (self_bias) {       // A.7 / A.8: bias from the same LN(z) rows
      BIAS = buf<T>(ar.bias);
      Epi e = epi_base(EPI_HEADS, g);
      e.out = BIAS;
      e.Lpad = Lp;
      if (!gemm(X, C, w + a.w_bias, nullptr, H, nullptr, R, C, H, e)) return false;
    }
    const float scale = 0.17677669529663687f;   // 1/sqrt(32)
    bool fused = std::is_same<T, bf16>::value && tc(0);
    if (fused) {
      // one launch: [q*scale | k | sigmoid(gate + bg) | v -> vt]
      Epi e = epi_base(EPI_STORE, g);
      e.out = QKG; e.ldo = 3 * C;
      e.scale = scale; e.scale_cols = C;
      e.bias = wf + at.bias_qkgv;
      e.act = ACT_SIGMOID; e.act_lo = 2 * C; e.act_hi = 3 * C;
      e.vt_from = 3 * C; e.vt = VT; e.Lpad = Lp;
      if (!gemm(X, C, nullptr, nullptr, 0, w16 + at.wqkgv, R, C, 4 * C, e)) return false;
    } else {
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
        if (!gemm(X, C, W, nullptr, C, nullptr, R, C, C, e)) return false;
      }
    }
    if (!attention(QKG, VT, BIAS, keymask, O, g.D1, L, H)) return false;
    Epi e = epi_base(EPI_RESID, g);
    e.bias = w + a.bo;
    e.resid = res; e.ldr = C;
    e.transposed = transposed ? 1 : 0;
    return gemm(O, C, w + a.wo, nullptr, C, w16 ? w16 + at.wo : nullptr, R, C, C, e);
  }

  bool transition_substep(float* res, long R, int C, const TransW& t, size_t w1t, size_t w2t) {
    int n = h->cfg.transition_n;
    RowGeom g{1, 1, (int)R};
    T* X = buf<T>(ar.x);
    T* Hb = buf<T>(ar.qkg);
    ln_rows(res, X, w + t.ln_g, w + t.ln_b, R, C, g, 0);
    Epi e1 = epi_base(EPI_STORE, g);
    e1.out = Hb; e1.ldo = n * C;
    e1.bias = w + t.b1;
    e1.act = ACT_RELU; e1.act_lo = 0; e1.act_hi = n * C;
    if (!gemm(X, C, w + t.w1, nullptr, n * C, w16 ? w16 + w1t : nullptr, R, C, n * C, e1)) return false;
    Epi e2 = epi_base(EPI_RESID, g);
    e2.bias = w + t.b2;
    e2.resid = res; e2.ldr = C;
    return gemm(Hb, n * C, w + t.w2, nullptr, C, w16 ? w16 + w2t : nullptr, R, n * C, C, e2);
  }

  bool opm_substep() {
    const pf_config& c = h->cfg;
    const OpmW& o = h->off.opm;
    long M = (long)B * S * N;
    double P = (double)B * N * N, cc = (double)c.c_opm * c.c_opm;
    T* X = buf<T>(ar.x);
    if constexpr (std::is_same<T, bf16>::value) {
      if (tc(0) && tc(3) && S <= 512) {
        // rows (b, i, s): the projection epilogue writes a|b transposed, [(b,i), 64, Spad], s contiguous
        RowGeom gt{B, N, S};
        int Sp = pad8(S);
        T* ABT = buf<T>(ar.vt);
        ln_rows(msa, X, w + o.ln_g, w + o.ln_b, M, c.c_m, gt, 1);
        Epi e = epi_base(EPI_STORE, gt);
        e.bias = wf + h->tc.opm_bias_ab;
        e.rowmask = RM_MSA; e.seq_mask = seq_mask; e.msa_mask = msa_mask; e.mask_transposed = 1;
        e.vt_from = 0; e.vt = ABT; e.Lpad = Sp;
        if (!gemm(X, c.c_m, nullptr, nullptr, 0, w16 + h->tc.opm_wab, M, c.c_m, 2 * c.c_opm, e)) return false;
        pb(KK_OPM, 2.0 * P * cc * S + 2.0 * P * cc * c.c_z, 2.0 * M * c.c_opm * es() + 8.0 * P * c.c_z);
        if (launch_opm_tc(h->tma, ABT, w16 + h->tc.opm_wout, w + o.bout, seq_mask, msa_mask, pair, B, S, Sp, N, st) != 0) {
          err = std::string("opm_tc: ") + tc_last_error();
          return false;
        }
        pe();
        return true;
      }
    }
    RowGeom g{B, S, N};
    T* OA = buf<T>(ar.oa);
    T* OB = buf<T>(ar.ob);
    ln_rows(msa, X, w + o.ln_g, w + o.ln_b, M, c.c_m, g, 0);
    for (int part = 0; part < 2; ++part) {
      Epi e = epi_base(EPI_STORE, g);
      e.out = part ? OB : OA; e.ldo = c.c_opm;
      e.bias = w + (part ? o.bb : o.ba);
      e.rowmask = RM_MSA; e.seq_mask = seq_mask; e.msa_mask = msa_mask;
      if (!gemm(X, c.c_m, w + (part ? o.wb : o.wa), nullptr, c.c_opm, nullptr, M, c.c_m, c.c_opm, e)) return false;
    }
    pb(KK_OPM, 2.0 * P * cc * S + 2.0 * P * cc * c.c_z, 2.0 * M * c.c_opm * es() + 8.0 * P * c.c_z);
    launch_opm_simt<T>(OA, OB, w + o.wout, w + o.bout, seq_mask, msa_mask, pair, B, S, N, c.c_opm, c.c_z, st);
    pe();
    return true;
  }

  bool trimul_substep(bool incoming) {
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
    size_t wa16 = incoming ? h->tc.ti_wa : h->tc.to_wa, wb16 = incoming ? h->tc.ti_wb : h->tc.to_wb;
    size_t wg16 = incoming ? h->tc.ti_wg : h->tc.to_wg, wz16 = incoming ? h->tc.ti_wz : h->tc.to_wz;
    for (int part = 0; part < 2; ++part) {
      // incoming (A.6) = outgoing on the transposed rows with the a/b projections swapped (SURVEY.md §0 finding 1)
      bool use_b = (part == 1) != incoming;
      Epi e = epi_base(EPI_GATED_CM, g);
      e.out = part ? BCM : ACM;
      e.Lpad = Np;
      e.bias = w + (use_b ? t.b_bp : t.b_ap);
      e.bias2 = w + (use_b ? t.b_bg : t.b_ag);
      e.rowmask = RM_PAIR; e.seq_mask = seq_mask;
      const bf16* wt = w16 ? w16 + (use_b ? wb16 : wa16) : nullptr;
      if (!gemm(X, c.c_z, w + (use_b ? t.w_bp : t.w_ap), w + (use_b ? t.w_bg : t.w_ag), c.c_tri, wt, P, c.c_z,
                c.c_tri, e))
        return false;
    }
    {
      Epi e = epi_base(EPI_STORE, g);
      e.out = G; e.ldo = c.c_z;
      e.bias = w + t.b_g;
      e.act = ACT_SIGMOID; e.act_lo = 0; e.act_hi = c.c_z;
      if (!gemm(X, c.c_z, w + t.w_g, nullptr, c.c_z, w16 ? w16 + wg16 : nullptr, P, c.c_z, c.c_z, e)) return false;
    }
    pb(KK_TRI, 2.0 * B * c.c_tri * (double)N * N * N, (double)B * c.c_tri * N * Np * (2.0 * es() + 4.0));
    bool done = false;
    if constexpr (std::is_same<T, bf16>::value) {
      if (tc(2)) {
        if (launch_tri_einsum_tc(h->tma, ACM, BCM, TCM, B * c.c_tri, N, Np, h->num_sms, st) != 0) {
          err = std::string("tri_einsum_tc: ") + tc_last_error();
          return false;
        }
        done = true;
      }
    }
    if (!done) launch_tri_einsum_simt<T>(ACM, BCM, TCM, B * c.c_tri, N, Np, st);
    pe();
    pb(KK_LNC, 0.0, (double)P * c.c_tri * (4.0 + es()));
    launch_lnc<T>(TCM, TN, w + t.ln_out_g, w + t.ln_out_b, B, c.c_tri, N, Np, st);
    pe();
    Epi e = epi_base(EPI_RESID, g);
    e.bias = w + t.b_z;
    e.resid = pair; e.ldr = c.c_z;
    e.gate = G; e.ldg = c.c_z;
    e.transposed = incoming ? 1 : 0;
    return gemm(TN, c.c_tri, w + t.w_z, nullptr, c.c_z, w16 ? w16 + wz16 : nullptr, P, c.c_tri, c.c_z, e);
  }

  bool run_substep(int block, int step) {
    const pf_config& c = h->cfg;
    w = h->w32 + (size_t)block * h->off.total;
    w16 = h->w16 ? h->w16 + (size_t)block * h->tc.total_bf16 : nullptr;
    wf = h->wf ? h->wf + (size_t)block * h->tc.total_f32 : nullptr;
    switch (step) {
      case 1: return attn_substep(msa, c.c_m, c.heads_msa, RowGeom{B, S, N}, false, h->off.row, h->tc.row, seq_mask,
                                  w + h->off.row.ln_z_g, w + h->off.row.ln_z_b, false);
      case 2: return attn_substep(msa, c.c_m, c.heads_msa, RowGeom{B, N, S}, true, h->off.col, h->tc.col, msa_mask,
                                  nullptr, nullptr, false);
      case 3: return transition_substep(msa, (long)B * S * N, c.c_m, h->off.msa_trans, h->tc.mt_w1, h->tc.mt_w2);
      case 4: return opm_substep();
      case 5: return trimul_substep(false);
      case 6: return trimul_substep(true);
      case 7: return attn_substep(pair, c.c_z, c.heads_pair, RowGeom{B, N, N}, false, h->off.tri_start,
                                  h->tc.tri_start, seq_mask, nullptr, nullptr, true);
      case 8: return attn_substep(pair, c.c_z, c.heads_pair, RowGeom{B, N, N}, true, h->off.tri_end, h->tc.tri_end,
                                  seq_mask, nullptr, nullptr, true);
      case 9: return transition_substep(pair, (long)B * N * N, c.c_z, h->off.pair_trans, h->tc.pt_w1, h->tc.pt_w2);
    }
    err = "substep not in 1..9";
    return false;
  }
};

static pf_status check_and_grow(pf_evoformer* h, const float* msa, const float* pair, const float* sm, const float* mm,
                                int B, int S, int N) {
  if (!h || !msa || !pair || !sm || !mm) return fail(PF_ERR_INVALID_ARG, "null argument");
  if (B < 1 || S < 1 || N < 1) return fail(PF_ERR_SHAPE, "B, S, N must be >= 1");
  if ((long)B * S > 65535 || (long)B * N > 65535) return fail(PF_ERR_SHAPE, "B*S and B*N must be <= 65535");
  size_t need = arena_layout(h->cfg, B, S, N).total;
  if (need > h->ws_bytes) {
    cudaDeviceSynchronize();
    cudaFree(h->ws);
    h->ws = nullptr;
    h->ws_bytes = 0;
    if (cudaMalloc(&h->ws, need) != cudaSuccess) {
      cudaGetLastError();
      return fail(PF_ERR_ALLOC, "cudaMalloc workspace");
    }
    h->ws_bytes = need;
  }
  return PF_OK;
}

template <typename T>
static pf_status run(pf_evoformer* h, float* msa, float* pair, const float* sm, const float* mm, int B, int S, int N,
                     int block0, int block1, int step0, int step1, cudaStream_t st) {
  Driver<T> d;
  d.h = h; d.st = st; d.B = B; d.S = S; d.N = N;
  d.msa = msa; d.pair = pair; d.seq_mask = sm; d.msa_mask = mm;
  d.ar = arena_layout(h->cfg, B, S, N);
  h->launches = 0;
  for (int blk = block0; blk < block1; ++blk)
    for (int step = step0; step <= step1; ++step) {
      if (!d.run_substep(blk, step)) return fail(PF_ERR_CUDA, d.err);
      cudaError_t e = cudaGetLastError();
      if (e != cudaSuccess)
        return fail(PF_ERR_CUDA, std::string("launch failed in block ") + std::to_string(blk) + " substep " +
                                     std::to_string(step) + ": " + cudaGetErrorString(e));
    }
  return PF_OK;
}

static pf_status dispatch(pf_evoformer* h, float* msa, float* pair, const float* sm, const float* mm, int B, int S,
                          int N, int block0, int block1, int step0, int step1, void* stream) {
  pf_status s = check_and_grow(h, msa, pair, sm, mm, B, S, N);
  if (s != PF_OK) return s;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (h->cfg.dtype == PF_F32) return run<float>(h, msa, pair, sm, mm, B, S, N, block0, block1, step0, step1, st);
  return run<bf16>(h, msa, pair, sm, mm, B, S, N, block0, block1, step0, step1, st);
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
  CUDA_TRY(cudaMemcpyAsync(dm, msa_host, nm, cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(dz, pair_host, nz, cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(ds, seq_mask_host, (size_t)B * N * 4, cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(dr, msa_mask_host, (size_t)B * S * 4, cudaMemcpyHostToDevice, st));
  pf_status s = pf_evoformer_forward(h, dm, dz, ds, dr, B, S, N, n_blocks, stream);
  if (s != PF_OK) return s;
  CUDA_TRY(cudaMemcpyAsync(msa_host, dm, nm, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemcpyAsync(pair_host, dz, nz, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return PF_OK;
}
