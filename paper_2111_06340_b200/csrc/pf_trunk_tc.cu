// tcgen05 path of the trunk (PF_BF16): device weight layout and the per-sub-step launch sequences of SURVEY.md §8(a).
// 16-bit MMA operands with fp32 accumulation, fp32 residual streams (R1).  Storage formats (reading R17):
// LayerNorm outputs and the weights they multiply are fp16 operands (bounded by construction; the weight values are the
// bf16-rounded ones of R15, which fp16 represents exactly inside its normal range 2^-14 .. 65504 — smaller magnitudes lose
// bits, larger ones are refused at create time, see F16Range), sigmoid gates are stored as fp16 (never an MMA operand), every other
// intermediate (q, k, v, P, o, transition hidden, triangle operands, outer-product operands, pair bias) is bf16.
// No arithmetic of the method lives here except two constants handed to the projection epilogues: log2(e)/sqrt(head_dim) on q
// (R12) and log2(e) on the pair bias, so that the attention kernel's softmax runs in the exp2 domain.
#include "pf_handle.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

namespace pf {

// ------------------------------------------------------------------------------------------------
// weights
// ------------------------------------------------------------------------------------------------
static uint16_t f32_to_bf16_bits(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  uint32_t lsb = (u >> 16) & 1;
  u += 0x7FFFu + lsb;
  return (uint16_t)(u >> 16);
}
static uint16_t f32_to_f16_bits(float f) {
  __half h = __float2half_rn(f);   // host-callable conversion
  uint16_t b;
  memcpy(&b, &h, 2);
  return b;
}

static F16Range* g_range = nullptr;   // set for the duration of one build_tc_block call (create is not re-entrant per handle)

// dst[n, k] = src[k, n]  (src row-major [K, ld_src], columns [0, Nout)) as 16-bit
static void put_transposed(std::vector<uint16_t>& dst, size_t at, const float* src, int K, int Nout, bool f16) {
  for (int n = 0; n < Nout; ++n)
    for (int k = 0; k < K; ++k) {
      float v = src[(size_t)k * Nout + n];
      if (f16 && g_range) {
        const float a = v < 0 ? -v : v;
        if (!(a <= 65504.0f)) g_range->overflow++;           // also catches NaN
        else if (a != 0.0f && a < 6.103515625e-05f) g_range->below_normal++;
      }
      dst[at + (size_t)n * K + k] = f16 ? f32_to_f16_bits(v) : f32_to_bf16_bits(v);
    }
}

TcBlock tc_layout(const pf_config& c) {
  TcBlock t{};
  size_t o = 0, f = 0;
  auto take = [&](size_t k) { size_t r = o; o += align_up(k, 64); return r; };
  auto takef = [&](size_t k) { size_t r = f; f += align_up(k, 32); return r; };
  auto attn = [&](int ch, int extra) {
    AttnT a{};
    a.w_in = take((size_t)(4 * ch + extra) * ch);
    a.b_in = takef((size_t)4 * ch + extra);
    a.wo = take((size_t)ch * ch);
    return a;
  };
  t.row = attn(c.c_m, 0);
  t.col = attn(c.c_m, 0);
  t.tri_start = attn(c.c_z, c.heads_pair);
  t.tri_end = attn(c.c_z, c.heads_pair);
  t.row_wbias = take((size_t)c.heads_msa * c.c_z);
  size_t n = c.transition_n;
  t.mt_w1 = take(n * c.c_m * c.c_m); t.mt_w2 = take(n * c.c_m * c.c_m);
  t.pt_w1 = take(n * c.c_z * c.c_z); t.pt_w2 = take(n * c.c_z * c.c_z);
  t.opm_wab = take((size_t)2 * c.c_opm * c.c_m);
  t.opm_bias_ab = takef((size_t)2 * c.c_opm);
  t.opm_wout = take((size_t)c.c_opm * c.c_opm * c.c_z);
  t.to_w = take((size_t)5 * c.c_tri * c.c_z); t.to_b = takef((size_t)5 * c.c_tri); t.to_wz = take((size_t)c.c_z * c.c_tri);
  t.ti_w = take((size_t)5 * c.c_tri * c.c_z); t.ti_b = takef((size_t)5 * c.c_tri); t.ti_wz = take((size_t)c.c_z * c.c_tri);
  t.total16 = o;
  t.total_f32 = f;
  return t;
}

void build_tc_block(const pf_config& c, const BlockW& off, const TcBlock& t, const float* w, std::vector<uint16_t>& w16,
                    size_t base16, std::vector<float>& wf, size_t basef, F16Range* range) {
  g_range = range;
  auto attn = [&](const AttnW& a, const AttnT& d, int ch, int heads, bool self_bias) {
    // column order of the fused projection: [q | k | gate | v (| pair-bias heads)], all fed by LN(x): fp16
    put_transposed(w16, base16 + d.w_in + (size_t)0 * ch * ch, w + a.wq, ch, ch, true);
    put_transposed(w16, base16 + d.w_in + (size_t)1 * ch * ch, w + a.wk, ch, ch, true);
    put_transposed(w16, base16 + d.w_in + (size_t)2 * ch * ch, w + a.wg, ch, ch, true);
    put_transposed(w16, base16 + d.w_in + (size_t)3 * ch * ch, w + a.wv, ch, ch, true);
    if (self_bias) put_transposed(w16, base16 + d.w_in + (size_t)4 * ch * ch, w + a.w_bias, ch, heads, true);
    int nb = 4 * ch + (self_bias ? heads : 0);
    for (int i = 0; i < nb; ++i) wf[basef + d.b_in + i] = 0.f;
    for (int i = 0; i < ch; ++i) wf[basef + d.b_in + 2 * ch + i] = w[a.bg + i];
    put_transposed(w16, base16 + d.wo, w + a.wo, ch, ch, false);
  };
  attn(off.row, t.row, c.c_m, c.heads_msa, false);
  attn(off.col, t.col, c.c_m, c.heads_msa, false);
  attn(off.tri_start, t.tri_start, c.c_z, c.heads_pair, true);
  attn(off.tri_end, t.tri_end, c.c_z, c.heads_pair, true);
  put_transposed(w16, base16 + t.row_wbias, w + off.row.w_bias, c.c_z, c.heads_msa, true);
  int n = c.transition_n;
  put_transposed(w16, base16 + t.mt_w1, w + off.msa_trans.w1, c.c_m, n * c.c_m, true);
  put_transposed(w16, base16 + t.mt_w2, w + off.msa_trans.w2, n * c.c_m, c.c_m, false);
  put_transposed(w16, base16 + t.pt_w1, w + off.pair_trans.w1, c.c_z, n * c.c_z, true);
  put_transposed(w16, base16 + t.pt_w2, w + off.pair_trans.w2, n * c.c_z, c.c_z, false);
  put_transposed(w16, base16 + t.opm_wab, w + off.opm.wa, c.c_m, c.c_opm, true);
  put_transposed(w16, base16 + t.opm_wab + (size_t)c.c_opm * c.c_m, w + off.opm.wb, c.c_m, c.c_opm, true);
  for (int i = 0; i < c.c_opm; ++i) {
    wf[basef + t.opm_bias_ab + i] = w[off.opm.ba + i];
    wf[basef + t.opm_bias_ab + c.c_opm + i] = w[off.opm.bb + i];
  }
  put_transposed(w16, base16 + t.opm_wout, w + off.opm.wout, c.c_opm * c.c_opm, c.c_z, true);   // fp16 as the outer product it multiplies
  // triangle multiplication: the einsum kernel contracts buffer 0 (rows i) with buffer 1 (rows j) along k.
  // outgoing (A.5): buffer 0 = a, buffer 1 = b.  incoming (A.6) runs on the transposed rows with a and b swapped
  // (SURVEY.md §0 finding 1): buffer 0 = b, buffer 1 = a.
  auto tri = [&](const TriMulW& s, size_t wdst, size_t bdst, size_t wz, bool swap) {
    const int ct = c.c_tri, cz = c.c_z;
    size_t blk = (size_t)ct * cz;
    size_t p0 = swap ? s.w_bp : s.w_ap, g0 = swap ? s.w_bg : s.w_ag, p1 = swap ? s.w_ap : s.w_bp, g1 = swap ? s.w_ag : s.w_bg;
    size_t bp0 = swap ? s.b_bp : s.b_ap, bg0 = swap ? s.b_bg : s.b_ag, bp1 = swap ? s.b_ap : s.b_bp, bg1 = swap ? s.b_ag : s.b_bg;
    put_transposed(w16, base16 + wdst + 0 * blk, w + p0, cz, ct, true);
    put_transposed(w16, base16 + wdst + 1 * blk, w + g0, cz, ct, true);
    put_transposed(w16, base16 + wdst + 2 * blk, w + p1, cz, ct, true);
    put_transposed(w16, base16 + wdst + 3 * blk, w + g1, cz, ct, true);
    put_transposed(w16, base16 + wdst + 4 * blk, w + s.w_g, cz, cz, true);
    for (int i = 0; i < ct; ++i) {
      wf[basef + bdst + 0 * ct + i] = w[bp0 + i];
      wf[basef + bdst + 1 * ct + i] = w[bg0 + i];
      wf[basef + bdst + 2 * ct + i] = w[bp1 + i];
      wf[basef + bdst + 3 * ct + i] = w[bg1 + i];
      wf[basef + bdst + 4 * ct + i] = w[s.b_g + i];
    }
    put_transposed(w16, base16 + wz, w + s.w_z, ct, cz, true);
  };
  tri(off.tri_out, t.to_w, t.to_b, t.to_wz, false);
  tri(off.tri_in, t.ti_w, t.ti_b, t.ti_wz, true);
  g_range = nullptr;
}


// ------------------------------------------------------------------------------------------------
// sub-step driver
// ------------------------------------------------------------------------------------------------
namespace {

constexpr float kLog2e = 1.4426950408889634f;

struct TcDriver {
  typedef G2Desc G2Desc_;
  pf_evoformer* h;
  cudaStream_t st;
  int B, S, N;
  float* msa;
  float* pair;
  const float* seq_mask;
  const float* msa_mask;
  Arena ar;
  const float* w;        // fp32 blob of the current block (device): LN parameters and un-fused biases
  const uint16_t* w16;   // 16-bit matrices of the current block
  const float* wf;       // fused fp32 biases of the current block
  std::string err;

  template <typename U>
  U* buf(size_t off) { return reinterpret_cast<U*>(h->ws + off); }
  const unsigned char* flags(size_t off) { return reinterpret_cast<const unsigned char*>(h->ws + off); }

  static G2Desc desc_base(int B, int D1, int D2, int K, int Nw) {
    G2Desc d;
    memset(&d, 0, sizeof(d));
    d.B = B; d.D1 = D1; d.D2 = D2; d.K = K; d.Nw = Nw;
    return d;
  }
  static G2Op op(int kind, int dst_col, int ncols = 64) {
    G2Op o;
    memset(&o, 0, sizeof(o));
    o.kind = kind; o.dst_col = dst_col; o.ncols = ncols; o.scale = 1.0f;
    return o;
  }

  // frac: share of the row tiles that is executed (mask-derived skipping), applied to the FLOP / byte tags
  bool gemm2(const G2Desc& d, double out_bytes, double frac) {
    double R = (double)d.B * d.D1 * d.D2 * frac;
    out_bytes *= frac;
    double in_bytes = R * d.K * (d.a_mode == 0 ? 4.0 : 2.0);
    h->prof_begin(KK_LNGEMM, 2.0 * R * d.K * d.Nw, in_bytes + out_bytes + 2.0 * d.K * d.Nw, st);
    if (launch_gemm2(h->tma, d, h->num_sms, st) != 0) {
      err = std::string("gemm2: ") + tc_last_error();
      return false;
    }
    h->prof_end(st);
    return true;
  }

  // Gated attention sub-step on a residual stream `res` viewed as rows (b, x in D1, y in D2), attention along y.
  //   transposed: rows are gathered from / scattered to the (b, y, x) layout of `res`  (A.2, A.8 via their identities)
  //   f_rows: active-tile flags of this row geometry; rl_off / rl_idx: the compacted row list of this attention (pf_flags.cu)
  // Where one attention's own parameters live: the handle's blobs for the main block, the extra-MSA stack's own buffers for
  // its row attention (there the residual stream has Kin = c_e = 64 channels while the attention runs on C = H x 32 columns:
  // heads of dimension 8 zero-padded to the 32 the attention core is built for).
  struct AttnPar {
    int Kin;                          // channels of the residual stream = LayerNorm width = reduction length of the projection
    const float *ln_g, *ln_b;
    const void* w_in;                 // fp16 [4C (+H), Kin]
    const float* b_in;                // fp32 [4C (+H)]
    const void* wo;                   // bf16 [Kin, C]
    const float* bo;                  // fp32 [Kin]
    float qscale;                     // 1 / sqrt(head dimension)  (R12)
  };
  AttnPar main_par(int C, const AttnW& a, const AttnT& at) const {
    return AttnPar{C, w + a.ln_g, w + a.ln_b, w16 + at.w_in, wf + at.b_in, w16 + at.wo, w + a.bo, 0.17677669529663687f};
  }

  bool attn_substep(float* res, int C, int H, int D1, int D2, bool transposed, const AttnW& a, const AttnPar& px,
                    const float* keymask, bool row_bias, bool self_bias, size_t f_rows, size_t rl_off, int rl_idx) {
    const double f_frac = rl_idx == 0 ? h->frac.msa : rl_idx == 1 ? h->frac.msat : h->frac.pair;
    const double a_frac = rl_idx == 0 ? h->frac.attn_row : rl_idx == 1 ? h->frac.attn_col : h->frac.attn_tri;
    const pf_config& c = h->cfg;
    const double R = (double)B * D1 * D2;
    const int L = D2, Lp = pad8(L);
    bf16* QKG = buf<bf16>(ar.qkg);
    bf16* VT = buf<bf16>(ar.vt);
    bf16* O = buf<bf16>(ar.o);
    bf16* BIAS = (row_bias || self_bias) ? buf<bf16>(ar.bias) : nullptr;
    if (row_bias && c.c_z == 128 && c.heads_msa <= 8 && (double)B * N * N < 4.0e9) {
      // A.1: beta[h,i,j] = Lin0(LN'(z[i,j]))_h — 16 bytes out per 512 bytes in: a streaming SIMT kernel (pf_simt.cu)
      h->prof_begin(KK_HEADS, 2.0 * B * N * N * c.c_z * c.heads_msa * h->frac.pair_rows,
                    (double)B * N * N * (c.c_z * 4.0 + c.heads_msa * 2.0) * h->frac.pair_rows, st);
      launch_ln_heads128(pair, w + a.ln_z_g, w + a.ln_z_b, w + a.w_bias, kLog2e, seq_mask, BIAS, B, N, pad8(N), c.heads_msa,
                         h->num_sms, st);
      h->prof_end(st);
    } else if (row_bias) {
      G2Desc d = desc_base(B, N, N, c.c_z, c.heads_msa);
      d.src = pair; d.gamma = w + a.ln_z_g; d.beta = w + a.ln_z_b;
      d.op_fmt = 1; d.Wt = w16 + h->tc.row_wbias;
      d.heads_out = BIAS; d.n_heads = c.heads_msa; d.Lpad = pad8(N);
      d.ops[0] = op(G2_HEADS, 0, c.heads_msa);
      d.ops[0].scale = kLog2e;
      d.n_ops = 1;
      d.tile_active = flags(ar.f_pair);
      if (!gemm2(d, (double)B * N * N * c.heads_msa * 2.0, h->frac.pair)) return false;
    }
    {
      const int Nw = 4 * C + (self_bias ? H : 0);
      G2Desc d = desc_base(B, D1, D2, px.Kin, Nw);
      d.src = res; d.src_transposed = transposed ? 1 : 0; d.gamma = px.ln_g; d.beta = px.ln_b;
      d.op_fmt = 1; d.Wt = px.w_in; d.bias = px.b_in;
      d.bias_lo = 2 * C; d.bias_n = C;   // only the gate columns carry a bias (R7)
      d.row_out[0] = QKG; d.row_ld[0] = 3 * C;
      d.vt_out = VT; d.vt_cols = C; d.Lpad = Lp;
      d.heads_out = BIAS; d.n_heads = H;
      int n = 0;
      for (int col = 0; col < 4 * C; col += 64, ++n) {
        int seg = col / C;
        if (seg < 3) {
          d.ops[n] = op(G2_ROW16, col);
          if (seg == 0) d.ops[n].scale = px.qscale * kLog2e;   // log2(e)/sqrt(d)  (R12)
          if (seg == 2) { d.ops[n].act = ACT_SIGMOID; d.ops[n].fmt = 1; }
        } else if (g2_pick_yt(D2) >= 64) {
          // V^T comes out of the MMA already transposed: the half-window holding these columns is computed operand-swapped
          d.ops[n] = op(G2_VTS, ((col - 3 * C) / 128) * 128);
          d.swap_mask |= 1u << (col / 128);
        } else {
          d.ops[n] = op(G2_VT, col - 3 * C);
        }
      }
      if (self_bias) {   // A.7 / A.8: beta from the same LN(z) rows
        d.ops[n] = op(G2_HEADS, 0, H);
        d.ops[n++].scale = kLog2e;
      }
      d.n_ops = n;
      d.tile_active = flags(f_rows);
      if (!gemm2(d, R * 4.0 * C * 2.0 + (self_bias ? R * H * 2.0 : 0.0), f_frac)) return false;
    }
    {
      double rows = R, Cc = C;
      h->prof_begin(KK_ATTN, 4.0 * rows * L * Cc * a_frac,
                    (5.0 * rows * Cc * 2.0 + (BIAS ? (double)B * H * L * L * 2.0 : 0.0)) * a_frac, st);
      if (launch_attn_tc(h->tma, QKG, VT, BIAS, keymask, O, B, D1, L, Lp, H, h->ws + rl_off, buf<int>(ar.rl_count) + rl_idx,
                         h->num_sms, st) != 0) {
        err = std::string("attn_tc: ") + tc_last_error();
        return false;
      }
      h->prof_end(st);
    }
    G2Desc d = desc_base(B, D1, D2, C, px.Kin);
    d.a_mode = 1; d.A = O; d.op_fmt = 0; d.Wt = px.wo; d.bias = px.bo;
    d.resid = res; d.resid_ld = px.Kin; d.resid_transposed = transposed ? 1 : 0;
    int n = 0;
    for (int col = 0; col < px.Kin; col += 64) d.ops[n++] = op(G2_RESID, col);
    d.n_ops = n;
    d.tile_active = flags(f_rows);
    return gemm2(d, R * px.Kin * 8.0, f_frac);
  }

  // A.3 / A.9: one fused kernel, the 4C-wide hidden activation stays on chip
  bool transition_substep(float* res, int D1, int D2, int C, const TransW& t, size_t w1t, size_t w2t, size_t f_lin) {
    const double R = (double)B * D1 * D2 * (C == h->cfg.c_m ? h->frac.msa_lin : h->frac.pair_lin);
    const double n4 = (double)h->cfg.transition_n * C;
    h->prof_begin(KK_TRANS, 4.0 * R * n4 * C, R * C * 8.0 + 4.0 * n4 * C, st);
    if (launch_transition_tc(h->tma, res, (long)B * D1 * D2, C, w + t.ln_g, w + t.ln_b, w16 + w1t, w + t.b1, w16 + w2t,
                             w + t.b2, flags(f_lin), h->num_sms, st) != 0) {
      err = std::string("transition_tc: ") + tc_last_error();
      return false;
    }
    h->prof_end(st);
    return true;
  }

  bool opm_substep() {
    const pf_config& c = h->cfg;
    const OpmW& o = h->off.opm;
    const double M = (double)B * S * N, P = (double)B * N * N, cc = (double)c.c_opm * c.c_opm;
    const int Sp = pad8(S);
    bf16* ABT = buf<bf16>(ar.vt);
    // rows (b, i, s) gathered from msa[(b, s, i)]: a | b masked and written transposed, [(b,i), 64, Spad], s contiguous
    if (c.c_m == 256 && c.c_opm == 32) {
      // 128 bytes out per KB in: a streaming kernel with the LayerNorm in registers and mma.sync for the 64 columns (pf_simt.cu)
      h->prof_begin(KK_OPMAB, 2.0 * M * c.c_m * 2.0 * c.c_opm * h->frac.msat_x,
                    M * (c.c_m * 4.0 + 2.0 * c.c_opm * 2.0) * h->frac.msat_x, st);
      launch_ln_opm_ab256(msa, w + o.ln_g, w + o.ln_b, w + o.wa, w + o.wb, w + o.ba, w + o.bb, seq_mask, msa_mask, ABT, B, S, N, Sp,
                          h->num_sms, st);
      h->prof_end(st);
    } else {
    G2Desc d = desc_base(B, N, S, c.c_m, 2 * c.c_opm);
    d.src = msa; d.src_transposed = 1; d.gamma = w + o.ln_g; d.beta = w + o.ln_b;
    d.op_fmt = 1; d.Wt = w16 + h->tc.opm_wab; d.bias = wf + h->tc.opm_bias_ab;
    d.rowmask = RM_MSA; d.seq_mask = seq_mask; d.msa_mask = msa_mask; d.mask_transposed = 1;
    d.vt_out = ABT; d.vt_cols = 2 * c.c_opm; d.Lpad = Sp;
    d.ops[0] = op(G2_VT, 0, 2 * c.c_opm);
    d.ops[0].fmt = 1;   // fp16 operands of the outer product
    d.ops[0].masked = 1;
    d.n_ops = 1;
    d.tile_active = flags(ar.f_msat_x);   // a, b are summed over s: masked s must be written as zeros
    if (!gemm2(d, M * 2.0 * c.c_opm * 2.0, h->frac.msat_x)) return false;
    }
    h->prof_begin(KK_OPM, (2.0 * P * cc * S + 2.0 * P * cc * c.c_z) * h->frac.opm,
                  (2.0 * M * c.c_opm * 2.0 + 8.0 * P * c.c_z) * h->frac.opm, st);
    if (launch_opm_tc(h->tma, ABT, reinterpret_cast<const bf16*>(w16 + h->tc.opm_wout), w + o.bout, seq_mask, msa_mask,
                      pair, B, S, Sp, N, st) != 0) {
      err = std::string("opm_tc: ") + tc_last_error();
      return false;
    }
    h->prof_end(st);
    return true;
  }

  bool trimul_substep(bool incoming) {
    const pf_config& c = h->cfg;
    const TriMulW& t = incoming ? h->off.tri_in : h->off.tri_out;
    const double P = (double)B * N * N;
    const int Np = pad8(N), ct = c.c_tri;
    bf16* ACM = buf<bf16>(ar.acm);
    bf16* BCM = buf<bf16>(ar.bcm);
    __half* G = buf<__half>(ar.g);
    bf16* TCM = buf<bf16>(ar.tcm);
    __half* TN = buf<__half>(ar.tn);
    {
      G2Desc d = desc_base(B, N, N, c.c_z, 5 * ct);
      d.src = pair; d.src_transposed = incoming ? 1 : 0; d.gamma = w + t.ln_in_g; d.beta = w + t.ln_in_b;
      d.op_fmt = 1; d.Wt = w16 + (incoming ? h->tc.ti_w : h->tc.to_w); d.bias = wf + (incoming ? h->tc.ti_b : h->tc.to_b);
      d.rowmask = RM_PAIR; d.seq_mask = seq_mask;
      d.cm_out[0] = ACM; d.cm_out[1] = BCM; d.cm_channels = ct; d.Lpad = Np;
      d.row_out[0] = G; d.row_ld[0] = c.c_z;
      for (int tile = 0; tile < 2; ++tile)
        for (int j = 0; j < 4; ++j) {
          if (g2_pick_yt(N) >= 64) {
            // both halves (p | gate) of the window are computed operand-swapped: the gated operand leaves the MMA channel-major
            d.ops[tile * 4 + j] = j < 2 ? op(G2_CMS, 0) : op(G2_SKIP, 0);
            d.swap_mask |= 3u << (2 * tile);
          } else {
            d.ops[tile * 4 + j] = j < 2 ? op(G2_CM_DUAL, j * 64) : op(G2_SKIP, 0);
          }
          d.ops[tile * 4 + j].map = tile;
        }
      for (int j = 0; j < 2; ++j) {
        d.ops[8 + j] = op(G2_ROW16, j * 64);
        d.ops[8 + j].act = ACT_SIGMOID;
        d.ops[8 + j].fmt = 1;
      }
      d.n_ops = 10;
      d.tile_active = flags(ar.f_pair_x);   // a, b are summed over k: masked k must be written as zeros
      if (!gemm2(d, P * 3.0 * ct * 2.0, h->frac.pair_x)) return false;
    }
    h->prof_begin(KK_TRI, 2.0 * B * ct * (double)N * N * N * h->frac.tri_k,
                  (double)B * ct * N * Np * (4.0 * h->frac.tri_k + 2.0), st);
    if (launch_tri_einsum_tc(h->tma, ACM, BCM, TCM, B * ct, N, Np, buf<int>(ar.kt_seq), ct, h->num_sms, st) != 0) {
      err = std::string("tri_einsum_tc: ") + tc_last_error();
      return false;
    }
    h->prof_end(st);
    h->prof_begin(KK_LNC, 0.0, P * ct * 4.0 * h->frac.lnc, st);
    launch_lnc_tc(TCM, TN, w + t.ln_out_g, w + t.ln_out_b, seq_mask, B, N, Np, st);
    h->prof_end(st);
    G2Desc d = desc_base(B, N, N, ct, c.c_z);
    d.a_mode = 1; d.A = TN; d.op_fmt = 1; d.Wt = w16 + (incoming ? h->tc.ti_wz : h->tc.to_wz); d.bias = w + t.b_z;
    d.resid = pair; d.resid_ld = c.c_z; d.resid_transposed = incoming ? 1 : 0;
    d.gate = G; d.ldg = c.c_z;
    d.ops[0] = op(G2_RESID, 0);
    d.ops[1] = op(G2_RESID, 64);
    d.n_ops = 2;
    d.tile_active = flags(ar.f_pair);
    return gemm2(d, P * c.c_z * 10.0, h->frac.pair);
  }
};

}  // namespace

// Host restatement of the skipping rules of pf_flags.cu, used only while profiling to scale the FLOP / byte tags.
static void host_work_fractions(pf_evoformer* h, const std::vector<float>& sg, const std::vector<float>& rho, int B, int S,
                                int N) {
  auto act = [&](int kind, int b, int x, int y, int D1, int D2) {
    if (kind == 3) return sg[(size_t)b * D1 + x] > 0.5f;
    const float mx = (kind == 0 ? rho : sg)[(size_t)b * D1 + x], my = (kind == 1 ? rho : sg)[(size_t)b * D2 + y];
    return mx * my > 0.5f;
  };
  auto tiles2d = [&](int kind, int D1, int D2) {
    const int yt = g2_pick_yt(D2), xt = 128 / yt;
    long on = 0, all = 0;
    for (int b = 0; b < B; ++b)
      for (int x0 = 0; x0 < D1; x0 += xt)
        for (int y0 = 0; y0 < D2; y0 += yt, ++all) {
          bool any = false;
          for (int x = x0; x < x0 + xt && x < D1 && !any; ++x)
            for (int y = y0; y < y0 + yt && y < D2 && !any; ++y) any = act(kind, b, x, y, D1, D2);
          on += any;
        }
    return all ? (double)on / all : 1.0;
  };
  auto tiles_lin = [&](int kind, int D1, int D2) {
    const long R = (long)B * D1 * D2, per = (long)D1 * D2;
    long on = 0, all = 0;
    for (long t0 = 0; t0 < R; t0 += 128, ++all) {
      bool any = false;
      for (long r = t0; r < t0 + 128 && r < R && !any; ++r) {
        const int b = (int)(r / per), rem = (int)(r % per);
        any = act(kind, b, rem / D2, rem % D2, D1, D2);
      }
      on += any;
    }
    return all ? (double)on / all : 1.0;
  };
  auto key_tiles = [&](const std::vector<float>& m, int b, int L) {
    int last = 0;
    for (int j = 0; j < L; ++j)
      if (m[(size_t)b * L + j] > 0.5f) last = j;
    return last / 64 + 1;
  };
  auto attn = [&](const std::vector<float>& rowm, int R, const std::vector<float>& keym, int L) {
    const int nkt = (L + 63) / 64;
    double on = 0;
    for (int b = 0; b < B; ++b) {
      const int kt = std::min(nkt, key_tiles(keym, b, L));
      for (int r = 0; r < R; ++r)
        if (rowm[(size_t)b * R + r] > 0.5f) on += kt;
    }
    return on / ((double)B * R * nkt);
  };
  pf_evoformer::WorkFrac f;
  f.msa = tiles2d(0, S, N);
  f.msat = tiles2d(1, N, S);
  f.pair = tiles2d(2, N, N);
  f.pair_x = tiles2d(3, N, N);
  f.msat_x = tiles2d(3, N, S);
  f.msa_lin = tiles_lin(0, S, N);
  f.pair_lin = tiles_lin(2, N, N);
  f.attn_row = attn(rho, S, sg, N);
  f.attn_col = attn(sg, N, rho, S);
  f.attn_tri = attn(sg, N, sg, N);
  {
    long on = 0, all = 0, rows = 0;
    double kb = 0;
    const int nkb = (N + 63) / 64;
    for (int b = 0; b < B; ++b) {
      for (int j = 0; j < N; j += 2, ++all) on += sg[(size_t)b * N + j] > 0.5f || (j + 1 < N && sg[(size_t)b * N + j + 1] > 0.5f);
      for (int i = 0; i < N; ++i) rows += sg[(size_t)b * N + i] > 0.5f;
      kb += std::min(nkb, key_tiles(sg, b, N));
    }
    f.opm = (double)on / all;
    f.lnc = (double)rows / ((double)B * N);
    {
      double pr = 0;
      for (int b = 0; b < B; ++b) {
        long cnt = 0;
        for (int i = 0; i < N; ++i) cnt += sg[(size_t)b * N + i] > 0.5f;
        pr += (double)cnt * cnt;
      }
      f.pair_rows = pr / ((double)B * N * N);
    }
    f.tri_k = kb / ((double)B * nkb);
  }
  h->frac = f;
}

bool tc_prepare_flags(pf_evoformer* h, const float* seq_mask, const float* msa_mask, int B, int S, int N, cudaStream_t st) {
  h->frac = pf_evoformer::WorkFrac();
  if (h->prof_on) {
    std::vector<float> sg((size_t)B * N), rho((size_t)B * S);
    if (cudaMemcpyAsync(sg.data(), seq_mask, sg.size() * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemcpyAsync(rho.data(), msa_mask, rho.size() * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
      return false;
    host_work_fractions(h, sg, rho, B, S, N);
  }
  const Arena ar = arena_layout(h->cfg, B, S, N);
  auto fl = [&](size_t off) { return reinterpret_cast<unsigned char*>(h->ws + off); };
  const long M = (long)B * S * N, P = (long)B * N * N;
  h->prof_begin(KK_FLAGS, 0.0, 0.0, st);
  {
    const int yt = g2_pick_yt(N);
    launch_tile_flags(seq_mask, msa_mask, 0, B, S, N, 128 / yt, yt, fl(ar.f_msa), g2_num_tiles(B, S, N), st);
    launch_tile_flags(seq_mask, msa_mask, 2, B, N, N, 128 / yt, yt, fl(ar.f_pair), g2_num_tiles(B, N, N), st);
    launch_tile_flags(seq_mask, msa_mask, 3, B, N, N, 128 / yt, yt, fl(ar.f_pair_x), g2_num_tiles(B, N, N), st);
  }
  {
    const int yt = g2_pick_yt(S);
    launch_tile_flags(seq_mask, msa_mask, 1, B, N, S, 128 / yt, yt, fl(ar.f_msat), g2_num_tiles(B, N, S), st);
    launch_tile_flags(seq_mask, msa_mask, 3, B, N, S, 128 / yt, yt, fl(ar.f_msat_x), g2_num_tiles(B, N, S), st);
  }
  launch_tile_flags(seq_mask, msa_mask, 0, B, S, N, 0, 0, fl(ar.f_msa_lin), (M + 127) / 128, st);
  launch_tile_flags(seq_mask, msa_mask, 2, B, N, N, 0, 0, fl(ar.f_pair_lin), (P + 127) / 128, st);
  launch_key_tiles(seq_mask, B, N, reinterpret_cast<int*>(h->ws + ar.kt_seq), st);
  launch_key_tiles(msa_mask, B, S, reinterpret_cast<int*>(h->ws + ar.kt_msa), st);
  int* kt_seq = reinterpret_cast<int*>(h->ws + ar.kt_seq);
  int* kt_msa = reinterpret_cast<int*>(h->ws + ar.kt_msa);
  int* cnt = reinterpret_cast<int*>(h->ws + ar.rl_count);
  launch_row_list(msa_mask, kt_seq, B, S, h->ws + ar.rl_row, cnt + 0, st);   // row attention: rows (b, s), keys = residues
  launch_row_list(seq_mask, kt_msa, B, N, h->ws + ar.rl_col, cnt + 1, st);   // column attention: rows (b, i), keys = sequences
  launch_row_list(seq_mask, kt_seq, B, N, h->ws + ar.rl_tri, cnt + 2, st);   // triangle attention: rows (b, i), keys = residues
  h->prof_end(st);
  h->launches += 11;   // prof_begin counted one of the twelve
  return cudaGetLastError() == cudaSuccess;
}

// Extra-MSA stack, MSA-side sub-steps 1-4 of one block (5-9 are the main block's pair stack on the inner handle).  The
// residual stream e has c_e = 64 channels; its row attention runs on H x 32 = 256 columns (heads zero-padded 8 -> 32), so all
// intermediates have the main block's shapes and live in the inner handle's arena.
bool tc_run_extra_substep(pf_evoformer* h, const ExtraOff& xo, const ExtraT& xt, const ExtraBlockDev& xb, float* e, float* pair,
                          const float* seq_mask, const float* msa_mask, int B, int S, int N, int block, int step,
                          cudaStream_t st, std::string& err) {
  const pf_config& c = h->cfg;
  if (step >= 5) return tc_run_substep(h, e, pair, seq_mask, msa_mask, B, S, N, block, step, st, err);
  TcDriver d;
  d.h = h; d.st = st; d.B = B; d.S = S; d.N = N;
  d.msa = e; d.pair = pair; d.seq_mask = seq_mask; d.msa_mask = msa_mask;
  d.ar = arena_layout(c, B, S, N);
  d.w = h->w32 + (size_t)block * h->off.total;
  d.w16 = h->w16 + (size_t)block * h->tc.total16;
  d.wf = h->wf + (size_t)block * h->tc.total_f32;
  const int ce = xb.c_e, H = xb.heads, C = 32 * H;
  const double M = (double)B * S * N;
  bool ok = false;
  if (step == 1) {
    TcDriver::AttnPar px{ce, xb.w32 + xo.row.ln_g, xb.w32 + xo.row.ln_b, xb.w16 + xt.row_w_in, xb.wf + xt.row_b_in,
                         xb.w16 + xt.row_wo, xb.w32 + xo.row.bo, 1.0f / sqrtf((float)xb.head_dim)};
    // LN'(z) and the pair-bias projection of this block sit in the inner handle's blob (same shapes as the main block's)
    ok = d.attn_substep(e, C, H, S, N, false, h->off.row, px, seq_mask, true, false, d.ar.f_msa, d.ar.rl_row, 0);
  } else if (step == 2) {
    h->prof_begin(KK_GLOBAL, 2.0 * M * ce * (2.0 * ce + 2.0 * xb.head_dim), M * ce * 12.0, st);
    launch_extra_global_col(e, seq_mask, msa_mask, xb.w32, xo.col, xb.o_glob, B, S, N, ce, H, st);
    h->prof_end(st);
    h->launches += 1;   // two kernels
    ok = true;
  } else if (step == 3) {
    // X.3 unfused: LN(e) W1 + b1 -> relu -> bf16 hidden [M, 4 c_e] in the arena; hidden W2 + b2 reduce-added into e
    const int n4 = c.transition_n * ce;
    bf16* Hb = d.buf<bf16>(d.ar.o);
    TcDriver::G2Desc_ g1 = TcDriver::desc_base(B, S, N, ce, n4);
    g1.src = e; g1.gamma = xb.w32 + xo.msa_trans.ln_g; g1.beta = xb.w32 + xo.msa_trans.ln_b;
    g1.op_fmt = 1; g1.Wt = xb.w16 + xt.tr_w1; g1.bias = xb.w32 + xo.msa_trans.b1;
    g1.row_out[0] = Hb; g1.row_ld[0] = n4;
    int n = 0;
    for (int col = 0; col < n4; col += 64, ++n) {
      g1.ops[n] = TcDriver::op(G2_ROW16, col);
      g1.ops[n].act = ACT_RELU;
    }
    g1.n_ops = n;
    g1.tile_active = d.flags(d.ar.f_msa);
    if (!d.gemm2(g1, M * n4 * 2.0, h->frac.msa)) { err = d.err; return false; }
    TcDriver::G2Desc_ g2 = TcDriver::desc_base(B, S, N, n4, ce);
    g2.a_mode = 1; g2.A = Hb; g2.op_fmt = 0; g2.Wt = xb.w16 + xt.tr_w2; g2.bias = xb.w32 + xo.msa_trans.b2;
    g2.resid = e; g2.resid_ld = ce;
    g2.ops[0] = TcDriver::op(G2_RESID, 0);
    g2.n_ops = 1;
    g2.tile_active = d.flags(d.ar.f_msa);
    ok = d.gemm2(g2, M * ce * 8.0, h->frac.msa);
  } else if (step == 4) {
    const double P = (double)B * N * N, cc = (double)c.c_opm * c.c_opm;
    const int Sp = pad8(S);
    bf16* ABT = d.buf<bf16>(d.ar.vt);
    TcDriver::G2Desc_ g = TcDriver::desc_base(B, N, S, ce, 2 * c.c_opm);
    g.src = e; g.src_transposed = 1; g.gamma = xb.w32 + xo.opm.ln_g; g.beta = xb.w32 + xo.opm.ln_b;
    g.op_fmt = 1; g.Wt = xb.w16 + xt.opm_wab; g.bias = xb.wf + xt.opm_bias_ab;
    g.rowmask = RM_MSA; g.seq_mask = seq_mask; g.msa_mask = msa_mask; g.mask_transposed = 1;
    g.vt_out = ABT; g.vt_cols = 2 * c.c_opm; g.Lpad = Sp;
    g.ops[0] = TcDriver::op(G2_VT, 0, 2 * c.c_opm);
    g.ops[0].fmt = 1;   // fp16 operands of the outer product
    g.ops[0].masked = 1;
    g.n_ops = 1;
    g.tile_active = d.flags(d.ar.f_msat_x);
    if (!d.gemm2(g, M * 2.0 * c.c_opm * 2.0, h->frac.msat_x)) { err = d.err; return false; }
    h->prof_begin(KK_OPM, (2.0 * P * cc * S + 2.0 * P * cc * c.c_z) * h->frac.opm,
                  (2.0 * M * c.c_opm * 2.0 + 8.0 * P * c.c_z) * h->frac.opm, st);
    if (launch_opm_tc(h->tma, ABT, reinterpret_cast<const bf16*>(d.w16 + h->tc.opm_wout), d.w + h->off.opm.bout, seq_mask,
                      msa_mask, pair, B, S, Sp, N, st) != 0) {
      err = std::string("opm_tc: ") + tc_last_error();
      return false;
    }
    h->prof_end(st);
    ok = true;
  } else {
    d.err = "substep not in 1..9";
  }
  if (!ok) err = d.err;
  return ok;
}

bool tc_run_substep(pf_evoformer* h, float* msa, float* pair, const float* seq_mask, const float* msa_mask, int B, int S,
                    int N, int block, int step, cudaStream_t st, std::string& err) {
  const pf_config& c = h->cfg;
  TcDriver d;
  d.h = h; d.st = st; d.B = B; d.S = S; d.N = N;
  d.msa = msa; d.pair = pair; d.seq_mask = seq_mask; d.msa_mask = msa_mask;
  d.ar = arena_layout(c, B, S, N);
  d.w = h->w32 + (size_t)block * h->off.total;
  d.w16 = h->w16 + (size_t)block * h->tc.total16;
  d.wf = h->wf + (size_t)block * h->tc.total_f32;
  bool ok = false;
  switch (step) {
    case 1: ok = d.attn_substep(msa, c.c_m, c.heads_msa, S, N, false, h->off.row, d.main_par(c.c_m, h->off.row, h->tc.row), seq_mask, true, false, d.ar.f_msa,
                                d.ar.rl_row, 0); break;
    case 2: ok = d.attn_substep(msa, c.c_m, c.heads_msa, N, S, true, h->off.col, d.main_par(c.c_m, h->off.col, h->tc.col), msa_mask, false, false, d.ar.f_msat,
                                d.ar.rl_col, 1); break;
    case 3: ok = d.transition_substep(msa, S, N, c.c_m, h->off.msa_trans, h->tc.mt_w1, h->tc.mt_w2, d.ar.f_msa_lin); break;
    case 4: ok = d.opm_substep(); break;
    case 5: ok = d.trimul_substep(false); break;
    case 6: ok = d.trimul_substep(true); break;
    case 7: ok = d.attn_substep(pair, c.c_z, c.heads_pair, N, N, false, h->off.tri_start, d.main_par(c.c_z, h->off.tri_start, h->tc.tri_start), seq_mask, false,
                                true, d.ar.f_pair, d.ar.rl_tri, 2); break;
    case 8: ok = d.attn_substep(pair, c.c_z, c.heads_pair, N, N, true, h->off.tri_end, d.main_par(c.c_z, h->off.tri_end, h->tc.tri_end), seq_mask, false,
                                true, d.ar.f_pair, d.ar.rl_tri, 2); break;
    case 9: ok = d.transition_substep(pair, N, N, c.c_z, h->off.pair_trans, h->tc.pt_w1, h->tc.pt_w2, d.ar.f_pair_lin); break;
    default: d.err = "substep not in 1..9";
  }
  if (!ok) err = d.err;
  return ok;
}

}  // namespace pf
