// The handle behind pf_evoformer_t, the weight-blob offsets and the device weight layout of the
// tensor-core path.  Shared by pf_api.cu (C ABI, fp32 SIMT driver) and pf_trunk_tc.cu (tcgen05 driver).
#pragma once
#include "../../include/pf_evoformer.h"
#include "pf_internal.h"

#include <string>
#include <vector>

namespace pf {

// ---- offsets (floats, within one block) into the fp32 blob, Appendix B order ----
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
BlockW block_offsets(const pf_config& c);

// ---- tensor-core weight set: 16-bit matrices [Nout, K] (K contiguous), offsets in 16-bit elements within one block.
// Matrices that multiply a LayerNorm output are stored as fp16 (reading R17: the values are the bf16-rounded
// weights of R15, which fp16 represents exactly when 2^-14 <= |w| <= 65504; F16Range counts the entries outside), all
// others as bf16.  Fused bias vectors are fp32 (offsets in floats).
struct F16Range {
  size_t overflow = 0;       // |w| > 65504 or NaN: refused by create
  size_t below_normal = 0;   // 0 < |w| < 2^-14: stored with fewer mantissa bits or flushed to zero
};
struct AttnT {
  size_t w_in;   // fp16 [4C (+H), C]: q | k | gate | v (| pair-bias heads for triangle attention)
  size_t b_in;   // fp32 [4C (+H)]: gate bias in its column range, zero elsewhere
  size_t wo;     // bf16 [C, C]
};
struct TcBlock {
  AttnT row, col, tri_start, tri_end;
  size_t row_wbias;                      // fp16 [H_m, c_z]  (LN'(z) -> pair bias of row attention)
  size_t mt_w1, mt_w2, pt_w1, pt_w2;     // transitions: W1 fp16 [4C, C], W2 bf16 [C, 4C]
  size_t opm_wab, opm_bias_ab, opm_wout; // fp16 [2 c_opm, c_m], fp32 [2 c_opm], bf16 [c_z, c_opm^2]
  // triangle multiplication: fp16 [5 c_t, c_z] = [p | gate] of the operand written to the first einsum buffer,
  // [p | gate] of the second, then the output gate g; fp32 bias [5 c_t] in the same order; W_z fp16 [c_z, c_t]
  size_t to_w, to_b, to_wz, ti_w, ti_b, ti_wz;
  size_t total16, total_f32;
};
TcBlock tc_layout(const pf_config& c);
void build_tc_block(const pf_config& c, const BlockW& off, const TcBlock& t, const float* w, std::vector<uint16_t>& w16,
                    size_t base16, std::vector<float>& wf, size_t basef, F16Range* range);

enum KernelKind { KK_LN = 0, KK_GEMM, KK_ATTN, KK_TRI, KK_LNC, KK_OPM, KK_LNGEMM, KK_TRANS, KK_FLAGS, KK_GLOBAL, KK_EMBED, KK_HEADS, KK_OPMAB, KK_COUNT };

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline int pad8(int v) { return (v + 7) / 8 * 8; }

struct Arena {
  size_t x, qkg, vt, o, bias, acm, bcm, g, tcm, tn, oa, ob;
  // mask-derived work flags (pf_flags.cu): active-tile bytes per row geometry, key-tile counts per protein
  size_t f_msa, f_msat, f_pair, f_msa_lin, f_pair_lin, f_pair_x, f_msat_x, kt_seq, kt_msa;
  // compacted attention row lists {row, key tiles} + their lengths: row attention (b,s), column attention (b,i), triangle (b,i)
  size_t rl_row, rl_col, rl_tri, rl_count;
  size_t total;
};
Arena arena_layout(const pf_config& c, int B, int S, int N);

}  // namespace pf

struct pf_evoformer {
  pf_config cfg;
  pf::BlockW off;
  pf::TcBlock tc;
  float* w32 = nullptr;      // device fp32 blob
  uint16_t* w16 = nullptr;   // device 16-bit transposed matrices (PF_BF16 only)
  float* wf = nullptr;       // device fused fp32 bias vectors (PF_BF16 only)
  char* ws = nullptr;        // workspace arena
  size_t ws_bytes = 0;
  size_t f16_below_normal = 0;   // weights stored as fp16 with |w| < 2^-14 (precision loss, pf_evoformer.h value-range note)
  int device = -1;           // the device the handle was created on (weights, workspace and kernel attributes live there)
  int ws_B = 0, ws_S = 0, ws_N = 0;   // shape of the arena layout the workspace currently holds (zero-filled when it changes)
  // CUDA graphs of whole forward calls on launch-bound shapes (pf_api.cu, dispatch_pass)
  struct GraphEntry { float* msa; float* pair; const float* sm; const float* mm; int B, S, N, block0, block1; cudaGraphExec_t exec; long long launches; };
  std::vector<GraphEntry> graphs;
  cudaStream_t cap_stream = nullptr;
  char* stage = nullptr;     // forward_host staging
  size_t stage_bytes = 0;
  // forward_host pipelines the batch in chunks of proteins: copy-in stream, the caller's stream for compute, copy-out stream
  cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
  cudaEvent_t host_ev[2 * 16 + 1] = {};   // per chunk (at most 16): inputs landed [c], compute done [16 + c]; [32]: call start
  int num_sms = 148;
  long long launches = 0;
  pf::TmaCtx* tma = nullptr;
  // per-launch CUDA-event profiling (pf_evoformer_set_profiling)
  bool prof_on = false;
  struct ProfRec { int kind; cudaEvent_t e0, e1; double flops, bytes; };
  std::vector<ProfRec> prof;
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_used = 0;
  // Fractions of the nominal (padded) work the mask-derived skipping leaves, computed on the host from the masks while
  // profiling is on, so that the per-launch FLOP / byte tags count executed work only.  1.0 when not profiling.
  struct WorkFrac {
    double msa = 1, msat = 1, pair = 1, msa_lin = 1, pair_lin = 1, pair_x = 1, msat_x = 1;   // active 128-row tiles per geometry
    double attn_row = 1, attn_col = 1, attn_tri = 1;                 // visited (row, key tile) pairs
    double opm = 1, tri_k = 1, lnc = 1;                              // active j pairs, visited k-blocks, unpadded rows i
    double pair_rows = 1;                                            // unmasked (i, j) pairs (pair-bias heads kernel)
  } frac;
  cudaEvent_t next_event() {
    if (ev_used == ev_pool.size()) {
      cudaEvent_t e;
      cudaEventCreate(&e);
      ev_pool.push_back(e);
    }
    return ev_pool[ev_used++];
  }
  // one kernel launch: counts it and, when profiling, brackets it with events on the launch stream
  void prof_begin(int kind, double flops, double bytes, cudaStream_t st) {
    launches++;
    if (!prof_on) return;
    ProfRec r{kind, next_event(), next_event(), flops, bytes};
    cudaEventRecord(r.e0, st);
    prof.push_back(r);
  }
  void prof_end(cudaStream_t st) {
    if (prof_on) cudaEventRecord(prof.back().e1, st);
  }
};

namespace pf {
// ---- extra-MSA stack (pf_extra.cu, readings X.1-X.9) ----
// offsets (floats) within one extra-MSA block of its fp32 blob (the order of pf_synth.extra_block_spec)
struct GlobalColW {
  size_t ln_g, ln_b, wq, wk, wv, wg, bg, wo, bo;
};
struct ExtraOff {
  AttnW row;                 // c = c_e, with LN'(z) and the pair-bias projection
  GlobalColW col;
  TransW msa_trans;
  OpmW opm;
  TriMulW tri_out, tri_in;
  AttnW tri_start, tri_end;
  TransW pair_trans;
  size_t total;
};
// prepared device matrices of the MSA-side modules of one extra block: 16-bit offsets / fp32 offsets
struct ExtraT {
  size_t row_w_in;           // fp16 [4 * 32 H, c_e]: q | k | gate | v with every head zero-padded from c_e / H to 32 rows
  size_t row_wo;             // bf16 [c_e, 32 H]
  size_t tr_w1, tr_w2;       // fp16 [4 c_e, c_e], bf16 [c_e, 4 c_e]
  size_t opm_wab;            // fp16 [2 c_opm, c_e]
  size_t total16;
  size_t row_b_in;           // fp32 [4 * 32 H]: gate bias in its (padded) column range
  size_t opm_bias_ab;        // fp32 [2 c_opm]
  size_t total_f32;
};
struct ExtraBlockDev {
  const float* w32;          // fp32 blob of this extra block (LayerNorm parameters, biases, the global attention's matrices)
  const uint16_t* w16;
  const float* wf;
  float* o_glob;             // [B, N, c_e] scratch of the global column attention
  int c_e, heads, head_dim;
};
void launch_extra_global_col(float* e, const float* seq_mask, const float* msa_mask, const float* w32, const GlobalColW& o,
                             float* o_glob, int B, int S, int N, int c_e, int heads, cudaStream_t st);
bool tc_run_extra_substep(pf_evoformer* inner, const ExtraOff& xo, const ExtraT& xt, const ExtraBlockDev& xb, float* e,
                          float* pair, const float* seq_mask, const float* msa_mask, int B, int S, int N, int block, int step,
                          cudaStream_t st, std::string& err);
// workspace of `h` for (B, S, N): grown and, when the shape changed, zero-filled in stream order (pf_api.cu)
bool ensure_workspace(pf_evoformer* h, int B, int S, int N, cudaStream_t st, std::string& err);

// tcgen05 path: one sub-step (1..9) of block `block`; returns false and sets err on failure.
// mask-derived work flags for one forward call (launched once, before the first block)
bool tc_prepare_flags(pf_evoformer* h, const float* seq_mask, const float* msa_mask, int B, int S, int N, cudaStream_t st);
bool tc_run_substep(pf_evoformer* h, float* msa, float* pair, const float* seq_mask, const float* msa_mask, int B, int S,
                    int N, int block, int step, cudaStream_t st, std::string& err);
}  // namespace pf
