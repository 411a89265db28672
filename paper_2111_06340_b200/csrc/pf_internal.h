// Internal declarations shared by the kernels and the C-ABI driver (not installed; include/pf_evoformer.h is the ABI).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <string>

typedef __nv_bfloat16 bf16;

namespace pf {

enum Act { ACT_NONE = 0, ACT_SIGMOID = 1, ACT_RELU = 2 };
enum RowMaskKind { RM_NONE = 0, RM_MSA = 1, RM_PAIR = 2 };
enum EpiKind { EPI_STORE = 0, EPI_GATED_CM = 1, EPI_RESID = 2, EPI_HEADS = 3 };

// Rows of a [B, D1, D2, C] activation: r = (b*D1 + x)*D2 + y.
struct RowGeom {
  int B, D1, D2;
};

// Epilogue of a projection GEMM  acc[r, n] = sum_k A[r,k] W[k,n]   (shared by the SIMT and tcgen05 kernels).
struct Epi {
  int kind;
  // EPI_STORE: v = acc * (n < scale_cols ? scale : 1) + bias[n]; act on n in [act_lo, act_hi); * rowmask(r);
  //            n < vt_from : out[r*ldo + n] ; n >= vt_from : vt[((r / D2)*(Nout-vt_from) + (n-vt_from))*Lpad + (r % D2)]
  int act, act_lo, act_hi;
  float scale;
  int scale_cols;
  const float* bias;    // [Nout] or null
  void* out;            // T*
  int ldo;
  int vt_from;          // >= Nout: no transposed columns
  void* vt;             // T*
  int Lpad;
  int rowmask;          // RowMaskKind
  const float* seq_mask;   // [B, N]
  const float* msa_mask;   // [B, S]
  RowGeom geom;
  int mask_transposed;  // RM_MSA only: rows are (b, i, s) instead of (b, s, i)
  // EPI_GATED_CM: v = pi(r) * sigmoid(acc2 + bias2[n]) * (acc + bias[n]) -> cm[((b*Nout + n)*D1 + x)*Lpad + y]
  const float* bias2;
  // EPI_RESID: resid[dst(r)*ldr + n] += (acc + bias[n]) * (gate ? gate[r*ldg + n] : 1); dst(r) = transposed ? (b, y, x) : r
  float* resid;
  int ldr;
  const void* gate;     // T*
  int ldg;
  int transposed;
  // EPI_HEADS: out[((b*Nout + n)*D1 + x)*Lpad + y] = acc * scale      (pair bias, [B, H, L, Lpad])
};

// ---- SIMT kernels (templated on the storage type T = float | bf16), pf_simt.cu ----
template <typename T>
void launch_ln_rows(const float* x, T* y, const float* gamma, const float* beta, long rows, int C,
                    RowGeom geom, int transposed, cudaStream_t st);
template <typename T>
void launch_gemm_simt(const T* A, int lda, const float* W, const float* W2, int ldw, long R, int K, int Nout,
                      const Epi& epi, cudaStream_t st);
template <typename T>
void launch_attn_simt(const T* qkg, const T* vt, const T* bias, const float* keymask, T* o, int B, int R, int L,
                      int Lpad, int H, cudaStream_t st);
template <typename T>
void launch_tri_einsum_simt(const T* a_cm, const T* b_cm, float* t_cm, int batch, int N, int Npad, cudaStream_t st);
template <typename T>
void launch_lnc(const float* t_cm, T* y, const float* gamma, const float* beta, const float* seq_mask /*optional: rows of
                padded residues are skipped*/, int B, int C, int N, int Npad, cudaStream_t st);
// pair-bias heads of the MSA row attention at c_z = 128, H <= 8 (pf_simt.cu): bias[b,h,i,j] = scale Lin0(LN'(z_ij))_h, W [128, H] fp32
void launch_ln_heads128(const float* z, const float* gamma, const float* beta, const float* W, float scale, const float* seq_mask,
                        bf16* out, int B, int N, int Lpad, int H, int num_sms, cudaStream_t st);
// outer-product-mean operands at c_m = 256, c_opm = 32 (pf_simt.cu): ab_t[(b,i), 64, Spad] = mu (LN(m) [W_a | W_b] + [b_a | b_b]), fp32 weights [256, 32]
void launch_ln_opm_ab256(const float* msa, const float* gamma, const float* beta, const float* Wa, const float* Wb, const float* ba,
                         const float* bb, const float* seq_mask, const float* msa_mask, bf16* out, int B, int S, int N, int Spad,
                         int num_sms, cudaStream_t st);
void launch_lnc_tc(const bf16* t_cm, __half* y, const float* gamma, const float* beta, const float* seq_mask, int B, int N,
                   int Npad, cudaStream_t st);
template <typename T>
void launch_opm_simt(const T* a, const T* b, const float* wout, const float* bout, const float* seq_mask,
                     const float* msa_mask, float* z, int B, int S, int N, int c_opm, int c_z, cudaStream_t st);

// ---- tcgen05 kernels (pf_tma.cu: TMA host side; pf_lngemm_tc.cu, pf_trans_tc.cu, pf_attn_tc.cu, pf_opm_tc.cu, pf_tri_tc.cu) ----
// Weights Wt are 16-bit [Nout, K] (K contiguous).
struct TmaCtx;   // holds the driver entry point for cuTensorMapEncodeTiled
TmaCtx* tma_ctx_create();
void tma_ctx_destroy(TmaCtx*);
// kernel attributes (dynamic shared memory sizes) for the CURRENT device; called by pf_evoformer_create, so a handle's kernels
// are configured on the handle's own device (no process-wide "configured" flags)
bool configure_gemm2_kernels();
bool configure_transition_kernels();
bool configure_attn_kernel();
bool configure_opm_kernel();
bool configure_tri_kernel();
const char* tc_last_error();
void tc_set_error(const std::string& s);
// ---- persistent LN-fused projection GEMM (pf_lngemm_tc.cu) ----
// Rows of the GEMM are (b, x in [0,D1), y in [0,D2)); one CTA tile = XT consecutive x times YT consecutive y (XT*YT = 128).
// The 64-column groups of the output are described by G2Op: what is done to the accumulator and where it goes.
// G2_VTS: like G2_VT, but the half-window it belongs to is computed with the operand roles SWAPPED (weights as the M side,
// the LayerNorm tile as the N side), so the accumulator already holds the transposed tile: TMEM lane = output column,
// TMEM column = tile row.  Group j of a window covers half j / 2 and tile rows [64 (j % 2), +64); needs YT >= 64.
// G2_CMS: G2_CM_DUAL on a window whose two halves (p | gate) are both operand-swapped: lane = channel, the group j (0 or 1)
// covers tile rows [64 j, +64); the row masks of the tile come from a small shared-memory table.
enum G2Kind { G2_SKIP = 0, G2_ROW16 = 1, G2_CM_DUAL = 2, G2_HEADS = 3, G2_VT = 4, G2_RESID = 5, G2_VTS = 6, G2_CMS = 7 };
struct G2Op {
  int kind;      // G2Kind
  int act;       // Act, applied after scale and bias (ROW16)
  int fmt;       // ROW16: 0 = bf16, 1 = fp16 output
  int map;       // ROW16: row_out index; CM_DUAL: cm_out index
  int dst_col;   // first destination column / channel / head
  int ncols;     // valid columns of this group (<= 64)
  float scale;   // ROW16 / HEADS: multiplies the accumulator before the bias
  int masked;    // VT: multiply by the row mask
};
constexpr int G2_MAX_OPS = 20;
// tile height along y for a [B, D1, D2] row grid: the power of two in [8, 128] that wastes the fewest rows (ties: largest)
inline int g2_pick_yt(int D2) {
  int best = 128;
  double best_eff = -1.0;
  for (int yt = 128; yt >= 8; yt >>= 1) {
    int tiles = (D2 + yt - 1) / yt;
    double eff = (double)D2 / ((double)tiles * yt);
    if (eff > best_eff + 1e-9) {
      best_eff = eff;
      best = yt;
    }
  }
  return best;
}
inline long g2_num_tiles(int B, int D1, int D2) {
  const int yt = g2_pick_yt(D2), xt = 128 / yt;
  return (long)B * ((D1 + xt - 1) / xt) * ((D2 + yt - 1) / yt);
}
struct G2Desc {
  int B, D1, D2;            // row geometry
  int K, Nw;                // K in {128, 256}; Nw = rows of Wt (GEMM columns including gate partners)
  int a_mode;               // 0: A = LayerNorm of fp32 rows gathered from src; 1: A = 16-bit [R, K] in GEMM row order (TMA)
  const float* src;         // a_mode 0: [B, D1, D2, K] fp32, or [B, D2, D1, K] when src_transposed
  int src_transposed;
  const float* gamma;
  const float* beta;
  const void* A;            // a_mode 1
  int op_fmt;               // MMA operand format: 0 bf16, 1 fp16 (A and Wt alike)
  const void* Wt;           // [Nw, K] 16-bit, K contiguous
  const float* bias;        // [Nw] fp32 or null
  int bias_lo, bias_n;      // columns [bias_lo, bias_lo + bias_n) may be non-zero (bias_n = 0: [bias_lo, Nw)); multiples of 64,
                            // at most 256 (K = 256) / 768 (K = 128) columns: the kernel keeps this range in shared memory
  int rowmask;              // RowMaskKind, applied by CM_DUAL and masked VT groups
  const float* seq_mask;
  const float* msa_mask;
  int mask_transposed;
  void* row_out[2];         // ROW16 destinations [R, row_ld] 16-bit in GEMM row order
  int row_ld[2];
  float* resid;             // RESID destination: [B, D1, D2, resid_ld], or [B, D2, D1, resid_ld] when resid_transposed
  int resid_ld;
  int resid_transposed;
  const void* gate;         // RESID: optional fp16 gate [R, ldg] in GEMM row order
  int ldg;
  void* cm_out[2];          // CM_DUAL: bf16 [(b, channel), D1, Lpad]
  int cm_channels;
  void* heads_out;          // HEADS: bf16 [b, n_heads, D1, Lpad]
  int n_heads;
  void* vt_out;             // VT: bf16 [((b, x), vt_cols), Lpad]
  int vt_cols;
  int Lpad;
  G2Op ops[G2_MAX_OPS];
  int n_ops;
  unsigned swap_mask;       // bit (2 nt + h): the 128 columns of half h of window nt are computed operand-swapped (G2_VTS groups)
  const unsigned char* tile_active;   // optional [num_tiles]: 0 = every row of the tile is masked, skip it (pf_flags.cu)
};
int launch_gemm2(TmaCtx* ctx, const G2Desc& d, int num_sms, cudaStream_t st);
// fused transition (pf_trans_tc.cu): res[R, C] += relu(LN(res) W1 + b1) W2 + b2; w1t fp16 [4C, C], w2t bf16 [C, 4C]
int launch_transition_tc(TmaCtx* ctx, float* res, long R, int C, const float* gamma, const float* beta, const void* w1t,
                         const float* b1, const void* w2t, const float* b2, const unsigned char* tile_active, int num_sms,
                         cudaStream_t st);
// rows: device list of int2 {b*R + r, key tiles to visit} of the rows to process, *n_rows its length (pf_flags.cu
// launch_row_list): rows all of whose queries are masked are not in it, key tiles past the last unmasked key are not visited
int launch_attn_tc(TmaCtx* ctx, const bf16* qkg, const bf16* vt, const bf16* bias, const float* keymask, bf16* o,
                   int B, int R, int L, int Lpad, int H, const void* rows, const int* n_rows, int num_sms, cudaStream_t st);
void launch_row_list(const float* rowmask, const int* key_tiles, int B, int R, void* rows, int* n_rows, cudaStream_t st);
// pf_flags.cu
void launch_tile_flags(const float* seq_mask, const float* msa_mask, int kind, int B, int D1, int D2, int XT, int YT,
                       unsigned char* flags, long num_tiles, cudaStream_t st);
void launch_key_tiles(const float* mask, int B, int L, int* key_tiles, cudaStream_t st);
// ab_t: [(b,i), 64 channels (a | b), Spad] bf16 masked projections; wout_t: [c_z, c_opm*c_opm] bf16
int launch_opm_tc(TmaCtx* ctx, const bf16* ab_t, const bf16* wout_t, const float* bout, const float* seq_mask,
                  const float* msa_mask, float* z, int B, int S, int Spad, int N, cudaStream_t st);
// key_tiles [batch / channels] (optional): the contraction stops after the last unmasked residue's 64-wide k-block
int launch_tri_einsum_tc(TmaCtx* ctx, const bf16* a_cm, const bf16* b_cm, bf16* t_cm, int batch, int N, int Npad,
                         const int* key_tiles, int channels, int num_sms, cudaStream_t st);

}  // namespace pf
