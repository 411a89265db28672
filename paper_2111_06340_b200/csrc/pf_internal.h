// Internal declarations shared by the kernels and the C-ABI driver (not installed; include/pf_evoformer.h is the ABI).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
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
void launch_lnc(const float* t_cm, T* y, const float* gamma, const float* beta, int B, int C, int N, int Npad,
                cudaStream_t st);
template <typename T>
void launch_opm_simt(const T* a, const T* b, const float* wout, const float* bout, const float* seq_mask,
                     const float* msa_mask, float* z, int B, int S, int N, int c_opm, int c_z, cudaStream_t st);

// ---- tcgen05 kernels (bf16), pf_gemm_tc.cu / pf_attn_tc.cu ----
// Weights Wt are bf16 [Nout, K] (K contiguous).  DUAL: Wt is [2*Nout_eff, K] = [Wp ; Wg] stacked per 128 columns.
struct TmaCtx;   // holds the driver entry point for cuTensorMapEncodeTiled
TmaCtx* tma_ctx_create();
void tma_ctx_destroy(TmaCtx*);
const char* tc_last_error();
void tc_set_error(const std::string& s);
int launch_gemm_tc(TmaCtx* ctx, const bf16* A, int lda, const bf16* Wt, long R, int K, int Nout, const Epi& epi,
                   int num_sms, cudaStream_t st);
int launch_attn_tc(TmaCtx* ctx, const bf16* qkg, const bf16* vt, const bf16* bias, const float* keymask, bf16* o,
                   int B, int R, int L, int Lpad, int H, int num_sms, cudaStream_t st);
// ab_t: [(b,i), 64 channels (a | b), Spad] bf16 masked projections; wout_t: [c_z, c_opm*c_opm] bf16
int launch_opm_tc(TmaCtx* ctx, const bf16* ab_t, const bf16* wout_t, const float* bout, const float* seq_mask,
                  const float* msa_mask, float* z, int B, int S, int Spad, int N, cudaStream_t st);
int launch_tri_einsum_tc(TmaCtx* ctx, const bf16* a_cm, const bf16* b_cm, float* t_cm, int batch, int N, int Npad,
                         int num_sms, cudaStream_t st);

}  // namespace pf
