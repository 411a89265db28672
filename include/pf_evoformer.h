/*
 * pf_evoformer.h — C ABI of the B200-native Evoformer trunk (the GPU stage ParaFold separates out).
 *
 * What is computed: the forward pass of AlphaFold's Evoformer trunk (named at PAPER.md:27 and
 * PAPER.md:61; AlphaFold v2.0.1 monomer), n_blocks blocks of the nine sub-steps of
 * SURVEY.md Appendix A.1-A.9, over a batch of proteins padded to one length bucket (PAPER.md:113:
 * proteins of similar length share one compiled model; here: one binary, runtime shapes).
 * BASELINE.json:north_star defines the two entry points (create / forward) and the scheduler.
 *
 * Conventions
 *   - Plain C, no torch types.  "dev" = CUDA device pointer on the current device, "host" = host pointer.
 *   - All tensors row-major, channels last.  B = batch, S = N_seq, N = N_res (padded bucket length).
 *   - Residual streams msa / pair are fp32 in HBM on both compute paths and are
 *     updated IN PLACE.
 *   - Masks are fp32 0/1: seq_mask[B,N], msa_mask[B,S] (R2).  Precondition: msa_mask[b,0]=1 and every
 *     protein has at least one unmasked residue.  Outputs at masked positions are unspecified but finite (R3).
 *   - Every call returns a pf_status; nothing throws or aborts across the ABI.  pf_last_error() gives a
 *     thread-local message for the last non-OK status.
 *   - A handle is not thread-safe; use one handle per stream.
 */
#ifndef PF_EVOFORMER_H_
#define PF_EVOFORMER_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pf_evoformer pf_evoformer_t;   /* opaque; owns device weights and a grow-only workspace */

typedef enum {
  PF_OK = 0,
  PF_ERR_INVALID_ARG = 1,
  PF_ERR_SHAPE = 2,
  PF_ERR_ALLOC = 3,
  PF_ERR_CUDA = 4,
  PF_ERR_ARCH = 5,            /* device is not compute capability 10.x */
  PF_ERR_UNIMPLEMENTED = 6
} pf_status;

typedef enum {
  PF_F32 = 0,        /* fp32 SIMT arithmetic everywhere (cfg1; tolerance max-abs 1e-4) */
  PF_BF16 = 1        /* 16-bit operands (bf16; fp16 for LayerNorm outputs, their weights and gates), fp32 accumulation on
                        tcgen05 tensor cores, fp32 residual streams */
} pf_dtype;

typedef struct {
  int c_m;            /* MSA channels (256) */
  int c_z;            /* pair channels (128) */
  int heads_msa;      /* 8  (heads_msa  * head_dim == c_m) */
  int heads_pair;     /* 4  (heads_pair * head_dim == c_z) */
  int head_dim;       /* must be 32 */
  int c_opm;          /* outer-product-mean hidden (32) */
  int c_tri;          /* triangle-multiplication hidden (128) */
  int transition_n;   /* transition expansion factor (4) */
  int n_blocks_max;   /* number of blocks whose weights the blob holds */
  pf_dtype dtype;
} pf_config;

/* Number of fp32 values one block occupies in the weights blob (SURVEY.md Appendix B layout,
 * every matrix row-major [in, out]); 1,829,952 for the AlphaFold dims. */
size_t pf_evoformer_block_floats(const pf_config* cfg);

/* Create a trunk.  weights_host: host fp32 blob of cfg->n_blocks_max blocks in Appendix-B order,
 * n_weight_floats its length (checked).  The blob is copied / converted to the device; the caller may
 * free it afterwards.  Errors: INVALID_ARG (null), SHAPE (bad dims, head_dim != 32, wrong blob length),
 * ARCH (not CC 10.x), ALLOC, CUDA.  (= north_star pf_evoformer_create(weights, c_m, c_z, heads).) */
pf_status pf_evoformer_create(pf_evoformer_t** out, const float* weights_host, size_t n_weight_floats,
                              const pf_config* cfg);

/* Run blocks [0, n_blocks) on dev msa[B,S,N,c_m] and dev pair[B,N,N,c_z] in place, asynchronously on
 * cuda_stream (a cudaStream_t, NULL = default stream).  Does not synchronise; reports launch-time errors.
 * Shapes are runtime arguments: a new (B,S,N) costs a workspace growth at most, never a rebuild.
 * Sub-step order inside a block: 1 row attention with pair bias (A.1), 2 column attention
 * (A.2), 3 MSA transition (A.3), 4 outer-product-mean (A.4, reads the updated msa), 5/6 triangle
 * multiplication outgoing/incoming (A.5/A.6), 7/8 triangle attention starting/ending node (A.7/A.8),
 * 9 pair transition (A.9).
 * Limits (PF_ERR_SHAPE / PF_ERR_CUDA with a message otherwise): S <= 65535 and N <= 65535; on the PF_BF16 path also
 * N <= 1024 and S <= 1024 (keys per attention row) and S <= 512 (outer-product-mean contraction length).  B is not
 * limited: batches beyond what one launch sequence takes (grid limits) are cut into chunks of proteins internally.
 * The current CUDA device must be the one the handle was created on (PF_ERR_INVALID_ARG otherwise).
 * Value range on the PF_BF16 path (reading R17): LayerNorm outputs, sigmoid gates, the weight matrices that
 * multiply a LayerNorm output, the pair bias, the gated triangle operands and their einsum (sums over N_res of products of
 * order one), the outer-product operands, the outer product (sums over N_seq) and W_out are held as fp16; q, k, v, the
 * attention probabilities, o and the transition hidden activation as bf16.  Precondition: those weights (after bf16 rounding, R15) lie in the fp16
 * normal range, 2^-14 <= |w| <= 65504 or w == 0 (smaller magnitudes lose bits or flush to zero), and LayerNorm outputs
 * gamma * xhat + beta stay below 65504 in magnitude (|xhat| <= sqrt(C)).  create() counts weights outside that range and
 * refuses blobs with overflowing ones (PF_ERR_SHAPE); the seeded R8 init has about 0.08 % of entries below 2^-14 (a
 * relative perturbation of those entries only, far below the bf16 tolerances).
 * Masked work: on the PF_BF16 path 128-row tiles, attention rows and key tiles whose outputs all lie at masked positions are
 * skipped (outputs there are unspecified but finite, as stated above); unmasked outputs do not depend on what the masked
 * positions of msa / pair contain.
 * Launch-bound shapes (PF_BF16, B * S * N <= 131072, n_blocks >= 2, profiling off): the launch sequence of the call is captured
 * into a CUDA graph the first time it is seen for these buffer addresses and this shape, and replayed on cuda_stream afterwards
 * (the mask-derived flags are computed inside the graph, so mask CONTENTS may change between calls).  At most 16 graphs are
 * kept per handle; a workspace growth drops them.  Environment variable PF_GRAPH=0 turns this off, PF_GRAPH=2 forces it for
 * every shape. */
pf_status pf_evoformer_forward(pf_evoformer_t* h, float* msa_dev, float* pair_dev,
                               const float* seq_mask_dev, const float* msa_mask_dev,
                               int B, int S, int N, int n_blocks, void* cuda_stream);

/* Test hook: run only sub-step `substep` (1..9) of block `block`. */
pf_status pf_evoformer_forward_substep(pf_evoformer_t* h, float* msa_dev, float* pair_dev,
                                       const float* seq_mask_dev, const float* msa_mask_dev,
                                       int B, int S, int N, int block, int substep, void* cuda_stream);

/* End-to-end convenience: the same computation with HOST buffers (pinned or pageable).  The batch is pipelined in
 * chunks of proteins: host->device copies on an internal copy stream, forward on cuda_stream, device->host copies on a
 * second internal copy stream (ordered after earlier work on cuda_stream); returns after everything has completed.
 * Chunk plan for B >= 16: B/16, seven chunks of ~B/8, B/16 proteins (B < 16: up to eight equal chunks); the environment
 * variable PF_HOST_CHUNKS=a,b,c,... (at most 16 positive sizes adding up to B, otherwise ignored) overrides it.
 * Device staging buffers and the copy streams are owned by the handle (grow-only). */
pf_status pf_evoformer_forward_host(pf_evoformer_t* h, float* msa_host, float* pair_host,
                                    const float* seq_mask_host, const float* msa_mask_host,
                                    int B, int S, int N, int n_blocks, void* cuda_stream);

/* Bytes of device workspace forward() needs for (B,S,N) (excluding msa/pair themselves and weights). */
size_t pf_evoformer_workspace_bytes(const pf_evoformer_t* h, int B, int S, int N);

/* Number of kernel launches the last forward()/forward_substep() call on this handle issued. */
long long pf_evoformer_last_launch_count(const pf_evoformer_t* h);

/* Per-launch timing (measurement aid).  While enabled, every kernel launch of forward() is
 * bracketed by two CUDA events on the launch stream and tagged with its kernel kind and its algorithmic FLOPs
 * (2*MAC of the contraction) and algorithmic HBM bytes (operands read once + results written once).
 * set_profiling(h, 1) clears earlier records and starts recording; set_profiling(h, 0) stops and clears.
 * get_profile synchronises on the recorded events and returns, for one kind in [0, pf_evoformer_profile_kinds()),
 * the totals since profiling was enabled: launches, device milliseconds, FLOPs, bytes. */
pf_status pf_evoformer_set_profiling(pf_evoformer_t* h, int enable);
int pf_evoformer_profile_kinds(void);
const char* pf_evoformer_profile_name(int kind);
pf_status pf_evoformer_get_profile(pf_evoformer_t* h, int kind, long long* launches, double* ms, double* flops,
                                   double* bytes);
/* The same records one by one, in launch order: record `index` in [0, pf_evoformer_profile_records(h)) -> its kind, device
 * milliseconds, FLOP and byte tags.  Errors: INVALID_ARG (null, index out of range), CUDA (event query failed). */
long long pf_evoformer_profile_records(const pf_evoformer_t* h);
pf_status pf_evoformer_get_profile_record(pf_evoformer_t* h, long long index, int* kind, double* ms, double* flops,
                                          double* bytes);

void pf_evoformer_destroy(pf_evoformer_t* h);

const char* pf_last_error(void);

/* ------------------------------------------------------------------------------------------------
 * Input / recycling embedders and the recycled trunk.  ParaFold's GPU stage reads the features its CPU
 * stage wrote and runs the network with "three recycling procedures" ("recycling",
 * PAPER.md:61).  PAPER.md prints no formula; the readings E.1-E.3 are:
 *   E.1 input embedder      z_ij = Lin_a(tf_i) + Lin_b(tf_j) + Lin_rel(onehot(clip(r_i - r_j, -R, R) + R))
 *                           m_si = Lin_m(msa_feat_si) + Lin_t(tf_i)
 *   E.2 recycling embedder  z_ij += LN_z(zprev_ij) + Lin_d(onehot_bins(|xprev_i - xprev_j|)),  m_0i += LN_m(mprev_0i)
 *                           (n_dist_bins lower edges evenly spaced from first_break to last_break; the last bin is open)
 *   E.3 recycled trunk      n_cycles x (E.1, E.2 with the previous cycle's trunk output — zeros in the first cycle —, trunk)
 * All arithmetic is fp32.  In pf_evoformer_forward_recycled xprev (previous positions, Angstrom) is an input held constant over
 * the cycles; NULL = no previous structure (no bin is set).  pf_fold_forward (further down) feeds it from the structure module.
 * ---------------------------------------------------------------------------------------------- */
typedef struct pf_embedder pf_embedder_t;   /* opaque; owns device weights and a small grow-only workspace */
typedef struct pf_extra_msa pf_extra_msa_t; /* the extra-MSA stack, declared further down */
typedef struct {
  int c_m;            /* MSA channels (256) */
  int c_z;            /* pair channels (128) */
  int tf_dim;         /* target features per residue (22) */
  int msa_dim;        /* MSA features per (sequence, residue) (49; at most 64) */
  int max_relpos;     /* R: relative positions are clipped to [-R, R] (32) */
  int n_dist_bins;    /* distance bins of the recycled positions (15) */
  float first_break;  /* lower edge of the first bin, Angstrom (3.25) */
  float last_break;   /* lower edge of the last bin (20.75) */
  int extra_dim;      /* extra-MSA features per (sequence, residue) (25; at most 32) */
  int c_e;            /* extra-MSA channels (64) */
} pf_embed_config;

/* fp32 values in the embedder weights blob, in this order, every matrix row-major [in, out]:
 * W_a[tf_dim,c_z] b_a | W_b b_b | W_rel[2R+1,c_z] b_rel | W_m[msa_dim,c_m] b_m | W_t[tf_dim,c_m] b_t | LN_m gamma beta [c_m] |
 * LN_z gamma beta [c_z] | W_d[n_dist_bins,c_z] b_d | W_e[extra_dim,c_e] b_e.  0 for a null / unsupported config. */
size_t pf_embedder_floats(const pf_embed_config* cfg);
/* Errors: INVALID_ARG (null), SHAPE (c_m, c_z not in {128, 256}; msa_dim > 64; blob length), ALLOC, CUDA. */
pf_status pf_embedder_create(pf_embedder_t** out, const float* weights_host, size_t n_weight_floats,
                             const pf_embed_config* cfg);
/* E.1 + E.2 for a batch, asynchronously on cuda_stream, IN PLACE: with has_prev != 0 dev msa[B,S,N,c_m] / pair[B,N,N,c_z] hold
 * the previous cycle's trunk output on entry (only row s = 0 of msa is read); with has_prev == 0 they are not read (previous
 * representations = 0).  On return they hold the embedded representations.  target_feat_dev [B,N,tf_dim] fp32,
 * residue_index_dev [B,N] int32, msa_feat_dev [B,S,N,msa_dim] fp32, x_prev_dev [B,N,3] fp32 or NULL.  Every position is
 * embedded (padding included: the embedders are per position; masks belong to the trunk). */
pf_status pf_embedder_forward(pf_embedder_t* e, const float* target_feat_dev, const int* residue_index_dev,
                              const float* msa_feat_dev, const float* x_prev_dev, int has_prev, float* msa_dev,
                              float* pair_dev, int B, int S, int N, void* cuda_stream);
/* E.4 extra-MSA embedder: dev extra_msa[B,S_e,N,c_e] = Lin_e(dev extra_msa_feat[B,S_e,N,extra_dim]). */
pf_status pf_embedder_forward_extra(pf_embedder_t* e, const float* extra_msa_feat_dev, float* extra_msa_dev, int B, int S_e,
                                    int N, void* cuda_stream);
long long pf_embedder_last_launch_count(const pf_embedder_t* e);
void pf_embedder_destroy(pf_embedder_t* e);
/* E.3: n_cycles x (pf_embedder_forward [, pf_embedder_forward_extra, pf_extra_msa_forward over n_extra_blocks blocks],
 * pf_evoformer_forward over n_blocks blocks) on cuda_stream; msa_dev / pair_dev are outputs (their contents on entry are
 * ignored).  x == NULL skips the extra-MSA stack (its three arguments and S_e, n_extra_blocks are then ignored); otherwise
 * extra_msa_dev [B,S_e,N,c_e] is a caller-owned scratch buffer and extra_msa_mask_dev [B,S_e] the stack's sequence mask.
 * n_cycles = 4 is AlphaFold's "three recycling procedures".
 * Errors: those of the calls it makes; SHAPE if n_cycles < 1 or the channel dims of the handles differ. */
pf_status pf_evoformer_forward_recycled(pf_evoformer_t* h, pf_embedder_t* e, pf_extra_msa_t* x, const float* target_feat_dev,
                                        const int* residue_index_dev, const float* msa_feat_dev, const float* x_prev_dev,
                                        const float* extra_msa_feat_dev, float* extra_msa_dev, const float* extra_msa_mask_dev,
                                        float* msa_dev, float* pair_dev, const float* seq_mask_dev, const float* msa_mask_dev,
                                        int B, int S, int S_e, int N, int n_blocks, int n_extra_blocks, int n_cycles,
                                        void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * Extra-MSA stack: the Evoformer block at c_e = 64 MSA channels with GLOBAL column attention over an MSA
 * of thousands of sequences, updating the same pair representation (part of the network the paper's GPU stage runs,
 * PAPER.md:61; AlphaFold v2.0.1 CASP14 preset).  PAPER.md prints no formula; readings X.1-X.9:
 *   X.1 MSA row attention with pair bias (A.1 at c_e channels, heads of dimension c_e / heads_msa)
 *   X.2 MSA column global attention: x = LN(e); qbar_i = sum_s mu_si x_si / (sum_s mu_si + 1e-10); q[i,h] = Lin0(qbar_i)_h / sqrt(d);
 *       ONE key / value head k[s,i], v[s,i] in R^d; P = softmax_s(q[i,h].k[s,i] + NEG(mu_si)); o[i,h] = sum_s P v[s,i];
 *       e[s,i] += Lin_o( sigmoid(Lin_g(x_si)) (.) concat_h o[i,h] )
 *   X.3 MSA transition (A.3 at c_e), X.4 outer-product-mean (A.4 from e into pair), X.5-X.9 the pair stack A.5-A.9.
 * 16-bit operands with fp32 accumulation and fp32 residual streams as PF_BF16 (X.2 runs in fp32).  Same conventions, masks
 * (R2, R3), in-place semantics and error behaviour as pf_evoformer_forward.  Limits: N <= 1024, N_seq <= ~2900, B <= 511.
 * Weights blob: n_blocks_max blocks of pf_extra_msa_block_floats values, the Appendix-B order at c_m = c_e with the column
 * attention's entry replaced by: LN gamma beta [c_e], W_q [c_e,c_e], W_k [c_e,d], W_v [c_e,d], W_g [c_e,c_e], b_g, W_o [c_e,c_e], b_o.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
  int c_e;            /* extra-MSA channels (64) */
  int c_z;            /* pair channels (128) */
  int heads_msa;      /* 8 heads of dimension c_e / heads_msa = 8 */
  int heads_pair;     /* 4 */
  int head_dim_pair;  /* 32 */
  int c_opm;          /* 32 */
  int c_tri;          /* 128 */
  int transition_n;   /* 4 */
  int n_blocks_max;   /* blocks in the blob (4 in AlphaFold) */
} pf_extra_config;
size_t pf_extra_msa_block_floats(const pf_extra_config* cfg);
pf_status pf_extra_msa_create(pf_extra_msa_t** out, const float* weights_host, size_t n_weight_floats,
                              const pf_extra_config* cfg);
/* blocks [0, n_blocks) on dev extra_msa[B,S,N,c_e] and dev pair[B,N,N,c_z], in place, asynchronously on cuda_stream */
pf_status pf_extra_msa_forward(pf_extra_msa_t* x, float* extra_msa_dev, float* pair_dev, const float* seq_mask_dev,
                               const float* extra_msa_mask_dev, int B, int S, int N, int n_blocks, void* cuda_stream);
/* test hook: sub-step `substep` (1..9 = X.1..X.9) of block `block` */
pf_status pf_extra_msa_forward_substep(pf_extra_msa_t* x, float* extra_msa_dev, float* pair_dev, const float* seq_mask_dev,
                                       const float* extra_msa_mask_dev, int B, int S, int N, int block, int substep,
                                       void* cuda_stream);
long long pf_extra_msa_last_launch_count(const pf_extra_msa_t* x);
/* per-launch timing as pf_evoformer_set_profiling / pf_evoformer_get_profile (same kinds) */
pf_status pf_extra_msa_set_profiling(pf_extra_msa_t* x, int enable);
pf_status pf_extra_msa_get_profile(pf_extra_msa_t* x, int kind, long long* launches, double* ms, double* flops, double* bytes);
void pf_extra_msa_destroy(pf_extra_msa_t* x);

/* ------------------------------------------------------------------------------------------------
 * Structure module and output heads: the last stage of the network the paper's GPU stage runs ("a new
 * Evoformer architecture" feeding "the structure module"; AlphaFold v2.0.1 monomer).
 * PAPER.md prints no formula; readings M.0-M.6 / H.1-H.5, per protein:
 *   M.0 s^single_i = Lin_single(m_0i)                         M.1 s^init = LN_s(s^single), zn = LN_z(z), s = Lin_in(s^init), T_i = (I, 0)
 *   M.2 invariant point attention, H heads: q, k, v = Lin0(s) [c per head]; query / key points qp, kp [P_q x 3], value points vp
 *       [P_v x 3] = Lin0(s) in the residue's frame, mapped to the global frame by T; b = Lin0(zn) [H];
 *       a_hij = softmax_j( sqrt(1/3) ( q_ih.k_jh / sqrt(c) + b_ijh - softplus(g_h) sqrt(2 / (9 P_q)) / 2 sum_p |T_i qp_ihp - T_j kp_jhp|^2 ) + NEG(sigma_j) )
 *       IPA_i = Lin_out( concat[ sum_j a zn_ij (H c_z) | sum_j a v_jh (H c) | T_i^-1 sum_j a T_j vp_jhp (H P_v 3) | its norms, sqrt(|.|^2 + 1e-8) (H P_v) ] )
 *   M.3 s = LN_ipa(s + IPA);  s = LN_tr(s + Lin_3(relu(Lin_2(relu(Lin_1(s))))))            (n_layers layers, weights shared)
 *   M.4 (b, c, d, u) = Lin_bb(s_i); R^upd from the unit quaternion (1, b, c, d) / |.|;  t_i <- R_i u + t_i, R_i <- R_i R^upd
 *   M.5 a = Lin_a1(s) + Lin_a2(s^init); twice a += Lin_rb(relu(Lin_ra(relu(a)))); alpha = Lin_alpha(relu(a)) [n_torsion, 2], normalised
 *   M.6 positions x_i = pos_scale t_i (Angstrom; the frame origin = C-alpha).  All-atom side-chain coordinates are not computed
 *       (they need per-residue ideal-geometry tables that are not on this box): x is what the recycling embedder (E.2) receives.
 *   H.1 distogram logits_ij = Lin_dg(z_ij) + Lin_dg(z_ji)    H.2 masked-MSA logits_si = Lin_mm(m_si)
 *   H.3 pLDDT_i = 100 sum_k softmax(Lin_l3(relu(Lin_l2(relu(Lin_l1(LN_l(s_i)))))))_k (k + 1/2) / n_lddt_bins
 *   H.4 predicted-aligned-error logits_ij = Lin_pae(z_ij) (not symmetrised)   H.5 experimentally-resolved logits_i = Lin_er(s_i)
 * All arithmetic is fp32 (tolerance 1e-4 max-abs against the fp64 oracle on s, frames in nanometres, angles; 1e-3 on x in
 * Angstrom and pLDDT in points).  Masked residues act as masked keys only; outputs at masked residues are unspecified but finite.
 * Weights blob (fp32, every matrix row-major [in, out]), in this order: W_single b | LN_s g b | LN_z g b | W_in b | W_q | W_k |
 * W_v [c_s, H c] | W_qp | W_kp [c_s, H P_q 3] | W_vp [c_s, H P_v 3] | W_b [c_z, H] | g_head [H] | W_out [H (c_z + c + 4 P_v), c_s] b |
 * LN_ipa g b | W_1 b W_2 b W_3 b | LN_tr g b | W_bb [c_s, 6] b | W_a1 b W_a2 b [c_s, c_r] | 2 x (W_ra b W_rb b [c_r, c_r]) |
 * W_alpha [c_r, 2 n_torsion] b | W_dg [c_z, n_dist_bins] b | W_mm [c_m, n_msa_classes] b | LN_l g b | W_l1 [c_s, c_l] b |
 * W_l2 [c_l, c_l] b | W_l3 [c_l, n_lddt_bins] b | W_pae [c_z, n_pae_bins] b | W_er [c_s, n_resolved] b.
 * ---------------------------------------------------------------------------------------------- */
typedef struct pf_structure pf_structure_t;   /* opaque; owns device weights and a grow-only workspace */
typedef struct {
  int c_m;            /* 256 */
  int c_z;            /* 128 */
  int c_s;            /* single-representation channels (384) */
  int heads;          /* IPA heads H (12; at most 32) */
  int c_ipa;          /* scalar channels per head c (16) */
  int n_qp;           /* query / key points per head P_q (4) */
  int n_pv;           /* value points per head P_v (8) */
  int n_layers;       /* default layer count (8) */
  int c_resnet;       /* torsion-angle resnet width (128) */
  int n_torsion;      /* 7 */
  int n_dist_bins;    /* distogram bins (64) */
  int n_msa_classes;  /* masked-MSA classes (23) */
  int n_lddt_bins;    /* pLDDT bins (50) */
  int c_lddt;         /* pLDDT head width (128) */
  int n_pae_bins;     /* predicted-aligned-error bins (64) */
  int n_resolved;     /* experimentally-resolved classes (37) */
  float pos_scale;    /* Angstrom per unit of frame translation (10) */
} pf_struct_config;
/* fp32 values in the blob described above; 0 for a null / unsupported config. */
size_t pf_structure_floats(const pf_struct_config* cfg);
/* Errors: INVALID_ARG (null), SHAPE (dims, blob length), ARCH, ALLOC, CUDA. */
pf_status pf_structure_create(pf_structure_t** out, const float* weights_host, size_t n_weight_floats,
                              const pf_struct_config* cfg);
/* M.0-M.6 (+ H.3) for a batch, asynchronously on cuda_stream.  Inputs (device, read only): msa[B,S,N,c_m] (only row s = 0 is
 * read), pair[B,N,N,c_z], seq_mask[B,N].  Outputs (device, each may be NULL): s_out[B,N,c_s], frames_out[B,N,12] (R row-major
 * 3 x 3, then t, nanometres), x_out[B,N,3] (Angstrom), alpha_out[B,N,n_torsion,2], plddt_out[B,N], resolved_out[B,N,n_resolved]
 * (H.5 logits).  n_layers >= 1 (the
 * config's value is the AlphaFold default).  Limit: heads x N x 4 bytes <= ~200 KB (N <= 4000 at 12 heads).
 * Errors: INVALID_ARG, SHAPE, ALLOC (workspace: ~N^2 (c_z + heads) floats per protein), CUDA. */
pf_status pf_structure_forward(pf_structure_t* h, const float* msa_dev, const float* pair_dev, const float* seq_mask_dev, int B,
                               int S, int N, int n_layers, float* s_out, float* frames_out, float* x_out, float* alpha_out,
                               float* plddt_out, float* resolved_out, void* cuda_stream);
/* H.1 / H.2 / H.4: distogram_out[B,N,N,n_dist_bins], masked_msa_out[B,S,N,n_msa_classes], pae_out[B,N,N,n_pae_bins] (device;
 * NULL skips a head). */
pf_status pf_heads_forward(pf_structure_t* h, const float* msa_dev, const float* pair_dev, int B, int S, int N,
                           float* distogram_out, float* masked_msa_out, float* pae_out, void* cuda_stream);
long long pf_structure_last_launch_count(const pf_structure_t* h);
void pf_structure_destroy(pf_structure_t* h);
/* H.3 for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the pLDDT head
 * (LN_l, two ReLU layers, logits, expectation — the same kernels as the tail of pf_structure_forward) with its intermediates in a
 * file-scope device array of PF_PLDDT_STATIC_SCRATCH_BYTES instead of the handle's workspace.  The call performs no cudaMalloc,
 * cudaFree or allocating library routine; every GPU that loads the library holds the array until the process exits.
 * s_dev[rows, c_s] (device, read only; rows = B N of the single representation s_out), plddt_out[rows] (device).  Asynchronous on
 * cuda_stream.  rows * (c_s + 2 c_lddt + n_lddt_bins) floats (each of the four segments rounded up to 256 bytes) must fit the
 * array: 3039 rows at the default dims; beyond that the call fails with PF_ERR_SHAPE and pf_last_error() states the sizes.
 * ALL calls in the process on one GPU share the one array (whatever the handle or stream): calls that overlap on the GPU race;
 * order them on one stream or with events.  The array keeps the previous call's contents; nothing in it needs clearing, each
 * launch reads only what the launch before it wrote in the same call.  The first call on a device resolves the array's device
 * address (cudaGetSymbolAddress) and may load the module: make it before a stream capture begins.
 * Errors: INVALID_ARG (null, wrong current device, device ordinal >= 64), SHAPE (rows < 1 or beyond the array), CUDA. */
#define PF_PLDDT_STATIC_SCRATCH_BYTES (8u << 20)
pf_status pf_plddt_forward_static(pf_structure_t* h, const float* s_dev, int rows, float* plddt_out, void* cuda_stream);
/* The whole GPU stage: n_cycles x (pf_embedder_forward with the PREVIOUS cycle's structure-module
 * positions — x_prev0_dev [B,N,3] or NULL (no previous structure) in the first cycle —, [extra-MSA stack], pf_evoformer_forward,
 * pf_structure_forward).  Arguments as pf_evoformer_forward_recycled; x_cycles_out [n_cycles,B,N,3] (device, required) receives the
 * positions after every cycle (the last slice is the prediction; earlier slices are what the next cycle's recycling embedder
 * read, so a checker can replay the distance-bin decisions); s_out / frames_out / alpha_out / plddt_out (may be NULL) are the
 * last cycle's.  pf_structure_last_launch_count(sm) then counts every launch of the call.
 * Errors: those of the calls it makes; INVALID_ARG if x_cycles_out is NULL. */
pf_status pf_fold_forward(pf_evoformer_t* h, pf_embedder_t* e, pf_extra_msa_t* x, pf_structure_t* sm,
                          const float* target_feat_dev, const int* residue_index_dev, const float* msa_feat_dev,
                          const float* x_prev0_dev, const float* extra_msa_feat_dev, float* extra_msa_dev,
                          const float* extra_msa_mask_dev, float* msa_dev, float* pair_dev, const float* seq_mask_dev,
                          const float* msa_mask_dev, int B, int S, int S_e, int N, int n_blocks, int n_extra_blocks, int n_cycles,
                          int n_layers, float* x_cycles_out, float* s_out, float* frames_out, float* alpha_out, float* plddt_out,
                          void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * Length-bucketing batch scheduler ("sort by length ... share the compiled model";
 * SURVEY.md §3(iv)).  Host only.  Proteins are sorted by descending length (largest first, as the paper
 * compiles for the largest), assigned to the smallest bucket >= length, and cut into batches of at most
 * max(1, floor(mem_budget_bytes / bytes_per_protein(bucket, S))) proteins of one bucket.
 * ---------------------------------------------------------------------------------------------- */
typedef struct pf_sched pf_sched_t;

/* buckets: ascending padded lengths (host ints).  S: N_seq used for the footprint estimate.
 * Errors: INVALID_ARG (null / not ascending / n_buckets < 1 / S < 1). */
pf_status pf_sched_create(pf_sched_t** out, const int* buckets, int n_buckets, size_t mem_budget_bytes, int S);
/* Errors: SHAPE if length < 1 or length > largest bucket. */
pf_status pf_sched_add(pf_sched_t* s, int protein_id, int length);
/* Writes up to cap protein ids and their lengths (lengths_out may be NULL) of the next batch and its bucket;
 * returns the batch size B (0 when drained, -1 on invalid arguments).  The first call freezes the queue order. */
int pf_sched_next_batch(pf_sched_t* s, int* ids_out, int* lengths_out, int cap, int* bucket_out);
/* Footprint model used for batching: residual streams + workspace, bytes per protein. */
size_t pf_sched_bytes_per_protein(int bucket, int S);
/* Cost of one protein for load balancing: GEMM FLOPs of one Evoformer block at its bucket (SURVEY.md §8(d) F(S,N)). */
double pf_sched_cost(int bucket, int S);
/* Multi-GPU is replicas only (PAPER.md:190 runs independent single-GPU tasks, PAPER.md:260 lists
 * multi-GPU inference as future work): this call shards the PROTEIN LIST, there is no data-path collective.
 * lengths[n], ascending buckets[n_buckets] (host ints) -> rank_out[n] in [0, world): longest-processing-time-first over
 * pf_sched_cost, ties to the lowest rank; deterministic, so every rank computes the same assignment without talking.
 * Errors: INVALID_ARG (null, world < 1, buckets not ascending), SHAPE (a length outside [1, largest bucket]). */
pf_status pf_sched_partition(const int* lengths, int n, const int* buckets, int n_buckets, int S, int world,
                             int* rank_out);
void pf_sched_destroy(pf_sched_t* s);

#ifdef __cplusplus
}
#endif
#endif /* PF_EVOFORMER_H_ */
