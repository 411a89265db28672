"""fp64 CPU oracle of the extra-MSA stack (TEST INFRASTRUCTURE — not part of the product path; only tests/,
__graft_entry__.smoke() and bench.py's reference legs may import it).

What it computes: SURVEY.md §8(f)1 — "extra-MSA stack variant: the same block at c_e = 64 with *global* column attention
and S_extra in the thousands", the part of the network ParaFold's GPU stage runs between the embedders and the 48-block
trunk ("complicated neural network"; AlphaFold v2.0.1, CASP14 preset).  PAPER.md prints no formula;
the reading X.1-X.9 of DESIGN.md §2c (the published AlphaFold 2 algorithm restated) is:

  X.1 MSA row attention with pair bias on e[s,i,:] in R^{c_e}: A.1 with c_e channels and H_e heads of dimension c_e / H_e
  X.2 MSA column GLOBAL attention: x = LN(e);  qbar_i = sum_s mu_si x_si / (sum_s mu_si + 1e-10);
      q[i,h] = Lin0_q(qbar_i)_h / sqrt(d);  k[s,i] = Lin0_k(x_si) in R^d and v[s,i] = Lin0_v(x_si) in R^d (ONE key / value head
      shared by all query heads);  L[i,h,s] = q[i,h].k[s,i] + NEG(mu_si);  P = softmax_s;  o[i,h] = sum_s P[i,h,s] v[s,i];
      G[s,i] = sigmoid(Lin_g(x_si));  e[s,i] += Lin_o( G[s,i] (.) concat_h o[i,h] )
  X.3 MSA transition (A.3 at c_e)            X.4 outer-product-mean (A.4 from e, into z)
  X.5 .. X.9 the pair stack of the main block (A.5 .. A.9), unchanged
Order: X.1 .. X.9 as in the main block (reading R0).  Everything except X.2 is the main-block function at other dimensions,
so it inherits those pins; X.2 is pinned in tests/test_oracle_extra.py (pure-Python loops; the single-sequence and uniform
closed forms; permutation of the MSA rows).  Parity with DeepMind's AlphaFold itself: **parity unpinned**.
"""
from __future__ import annotations

import numpy as np

from . import evoformer_ref as ref
from .evoformer_ref import _f64, layer_norm, linear, neg, sigmoid, softmax

GLOBAL_Q_EPS = 1e-10


def msa_col_global_attention(e, seq_mask, msa_mask, w, head_dim):
    """X.2 on e[S, N, c_e]."""
    e = _f64(e)
    S, N, _ = e.shape
    x = layer_norm(e, w["ln_g"], w["ln_b"])
    mu = _f64(msa_mask)[:, None] * _f64(seq_mask)[None, :]                        # mu[s, i]
    qbar = (mu[:, :, None] * x).sum(axis=0) / (mu.sum(axis=0)[:, None] + GLOBAL_Q_EPS)   # [N, c_e]
    q = linear(qbar, w["wq"]) / np.sqrt(float(head_dim))                           # [N, H d]
    H = q.shape[-1] // head_dim
    qh = q.reshape(N, H, head_dim)
    k = linear(x, w["wk"])                                                          # [S, N, d]
    v = linear(x, w["wv"])                                                          # [S, N, d]
    logits = np.einsum("ihd,sid->ihs", qh, k) + np.transpose(neg(mu), (1, 0))[:, None, :]
    P = softmax(logits, axis=-1)                                                    # over s
    o = np.einsum("ihs,sid->ihd", P, v).reshape(N, H * head_dim)
    gate = sigmoid(linear(x, w["wg"], w["bg"]))                                     # [S, N, H d]
    return e + linear(gate * o[None, :, :], w["wo"], w["bo"])


SUBSTEPS = ("row", "col_global", "msa_trans", "opm", "tri_mul_out", "tri_mul_in", "tri_att_start", "tri_att_end", "pair_trans")


def substep(step, e, z, seq_mask, msa_mask, w, head_dim_msa=8, head_dim_pair=32):
    """Sub-step ``step`` (1..9) of one extra-MSA block; returns (e, z)."""
    e, z = _f64(e), _f64(z)
    if step == 1:
        e = ref.msa_row_attention(e, z, seq_mask, msa_mask, w["row"], head_dim_msa)
    elif step == 2:
        e = msa_col_global_attention(e, seq_mask, msa_mask, w["col_global"], head_dim_msa)
    elif step == 3:
        e = ref.transition(e, w["msa_trans"])
    elif step == 4:
        z = ref.outer_product_mean(e, z, seq_mask, msa_mask, w["opm"])
    elif 5 <= step <= 9:
        _, z = ref.substep(step, e, z, seq_mask, msa_mask, w, head_dim_pair)
    else:
        raise ValueError(f"substep {step} not in 1..9")
    return e, z


def extra_msa_block(e, z, seq_mask, msa_mask, w, head_dim_msa=8, head_dim_pair=32):
    for step in range(1, 10):
        e, z = substep(step, e, z, seq_mask, msa_mask, w, head_dim_msa, head_dim_pair)
    return e, z


def extra_msa_stack(e, z, seq_mask, msa_mask, blocks, head_dim_msa=8, head_dim_pair=32):
    """n blocks with distinct weights; only z leaves the stack (e is dropped by the caller)."""
    for w in blocks:
        e, z = extra_msa_block(e, z, seq_mask, msa_mask, w, head_dim_msa, head_dim_pair)
    return e, z


def msa_col_global_attention_at(e, seq_mask, msa_mask, w, s, i, head_dim):
    """X.2 at one output position (s, i): only column i of e enters (sampled oracle for the large shapes)."""
    x = layer_norm(_f64(e[:, i]), w["ln_g"], w["ln_b"])                             # [S, c_e]
    mu = _f64(msa_mask) * float(seq_mask[i])
    qbar = (mu[:, None] * x).sum(axis=0) / (mu.sum() + GLOBAL_Q_EPS)
    q = linear(qbar, w["wq"]) / np.sqrt(float(head_dim))
    H = q.shape[-1] // head_dim
    k = linear(x, w["wk"])
    v = linear(x, w["wv"])
    o = np.zeros(H * head_dim)
    for h in range(H):
        P = softmax(k @ q[h * head_dim:(h + 1) * head_dim] + neg(mu))
        o[h * head_dim:(h + 1) * head_dim] = P @ v
    gate = sigmoid(linear(x[s], w["wg"], w["bg"]))
    return _f64(e[s, i]) + linear(gate * o, w["wo"], w["bo"])
