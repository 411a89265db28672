"""fp64 CPU oracle of the input / recycling embedders and the recycled trunk (TEST INFRASTRUCTURE — not part of the
product path; only tests/, __graft_entry__.smoke() and bench.py's reference legs may import it).

What it computes: SURVEY.md §8(f)2 — "recycling wrapper + input/recycling embedders", the part of the GPU stage that turns
the features ParaFold's CPU stage wrote (features.pkl) into the trunk's inputs and feeds the trunk's outputs
back ("three recycling procedures"; "recycling").  PAPER.md prints no formula; what follows is
the reading E.1-E.3 of DESIGN.md §2b (the published AlphaFold 2 algorithm restated; AlphaFold v2.0.1 monomer):

  E.1 input embedder     a_i = Lin_a(tf_i), b_j = Lin_b(tf_j), z_ij = a_i + b_j + Lin_rel(onehot(clip(r_i - r_j, -R, R) + R)),
                         m_si = Lin_m(msa_feat_si) + Lin_t(tf_i)
  E.2 recycling embedder z_ij += LN_z(zprev_ij) + Lin_d(onehot_bins(|xprev_i - xprev_j|)),   m_0i += LN_m(mprev_0i)
                         bins: K lower edges e_k evenly spaced from first_break to last_break; d falls in bin k when
                         e_k^2 < d^2 < e_{k+1}^2 (e_K = infinity); below e_0 no bin is set (the one-hot is all zero)
  E.3 recycled trunk     for c in 0 .. n_cycles-1: (m, z) = E.1(features); E.2 with the previous cycle's (m_0, z) — zeros in
                         the first cycle —; optionally the extra-MSA stack: e = Lin_e(extra_msa_feat) (E.4), (e, z) =
                         extra_stack(e, z) (oracle/extra_msa_ref.py), e dropped; (m, z) = trunk(m, z).  xprev comes from the structure module, which is not built
                         (SURVEY.md §8(f)4): it is an input held constant over the cycles (zeros = "no previous structure").

The bin decision is a floating-point comparison deciding an integer: both sides take it in fp32 with the same operation
order ((dx*dx + dy*dy) + dz*dz, no fused multiply-add), so that the one-hot index agrees bit for bit.
Pins: tests/test_oracle_embed.py (row-gather closed forms, numpy searchsorted for the bins, LN(0) = beta, pure-Python
loops on tiny inputs, the first cycle's closed form).  Parity with DeepMind's AlphaFold itself: **parity unpinned**.
"""
from __future__ import annotations

import numpy as np

from .evoformer_ref import F64, _f64, evoformer_trunk, layer_norm, linear
from .extra_msa_ref import extra_msa_stack


def relpos_index(residue_index, max_relpos):
    """clip(r_i - r_j, -R, R) + R in [0, 2R]  (E.1)."""
    r = np.asarray(residue_index, dtype=np.int64)
    return np.clip(r[:, None] - r[None, :], -max_relpos, max_relpos) + max_relpos


def one_hot(idx, n):
    out = np.zeros(idx.shape + (n,), dtype=F64)
    np.put_along_axis(out, idx[..., None], 1.0, axis=-1)
    return out


def input_embedder(target_feat, residue_index, msa_feat, w, max_relpos=32):
    """E.1 -> (m[S,N,c_m], z[N,N,c_z])."""
    tf = _f64(target_feat)
    a = linear(tf, w["w_a"], w["b_a"])
    b = linear(tf, w["w_b"], w["b_b"])
    rel = one_hot(relpos_index(residue_index, max_relpos), 2 * max_relpos + 1)
    z = a[:, None, :] + b[None, :, :] + linear(rel, w["w_rel"], w["b_rel"])
    m = linear(_f64(msa_feat), w["w_m"], w["b_m"]) + linear(tf, w["w_t"], w["b_t"])[None, :, :]
    return m, z


def bin_edges(n_bins, first_break, last_break):
    return np.linspace(first_break, last_break, n_bins)


def distance_one_hot(x, n_bins, first_break, last_break):
    """onehot_bins(|x_i - x_j|) [N, N, n_bins]; the comparison runs in fp32 (see the module header)."""
    x = np.asarray(x, dtype=np.float32)
    d = x[:, None, :] - x[None, :, :]
    d2 = (d[..., 0] * d[..., 0] + d[..., 1] * d[..., 1]) + d[..., 2] * d[..., 2]        # fp32, this order
    e = bin_edges(n_bins, first_break, last_break).astype(np.float32)
    lo = e * e
    hi = np.concatenate([lo[1:], np.array([np.inf], dtype=np.float32)])
    return ((d2[..., None] > lo) & (d2[..., None] < hi)).astype(F64)


def recycling_embedder(m, z, m0_prev, z_prev, x_prev, w, n_bins=15, first_break=3.25, last_break=20.75):
    """E.2 -> (m, z) with the previous cycle's first MSA row, pair representation and positions folded in."""
    m, z = _f64(m).copy(), _f64(z)
    dg = distance_one_hot(x_prev, n_bins, first_break, last_break)
    z = z + layer_norm(z_prev, w["ln_z_g"], w["ln_z_b"]) + linear(dg, w["w_d"], w["b_d"])
    m[0] = m[0] + layer_norm(m0_prev, w["ln_m_g"], w["ln_m_b"])
    return m, z


def embed_cycle(target_feat, residue_index, msa_feat, m0_prev, z_prev, x_prev, w, max_relpos=32, n_bins=15,
                first_break=3.25, last_break=20.75):
    """E.1 followed by E.2 (what one call of the CUDA embedder computes)."""
    m, z = input_embedder(target_feat, residue_index, msa_feat, w, max_relpos)
    return recycling_embedder(m, z, m0_prev, z_prev, x_prev, w, n_bins, first_break, last_break)


def extra_msa_embedder(extra_msa_feat, w):
    """E.4  e_si = Lin_e(extra_msa_feat_si)."""
    return linear(_f64(extra_msa_feat), w["w_e"], w["b_e"])


def recycled_trunk(target_feat, residue_index, msa_feat, x_prev, seq_mask, msa_mask, w_embed, blocks, n_cycles,
                   head_dim=32, extra=None, **kw):
    """E.3 for one protein -> (m, z) after the last cycle's trunk.
    extra = (extra_msa_feat[S_e,N,F], extra_msa_mask[S_e], extra_blocks, head_dim_msa) runs the extra-MSA stack between the
    embedders and the trunk in every cycle."""
    S, N = np.asarray(msa_feat).shape[:2]
    c_m, c_z = np.asarray(w_embed["w_m"]).shape[1], np.asarray(w_embed["w_a"]).shape[1]
    m0_prev, z_prev = np.zeros((N, c_m)), np.zeros((N, N, c_z))
    m = z = None
    for _ in range(n_cycles):
        m, z = embed_cycle(target_feat, residue_index, msa_feat, m0_prev, z_prev, x_prev, w_embed, **kw)
        if extra is not None:
            xf, xmask, xblocks, xhd = extra
            _, z = extra_msa_stack(extra_msa_embedder(xf, w_embed), z, seq_mask, xmask, xblocks, xhd, head_dim)
        m, z = evoformer_trunk(m, z, seq_mask, msa_mask, blocks, head_dim)
        m0_prev, z_prev = m[0], z
    return m, z
