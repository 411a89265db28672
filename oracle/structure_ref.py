"""fp64 CPU oracle of the structure module and the output heads (TEST INFRASTRUCTURE — not part of the product path;
only tests/, __graft_entry__.smoke() and bench.py's reference legs may import it).

What it computes: SURVEY.md §8(f)4 — "structure module + heads", the last stage of the network the paper's GPU stage runs
("a new Evoformer architecture" feeding "the structure module"; AlphaFold v2.0.1 monomer,
PAPER.md:127).  PAPER.md prints no formula; what follows is the reading M.0-M.6 / H.1-H.5 of DESIGN.md §2d (the published
AlphaFold 2 algorithm restated in this repository's notation).  One protein, no batch axis:

  M.0 single representation   s^single_i = Lin_single(m_0i)                                  (first MSA row, c_m -> c_s)
  M.1 initialisation          s^init = LN_s(s^single),  zn = LN_z(z),  s = Lin_in(s^init),  T_i = (R_i, t_i) = (I, 0)
  M.2 invariant point attention (H heads, c channels, P_q query points, P_v value points per head)
        q, k, v = Lin0(s)  [N,H,c];   qp, kp [N,H,P_q,3], vp [N,H,P_v,3] = Lin0(s)  (local frame);   b = Lin0(zn) [N,N,H]
        qg_ihp = R_i qp_ihp + t_i  (same for kg, vg);   w_C = sqrt(2 / (9 P_q)),  w_L = sqrt(1/3),  gamma_h = softplus(g_h)
        a_hij = softmax_j( w_L ( q_ih.k_jh / sqrt(c) + b_ijh - gamma_h w_C / 2 sum_p |qg_ihp - kg_jhp|^2 ) + NEG(sigma_j) )
        ot_ih = sum_j a_hij zn_ij  [c_z],   o_ih = sum_j a_hij v_jh  [c],   op_ihp = R_i^T ( sum_j a_hij vg_jhp - t_i )  [3]
        IPA_i = Lin_out( concat[ ot_i (H c_z) | o_i (H c) | op_i (H P_v 3) | sqrt(|op_ihp|^2 + 1e-8) (H P_v) ] )
  M.3 layer (weights SHARED by all n_layers)
        s = LN_ipa(s + IPA(s, zn, T));   s = LN_tr(s + Lin_3(relu(Lin_2(relu(Lin_1(s))))))
  M.4 backbone update         (b, c, d, u) = Lin_bb(s_i);  unit quaternion (1, b, c, d) / sqrt(1 + b^2 + c^2 + d^2) -> R^upd;
                              T_i <- T_i o (R^upd, u):   t_i <- R_i u + t_i,  R_i <- R_i R^upd
  M.5 torsion angles (after the last layer)
        a = Lin_a1(s_i) + Lin_a2(s^init_i);  twice: a <- a + Lin_rb(relu(Lin_ra(relu(a))));
        alpha = Lin_alpha(relu(a)) [n_torsion, 2],  alpha_hat = alpha / sqrt(|alpha|^2 + 1e-12)
  M.6 outputs                 s (final), frames (R_i, t_i), positions x_i = pos_scale t_i  (Angstrom; the frame origin is
                              the C-alpha atom), alpha_hat
  H.1 distogram               logits_ij = Lin_dg(z_ij) + Lin_dg(z_ji)                         [N,N,n_dist_bins]
  H.2 masked-MSA              logits_si = Lin_mm(m_si)                                         [S,N,n_msa_classes]
  H.3 pLDDT                   l_i = Lin_l3(relu(Lin_l2(relu(Lin_l1(LN_l(s_i))))))  [n_lddt_bins];  p = softmax(l);
                              plddt_i = 100 sum_k p_k (k + 1/2) / n_lddt_bins
  H.4 predicted aligned error logits_ij = Lin_pae(z_ij)   [N,N,n_pae_bins]   (NOT symmetrised: error of j in the frame of i)
  H.5 experimentally resolved logits_i = Lin_er(s_i)      [N,n_resolved]

Masked residues enter only as attention keys (NEG(sigma_j)); outputs at masked residues are unspecified (R3).
All-atom side-chain coordinates are NOT computed: they need the ideal-geometry tables of the amino acids, which are data of
a third-party project and not on this box; the positions handed to the recycling embedder (E.2) are the C-alpha positions
x_i of M.6 (reading M.6 in DESIGN.md).

Pins: tests/test_oracle_structure.py — scipy's Rotation for the quaternion map and the frame composition, invariance of
(s, alpha_hat, plddt) and equivariance of the frames under a global rigid motion of the incoming frames (the property the
attention is named for), pure-Python index loops for M.2 on a tiny input, closed forms (zero point weights reduce M.2 to
plain biased attention = torch scaled_dot_product_attention; W_bb = 0 keeps T = identity), softmax rows sum to one,
padding invariance with a negative control, H.1 symmetry, plddt in [0, 100] and its one-hot closed form.
Parity with DeepMind's AlphaFold itself: **parity unpinned**.
"""
from __future__ import annotations

import numpy as np

from .evoformer_ref import F64, NEG_INF_SCALE, _f64, layer_norm, linear, softmax

IPA_NORM_EPS = 1e-8
ANGLE_EPS = 1e-12


def relu(x):
    return np.maximum(_f64(x), 0.0)


def softplus(x):
    x = _f64(x)
    return np.log1p(np.exp(-np.abs(x))) + np.maximum(x, 0.0)


def quat_to_rot(b, c, d):
    """M.4: rotation matrix of the unit quaternion (1, b, c, d) / sqrt(1 + b^2 + c^2 + d^2); inputs [...]-shaped."""
    b, c, d = _f64(b), _f64(c), _f64(d)
    n = np.sqrt(1.0 + b * b + c * c + d * d)
    a, b, c, d = 1.0 / n, b / n, c / n, d / n
    R = np.empty(b.shape + (3, 3), dtype=F64)
    R[..., 0, 0] = a * a + b * b - c * c - d * d
    R[..., 0, 1] = 2 * (b * c - a * d)
    R[..., 0, 2] = 2 * (b * d + a * c)
    R[..., 1, 0] = 2 * (b * c + a * d)
    R[..., 1, 1] = a * a - b * b + c * c - d * d
    R[..., 1, 2] = 2 * (c * d - a * b)
    R[..., 2, 0] = 2 * (b * d - a * c)
    R[..., 2, 1] = 2 * (c * d + a * b)
    R[..., 2, 2] = a * a - b * b - c * c + d * d
    return R


def compose_frames(R, t, R_upd, u):
    """M.4: T o (R_upd, u) = (R R_upd, R u + t) per residue."""
    return np.einsum("nab,nbc->nac", R, R_upd), np.einsum("nab,nb->na", R, u) + t


def invariant_point_attention(s, zn, R, t, seq_mask, w, heads, c, n_qp, n_pv, return_weights=False):
    """M.2 -> IPA_i [N, c_s]."""
    s, zn = _f64(s), _f64(zn)
    N = s.shape[0]
    H = heads
    q = linear(s, w["w_q"]).reshape(N, H, c)
    k = linear(s, w["w_k"]).reshape(N, H, c)
    v = linear(s, w["w_v"]).reshape(N, H, c)
    qp = linear(s, w["w_qp"]).reshape(N, H, n_qp, 3)
    kp = linear(s, w["w_kp"]).reshape(N, H, n_qp, 3)
    vp = linear(s, w["w_vp"]).reshape(N, H, n_pv, 3)
    b = linear(zn, w["w_b"])                                            # [N, N, H]
    qg = np.einsum("nab,nhpb->nhpa", R, qp) + t[:, None, None, :]
    kg = np.einsum("nab,nhpb->nhpa", R, kp) + t[:, None, None, :]
    vg = np.einsum("nab,nhpb->nhpa", R, vp) + t[:, None, None, :]
    w_c = np.sqrt(2.0 / (9.0 * n_qp))
    w_l = np.sqrt(1.0 / 3.0)
    gamma = softplus(w["g_head"])                                       # [H]
    qk = np.einsum("ihc,jhc->hij", q, k) / np.sqrt(c)
    d2 = ((qg[:, None] - kg[None, :]) ** 2).sum(axis=(-1, -2))          # [N(i), N(j), H]
    logits = w_l * (qk + np.transpose(b, (2, 0, 1)) - (gamma * w_c / 2.0)[:, None, None] * np.transpose(d2, (2, 0, 1)))
    logits = logits + NEG_INF_SCALE * (_f64(seq_mask)[None, None, :] - 1.0)
    a = softmax(logits, axis=-1)                                        # [H, N, N]
    ot = np.einsum("hij,ijc->ihc", a, zn)                               # [N, H, c_z]
    o = np.einsum("hij,jhc->ihc", a, v)                                 # [N, H, c]
    og = np.einsum("hij,jhpa->ihpa", a, vg)                             # [N, H, P_v, 3] global
    op = np.einsum("nba,nhpb->nhpa", R, og - t[:, None, None, :])       # R^T (og - t)
    nrm = np.sqrt((op ** 2).sum(axis=-1) + IPA_NORM_EPS)                # [N, H, P_v]
    cat = np.concatenate([ot.reshape(N, -1), o.reshape(N, -1), op.reshape(N, -1), nrm.reshape(N, -1)], axis=-1)
    out = linear(cat, w["w_out"], w["b_out"])
    return (out, a) if return_weights else out


def structure_transition(s, w):
    """M.3, second half: Lin_3(relu(Lin_2(relu(Lin_1(s)))))."""
    h = relu(linear(s, w["w_t1"], w["b_t1"]))
    h = relu(linear(h, w["w_t2"], w["b_t2"]))
    return linear(h, w["w_t3"], w["b_t3"])


def backbone_update(s, R, t, w):
    """M.4 -> (R, t)."""
    y = linear(s, w["w_bb"], w["b_bb"])                                 # [N, 6]
    return compose_frames(R, t, quat_to_rot(y[:, 0], y[:, 1], y[:, 2]), y[:, 3:6])


def torsion_angles(s, s_init, w, n_torsion):
    """M.5 -> alpha_hat [N, n_torsion, 2]."""
    a = linear(s, w["w_a1"], w["b_a1"]) + linear(s_init, w["w_a2"], w["b_a2"])
    for r in (1, 2):
        a = a + linear(relu(linear(relu(a), w[f"w_r{r}a"], w[f"b_r{r}a"])), w[f"w_r{r}b"], w[f"b_r{r}b"])
    alpha = linear(relu(a), w["w_alpha"], w["b_alpha"]).reshape(-1, n_torsion, 2)
    return alpha / np.sqrt((alpha ** 2).sum(axis=-1, keepdims=True) + ANGLE_EPS)


def single_representation(m0, w):
    """M.0."""
    return linear(m0, w["w_single"], w["b_single"])


def structure_module(m0, z, seq_mask, w, heads=12, c=16, n_qp=4, n_pv=8, n_layers=8, n_torsion=7, pos_scale=10.0,
                     frames=None):
    """M.0-M.6 for one protein -> dict(s, R, t, x, alpha, s_init).  frames = (R, t) replaces the identity start (tests)."""
    s_init = layer_norm(single_representation(m0, w), w["ln_s_g"], w["ln_s_b"])
    zn = layer_norm(z, w["ln_z_g"], w["ln_z_b"])
    s = linear(s_init, w["w_in"], w["b_in"])
    N = s.shape[0]
    if frames is None:
        R, t = np.tile(np.eye(3), (N, 1, 1)), np.zeros((N, 3))
    else:
        R, t = _f64(frames[0]).copy(), _f64(frames[1]).copy()
    for _ in range(n_layers):
        s = layer_norm(s + invariant_point_attention(s, zn, R, t, seq_mask, w, heads, c, n_qp, n_pv),
                       w["ln_ipa_g"], w["ln_ipa_b"])
        s = layer_norm(s + structure_transition(s, w), w["ln_tr_g"], w["ln_tr_b"])
        R, t = backbone_update(s, R, t, w)
    alpha = torsion_angles(s, s_init, w, n_torsion)
    return {"s": s, "R": R, "t": t, "x": pos_scale * t, "alpha": alpha, "s_init": s_init}


def distogram_logits(z, w):
    """H.1."""
    half = linear(z, w["w_dg"], w["b_dg"])
    return half + np.transpose(half, (1, 0, 2))


def masked_msa_logits(m, w):
    """H.2."""
    return linear(m, w["w_mm"], w["b_mm"])


def plddt(s, w):
    """H.3 -> (logits [N, n_bins], plddt [N])."""
    h = layer_norm(s, w["ln_l_g"], w["ln_l_b"])
    h = relu(linear(h, w["w_l1"], w["b_l1"]))
    h = relu(linear(h, w["w_l2"], w["b_l2"]))
    logits = linear(h, w["w_l3"], w["b_l3"])
    nb = logits.shape[-1]
    centers = (np.arange(nb, dtype=F64) + 0.5) / nb
    return logits, 100.0 * (softmax(logits, axis=-1) * centers).sum(axis=-1)


def pae_logits(z, w):
    """H.4."""
    return linear(z, w["w_pae"], w["b_pae"])


def resolved_logits(s, w):
    """H.5."""
    return linear(s, w["w_er"], w["b_er"])


def fold(target_feat, residue_index, msa_feat, seq_mask, msa_mask, w_embed, blocks, w_struct, n_cycles, x_prev0=None,
         x_forced=None, head_dim=32, extra=None, struct_kw=None, **embed_kw):
    """The whole GPU stage for one protein: n_cycles x (E.1, E.2 with the previous cycle's first MSA
    row, pair representation and structure-module positions, [extra-MSA stack], trunk, M.0-M.6).
    x_prev0 [N,3] or None: positions the first cycle's recycling embedder sees (None = no bin set).
    x_forced: optional list of n_cycles - 1 position arrays used INSTEAD of this function's own positions as the recycling
    input of cycles 1 .. n_cycles-1.  The distance bins are a floating-point comparison deciding an integer; a checker hands
    in the positions the other implementation produced so that both sides decide on the same numbers.
    -> dict(m, z, x_cycles [n_cycles, N, 3], and the last cycle's structure_module outputs)."""
    from .embed_ref import embed_cycle, extra_msa_embedder
    from .evoformer_ref import evoformer_trunk
    from .extra_msa_ref import extra_msa_stack
    N = np.asarray(msa_feat).shape[1]
    c_m, c_z = np.asarray(w_embed["w_m"]).shape[1], np.asarray(w_embed["w_a"]).shape[1]
    m0_prev, z_prev = np.zeros((N, c_m)), np.zeros((N, N, c_z))
    x_prev = np.zeros((N, 3)) if x_prev0 is None else x_prev0
    xs, out, m, z = [], None, None, None
    for cyc in range(n_cycles):
        m, z = embed_cycle(target_feat, residue_index, msa_feat, m0_prev, z_prev, x_prev, w_embed, **embed_kw)
        if extra is not None:
            xf, xmask, xblocks, xhd = extra
            _, z = extra_msa_stack(extra_msa_embedder(xf, w_embed), z, seq_mask, xmask, xblocks, xhd, head_dim)
        m, z = evoformer_trunk(m, z, seq_mask, msa_mask, blocks, head_dim)
        out = structure_module(m[0], z, seq_mask, w_struct, **(struct_kw or {}))
        xs.append(out["x"])
        m0_prev, z_prev = m[0], z
        x_prev = out["x"] if x_forced is None or cyc >= len(x_forced) else x_forced[cyc]
    res = dict(out)
    res.update(m=m, z=z, x_cycles=np.stack(xs))
    return res
