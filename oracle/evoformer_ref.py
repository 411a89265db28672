"""fp64 CPU oracle of one Evoformer block (TEST INFRASTRUCTURE — not part of the product path).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this package.  It shares no code with ``paper_2111_06340_b200`` (the CUDA path) and
never imports it.  Everything is plain numpy in float64; a matmul / einsum is the only library
primitive used as a step.  No blocking, fusion or reordering: logits and softmax weights are
materialised in full, sums are written as the definition states them.

What it computes: the Evoformer trunk named at PAPER.md:27 and PAPER.md:61 (AlphaFold v2.0.1 monomer,
PAPER.md:127), in the reading SURVEY.md Appendix A.1-A.9 gives of it (the paper itself prints no
formula; readings R0-R16 of SURVEY.md §8(c) apply and are listed in DESIGN.md).  Each function
below cites the Appendix-A item it follows and uses its notation:
    m[s,i,:]  MSA representation,  z[i,j,:]  pair representation (one protein, no batch axis),
    sigma_i = seq_mask, rho_s = msa_mask, mu_si = rho_s sigma_i, pi_ij = sigma_i sigma_j,
    NEG(mask) = 1e9 (mask - 1), head h owns columns [h d, (h+1) d).

Pins (tests/test_oracle_*.py, ``-m "not gpu"``): library routines (torch layer_norm /
scaled_dot_product_attention in fp64), closed forms (S=1 outer product, N=1 triangle update, W_q=0
uniform attention), index-by-index pure-Python loops on tiny inputs, the transposition identities
A.6/A.8, padding invariance, MSA-row permutation, softmax normalisation, zero-output-weights identity.
Parity with DeepMind's AlphaFold itself: **parity unpinned** (no trained weights, code or supplement
on this box); only the Appendix-A reading is pinned.
"""
from __future__ import annotations

import numpy as np

NEG_INF_SCALE = 1e9      # R3: additive mask 1e9 * (mask - 1)
LN_EPS = 1e-5            # R4
OPM_EPS = 1e-3           # R5

F64 = np.float64


def _f64(x):
    return np.asarray(x, dtype=F64)


# ----------------------------------------------------------------------------------------------
# primitives
# ----------------------------------------------------------------------------------------------

def layer_norm(x, gamma, beta, eps=LN_EPS):
    """R4: biased variance over the channel axis, eps inside the sqrt, affine gamma/beta."""
    x = _f64(x)
    mean = x.mean(axis=-1, keepdims=True)
    var = ((x - mean) ** 2).mean(axis=-1, keepdims=True)
    return (x - mean) / np.sqrt(var + eps) * _f64(gamma) + _f64(beta)


def linear(x, w, b=None):
    """Lin(x) = x W + b with W row-major [in, out] (Appendix B); Lin0 when b is None."""
    y = _f64(x) @ _f64(w)
    if b is not None:
        y = y + _f64(b)
    return y


def sigmoid(x):
    x = _f64(x)
    return 1.0 / (1.0 + np.exp(-x))


def softmax(logits, axis=-1):
    logits = _f64(logits)
    e = np.exp(logits - logits.max(axis=axis, keepdims=True))
    return e / e.sum(axis=axis, keepdims=True)


def neg(mask):
    """NEG(mask) = 1e9 (mask - 1)  (R3)."""
    return NEG_INF_SCALE * (_f64(mask) - 1.0)


# ----------------------------------------------------------------------------------------------
# gated attention core shared by A.1 / A.2 / A.7 / A.8 in its plain form
# ----------------------------------------------------------------------------------------------

def gated_attention_weights(q, k, bias, key_mask, head_dim):
    """P[r,h,i,j] = softmax_j( q[r,i,h].k[r,j,h]/sqrt(d) + bias[h,i,j] + NEG(key_mask[r,j]) ).

    q, k: [R, L, H*d]; bias: [H, L, L] or None; key_mask: [R, L].  R12: scale before the bias.
    """
    R, L, C = q.shape
    H = C // head_dim
    qh = _f64(q).reshape(R, L, H, head_dim)
    kh = _f64(k).reshape(R, L, H, head_dim)
    logits = np.einsum("rihd,rjhd->rhij", qh, kh) / np.sqrt(float(head_dim))
    if bias is not None:
        logits = logits + _f64(bias)[None, :, :, :]
    logits = logits + neg(key_mask)[:, None, None, :]
    return softmax(logits, axis=-1)


def gated_attention(x, bias, key_mask, w, head_dim):
    """o[r,i] = Lin_o( concat_h G[r,i,h] (.) sum_j P[r,h,i,j] v[r,j,h] )  for x: [R, L, C]."""
    R, L, C = x.shape
    q = linear(x, w["wq"])
    k = linear(x, w["wk"])
    v = linear(x, w["wv"])
    gate = sigmoid(linear(x, w["wg"], w["bg"]))
    H = q.shape[-1] // head_dim
    P = gated_attention_weights(q, k, bias, key_mask, head_dim)
    vh = v.reshape(R, L, H, head_dim)
    o = np.einsum("rhij,rjhd->rihd", P, vh).reshape(R, L, H * head_dim)
    return linear(gate * o, w["wo"], w["bo"])


# ----------------------------------------------------------------------------------------------
# A.1 - A.9
# ----------------------------------------------------------------------------------------------

def msa_row_attention(m, z, seq_mask, msa_mask, w, head_dim=32):
    """A.1  m[s,i] += Lin(concat_h G (.) sum_j softmax_j(q.k/sqrt d + beta[h,i,j] + NEG(mu_sj)) v)."""
    m, z = _f64(m), _f64(z)
    x = layer_norm(m, w["ln_g"], w["ln_b"])
    y = layer_norm(z, w["ln_z_g"], w["ln_z_b"])
    beta = np.transpose(linear(y, w["w_bias"]), (2, 0, 1))          # [H, i, j]
    mu = _f64(msa_mask)[:, None] * _f64(seq_mask)[None, :]            # mu[s, j]
    return m + gated_attention(x, beta, mu, w, head_dim)


def msa_col_attention(m, seq_mask, msa_mask, w, head_dim=32):
    """A.2  attention along s for every residue i: keys t masked by mu_ti, no bias."""
    m = _f64(m)
    x = layer_norm(m, w["ln_g"], w["ln_b"])
    xt = np.transpose(x, (1, 0, 2))                                   # [i, s, c]
    mu_t = _f64(seq_mask)[:, None] * _f64(msa_mask)[None, :]          # mu[i, t] = rho_t sigma_i
    upd = gated_attention(xt, None, mu_t, w, head_dim)               # [i, s, c]
    return m + np.transpose(upd, (1, 0, 2))


def transition(x, w):
    """A.3 / A.9  x += Lin2(relu(Lin1(LN(x))))."""
    x = _f64(x)
    h = linear(layer_norm(x, w["ln_g"], w["ln_b"]), w["w1"], w["b1"])
    return x + linear(np.maximum(h, 0.0), w["w2"], w["b2"])


def outer_product_mean(m, z, seq_mask, msa_mask, w):
    """A.4  z[i,j] += Lin_out( vec(sum_s a[s,i] (x) b[s,j]) / (1e-3 + n_ij) ), vec index c1*c_opm + c2 (R5, R6)."""
    m, z = _f64(m), _f64(z)
    S, N, _ = m.shape
    x = layer_norm(m, w["ln_g"], w["ln_b"])
    mu = _f64(msa_mask)[:, None] * _f64(seq_mask)[None, :]            # [s, i]
    a = mu[:, :, None] * linear(x, w["wa"], w["ba"])                  # [s, i, c1]
    b = mu[:, :, None] * linear(x, w["wb"], w["bb"])                  # [s, j, c2]
    c = a.shape[-1]
    O = np.einsum("sic,sjd->ijcd", a, b).reshape(N, N, c * c)
    n = np.einsum("si,sj->ij", mu, mu)
    return z + linear(O / (OPM_EPS + n)[:, :, None], w["wout"], w["bout"])


def _tri_mul_ab_g(z, seq_mask, w):
    x = layer_norm(z, w["ln_in_g"], w["ln_in_b"])
    pi = _f64(seq_mask)[:, None] * _f64(seq_mask)[None, :]
    a = pi[:, :, None] * sigmoid(linear(x, w["w_ag"], w["b_ag"])) * linear(x, w["w_ap"], w["b_ap"])
    b = pi[:, :, None] * sigmoid(linear(x, w["w_bg"], w["b_bg"])) * linear(x, w["w_bp"], w["b_bp"])
    g = sigmoid(linear(x, w["w_g"], w["b_g"]))
    return a, b, g


def triangle_mult_outgoing(z, seq_mask, w):
    """A.5  t[i,j,c] = sum_k a[i,k,c] b[j,k,c];  z[i,j] += g[i,j] (.) Lin_z(LN_out(t[i,j]))."""
    z = _f64(z)
    a, b, g = _tri_mul_ab_g(z, seq_mask, w)
    t = np.einsum("ikc,jkc->ijc", a, b)
    return z + g * linear(layer_norm(t, w["ln_out_g"], w["ln_out_b"]), w["w_z"], w["b_z"])


def triangle_mult_incoming(z, seq_mask, w):
    """A.6  as A.5 with t[i,j,c] = sum_k a[k,i,c] b[k,j,c]."""
    z = _f64(z)
    a, b, g = _tri_mul_ab_g(z, seq_mask, w)
    t = np.einsum("kic,kjc->ijc", a, b)
    return z + g * linear(layer_norm(t, w["ln_out_g"], w["ln_out_b"]), w["w_z"], w["b_z"])


def triangle_attention_start(z, seq_mask, w, head_dim=32):
    """A.7  L[i,h,j,k] = q[i,j,h].k[i,k,h]/sqrt d + beta[h,j,k] + NEG(pi_ik); softmax over k."""
    z = _f64(z)
    x = layer_norm(z, w["ln_g"], w["ln_b"])
    beta = np.transpose(linear(x, w["w_bias"]), (2, 0, 1))            # beta[h, j, k]
    pi = _f64(seq_mask)[:, None] * _f64(seq_mask)[None, :]            # pi[i, k]
    return z + gated_attention(x, beta, pi, w, head_dim)


def triangle_attention_end(z, seq_mask, w, head_dim=32):
    """A.8  L[i,j,h,k] = q[i,j,h].k[k,j,h]/sqrt d + beta[h,k,i] + NEG(pi_kj); softmax over k;
    o[i,j,h] = G[i,j,h] (.) sum_k P v[k,j,h].  Written directly in the index form (not via A.7)."""
    z = _f64(z)
    N = z.shape[0]
    x = layer_norm(z, w["ln_g"], w["ln_b"])
    q = linear(x, w["wq"])
    k = linear(x, w["wk"])
    v = linear(x, w["wv"])
    gate = sigmoid(linear(x, w["wg"], w["bg"]))
    H = q.shape[-1] // head_dim
    beta = linear(x, w["w_bias"])                                     # beta[a, b, h] from x[a, b]
    qh = q.reshape(N, N, H, head_dim)
    kh = k.reshape(N, N, H, head_dim)
    vh = v.reshape(N, N, H, head_dim)
    logits = np.einsum("ijhd,kjhd->ijhk", qh, kh) / np.sqrt(float(head_dim))
    logits = logits + np.transpose(beta, (1, 2, 0))[:, None, :, :]    # [i, 1, h, k] <- beta[k, i, h]
    pi = _f64(seq_mask)[:, None] * _f64(seq_mask)[None, :]            # pi[k, j]
    logits = logits + np.transpose(neg(pi), (1, 0))[None, :, None, :]  # [1, j, 1, k] <- NEG(pi[k, j])
    P = softmax(logits, axis=-1)
    o = np.einsum("ijhk,kjhd->ijhd", P, vh).reshape(N, N, H * head_dim)
    return z + linear(gate * o, w["wo"], w["bo"])


# ----------------------------------------------------------------------------------------------
# block and trunk
# ----------------------------------------------------------------------------------------------

SUBSTEPS = ("row", "col", "msa_trans", "opm", "tri_mul_out", "tri_mul_in",
            "tri_att_start", "tri_att_end", "pair_trans")


def substep(step, m, z, seq_mask, msa_mask, w, head_dim=32):
    """Apply sub-step ``step`` (1..9, SURVEY.md §8(a) order) of one block; returns (m, z)."""
    m, z = _f64(m), _f64(z)
    if step == 1:
        m = msa_row_attention(m, z, seq_mask, msa_mask, w["row"], head_dim)
    elif step == 2:
        m = msa_col_attention(m, seq_mask, msa_mask, w["col"], head_dim)
    elif step == 3:
        m = transition(m, w["msa_trans"])
    elif step == 4:
        z = outer_product_mean(m, z, seq_mask, msa_mask, w["opm"])
    elif step == 5:
        z = triangle_mult_outgoing(z, seq_mask, w["tri_mul_out"])
    elif step == 6:
        z = triangle_mult_incoming(z, seq_mask, w["tri_mul_in"])
    elif step == 7:
        z = triangle_attention_start(z, seq_mask, w["tri_att_start"], head_dim)
    elif step == 8:
        z = triangle_attention_end(z, seq_mask, w["tri_att_end"], head_dim)
    elif step == 9:
        z = transition(z, w["pair_trans"])
    else:
        raise ValueError(f"substep {step} not in 1..9")
    return m, z


def evoformer_block(m, z, seq_mask, msa_mask, w, head_dim=32):
    """One block: A.1, A.2, A.3 on m; A.4 reads the updated m; A.5 .. A.9 on z (R0 ordering)."""
    for step in range(1, 10):
        m, z = substep(step, m, z, seq_mask, msa_mask, w, head_dim)
    return m, z


def evoformer_trunk(m, z, seq_mask, msa_mask, blocks, head_dim=32):
    """n_blocks blocks with distinct weights, one protein."""
    for w in blocks:
        m, z = evoformer_block(m, z, seq_mask, msa_mask, w, head_dim)
    return m, z


def evoformer_trunk_batched(msa, pair, seq_mask, msa_mask, blocks, head_dim=32):
    """Batch wrapper: proteins are independent."""
    ms, zs = [], []
    for b in range(msa.shape[0]):
        m, z = evoformer_trunk(msa[b], pair[b], seq_mask[b], msa_mask[b], blocks, head_dim)
        ms.append(m)
        zs.append(z)
    return np.stack(ms), np.stack(zs)
