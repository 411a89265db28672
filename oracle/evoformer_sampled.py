"""Sampled-output fp64 oracle (TEST INFRASTRUCTURE — not part of the product path).

``evoformer_ref`` evaluates a sub-step for every position; at the benchmarked sizes (N_seq 512, N_res
384 / 768: BASELINE.json configs[2..4]) that is minutes of fp64 work per block (SURVEY.md §8(c)
"Feasibility").  The functions here evaluate the SAME Appendix-A formulas for ONE output position:
given the sub-step's input tensors they return the updated m[s,i,:] (sub-steps 1-3) or z[i,j,:]
(sub-steps 4-9).  Each is the definition written out for that position, in the notation of
``evoformer_ref`` (sigma, rho, mu, pi, NEG, head h owns columns [h d, (h+1) d)); the only library
steps are matmuls.  Pin: ``tests/test_oracle_sampled.py`` compares every function with the
full-tensor oracle at every position of small ragged problems (<= 1e-12), so each inherits the pins
of ``evoformer_ref``.

Optional switch ``rnd`` (reading R16, "quantisation-aware oracle"): a ``Rounding`` object rounds
intermediate values at the points where the bf16 CUDA path stores them in 16 bits (R17:
LayerNorm outputs, gates, pair bias, outer-product and triangle operands and results fp16; q, k, v, P, o,
transition hidden bf16).  The arithmetic between those points stays fp64.  With ``rnd=None`` (the
default) no rounding happens and the functions ARE the plain oracle; the switch exists so that a
difference GPU - oracle can be split into the part the storage formats cause by themselves
(quantised - plain) and the rest (GPU - quantised).  The quantised mode is a model of the storage
formats, not a definition of correct; tolerances are always checked against the plain mode.
"""
from __future__ import annotations

import numpy as np

from .evoformer_ref import F64, OPM_EPS, _f64, layer_norm, linear, neg, sigmoid, softmax

LOG2E = 1.4426950408889634


class Rounding:
    """Storage-format rounding (R16 / R17).  ``Rounding(False)`` is the identity."""

    def __init__(self, on=True):
        self.on = bool(on)

    def f16(self, x):
        """Round to the nearest IEEE fp16 value (ties to even), returned as fp64."""
        if not self.on:
            return _f64(x)
        return np.asarray(x, dtype=np.float16).astype(F64)

    def bf16(self, x):
        """Round to the nearest bfloat16 value (ties to even) through fp32, returned as fp64."""
        if not self.on:
            return _f64(x)
        a = np.ascontiguousarray(x, dtype=np.float32)
        u = a.view(np.uint32).astype(np.uint64)
        u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
        return u.astype(np.uint32).view(np.float32).reshape(a.shape).astype(F64)

    def gate(self, pre):
        """sigmoid of a gate pre-activation, held in fp16 (R17).  The CUDA path rounds the pre-activation to fp16 and
        evaluates 0.5 + 0.5 tanh(x / 2) in fp16 arithmetic; modelled as fp16(pre) -> exact sigmoid -> fp16."""
        if not self.on:
            return sigmoid(pre)
        return self.f16(sigmoid(self.f16(pre)))


PLAIN = Rounding(False)


def _ln(x, g, b, r):
    """LayerNorm output as the MMA operand: fp16 on the quantised path (R17)."""
    return r.f16(layer_norm(x, g, b))


def _lin(x, w, b, r):
    """Linear fed by a LayerNorm output: its weight matrix is an fp16 operand too (R17; exact for bf16-rounded weights in
    the fp16 normal range)."""
    return linear(x, r.f16(w), b)


# ----------------------------------------------------------------------------------------------
# one query of the gated attention shared by A.1 / A.2 / A.7 / A.8
# ----------------------------------------------------------------------------------------------

def _gated_attention_one_query(xq, xk, beta_q, key_mask, w, head_dim, r):
    """Lin_o( concat_h G_h (.) sum_j softmax_j( q_h.k_jh / sqrt(d) + beta_q[j,h] + NEG(key_mask_j) ) v_jh ).

    xq: [C] LayerNorm output at the query position; xk: [L, C] at the L key positions; beta_q: [L, H] pair bias of this
    query towards every key, or None; key_mask: [L].  R12: scale before the bias.
    """
    L, C = xk.shape
    H = C // head_dim
    q = _lin(xq, w["wq"], None, r)
    k = r.bf16(_lin(xk, w["wk"], None, r))
    v = r.bf16(_lin(xk, w["wv"], None, r))
    gate = r.gate(_lin(xq, w["wg"], w["bg"], r))
    if r.on:
        # storage points of the CUDA path: q carries log2(e)/sqrt(d) (bf16), the bias log2(e) (fp16); the softmax runs in the
        # exp2 domain — the same real function (R12)
        q = r.bf16(q * (LOG2E / np.sqrt(float(head_dim)))) / LOG2E * np.sqrt(float(head_dim))
        if beta_q is not None:
            beta_q = r.f16(_f64(beta_q) * LOG2E) / LOG2E
    o = np.zeros(C, dtype=F64)
    for h in range(H):
        cols = slice(h * head_dim, (h + 1) * head_dim)
        logits = k[:, cols] @ q[cols] / np.sqrt(float(head_dim))
        if beta_q is not None:
            logits = logits + _f64(beta_q)[:, h]
        logits = logits + neg(key_mask)
        if r.on:
            # P is stored as bf16 un-normalised (exp of logit - max), the normaliser is the fp32 sum of the unrounded terms
            e = np.exp(logits - logits.max())
            o[cols] = (r.bf16(e) @ v[:, cols]) / e.sum()
        else:
            o[cols] = softmax(logits) @ v[:, cols]
    o = r.bf16(gate * o)
    return linear(o, w["wo"], w["bo"])


# ----------------------------------------------------------------------------------------------
# A.1 - A.9 at one output position
# ----------------------------------------------------------------------------------------------

def msa_row_attention_at(m, z, seq_mask, msa_mask, w, s, i, head_dim=32, rnd=None):
    """A.1 at (s, i): keys are the residues j of MSA row s; beta[h,i,j] = Lin0(LN'(z[i,j]))_h; key mask mu_sj."""
    r = rnd or PLAIN
    x = _ln(m[s], w["ln_g"], w["ln_b"], r)                            # [N, c_m]: row s
    y = _ln(z[i], w["ln_z_g"], w["ln_z_b"], r)                        # [N, c_z]: pair row i
    beta = _lin(y, w["w_bias"], None, r)                              # beta[j, h]
    mu = _f64(msa_mask)[s] * _f64(seq_mask)                           # mu[s, j]
    return _f64(m[s, i]) + _gated_attention_one_query(x[i], x, beta, mu, w, head_dim, r)


def msa_col_attention_at(m, seq_mask, msa_mask, w, s, i, head_dim=32, rnd=None):
    """A.2 at (s, i): keys are the sequences t of MSA column i; no bias; key mask mu_ti = rho_t sigma_i."""
    r = rnd or PLAIN
    x = _ln(m[:, i], w["ln_g"], w["ln_b"], r)                         # [S, c_m]: column i
    mu = _f64(msa_mask) * _f64(seq_mask)[i]
    return _f64(m[s, i]) + _gated_attention_one_query(x[s], x, None, mu, w, head_dim, r)


def transition_at(x_row, w, rnd=None):
    """A.3 / A.9 for one row: x + Lin2(relu(Lin1(LN(x))))."""
    r = rnd or PLAIN
    h = _lin(_ln(x_row, w["ln_g"], w["ln_b"], r), w["w1"], w["b1"], r)
    return _f64(x_row) + linear(r.bf16(np.maximum(h, 0.0)), w["w2"], w["b2"])


def outer_product_mean_at(m, z, seq_mask, msa_mask, w, i, j, rnd=None):
    """A.4 at (i, j): z[i,j] + Lin_out( vec(sum_s a[s,i] (x) b[s,j]) / (1e-3 + n_ij) ), vec index c1*c_opm + c2."""
    r = rnd or PLAIN
    rho, sg = _f64(msa_mask), _f64(seq_mask)
    xi = _ln(m[:, i], w["ln_g"], w["ln_b"], r)                        # [S, c_m]
    xj = _ln(m[:, j], w["ln_g"], w["ln_b"], r)
    a = r.f16((rho * sg[i])[:, None] * _lin(xi, w["wa"], w["ba"], r))   # a[s, c1] = mu_si Lin_a(x[s,i])
    b = r.f16((rho * sg[j])[:, None] * _lin(xj, w["wb"], w["bb"], r))   # b[s, c2] = mu_sj Lin_b(x[s,j])
    O = r.f16(a.T @ b)                                                # O[c1, c2] = sum_s a[s,c1] b[s,c2]
    n = float(np.sum((rho * sg[i]) * (rho * sg[j])))
    if r.on:
        # the CUDA path contracts the 16-bit outer product with W_out first and divides afterwards (the same by linearity)
        return _f64(z[i, j]) + linear(O.reshape(-1), w["wout"]) / (OPM_EPS + n) + _f64(w["bout"])
    return _f64(z[i, j]) + linear(O.reshape(-1) / (OPM_EPS + n), w["wout"], w["bout"])


def _tri_operand(x, pi, wp, bp, wg, bg, r):
    """pi (.) sigmoid(Lin_g(x)) (.) Lin_p(x) for the rows of x ([L, c_z]) with pair masks pi ([L])."""
    return r.f16(pi[:, None] * sigmoid(_lin(x, wg, bg, r)) * _lin(x, wp, bp, r))


def triangle_mult_outgoing_at(z, seq_mask, w, i, j, rnd=None):
    """A.5 at (i, j): t[c] = sum_k a[i,k,c] b[j,k,c];  z[i,j] + g[i,j] (.) Lin_z(LN_out(t))."""
    r = rnd or PLAIN
    sg = _f64(seq_mask)
    xi = _ln(z[i], w["ln_in_g"], w["ln_in_b"], r)                     # rows (i, k), all k
    xj = _ln(z[j], w["ln_in_g"], w["ln_in_b"], r)                     # rows (j, k)
    a = _tri_operand(xi, sg[i] * sg, w["w_ap"], w["b_ap"], w["w_ag"], w["b_ag"], r)   # a[k, c] = a[i,k,c]
    b = _tri_operand(xj, sg[j] * sg, w["w_bp"], w["b_bp"], w["w_bg"], w["b_bg"], r)   # b[k, c] = b[j,k,c]
    t = r.f16(np.sum(a * b, axis=0))
    g = r.gate(_lin(xi[j], w["w_g"], w["b_g"], r))
    return _f64(z[i, j]) + g * _lin(_ln(t, w["ln_out_g"], w["ln_out_b"], r), w["w_z"], w["b_z"], r)


def triangle_mult_incoming_at(z, seq_mask, w, i, j, rnd=None):
    """A.6 at (i, j): t[c] = sum_k a[k,i,c] b[k,j,c]."""
    r = rnd or PLAIN
    sg = _f64(seq_mask)
    xi = _ln(z[:, i], w["ln_in_g"], w["ln_in_b"], r)                  # rows (k, i), all k
    xj = _ln(z[:, j], w["ln_in_g"], w["ln_in_b"], r)                  # rows (k, j)
    a = _tri_operand(xi, sg * sg[i], w["w_ap"], w["b_ap"], w["w_ag"], w["b_ag"], r)   # a[k, c] = a[k,i,c]
    b = _tri_operand(xj, sg * sg[j], w["w_bp"], w["b_bp"], w["w_bg"], w["b_bg"], r)   # b[k, c] = b[k,j,c]
    t = r.f16(np.sum(a * b, axis=0))
    xij = _ln(z[i, j], w["ln_in_g"], w["ln_in_b"], r)
    g = r.gate(_lin(xij, w["w_g"], w["b_g"], r))
    return _f64(z[i, j]) + g * _lin(_ln(t, w["ln_out_g"], w["ln_out_b"], r), w["w_z"], w["b_z"], r)


def triangle_attention_start_at(z, seq_mask, w, i, j, head_dim=32, rnd=None):
    """A.7 at (i, j): keys k along row i; L[h,k] = q[i,j,h].k[i,k,h]/sqrt d + beta[h,j,k] + NEG(pi_ik)."""
    r = rnd or PLAIN
    sg = _f64(seq_mask)
    xi = _ln(z[i], w["ln_g"], w["ln_b"], r)                           # rows (i, k)
    xj = _ln(z[j], w["ln_g"], w["ln_b"], r)                           # rows (j, k): beta[h,j,k] = Lin0(x[j,k])_h
    beta = _lin(xj, w["w_bias"], None, r)                             # beta[k, h]
    return _f64(z[i, j]) + _gated_attention_one_query(xi[j], xi, beta, sg[i] * sg, w, head_dim, r)


def triangle_attention_end_at(z, seq_mask, w, i, j, head_dim=32, rnd=None):
    """A.8 at (i, j): keys k along column j; L[h,k] = q[i,j,h].k[k,j,h]/sqrt d + beta[h,k,i] + NEG(pi_kj)."""
    r = rnd or PLAIN
    sg = _f64(seq_mask)
    xj = _ln(z[:, j], w["ln_g"], w["ln_b"], r)                        # rows (k, j)
    xi = _ln(z[:, i], w["ln_g"], w["ln_b"], r)                        # rows (k, i): beta[h,k,i] = Lin0(x[k,i])_h
    beta = _lin(xi, w["w_bias"], None, r)                             # beta[k, h]
    return _f64(z[i, j]) + _gated_attention_one_query(xj[i], xj, beta, sg * sg[j], w, head_dim, r)


def substep_at(step, m, z, seq_mask, msa_mask, w, pos, head_dim=32, rnd=None):
    """Output of sub-step ``step`` (1..9, SURVEY.md §8(a) order) of one block at one position of one protein:
    pos = (s, i) -> updated m[s,i,:] for steps 1-3; pos = (i, j) -> updated z[i,j,:] for steps 4-9."""
    p, q = int(pos[0]), int(pos[1])
    if step == 1:
        return msa_row_attention_at(m, z, seq_mask, msa_mask, w["row"], p, q, head_dim, rnd)
    if step == 2:
        return msa_col_attention_at(m, seq_mask, msa_mask, w["col"], p, q, head_dim, rnd)
    if step == 3:
        return transition_at(m[p, q], w["msa_trans"], rnd)
    if step == 4:
        return outer_product_mean_at(m, z, seq_mask, msa_mask, w["opm"], p, q, rnd)
    if step == 5:
        return triangle_mult_outgoing_at(z, seq_mask, w["tri_mul_out"], p, q, rnd)
    if step == 6:
        return triangle_mult_incoming_at(z, seq_mask, w["tri_mul_in"], p, q, rnd)
    if step == 7:
        return triangle_attention_start_at(z, seq_mask, w["tri_att_start"], p, q, head_dim, rnd)
    if step == 8:
        return triangle_attention_end_at(z, seq_mask, w["tri_att_end"], p, q, head_dim, rnd)
    if step == 9:
        return transition_at(z[p, q], w["pair_trans"], rnd)
    raise ValueError(f"substep {step} not in 1..9")


def substep_all(step, m, z, seq_mask, msa_mask, w, head_dim=32, rnd=None):
    """The whole sub-step through ``substep_at`` at every position (small problems only: quantisation-aware block floors)."""
    m, z = _f64(m), _f64(z)
    if step <= 3:
        out = np.empty_like(m)
        for s in range(m.shape[0]):
            for i in range(m.shape[1]):
                out[s, i] = substep_at(step, m, z, seq_mask, msa_mask, w, (s, i), head_dim, rnd)
        return out, z
    out = np.empty_like(z)
    for i in range(z.shape[0]):
        for j in range(z.shape[1]):
            out[i, j] = substep_at(step, m, z, seq_mask, msa_mask, w, (i, j), head_dim, rnd)
    return m, out


def block_all(m, z, seq_mask, msa_mask, w, head_dim=32, rnd=None):
    """One block, sub-steps 1..9 in order, every position through ``substep_at``."""
    for step in range(1, 10):
        m, z = substep_all(step, m, z, seq_mask, msa_mask, w, head_dim, rnd)
    return m, z
