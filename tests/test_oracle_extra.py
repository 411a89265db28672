"""Pins of oracle/extra_msa_ref.py: the global column attention X.2 (everything else in the extra-MSA block is a main-block
function at other dimensions and carries those pins)."""
import math

import numpy as np
import pytest

import pf_synth as ps
from oracle import evoformer_ref as ref
from oracle import extra_msa_ref as ex

D = ps.EXTRA


@pytest.fixture(scope="module")
def case():
    S, N = 6, 5
    w = ps.make_extra_weights(111, 1)[0]
    e, z, _, _ = ps.make_extra_inputs(112, 1, S, N)
    sig = np.array([1.0, 1, 0, 1, 1])
    rho = np.array([1.0, 0, 1, 1, 0, 1])
    return w, e[0].astype(np.float64), z[0].astype(np.float64), sig, rho


def test_spec_sizes():
    assert ps.extra_block_floats() == sum(int(np.prod(s)) for _, it in ps.extra_block_spec() for _, s, _ in it)
    names = [m for m, _ in ps.extra_block_spec()]
    assert names == list(ex.SUBSTEPS)
    assert dict(ps.extra_block_spec())["col_global"][3][1] == (64, 8)       # wk: ONE key head of dimension 8


def test_global_attention_brute_force(case):
    w, e, z, sig, rho = case
    wc = w["col_global"]
    out = ex.msa_col_global_attention(e, sig, rho, wc, D.head_dim_msa)
    S, N, C = e.shape
    d, H = D.head_dim_msa, D.heads_msa

    def ln(v):
        mu = sum(v) / len(v)
        var = sum((t - mu) ** 2 for t in v) / len(v)
        return [(t - mu) / math.sqrt(var + 1e-5) * float(g) + float(b) for t, g, b in zip(v, wc["ln_g"], wc["ln_b"])]

    def lin(v, W, b=None):
        return [sum(v[k] * float(W[k, n]) for k in range(len(v))) + (float(b[n]) if b is not None else 0.0) for n in range(W.shape[1])]

    for i in (0, 3):
        x = [ln([float(t) for t in e[s, i]]) for s in range(S)]
        mu = [float(rho[s]) * float(sig[i]) for s in range(S)]
        den = sum(mu) + 1e-10
        qbar = [sum(mu[s] * x[s][c] for s in range(S)) / den for c in range(C)]
        q = [t / math.sqrt(d) for t in lin(qbar, wc["wq"])]
        k = [lin(x[s], wc["wk"]) for s in range(S)]
        v = [lin(x[s], wc["wv"]) for s in range(S)]
        o = []
        for h in range(H):
            lg = [sum(q[h * d + c] * k[s][c] for c in range(d)) + 1e9 * (mu[s] - 1.0) for s in range(S)]
            mx = max(lg)
            p = [math.exp(t - mx) for t in lg]
            tot = sum(p)
            o += [sum(p[s] / tot * v[s][c] for s in range(S)) for c in range(d)]
        for s in (0, 2, 5):
            g = [1.0 / (1.0 + math.exp(-t)) for t in lin(x[s], wc["wg"], wc["bg"])]
            upd = lin([g[c] * o[c] for c in range(C)], wc["wo"], wc["bo"])
            for c in (0, 17, 63):
                assert abs(out[s, i, c] - (e[s, i, c] + upd[c])) < 1e-10
    # sampled form agrees everywhere
    for s in range(S):
        for i in range(N):
            assert np.abs(ex.msa_col_global_attention_at(e, sig, rho, wc, s, i, D.head_dim_msa) - out[s, i]).max() < 1e-12


def test_single_sequence_closed_form(case):
    """S = 1: the softmax over one key is 1, so o = v and e += Lin_o(G (.) tile_H(Lin_v(x)))."""
    w, e, z, sig, rho = case
    wc = w["col_global"]
    e1 = e[:1]
    out = ex.msa_col_global_attention(e1, np.ones(5), np.ones(1), wc, D.head_dim_msa)
    x = ref.layer_norm(e1, wc["ln_g"], wc["ln_b"])
    v = ref.linear(x, wc["wv"])
    g = ref.sigmoid(ref.linear(x, wc["wg"], wc["bg"]))
    exp = e1 + ref.linear(g * np.tile(v, (1, 1, D.heads_msa)), wc["wo"], wc["bo"])
    assert np.abs(out - exp).max() < 1e-12


def test_zero_query_weights_give_the_masked_mean_of_v(case):
    """W_q = 0 -> uniform weights over the unmasked sequences: o = masked mean of v (the same for every head)."""
    w, e, z, sig, rho = case
    wc = dict(w["col_global"])
    wc["wq"] = np.zeros_like(wc["wq"])
    out = ex.msa_col_global_attention(e, sig, rho, wc, D.head_dim_msa)
    x = ref.layer_norm(e, wc["ln_g"], wc["ln_b"])
    v = ref.linear(x, wc["wv"])
    g = ref.sigmoid(ref.linear(x, wc["wg"], wc["bg"]))
    for i in (0, 1, 3, 4):                                   # unmasked residues: mean over the unmasked sequences
        vm = (rho[:, None] * v[:, i]).sum(0) / rho.sum()
        exp = e[:, i] + ref.linear(g[:, i] * np.tile(vm, D.heads_msa)[None, :], wc["wo"], wc["bo"])
        assert np.abs(out[:, i] - exp).max() < 1e-12


def test_row_permutation_equivariance_and_padding(case):
    w, e, z, sig, rho = case
    wc = w["col_global"]
    out = ex.msa_col_global_attention(e, sig, rho, wc, D.head_dim_msa)
    perm = np.array([3, 0, 5, 1, 2, 4])
    outp = ex.msa_col_global_attention(e[perm], sig, rho[perm], wc, D.head_dim_msa)
    assert np.abs(outp - out[perm]).max() < 1e-12
    e2 = e.copy()
    g = ps.rng(113)
    e2[rho == 0] = 3.0 * g.standard_normal(e2[rho == 0].shape)          # other garbage in the masked sequences
    e2[:, sig == 0] = 3.0 * g.standard_normal(e2[:, sig == 0].shape)    # and at the masked residue
    out2 = ex.msa_col_global_attention(e2, sig, rho, wc, D.head_dim_msa)
    keep = (rho[:, None] * sig[None, :]) > 0
    assert np.abs(out2[keep] - out[keep]).max() < 1e-12                 # unmasked outputs do not see it (R3)
    assert np.abs(out2[~keep] - out[~keep]).max() > 1e-3 and np.isfinite(out2).all()


def test_block_order_and_pair_stack_reuse(case):
    w, e, z, sig, rho = case
    e1, z1 = ex.extra_msa_block(e, z, sig, rho, w)
    a, b = e, z
    a = ref.msa_row_attention(a, b, sig, rho, w["row"], 8)
    a = ex.msa_col_global_attention(a, sig, rho, w["col_global"], 8)
    a = ref.transition(a, w["msa_trans"])
    b = ref.outer_product_mean(a, b, sig, rho, w["opm"])
    b = ref.triangle_mult_outgoing(b, sig, w["tri_mul_out"])
    b = ref.triangle_mult_incoming(b, sig, w["tri_mul_in"])
    b = ref.triangle_attention_start(b, sig, w["tri_att_start"], 32)
    b = ref.triangle_attention_end(b, sig, w["tri_att_end"], 32)
    b = ref.transition(b, w["pair_trans"])
    assert np.abs(e1 - a).max() < 1e-12 and np.abs(z1 - b).max() < 1e-12
