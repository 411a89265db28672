"""Pin the fp64 oracle to library routines, closed forms and the invariants BASELINE.json north_star lists.

SURVEY.md §8(c) "What pins each part".  All CPU, fp64.
"""
import copy

import numpy as np
import pytest
import torch

import oracle
import pf_synth as ps

D = ps.AF2


@pytest.fixture(scope="module")
def w_full():
    return ps.make_block_weights(11, 0, D)


@pytest.fixture(scope="module")
def small_case(w_full):
    S, N = 6, 10
    msa, pair, _, _ = ps.make_inputs(11, 1, S, N, D)
    sig = np.ones(N)
    sig[7:] = 0
    rho = np.ones(S)
    rho[[2, 4]] = 0
    return S, N, msa[0].astype(np.float64), pair[0].astype(np.float64), sig, rho


# ---- LayerNorm --------------------------------------------------------------------------------

def test_layer_norm_matches_torch_and_moments():
    g = ps.rng(3)
    x = g.standard_normal((5, 7, 128)) * 3 + 1.5
    gamma, beta = g.standard_normal(128), g.standard_normal(128)
    ref = torch.nn.functional.layer_norm(torch.from_numpy(x), (128,), torch.from_numpy(gamma),
                                         torch.from_numpy(beta), eps=1e-5).numpy()
    assert np.abs(oracle.layer_norm(x, gamma, beta) - ref).max() < 1e-12
    y = oracle.layer_norm(x, np.ones(128), np.zeros(128))
    assert np.abs(y.mean(-1)).max() < 1e-12
    var = x.var(-1)
    assert np.abs(y.var(-1) - var / (var + 1e-5)).max() < 1e-12


# ---- transitions and projections vs torch matmul chain ---------------------------------------------

def test_transition_matches_torch(w_full, small_case):
    S, N, m, z, sig, rho = small_case
    for x, w in ((m, w_full["msa_trans"]), (z, w_full["pair_trans"])):
        t = {k: torch.from_numpy(np.asarray(v, dtype=np.float64)) for k, v in w.items()}
        xt = torch.from_numpy(x)
        h = torch.nn.functional.layer_norm(xt, (x.shape[-1],), t["ln_g"], t["ln_b"], 1e-5)
        ref = xt + torch.relu(h @ t["w1"] + t["b1"]) @ t["w2"] + t["b2"]
        assert np.abs(oracle.transition(x, w) - ref.numpy()).max() < 1e-11


# ---- softmax ------------------------------------------------------------------------------------

def test_attention_weights_normalised(w_full, small_case):
    S, N, m, z, sig, rho = small_case
    w = w_full["row"]
    x = oracle.layer_norm(m, w["ln_g"], w["ln_b"])
    q, k = oracle.linear(x, w["wq"]), oracle.linear(x, w["wk"])
    mu = rho[:, None] * sig[None, :]
    P = oracle.gated_attention_weights(q, k, None, mu, D.head_dim)
    assert P.min() >= 0.0
    assert np.abs(P.sum(-1) - 1.0).max() < 1e-13
    # masked keys carry exactly zero weight wherever the row has an unmasked key
    live = rho > 0
    assert np.all(P[live][:, :, :, sig == 0] == 0.0)
    # fully masked rows stay finite and normalised (R3: their values are unspecified, never compared)
    assert np.isfinite(P[~live]).all() and np.abs(P[~live].sum(-1) - 1.0).max() < 1e-12


def _online_softmax_attention(q, k, v, bias, keyneg, block):
    """Blocked / online-softmax restatement (flash-style) in fp64, used only as a cross-check."""
    L, d = q.shape
    mx = np.full(L, -np.inf)
    den = np.zeros(L)
    acc = np.zeros((L, v.shape[1]))
    for j0 in range(0, L, block):
        j1 = min(L, j0 + block)
        s = q @ k[j0:j1].T / np.sqrt(d) + bias[:, j0:j1] + keyneg[None, j0:j1]
        new = np.maximum(mx, s.max(1))
        scale = np.exp(mx - new)
        p = np.exp(s - new[:, None])
        den = den * scale + p.sum(1)
        acc = acc * scale[:, None] + p @ v[j0:j1]
        mx = new
    return acc / den[:, None]


def test_naive_vs_blocked_attention():
    g = ps.rng(5)
    L, d = 13, 8
    q, k, v = (g.standard_normal((L, d)) for _ in range(3))
    bias = g.standard_normal((L, L))
    mask = np.ones(L)
    mask[[3, 9]] = 0
    P = oracle.gated_attention_weights(q[None], k[None], bias[None], mask[None], d)[0, 0]
    naive = P @ v
    for block in (1, 4, 5, 13):
        blk = _online_softmax_attention(q, k, v, bias, oracle.neg(mask), block)
        assert np.abs(naive - blk).max() < 1e-12


# ---- gated attention special cases -----------------------------------------------------------------

def test_gate_one_equals_torch_sdpa(w_full):
    g = ps.rng(6)
    R, L, C, H, d = 3, 9, 256, 8, 32
    x = g.standard_normal((R, L, C))
    bias = g.standard_normal((H, L, L))
    mask = np.ones((R, L))
    mask[:, 6:] = 0
    w = {k: np.asarray(v, dtype=np.float64) for k, v in w_full["col"].items()}
    w["wg"] = np.zeros_like(w["wg"])
    w["bg"] = np.full_like(w["bg"], 40.0)            # sigmoid(40) == 1 to 1e-17
    got = oracle.gated_attention(x, bias, mask, w, d)
    T = torch.from_numpy
    q = (T(x) @ T(w["wq"])).reshape(R, L, H, d).permute(0, 2, 1, 3)
    k = (T(x) @ T(w["wk"])).reshape(R, L, H, d).permute(0, 2, 1, 3)
    v = (T(x) @ T(w["wv"])).reshape(R, L, H, d).permute(0, 2, 1, 3)
    am = T(bias)[None] + T(oracle.neg(mask))[:, None, None, :]
    o = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=am)   # scale 1/sqrt(d)
    ref = o.permute(0, 2, 1, 3).reshape(R, L, C) @ T(w["wo"]) + T(w["bo"])
    assert np.abs(got - ref.numpy()).max() < 1e-11


def test_zero_query_gives_gated_masked_mean(w_full):
    g = ps.rng(7)
    R, L, C, d = 2, 7, 256, 32
    x = g.standard_normal((R, L, C))
    mask = np.ones((R, L))
    mask[0, 5:] = 0
    w = {k: np.asarray(v, dtype=np.float64) for k, v in w_full["col"].items()}
    w["wq"] = np.zeros_like(w["wq"])
    got = oracle.gated_attention(x, None, mask, w, d)
    v = x @ w["wv"]
    mean_v = (mask[:, :, None] * v).sum(1, keepdims=True) / mask.sum(1)[:, None, None]
    gate = 1 / (1 + np.exp(-(x @ w["wg"] + w["bg"])))
    ref = (gate * mean_v) @ w["wo"] + w["bo"]
    assert np.abs(got - ref).max() < 1e-11


# ---- outer product mean ---------------------------------------------------------------------------

def test_opm_single_sequence_closed_form(w_full):
    g = ps.rng(8)
    N = 5
    m = g.standard_normal((1, N, D.c_m))
    z = g.standard_normal((N, N, D.c_z))
    w = w_full["opm"]
    x = oracle.layer_norm(m, w["ln_g"], w["ln_b"])[0]
    a = x @ np.float64(w["wa"]) + w["ba"]
    b = x @ np.float64(w["wb"]) + w["bb"]
    ref = np.empty_like(z)
    for i in range(N):
        for j in range(N):
            ref[i, j] = z[i, j] + (np.outer(a[i], b[j]).reshape(-1) / (1 + 1e-3)) @ np.float64(w["wout"]) + w["bout"]
    got = oracle.outer_product_mean(m, z, np.ones(N), np.ones(1), w)
    assert np.abs(got - ref).max() < 1e-11


def test_opm_matches_torch_einsum_route(w_full, small_case):
    S, N, m, z, sig, rho = small_case
    w = {k: torch.from_numpy(np.asarray(v, dtype=np.float64)) for k, v in w_full["opm"].items()}
    mt = torch.from_numpy(m)
    x = torch.nn.functional.layer_norm(mt, (D.c_m,), w["ln_g"], w["ln_b"], 1e-5)
    mu = torch.from_numpy(rho[:, None] * sig[None, :])
    a = mu[..., None] * (x @ w["wa"] + w["ba"])
    b = mu[..., None] * (x @ w["wb"] + w["bb"])
    O = torch.einsum("sic,sjd->ijcd", a, b).reshape(N, N, -1)
    n = mu.T @ mu
    ref = torch.from_numpy(z) + (O / (1e-3 + n)[..., None]) @ w["wout"] + w["bout"]
    got = oracle.outer_product_mean(m, z, sig, rho, w_full["opm"])
    assert np.abs(got - ref.numpy()).max() < 1e-11


# ---- triangle identities (SURVEY.md §0 finding 1) -----------------------------------------------------

def test_incoming_is_outgoing_on_transpose_with_swapped_ab(w_full, small_case):
    S, N, m, z, sig, rho = small_case
    w = w_full["tri_mul_in"]
    sw = dict(w)
    for proj in ("p", "g"):
        for kind in ("w", "b"):
            sw[f"{kind}_a{proj}"], sw[f"{kind}_b{proj}"] = w[f"{kind}_b{proj}"], w[f"{kind}_a{proj}"]
    zt = np.transpose(z, (1, 0, 2))
    inc = oracle.triangle_mult_incoming(z, sig, w)
    out_t = np.transpose(oracle.triangle_mult_outgoing(zt, sig, sw), (1, 0, 2))
    assert np.abs(inc - out_t).max() < 1e-12
    # without the a<->b swap the identity must NOT hold (guards against a symmetric bug)
    out_noswap = np.transpose(oracle.triangle_mult_outgoing(zt, sig, w), (1, 0, 2))
    assert np.abs(inc - out_noswap).max() > 1e-2


def test_triangle_mult_single_residue_closed_form(w_full):
    g = ps.rng(9)
    z = g.standard_normal((1, 1, D.c_z))
    for name, fn in (("tri_mul_out", oracle.triangle_mult_outgoing), ("tri_mul_in", oracle.triangle_mult_incoming)):
        w = {k: np.asarray(v, dtype=np.float64) for k, v in w_full[name].items()}
        x = oracle.layer_norm(z, w["ln_in_g"], w["ln_in_b"])[0, 0]
        sg = lambda t: 1 / (1 + np.exp(-t))
        a = sg(x @ w["w_ag"] + w["b_ag"]) * (x @ w["w_ap"] + w["b_ap"])
        b = sg(x @ w["w_bg"] + w["b_bg"]) * (x @ w["w_bp"] + w["b_bp"])
        gt = sg(x @ w["w_g"] + w["b_g"])
        t = oracle.layer_norm(a * b, w["ln_out_g"], w["ln_out_b"])
        ref = z[0, 0] + gt * (t @ w["w_z"] + w["b_z"])
        assert np.abs(fn(z, np.ones(1), w_full[name])[0, 0] - ref).max() < 1e-12


def test_ending_node_is_starting_node_on_transpose(w_full, small_case):
    S, N, m, z, sig, rho = small_case
    w = w_full["tri_att_end"]
    zt = np.transpose(z, (1, 0, 2))
    end = oracle.triangle_attention_end(z, sig, w)
    start_t = np.transpose(oracle.triangle_attention_start(zt, sig, w), (1, 0, 2))
    assert np.abs(end - start_t).max() < 1e-12
    assert np.abs(end - oracle.triangle_attention_start(z, sig, w)).max() > 1e-2


# ---- padding invariance (north_star) ----------------------------------------------------------------

def test_padding_does_not_change_unpadded_outputs(w_full):
    S, N, Sp, Np = 5, 9, 8, 14
    msa, pair, _, _ = ps.make_inputs(21, 1, S, N, D)
    m, z = msa[0].astype(np.float64), pair[0].astype(np.float64)
    g = ps.rng(22)
    mp = 3.0 * g.standard_normal((Sp, Np, D.c_m))
    zp = 3.0 * g.standard_normal((Np, Np, D.c_z))
    mp[:S, :N] = m
    zp[:N, :N] = z
    sig, rho = np.zeros(Np), np.zeros(Sp)
    sig[:N] = 1
    rho[:S] = 1
    m_ref, z_ref = oracle.evoformer_block(m, z, np.ones(N), np.ones(S), w_full)
    m_pad, z_pad = oracle.evoformer_block(mp, zp, sig, rho, w_full)
    assert np.abs(m_pad[:S, :N] - m_ref).max() < 1e-9
    assert np.abs(z_pad[:N, :N] - z_ref).max() < 1e-9
    assert np.isfinite(m_pad).all() and np.isfinite(z_pad).all()


# ---- MSA row permutation (north_star) ---------------------------------------------------------------

def test_msa_row_permutation(w_full, small_case):
    S, N, m, z, sig, rho = small_case
    perm = np.array([0, 3, 1, 5, 2, 4])
    m1, z1 = oracle.evoformer_block(m, z, sig, rho, w_full)
    m2, z2 = oracle.evoformer_block(m[perm], z, sig, rho[perm], w_full)
    live = sig > 0
    assert np.abs(z2[live][:, live] - z1[live][:, live]).max() < 1e-10        # OPM invariant
    lr = rho[perm] > 0
    assert np.abs(m2[lr][:, live] - m1[perm][lr][:, live]).max() < 1e-10      # column attention equivariant


# ---- whole block ------------------------------------------------------------------------------------

def test_zero_output_layers_make_block_identity(w_full, small_case):
    S, N, m, z, sig, rho = small_case
    w = copy.deepcopy(w_full)
    for mod, names in (("row", ("wo", "bo")), ("col", ("wo", "bo")), ("msa_trans", ("w2", "b2")),
                       ("opm", ("wout", "bout")), ("tri_mul_out", ("w_z", "b_z")), ("tri_mul_in", ("w_z", "b_z")),
                       ("tri_att_start", ("wo", "bo")), ("tri_att_end", ("wo", "bo")), ("pair_trans", ("w2", "b2"))):
        for n in names:
            w[mod][n] = np.zeros_like(w[mod][n])
    m1, z1 = oracle.evoformer_block(m, z, sig, rho, w)
    assert np.array_equal(m1, m) and np.array_equal(z1, z)


def test_every_substep_changes_only_its_stream(w_full, small_case):
    S, N, m, z, sig, rho = small_case
    for step in range(1, 10):
        m1, z1 = oracle.substep(step, m, z, sig, rho, w_full)
        if step <= 3:
            assert np.array_equal(z1, z) and np.abs(m1 - m).max() > 1e-3
        else:
            assert np.array_equal(m1, m) and np.abs(z1 - z).max() > 1e-3


def test_blob_roundtrip_and_size():
    assert ps.block_floats(D) == 1829952          # SURVEY.md Appendix B total
    w = ps.make_weights(5, 2, D, bf16_weights=True)
    blob = ps.pack_blob(w, D)
    back = ps.unpack_blob(blob, 2, D)
    for a, b in zip(w, back):
        for mod in a:
            for name in a[mod]:
                assert np.array_equal(a[mod][name], b[mod][name])
    # R15: W matrices are bf16-representable (low 16 bits of the fp32 pattern are zero)
    assert (w[0]["row"]["wq"].view(np.uint32) & 0xFFFF).max() == 0
    assert (w[0]["row"]["bg"].view(np.uint32) & 0xFFFF).max() != 0


def test_round_to_bf16_matches_torch():
    x = ps.rng(1).standard_normal(10000).astype(np.float32) * 7
    ref = torch.from_numpy(x).to(torch.bfloat16).to(torch.float32).numpy()
    assert np.array_equal(ps.round_to_bf16(x), ref)
