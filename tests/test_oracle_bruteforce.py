"""Pin the fp64 oracle against index-by-index pure-Python loops on tiny inputs.

The loops below are written straight from the index forms of SURVEY.md Appendix A.1-A.9 with
`math` scalars only (no numpy arithmetic, no einsum, no matmul), so a transposed operand, a wrong
index, a dropped bias/mask/gate or a wrong flatten order in ``oracle/`` fails here.
"""
import math

import numpy as np
import pytest

import oracle
import pf_synth as ps

TOL = 1e-11


# ---- scalar helpers ---------------------------------------------------------------------------

def _ln(vec, g, b):
    n = len(vec)
    mean = sum(vec) / n
    var = sum((v - mean) ** 2 for v in vec) / n
    return [(v - mean) / math.sqrt(var + 1e-5) * g[c] + b[c] for c, v in enumerate(vec)]


def _lin(vec, W, b=None):
    out = []
    for o in range(len(W[0])):
        acc = sum(vec[i] * W[i][o] for i in range(len(vec)))
        out.append(acc + (b[o] if b is not None else 0.0))
    return out


def _sg(x):
    return 1.0 / (1.0 + math.exp(-x))


def _softmax(v):
    mx = max(v)
    e = [math.exp(x - mx) for x in v]
    s = sum(e)
    return [x / s for x in e]


def _L(a):
    return np.asarray(a, dtype=np.float64).tolist()


def _w(w):
    return {k: _L(v) for k, v in w.items()}


@pytest.fixture(scope="module")
def case(tiny_dims):
    d = tiny_dims
    S, N = 3, 4
    w = ps.make_block_weights(7, 0, d)
    msa, pair, _, _ = ps.make_inputs(7, 1, S, N, d)
    seq_mask = np.array([1, 1, 0, 1], dtype=np.float64)      # a hole, not just a suffix
    msa_mask = np.array([1, 0, 1], dtype=np.float64)
    return d, S, N, w, msa[0].astype(np.float64), pair[0].astype(np.float64), seq_mask, msa_mask


# ---- A.1 ---------------------------------------------------------------------------------------

def test_row_attention_loops(case):
    d, S, N, w, m, z, sig, rho = case
    W = _w(w["row"])
    H, dh = d.heads_msa, d.head_dim
    ml, zl = _L(m), _L(z)
    x = [[_ln(ml[s][i], W["ln_g"], W["ln_b"]) for i in range(N)] for s in range(S)]
    y = [[_ln(zl[i][j], W["ln_z_g"], W["ln_z_b"]) for j in range(N)] for i in range(N)]
    beta = [[_lin(y[i][j], W["w_bias"]) for j in range(N)] for i in range(N)]     # [i][j][h]
    out = np.zeros_like(m)
    for s in range(S):
        q = [_lin(x[s][i], W["wq"]) for i in range(N)]
        k = [_lin(x[s][i], W["wk"]) for i in range(N)]
        v = [_lin(x[s][i], W["wv"]) for i in range(N)]
        G = [[_sg(t) for t in _lin(x[s][i], W["wg"], W["bg"])] for i in range(N)]
        for i in range(N):
            o = [0.0] * (H * dh)
            for h in range(H):
                logits = []
                for j in range(N):
                    dot = sum(q[i][h * dh + c] * k[j][h * dh + c] for c in range(dh))
                    logits.append(dot / math.sqrt(dh) + beta[i][j][h] + 1e9 * (rho[s] * sig[j] - 1.0))
                P = _softmax(logits)
                for c in range(dh):
                    o[h * dh + c] = G[i][h * dh + c] * sum(P[j] * v[j][h * dh + c] for j in range(N))
            upd = _lin(o, W["wo"], W["bo"])
            for c in range(d.c_m):
                out[s, i, c] = ml[s][i][c] + upd[c]
    got = oracle.msa_row_attention(m, z, sig, rho, w["row"], dh)
    assert np.abs(got - out).max() < TOL


# ---- A.2 ---------------------------------------------------------------------------------------

def test_col_attention_loops(case):
    d, S, N, w, m, z, sig, rho = case
    W = _w(w["col"])
    H, dh = d.heads_msa, d.head_dim
    ml = _L(m)
    x = [[_ln(ml[s][i], W["ln_g"], W["ln_b"]) for i in range(N)] for s in range(S)]
    out = np.zeros_like(m)
    for i in range(N):
        q = [_lin(x[s][i], W["wq"]) for s in range(S)]
        k = [_lin(x[s][i], W["wk"]) for s in range(S)]
        v = [_lin(x[s][i], W["wv"]) for s in range(S)]
        G = [[_sg(t) for t in _lin(x[s][i], W["wg"], W["bg"])] for s in range(S)]
        for s in range(S):
            o = [0.0] * (H * dh)
            for h in range(H):
                logits = []
                for t in range(S):
                    dot = sum(q[s][h * dh + c] * k[t][h * dh + c] for c in range(dh))
                    logits.append(dot / math.sqrt(dh) + 1e9 * (rho[t] * sig[i] - 1.0))
                P = _softmax(logits)
                for c in range(dh):
                    o[h * dh + c] = G[s][h * dh + c] * sum(P[t] * v[t][h * dh + c] for t in range(S))
            upd = _lin(o, W["wo"], W["bo"])
            for c in range(d.c_m):
                out[s, i, c] = ml[s][i][c] + upd[c]
    got = oracle.msa_col_attention(m, sig, rho, w["col"], dh)
    assert np.abs(got - out).max() < TOL


# ---- A.3 / A.9 ---------------------------------------------------------------------------------

@pytest.mark.parametrize("which", ["msa_trans", "pair_trans"])
def test_transition_loops(case, which):
    d, S, N, w, m, z, sig, rho = case
    W = _w(w[which])
    x = m if which == "msa_trans" else z
    xl = _L(x)
    out = np.zeros_like(x)
    for a in range(x.shape[0]):
        for b in range(x.shape[1]):
            h = [max(t, 0.0) for t in _lin(_ln(xl[a][b], W["ln_g"], W["ln_b"]), W["w1"], W["b1"])]
            u = _lin(h, W["w2"], W["b2"])
            for c in range(x.shape[2]):
                out[a, b, c] = xl[a][b][c] + u[c]
    assert np.abs(oracle.transition(x, w[which]) - out).max() < TOL


# ---- A.4 ---------------------------------------------------------------------------------------

def test_outer_product_mean_loops(case):
    d, S, N, w, m, z, sig, rho = case
    W = _w(w["opm"])
    co = d.c_opm
    ml, zl = _L(m), _L(z)
    a = [[None] * N for _ in range(S)]
    b = [[None] * N for _ in range(S)]
    for s in range(S):
        for i in range(N):
            x = _ln(ml[s][i], W["ln_g"], W["ln_b"])
            mu = rho[s] * sig[i]
            a[s][i] = [mu * t for t in _lin(x, W["wa"], W["ba"])]
            b[s][i] = [mu * t for t in _lin(x, W["wb"], W["bb"])]
    out = np.zeros_like(z)
    for i in range(N):
        for j in range(N):
            n_ij = sum(rho[s] * sig[i] * rho[s] * sig[j] for s in range(S))
            vec = [0.0] * (co * co)
            for c1 in range(co):
                for c2 in range(co):
                    vec[c1 * co + c2] = sum(a[s][i][c1] * b[s][j][c2] for s in range(S)) / (1e-3 + n_ij)
            u = _lin(vec, W["wout"], W["bout"])
            for c in range(d.c_z):
                out[i, j, c] = zl[i][j][c] + u[c]
    got = oracle.outer_product_mean(m, z, sig, rho, w["opm"])
    assert np.abs(got - out).max() < TOL


# ---- A.5 / A.6 ---------------------------------------------------------------------------------

@pytest.mark.parametrize("incoming", [False, True])
def test_triangle_mult_loops(case, incoming):
    d, S, N, w, m, z, sig, rho = case
    name = "tri_mul_in" if incoming else "tri_mul_out"
    W = _w(w[name])
    ct = d.c_tri
    zl = _L(z)
    a = [[None] * N for _ in range(N)]
    b = [[None] * N for _ in range(N)]
    g = [[None] * N for _ in range(N)]
    for i in range(N):
        for k in range(N):
            x = _ln(zl[i][k], W["ln_in_g"], W["ln_in_b"])
            pi = sig[i] * sig[k]
            ap, ag = _lin(x, W["w_ap"], W["b_ap"]), _lin(x, W["w_ag"], W["b_ag"])
            bp, bg = _lin(x, W["w_bp"], W["b_bp"]), _lin(x, W["w_bg"], W["b_bg"])
            a[i][k] = [pi * _sg(ag[c]) * ap[c] for c in range(ct)]
            b[i][k] = [pi * _sg(bg[c]) * bp[c] for c in range(ct)]
            g[i][k] = [_sg(t) for t in _lin(x, W["w_g"], W["b_g"])]
    out = np.zeros_like(z)
    for i in range(N):
        for j in range(N):
            if incoming:
                t = [sum(a[k][i][c] * b[k][j][c] for k in range(N)) for c in range(ct)]
            else:
                t = [sum(a[i][k][c] * b[j][k][c] for k in range(N)) for c in range(ct)]
            u = _lin(_ln(t, W["ln_out_g"], W["ln_out_b"]), W["w_z"], W["b_z"])
            for c in range(d.c_z):
                out[i, j, c] = zl[i][j][c] + g[i][j][c] * u[c]
    fn = oracle.triangle_mult_incoming if incoming else oracle.triangle_mult_outgoing
    assert np.abs(fn(z, sig, w[name]) - out).max() < TOL


# ---- A.7 / A.8 ---------------------------------------------------------------------------------

@pytest.mark.parametrize("ending", [False, True])
def test_triangle_attention_loops(case, ending):
    d, S, N, w, m, z, sig, rho = case
    name = "tri_att_end" if ending else "tri_att_start"
    W = _w(w[name])
    H, dh = d.heads_pair, d.head_dim
    zl = _L(z)
    x = [[_ln(zl[i][j], W["ln_g"], W["ln_b"]) for j in range(N)] for i in range(N)]
    q = [[_lin(x[i][j], W["wq"]) for j in range(N)] for i in range(N)]
    k = [[_lin(x[i][j], W["wk"]) for j in range(N)] for i in range(N)]
    v = [[_lin(x[i][j], W["wv"]) for j in range(N)] for i in range(N)]
    G = [[[_sg(t) for t in _lin(x[i][j], W["wg"], W["bg"])] for j in range(N)] for i in range(N)]
    beta = [[_lin(x[i][j], W["w_bias"]) for j in range(N)] for i in range(N)]     # beta[a][b][h] from x[a][b]
    out = np.zeros_like(z)
    for i in range(N):
        for j in range(N):
            o = [0.0] * (H * dh)
            for h in range(H):
                logits = []
                for kk in range(N):
                    if ending:   # A.8: q[i,j].k[kk,j] + beta[h,kk,i] + NEG(pi_{kk,j})
                        dot = sum(q[i][j][h * dh + c] * k[kk][j][h * dh + c] for c in range(dh))
                        logits.append(dot / math.sqrt(dh) + beta[kk][i][h] + 1e9 * (sig[kk] * sig[j] - 1.0))
                    else:        # A.7: q[i,j].k[i,kk] + beta[h,j,kk] + NEG(pi_{i,kk})
                        dot = sum(q[i][j][h * dh + c] * k[i][kk][h * dh + c] for c in range(dh))
                        logits.append(dot / math.sqrt(dh) + beta[j][kk][h] + 1e9 * (sig[i] * sig[kk] - 1.0))
                P = _softmax(logits)
                for c in range(dh):
                    if ending:
                        acc = sum(P[kk] * v[kk][j][h * dh + c] for kk in range(N))
                    else:
                        acc = sum(P[kk] * v[i][kk][h * dh + c] for kk in range(N))
                    o[h * dh + c] = G[i][j][h * dh + c] * acc
            u = _lin(o, W["wo"], W["bo"])
            for c in range(d.c_z):
                out[i, j, c] = zl[i][j][c] + u[c]
    fn = oracle.triangle_attention_end if ending else oracle.triangle_attention_start
    assert np.abs(fn(z, sig, w[name], dh) - out).max() < TOL


def test_block_order(case):
    """R0 ordering: OPM (step 4) must read the m updated by steps 1-3; the block is steps 1..9 in order."""
    d, S, N, w, m, z, sig, rho = case
    dh = d.head_dim
    m1 = oracle.msa_row_attention(m, z, sig, rho, w["row"], dh)
    m2 = oracle.msa_col_attention(m1, sig, rho, w["col"], dh)
    m3 = oracle.transition(m2, w["msa_trans"])
    z1 = oracle.outer_product_mean(m3, z, sig, rho, w["opm"])
    z2 = oracle.triangle_mult_outgoing(z1, sig, w["tri_mul_out"])
    z3 = oracle.triangle_mult_incoming(z2, sig, w["tri_mul_in"])
    z4 = oracle.triangle_attention_start(z3, sig, w["tri_att_start"], dh)
    z5 = oracle.triangle_attention_end(z4, sig, w["tri_att_end"], dh)
    z6 = oracle.transition(z5, w["pair_trans"])
    mb, zb = oracle.evoformer_block(m, z, sig, rho, w, dh)
    assert np.array_equal(mb, m3) and np.array_equal(zb, z6)
    # OPM on the *old* m must differ (guards against reading the stale stream)
    assert np.abs(oracle.outer_product_mean(m, z, sig, rho, w["opm"]) - z1).max() > 1e-3
