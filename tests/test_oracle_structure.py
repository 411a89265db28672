"""Pins of the structure-module / heads oracle (oracle/structure_ref.py; readings M.0-M.6, H.1-H.5 of DESIGN.md §2d) against
things other than itself: scipy's Rotation, homogeneous 4x4 matrices, torch's attention and softplus, pure-Python index
loops, the rigid-motion invariance the attention is named for, closed forms and padding invariance (with negative controls).
"""
import math

import numpy as np
import pytest
import torch
from scipy.spatial.transform import Rotation

import pf_synth as ps
from oracle import structure_ref as sr

D = ps.STRUCT
SMALL = ps.StructDims(c_m=12, c_z=5, c_s=8, heads=2, c_ipa=3, n_qp=2, n_pv=2, n_layers=2, c_resnet=6, n_torsion=3,
                      n_dist_bins=7, n_msa_classes=4, n_lddt_bins=5, c_lddt=6, n_pae_bins=6, n_resolved=3)


def _kw(d):
    return dict(heads=d.heads, c=d.c_ipa, n_qp=d.n_qp, n_pv=d.n_pv)


def _random_frames(seed, n):
    g = ps.rng(seed, 77)
    R = Rotation.from_rotvec(g.standard_normal((n, 3))).as_matrix()
    return R, g.standard_normal((n, 3))


def _inputs(seed, N, d, lengths=None):
    main = ps.Dims(c_m=d.c_m, c_z=d.c_z)
    m, z, sm, _ = ps.make_inputs(seed, 1, 3, N, main, lengths=lengths)
    return m[0], z[0], sm[0]


def test_quaternion_map_matches_scipy():
    g = ps.rng(5, 1)
    bcd = g.standard_normal((50, 3)) * 2.0
    ours = sr.quat_to_rot(bcd[:, 0], bcd[:, 1], bcd[:, 2])
    q = np.concatenate([bcd, np.ones((50, 1))], axis=1)          # scipy: scalar last, normalises
    ref = Rotation.from_quat(q).as_matrix()
    assert np.abs(ours - ref).max() < 1e-13
    assert np.abs(np.einsum("nab,ncb->nac", ours, ours) - np.eye(3)).max() < 1e-13
    assert np.allclose(np.linalg.det(ours), 1.0)


def test_frame_composition_matches_homogeneous_matrices():
    R1, t1 = _random_frames(1, 6)
    R2, t2 = _random_frames(2, 6)
    R, t = sr.compose_frames(R1, t1, R2, t2)
    for n in range(6):
        A, B = np.eye(4), np.eye(4)
        A[:3, :3], A[:3, 3] = R1[n], t1[n]
        B[:3, :3], B[:3, 3] = R2[n], t2[n]
        C = A @ B
        assert np.abs(C[:3, :3] - R[n]).max() < 1e-13 and np.abs(C[:3, 3] - t[n]).max() < 1e-13


def test_softplus_matches_torch():
    x = np.linspace(-30, 30, 101)
    assert np.abs(sr.softplus(x) - torch.nn.functional.softplus(torch.from_numpy(x), threshold=1e9).numpy()).max() < 1e-13


def test_ipa_pure_python_loops():
    d = SMALL
    N = 5
    w = ps.make_struct_weights(3, d)
    g = ps.rng(9, 1)
    s = g.standard_normal((N, d.c_s))
    zn = g.standard_normal((N, N, d.c_z))
    R, t = _random_frames(4, N)
    mask = np.array([1, 1, 0, 1, 1], dtype=np.float64)           # a hole among the keys
    got, a_got = sr.invariant_point_attention(s, zn, R, t, mask, w, return_weights=True, **_kw(d))
    H, c, Pq, Pv = d.heads, d.c_ipa, d.n_qp, d.n_pv
    W = {k: np.asarray(v, dtype=np.float64) for k, v in w.items()}

    def lin0(x, M):
        return [sum(x[a] * M[a][o] for a in range(len(x))) for o in range(len(M[0]))]

    def glob(n, p):   # R_n p + t_n
        return [sum(R[n][a][b] * p[b] for b in range(3)) + t[n][a] for a in range(3)]

    q = [lin0(s[n], W["w_q"]) for n in range(N)]
    k = [lin0(s[n], W["w_k"]) for n in range(N)]
    v = [lin0(s[n], W["w_v"]) for n in range(N)]
    qp = [lin0(s[n], W["w_qp"]) for n in range(N)]
    kp = [lin0(s[n], W["w_kp"]) for n in range(N)]
    vp = [lin0(s[n], W["w_vp"]) for n in range(N)]
    wc, wl = math.sqrt(2.0 / (9.0 * Pq)), math.sqrt(1.0 / 3.0)
    out = np.zeros((N, d.c_s))
    for i in range(N):
        cat_t, cat_o, cat_p, cat_n = [], [], [], []
        for h in range(H):
            gam = math.log(1.0 + math.exp(W["g_head"][h]))
            logit = []
            for j in range(N):
                qk = sum(q[i][h * c + e] * k[j][h * c + e] for e in range(c)) / math.sqrt(c)
                bij = sum(zn[i][j][e] * W["w_b"][e][h] for e in range(d.c_z))
                d2 = 0.0
                for p in range(Pq):
                    a = glob(i, qp[i][(h * Pq + p) * 3:(h * Pq + p) * 3 + 3])
                    b = glob(j, kp[j][(h * Pq + p) * 3:(h * Pq + p) * 3 + 3])
                    d2 += sum((a[x] - b[x]) ** 2 for x in range(3))
                logit.append(wl * (qk + bij - gam * wc / 2.0 * d2) + 1e9 * (mask[j] - 1.0))
            mx = max(logit)
            e = [math.exp(x - mx) for x in logit]
            a = [x / sum(e) for x in e]
            assert abs(sum(a) - 1.0) < 1e-12 and a[2] == 0.0
            for j in range(N):
                assert abs(a[j] - a_got[h, i, j]) < 1e-12
            cat_t += [sum(a[j] * zn[i][j][e2] for j in range(N)) for e2 in range(d.c_z)]
            cat_o += [sum(a[j] * v[j][h * c + e2] for j in range(N)) for e2 in range(c)]
            for p in range(Pv):
                og = [0.0, 0.0, 0.0]
                for j in range(N):
                    gj = glob(j, vp[j][(h * Pv + p) * 3:(h * Pv + p) * 3 + 3])
                    og = [og[x] + a[j] * gj[x] for x in range(3)]
                loc = [sum(R[i][b][x] * (og[b] - t[i][b]) for b in range(3)) for x in range(3)]   # R^T (og - t)
                cat_p += loc
                cat_n.append(math.sqrt(sum(x * x for x in loc) + 1e-8))
        cat = cat_t + cat_o + cat_p + cat_n
        assert len(cat) == d.c_cat
        out[i] = [sum(cat[a2] * W["w_out"][a2][o] for a2 in range(d.c_cat)) + W["b_out"][o] for o in range(d.c_s)]
    assert np.abs(out - got).max() < 1e-11


def test_ipa_without_points_is_plain_biased_attention():
    """w_qp = w_kp = 0 with identity frames: the point term vanishes and the scalar output is torch's attention."""
    d = SMALL
    N = 7
    w = dict(ps.make_struct_weights(4, d))
    w["w_qp"] = np.zeros_like(w["w_qp"])
    w["w_kp"] = np.zeros_like(w["w_kp"])
    H, c = d.heads, d.c_ipa
    sel = np.zeros((d.c_cat, d.c_s))
    o_lo = H * d.c_z
    for e in range(H * c):
        sel[o_lo + e, e] = 1.0                                   # Lin_out picks the scalar block o
    w["w_out"], w["b_out"] = sel, np.zeros(d.c_s)
    g = ps.rng(11, 1)
    s = g.standard_normal((N, d.c_s))
    zn = g.standard_normal((N, N, d.c_z))
    mask = np.array([1, 1, 1, 0, 1, 1, 0], dtype=np.float64)
    got = sr.invariant_point_attention(s, zn, np.tile(np.eye(3), (N, 1, 1)), np.zeros((N, 3)), mask, w, **_kw(d))[:, :H * c]
    wl = math.sqrt(1.0 / 3.0)
    tq = torch.from_numpy((s @ w["w_q"].astype(np.float64)).reshape(N, H, c)).permute(1, 0, 2)
    tk = torch.from_numpy((s @ w["w_k"].astype(np.float64)).reshape(N, H, c)).permute(1, 0, 2)
    tv = torch.from_numpy((s @ w["w_v"].astype(np.float64)).reshape(N, H, c)).permute(1, 0, 2)
    bias = torch.from_numpy(wl * np.transpose(zn @ w["w_b"].astype(np.float64), (2, 0, 1)) + 1e9 * (mask[None, None, :] - 1.0))
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, attn_mask=bias, scale=wl / math.sqrt(c))
    assert np.abs(ref.permute(1, 0, 2).reshape(N, H * c).numpy() - got).max() < 1e-12


def test_rigid_motion_invariance_and_equivariance():
    """A global rigid motion of the incoming frames leaves s, the angles and pLDDT unchanged and moves the outgoing frames
    with it; moving ONE residue's frame does change the result (negative control)."""
    d = SMALL
    N = 9
    w = ps.make_struct_weights(5, d)
    m0, z, mask = _inputs(6, N, d, lengths=[7])
    m0 = m0[0]
    R, t = _random_frames(7, N)
    Rg, tg = _random_frames(8, 1)
    Rg, tg = Rg[0], tg[0]
    kw = dict(n_layers=d.n_layers, n_torsion=d.n_torsion, **_kw(d))
    a = sr.structure_module(m0, z, mask, w, frames=(R, t), **kw)
    b = sr.structure_module(m0, z, mask, w, frames=(Rg @ R, t @ Rg.T + tg), **kw)
    v = mask > 0
    assert np.abs(a["s"][v] - b["s"][v]).max() < 1e-10
    assert np.abs(a["alpha"][v] - b["alpha"][v]).max() < 1e-10
    assert np.abs(Rg @ a["R"][v] - b["R"][v]).max() < 1e-10
    assert np.abs(a["t"][v] @ Rg.T + tg - b["t"][v]).max() < 1e-10
    assert np.abs(sr.plddt(a["s"], w)[1][v] - sr.plddt(b["s"], w)[1][v]).max() < 1e-8
    t2 = t.copy()
    t2[1] += 0.5
    c = sr.structure_module(m0, z, mask, w, frames=(R, t2), **kw)
    assert np.abs(a["s"][v] - c["s"][v]).max() > 1e-3


def test_zero_backbone_update_keeps_identity_frames():
    d = SMALL
    N = 6
    w = dict(ps.make_struct_weights(6, d))
    w["w_bb"], w["b_bb"] = np.zeros_like(w["w_bb"]), np.zeros_like(w["b_bb"])
    m0, z, mask = _inputs(7, N, d)
    o = sr.structure_module(m0[0], z, mask, w, n_layers=3, n_torsion=d.n_torsion, **_kw(d))
    assert np.abs(o["R"] - np.eye(3)).max() == 0.0 and np.abs(o["t"]).max() == 0.0 and np.abs(o["x"]).max() == 0.0


def test_backbone_update_is_a_right_composition():
    """t moves by R u (the update is expressed in the residue's own frame), checked against scipy."""
    d = SMALL
    N = 4
    w = ps.make_struct_weights(8, d)
    g = ps.rng(3, 3)
    s = g.standard_normal((N, d.c_s))
    R, t = _random_frames(9, N)
    R2, t2 = sr.backbone_update(s, R, t, w)
    y = s @ w["w_bb"].astype(np.float64) + w["b_bb"]
    Ru = Rotation.from_quat(np.concatenate([y[:, :3], np.ones((N, 1))], axis=1))
    ref_R = (Rotation.from_matrix(R) * Ru).as_matrix()
    ref_t = Rotation.from_matrix(R).apply(y[:, 3:]) + t
    assert np.abs(ref_R - R2).max() < 1e-12 and np.abs(ref_t - t2).max() < 1e-12


def test_padding_invariance_with_negative_control():
    d = SMALL
    N, L = 10, 7
    w = ps.make_struct_weights(9, d)
    m0, z, mask = _inputs(10, N, d, lengths=[L])
    kw = dict(n_layers=d.n_layers, n_torsion=d.n_torsion, **_kw(d))
    a = sr.structure_module(m0[0], z, mask, w, **kw)
    m2, z2 = m0[0].copy(), z.copy()
    m2[L:] *= 3.0
    z2[L:] *= -2.0
    z2[:, L:] += 5.0
    b = sr.structure_module(m2, z2, mask, w, **kw)
    for key in ("s", "R", "t", "alpha"):
        assert np.abs(a[key][:L] - b[key][:L]).max() < 1e-10, key
    crop = sr.structure_module(m0[0][:L], z[:L, :L], mask[:L], w, **kw)
    assert np.abs(a["s"][:L] - crop["s"]).max() < 1e-10
    z3 = z.copy()
    z3[1, 2, 0] += 3.0                                           # an unmasked pair does matter (one channel: LN_z removes a shift of all)
    c = sr.structure_module(m0[0], z3, mask, w, **kw)
    assert np.abs(a["s"][:L] - c["s"][:L]).max() > 1e-4


def test_angles_are_unit_vectors():
    d = SMALL
    w = ps.make_struct_weights(10, d)
    g = ps.rng(1, 9)
    al = sr.torsion_angles(g.standard_normal((5, d.c_s)), g.standard_normal((5, d.c_s)), w, d.n_torsion)
    assert al.shape == (5, d.n_torsion, 2) and np.abs((al ** 2).sum(-1) - 1.0).max() < 1e-9


def test_distogram_is_symmetric_and_matches_loops():
    d = SMALL
    w = ps.make_struct_weights(11, d)
    z = ps.rng(2, 9).standard_normal((4, 4, d.c_z))
    lg = sr.distogram_logits(z, w)
    assert np.abs(lg - np.transpose(lg, (1, 0, 2))).max() < 1e-14
    W, bb = w["w_dg"].astype(np.float64), w["b_dg"].astype(np.float64)
    for i in range(4):
        for j in range(4):
            for o in range(d.n_dist_bins):
                ref = sum((z[i, j, e] + z[j, i, e]) * W[e, o] for e in range(d.c_z)) + 2.0 * bb[o]
                assert abs(ref - lg[i, j, o]) < 1e-12


def test_masked_msa_head_is_a_row_linear():
    d = SMALL
    w = ps.make_struct_weights(12, d)
    m = ps.rng(4, 9).standard_normal((2, 3, d.c_m))
    lg = sr.masked_msa_logits(m, w)
    ref = torch.nn.functional.linear(torch.from_numpy(m), torch.from_numpy(w["w_mm"].astype(np.float64).T),
                                     torch.from_numpy(w["b_mm"].astype(np.float64))).numpy()
    assert lg.shape == (2, 3, d.n_msa_classes) and np.abs(lg - ref).max() < 1e-13


def test_plddt_closed_forms():
    d = SMALL
    w = dict(ps.make_struct_weights(13, d))
    s = ps.rng(5, 9).standard_normal((6, d.c_s))
    _, p = sr.plddt(s, w)
    assert (p >= 0).all() and (p <= 100).all()
    w["w_l3"] = np.zeros_like(w["w_l3"])
    for k in range(d.n_lddt_bins):
        b3 = np.full(d.n_lddt_bins, -1e4)
        b3[k] = 0.0
        w["b_l3"] = b3
        _, p = sr.plddt(s, w)
        assert np.abs(p - 100.0 * (k + 0.5) / d.n_lddt_bins).max() < 1e-9
    w["b_l3"] = np.zeros(d.n_lddt_bins)                          # uniform distribution: the mean of the bin centres
    _, p = sr.plddt(s, w)
    assert np.abs(p - 50.0).max() < 1e-9


def test_full_dims_run_and_shapes():
    w = ps.make_struct_weights(1)
    m, z, sm, _ = ps.make_inputs(3, 1, 2, 12, lengths=[10])
    o = sr.structure_module(m[0, 0], z[0], sm[0], w)
    assert o["s"].shape == (12, D.c_s) and o["alpha"].shape == (12, 7, 2) and o["x"].shape == (12, 3)
    assert np.abs(o["x"] - D.pos_scale * o["t"]).max() == 0.0
    assert all(np.isfinite(v).all() for v in o.values())
    assert len(ps.pack_struct_blob(w)) == ps.struct_floats()


def test_fold_composes_the_pinned_parts():
    """fold = recycled trunk (oracle/embed_ref.py, pinned in test_oracle_embed.py) + structure module per cycle; forcing the
    function's own positions back in changes nothing, forcing other positions changes the next cycle (negative control)."""
    from oracle import embed_ref
    S, N = 3, 10
    blocks = ps.make_weights(2, 1)
    we, wst = ps.make_embed_weights(2), ps.make_struct_weights(2)
    tf, ri, mf, _ = ps.make_features(5, 1, S, N)
    _, _, sm, mm = ps.make_inputs(5, 1, S, N, lengths=[8])
    kw = dict(struct_kw=dict(n_layers=2))
    one = sr.fold(tf[0], ri[0], mf[0], sm[0], mm[0], we, blocks, wst, 1, **kw)
    m1, z1 = embed_ref.recycled_trunk(tf[0], ri[0], mf[0], np.zeros((N, 3)), sm[0], mm[0], we, blocks, 1)
    assert np.abs(one["m"] - m1).max() == 0.0 and np.abs(one["z"] - z1).max() == 0.0
    ref = sr.structure_module(m1[0], z1, sm[0], wst, n_layers=2)
    assert np.abs(one["x_cycles"][0] - ref["x"]).max() == 0.0 and np.abs(one["s"] - ref["s"]).max() == 0.0
    two = sr.fold(tf[0], ri[0], mf[0], sm[0], mm[0], we, blocks, wst, 2, **kw)
    assert np.abs(two["x_cycles"][0] - one["x_cycles"][0]).max() == 0.0
    same = sr.fold(tf[0], ri[0], mf[0], sm[0], mm[0], we, blocks, wst, 2, x_forced=[two["x_cycles"][0]], **kw)
    assert np.abs(same["z"] - two["z"]).max() == 0.0
    # second cycle by hand: the recycling embedder sees the first cycle's m_0, z and positions
    m2, z2 = embed_ref.embed_cycle(tf[0], ri[0], mf[0], one["m"][0], one["z"], one["x_cycles"][0], we)
    from oracle import evoformer_trunk
    m2, z2 = evoformer_trunk(m2, z2, sm[0], mm[0], blocks, 32)
    assert np.abs(two["m"] - m2).max() < 1e-12 and np.abs(two["z"] - z2).max() < 1e-12
    other = sr.fold(tf[0], ri[0], mf[0], sm[0], mm[0], we, blocks, wst, 2, x_forced=[two["x_cycles"][0] * 3.0 + 7.0], **kw)
    v = sm[0] > 0
    assert np.abs(other["z"][np.ix_(v, v)] - two["z"][np.ix_(v, v)]).max() > 1e-3


def test_pae_and_resolved_heads_are_row_linears():
    """H.4 / H.5 against torch's linear; H.4 is not symmetric (unlike the distogram)."""
    d = SMALL
    w = ps.make_struct_weights(14, d)
    g = ps.rng(6, 9)
    z = g.standard_normal((4, 4, d.c_z))
    s = g.standard_normal((4, d.c_s))
    lin = torch.nn.functional.linear
    pae = sr.pae_logits(z, w)
    ref = lin(torch.from_numpy(z), torch.from_numpy(w["w_pae"].astype(np.float64).T), torch.from_numpy(w["b_pae"].astype(np.float64))).numpy()
    assert pae.shape == (4, 4, d.n_pae_bins) and np.abs(pae - ref).max() < 1e-13
    assert np.abs(pae - np.transpose(pae, (1, 0, 2))).max() > 1e-3
    er = sr.resolved_logits(s, w)
    ref = lin(torch.from_numpy(s), torch.from_numpy(w["w_er"].astype(np.float64).T), torch.from_numpy(w["b_er"].astype(np.float64))).numpy()
    assert er.shape == (4, d.n_resolved) and np.abs(er - ref).max() < 1e-13
