"""pf_plddt_forward_static (include/pf_evoformer.h): the pLDDT head H.3 with its intermediates in a file-scope device array,
for callers that cannot call cudaMalloc.  Checked against the existing path (the pLDDT tail of pf_structure_forward, whose
workspace is cudaMalloc'ed) on two calls in a row that share the array, against the fp64 oracle on a cold start, and for the
size limit.  Tolerance: the one tests/test_gpu_structure.py uses for pLDDT (1e-3 max-abs on a 0..100 scale); the two paths run
the same kernels, so they are expected to agree exactly.  Named test_zz_* so that pytest collects it last."""
import numpy as np
import pytest

import paper_2111_06340_b200 as pf
import pf_synth as ps
from oracle import structure_ref as sr

pytestmark = pytest.mark.gpu

TOL_PLDDT = 1e-3
D = ps.STRUCT
MAX_ROWS = 3039          # default dims: rows * (384 + 2 * 128 + 50) floats, segments rounded to 256 B, in 8 MiB


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_static_scratch_cold_start_matches_oracle():
    """The new entry point is the first thing this handle runs: the array's device address is resolved inside the call."""
    import torch
    w = ps.make_struct_weights(21)
    h = pf.StructureModule(ps.pack_struct_blob(w), pf.make_struct_config())
    s = ps.rng(22, 1).standard_normal((77, D.c_s)).astype(np.float32) * 2.0
    out = torch.full((77,), -1.0, device="cuda")
    h.plddt_static(_dev(s), out)
    torch.cuda.synchronize()
    assert h.last_launch_count() == 5
    _, ref = sr.plddt(s.astype(np.float64), w)
    h.close()
    assert np.abs(out.cpu().numpy() - ref).max() <= TOL_PLDDT


def test_static_scratch_matches_existing_path_twice_in_a_row():
    """Existing path: pf_structure_forward (s_out, plddt_out).  New path on that s_out, two calls back to back: a large batch, then
    a smaller one that leaves the first call's values in the rest of the shared array, then the large one again."""
    import torch
    w = ps.make_struct_weights(5)
    h = pf.StructureModule(ps.pack_struct_blob(w), pf.make_struct_config())
    cases = []
    for seed, (B, S, N, lengths) in enumerate([(2, 2, 150, [150, 131]), (1, 3, 45, None)]):
        msa, pair, sm, _ = ps.make_inputs(30 + seed, B, S, N, lengths=lengths)
        s = torch.empty((B, N, D.c_s), device="cuda")
        pl = torch.empty((B, N), device="cuda")
        h.forward(_dev(msa), _dev(pair), _dev(sm), 2, s_out=s, plddt_out=pl)
        torch.cuda.synchronize()
        cases.append((s, pl))
    free0, _ = torch.cuda.mem_get_info()
    outs = [torch.full_like(pl, float("nan")) for _, pl in cases] + [torch.full_like(cases[0][1], float("nan"))]
    h.plddt_static(cases[0][0], outs[0])
    h.plddt_static(cases[1][0], outs[1])         # same stream: ordered after the first, reuses the same array
    h.plddt_static(cases[0][0], outs[2])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    h.close()
    assert free0 - free1 < (1 << 20), "the allocation-free entry point took device memory"
    for got, (_, want) in zip(outs, [cases[0], cases[1], cases[0]]):
        g, r = got.cpu().numpy(), want.cpu().numpy()
        assert np.isfinite(g).all()
        assert np.abs(g - r).max() <= TOL_PLDDT
        assert np.array_equal(g, r)              # same kernels, same order of operations


def test_static_scratch_limit():
    import torch
    w = ps.make_struct_weights(5)
    h = pf.StructureModule(ps.pack_struct_blob(w), pf.make_struct_config())
    s = torch.zeros((MAX_ROWS + 1, D.c_s), device="cuda")
    s[:MAX_ROWS] = _dev(ps.rng(23, 1).standard_normal((MAX_ROWS, D.c_s)).astype(np.float32))
    out = torch.full((MAX_ROWS + 1,), -1.0, device="cuda")
    h.plddt_static(s[:MAX_ROWS], out[:MAX_ROWS])           # the largest size the array holds
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    idx = [0, 1, MAX_ROWS // 2, MAX_ROWS - 2, MAX_ROWS - 1]
    _, ref = sr.plddt(s[idx].cpu().numpy().astype(np.float64), w)
    assert np.abs(got[idx] - ref).max() <= TOL_PLDDT
    assert got[MAX_ROWS] == -1.0
    with pytest.raises(pf.PfError, match="static array holds"):
        h.plddt_static(s, out)
    with pytest.raises(pf.PfError):
        h.plddt_static(s[:0], out[:0])
    h.close()
