"""Stand-ins for compute-sanitizer (closed on this GPU pool, profiles/r02_sanitizer.md): guard bands around the caller's
tensors and run-to-run bit identity of the tcgen05 path."""
import numpy as np
import pytest

import paper_2111_06340_b200 as pf
import pf_synth as ps
from gpu_util import errors, run_oracle, valid_masks

pytestmark = pytest.mark.gpu

GUARD = 4096          # floats on each side


def _guarded(a, dev):
    import torch
    flat = torch.full((a.size + 2 * GUARD,), -123456.75, device=dev, dtype=torch.float32)
    view = flat[GUARD:GUARD + a.size].view(*a.shape)
    view.copy_(torch.from_numpy(a))
    return flat, view


@pytest.mark.parametrize("B,S,N", [(2, 17, 50), (1, 3, 129), (2, 20, 72)])
def test_guard_bands_around_user_tensors_stay_intact(B, S, N):
    import torch
    dev = torch.device("cuda:0")
    blocks = ps.make_weights(121, 1, bf16_weights=True)
    lengths = ps.rng(122, N).integers(N // 2, N + 1, size=B)
    msa, pair, sm, mm = ps.make_inputs(123, B, S, N, lengths=lengths, msa_mask_frac_max=0.3)
    fm, m = _guarded(msa, dev)
    fz, z = _guarded(pair, dev)
    fs, smd = _guarded(sm, dev)
    fr, mmd = _guarded(mm, dev)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(1, pf.PF_BF16))
    h.forward(m, z, smd, mmd, 1)
    torch.cuda.synchronize()
    h.close()
    for name, flat in (("msa", fm), ("pair", fz), ("seq_mask", fs), ("msa_mask", fr)):
        g = torch.cat([flat[:GUARD], flat[-GUARD:]])
        assert bool((g == -123456.75).all()), f"guard band of {name} was written"
    assert np.array_equal(smd.cpu().numpy(), sm) and np.array_equal(mmd.cpu().numpy(), mm)
    mr, zr = run_oracle(blocks, msa, pair, sm, mm)
    vm, vz = valid_masks(sm, mm)
    em, rm = errors(m.cpu().numpy(), mr, vm)
    ez, rz = errors(z.cpu().numpy(), zr, vz)
    assert em <= 3e-2 and ez <= 3e-2 and rm <= 1e-2 and rz <= 1e-2


def test_repeated_runs_are_bit_identical():
    import torch
    dev = torch.device("cuda:0")
    B, S, N, nb = 3, 96, 200, 2
    blocks = ps.make_weights(124, nb, bf16_weights=True)
    msa, pair, sm, mm = ps.make_inputs(125, B, S, N, lengths=[200, 131, 77], msa_mask_frac_max=0.3)
    smd, mmd = torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev)
    vm, vz = valid_masks(sm, mm)
    outs = []
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
    for rep in range(4):
        if rep == 3:
            h.close()
            h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
        m, z = torch.from_numpy(msa).to(dev), torch.from_numpy(pair).to(dev)
        h.forward(m, z, smd, mmd, nb)
        torch.cuda.synchronize()
        outs.append((m.cpu().numpy()[vm], z.cpu().numpy()[vz]))
    h.close()
    for mo, zo in outs[1:]:
        assert np.array_equal(mo, outs[0][0]) and np.array_equal(zo, outs[0][1])
