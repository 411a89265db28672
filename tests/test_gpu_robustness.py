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


def test_tmem_operand_kernels_bit_identical_under_load():
    """The transition, outer-product and attention kernels keep the intermediate of their two chained GEMMs in tensor memory and
    let a later tcgen05.mma overwrite columns an earlier one of the same thread read as its A operand, relying on issue-order
    execution (no barrier in between).  A violated ordering would show as run-to-run differences once every SM works through
    many tiles: eight repetitions of one block at a batch that gives each persistent CTA dozens of tiles must agree bit for
    bit on every valid element."""
    import torch
    dev = torch.device("cuda:0")
    B, S, N, nb = 24, 128, 128, 1
    blocks = ps.make_weights(131, nb, bf16_weights=True)
    msa, pair, sm, mm = ps.make_inputs(132, B, S, N, lengths=[128 - 3 * i for i in range(B)], msa_mask_frac_max=0.3)
    smd, mmd = torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev)
    m0, z0 = torch.from_numpy(msa).to(dev), torch.from_numpy(pair).to(dev)
    vm, vz = valid_masks(sm, mm)
    vmd, vzd = torch.from_numpy(vm).to(dev), torch.from_numpy(vz).to(dev)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
    ref = None
    for rep in range(8):
        m, z = m0.clone(), z0.clone()
        h.forward(m, z, smd, mmd, nb)
        torch.cuda.synchronize()
        m, z = m[vmd], z[vzd]
        assert bool(torch.isfinite(m).all()) and bool(torch.isfinite(z).all())
        if ref is None:
            ref = (m, z)
        else:
            assert torch.equal(m, ref[0]) and torch.equal(z, ref[1]), f"run {rep} differs from run 0"
    h.close()


def test_cuda_graph_replay_matches_direct_launches():
    """Small shapes are launch-bound, so whole forward calls on them are captured into a CUDA graph per (buffers, shape) and
    replayed (pf_api.cu, dispatch_pass).  The graph holds the mask-flag kernels too, so changing the CONTENTS of the masks
    between replays must give what a direct launch sequence gives (profiling on = no graph), bit for bit."""
    import torch
    B, S, N, nb = 2, 10, 72, 2
    blocks = ps.make_weights(61, nb, bf16_weights=True)
    msa, pair, sm1, mm1 = ps.make_inputs(62, B, S, N, lengths=[72, 50], msa_mask_frac_max=0.3)
    _, _, sm2, mm2 = ps.make_inputs(63, B, S, N, lengths=[33, 72], msa_mask_frac_max=0.3)
    hg = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
    hd = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
    hd.set_profiling(True)
    m = torch.empty((B, S, N, 256), device="cuda")
    z = torch.empty((B, N, N, 128), device="cuda")
    smd = torch.empty((B, N), device="cuda")
    mmd = torch.empty((B, S), device="cuda")
    outs = {}
    for tag, h in (("graph", hg), ("direct", hd)):
        for k, (sm, mm) in enumerate(((sm1, mm1), (sm2, mm2), (sm1, mm1))):
            m.copy_(torch.from_numpy(msa))
            z.copy_(torch.from_numpy(pair))
            smd.copy_(torch.from_numpy(sm))
            mmd.copy_(torch.from_numpy(mm))
            h.forward(m, z, smd, mmd, nb)          # same buffers every time: the second and third call replay the graph
            torch.cuda.synchronize()
            outs[(tag, k)] = (m.cpu().numpy().copy(), z.cpu().numpy().copy())
    hg.close()
    hd.close()
    for k, (sm, mm) in enumerate(((sm1, mm1), (sm2, mm2), (sm1, mm1))):
        vm = (mm[:, :, None] * sm[:, None, :]) > 0
        vz = (sm[:, :, None] * sm[:, None, :]) > 0
        assert np.isfinite(outs[("graph", k)][0]).all() and np.isfinite(outs[("graph", k)][1]).all()
        assert np.array_equal(outs[("graph", k)][0][vm], outs[("direct", k)][0][vm]), k
        assert np.array_equal(outs[("graph", k)][1][vz], outs[("direct", k)][1][vz]), k
