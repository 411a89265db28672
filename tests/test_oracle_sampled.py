"""Pin the sampled-output oracle (oracle/evoformer_sampled.py) to the full-tensor oracle, which carries the pins of
tests/test_oracle_pins.py and tests/test_oracle_bruteforce.py: at EVERY position of a small ragged problem (a hole in
seq_mask, masked MSA rows, AlphaFold channel dims) the one-position functions must reproduce the full-tensor result to
1e-12, in plain mode and with the rounding switch constructed but off.  The quantisation-aware mode (R16) is a model of
the storage formats, not a definition: it is only required to stay close to the plain result (well inside the bf16
tolerances) and to actually differ from it (the switch does something).
"""
import numpy as np
import pytest

import oracle
import pf_synth as ps
from oracle import evoformer_sampled as sm


@pytest.fixture(scope="module")
def case():
    S, N = 5, 9
    w = ps.make_block_weights(71, 0, ps.AF2, bf16_weights=True)
    msa, pair, _, _ = ps.make_inputs(72, 1, S, N)
    sig = np.ones(N)
    sig[[3, 7, 8]] = 0          # a hole and a padded tail
    rho = np.ones(S)
    rho[2] = 0
    return w, msa[0].astype(np.float64), pair[0].astype(np.float64), sig, rho


@pytest.mark.parametrize("step", range(1, 10))
@pytest.mark.parametrize("rnd", [None, sm.Rounding(False)])
def test_every_position_matches_full_oracle(case, step, rnd):
    w, m, z, sig, rho = case
    mr, zr = oracle.substep(step, m, z, sig, rho, w)
    ms, zs = sm.substep_all(step, m, z, sig, rho, w, rnd=rnd)
    assert np.abs(ms - mr).max() < 1e-12 and np.abs(zs - zr).max() < 1e-12


def test_sampled_positions_on_a_non_square_problem():
    """Index order: S != N and distinct (s, i) / (i, j) so that a swapped index pair cannot cancel."""
    S, N = 7, 4
    w = ps.make_block_weights(73, 0, ps.AF2)
    msa, pair, _, _ = ps.make_inputs(74, 1, S, N)
    m, z = msa[0].astype(np.float64), pair[0].astype(np.float64)
    sig, rho = np.array([1.0, 1, 0, 1]), np.array([1.0, 0, 1, 1, 1, 0, 1])
    for step in range(1, 10):
        mr, zr = oracle.substep(step, m, z, sig, rho, w)
        for pos in ((6, 1), (0, 3)) if step <= 3 else ((3, 0), (1, 3)):
            got = sm.substep_at(step, m, z, sig, rho, w, pos)
            ref = (mr if step <= 3 else zr)[pos]
            assert np.abs(got - ref).max() < 1e-12, (step, pos)


def test_float32_inputs_are_accepted(case):
    """The GPU tests hand fp32 arrays (the residual streams as the CUDA path saw them): same values as their fp64 copies."""
    w, m, z, sig, rho = case
    m32, z32 = m.astype(np.float32), z.astype(np.float32)
    for step, pos in ((1, (1, 4)), (4, (2, 5)), (6, (5, 1)), (8, (0, 6))):
        a = sm.substep_at(step, m32, z32, sig.astype(np.float32), rho.astype(np.float32), w, pos)
        b = sm.substep_at(step, m32.astype(np.float64), z32.astype(np.float64), sig, rho, w, pos)
        assert np.array_equal(a, b)


def test_rounding_helpers():
    r = sm.Rounding(True)
    x = np.array([1.0, 1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -9, -3.14159, 1e-30, 65504.0])
    b = r.bf16(x)
    assert b[0] == 1.0 and b[1] == 1.0 and b[2] == 1.0 + 2.0 ** -7      # ties to even, then round up
    assert abs(b[3] + 3.14159) <= 2.0 ** -7 and b[4] > 0
    h = r.f16(x)
    assert h[1] == 1.0 + 2.0 ** -8 and h[4] == 0.0 and h[5] == 65504.0  # 11-bit mantissa; flush below the subnormals
    assert np.array_equal(sm.Rounding(False).bf16(x), x) and np.array_equal(sm.Rounding(False).f16(x), x)
    g = r.gate(np.array([0.0, 30.0, -30.0]))
    assert g[0] == 0.5 and g[1] == 1.0 and 0.0 <= g[2] < 1e-7


@pytest.mark.parametrize("step", range(1, 10))
def test_quantised_mode_is_close_but_not_identical(case, step):
    w, m, z, sig, rho = case
    mr, zr = oracle.substep(step, m, z, sig, rho, w)
    mq, zq = sm.substep_all(step, m, z, sig, rho, w, rnd=sm.Rounding(True))
    vm = (rho[:, None] * sig[None, :]) > 0
    vz = (sig[:, None] * sig[None, :]) > 0
    d = np.abs(mq - mr)[vm].max() if step <= 3 else np.abs(zq - zr)[vz].max()
    assert 0.0 < d < 3e-2, (step, d)
