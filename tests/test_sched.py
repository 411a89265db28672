"""Length-bucketing batch scheduler (host logic, no GPU): PAPER.md:113, SURVEY.md §3(iv)."""
import pytest
from hypothesis import given, settings
from hypothesis import strategies as st

import paper_2111_06340_b200 as pf
import pf_synth as ps

BUCKETS = list(ps.CFG5_BUCKETS)


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2111_06340_b200 import build
    build.build()


@settings(max_examples=60, deadline=None)
@given(lengths=st.lists(st.integers(1, 320), min_size=0, max_size=200),
       budget_gb=st.integers(0, 64), S=st.sampled_from([1, 128, 512]))
def test_every_protein_once_bucket_fits_budget_respected(lengths, budget_gb, S):
    budget = budget_gb << 30
    s = pf.Scheduler(BUCKETS, budget, S)
    for i, L in enumerate(lengths):
        s.add(i, L)
    seen = []
    prev_bucket = None
    for ids, lens, bucket in s.batches():
        assert bucket in BUCKETS
        assert all(L <= bucket for L in lens)
        smaller = [b for b in BUCKETS if b < bucket]
        assert all(not smaller or L > smaller[-1] for L in lens)       # smallest bucket that fits
        per = pf.bytes_per_protein(bucket, S)
        assert len(ids) == 1 or len(ids) * per <= budget               # budget respected (a single protein always runs)
        assert [lengths[i] for i in ids] == lens
        if prev_bucket is not None:
            assert bucket <= prev_bucket                               # largest first
        prev_bucket = bucket
        seen += ids
    assert sorted(seen) == list(range(len(lengths)))
    s.close()


def test_rejects_bad_input():
    with pytest.raises(pf.PfError):
        pf.Scheduler([128, 64], 1 << 30, 128)
    s = pf.Scheduler(BUCKETS, 1 << 30, 128)
    with pytest.raises(pf.PfError):
        s.add(0, 321)
    with pytest.raises(pf.PfError):
        s.add(0, 0)


def test_cfg5_bucket_population():
    """R10: the log-normal length law populates all five buckets."""
    lens = ps.cfg5_lengths(5)
    s = pf.Scheduler(BUCKETS, 8 << 30, 512)
    for i, L in enumerate(lens):
        s.add(i, int(L))
    counts = {b: 0 for b in BUCKETS}
    for ids, _, bucket in s.batches():
        counts[bucket] += len(ids)
    assert sum(counts.values()) == 2000 and all(v > 20 for v in counts.values())
