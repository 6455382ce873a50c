"""measurement aids of the boundary (pd_measure_fp64_rate, pd_measure_pair_exchange): they run, allocate nothing that
stays, and agree with each other where they time the same thing."""
import pytest

pytestmark = pytest.mark.gpu


def test_issue_rate_probes_run_and_agree():
    from paper_2309_11273_b200 import pd
    pd.measure_pair_exchange(2)                         # brings the clocks up: the figures below are compared with each other
    r = pd.measure_pair_exchange(3)
    assert set(r) == {"dfma_per_s", "shift64_per_s", "shift64_plus_5dfma_per_s", "smem_double_per_s"}
    assert all(v > 1e10 for v in r.values())
    f = pd.measure_fp64_rate(3)
    assert 0.6 <= r["dfma_per_s"] / f <= 1.6           # the same DFMA stream, timed by two kernels
    # a group holds 5 DFMA: it cannot run faster than the FP64 pipe alone allows
    assert r["shift64_plus_5dfma_per_s"] * 5.0 <= max(r["dfma_per_s"], f) * 1.25
