"""accLB_stats_increments_static: the structure functions through the entry point that allocates nothing (its accumulators
are a fixed `static __device__` array inside the library) against the existing path accLB_stats_increments (caller-owned
scratch block), on two calls in a row with different inputs -- the shared array keeps the last call's contents, so the
second call shows that it is cleared.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2505_01126_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-11  # the tolerance of tests/test_stats.py: |difference| / S_2^{p/2}; the two paths differ by the order of the atomic adds


def close(a, b):
    a, b = np.array(a), np.array(b)
    scale = b[:, :1] ** (np.array([2, 3, 4]) / 2.0)
    return (np.abs(a - b) / scale).max() < TOL


def test_static_scratch_entry_point_matches_the_scratch_block_path(acclb):
    import torch

    n = 64
    ua = torch.from_numpy(np.ascontiguousarray(wl.hit_velocity(n))).cuda()
    rng = np.random.default_rng(11)
    ub = torch.from_numpy(rng.standard_normal((3, 20, 12, 30))).cuda()   # non-cubic, other magnitudes (sums ~1e5 times larger)
    ra, rb = [1, 2, 3, 4, 8, 16, 31], [5, 1]
    want_a, want_b = acclb.stats_increments(ua, ra), acclb.stats_increments(ub, rb)
    acclb.stats_increments_static(ua, [1])                               # warm-up: the symbol address is looked up once per device
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    got_a = acclb.stats_increments_static(ua, ra)                        # first call
    got_b = acclb.stats_increments_static(ub, rb)                        # second call: fewer separations, other field
    got_a2 = acclb.stats_increments_static(ua, ra)                       # and back
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                         # no device allocation behind the caller's back
    assert close(got_a, want_a), (got_a, want_a)
    assert close(got_b, want_b), (got_b, want_b)
    assert close(got_a2, want_a), (got_a2, want_a)
    # the limit: at most STATS_STATIC_MAX_NR separations; beyond that a clear error and no launch
    assert acclb.STATS_STATIC_MAX_NR == 64
    r64 = list(range(60)) + [61, 62, 63, 64]                             # (60 is a period of all three axes of ub: S = 0 there)
    full = acclb.stats_increments_static(ub, r64)
    assert close(full[1:], acclb.stats_increments(ub, r64[1:])) and full[0] == [0.0, 0.0, 0.0]
    with pytest.raises(acclb.AccLBError, match="at most 64"):
        acclb.stats_increments_static(ub, list(range(65)))
    with pytest.raises(acclb.AccLBError):
        acclb.stats_increments_static(ub, [-1])
    # a non-default stream
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        s.wait_stream(torch.cuda.default_stream())
        assert close(acclb.stats_increments_static(ua, ra), want_a)
