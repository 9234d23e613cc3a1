"""SLO-aware latency controller (PAPER.md 4.5; include/bm.h bm_salc_*): host logic, no GPU.
The expected values are worked out by hand from the rule the paper states and DESIGN.md reading A21."""
import math

import pytest
import torch


def test_threshold_starts_at_no_merging_and_follows_p259():
    import paper_2607_04164_b200 as bm
    c = bm.Salc(slo=100.0, warn_frac=0.8, decrease=0.5, increase=0.1, window=4)
    assert c.threshold == 1.0                                   # threshold = 1.0, no merging
    # inside the band [80, 100]: nothing moves
    assert c.observe(90.0) == 1.0 and c.observe(95.0) == 1.0
    # window (90, 95, 120): P90 = ceil(0.9*3) = 3rd smallest = 120 > SLO -> multiplicative decrease
    assert c.observe(120.0) == 0.5
    # window (90, 95, 120, 70): P90 = ceil(3.6) = 4th smallest = 120 -> again
    assert c.observe(70.0) == 0.25
    # the window slides: (95, 120, 70, 60) still holds 120
    assert c.observe(60.0) == 0.125
    # (120, 70, 60, 50) -> 0.0625; then 120 leaves: (70, 60, 50, 40): P90 = 70 < 80 -> linear increase
    assert c.observe(50.0) == 0.0625
    assert c.observe(40.0) == pytest.approx(0.1625)
    assert c.p90() == 70.0
    for _ in range(20):                                          # saturates at 1
        c.observe(10.0)
    assert c.threshold == 1.0


def test_p90_is_nearest_rank():
    import paper_2607_04164_b200 as bm
    c = bm.Salc(slo=1e9, warn_frac=1e-9, window=10)
    vals = [5, 1, 9, 3, 7, 2, 8, 4, 6, 10]
    for i, v in enumerate(vals, 1):
        c.observe(float(v))
        assert c.p90() == sorted(vals[:i])[math.ceil(0.9 * i) - 1]
    assert c.threshold == 1.0                                   # never left the band


def test_bad_arguments():
    import paper_2607_04164_b200 as bm
    for kw in (dict(slo=0.0), dict(slo=1.0, decrease=1.0), dict(slo=1.0, increase=0.0), dict(slo=1.0, window=0),
               dict(slo=1.0, window=257), dict(slo=1.0, warn_frac=1.5)):
        with pytest.raises(bm.BmError):
            bm.Salc(**kw)


def test_cold_mask_from_threshold():
    import paper_2607_04164_b200 as bm
    w = torch.tensor([50, 3, 20, 3, 0, 7, 90, 1], dtype=torch.int32)
    assert bm.bm_salc_cold_mask(w, 1.0).tolist() == [0] * 8      # zero brownout
    assert bm.bm_salc_cold_mask(w, 0.0).tolist() == [1] * 8      # full brownout
    # threshold 0.5 -> the 4 least-used experts: e4 (0), e7 (1), then the tie 3 = 3 -> lower index first: e1, e3
    assert bm.bm_salc_cold_mask(w, 0.5).tolist() == [0, 1, 0, 1, 1, 0, 0, 1]
    # threshold 0.625 -> round(0.375 * 8) = 3 coldest: e4, e7, e1
    assert bm.bm_salc_cold_mask(w, 0.625).tolist() == [0, 1, 0, 0, 1, 0, 0, 1]
    with pytest.raises(bm.BmError):
        bm.bm_salc_cold_mask(w, 1.5)
