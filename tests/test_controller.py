"""CPU tests of the caller-side adaptive time-step controller (C11)."""
from paper_2403_07666_b200.controller import AdaptiveDt


def test_halves_doubles_and_clamps():
    c = AdaptiveDt(J_ref=1.0, dt=1e-4)
    assert c.update(0.03, 0) == 5e-5            # s > 0.02: halve
    assert c.update(0.03, 0) == 2.5e-5
    assert c.update(0.01, 0) == 2.5e-5          # between the thresholds: keep
    assert c.update(0.001, 0) == 5e-5           # s < 0.005: double
    assert c.update(0.0, 0) == 1e-4 and c.update(0.0, 0) == 1e-4      # clamped at dt_max
    for _ in range(12):
        c.update(1.0, 0)
    assert c.dt == 1e-6                          # clamped at dt_min


def test_event_holds_dt_min_for_ten_steps():
    c = AdaptiveDt(J_ref=1.0, dt=1e-4)
    assert c.update(0.0, 1) == 1e-6              # an event: dt_min for the next 10 steps
    for _ in range(9):
        assert c.update(0.0, 0) == 1e-6
    assert c.update(0.0, 0) == 2e-6              # released: grows again
    assert c.update(0.0, 4) == 4e-6              # bit 2 (CG maxit) is not an event
