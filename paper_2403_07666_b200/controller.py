"""Caller-side adaptive time-step controller for config 3 (BASELINE.json configs[3]:
"adaptive dt in [1e-6, 1e-4] s").  Host logic only: dt is an argument of qs_step, the library reports
max_c |J^{k+1} - J^k| (qs_stats_t.dJ_max) and the event word; this module turns them into the next dt.

Rule (C11): s = dJ_max / J_ref with J_ref = Jc0 (1 - T_bath/Tc)^2;  s > 0.02 -> dt = max(dt/2, dt_min);
s < 0.005 -> dt = min(2 dt, dt_max);  any event flag -> dt = dt_min for the next `hold` steps.
"""
from __future__ import annotations

import dataclasses


@dataclasses.dataclass
class AdaptiveDt:
    J_ref: float
    dt: float = 1e-4
    dt_min: float = 1e-6
    dt_max: float = 1e-4
    shrink_above: float = 0.02
    grow_below: float = 0.005
    hold: int = 10
    _held: int = 0

    def update(self, dJ_max: float, event_word: int) -> float:
        """Digest the outcome of the step just taken with self.dt; returns the dt of the next step."""
        if event_word & 3:                       # flux jump started or quench flag set
            self._held = self.hold
        if self._held > 0:
            self._held -= 1
            self.dt = self.dt_min
            return self.dt
        s = dJ_max / self.J_ref
        if s > self.shrink_above:
            self.dt = max(0.5 * self.dt, self.dt_min)
        elif s < self.grow_below:
            self.dt = min(2.0 * self.dt, self.dt_max)
        return self.dt


def reference_current_density(material, geometry) -> float:
    """J_ref of C11: Jc0 (1 - T_bath/Tc)^2."""
    return material.Jc0 * (1.0 - geometry.T_bath / material.Tc) ** 2


def run_adaptive(sim, geometry, material, I_ramp: float, steps: int, dt0: float = 1e-4, on_step=None):
    """Advance `sim` (a QS handle) `steps` steps under the C11 controller; returns the list of dt taken."""
    ctl = AdaptiveDt(J_ref=reference_current_density(material, geometry), dt=dt0)
    taken = []
    for _ in range(steps):
        dt = ctl.dt
        rc = sim.step(dt, I_ramp)
        st = sim.stats()
        taken.append(dt)
        if on_step is not None:
            on_step(dt, rc, st)
        ctl.update(st["dJ_max"], rc)
    return taken
