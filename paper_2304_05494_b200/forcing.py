"""Bulk-flow controller of a forced channel: host logic on top of the C ABI ("forcing term evaluations (sum
reduction)").  Every step it reads the volume integrals of the state (streams_get_sums, fixed-order reductions on the
device) and resets the uniform streamwise acceleration (streams_set_body_force) so that the bulk momentum returns to its
target: with M = sum(rho dV) and P = sum(rho u dV), a force g acting over the next step changes P by g M dt, so
g <- g_balance + (P_target - P) / (M dt), where g_balance is the running estimate of the force that balances the wall
friction (the previous g corrected by the drift it left).  No field data leaves the device."""
from __future__ import annotations


class BulkFlowController:
    def __init__(self, solver, direction: int = 0, target=None):
        self.s = solver
        self.d = direction
        sums = solver.get_sums(0)
        self.target = float(sums[1 + direction]) if target is None else float(target)
        self.g = [0.0, 0.0, 0.0]
        self.prev_p = float(sums[1 + direction])

    def step(self, nsteps: int = 1):
        """Advance nsteps steps, one at a time, re-evaluating the force after each.  Returns (dt, time, g, P / P_target)."""
        dt = t = 0.0
        ratio = 1.0
        for _ in range(nsteps):
            dt, t = self.s.step(1)
            sums = self.s.get_sums(0)
            mass, p = float(sums[0]), float(sums[1 + self.d])
            # the force that would have kept P constant over the step just taken ...
            g_balance = self.g[self.d] - (p - self.prev_p) / (mass * dt)
            # ... plus what brings P back to the target over the next one
            self.g[self.d] = g_balance + (self.target - p) / (mass * dt)
            self.s.set_body_force(self.g)
            self.prev_p = p
            ratio = p / self.target if self.target != 0.0 else 1.0
        return dt, t, list(self.g), ratio
