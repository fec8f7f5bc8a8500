"""Seeded synthetic input generators shared by the oracle tests, the CUDA parity tests and bench.py.

This module holds NONE of the method's arithmetic (no lens equation, no polynomial, no areas): it only
produces source centres zeta (centre-of-mass frame, Einstein-radius units), lens parameters (s, q), source
radii rho and the model indirection, with the shapes and distributions BASELINE.json's five configs name.
The recipes are stated in DESIGN.md ("Input recipe") and follow SURVEY.md section 8(d).

Conventions
-----------
* Frame: the paper's centre-of-mass frame (Eq. 2): primary at z1 = -q s/(1+q), secondary at
  z2 = +s/(1+q), both on the real axis.
* Trajectory: zeta(tau) = -(tau + i u0) e^{i alpha} + o with tau = (t - t0)/tE; o = z1 where the config says
  "primary at origin" (configs 1, 2) and o = 0 otherwise (config 3).  With this sign the source passes the
  origin on the planet's side for u0 > 0, alpha in (0, pi), which is what realises config 2's
  "central-caustic crossing".
* RNG: numpy.random.default_rng(seed); arrays are drawn in the order listed, whole-array draws.
"""
from .configs import (Workload, config1, config2, config3, config4, config5, domain_corners, fig1_case, fig2_case,
                      fig5_map, fig6_case, fig7_grid, get, lowq_sweep, trajectory)

__all__ = ["Workload", "config1", "config2", "config3", "config4", "config5", "fig1_case", "fig2_case",
           "fig5_map", "fig6_case", "fig7_grid", "lowq_sweep", "domain_corners", "get", "trajectory"]
