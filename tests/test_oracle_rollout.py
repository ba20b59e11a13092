"""Pins of the oracle's full-step rollout (forward + backward pass): the end-to-end
parameter gradient against central finite differences of the loss (the paper's own validation method,
PAPER.md:L430-434, App. F) and against a closed form."""
import numpy as np
import pytest

from oracle import nf_oracle as orc
from paper_2405_14903_b200 import workloads as wl


def _case(n):
    P = wl.config2_params(n)
    bc = orc.BC(P["bc_types"], P["bc_values"])
    U0 = [np.zeros(s) for s in wl.face_shapes(n, n, n)]
    return P, bc, U0


def test_rollout_gradient_matches_finite_differences():
    """BASELINE.json configs[1] shape at 12^3, 3 steps: dJ/dtheta through advection, projection, the weight
    builder and the solid velocity == central difference of J (h = 1e-5; the paper uses 1.2e-5)."""
    P, bc, U0 = _case(12)
    loss = orc.loss_sum_u2(P["loss_lo"], P["loss_hi"])

    def run(theta):
        return orc.rollout(U0, lambda s: wl.config2_solid(P, s, theta, dtype=np.float64), 3, P["dt"], P["dx"],
                           P["dt_over_rho"], bc, loss)

    J, dJ, _ = run(0.5)
    h = 1e-5
    fd = (run(0.5 + h)[0] - run(0.5 - h)[0]) / (2 * h)
    assert J > 0
    assert abs(dJ - fd) <= 1e-7 * abs(fd)


def test_rollout_gradient_wrt_initial_velocity_finite_differences():
    """dJ/dU0 in a random direction == directional central difference (moving plates, random initial velocity)."""
    P, bc, _ = _case(10)
    rng = np.random.default_rng(3)
    U0 = [0.3 * rng.standard_normal(s) for s in wl.face_shapes(10, 10, 10)]
    D = [rng.standard_normal(s) for s in wl.face_shapes(10, 10, 10)]
    loss = orc.loss_sum_u2(P["loss_lo"], P["loss_hi"])
    sf = lambda s: wl.config2_solid(P, s, 0.5, dtype=np.float64)

    def run(eps):
        return orc.rollout([a + eps * d for a, d in zip(U0, D)], sf, 2, P["dt"], P["dx"], P["dt_over_rho"], bc, loss)

    _, _, g = run(0.0)
    h = 1e-6
    fd = (run(h)[0] - run(-h)[0]) / (2 * h)
    an = sum(float(np.sum(a * d)) for a, d in zip(g, D))
    assert abs(an - fd) <= 1e-6 * max(abs(fd), 1e-12)


def test_rollout_frozen_geometry_closed_form():
    """Geometry frozen (phi of theta_0 at every step, d phi/d theta = 0), advection off, fluid at rest: U is linear
    in theta through U_s only, so J = C theta^2 and dJ/dtheta = 2 J / theta exactly."""
    P, bc, U0 = _case(12)
    loss = orc.loss_sum_u2(P["loss_lo"], P["loss_hi"])
    theta = 0.37

    def sf(step):
        phi, _, _, _ = wl.config2_solid(P, step, 0.5, dtype=np.float64)   # frozen shape
        _, us, _, dus = wl.config2_solid(P, step, theta, dtype=np.float64)  # velocity of amplitude theta
        return phi, us, np.zeros_like(phi), dus

    J, dJ, _ = orc.rollout(U0, sf, 2, P["dt"], P["dx"], P["dt_over_rho"], bc, loss, advect_on=False)
    assert J > 0
    assert abs(dJ - 2 * J / theta) <= 1e-9 * abs(dJ)
