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


# ---------------------------------------------------------------------------------------------------------
# CFL sub-stepped frames (reading R24)
# ---------------------------------------------------------------------------------------------------------
def _substep_case(n=10, amp=1.5):
    P = wl.config2_params(n)
    bc = orc.BC(P["bc_types"], P["bc_values"])
    rng = np.random.default_rng(8)
    U0 = [amp * rng.standard_normal(s) for s in wl.face_shapes(n, n, n)]   # max|U| dt_frame / dx ~ 2.5: sub-steps
    dt_frame, rho = 1.0 / n, 2.0 / 1.0
    sf = lambda theta: (lambda t: wl.config2_solid(P, t / P["dt"], theta, dtype=np.float64))
    return P, bc, U0, dt_frame, rho, sf


def test_cfl_dt_policy():
    """dt = t_left / n with n the smallest integer that satisfies dt <= cfl dx / max|U| (R24)."""
    U = [np.array([[[0.0, -3.0]]]), np.array([[[1.0], [2.0]]]), np.array([[[0.5]], [[0.1]]])]
    assert orc.max_speed(U) == 3.0
    assert orc.cfl_dt(U, 1.0, 0.5, 1.0) == pytest.approx(1.0 / 6)      # 1.0 * 3 / 0.5 = 6 sub-steps
    assert orc.cfl_dt(U, 1.0, 0.5, 2.0) == pytest.approx(1.0 / 3)
    assert orc.cfl_dt(U, 0.1, 0.5, 1.0) == pytest.approx(0.1)          # already small enough: one step
    assert orc.cfl_dt([np.zeros((1, 1, 2))] * 3, 0.7, 0.5, 1.0) == 0.7  # fluid at rest
    assert orc.cfl_dt(U, 1.0, 0.5, 1.0, max_substeps=4) == pytest.approx(0.25)


def test_substepped_rollout_covers_the_frames_and_reduces_to_the_plain_rollout():
    P, bc, U0, dt_frame, rho, sf = _substep_case()
    loss = orc.loss_sum_u2(P["loss_lo"], P["loss_hi"])
    J, dJ, g, used = orc.rollout_substepped(U0, sf(0.5), 2, dt_frame, P["dx"], rho, bc, loss, cfl=1.0)
    assert all(len(d) >= 2 for d in used)                              # the CFL condition did cut the frames
    for d in used:
        assert sum(d) == pytest.approx(dt_frame, rel=1e-12)
    # every sub-step respected the condition with the velocity it started from: replaying the same sizes gives the
    # same answer, and a huge cfl (one sub-step per frame) is the plain rollout with dt = dt_frame
    J2, dJ2, _, _ = orc.rollout_substepped(U0, sf(0.5), 2, dt_frame, P["dx"], rho, bc, loss, dts=used)
    assert J2 == pytest.approx(J, rel=1e-13) and dJ2 == pytest.approx(dJ, rel=1e-10)
    J3, dJ3, g3, used3 = orc.rollout_substepped(U0, sf(0.5), 2, dt_frame, P["dx"], rho, bc, loss, cfl=1e9)
    assert [len(d) for d in used3] == [1, 1]
    Jp, dJp, gp = orc.rollout(U0, lambda s: wl.config2_solid(P, s * dt_frame / P["dt"], 0.5, dtype=np.float64), 2,
                              dt_frame, P["dx"], dt_frame / rho, bc, loss)
    assert J3 == pytest.approx(Jp, rel=1e-12) and dJ3 == pytest.approx(dJp, rel=1e-9)


def test_substepped_rollout_gradient_matches_finite_differences():
    """dJ/dtheta and dJ/dU0 through CFL sub-steps == central differences of the loss with the sub-step sizes held
    fixed (R24: dt is a constant of the backward pass; PAPER.md:L430-434 validates gradients the same way)."""
    P, bc, U0, dt_frame, rho, sf = _substep_case()
    loss = orc.loss_sum_u2(P["loss_lo"], P["loss_hi"])
    J, dJ, g, used = orc.rollout_substepped(U0, sf(0.5), 2, dt_frame, P["dx"], rho, bc, loss, cfl=1.0)
    h = 1e-5
    Jp = orc.rollout_substepped(U0, sf(0.5 + h), 2, dt_frame, P["dx"], rho, bc, loss, dts=used)[0]
    Jm = orc.rollout_substepped(U0, sf(0.5 - h), 2, dt_frame, P["dx"], rho, bc, loss, dts=used)[0]
    fd = (Jp - Jm) / (2 * h)
    assert abs(dJ - fd) <= 1e-6 * abs(fd)
    rng = np.random.default_rng(4)
    D = [rng.standard_normal(a.shape) for a in U0]
    h = 1e-6
    Jp = orc.rollout_substepped([a + h * d for a, d in zip(U0, D)], sf(0.5), 2, dt_frame, P["dx"], rho, bc, loss, dts=used)[0]
    Jm = orc.rollout_substepped([a - h * d for a, d in zip(U0, D)], sf(0.5), 2, dt_frame, P["dx"], rho, bc, loss, dts=used)[0]
    an = sum(float(np.sum(a * d)) for a, d in zip(g, D))
    assert abs(an - (Jp - Jm) / (2 * h)) <= 1e-6 * abs(an)
