"""Pins of the oracle's viscosity step (Eq. 3, L359-361 Eq. 13): closed-form
eigenmodes, conservation, symmetry (the backward pass applies the same matrix, Eq. 8), the explicit heat-equation
limit, and the end-to-end rollout gradient with viscosity against finite differences."""
import numpy as np

from oracle import nf_oracle as orc
from paper_2405_14903_b200 import workloads as wl


def test_viscosity_cosine_eigenmode_closed_form():
    """On a lattice with nothing outside it G^T G is diagonalised by the DCT-II modes cos(pi m (i + 1/2) / n) with
    eigenvalue 2 - 2 cos(pi m / n) per axis: one mode per component, different lattices."""
    nx, ny, nz = 9, 6, 5
    shapes = wl.face_shapes(nx, ny, nz)
    nu, dt, dx = 0.37, 0.01, 0.1
    k = nu * dt / dx ** 2
    U, lam = [], []
    for (ez, ey, ex), (mx, my, mz) in zip(shapes, [(2, 1, 0), (0, 3, 2), (4, 0, 1)]):
        cx = np.cos(np.pi * mx * (np.arange(ex) + 0.5) / ex)
        cy = np.cos(np.pi * my * (np.arange(ey) + 0.5) / ey)
        cz = np.cos(np.pi * mz * (np.arange(ez) + 0.5) / ez)
        U.append(cz[:, None, None] * cy[None, :, None] * cx[None, None, :])
        lam.append((2 - 2 * np.cos(np.pi * mx / ex)) + (2 - 2 * np.cos(np.pi * my / ey)) + (2 - 2 * np.cos(np.pi * mz / ez)))
    out = orc.viscosity(U, nu, dt, dx)
    for o, u, l in zip(out, U, lam):
        assert np.max(np.abs(o - (1 - k * l) * u)) <= 1e-14


def test_viscosity_constants_conservation_and_symmetry():
    rng = np.random.default_rng(4)
    shapes = wl.face_shapes(7, 5, 6)
    nu, dt, dx = 0.8, 0.02, 0.25
    ones = [np.full(s, 2.5) for s in shapes]
    assert all(np.array_equal(o, a) for o, a in zip(orc.viscosity(ones, nu, dt, dx), ones))  # no flux through the ends
    A = [rng.standard_normal(s) for s in shapes]
    B = [rng.standard_normal(s) for s in shapes]
    LA, LB = orc.viscosity(A, nu, dt, dx), orc.viscosity(B, nu, dt, dx)
    for a, la in zip(A, LA):
        assert abs(la.sum() - a.sum()) <= 1e-12 * np.abs(a).sum()                           # momentum is conserved
    lhs = sum(float(np.sum(x * y)) for x, y in zip(LA, B))
    rhs = sum(float(np.sum(x * y)) for x, y in zip(A, LB))
    assert abs(lhs - rhs) <= 1e-13 * abs(lhs)                                               # self-adjoint (Eq. 8)


def test_viscosity_matches_heat_equation_step():
    """Interior points: f + nu dt * (7-point Laplacian) / dx^2, written out by hand."""
    rng = np.random.default_rng(1)
    shapes = wl.face_shapes(6, 6, 6)
    U = [rng.standard_normal(s) for s in shapes]
    nu, dt, dx = 0.3, 0.05, 0.5
    out = orc.viscosity(U, nu, dt, dx)
    f, o = U[1], out[1]
    k_, j_, i_ = 2, 3, 2
    lap = (f[k_, j_, i_ + 1] + f[k_, j_, i_ - 1] + f[k_, j_ + 1, i_] + f[k_, j_ - 1, i_] + f[k_ + 1, j_, i_]
           + f[k_ - 1, j_, i_] - 6 * f[k_, j_, i_]) / dx ** 2
    assert abs(o[k_, j_, i_] - (f[k_, j_, i_] + nu * dt * lap)) <= 1e-14


def test_rollout_with_viscosity_gradient_matches_finite_differences():
    n = 10
    P = wl.config2_params(n)
    bc = orc.BC(P["bc_types"], P["bc_values"])
    rng = np.random.default_rng(8)
    U0 = [0.2 * rng.standard_normal(s) for s in wl.face_shapes(n, n, n)]
    loss = orc.loss_sum_u2(P["loss_lo"], P["loss_hi"])
    nu = 0.05 * P["dx"] ** 2 / P["dt"]      # nu dt / dx^2 = 0.05

    def run(theta):
        return orc.rollout(U0, lambda s: wl.config2_solid(P, s, theta, dtype=np.float64), 2, P["dt"], P["dx"],
                           P["dt_over_rho"], bc, loss, nu=nu)

    J, dJ, _ = run(0.5)
    h = 1e-5
    fd = (run(0.5 + h)[0] - run(0.5 - h)[0]) / (2 * h)
    assert abs(dJ - fd) <= 1e-6 * abs(fd)
    J0 = orc.rollout(U0, lambda s: wl.config2_solid(P, s, 0.5, dtype=np.float64), 2, P["dt"], P["dx"],
                     P["dt_over_rho"], bc, loss)[0]
    assert abs(J - J0) > 1e-6 * abs(J0)     # (the viscosity step is really in the path)
