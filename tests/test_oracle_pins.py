"""Pins for oracle/nf_oracle.py against things other than itself: the paper's printed formula, closed
forms, dense direct solves, invariants, finite differences, brute force.  CPU only."""
import os

import numpy as np
import pytest

from oracle import nf_oracle as O
from paper_2405_14903_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


# ----------------------------------------------------------------------------------------------------
# weights (a-1)
# ----------------------------------------------------------------------------------------------------
def test_alpha_printed_formula():
    """alpha = 1/2 * phiA/(phiA-phiB) * phiA/(phiA-phiD) when only corner A is in the fluid."""
    pa, pb, pc, pd = 0.3, -0.5, -0.9, -0.2
    expect = 0.5 * (0.3 / 0.8) * (0.3 / 0.5)
    for rot in range(4):  # the fluid corner may be any of the four
        vals = np.roll([pa, pb, pc, pd], rot)
        assert abs(O.area_fraction(*vals) - expect) < 1e-15
    # and mirrored orientation (B and D exchanged) gives the same area
    assert abs(O.area_fraction(pa, pd, pc, pb) - expect) < 1e-15


def _polygon_area(vals):
    """Brute force, independent of the case table: walk the unit square's boundary, collect fluid corners and
    linear zero crossings, shoelace the polygon.  Valid when the fluid region is one polygon
    (every case except the diagonal one)."""
    corners = [(0.0, 0.0), (1.0, 0.0), (1.0, 1.0), (0.0, 1.0)]
    pts = []
    for q in range(4):
        a, b = vals[q], vals[(q + 1) % 4]
        if a > 0:
            pts.append(corners[q])
        if (a > 0) != (b > 0):
            t = a / (a - b)
            pts.append((corners[q][0] + t * (corners[(q + 1) % 4][0] - corners[q][0]),
                        corners[q][1] + t * (corners[(q + 1) % 4][1] - corners[q][1])))
    if len(pts) < 3:
        return 0.0
    s = 0.0
    for q in range(len(pts)):
        x0, y0 = pts[q]
        x1, y1 = pts[(q + 1) % len(pts)]
        s += x0 * y1 - x1 * y0
    return abs(s) / 2


def test_alpha_brute_force_polygon():
    rng = np.random.default_rng(7)
    n_checked = {1: 0, 2: 0, 3: 0}
    for _ in range(4000):
        vals = rng.uniform(-1, 1, 4)
        f = vals > 0
        s = int(f.sum())
        if s in (0, 4) or (s == 2 and f[0] == f[2]):
            continue
        ref = _polygon_area(vals)
        if ref < 1e-3:
            continue
        got = float(O.area_fraction(*vals))
        assert abs(got - ref) < 1e-13, (vals, got, ref)
        n_checked[s] += 1
    assert min(n_checked.values()) > 200


def test_alpha_diagonal_case():
    """Two opposite fluid corners: mean > 0 joins the fluid (1 - two solid triangles), else two fluid
    triangles (R3); both branches by hand."""
    a, b, c, d = 0.9, -0.1, 0.8, -0.2  # mean > 0
    solid = 0.5 * (0.1 / 1.0) * (0.1 / 0.9) + 0.5 * (0.2 / 1.1) * (0.2 / 1.0)
    assert abs(O.area_fraction(a, b, c, d) - (1 - solid)) < 1e-15
    assert abs(O.area_fraction(b, c, d, a) - (1 - solid)) < 1e-15  # rotated
    a, b, c, d = 0.1, -0.9, 0.2, -0.8  # mean < 0
    fluid = 0.5 * (0.1 / 1.0) * (0.1 / 0.9) + 0.5 * (0.2 / 1.1) * (0.2 / 1.0)
    assert abs(O.area_fraction(a, b, c, d) - fluid) < 1e-15


def test_alpha_trivial_and_clamp():
    assert O.area_fraction(1, 2, 3, 4) == 1.0
    assert O.area_fraction(-1, -2, -3, -4) == 0.0
    assert O.area_fraction(0.0, -1, -1, -1) == 0.0  # phi == 0 counts as solid (R1)
    # tiny weight: 0.5 * (0.01/1.01)^2 = 4.9e-5 < 1e-4 -> 0 (R4)
    assert O.area_fraction(0.01, -1, -1, -1) == 0.0
    assert O.area_fraction(0.02, -1, -1, -1) > 1e-4


def test_alpha_planar_exact():
    """Axis-aligned plane x = 3.3 (fluid where x > 3.3): v- and w-faces of the cut column have alpha = 0.7,
    u-faces are 0 or 1 (marching squares is exact for planar interfaces)."""
    nx, ny, nz = 8, 5, 4
    x, y, z = W.node_coords(nx, ny, nz)
    phi = (x - 3.3) + 0 * y + 0 * z
    bc = O.BC((1,) * 6)  # Dirichlet everywhere so that no wall zeroing interferes
    au, av, aw = O.face_weights(phi, bc)
    assert np.allclose(au[:, :, :4], 0) and np.allclose(au[:, :, 4:], 1)
    assert np.allclose(av[:, :, 3], 0.7, atol=1e-14) and np.allclose(av[:, :, :3], 0) and np.allclose(av[:, :, 4:], 1)
    assert np.allclose(aw[:, :, 3], 0.7, atol=1e-14)
    # oblique plane x + y = 4.5 through a w-face: exact polygon area of {x+y>4.5} in the unit square
    phi = (x + y - 4.5) / np.sqrt(2) + 0 * z
    _, _, aw = O.face_weights(phi, bc)
    # face x in [2,3], y in [2,3]: solid corner triangle of legs 1/2 -> 7/8; face x in [1,2]: fluid triangle 1/8
    assert abs(aw[0, 2, 2] - 0.875) < 1e-14 and abs(aw[0, 2, 1] - 0.125) < 1e-14
    assert abs(aw[0, 2, 3] - 1) < 1e-14 and abs(aw[0, 2, 0]) < 1e-14


def test_alpha_axis_permutation_symmetry():
    rng = np.random.default_rng(3)
    phi = rng.uniform(-1, 1, (5, 6, 7))
    bc = O.BC((1,) * 6)
    au, av, aw = O.face_weights(phi, bc)
    # swap x and z
    au2, av2, aw2 = O.face_weights(phi.transpose(2, 1, 0).copy(), bc)
    assert np.allclose(aw2, au.transpose(2, 1, 0), atol=1e-15)
    assert np.allclose(av2, av.transpose(2, 1, 0), atol=1e-15)
    # swap x and y
    au3, av3, aw3 = O.face_weights(phi.transpose(0, 2, 1).copy(), bc)
    assert np.allclose(av3, au.transpose(0, 2, 1), atol=1e-15)
    assert np.allclose(aw3, aw.transpose(0, 2, 1), atol=1e-15)


def test_alpha_continuity_across_cases():
    """The area is continuous where a corner changes sign and the topology does not change: all
    non-diagonal transitions; into the diagonal case from s=1 when the decider separates (mean <= 0) and
    from s=3 when it joins (mean > 0).  (Across the decider itself the marching-squares area jumps; R3.)"""
    eps = 1e-9
    cases = []
    for base in (np.array([0.4, 0.7, -0.3, -0.6]), np.array([-0.4, 0.7, 0.3, 0.6]), np.array([0.4, -0.7, -0.3, -0.6])):
        for rot in range(4):
            v = np.roll(base, rot)
            for q in range(4):
                w = v.copy(); w[q] = 0
                f = w > 0
                if not (f[(q + 1) % 4] == f[(q - 1) % 4] and f[(q + 1) % 4] != f[(q + 2) % 4] and not f[(q + 1) % 4]):
                    cases.append((v, q))  # corner q's sign change cannot create a diagonal pattern
    cases.append((np.array([0.0, -0.5, 0.3, -0.4]), 0))  # s=1 -> diagonal, mean < 0: separated
    cases.append((np.array([0.5, -0.1, 0.4, 0.0]), 3))   # s=3 -> diagonal, mean > 0: joined
    assert len(cases) > 20
    for v, q in cases:
        lo, hi = v.copy(), v.copy()
        lo[q], hi[q] = -eps, eps
        assert abs(O.area_fraction(*lo) - O.area_fraction(*hi)) < 1e-6, (v, q)


def _golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "config1_worked_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v, t = line.split()
        out[k] = (float(v), float(t))
    return out


def _check(gold, key, val):
    ref, tol = gold[key]
    if tol == 0:
        assert val == ref, (key, val, ref)
    else:
        assert abs(val - ref) <= tol * abs(ref), (key, val, ref)


@pytest.fixture(scope="module")
def cfg1():
    c = W.config1()
    bc = O.BC(c["bc_types"], c["bc_values"])
    alpha = O.face_weights(c["phi"], bc)
    return c, bc, alpha


def test_config1_weights_golden(cfg1):
    """tests/golden/config1_worked_example.txt."""
    c, bc, alpha = cfg1
    gold = _golden()
    for a in alpha:
        _check(gold, "sum_alpha_per_family", float(a.sum()))
        _check(gold, "faces_cut_per_family", int(((a > 0) & (a < 1)).sum()))
        _check(gold, "faces_closed_per_family", int((a == 0).sum()))
    act = O.active_cells(alpha)
    _check(gold, "cells_active", int(act.sum()))
    _check(gold, "cells_inactive", int((~act).sum()))
    _check(gold, "solid_cross_section_plane_i16", float((1 - alpha[0][:, :, 16]).sum()))
    # curved interface: second-order accurate area of the R = 8 disc
    assert abs((1 - alpha[0][:, :, 16]).sum() - np.pi * 64) / (np.pi * 64) < 5e-3


def test_config1_projection_and_adjoint_golden(cfg1):
    c, bc, alpha = cfg1
    gold = _golden()
    U = [a.astype(np.float64) for a in c["U"]]
    g = [a.astype(np.float64) for a in c["g"]]
    _check(gold, "norm_Uhat", float(np.sqrt(sum((a ** 2).sum() for a in U))))
    cc = c["dt_over_rho"] / c["dx"]
    us0 = O.effective_solid_velocity(None, [a.shape for a in U], bc)
    b = O.rhs(U, alpha, us0, cc, bc)
    _check(gold, "norm_b", float(np.linalg.norm(b)))
    assert abs(b.sum()) < 1e-10
    Un, p = O.project(U, alpha, None, c["dx"], c["dt_over_rho"], bc, tol=1e-13)
    _check(gold, "norm_p", float(np.linalg.norm(p)))
    _check(gold, "max_abs_p", float(np.abs(p).max()))
    _check(gold, "norm_Unew", float(np.sqrt(sum((a ** 2).sum() for a in Un))))
    assert np.abs(O.weighted_divergence(Un, alpha, None, bc)).max() < 1e-10
    gU, ga, gus, y = O.project_adjoint(g, alpha, p, U, None, c["dx"], c["dt_over_rho"], bc, tol=1e-13)
    Mg = [np.where(a > 0, x, 0) for a, x in zip(alpha, g)]
    _check(gold, "norm_gp", float(np.linalg.norm(cc * O.grad_T(*Mg))))
    _check(gold, "norm_y", float(np.linalg.norm(y)))
    _check(gold, "norm_gUhat", float(np.sqrt(sum((a ** 2).sum() for a in gU))))
    d1 = sum((a * b_).sum() for a, b_ in zip(Un, g))
    d2 = sum((a * b_).sum() for a, b_ in zip(U, gU))
    _check(gold, "dot_Unew_g", float(d1))
    assert abs(d1 - d2) < 1e-10 * abs(d1)  # <P x, y> = <x, P^T y>   (north_star pin, 1e-10)
    _check(gold, "norm_galpha_open", float(np.sqrt(sum(((x * (a > 0)) ** 2).sum() for x, a in zip(ga, alpha)))))


# ----------------------------------------------------------------------------------------------------
# operators and solve (a-2 .. a-6)
# ----------------------------------------------------------------------------------------------------
def _random_alpha(rng, nx, ny, nz, bc, closed_frac=0.2):
    shapes = W.face_shapes(nx, ny, nz)
    alpha = []
    for sh in shapes:
        a = rng.uniform(0, 1, sh)
        a[rng.uniform(0, 1, sh) < closed_frac] = 0
        a[rng.uniform(0, 1, sh) < 0.4] = 1
        alpha.append(a)
    O.apply_wall_bc(*alpha, bc)
    return alpha


def _assemble_by_faces(alpha, c, nx, ny, nz):
    """Independent dense assembly: loop over interior faces and Dirichlet-open boundary faces, add the 2x2
    (or 1x1) element matrix c*alpha*[[1,-1],[-1,1]]."""
    n = nx * ny * nz
    A = np.zeros((n, n))
    idx = lambda i, j, k: (k * ny + j) * nx + i
    au, av, aw = alpha
    for k in range(nz):
        for j in range(ny):
            for i in range(nx + 1):
                a = c * au[k, j, i]
                cells = [idx(ii, j, k) for ii in (i - 1, i) if 0 <= ii < nx]
                _add(A, cells, a)
    for k in range(nz):
        for j in range(ny + 1):
            for i in range(nx):
                a = c * av[k, j, i]
                cells = [idx(i, jj, k) for jj in (j - 1, j) if 0 <= jj < ny]
                _add(A, cells, a)
    for k in range(nz + 1):
        for j in range(ny):
            for i in range(nx):
                a = c * aw[k, j, i]
                cells = [idx(i, j, kk) for kk in (k - 1, k) if 0 <= kk < nz]
                _add(A, cells, a)
    return A


def _add(A, cells, a):
    if len(cells) == 2:
        p, q = cells
        A[p, p] += a; A[q, q] += a; A[p, q] -= a; A[q, p] -= a
    else:
        A[cells[0], cells[0]] += a


@pytest.mark.parametrize("dirichlet", [False, True])
def test_operator_dense_and_direct_solve_8cubed(dirichlet):
    """north_star pin: dense direct solve on an 8^3 grid."""
    rng = np.random.default_rng(11)
    n = 8
    bc = O.BC((1, 0, 0, 1, 0, 0) if dirichlet else (0,) * 6, (0.7, 0, 0, -0.4, 0, 0) if dirichlet else (0,) * 6)
    alpha = _random_alpha(rng, n, n, n, bc, closed_frac=0.1)
    alpha = list(W.keep_largest_component(*alpha)[:3])
    c = 3.7
    A = _assemble_by_faces(alpha, c, n, n, n)
    assert np.abs(A - A.T).max() == 0
    x = rng.standard_normal((n, n, n))
    assert np.abs(O.apply_A(x, alpha, c).ravel() - A @ x.ravel()).max() < 1e-12
    assert np.abs(O.diag_A(alpha, c).ravel() - np.diag(A)).max() < 1e-13
    if not dirichlet:
        assert np.abs(A.sum(axis=1)).max() < 1e-12  # row sums 0 without Dirichlet
    act = O.active_cells(alpha)
    b = np.where(act, rng.standard_normal((n, n, n)), 0)
    if dirichlet:
        ia = np.flatnonzero(act.ravel())
        ref = np.zeros(n ** 3)
        ref[ia] = np.linalg.solve(A[np.ix_(ia, ia)], b.ravel()[ia])  # SPD block: direct solve
    else:
        b = np.where(act, b - b[act].mean(), 0)
        ia = np.flatnonzero(act.ravel())
        # pin one cell, solve the reduced SPD system, then remove the mean
        keep = ia[1:]
        ref = np.zeros(n ** 3)
        ref[keep] = np.linalg.solve(A[np.ix_(keep, keep)], b.ravel()[keep])
        ref[ia] -= ref[ia].mean()
    info = {}
    got = O.solve(b, alpha, c, bc, tol=1e-13, info=info)
    assert np.abs(got.ravel() - ref).max() < 1e-10 * max(1.0, np.abs(ref).max())
    got2 = O.solve_dense(b, alpha, c, bc)
    assert np.abs(got2.ravel() - ref).max() < 1e-9 * max(1.0, np.abs(ref).max())


def test_grad_and_grad_T_are_transposes():
    rng = np.random.default_rng(5)
    nx, ny, nz = 5, 4, 3
    p = rng.standard_normal((nz, ny, nx))
    f = [rng.standard_normal(s) for s in W.face_shapes(nx, ny, nz)]
    lhs = sum((a * b).sum() for a, b in zip(O.grad(p), f))
    rhs = (p * O.grad_T(*f)).sum()
    assert abs(lhs - rhs) < 1e-12
    # explicit small case: G p on a 1-D row
    p1 = np.array([[[1.0, 4.0, 9.0]]])
    gu, _, _ = O.grad(p1, ghost=(10.0, 20.0, 0, 0, 0, 0))
    assert np.allclose(gu.ravel(), [1 - 10, 3, 5, 20 - 9])


def test_solve_neumann_box_dct_closed_form():
    """No solids, closed walls: A = c G^T G is diagonalised by the DCT-II with eigenvalues
    c * sum_d (2 - 2 cos(pi k_d / n_d))."""
    from scipy.fft import dctn, idctn
    rng = np.random.default_rng(2)
    nx, ny, nz = 12, 9, 7
    bc = O.BC()
    alpha = [np.ones(s) for s in W.face_shapes(nx, ny, nz)]
    O.apply_wall_bc(*alpha, bc)
    c = 2.5
    b = rng.standard_normal((nz, ny, nx))
    b -= b.mean()
    lam = c * ((2 - 2 * np.cos(np.pi * np.arange(nz) / nz))[:, None, None]
               + (2 - 2 * np.cos(np.pi * np.arange(ny) / ny))[None, :, None]
               + (2 - 2 * np.cos(np.pi * np.arange(nx) / nx))[None, None, :])
    bh = dctn(b, type=2, norm="ortho")
    lam[0, 0, 0] = 1.0
    bh[0, 0, 0] = 0.0
    ref = idctn(bh / lam, type=2, norm="ortho")
    got = O.solve(b, alpha, c, bc, tol=1e-14)
    assert np.abs(got - ref).max() < 1e-12


def test_manufactured_sin_solution_second_order():
    """north_star pin: p* = sin(pi x) sin(pi y) sin(pi z) on the unit cube, recovered through `project` with
    closed walls from Uhat = grad p* sampled at face centres (dt/rho = 1): max-norm error decays as h^2."""
    errs = []
    for n in (8, 16, 32):
        dx = 1.0 / n
        bc = O.BC()
        alpha = [np.ones(s) for s in W.face_shapes(n, n, n)]
        O.apply_wall_bc(*alpha, bc)
        U = []
        for comp in range(3):
            fx, fy, fz = (a * dx for a in W.face_coords(n, n, n, comp))
            s = [np.sin(np.pi * fx), np.sin(np.pi * fy), np.sin(np.pi * fz)]
            cs = [np.cos(np.pi * fx), np.cos(np.pi * fy), np.cos(np.pi * fz)]
            t = [s[0], s[1], s[2]]
            t[comp] = np.pi * cs[comp]
            U.append(t[0] * t[1] * t[2] * np.ones(W.face_shapes(n, n, n)[comp]))
        Un, p = O.project(U, alpha, None, dx, 1.0, bc, tol=1e-13)
        cx = (np.arange(n) + 0.5) * dx
        pstar = np.sin(np.pi * cx)[None, None, :] * np.sin(np.pi * cx)[None, :, None] * np.sin(np.pi * cx)[:, None, None]
        pstar = pstar - pstar.mean()
        errs.append(np.abs(p - pstar).max())
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.7 < errs[1] / errs[2] < 4.3, errs
    # SURVEY.md §8c.4 prints 1.168e-3 (n=16) and 2.965e-4 (n=32) for this set-up
    assert abs(errs[1] - 1.168e-3) < 2e-6 and abs(errs[2] - 2.965e-4) < 1e-6, errs


def _random_case(seed, nx=6, ny=5, nz=4, dirichlet=True, with_us=True):
    rng = np.random.default_rng(seed)
    bc = O.BC((1, 1, 0, 0, 0, 1) if dirichlet else (0,) * 6, (0.8, -0.3, 0, 0, 0, 0.5) if dirichlet else (0,) * 6)
    alpha = _random_alpha(rng, nx, ny, nz, bc, closed_frac=0.15)
    alpha = list(W.keep_largest_component(*alpha)[:3])
    U = [rng.standard_normal(s) for s in W.face_shapes(nx, ny, nz)]
    us = [rng.standard_normal(s) for s in W.face_shapes(nx, ny, nz)] if with_us else None
    g = [rng.standard_normal(s) for s in W.face_shapes(nx, ny, nz)]
    return bc, alpha, U, us, g


@pytest.mark.parametrize("dirichlet", [False, True])
def test_projection_zero_weighted_divergence_and_idempotence(dirichlet):
    """north_star pin: zero discrete divergence after projection (Eqs. 4-5)."""
    bc, alpha, U, us, g = _random_case(21, dirichlet=dirichlet, with_us=dirichlet)
    if not dirichlet:
        us = None
    dx = 0.25
    Un, p = O.project(U, alpha, us, dx, 0.6, bc, tol=1e-14)
    div = O.weighted_divergence(Un, alpha, us, bc)
    if dirichlet:
        assert np.abs(div).max() < 1e-11
        # homogeneous part is a projector only for zero data; check S-orthogonality of the correction instead
    else:
        assert np.abs(div).max() < 1e-11
        Un2, _ = O.project(Un, alpha, None, dx, 0.6, bc, tol=1e-14)
        assert max(np.abs(a - b).max() for a, b in zip(Un, Un2)) < 1e-11


def test_singular_incompatible_solid_flux_is_handled():
    """Closed box, U_s with net flux: b has a mean; it is removed (R12) and the residual divergence is the
    constant mean only."""
    bc, alpha, U, us, g = _random_case(22, dirichlet=False, with_us=True)
    Un, p = O.project(U, alpha, us, 0.25, 1.0, bc, tol=1e-14)
    div = O.weighted_divergence(Un, alpha, us, bc)
    act = O.active_cells(alpha)
    assert np.abs(div[act] - div[act].mean()).max() < 1e-11
    assert abs(p[act].mean()) < 1e-13


@pytest.mark.parametrize("dirichlet", [False, True])
def test_adjoint_dot_product(dirichlet):
    """north_star pin: <P x, y> = <x, P^T y> to 1e-10 (U_s = 0, homogeneous Dirichlet data)."""
    bc, alpha, U, _, g = _random_case(31, dirichlet=dirichlet, with_us=False)
    bc = O.BC(bc.types, (0.0,) * 6)
    Un, p = O.project(U, alpha, None, 0.2, 0.7, bc, tol=1e-14)
    gU, _, _, _ = O.project_adjoint(g, alpha, p, U, None, 0.2, 0.7, bc, tol=1e-14)
    lhs = sum((a * b).sum() for a, b in zip(Un, g))
    rhs = sum((a * b).sum() for a, b in zip(U, gU))
    assert abs(lhs - rhs) <= 1e-10 * abs(lhs)


@pytest.mark.parametrize("dirichlet", [False, True])
def test_adjoint_finite_differences(dirichlet):
    """PAPER.md:L430-434 method (central differences), J = <g, U^{n+1}>, w.r.t. Uhat, U_s and alpha.
    Pins the derived sign of Eq. 9a's second term (R9) and the derived Eq. 9b (R10)."""
    bc, alpha, U, us, g = _random_case(41, dirichlet=dirichlet, with_us=True)
    dx, dtr = 0.2, 0.7
    # keep alpha away from 0 on open faces so the FD step does not cross the open/closed switch
    alpha = [np.where(a > 0, np.maximum(a, 0.05), 0) for a in alpha]

    def J(U_, us_, alpha_):
        Un, _ = O.project(U_, alpha_, us_, dx, dtr, bc, tol=1e-14)
        return sum((a * b).sum() for a, b in zip(Un, g))

    Un, p = O.project(U, alpha, us, dx, dtr, bc, tol=1e-14)
    gU, ga, gus, _ = O.project_adjoint(g, alpha, p, U, us, dx, dtr, bc, tol=1e-14)
    rng = np.random.default_rng(0)
    h = 1e-6
    for which, grad_ in (("U", gU), ("us", gus), ("alpha", ga)):
        d = [rng.standard_normal(a.shape) for a in U]
        if which == "alpha":
            d = [np.where((a > 0), x, 0) for a, x in zip(alpha, d)]  # closed faces stay closed
        if not dirichlet and which == "us":
            # singular system: J is defined after mean removal; any direction is fine
            pass
        args_p = dict(U=U, us=us, alpha=alpha)
        args_m = dict(U=U, us=us, alpha=alpha)
        args_p[which] = [a + h * x for a, x in zip(args_p[which], d)]
        args_m[which] = [a - h * x for a, x in zip(args_m[which], d)]
        fd = (J(args_p["U"], args_p["us"], args_p["alpha"]) - J(args_m["U"], args_m["us"], args_m["alpha"])) / (2 * h)
        an = sum((a * x).sum() for a, x in zip(grad_, d))
        assert abs(fd - an) <= 2e-7 * max(1.0, abs(an)), (which, fd, an)


# ----------------------------------------------------------------------------------------------------
# advection (a-8, a-9) and weights adjoint (a-10)
# ----------------------------------------------------------------------------------------------------
def test_advect_constant_field_unchanged():
    nx, ny, nz = 6, 5, 4
    U = [np.full(s, v) for s, v in zip(W.face_shapes(nx, ny, nz), (0.7, -0.4, 0.2))]
    out = O.advect(U, dt=0.3, dx=0.5)
    for a, b in zip(out, U):
        assert np.abs(a - b).max() < 1e-15


def test_advect_linear_field_closed_form():
    """u = a x (trilinear interpolation is exact): x_m = x(1 - a dt/2), x_b = x - dt a x_m,
    out = a x_b = a x (1 - a dt + a^2 dt^2 / 2) away from the clamps."""
    nx, ny, nz = 10, 4, 3
    dx, dt, a = 0.5, 0.2, 0.8
    shu, shv, shw = W.face_shapes(nx, ny, nz)
    xu = np.arange(nx + 1) * dx
    U = [np.broadcast_to(a * xu, shu).copy(), np.zeros(shv), np.zeros(shw)]
    out = O.advect(U, dt, dx)
    expect = a * xu * (1 - a * dt + 0.5 * a * a * dt * dt)
    assert np.abs(out[0] - expect).max() < 1e-14


def test_interp_reproduces_samples_and_midpoints():
    rng = np.random.default_rng(9)
    nx, ny, nz = 4, 3, 5
    v = rng.standard_normal(W.face_shapes(nx, ny, nz)[1])
    # at its own sample positions (i+1/2, j, k+1/2)
    pos = W.face_coords(nx, ny, nz, 1)
    pos = [np.broadcast_to(p, v.shape) for p in pos]
    assert np.abs(O.interp(v, 1, pos) - v).max() < 1e-15
    # halfway between two samples in y
    got = O.interp(v, 1, [np.array(1.5), np.array(0.5), np.array(2.5)])
    assert abs(got - 0.5 * (v[2, 0, 1] + v[2, 1, 1])) < 1e-15
    # clamped outside the lattice
    got = O.interp(v, 1, [np.array(-3.0), np.array(1.0), np.array(2.5)])
    assert abs(got - v[2, 1, 0]) < 1e-15


def test_advect_adjoint_finite_differences():
    """Random field with CFL up to ~1.5 so back-traces cross cells and hit the clamps."""
    rng = np.random.default_rng(13)
    nx, ny, nz = 6, 5, 4
    dx, dt = 0.5, 0.25
    U = [3.0 * rng.uniform(-1, 1, s) for s in W.face_shapes(nx, ny, nz)]
    g = [rng.standard_normal(s) for s in W.face_shapes(nx, ny, nz)]
    gU = O.advect_adjoint(U, g, dt, dx)
    h = 1e-6
    for trial in range(4):
        d = [rng.standard_normal(a.shape) for a in U]
        Jp = sum((a * b).sum() for a, b in zip(O.advect([a + h * x for a, x in zip(U, d)], dt, dx), g))
        Jm = sum((a * b).sum() for a, b in zip(O.advect([a - h * x for a, x in zip(U, d)], dt, dx), g))
        fd = (Jp - Jm) / (2 * h)
        an = sum((a * x).sum() for a, x in zip(gU, d))
        assert abs(fd - an) <= 1e-7 * max(1.0, abs(an)), (fd, an)


def test_weights_adjoint_finite_differences():
    rng = np.random.default_rng(17)
    nx, ny, nz = 5, 4, 3
    phi = rng.uniform(-1, 1, (nz + 1, ny + 1, nx + 1))
    phi[np.abs(phi) < 0.05] = 0.3  # keep corners away from sign changes under the FD step
    bc = O.BC((0, 1, 0, 0, 1, 0))
    ga = [rng.standard_normal(s) for s in W.face_shapes(nx, ny, nz)]
    gphi = O.weights_adjoint(phi, *ga, bc)
    h = 1e-6
    for trial in range(4):
        d = rng.standard_normal(phi.shape)
        ap = O.face_weights(phi + h * d, bc)
        am = O.face_weights(phi - h * d, bc)
        # skip faces that cross the alpha < 1e-4 clamp or the diagonal tie-break under the perturbation
        fd = sum((g_ * (p_ - m_)).sum() for g_, p_, m_ in zip(ga, ap, am)) / (2 * h)
        an = (gphi * d).sum()
        assert abs(fd - an) <= 1e-6 * max(1.0, abs(an)), (fd, an)


def test_keep_largest_component():
    nx, ny, nz = 6, 3, 3
    alpha = [np.ones(s) for s in W.face_shapes(nx, ny, nz)]
    O.apply_wall_bc(*alpha, O.BC())
    alpha[0][:, :, 2] = 0  # wall between cells i<2 and i>=2
    au, av, aw, ncomp = W.keep_largest_component(*alpha)
    assert ncomp == 2
    act = O.active_cells([au, av, aw])
    assert not act[:, :, :2].any() and act[:, :, 2:].all()


# ---------------------------------------------------------------------------------------------------------
# R12 per fluid component: labels, compatibility and gauge of every singular component
# ---------------------------------------------------------------------------------------------------------
def _flood_fill_labels(alpha):
    """Brute force: breadth-first search over cells, stepping through faces with alpha > 0 (pure Python)."""
    au, av, aw = alpha
    nz, ny, nx = au.shape[0], au.shape[1], au.shape[2] - 1
    act = O.active_cells(alpha)
    lab = np.zeros((nz, ny, nx), dtype=int)
    cur = 0
    for k0 in range(nz):
        for j0 in range(ny):
            for i0 in range(nx):
                if not act[k0, j0, i0] or lab[k0, j0, i0]:
                    continue
                cur += 1
                lab[k0, j0, i0] = cur
                todo = [(k0, j0, i0)]
                while todo:
                    k, j, i = todo.pop()
                    nbs = []
                    if i > 0 and au[k, j, i] > 0: nbs.append((k, j, i - 1))
                    if i + 1 < nx and au[k, j, i + 1] > 0: nbs.append((k, j, i + 1))
                    if j > 0 and av[k, j, i] > 0: nbs.append((k, j - 1, i))
                    if j + 1 < ny and av[k, j + 1, i] > 0: nbs.append((k, j + 1, i))
                    if k > 0 and aw[k, j, i] > 0: nbs.append((k - 1, j, i))
                    if k + 1 < nz and aw[k + 1, j, i] > 0: nbs.append((k + 1, j, i))
                    for c in nbs:
                        if not lab[c]:
                            lab[c] = cur
                            todo.append(c)
    return lab


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_components_equal_brute_force_flood_fill(seed):
    rng = np.random.default_rng(seed)
    nx, ny, nz = 7, 6, 5
    alpha = [np.where(rng.uniform(size=s) < 0.55, 0.0, rng.uniform(0.1, 1, s)) for s in
             [(nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)]]
    bc = O.BC((1, 0, 0, 0, 0, 1))
    O.apply_wall_bc(*alpha, bc)
    lab, sing = O.components(alpha, bc)
    ref = _flood_fill_labels(alpha)
    assert np.array_equal(lab > 0, ref > 0) and lab.max() == ref.max() and lab.max() >= 2
    # same partition: the pairs (label, reference label) are one to one
    pairs = set(zip(lab[lab > 0].tolist(), ref[ref > 0].tolist()))
    assert len(pairs) == lab.max()
    # singular flag by hand: a component is regular iff one of its cells has an open face on a Dirichlet boundary
    for c in range(1, lab.max() + 1):
        m = lab == c
        touches = bool(np.any(alpha[0][:, :, 0][m[:, :, 0]] > 0) or np.any(alpha[2][-1][m[-1]] > 0))
        assert sing[c] == (not touches)


def test_solve_two_pockets_matches_pseudo_inverse():
    """A wall of closed faces splits an 8 x 6 x 5 box into a pocket with a Dirichlet face and a closed pocket (its
    block of A has the constant null vector): the CG solve with per-component compatibility and gauge (R12) equals
    the pseudo-inverse solution of the dense matrix; the regular pocket keeps its mean, the closed one has none."""
    rng = np.random.default_rng(5)
    nx, ny, nz = 8, 6, 5
    alpha = [rng.uniform(0.2, 1, s) for s in [(nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)]]
    alpha[0][:, :, 4] = 0.0
    bc = O.BC((1, 0, 0, 0, 0, 0), (0.3, 0, 0, 0, 0, 0))
    O.apply_wall_bc(*alpha, bc)
    lab, sing = O.components(alpha, bc)
    assert lab.max() == 2 and sing.tolist() == [False, False, True]
    assert O.is_singular(alpha, bc) is False      # (the global flag says "regular": not enough for the closed pocket)
    b = rng.standard_normal((nz, ny, nx))
    x = O.solve(b, alpha, 1.7, bc, tol=1e-13)
    xd = O.solve_dense(b, alpha, 1.7, bc)
    assert np.max(np.abs(x - xd)) <= 1e-9 * np.max(np.abs(xd))
    assert abs(x[lab == 2].mean()) <= 1e-12 and abs(x[lab == 1].mean()) > 1e-3
    # the residual that is left is exactly the incompatible part of b: its mean over the closed pocket
    res = b - O.apply_A(x, alpha, 1.7)
    assert np.max(np.abs(res[lab == 1])) <= 1e-10
    assert np.max(np.abs(res[lab == 2] - b[lab == 2].mean())) <= 1e-10


def test_projection_with_closed_pocket_is_divergence_free_where_it_can_be():
    """Projection on the two-pocket box with a solid velocity: zero weighted divergence in the pocket with the outlet;
    in the closed pocket the divergence that remains is the constant the incompatible boundary flux forces."""
    rng = np.random.default_rng(6)
    nx, ny, nz = 8, 6, 5
    shp = [(nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)]
    alpha = [rng.uniform(0.2, 1, s) for s in shp]
    alpha[0][:, :, 4] = 0.0
    bc = O.BC((1, 0, 0, 0, 0, 0))
    O.apply_wall_bc(*alpha, bc)
    U = [rng.standard_normal(s) for s in shp]
    us = [0.1 * rng.standard_normal(s) for s in shp]
    Un, p = O.project(U, alpha, us, 0.125, 0.9, bc)
    lab, _ = O.components(alpha, bc)
    div = O.weighted_divergence(Un, alpha, us, bc)
    assert np.max(np.abs(div[lab == 1])) <= 1e-9
    assert np.max(np.abs(div[lab == 2] - div[lab == 2].mean())) <= 1e-9
