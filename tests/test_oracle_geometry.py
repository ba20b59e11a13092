"""Pins for oracle/nf_geom_oracle.py against what PAPER.md:L339-347 and the mathematics fix:
the construction constraints of appendix A checked from their wording, closed forms (circle limit, rigid motion,
uniform growth, slab caps), an independent evaluation of the true Bezier curves (de Casteljau + winding number),
finite differences, and the level-set transport identity that ties the velocity to the distance."""
import numpy as np
import pytest

from oracle import nf_geom_oracle as G


def rand_params(rng, K, N, z0=0.17, z1=0.81, c=(0.5, 0.5), r=0.25, jitter=0.25):
    p = np.zeros(G.n_params(K, N))
    p[0], p[1] = z0, z1
    keys = p[2:].reshape(K, 2 + 2 * N)
    keys[:, 0] = c[0] + 0.03 * rng.standard_normal(K)
    keys[:, 1] = c[1] + 0.03 * rng.standard_normal(K)
    keys[:, 2:] = r * (1 + jitter * rng.uniform(-1, 1, (K, 2 * N)))
    return p


def de_casteljau(P, t):
    """Independent evaluation of a cubic Bezier curve by repeated linear interpolation."""
    P = [np.asarray(q, dtype=np.float64) for q in P]
    while len(P) > 1:
        P = [(1 - t) * P[i] + t * P[i + 1] for i in range(len(P) - 1)]
    return P[0]


# --- appendix A's construction constraints, from the wording (L341) -------------------------------------------------
def test_control_points_satisfy_appendix_A():
    rng = np.random.default_rng(1)
    N = 5
    c = np.array([0.3, -0.2])
    r1, r2 = rng.uniform(0.5, 1.5, N), rng.uniform(0.5, 1.5, N)
    e0, p0, p1, e1 = G.control_points(c, r1, r2)
    for i in range(N):
        ip = (i + 1) % N
        # "e1^i = e0^{(i+1)%N}"
        assert np.allclose(e1[i], e0[ip], atol=1e-15)
        # "each Bezier curve spans an arc of 2 pi / N": its endpoints sit at the polar angles theta_i, theta_{i+1}
        for e, th in ((e0[i], 2 * np.pi * i / N), (e1[i], 2 * np.pi * (i + 1) / N)):
            d = e - c
            assert abs(np.sin(np.arctan2(d[1], d[0]) - th)) < 1e-14 and np.cos(np.arctan2(d[1], d[0]) - th) > 0
        # "control points ... at an angular displacement of 2 pi / (3N) from their corresponding curve endpoint"
        a0 = np.arctan2(*(p0[i] - c)[::-1]) - 2 * np.pi * i / N
        a1 = 2 * np.pi * (i + 1) / N - np.arctan2(*(p1[i] - c)[::-1])
        assert abs(np.angle(np.exp(1j * a0)) - 2 * np.pi / (3 * N)) < 1e-14
        assert abs(np.angle(np.exp(1j * a1)) - 2 * np.pi / (3 * N)) < 1e-14
        # "polar coordinate distance of the two control points" = rho1, rho2
        assert np.isclose(np.linalg.norm(p0[i] - c), r1[i]) and np.isclose(np.linalg.norm(p1[i] - c), r2[i])
        # "colinearity of each pair of p1^i, e1^i, p0^{(i+1)%N}", the endpoint between the two
        u, v = e1[i] - p1[i], p0[ip] - e1[i]
        assert abs(u[0] * v[1] - u[1] * v[0]) < 1e-14 and u @ v > 0


def test_polyline_vertices_are_on_the_bezier_curves():
    rng = np.random.default_rng(2)
    N, M = 4, 7
    c = np.array([0.1, 0.2])
    r1, r2 = rng.uniform(0.5, 1.5, N), rng.uniform(0.5, 1.5, N)
    e0, p0, p1, e1 = G.control_points(c, r1, r2)
    V = G.polyline(c, r1, r2, M)
    assert V.shape == (N * M, 2)
    for i in range(N):
        for m in range(M):
            assert np.allclose(V[i * M + m], de_casteljau([e0[i], p0[i], p1[i], e1[i]], m / M), atol=1e-14)


# --- closed form: equal radii -> circle ------------------------------------------------------------------------------
def test_equal_radii_give_a_circle():
    """rho = R / cos(delta) on every control point: endpoints at radius R with tangents normal to the radius, inner
    control points at distance R tan(delta) along the tangent -- the standard cubic approximation of a circular
    arc, exact to O((2 pi / N)^6) R; with N = 24, M = 16 the polygon's sag R (1 - cos(pi / (N M))) = 3.4e-5 R
    dominates."""
    N, M, R = 24, 16, 0.3
    dl = 2 * np.pi / (3 * N)
    c = np.array([0.45, 0.55])
    r = np.full(N, R / np.cos(dl))
    rng = np.random.default_rng(3)
    X, Y = rng.uniform(0, 1, 400), rng.uniform(0, 1, 400)
    d = G.sdf2d(c, r, r, M, X, Y)
    exact = np.hypot(X - c[0], Y - c[1]) - R
    assert np.max(np.abs(d - exact)) < 5e-5 * R + 1e-12
    assert np.all(np.sign(d[np.abs(exact) > 1e-4]) == np.sign(exact[np.abs(exact) > 1e-4]))


# --- brute force on the true curve -----------------------------------------------------------------------------------
def test_distance_and_sign_against_dense_sampling_of_the_true_curve():
    rng = np.random.default_rng(4)
    N, M = 6, 48
    c = np.array([0.5, 0.5])
    r1, r2 = rng.uniform(0.2, 0.4, N), rng.uniform(0.2, 0.4, N)
    e0, p0, p1, e1 = G.control_points(c, r1, r2)
    ts = np.linspace(0, 1, 4001)[:-1]
    pts = np.concatenate([np.stack([de_casteljau([e0[i], p0[i], p1[i], e1[i]], t) for t in ts]) for i in range(N)])
    X, Y = rng.uniform(0, 1, 150), rng.uniform(0, 1, 150)
    d = G.sdf2d(c, r1, r2, M, X, Y)
    brute = np.sqrt(np.min((X[:, None] - pts[None, :, 0]) ** 2 + (Y[:, None] - pts[None, :, 1]) ** 2, axis=1))
    # polygon sag <= max|B''| / (8 M^2) <= 6 * (control polygon diameter) / (8 M^2)
    sag = 6 * 0.8 / (8 * M * M)
    assert np.max(np.abs(np.abs(d) - brute)) < sag + 1e-4
    # sign: winding number of the dense curve about the point (independent of the crossing test)
    ang = np.unwrap(np.arctan2(pts[None, :, 1] - Y[:, None], pts[None, :, 0] - X[:, None]), axis=1)
    closed = np.arctan2(pts[0, 1] - Y, pts[0, 0] - X)
    wind = np.round((ang[:, -1] + np.angle(np.exp(1j * (closed - ang[:, -1]))) - ang[:, 0]) / (2 * np.pi))
    far = brute > 2 * sag
    assert np.all((wind[far] != 0) == (d[far] < 0))


# --- z interpolation and slab ------------------------------------------------------------------------------------------
def test_key_sections_are_interpolated_and_evenly_spaced():
    rng = np.random.default_rng(5)
    K, N = 4, 3
    p = rand_params(rng, K, N, z0=0.2, z1=0.8)
    z0, z1, c, r1, r2 = G.unpack(p, K, N)
    for k in range(K):
        ck, r1k, r2k = G.section_at(p, K, N, z0 + (z1 - z0) * k / (K - 1))[:3]
        assert np.allclose(ck, c[k]) and np.allclose(r1k, r1[k]) and np.allclose(r2k, r2[k])
    ck, r1k, _ = G.section_at(p, K, N, z0 + (z1 - z0) * 1.5 / (K - 1))[:3]
    assert np.allclose(ck, 0.5 * (c[1] + c[2])) and np.allclose(r1k, 0.5 * (r1[1] + r1[2]))
    # outside [z0, z1] the end sections are held
    assert np.allclose(G.section_at(p, K, N, 0.0)[0], c[0]) and np.allclose(G.section_at(p, K, N, 1.0)[0], c[-1])


def test_extruded_circle_is_a_cylinder():
    N, M, R = 24, 16, 0.25
    n, dx = 16, 1.0 / 16
    dl = 2 * np.pi / (3 * N)
    p = np.zeros(G.n_params(1, N))
    p[0], p[1], p[2], p[3] = 0.3, 0.7, 0.5, 0.5
    p[4:] = R / np.cos(dl)
    phi = G.sdf_nodes(p, 1, N, M, n, n, n, dx)
    k, j, i = np.meshgrid(*(np.arange(n + 1) * dx,) * 3, indexing="ij")
    exact = np.maximum(np.hypot(i - 0.5, j - 0.5) - R, np.maximum(0.3 - k, k - 0.7))
    assert np.max(np.abs(phi - exact)) < 5e-5 * R
    assert np.allclose(G.sdf_nodes(p, 1, N, M, n, n, n, dx, complement=True), -phi)


def test_csg_is_set_union_and_intersection():
    rng = np.random.default_rng(6)
    a, b = rng.standard_normal((5, 6, 7)), rng.standard_normal((5, 6, 7))
    # phi < 0 = solid: a point is in the union iff it is in either solid, in the intersection iff in both
    assert np.array_equal(G.csg("union", a, b) < 0, (a < 0) | (b < 0))
    assert np.array_equal(G.csg("intersection", a, b) < 0, (a < 0) & (b < 0))
    g = rng.standard_normal(a.shape)
    for op in ("union", "intersection"):
        ga, gb = G.csg_adjoint(op, a, b, g)
        assert np.array_equal(ga + gb, g) and np.all((ga == 0) | (gb == 0))
        h = 1e-7
        da, db = rng.standard_normal(a.shape), rng.standard_normal(a.shape)
        fd = np.sum(g * (G.csg(op, a + h * da, b + h * db) - G.csg(op, a - h * da, b - h * db))) / (2 * h)
        assert np.isclose(fd, np.sum(ga * da) + np.sum(gb * db), rtol=1e-6)


# --- adjoint: finite differences -----------------------------------------------------------------------------------------
@pytest.mark.parametrize("K,N,complement", [(1, 4, False), (3, 4, False), (2, 5, True)])
def test_sdf_adjoint_matches_finite_differences(K, N, complement):
    rng = np.random.default_rng(7 + K)
    M, n, dx = 6, 10, 0.1
    p = rand_params(rng, K, N, z0=0.23, z1=0.78)
    gphi = rng.standard_normal((n + 1, n + 1, n + 1))
    g = G.sdf_nodes_adjoint(p, K, N, M, n, n, n, dx, gphi, complement)
    J = lambda q: np.sum(gphi * G.sdf_nodes(q, K, N, M, n, n, n, dx, complement))
    h = 1e-6
    fd = np.zeros_like(p)
    for a in range(len(p)):
        e = np.zeros_like(p); e[a] = h
        fd[a] = (J(p + e) - J(p - e)) / (2 * h)
    # phi is piecewise smooth in params (the closest segment can switch): a node within h of a switch costs O(h)
    assert np.max(np.abs(g - fd)) < 2e-4 * max(1.0, np.max(np.abs(fd)))
    assert np.max(np.abs(fd)) > 1.0


# --- velocity: closed forms and the transport identity ----------------------------------------------------------------------
def circle_params(N, R, c, z0, z1, K=1):
    dl = 2 * np.pi / (3 * N)
    p = np.zeros(G.n_params(K, N))
    p[0], p[1] = z0, z1
    keys = p[2:].reshape(K, 2 + 2 * N)
    keys[:, 0], keys[:, 1], keys[:, 2:] = c[0], c[1], R / np.cos(dl)
    return p


def test_velocity_of_a_translating_and_growing_cylinder():
    """The polygon's normal deviates from the circle's by at most half its turning angle, pi / (N M) = 2.0e-3 rad,
    so (nh . v) nh is within 2 |v| pi / (N M) = 3.3e-3 of the circle's value."""
    N, M, R, K = 24, 64, 0.25, 2
    n, dx = 12, 1.0 / 12
    p = circle_params(N, R, (0.5, 0.5), 0.2, 0.8, K)
    # rigid translation (a, b) of every key section, caps moving at zd0, zd1
    pd = np.zeros_like(p)
    a, b, zd0, zd1 = 0.7, -0.4, 0.3, -0.2
    kd = pd[2:].reshape(K, 2 + 2 * N)
    kd[:, 0], kd[:, 1] = a, b
    pd[0], pd[1] = zd0, zd1
    us, vs, ws = G.solid_velocity_faces(p, pd, K, N, M, n, n, n, dx)

    def closed(X, Y, z):
        rx, ry = X - 0.5, Y - 0.5
        r = np.hypot(rx, ry)
        nx_, ny_ = rx / r, ry / r
        # moving caps change s = (z - z0)/(z1 - z0) but both key sections are equal, so the section is unchanged
        vn = a * nx_ + b * ny_
        slab = np.maximum(0.2 - z, z - 0.8) > (r - R)
        zd = np.where(0.2 - z >= z - 0.8, zd0, zd1)
        return np.where(slab, 0, vn * nx_), np.where(slab, 0, vn * ny_), np.where(slab, zd, 0)
    k, j, i = np.meshgrid((np.arange(n) + 0.5) * dx, (np.arange(n) + 0.5) * dx, np.arange(n + 1) * dx, indexing="ij")
    assert np.max(np.abs(us - closed(i, j, k)[0])) < 3.5e-3
    k, j, i = np.meshgrid(np.arange(n + 1) * dx, (np.arange(n) + 0.5) * dx, (np.arange(n) + 0.5) * dx, indexing="ij")
    assert np.max(np.abs(ws - closed(i, j, k)[2])) < 1e-12
    # uniform growth: rho_dot = g rho on every control point -> the circle's radius grows at g R
    pd = np.zeros_like(p)
    pd[2:].reshape(K, 2 + 2 * N)[:, 2:] = 0.5 * p[2:].reshape(K, 2 + 2 * N)[:, 2:]
    us, vs, ws = G.solid_velocity_faces(p, pd, K, N, M, n, n, n, dx)
    k, j, i = np.meshgrid((np.arange(n) + 0.5) * dx, np.arange(n + 1) * dx, (np.arange(n) + 0.5) * dx, indexing="ij")
    r = np.hypot(i - 0.5, j - 0.5)
    inslab = (k > 0.2) & (k < 0.8) & (np.maximum(0.2 - k, k - 0.8) <= r - R)
    assert np.max(np.abs(vs - 0.5 * R * (j - 0.5) / r)[inslab]) < 1e-3
    assert np.all(ws == 0)


def test_velocity_transports_the_distance_field():
    """phi_t + U_s . grad(phi) = 0 for the surface moving along its normal: d/dh phi(params + h pdot) at a fixed
    point equals -(U_s . grad phi), grad phi by central differences in space."""
    rng = np.random.default_rng(11)
    K, N, M = 3, 4, 8
    p = rand_params(rng, K, N, z0=-1.0, z1=2.0)       # slab far away: the cross-section term is the active one
    pd = rng.standard_normal(p.shape) * 0.1
    pd[0] = pd[1] = 0.0
    X, Y = rng.uniform(0.1, 0.9, 60), rng.uniform(0.1, 0.9, 60)
    z = 0.37
    us, vs, _, _ = G._velocity_points(p, pd, K, N, M, X, Y, z)
    h = 1e-6

    def phi(q, X, Y):
        c, r1, r2 = G.section_at(q, K, N, z)[:3]
        return G.sdf2d(c, r1, r2, M, X, Y)
    phit = (phi(p + h * pd, X, Y) - phi(p - h * pd, X, Y)) / (2 * h)
    gx = (phi(p, X + h, Y) - phi(p, X - h, Y)) / (2 * h)
    gy = (phi(p, X, Y + h) - phi(p, X, Y - h)) / (2 * h)
    assert np.max(np.abs(phit + us * gx + vs * gy)) < 1e-6
    assert np.max(np.abs(phit)) > 1e-2


def test_velocity_is_linear_in_pdot_and_adjoint_is_its_transpose():
    rng = np.random.default_rng(12)
    K, N, M, n, dx = 2, 3, 4, 5, 0.2
    p = rand_params(rng, K, N, z0=0.25, z1=0.75)
    a, b = rng.standard_normal(p.shape), rng.standard_normal(p.shape)
    va = G.solid_velocity_faces(p, a, K, N, M, n, n, n, dx)
    vb = G.solid_velocity_faces(p, b, K, N, M, n, n, n, dx)
    vab = G.solid_velocity_faces(p, 2 * a - 3 * b, K, N, M, n, n, n, dx)
    for x, y, xy in zip(va, vb, vab):
        assert np.allclose(xy, 2 * x - 3 * y, atol=1e-12)
    gs = [rng.standard_normal(x.shape) for x in va]
    gp = G.solid_velocity_faces_adjoint(p, K, N, M, n, n, n, dx, *gs)
    assert np.isclose(sum(np.sum(x * g) for x, g in zip(va, gs)), gp @ a, rtol=1e-10)
    # band: faces farther than the band from the primitive keep what they had
    phi_u = G._velocity_points(p, a, K, N, M, *np.meshgrid(np.arange(n + 1) * dx, (np.arange(n) + 0.5) * dx), 2.5 * dx)[3]
    keep = [np.full(x.shape, 7.0) for x in va]
    vb = G.solid_velocity_faces(p, a, K, N, M, n, n, n, dx, band=0.1, out=keep)
    assert np.array_equal(vb[0][2] == 7.0, phi_u > 0.1) and np.array_equal(vb[0][2][phi_u <= 0.1], va[0][2][phi_u <= 0.1])
    assert 0 < np.count_nonzero(phi_u <= 0.1) < phi_u.size


# --- the co-design loop: finite differences of the loss through full time steps ---------------------------------------------
def _rollout_setup():
    from oracle import nf_oracle as orc
    n, dx = 10, 0.1
    bc = orc.BC((1, 1, 0, 0, 0, 0), (1.0, 0.0, 0, 0, 0, 0))
    rng = np.random.default_rng(21)
    U0 = [0.2 * rng.standard_normal(s) for s in ((n, n, n + 1), (n, n + 1, n), (n + 1, n, n))]
    pA = rand_params(rng, 2, 4, z0=0.22, z1=0.77, c=(0.38, 0.5), r=0.17)
    pB = rand_params(rng, 1, 3, z0=0.31, z1=0.68, c=(0.7, 0.45), r=0.12)
    dB = 0.3 * rng.standard_normal(pB.shape)

    def loss(U):
        return 0.5 * sum(float(np.sum(a * a)) for a in U), [a.copy() for a in U]
    return orc, n, dx, bc, U0, pA, pB, dB, loss


def test_design_gradient_of_a_rollout_matches_finite_differences():
    """dJ/dparams of a static shape (the paper's design tasks) through 2 full steps: sum over steps of the per-step
    gradient against a central difference of the loss (the paper's own validation method, L430-434)."""
    orc, n, dx, bc, U0, pA, pB, dB, loss = _rollout_setup()
    prims = lambda a, b: (lambda step: [(a, None, 2, 4, 5), (b, None, 1, 3, 6)])
    J, grads, gU0 = G.rollout_parametric(U0, prims(pA, pB), 2, 0.04, dx, 1.0, bc, loss)
    gA = sum(g[0][0] for g in grads)
    gB = sum(g[1][0] for g in grads)
    assert grads[0][0][1] is None
    rng = np.random.default_rng(2)
    for _ in range(2):
        dA, dBdir = rng.standard_normal(pA.shape) * 0.02, rng.standard_normal(pB.shape) * 0.02
        h = 1e-4
        Jp = G.rollout_parametric(U0, prims(pA + h * dA, pB + h * dBdir), 2, 0.04, dx, 1.0, bc, loss)[0]
        Jm = G.rollout_parametric(U0, prims(pA - h * dA, pB - h * dBdir), 2, 0.04, dx, 1.0, bc, loss)[0]
        fd = (Jp - Jm) / (2 * h)
        an = gA @ dA + gB @ dBdir
        assert abs(fd - an) < 2e-3 * max(abs(fd), abs(an)), (fd, an)
        assert abs(fd) > 1e-4


def test_control_gradient_of_a_rollout_matches_finite_differences():
    """dJ/dpdot of a moving primitive (the paper's control tasks): U_s is linear in pdot and phi does not depend on it,
    so the transpose is exact and the loss is quadratic in pdot."""
    orc, n, dx, bc, U0, pA, pB, dB, loss = _rollout_setup()
    band = 0.15
    prims = lambda d: (lambda step: [(pA, None, 2, 4, 5), (pB, d * (1.0 if step == 1 else -0.5), 1, 3, 6)])
    J, grads, _ = G.rollout_parametric(U0, prims(dB), 2, 0.04, dx, 1.0, bc, loss, band=band)
    rng = np.random.default_rng(3)
    dd = rng.standard_normal(pB.shape) * 0.1
    h = 1e-3
    Jp = G.rollout_parametric(U0, prims(dB + h * dd), 2, 0.04, dx, 1.0, bc, loss, band=band)[0]
    Jm = G.rollout_parametric(U0, prims(dB - h * dd), 2, 0.04, dx, 1.0, bc, loss, band=band)[0]
    fd = (Jp - Jm) / (2 * h)
    an = grads[0][1][1] @ dd - 0.5 * (grads[1][1][1] @ dd)
    assert abs(fd - an) < 1e-6 * max(abs(fd), abs(an)), (fd, an)
    assert abs(fd) > 1e-6
