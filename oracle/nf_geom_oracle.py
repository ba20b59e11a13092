"""fp64 CPU oracle for the differentiable parametric geometry: polar-Bezier cross-sections,
key sections along z, CSG, the node SDF phi, its adjoint to the parameters, and the solid velocity of a moving
geometry.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It shares no code with the CUDA path (paper_2405_14903_b200/csrc) and never imports it.  Plain NumPy, float64, in the
order and notation of PAPER.md:L55-67 (section 2.2) and L337-347 (appendix A), with the readings R25-R31 of
DESIGN.md section 3 (the appendix leaves the endpoint radius, the z-interpolation -- Eq. 10 is garbled --, the
distance computation and the velocity function open).

Parameter vector of one "closed 3-D surface" with K key cross-sections of N cubic Bezier curves each
("The parametrization includes z=z0 and z1 ... and the parameters for each key cross-section"):
    params = [z0, z1,  then for key k = 0..K-1:  cx_k, cy_k, rho1_k[0..N-1], rho2_k[0..N-1]]      (2 + K (2 + 2N))
in physical units; node (i, j, k) of the grid sits at (i dx, j dx, k dx); phi arrays are [k, j, i] like nf_oracle.

Sign convention (R2): phi > 0 in the fluid.  A primitive is solid INSIDE its closed surface (phi < 0
there); `complement=True` flips it (fluid inside: a chamber).

parity unpinned: nothing in this file.  Pins: tests/test_oracle_geometry.py.  rollout_parametric composes this
file with oracle/nf_oracle.py (the only import between the two oracle modules).
"""
import numpy as np


def n_params(K, N):
    return 2 + K * (2 + 2 * N)


def unpack(params, K, N):
    """-> z0, z1, c (K,2), rho1 (K,N), rho2 (K,N)."""
    p = np.asarray(params, dtype=np.float64)
    assert p.shape == (n_params(K, N),)
    keys = p[2:].reshape(K, 2 + 2 * N)
    return p[0], p[1], keys[:, 0:2], keys[:, 2:2 + N], keys[:, 2 + N:]


# ----------------------------------------------------------------------------------------------------
# 3-D: key cross-sections interpolated along z              PAPER.md:L343-347 (Eq. 10, garbled; R27)
# ----------------------------------------------------------------------------------------------------
def section_at(params, K, N, z):
    """Centre and control radii of the cross-section at height z: the K key sections sit evenly spaced on
    [z0, z1] (L343 "assumed to be evenly spaced") and the section in between is their piecewise-linear interpolant
    in s = (z - z0)/(z1 - z0) clamped to [0, 1] (R27).  -> (c (2,), rho1 (N,), rho2 (N,), k0, lam, s, clamped)."""
    z0, z1, c, r1, r2 = unpack(params, K, N)
    s_raw = (z - z0) / (z1 - z0)
    s = min(max(s_raw, 0.0), 1.0)
    clamped = not (0.0 < s_raw < 1.0)
    if K == 1:
        return c[0].copy(), r1[0].copy(), r2[0].copy(), 0, 0.0, s, True
    t = s * (K - 1)
    k0 = min(int(np.floor(t)), K - 2)
    lam = t - k0
    return ((1 - lam) * c[k0] + lam * c[k0 + 1], (1 - lam) * r1[k0] + lam * r1[k0 + 1],
            (1 - lam) * r2[k0] + lam * r2[k0 + 1], k0, lam, s, clamped)


# ----------------------------------------------------------------------------------------------------
# 2-D: N connected cubic Bezier curves in the polar frame       PAPER.md:L339-341 (R25, R26)
# ----------------------------------------------------------------------------------------------------
def control_points(c, rho1, rho2):
    """Control polygon of the closed curve: curve i spans [theta_i, theta_{i+1}], theta_i = 2 pi i / N; its inner
    control points sit at an angular displacement delta = 2 pi / (3N) from the curve's endpoints (L341):
        p0_i = c + rho1_i (cos, sin)(theta_i + delta),   p1_i = c + rho2_i (cos, sin)(theta_{i+1} - delta);
    the endpoint e1_i = e0_{i+1} lies on the ray theta_{i+1} (the curve "spans an arc of 2 pi / N") and on the line
    p1_i -- p0_{i+1} (L341 "colinearity"), which puts it at the radius
        r_i = 2 cos(delta) rho2_i rho1_{i+1} / (rho2_i + rho1_{i+1})                                   (R25).
    -> e0, p0, p1, e1, each (N, 2)."""
    N = len(rho1)
    th = 2 * np.pi * np.arange(N + 1) / N
    dl = 2 * np.pi / (3 * N)
    a = rho2                      # rho2_i
    b = np.roll(rho1, -1)         # rho1_{i+1}
    re = 2 * np.cos(dl) * a * b / (a + b)           # radius of e1_i
    e1 = c + re[:, None] * np.stack([np.cos(th[1:]), np.sin(th[1:])], axis=1)
    e0 = np.roll(e1, 1, axis=0)                      # e0_i = e1_{i-1}
    p0 = c + rho1[:, None] * np.stack([np.cos(th[:-1] + dl), np.sin(th[:-1] + dl)], axis=1)
    p1 = c + rho2[:, None] * np.stack([np.cos(th[1:] - dl), np.sin(th[1:] - dl)], axis=1)
    return e0, p0, p1, e1


def bernstein3(t):
    return np.array([(1 - t) ** 3, 3 * (1 - t) ** 2 * t, 3 * (1 - t) * t ** 2, t ** 3])


def polyline(c, rho1, rho2, M):
    """The curve as the method sees it (R26): every Bezier curve sampled at t = m / M, m = 0..M-1 -> the closed
    polygon V[0..NM-1] (vertex i M + m on curve i), the distance computation of L141 being the exact distance to
    that polygon."""
    e0, p0, p1, e1 = control_points(c, rho1, rho2)
    N = len(rho1)
    V = np.zeros((N * M, 2))
    for i in range(N):
        for m in range(M):
            B = bernstein3(m / M)
            V[i * M + m] = B[0] * e0[i] + B[1] * p0[i] + B[2] * p1[i] + B[3] * e1[i]
    return V


def _closest_on_polygon(V, X, Y):
    """For points (X, Y) (arrays): squared distance to the closed polygon V, the segment index, the parameter tau
    on it, and the even-odd crossing parity (True = inside)."""
    n = len(V)
    best = np.full(X.shape, np.inf)
    bk = np.zeros(X.shape, dtype=np.int64)
    bt = np.zeros(X.shape)
    inside = np.zeros(X.shape, dtype=bool)
    for k in range(n):
        ax, ay = V[k]
        bx, by = V[(k + 1) % n]
        ex, ey = bx - ax, by - ay
        l2 = ex * ex + ey * ey
        tau = ((X - ax) * ex + (Y - ay) * ey) / l2 if l2 > 0 else np.zeros(X.shape)
        tau = np.clip(tau, 0.0, 1.0)
        qx, qy = ax + tau * ex, ay + tau * ey
        d2 = (X - qx) ** 2 + (Y - qy) ** 2
        upd = d2 < best
        best = np.where(upd, d2, best)
        bk = np.where(upd, k, bk)
        bt = np.where(upd, tau, bt)
        # ray towards +x from (X, Y): the edge crosses it iff its ends straddle Y and the crossing lies right of X
        strad = (ay > Y) != (by > Y)
        with np.errstate(divide="ignore", invalid="ignore"):
            xc = ax + (Y - ay) * ex / ey
        inside ^= strad & (X < xc)
    return best, bk, bt, inside


def sdf2d(c, rho1, rho2, M, X, Y):
    """Signed distance (negative inside) of points to the cross-section's polygon."""
    d2, _, _, inside = _closest_on_polygon(polyline(c, rho1, rho2, M), X, Y)
    return np.where(inside, -1.0, 1.0) * np.sqrt(d2)


# ----------------------------------------------------------------------------------------------------
# phi on the grid nodes                                       PAPER.md:L89 ("SDF phi^{n+1} ... derived from the solid")
# ----------------------------------------------------------------------------------------------------
def sdf_nodes(params, K, N, M, nx, ny, nz, dx, complement=False):
    """phi[k, j, i] at node (i dx, j dx, k dx): d = max(d2(x, y; section(z)), z0 - z, z - z1) -- the cross-section's
    signed distance intersected with the slab z0 <= z <= z1 (R28) -- and phi = d (solid inside) or -d (complement)."""
    z0, z1 = float(params[0]), float(params[1])
    X, Y = np.meshgrid(np.arange(nx + 1) * dx, np.arange(ny + 1) * dx, indexing="xy")  # [j, i]
    phi = np.zeros((nz + 1, ny + 1, nx + 1))
    for k in range(nz + 1):
        z = k * dx
        c, r1, r2 = section_at(params, K, N, z)[:3]
        d = np.maximum(sdf2d(c, r1, r2, M, X, Y), max(z0 - z, z - z1))
        phi[k] = -d if complement else d
    return phi


def csg(op, a, b):
    """CSG on solids with phi > 0 = fluid ("Union and intersection"): the union of two solids is the
    min of their phi, the intersection the max (R29)."""
    return np.minimum(a, b) if op == "union" else np.maximum(a, b)


def csg_adjoint(op, a, b, gout):
    """Routes dJ/dphi_out to the operand that supplied the value (ties -> a)."""
    take_a = (a <= b) if op == "union" else (a >= b)
    return np.where(take_a, gout, 0.0), np.where(take_a, 0.0, gout)


# ----------------------------------------------------------------------------------------------------
# dJ/dphi -> dJ/dparams
# ----------------------------------------------------------------------------------------------------
def _section_grad_to_params(g, K, N, k0, lam, s, clamped, params, gc, gr1, gr2, z):
    """Adds the gradient w.r.t. the interpolated section (gc (2,), gr1 (N,), gr2 (N,)) to g (params layout)."""
    z0, z1, c, r1, r2 = unpack(params, K, N)
    W = 2 + 2 * N

    def key_slice(k):
        return slice(2 + k * W, 2 + (k + 1) * W)
    gsec = np.concatenate([gc, gr1, gr2])
    if K == 1:
        g[key_slice(0)] += gsec
        return
    g[key_slice(k0)] += (1 - lam) * gsec
    g[key_slice(k0 + 1)] += lam * gsec
    if not clamped:
        # d section / d s = (K-1) (key[k0+1] - key[k0]);  s = (z - z0) / (z1 - z0)
        dsec = (K - 1) * (np.asarray(params)[key_slice(k0 + 1)] - np.asarray(params)[key_slice(k0)])
        gs = float(gsec @ dsec)
        g[0] += gs * (z - z1) / (z1 - z0) ** 2
        g[1] += gs * (-(z - z0)) / (z1 - z0) ** 2


def sdf_nodes_adjoint(params, K, N, M, nx, ny, nz, dx, gphi, complement=False):
    """g[params] = sum over nodes of gphi * d phi / d params, the hand-written reverse of sdf_nodes:
    slab term active -> z0 / z1 only; else with q = (1 - tau) V_k + tau V_{k+1} the closest point and
    nh = (x - q)/|x - q|: d d2 / d V_k = -sgn (1 - tau) nh, d d2 / d V_{k+1} = -sgn tau nh (tau is stationary or
    clamped), then V -> Bezier control points (Bernstein weights) -> (c, rho1, rho2) of the section (the endpoint
    radius by the quotient rule) -> the key sections and z0, z1."""
    params = np.asarray(params, dtype=np.float64)
    z0, z1 = params[0], params[1]
    g = np.zeros_like(params)
    th = 2 * np.pi * np.arange(N + 1) / N
    dl = 2 * np.pi / (3 * N)
    X, Y = np.meshgrid(np.arange(nx + 1) * dx, np.arange(ny + 1) * dx, indexing="xy")
    sign_out = -1.0 if complement else 1.0
    for k in range(nz + 1):
        z = k * dx
        gd = sign_out * gphi[k]
        if not np.any(gd):
            continue
        c, r1, r2, k0, lam, s, clamped = section_at(params, K, N, z)
        V = polyline(c, r1, r2, M)
        d2, bk, bt, inside = _closest_on_polygon(V, X, Y)
        sgn = np.where(inside, -1.0, 1.0)
        dist = np.sqrt(d2)
        slab = max(z0 - z, z - z1)
        use_slab = slab > sgn * dist
        # slab
        gsl = float(np.sum(gd[use_slab]))
        if z0 - z >= z - z1:
            g[0] += gsl
        else:
            g[1] -= gsl
        # cross-section
        gV = np.zeros_like(V)
        n = len(V)
        js, is_ = np.nonzero((~use_slab) & (gd != 0) & (dist > 0))
        for j, i in zip(js, is_):
            kk, tau = bk[j, i], bt[j, i]
            q = (1 - tau) * V[kk] + tau * V[(kk + 1) % n]
            nh = (np.array([X[j, i], Y[j, i]]) - q) / dist[j, i]
            gq = -sgn[j, i] * nh * gd[j, i]
            gV[kk] += (1 - tau) * gq
            gV[(kk + 1) % n] += tau * gq
        if not np.any(gV):
            continue
        # V -> control points
        gE0 = np.zeros((N, 2)); gP0 = np.zeros((N, 2)); gP1 = np.zeros((N, 2)); gE1 = np.zeros((N, 2))
        for i in range(N):
            for m in range(M):
                B = bernstein3(m / M)
                gv = gV[i * M + m]
                gE0[i] += B[0] * gv; gP0[i] += B[1] * gv; gP1[i] += B[2] * gv; gE1[i] += B[3] * gv
        # control points -> (c, rho1, rho2)
        gc = (gE0 + gP0 + gP1 + gE1).sum(axis=0)
        gr1 = np.zeros(N); gr2 = np.zeros(N)
        for i in range(N):
            gr1[i] += gP0[i] @ np.array([np.cos(th[i] + dl), np.sin(th[i] + dl)])
            gr2[i] += gP1[i] @ np.array([np.cos(th[i + 1] - dl), np.sin(th[i + 1] - dl)])
            # endpoint e1_i = e0_{i+1}, radius r = 2 cos(dl) a b / (a + b), a = rho2_i, b = rho1_{i+1}
            ip = (i + 1) % N
            ge = (gE1[i] + gE0[ip]) @ np.array([np.cos(th[i + 1]), np.sin(th[i + 1])])
            a, b = r2[i], r1[ip]
            gr2[i] += ge * 2 * np.cos(dl) * b * b / (a + b) ** 2
            gr1[ip] += ge * 2 * np.cos(dl) * a * a / (a + b) ** 2
        _section_grad_to_params(g, K, N, k0, lam, s, clamped, params, gc, gr1, gr2, z)
    return g


# ----------------------------------------------------------------------------------------------------
# solid velocity of a moving geometry                         PAPER.md:L89, L132 ("velocity ... of the geometry U_s")
# ----------------------------------------------------------------------------------------------------
def _velocity_points(params, pdot, K, N, M, X, Y, z):
    """At points (X, Y) of the plane z: the velocity of the surface along its own in-plane normal (R30).  With
    q the closest point of the section's polygon (segment k, parameter tau held fixed) and nh the unit vector from
    q to the point, qdot = (1 - tau) Vdot_k + tau Vdot_{k+1} is q's velocity under params(t) moving at pdot at
    fixed z, and the solid velocity is its normal part (nh . qdot) nh; where the slab term of R28 is the active one
    the surface is a cap moving at (0, 0, z0dot) or (0, 0, z1dot).  -> (us, vs, ws, d) arrays like X, d the
    primitive's signed distance max(d2, slab) there."""
    params = np.asarray(params, dtype=np.float64)
    pdot = np.asarray(pdot, dtype=np.float64)
    z0, z1 = params[0], params[1]
    c, r1, r2, k0, lam, s, clamped = section_at(params, K, N, z)
    V = polyline(c, r1, r2, M)
    # Vdot: derivative of the vertices along pdot at fixed z (forward mode, written out)
    W = 2 + 2 * N
    if K == 1:
        secdot = pdot[2:2 + W].copy()
    else:
        kA = slice(2 + k0 * W, 2 + (k0 + 1) * W)
        kB = slice(2 + (k0 + 1) * W, 2 + (k0 + 2) * W)
        secdot = (1 - lam) * pdot[kA] + lam * pdot[kB]
        if not clamped:
            sdot = (pdot[0] * (z - z1) - pdot[1] * (z - z0)) / (z1 - z0) ** 2
            secdot = secdot + sdot * (K - 1) * (params[kB] - params[kA])
    cd, r1d, r2d = secdot[0:2], secdot[2:2 + N], secdot[2 + N:]
    th = 2 * np.pi * np.arange(N + 1) / N
    dl = 2 * np.pi / (3 * N)
    a, b = r2, np.roll(r1, -1)
    ad, bd = r2d, np.roll(r1d, -1)
    red = 2 * np.cos(dl) * (b * b * ad + a * a * bd) / (a + b) ** 2
    e1d = cd + red[:, None] * np.stack([np.cos(th[1:]), np.sin(th[1:])], axis=1)
    e0d = np.roll(e1d, 1, axis=0)
    p0d = cd + r1d[:, None] * np.stack([np.cos(th[:-1] + dl), np.sin(th[:-1] + dl)], axis=1)
    p1d = cd + r2d[:, None] * np.stack([np.cos(th[1:] - dl), np.sin(th[1:] - dl)], axis=1)
    Vd = np.zeros_like(V)
    for i in range(N):
        for m in range(M):
            B = bernstein3(m / M)
            Vd[i * M + m] = B[0] * e0d[i] + B[1] * p0d[i] + B[2] * p1d[i] + B[3] * e1d[i]
    d2, bk, bt, inside = _closest_on_polygon(V, X, Y)
    n = len(V)
    dist = np.sqrt(d2)
    sgn = np.where(inside, -1.0, 1.0)
    q = (1 - bt)[..., None] * V[bk] + bt[..., None] * V[(bk + 1) % n]
    qd = (1 - bt)[..., None] * Vd[bk] + bt[..., None] * Vd[(bk + 1) % n]
    with np.errstate(divide="ignore", invalid="ignore"):
        nhx = np.where(dist > 0, (X - q[..., 0]) / dist, 0.0)
        nhy = np.where(dist > 0, (Y - q[..., 1]) / dist, 0.0)
    vn = nhx * qd[..., 0] + nhy * qd[..., 1]
    us, vs, ws = vn * nhx, vn * nhy, np.zeros_like(vn)
    slab = max(z0 - z, z - z1)
    use_slab = slab > sgn * dist
    zdot = pdot[0] if (z0 - z >= z - z1) else pdot[1]
    us = np.where(use_slab, 0.0, us)
    vs = np.where(use_slab, 0.0, vs)
    ws = np.where(use_slab, zdot, ws)
    return us, vs, ws, np.maximum(sgn * dist, slab)


def solid_velocity_faces(params, pdot, K, N, M, nx, ny, nz, dx, band=np.inf, out=None):
    """U_s on the MAC faces (layout of nf_oracle: us (nz, ny, nx+1), vs (nz, ny+1, nx), ws (nz+1, ny, nx)): each
    component sampled at its own face centres.  Only faces whose distance to the primitive is <= band are written
    (R30: several moving parts are composed by one call each with a band of a few dx; the default writes all);
    the others keep `out`'s values (zero if out is None)."""
    if out is None:
        us = np.zeros((nz, ny, nx + 1)); vs = np.zeros((nz, ny + 1, nx)); ws = np.zeros((nz + 1, ny, nx))
    else:
        us, vs, ws = (np.array(a, dtype=np.float64) for a in out)
    xi, xc = np.arange(nx + 1) * dx, (np.arange(nx) + 0.5) * dx
    yj, yc = np.arange(ny + 1) * dx, (np.arange(ny) + 0.5) * dx
    for k in range(nz):
        z = (k + 0.5) * dx
        X, Y = np.meshgrid(xi, yc, indexing="xy")
        r = _velocity_points(params, pdot, K, N, M, X, Y, z)
        us[k] = np.where(r[3] <= band, r[0], us[k])
        X, Y = np.meshgrid(xc, yj, indexing="xy")
        r = _velocity_points(params, pdot, K, N, M, X, Y, z)
        vs[k] = np.where(r[3] <= band, r[1], vs[k])
    X, Y = np.meshgrid(xc, yc, indexing="xy")
    for k in range(nz + 1):
        r = _velocity_points(params, pdot, K, N, M, X, Y, k * dx)
        ws[k] = np.where(r[3] <= band, r[2], ws[k])
    return us, vs, ws


def solid_velocity_faces_adjoint(params, K, N, M, nx, ny, nz, dx, gus, gvs, gws, band=np.inf):
    """dJ/dpdot = J_v^T (gus, gvs, gws): U_s is linear in pdot, so the transpose is assembled column by column from
    solid_velocity_faces on the unit vectors (the definition of the transpose; R31: the dependence of U_s on
    params themselves -- through the closest point and the normal -- is not differentiated)."""
    P = n_params(K, N)
    g = np.zeros(P)
    for a in range(P):
        e = np.zeros(P); e[a] = 1.0
        us, vs, ws = solid_velocity_faces(params, e, K, N, M, nx, ny, nz, dx, band)
        g[a] = np.sum(us * gus) + np.sum(vs * gvs) + np.sum(ws * gws)
    return g


# ----------------------------------------------------------------------------------------------------
# the co-design loop: parametric geometry inside the time stepping
# ----------------------------------------------------------------------------------------------------
def rollout_parametric(U0, prims_fn, nsteps, dt, dx, dt_over_rho, bc, loss_fn, tol=1e-12, advect_on=True, band=np.inf):
    """N steps "advect -> geometry at t^{n+1} -> project" (R15) with the solid given by parametric primitives, and
    the backward pass down to the parameters (L132-141).

    prims_fn(step) -> list of (params, pdot or None, K, N, M) for step = 1..N: the solid is the union (R29) of the
    primitives; a primitive with pdot moves and supplies U_s on the faces within `band` of it (R30), in list order.
    Returns (J, grads, dJ/dU0), grads[step-1][i] = (dJ/dparams, dJ/dpdot or None) of primitive i at that step:
    dJ/dparams through phi only (Eq. 9a -> weight builder -> union -> distance, L141), dJ/dpdot the transpose of the
    velocity map applied to Eq. 9b's dJ/dU_s (R31)."""
    from . import nf_oracle as orc
    U = [np.asarray(a, dtype=np.float64) for a in U0]
    nz, ny, nx = U[0].shape[0], U[0].shape[1], U[0].shape[2] - 1
    tape = []
    for n in range(1, nsteps + 1):
        Uprev = U
        Ut = orc.advect(U, dt, dx) if advect_on else [a.copy() for a in U]
        prims = prims_fn(n)
        phis = [sdf_nodes(p, K, N, M, nx, ny, nz, dx) for (p, pd, K, N, M) in prims]
        partial = [phis[0]]
        for f in phis[1:]:
            partial.append(csg("union", partial[-1], f))
        phi = partial[-1]
        us = None
        for (p, pd, K, N, M) in prims:
            if pd is not None:
                us = solid_velocity_faces(p, pd, K, N, M, nx, ny, nz, dx, band, us)
        alpha = orc.face_weights(phi, bc)
        U, pr = orc.project(Ut, alpha, us, dx, dt_over_rho, bc, tol=tol)
        tape.append((Uprev, Ut, prims, phis, partial, us, alpha, pr, phi))
    J, g = loss_fn(U)
    g = [np.asarray(a, dtype=np.float64) for a in g]
    grads = [None] * nsteps
    for n in range(nsteps, 0, -1):
        Uprev, Ut, prims, phis, partial, us, alpha, pr, phi = tape[n - 1]
        g_ut, g_alpha, g_us, _ = orc.project_adjoint(g, alpha, pr, Ut, us, dx, dt_over_rho, bc, tol=tol)
        g_phi = orc.weights_adjoint(phi, g_alpha[0], g_alpha[1], g_alpha[2], bc)
        gphis = [None] * len(prims)
        for i in range(len(prims) - 1, 0, -1):
            g_phi, gphis[i] = csg_adjoint("union", partial[i - 1], phis[i], g_phi)
        gphis[0] = g_phi
        # a face's U_s was written by the LAST moving primitive whose band covers it: walk the list backwards and
        # clear dJ/dU_s on the faces a primitive owns once it has taken them (its velocity map with pdot = 0 writes 0
        # exactly there)
        g_us = [a.copy() for a in g_us]
        out = [None] * len(prims)
        for i in range(len(prims) - 1, -1, -1):
            p, pd, K, N, M = prims[i]
            gp = sdf_nodes_adjoint(p, K, N, M, nx, ny, nz, dx, gphis[i])
            gd = None
            if pd is not None:
                gd = solid_velocity_faces_adjoint(p, K, N, M, nx, ny, nz, dx, *g_us, band=band)
                g_us = list(solid_velocity_faces(p, np.zeros_like(np.asarray(p, dtype=np.float64)), K, N, M, nx, ny,
                                                 nz, dx, band, out=g_us))
            out[i] = (gp, gd)
        grads[n - 1] = out
        g = orc.advect_adjoint(Uprev, g_ut, dt, dx) if advect_on else g_ut
    return J, grads, g
