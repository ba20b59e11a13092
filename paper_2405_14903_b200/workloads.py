"""Seeded synthetic inputs for the five BASELINE.json configs (DESIGN.md §5 gives the recipes).

This module serves BOTH the oracle tests and the CUDA path and therefore holds none of the method's
arithmetic: it only draws random fields and evaluates closed-form geometry (signed distances and rigid /
prescribed solid velocities) -- the *inputs* the paper says "can be derived from the solid geometry"
(PAPER.md:L89).  It imports neither oracle/ nor the CUDA binding.

All arrays are float32, C-ordered [k, j, i] (x fastest):
  phi: nodes (nz+1, ny+1, nx+1), > 0 in fluid;  u: (nz, ny, nx+1);  v: (nz, ny+1, nx);  w: (nz+1, ny, nx).
Lengths are in cell units unless stated otherwise.
"""
import numpy as np

CLOSED, DIRICHLET = 0, 1


def face_shapes(nx, ny, nz):
    return (nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)


def node_coords(nx, ny, nz, dtype=np.float64):
    k, j, i = np.meshgrid(np.arange(nz + 1, dtype=dtype), np.arange(ny + 1, dtype=dtype),
                          np.arange(nx + 1, dtype=dtype), indexing="ij", sparse=True)
    return i, j, k


def face_coords(nx, ny, nz, comp, dtype=np.float64):
    """Cell-unit positions of the faces of family comp (0: x-faces at (i, j+1/2, k+1/2), ...)."""
    sh = face_shapes(nx, ny, nz)[comp]
    off = [(0.0, 0.5, 0.5), (0.5, 0.0, 0.5), (0.5, 0.5, 0.0)][comp]
    k, j, i = np.meshgrid(np.arange(sh[0], dtype=dtype), np.arange(sh[1], dtype=dtype),
                          np.arange(sh[2], dtype=dtype), indexing="ij", sparse=True)
    return i + off[0], j + off[1], k + off[2]


def random_velocity(rng, nx, ny, nz, kind="uniform"):
    out = []
    for sh in face_shapes(nx, ny, nz):
        a = rng.uniform(-1, 1, sh) if kind == "uniform" else rng.standard_normal(sh)
        out.append(a.astype(np.float32))
    return out


# ------------------------------------------------------------------------------------------------------
# closed-form signed distances (phi > 0 outside the solid = fluid)
# ------------------------------------------------------------------------------------------------------
def sdf_sphere(x, y, z, c, r):
    return np.sqrt((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2) - r


def sdf_box(x, y, z, c, half, rot_y=0.0):
    """Exact SDF of a box with half-extents `half`, centre c, rotated by rot_y about the y axis."""
    cs, sn = np.cos(rot_y), np.sin(rot_y)
    dx_, dy_, dz_ = x - c[0], y - c[1], z - c[2]
    # rotate the query point by -rot_y into the box frame
    lx = cs * dx_ - sn * dz_
    lz = sn * dx_ + cs * dz_
    qx, qy, qz = np.abs(lx) - half[0], np.abs(dy_) - half[1], np.abs(lz) - half[2]
    outside = np.sqrt(np.maximum(qx, 0) ** 2 + np.maximum(qy, 0) ** 2 + np.maximum(qz, 0) ** 2)
    inside = np.minimum(np.maximum(qx, np.maximum(qy, qz)), 0)
    return outside + inside


# ------------------------------------------------------------------------------------------------------
# config 1: 32^3 sphere, one projection forward + adjoint           (BASELINE.json configs[0])
# ------------------------------------------------------------------------------------------------------
def config1(n=32, seed=1001, radius=None):
    rng = np.random.default_rng(seed)
    u, v, w = random_velocity(rng, n, n, n, "uniform")
    gu, gv, gw = random_velocity(rng, n, n, n, "normal")
    x, y, z = node_coords(n, n, n)
    r = n / 4.0 if radius is None else radius
    phi = sdf_sphere(x, y, z, (n / 2.0,) * 3, r).astype(np.float32)
    return dict(nx=n, ny=n, nz=n, dx=1.0 / n, dt_over_rho=1.0, bc_types=(CLOSED,) * 6, bc_values=(0.0,) * 6,
                phi=phi, us=None, U=[u, v, w], g=[gu, gv, gw], tol=1e-6, maxit=200)


# ------------------------------------------------------------------------------------------------------
# config 2: 64^3, two oscillating plates, 10 full steps, dJ/dtheta      (BASELINE.json configs[1])
# ------------------------------------------------------------------------------------------------------
def config2_params(n=64):
    s = n / 64.0
    return dict(nx=n, ny=n, nz=n, dx=1.0 / n, dt=0.5 / n, dt_over_rho=0.5 / n, steps=10, T=40, theta=0.5,
                half=(16 * s, 24 * s, 2.0), centres=((32 * s, 32 * s, 16 * s), (32 * s, 32 * s, 48 * s)),
                bc_types=(CLOSED,) * 6, bc_values=(0.0,) * 6, loss_lo=int(24 * s), loss_hi=int(40 * s),
                tol=1e-6, maxit=200)


def config2_solid(P, step, theta, dtype=np.float32):
    """phi and u_s at time level `step` (1-based: t^{n+1} of step n, R15) for amplitude theta.
    Plate velocity theta*sin(2 pi t/T) x_hat; displacement s(t) = theta (T dt/2 pi)(1-cos(2 pi t/T))/dx cells.
    Also returns d phi/d theta and d u_s/d theta (closed form) for the end-to-end gradient."""
    n = P["nx"]
    T, dt, dx = P["T"], P["dt"], P["dx"]
    ang = 2 * np.pi * step / T
    vel = theta * np.sin(ang)
    dvel = np.sin(ang)
    shift = theta * (T * dt / (2 * np.pi)) * (1 - np.cos(ang)) / dx
    dshift = (T * dt / (2 * np.pi)) * (1 - np.cos(ang)) / dx
    x, y, z = node_coords(n, n, n)
    phis = [sdf_box(x, y, z, (c[0] + shift, c[1], c[2]), P["half"]) for c in P["centres"]]
    phi = np.minimum(phis[0], phis[1])
    # d phi / d theta = -d phi/d x * dshift ; central difference of the closed form in fp64 (h = 1e-6 cells)
    h = 1e-6
    ph = [np.minimum(*[sdf_box(x, y, z, (c[0] + shift + e, c[1], c[2]), P["half"]) for c in P["centres"]])
          for e in (h, -h)]
    dphi = (ph[0] - ph[1]) / (2 * h) * dshift
    shu, shv, shw = face_shapes(n, n, n)
    us = [np.full(shu, vel, dtype=dtype), np.zeros(shv, dtype=dtype), np.zeros(shw, dtype=dtype)]
    dus = [np.full(shu, dvel, dtype=np.float64), np.zeros(shv), np.zeros(shw)]
    return phi.astype(dtype), us, dphi, dus


# ------------------------------------------------------------------------------------------------------
# config 3: 128^3 chamber pump with a Dirichlet outlet                  (BASELINE.json configs[2])
# ------------------------------------------------------------------------------------------------------
def config3_params(n=128, seed=1003):
    s = n / 128.0
    rng = np.random.default_rng(seed)
    axes = np.array([56.0, 40.0, 40.0]) * s
    centre = np.array([64.0, 64.0, 64.0]) * s
    # 16 seeded points on the ellipsoid surface
    d = rng.standard_normal((16, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    bumps = centre + d * axes
    theta = rng.normal(0.0, 0.2, 16)
    return dict(nx=n, ny=n, nz=n, dx=1.0 / n, dt=0.5 / n, dt_over_rho=0.5 / n, steps=50, period=50,
                axes=axes, centre=centre, tube_r=max(6.0 * s, 2.0), sigma=10.0 * s, bumps=bumps, theta=theta,
                bc_types=(CLOSED, DIRICHLET, CLOSED, CLOSED, CLOSED, CLOSED), bc_values=(0.0,) * 6,
                tol=1e-6, maxit=400)


def _config3_fluid_sdf(P, x, y, z):
    """Negative inside the fluid region (ellipsoid union tube)."""
    a, c = P["axes"], P["centre"]
    X, Y, Z = x - c[0], y - c[1], z - c[2]
    k0 = np.sqrt((X / a[0]) ** 2 + (Y / a[1]) ** 2 + (Z / a[2]) ** 2)
    k1 = np.sqrt((X / a[0] ** 2) ** 2 + (Y / a[1] ** 2) ** 2 + (Z / a[2] ** 2) ** 2)
    with np.errstate(divide="ignore", invalid="ignore"):
        ell = np.where(k1 > 0, k0 * (k0 - 1.0) / np.where(k1 > 0, k1, 1.0), -min(a))
    # tube along +x from the ellipsoid centre to beyond the +x face
    rad = np.sqrt(Y ** 2 + Z ** 2) - P["tube_r"]
    tube = np.maximum(rad, -X)  # half-infinite cylinder x >= centre
    return np.minimum(ell, tube)


def config3_solid(P, step, theta=None, dtype=np.float32):
    """Static phi; wall velocity u_s = n * sum_k theta_k sin(2 pi t/period) exp(-|x-c_k|^2/2 sigma^2),
    n = -grad(phi)/|grad(phi)| (pointing into the solid).  Returns phi, us, and the per-parameter basis
    d u_s/d theta_k as a callable-free list only when theta is given as 'basis' (kept small: faces near
    the wall dominate, but the arrays are dense)."""
    n = P["nx"]
    th = P["theta"] if theta is None else np.asarray(theta, dtype=np.float64)
    x, y, z = node_coords(n, n, n)
    phi = -_config3_fluid_sdf(P, x, y, z)
    mod = np.sin(2 * np.pi * step / P["period"])
    us = []
    h = 1e-3
    for comp in range(3):
        fx, fy, fz = face_coords(n, n, n, comp)
        f0 = -_config3_fluid_sdf(P, fx, fy, fz)
        gx = (-_config3_fluid_sdf(P, fx + h, fy, fz) + _config3_fluid_sdf(P, fx - h, fy, fz)) / (2 * h)
        gy = (-_config3_fluid_sdf(P, fx, fy + h, fz) + _config3_fluid_sdf(P, fx, fy - h, fz)) / (2 * h)
        gz = (-_config3_fluid_sdf(P, fx, fy, fz + h) + _config3_fluid_sdf(P, fx, fy, fz - h)) / (2 * h)
        nrm = np.sqrt(gx ** 2 + gy ** 2 + gz ** 2) + 1e-12
        ncomp = -(gx, gy, gz)[comp] / nrm
        amp = 0.0
        for kk in range(16):
            ck = P["bumps"][kk]
            amp = amp + th[kk] * np.exp(-((fx - ck[0]) ** 2 + (fy - ck[1]) ** 2 + (fz - ck[2]) ** 2)
                                         / (2 * P["sigma"] ** 2))
        us.append((ncomp * amp * mod * np.ones_like(f0)).astype(dtype))
    return phi.astype(dtype), us


def config3_us_basis(P, step, kk):
    """d u_s / d theta_kk (float64 face arrays) -- u_s is linear in theta."""
    e = np.zeros(16)
    e[kk] = 1.0
    _, us = config3_solid(P, step, theta=e, dtype=np.float64)
    return us


# ------------------------------------------------------------------------------------------------------
# config 4: 256^3 channel with a rotating gate (the headline workload)     (BASELINE.json configs[3])
# ------------------------------------------------------------------------------------------------------
def config4_params(n=256, seed=1004):
    s = n / 256.0
    return dict(nx=n, ny=n, nz=n, dx=1.0 / n, dt=0.5 / n, dt_over_rho=0.5 / n, steps=20, seed=seed,
                half=(2.0, 64.0 * s, 32.0 * s), centre=(128.0 * s,) * 3, omega_step=0.05,
                bc_types=(DIRICHLET, DIRICHLET, CLOSED, CLOSED, CLOSED, CLOSED),
                bc_values=(1.0, 0.0, 0.0, 0.0, 0.0, 0.0), tol=1e-6, maxit=400)


def config4_initial_velocity(P):
    rng = np.random.default_rng(P["seed"])
    n = P["nx"]
    shu, shv, shw = face_shapes(n, n, n)
    u = (1.0 + 0.01 * rng.standard_normal(shu)).astype(np.float32)
    v = (0.01 * rng.standard_normal(shv)).astype(np.float32)
    w = (0.01 * rng.standard_normal(shw)).astype(np.float32)
    return [u, v, w]


def config4_solid(P, step, omega_step=None, dtype=np.float32):
    """phi of the plate rotated by omega_step*step about y, and u_s = omega x (x - c) everywhere
    (world units: omega = omega_step/dt, lengths * dx)."""
    n = P["nx"]
    om = P["omega_step"] if omega_step is None else omega_step
    x, y, z = node_coords(n, n, n)
    phi = sdf_box(x, y, z, P["centre"], P["half"], rot_y=om * step)
    wv = om / P["dt"] * P["dx"]  # velocity per cell of lever arm
    us = []
    c = P["centre"]
    for comp in range(3):
        fx, fy, fz = face_coords(n, n, n, comp)
        # omega = (0, wy, 0):  omega x r = (wy*rz, 0, -wy*rx)
        if comp == 0:
            a = wv * (fz - c[2]) + 0 * fx + 0 * fy
        elif comp == 1:
            a = 0 * (fx + fy + fz)
        else:
            a = -wv * (fx - c[0]) + 0 * fy + 0 * fz
        us.append(np.ascontiguousarray(np.broadcast_to(a, face_shapes(n, n, n)[comp])).astype(dtype))
    return phi.astype(dtype), us


# ------------------------------------------------------------------------------------------------------
# config 5: solver sweep, 200 random spheres                             (BASELINE.json configs[4])
# ------------------------------------------------------------------------------------------------------
def config5_phi(n, seed=1005, nspheres=200, dtype=np.float32):
    rng = np.random.default_rng(seed + n)
    centres = rng.uniform(0, n, (nspheres, 3))
    radii = rng.uniform(2, 12, nspheres)
    phi = np.full((n + 1, n + 1, n + 1), 1e9, dtype=np.float32)
    ax = np.arange(n + 1, dtype=np.float32)
    for c, r in zip(centres, radii):
        lo = np.maximum(np.floor(c - r - 3).astype(int), 0)
        hi = np.minimum(np.ceil(c + r + 3).astype(int) + 1, n + 1)
        if np.any(hi <= lo):
            continue
        zz = ax[lo[2]:hi[2], None, None]; yy = ax[None, lo[1]:hi[1], None]; xx = ax[None, None, lo[0]:hi[0]]
        d = np.sqrt((xx - c[0]) ** 2 + (yy - c[1]) ** 2 + (zz - c[2]) ** 2) - r
        sub = phi[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]]
        np.minimum(sub, d.astype(np.float32), out=sub)
    # far from every sphere the exact distance is irrelevant (all four corners positive -> alpha = 1)
    np.minimum(phi, 3.0, out=phi)
    return phi.astype(dtype)


def config5_rhs(n, active, seed=1005):
    rng = np.random.default_rng(seed + 7 * n)
    b = rng.standard_normal((n, n, n)).astype(np.float32)
    b = np.where(active, b, 0).astype(np.float64)
    b = np.where(active, b - b.sum() / max(int(active.sum()), 1), 0.0)
    return b.astype(np.float32)


def fluid_components(au, av, aw):
    """Labels (1..K, 0 = inactive) of the face-connected sets of active cells, and K.  Graph utility only (labels the
    doubled lattice: cells at odd sites, open interior faces between them): used to draw right-hand sides that are
    compatible on every closed fluid pocket (BASELINE.json configs[4]: 'RHS i.i.d. N(0,1) with its mean removed')."""
    from scipy import ndimage
    nz, ny, nx = au.shape[0], au.shape[1], au.shape[2] - 1
    act = (au[:, :, :-1] + au[:, :, 1:] + av[:, :-1, :] + av[:, 1:, :] + aw[:-1] + aw[1:]) > 0
    lat = np.zeros((2 * nz + 1, 2 * ny + 1, 2 * nx + 1), dtype=bool)
    lat[1::2, 1::2, 1::2] = act
    lat[1::2, 1::2, 2:-1:2] = au[:, :, 1:-1] > 0
    lat[1::2, 2:-1:2, 1::2] = av[:, 1:-1, :] > 0
    lat[2:-1:2, 1::2, 1::2] = aw[1:-1] > 0
    lab, _ = ndimage.label(lat)
    cl = np.where(act, lab[1::2, 1::2, 1::2], 0)
    ids = np.unique(cl[act])
    remap = np.zeros(int(lab.max()) + 1, dtype=np.int64)
    remap[ids] = np.arange(1, ids.size + 1)
    return remap[cl], int(ids.size)


def config5_rhs_per_component(n, labels, seed=1005):
    """N(0,1) on the active cells with the mean over every fluid component removed (closed walls: every component is
    singular, so this is the compatible right-hand side of configs[4] without discarding any pocket)."""
    rng = np.random.default_rng(seed + 7 * n)
    b = np.where(labels > 0, rng.standard_normal((n, n, n)).astype(np.float32), 0).astype(np.float64)
    K = int(labels.max())
    sums = np.bincount(labels.ravel(), weights=b.ravel(), minlength=K + 1)
    cnt = np.maximum(np.bincount(labels.ravel(), minlength=K + 1), 1)
    mean = sums / cnt
    mean[0] = 0.0
    return (b - mean[labels]).astype(np.float32)


def keep_largest_component(au, av, aw):
    """Zero every face weight that does not touch the largest face-connected set of active cells
    (R12: the library removes the null space globally, so inputs must have one fluid component).
    Graph utility only: labels the doubled lattice (cells at even sites, open faces at odd sites)."""
    from scipy import ndimage
    nz, ny, nx = au.shape[0], au.shape[1], au.shape[2] - 1
    lat = np.zeros((2 * nz + 1, 2 * ny + 1, 2 * nx + 1), dtype=bool)
    lat[1::2, 1::2, 0::2] = au > 0
    lat[1::2, 0::2, 1::2] = av > 0
    lat[0::2, 1::2, 1::2] = aw > 0
    act = (au[:, :, :-1] + au[:, :, 1:] + av[:, :-1, :] + av[:, 1:, :] + aw[:-1] + aw[1:]) > 0
    lat[1::2, 1::2, 1::2] = act
    lab, nlab = ndimage.label(lat)
    cl = lab[1::2, 1::2, 1::2]
    if nlab <= 1:
        return au, av, aw, 1 if nlab else 0
    counts = np.bincount(cl[act].ravel(), minlength=nlab + 1)
    counts[0] = 0
    best = int(np.argmax(counts))
    ncomp = int(np.count_nonzero(counts))
    au = np.where(lab[1::2, 1::2, 0::2] == best, au, 0).astype(au.dtype)
    av = np.where(lab[1::2, 0::2, 1::2] == best, av, 0).astype(av.dtype)
    aw = np.where(lab[0::2, 1::2, 1::2] == best, aw, 0).astype(aw.dtype)
    return au, av, aw, ncomp


# ------------------------------------------------------------------------------------------------------
# NEXT-2: seeded parameter vectors of a polar-Bezier primitive (layout of include/nf.h: [z0, z1, K x (cx, cy,
# rho1[N], rho2[N])]).  Only draws numbers and fills the layout -- none of the geometry's arithmetic lives here.
# ------------------------------------------------------------------------------------------------------
def geom_n_params(K, N):
    return 2 + K * (2 + 2 * N)


def geom_random_params(seed, K, N, z0, z1, centre, radius, jitter=0.25, centre_jitter=0.03):
    """Radii radius * (1 +- jitter) on every control point, centres scattered by centre_jitter * radius."""
    rng = np.random.default_rng(seed)
    p = np.zeros(geom_n_params(K, N), dtype=np.float64)
    p[0], p[1] = z0, z1
    keys = p[2:].reshape(K, 2 + 2 * N)
    keys[:, 0] = centre[0] + centre_jitter * radius * rng.standard_normal(K)
    keys[:, 1] = centre[1] + centre_jitter * radius * rng.standard_normal(K)
    keys[:, 2:] = radius * (1.0 + jitter * rng.uniform(-1.0, 1.0, (K, 2 * N)))
    return p.astype(np.float32)


def geom_random_rates(seed, K, N, scale=1.0):
    rng = np.random.default_rng(seed)
    return (scale * rng.standard_normal(geom_n_params(K, N))).astype(np.float32)
