"""fp64 CPU oracle for the NeuralFluid pressure projection (forward + adjoint), advection and the
face-weight builder.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It shares no code with the CUDA path (paper_2405_14903_b200/csrc) and never imports it.
Everything is plain NumPy in float64, written in the order and notation of the paper
(/root/reference/PAPER.md, cited as PAPER.md:Lnnn) with the readings listed in DESIGN.md §3 ("R<n>").

Conventions ("pressures stored at cell centers and velocities at cell faces"):
  * arrays are C-ordered [k, j, i] (x fastest).  p: (nz, ny, nx).  u: (nz, ny, nx+1) -- u[k,j,i] is the
    x-face between cells i-1 and i.  v: (nz, ny+1, nx).  w: (nz+1, ny, nx).  phi: nodes (nz+1, ny+1, nx+1).
  * G  (cells -> faces, "matrix (1/dx) G for gradient operator"): (G p)_u[i] = p[i] - p[i-1].
  * G^T (faces -> cells): (G^T f)[i,j,k] = f_u[i] - f_u[i+1] + f_v[j] - f_v[j+1] + f_w[k] - f_w[k+1]
    so that -(1/dx) G^T is the divergence.
  * S = diag(alpha), c = dt/(rho dx), A = c G^T S G (Eq. 4).
  * domain faces 0..5 = -x,+x,-y,+y,-z,+z; bc type 0 = closed wall (alpha forced to 0, wall at rest, R19),
    type 1 = Dirichlet: a ghost cell one dx outside holds p_D (R6).

Parity status of each function is listed in DESIGN.md §4; the pins live in tests/test_oracle_*.py.
  parity unpinned: nothing in this file (solver iteration counts are not part of the oracle).
"""
import numpy as np

ALPHA_EPS = 1e-4  # R4: alpha < 1e-4 -> 0 (paper silent)


class BC:
    """Domain boundary conditions: type[f] in {0 closed wall, 1 Dirichlet}, value[f] = p_D (R6)."""

    def __init__(self, types=(0,) * 6, values=(0.0,) * 6):
        self.types = tuple(int(t) for t in types)
        self.values = tuple(float(v) for v in values)

    def ghost(self, homogeneous=False):
        return [0.0 if (homogeneous or self.types[f] == 0) else self.values[f] for f in range(6)]


# ----------------------------------------------------------------------------------------------------
# a-1  face weights from the node SDF
# ----------------------------------------------------------------------------------------------------
def _tri(pa, pb, pd):
    """Area of the corner triangle AEF cut off at corner A with edge neighbours B and D:
    1/2 * phi_A/(phi_A-phi_B) * phi_A/(phi_A-phi_D)      (the printed formula).
    Valid whenever sign(phi_A) differs from sign(phi_B) and sign(phi_D)."""
    return 0.5 * (pa / (pa - pb)) * (pa / (pa - pd))


def area_fraction(pa, pb, pc, pd):
    """Fluid area fraction of a unit square face whose corners, in cyclic order A,B,C,D, carry the SDF
    values pa..pd (phi > 0 in fluid, phi == 0 counts as solid, R1).  Marching-squares contour with linear
    edge crossings ("marching cube ... intersection points between this contour and the
    grid faces"); the one case the paper prints (one fluid corner) is _tri; the others are the same
    construction (R3).  Inputs may be arrays (float or complex: the complex form is used for the
    complex-step derivative in weights_adjoint; case selection always uses the real part)."""
    pa, pb, pc, pd = (np.asarray(x) for x in (pa, pb, pc, pd))
    fa, fb, fc, fd = (x.real > 0 for x in (pa, pb, pc, pd))
    s = fa.astype(int) + fb + fc + fd
    out = np.zeros(np.broadcast(pa, pb, pc, pd).shape, dtype=np.result_type(pa, pb, pc, pd, np.float64))
    P = [np.broadcast_to(x, out.shape) for x in (pa, pb, pc, pd)]
    F = [np.broadcast_to(x, out.shape) for x in (fa, fb, fc, fd)]
    s = np.broadcast_to(s, out.shape)
    out[s == 4] = 1.0
    with np.errstate(divide="ignore", invalid="ignore"):
        for q in range(4):  # corner q with cyclic neighbours q+1 and q-1
            A, B, D, C = P[q], P[(q + 1) % 4], P[(q - 1) % 4], P[(q + 2) % 4]
            # s == 1, fluid corner q: the printed formula
            m = (s == 1) & F[q]
            out[m] = _tri(A[m], B[m], D[m])
            # s == 3, solid corner q: 1 - (solid triangle)
            m = (s == 3) & ~F[q]
            out[m] = 1.0 - _tri(A[m], B[m], D[m])
            # s == 2 adjacent: fluid corners q and q+1; their solid neighbours are q-1 (of q) and q+2 (of q+1)
            m = (s == 2) & F[q] & F[(q + 1) % 4]
            out[m] = 0.5 * (A[m] / (A[m] - D[m]) + B[m] / (B[m] - C[m]))
        # s == 2 diagonal: tie-break on the mean of the four values (R3)
        for q in range(2):
            A, B, C, D = P[q], P[q + 1], P[(q + 2) % 4], P[(q + 3) % 4]
            m = (s == 2) & F[q] & F[(q + 2) % 4]  # fluid at q and q+2, solid at q+1 and q+3
            mean = 0.25 * (A + B + C + D).real
            mj = m & (mean > 0)  # fluid joined: 1 - two solid triangles
            out[mj] = 1.0 - _tri(B[mj], C[mj], A[mj]) - _tri(D[mj], A[mj], C[mj])
            ms = m & ~(mean > 0)  # fluid separated: two fluid triangles
            out[ms] = _tri(A[ms], B[ms], D[ms]) + _tri(C[ms], D[ms], B[ms])
    out[out.real < ALPHA_EPS] = 0.0  # R4
    return out


def face_weights(phi, bc=BC()):
    """alpha for every face of the three families from node SDF phi (nz+1, ny+1, nx+1).
    x-face (i,j,k) has corners at nodes (i, j..j+1, k..k+1) (R2).  Closed-wall domain faces get 0 (R19);
    Dirichlet domain faces keep the SDF-derived value (R22)."""
    phi = np.asarray(phi, dtype=np.float64 if not np.iscomplexobj(phi) else np.complex128)
    # cyclic corner order A,B,C,D around each face
    au = area_fraction(phi[:-1, :-1, :], phi[:-1, 1:, :], phi[1:, 1:, :], phi[1:, :-1, :])
    av = area_fraction(phi[:-1, :, :-1], phi[:-1, :, 1:], phi[1:, :, 1:], phi[1:, :, :-1])
    aw = area_fraction(phi[:, :-1, :-1], phi[:, :-1, 1:], phi[:, 1:, 1:], phi[:, 1:, :-1])
    apply_wall_bc(au, av, aw, bc)
    return au, av, aw


def apply_wall_bc(au, av, aw, bc):
    """Closed-wall domain faces: alpha = 0 (R19)."""
    if bc.types[0] == 0: au[:, :, 0] = 0
    if bc.types[1] == 0: au[:, :, -1] = 0
    if bc.types[2] == 0: av[:, 0, :] = 0
    if bc.types[3] == 0: av[:, -1, :] = 0
    if bc.types[4] == 0: aw[0] = 0
    if bc.types[5] == 0: aw[-1] = 0


def weights_adjoint(phi, gau, gav, gaw, bc=BC()):
    """dJ/dphi at nodes given dJ/dalpha on faces ("back-propagating dJ/dS first through
    the SDF phi").  d alpha/d phi is taken by the complex-step derivative of area_fraction (exact to
    rounding: each case is a rational function; case selection is on the real part)."""
    phi = np.asarray(phi, dtype=np.float64)
    h = 1e-30
    g = np.zeros_like(phi)
    gau, gav, gaw = (np.array(x, dtype=np.float64) for x in (gau, gav, gaw))
    apply_wall_bc(gau, gav, gaw, bc)  # closed-wall faces do not depend on phi
    sl = slice(None)
    fam = [  # (gradient array, the four corner index tuples in the same order as face_weights)
        (gau, [(slice(0, -1), slice(0, -1), sl), (slice(0, -1), slice(1, None), sl),
               (slice(1, None), slice(1, None), sl), (slice(1, None), slice(0, -1), sl)]),
        (gav, [(slice(0, -1), sl, slice(0, -1)), (slice(0, -1), sl, slice(1, None)),
               (slice(1, None), sl, slice(1, None)), (slice(1, None), sl, slice(0, -1))]),
        (gaw, [(sl, slice(0, -1), slice(0, -1)), (sl, slice(0, -1), slice(1, None)),
               (sl, slice(1, None), slice(1, None)), (sl, slice(1, None), slice(0, -1))]),
    ]
    for ga, corners in fam:
        vals = [phi[c] for c in corners]
        for q in range(4):
            pert = [v.astype(np.complex128) for v in vals]
            pert[q] = pert[q] + 1j * h
            dadp = area_fraction(*pert).imag / h
            g[corners[q]] += ga * dadp
    return g


# ----------------------------------------------------------------------------------------------------
# operators G, G^T, A
# ----------------------------------------------------------------------------------------------------
def grad(p, ghost=(0.0,) * 6):
    """G p with ghost values outside the six domain faces (R6)."""
    nz, ny, nx = p.shape
    gu = np.empty((nz, ny, nx + 1)); gv = np.empty((nz, ny + 1, nx)); gw = np.empty((nz + 1, ny, nx))
    gu[:, :, 1:nx] = p[:, :, 1:] - p[:, :, :-1]
    gu[:, :, 0] = p[:, :, 0] - ghost[0]
    gu[:, :, nx] = ghost[1] - p[:, :, nx - 1]
    gv[:, 1:ny, :] = p[:, 1:, :] - p[:, :-1, :]
    gv[:, 0, :] = p[:, 0, :] - ghost[2]
    gv[:, ny, :] = ghost[3] - p[:, ny - 1, :]
    gw[1:nz] = p[1:] - p[:-1]
    gw[0] = p[0] - ghost[4]
    gw[nz] = ghost[5] - p[nz - 1]
    return gu, gv, gw


def grad_T(fu, fv, fw):
    """G^T f (minus the net outflow of a cell)."""
    return (fu[:, :, :-1] - fu[:, :, 1:]) + (fv[:, :-1, :] - fv[:, 1:, :]) + (fw[:-1] - fw[1:])


def apply_A(p, alpha, c):
    """A p = c G^T S G p with homogeneous ghosts."""
    gu, gv, gw = grad(p)
    return c * grad_T(alpha[0] * gu, alpha[1] * gv, alpha[2] * gw)


def diag_A(alpha, c):
    au, av, aw = alpha
    return c * (au[:, :, :-1] + au[:, :, 1:] + av[:, :-1, :] + av[:, 1:, :] + aw[:-1] + aw[1:])


def active_cells(alpha):
    return diag_A(alpha, 1.0) > 0


def is_singular(alpha, bc):
    """True when no Dirichlet domain face carries an open face weight: EVERY fluid component is singular (R12)."""
    au, av, aw = alpha
    planes = [au[:, :, 0], au[:, :, -1], av[:, 0, :], av[:, -1, :], aw[0], aw[-1]]
    return not any(bc.types[f] == 1 and np.any(planes[f] > 0) for f in range(6))


def components(alpha, bc):
    """Fluid components (R12): the connected components of the active cells, two cells being connected when the face
    between them is open (alpha > 0).  Returns (labels, singular): labels[k, j, i] in 1..K on active cells and 0 on
    inactive ones; singular[c] (c = 0..K, entry 0 unused) is True when component c touches no open face of a Dirichlet
    domain boundary -- A restricted to it then has the constant null vector.  The labelling itself is a library
    primitive (scipy.ndimage.label with its default face connectivity) applied to the doubled lattice whose odd sites
    are the cells and whose sites between two cells are the faces; pinned by a brute-force flood fill."""
    from scipy import ndimage
    au, av, aw = (np.asarray(a) for a in alpha)
    nz, ny, nx = au.shape[0], au.shape[1], au.shape[2] - 1
    act = active_cells([au, av, aw])
    lat = np.zeros((2 * nz + 1, 2 * ny + 1, 2 * nx + 1), dtype=bool)
    lat[1::2, 1::2, 1::2] = act
    lat[1::2, 1::2, 2:-1:2] = au[:, :, 1:-1] > 0   # interior faces only: a boundary face connects to no second cell
    lat[1::2, 2:-1:2, 1::2] = av[:, 1:-1, :] > 0
    lat[2:-1:2, 1::2, 1::2] = aw[1:-1] > 0
    lab, _ = ndimage.label(lat)
    cl = lab[1::2, 1::2, 1::2]
    ids = np.unique(cl[act])
    remap = np.zeros(int(lab.max()) + 1, dtype=np.int64)
    remap[ids] = np.arange(1, ids.size + 1)
    labels = np.where(act, remap[cl], 0)
    K = int(ids.size)
    singular = np.ones(K + 1, dtype=bool)
    planes = [(au[:, :, 0], labels[:, :, 0]), (au[:, :, -1], labels[:, :, -1]), (av[:, 0, :], labels[:, 0, :]),
              (av[:, -1, :], labels[:, -1, :]), (aw[0], labels[0]), (aw[-1], labels[-1])]
    for f in range(6):
        if bc.types[f] == 1:
            w, l = planes[f]
            singular[np.unique(l[w > 0])] = False
    singular[0] = False
    return labels, singular


def remove_component_means(x, labels, singular):
    """x minus, on every singular component, its mean over that component (R12: compatibility of b, gauge of p)."""
    K = singular.size - 1
    sums = np.bincount(labels.ravel(), weights=x.ravel(), minlength=K + 1)
    cnt = np.maximum(np.bincount(labels.ravel(), minlength=K + 1), 1)
    mean = np.where(singular, sums / cnt, 0.0)
    return x - mean[labels]


def effective_solid_velocity(us, shapes, bc):
    """U_s with closed-wall faces at rest (R19).  us = None means zero."""
    out = []
    for a, s in zip(us if us is not None else (None, None, None), shapes):
        out.append(np.zeros(s) if a is None else np.array(a, dtype=np.float64))
    if bc.types[0] == 0: out[0][:, :, 0] = 0
    if bc.types[1] == 0: out[0][:, :, -1] = 0
    if bc.types[2] == 0: out[1][:, 0, :] = 0
    if bc.types[3] == 0: out[1][:, -1, :] = 0
    if bc.types[4] == 0: out[2][0] = 0
    if bc.types[5] == 0: out[2][-1] = 0
    return out


def rhs(uhat, alpha, us, c, bc):
    """b = G^T (S Uhat + (I-S) U_s)  (Eq. 4 right-hand side) plus the known Dirichlet ghost
    terms moved from the left-hand side: - c G^T S G(0; ghost = p_D)  (R6)."""
    flux = [a * u + (1.0 - a) * s for a, u, s in zip(alpha, uhat, us)]
    b = grad_T(*flux)
    g0 = grad(np.zeros(b.shape), bc.ghost())
    b -= c * grad_T(alpha[0] * g0[0], alpha[1] * g0[1], alpha[2] * g0[2])
    return b


# ----------------------------------------------------------------------------------------------------
# a-3..a-5 as their plain definition: solve A p = b        (DESIGN.md §4 "definition")
# ----------------------------------------------------------------------------------------------------
def solve(b, alpha, c, bc, tol=1e-12, maxit=200000, info=None):
    """Solve A p = b.  MGPCG is only a fast way to reach this; the oracle uses
    Jacobi-preconditioned CG in fp64 to a relative residual `tol` (R11: ||r||_2 <= tol ||b||_2, x0 = 0).
    Inactive cells (diag 0) get p = 0 and b = 0.  A is block diagonal over the fluid components (R12); on every
    component without an open Dirichlet face the block has the constant null vector: the mean of b over that
    component is removed (compatibility) and the solution has zero mean over it (gauge)."""
    act = active_cells(alpha)
    labels, singc = components(alpha, bc)
    sing = bool(singc.any())
    b = np.where(act, b, 0.0)
    if sing:
        b = remove_component_means(b, labels, singc)
    d = diag_A(alpha, c)
    dinv = np.where(act, 1.0 / np.where(act, d, 1.0), 0.0)
    x = np.zeros_like(b)
    bb = float(np.vdot(b, b))
    it = 0
    if bb > 0:
        r = b.copy()
        z = dinv * r
        p = z.copy()
        rz = float(np.vdot(r, z))
        while it < maxit:
            q = apply_A(p, alpha, c)
            a = rz / float(np.vdot(p, q))
            x += a * p
            r -= a * q
            it += 1
            if float(np.vdot(r, r)) <= tol * tol * bb:
                break
            z = dinv * r
            rz_new = float(np.vdot(r, z))
            p = z + (rz_new / rz) * p
            rz = rz_new
    if sing:
        x = remove_component_means(x, labels, singc)
    if info is not None:
        info["iters"] = it
        info["relres"] = float(np.linalg.norm(b - apply_A(x, alpha, c)) / np.sqrt(bb)) if bb > 0 else 0.0
    return x


def solve_dense(b, alpha, c, bc):
    """Same definition by dense assembly + pseudo-inverse (small grids only; pin for `solve`)."""
    shape = b.shape
    n = b.size
    act = active_cells(alpha)
    Am = np.zeros((n, n))
    e = np.zeros(n)
    for col in range(n):
        e[col] = 1.0
        Am[:, col] = apply_A(e.reshape(shape), alpha, c).ravel()
        e[col] = 0.0
    # the pseudo-inverse IS the per-component definition: it drops the part of b in the null space (the mean over
    # every singular component) and returns the solution orthogonal to the null space (zero mean over each of them)
    bb = np.where(act, b, 0.0)
    x = (np.linalg.pinv(Am, rcond=1e-12, hermitian=True) @ bb.ravel()).reshape(shape)
    return np.where(act, x, 0.0)


# ----------------------------------------------------------------------------------------------------
# a-2, a-6  projection                         PAPER.md:L99-107 (Eqs. 4, 5)
# ----------------------------------------------------------------------------------------------------
def project(uhat, alpha, us, dx, dt_over_rho=1.0, bc=BC(), tol=1e-12, info=None):
    """Returns (U^{n+1}, P).  Eq. 4 solve, then Eq. 5 on open faces; faces with alpha = 0 take the solid
    velocity (R7; closed domain walls are at rest, R19)."""
    c = dt_over_rho / dx
    uhat = [np.asarray(a, dtype=np.float64) for a in uhat]
    alpha = [np.asarray(a, dtype=np.float64) for a in alpha]
    us = effective_solid_velocity(us, [a.shape for a in uhat], bc)
    b = rhs(uhat, alpha, us, c, bc)
    p = solve(b, alpha, c, bc, tol=tol, info=info)
    gp = grad(p, bc.ghost())
    unew = [np.where(a > 0, u - c * g, s) for a, u, g, s in zip(alpha, uhat, gp, us)]
    return unew, p


def weighted_divergence(u, alpha, us, bc):
    """G^T (S U + (I-S) U_s): zero after projection (follows from Eqs. 4-5)."""
    us = effective_solid_velocity(us, [a.shape for a in u], bc)
    return grad_T(*[a * x + (1.0 - a) * s for a, x, s in zip(alpha, u, us)])


# ----------------------------------------------------------------------------------------------------
# a-7  adjoint projection                      PAPER.md:L115-124 (Eqs. 6, 7), L134-139 (Eq. 9)
# ----------------------------------------------------------------------------------------------------
def project_adjoint(g, alpha, p_saved, uhat, us, dx, dt_over_rho=1.0, bc=BC(), tol=1e-12, info=None):
    """Given g = dJ/dU^{n+1}: returns (dJ/dUhat, dJ/dalpha, dJ/dU_s, y).
    Eq. 6 (column form, R8): dJ/dP = -c G^T (M g), M = [alpha > 0] (R7).
    A y = dJ/dP with the same A.
    Eq. 7: dJ/dUhat = M g + S G y.
    Eq. 9a with the derived minus sign (R9): dJ/dalpha_f = (G y)_f [ (Uhat - U_s)_f - c (G p)_f ].
    Eq. 9b in the derived form (R10): dJ/dU_s = (I - M) g + (I - S) G y; zero on closed walls (R19)."""
    c = dt_over_rho / dx
    g = [np.asarray(a, dtype=np.float64) for a in g]
    alpha = [np.asarray(a, dtype=np.float64) for a in alpha]
    uhat = [np.asarray(a, dtype=np.float64) for a in uhat]
    us = effective_solid_velocity(us, [a.shape for a in g], bc)
    Mg = [np.where(a > 0, x, 0.0) for a, x in zip(alpha, g)]
    gp_rhs = -c * grad_T(*Mg)
    y = solve(gp_rhs, alpha, c, bc, tol=tol, info=info)
    Gy = grad(y)  # homogeneous ghosts: the ghost pressure is data, not an unknown
    Gp = grad(np.asarray(p_saved, dtype=np.float64), bc.ghost())
    g_uhat = [m + a * gy for m, a, gy in zip(Mg, alpha, Gy)]
    g_alpha = [gy * ((u - s) - c * gp) for gy, u, s, gp in zip(Gy, uhat, us, Gp)]
    g_us = [(x - m) + (1.0 - a) * gy for x, m, a, gy in zip(g, Mg, alpha, Gy)]
    apply_wall_mask(g_us, g_alpha, bc)
    return g_uhat, g_alpha, g_us, y


def apply_wall_mask(g_us, g_alpha, bc):
    """Closed-wall faces: alpha is forced to 0 and the wall is at rest, so neither depends on the
    caller's arrays there (R19)."""
    for arrs in (g_us, g_alpha):
        if bc.types[0] == 0: arrs[0][:, :, 0] = 0
        if bc.types[1] == 0: arrs[0][:, :, -1] = 0
        if bc.types[2] == 0: arrs[1][:, 0, :] = 0
        if bc.types[3] == 0: arrs[1][:, -1, :] = 0
        if bc.types[4] == 0: arrs[2][0] = 0
        if bc.types[5] == 0: arrs[2][-1] = 0


# ----------------------------------------------------------------------------------------------------
# a-8, a-9  semi-Lagrangian advection and its adjoint     PAPER.md:L80-82 (Eq. 2), L353-357 (Eqs. 11-12)
# ----------------------------------------------------------------------------------------------------
_OFFS = [(0.0, 0.5, 0.5), (0.5, 0.0, 0.5), (0.5, 0.5, 0.0)]  # position of component c's samples in a cell


def _locate(f, comp, pos):
    """Lattice coordinates of component `comp` at positions pos (cell units), clamped to the lattice
    (R14).  Returns base indices, fractions, and the mask of un-clamped axes."""
    idx, frac, free = [], [], []
    for d in range(3):  # d = 0,1,2 -> x,y,z ; array axis = 2-d
        n = f.shape[2 - d]
        t = pos[d] - _OFFS[comp][d]
        tc = np.clip(t, 0.0, n - 1.0)
        i0 = np.minimum(np.floor(tc).astype(np.int64), n - 2) if n > 1 else np.zeros(tc.shape, np.int64)
        idx.append(i0)
        frac.append(tc - i0)
        free.append((t >= 0.0) & (t <= n - 1.0))
    return idx, frac, free


def interp(f, comp, pos):
    """Trilinear interpolation of staggered component `comp` (array f) at pos = (x, y, z) in cell units."""
    (ix, iy, iz), (fx, fy, fz), _ = _locate(f, comp, pos)
    out = 0.0
    for dz in (0, 1):
        for dy in (0, 1):
            for dx_ in (0, 1):
                wgt = (fx if dx_ else 1 - fx) * (fy if dy else 1 - fy) * (fz if dz else 1 - fz)
                out = out + wgt * f[np.minimum(iz + dz, f.shape[0] - 1), np.minimum(iy + dy, f.shape[1] - 1),
                                    np.minimum(ix + dx_, f.shape[2] - 1)]
    return out


def _face_positions(shape, comp):
    k, j, i = np.meshgrid(*(np.arange(s, dtype=np.float64) for s in shape), indexing="ij")
    o = _OFFS[comp]
    return [i + o[0], j + o[1], k + o[2]]


def advect(U, dt, dx):
    """Two-stage back-trace evaluated pointwise at every face (R20):
    v0 = U^n(x); x_m = x - 1/2 dt v0 (Eq. 11); v_m = U^n(x_m); x_b = x - dt v_m (Eq. 12);
    out_c(x) = U^n_c(x_b).  Positions in cell units, hence dt/dx."""
    U = [np.asarray(a, dtype=np.float64) for a in U]
    s = dt / dx
    out = []
    for comp in range(3):
        x = _face_positions(U[comp].shape, comp)
        v0 = [interp(U[d], d, x) for d in range(3)]
        xm = [x[d] - 0.5 * s * v0[d] for d in range(3)]
        vm = [interp(U[d], d, xm) for d in range(3)]
        xb = [x[d] - s * vm[d] for d in range(3)]
        out.append(interp(U[comp], comp, xb))
    return out


def _interp_adjoint(f, comp, pos, gbar, gf):
    """Reverse of `interp`: scatters gbar * weight into gf and returns d(out)/d(pos) * gbar per axis
    (zero on clamped axes)."""
    (ix, iy, iz), (fx, fy, fz), free = _locate(f, comp, pos)
    gpos = [0.0, 0.0, 0.0]
    sh = f.shape
    for dz in (0, 1):
        for dy in (0, 1):
            for dx_ in (0, 1):
                wx, wy, wz = (fx if dx_ else 1 - fx), (fy if dy else 1 - fy), (fz if dz else 1 - fz)
                kk, jj, ii = np.minimum(iz + dz, sh[0] - 1), np.minimum(iy + dy, sh[1] - 1), np.minimum(ix + dx_, sh[2] - 1)
                np.add.at(gf, (kk, jj, ii), gbar * wx * wy * wz)
                val = f[kk, jj, ii]
                gpos[0] = gpos[0] + gbar * val * (1 if dx_ else -1) * wy * wz
                gpos[1] = gpos[1] + gbar * val * wx * (1 if dy else -1) * wz
                gpos[2] = gpos[2] + gbar * val * wx * wy * (1 if dz else -1)
    return [np.where(free[d], gpos[d], 0.0) for d in range(3)]


def advect_adjoint(U, gout, dt, dx):
    """dJ/dU^n given dJ/dUtilde (Eq. 8: (dB/dU^n U^n + B(U^n))^T applied to the
    incoming gradient), as the hand-written reverse of `advect`."""
    U = [np.asarray(a, dtype=np.float64) for a in U]
    gout = [np.asarray(a, dtype=np.float64) for a in gout]
    s = dt / dx
    gU = [np.zeros_like(a) for a in U]
    for comp in range(3):
        x = _face_positions(U[comp].shape, comp)
        v0 = [interp(U[d], d, x) for d in range(3)]
        xm = [x[d] - 0.5 * s * v0[d] for d in range(3)]
        vm = [interp(U[d], d, xm) for d in range(3)]
        xb = [x[d] - s * vm[d] for d in range(3)]
        gxb = _interp_adjoint(U[comp], comp, xb, gout[comp], gU[comp])
        gvm = [-s * gxb[d] for d in range(3)]
        gxm = [0.0, 0.0, 0.0]
        for d in range(3):
            t = _interp_adjoint(U[d], d, xm, gvm[d], gU[d])
            gxm = [gxm[e] + t[e] for e in range(3)]
        gv0 = [-0.5 * s * gxm[d] for d in range(3)]
        for d in range(3):
            _interp_adjoint(U[d], d, x, gv0[d], gU[d])
    return gU


# ----------------------------------------------------------------------------------------------------
# viscosity         PAPER.md:L84-87 (Eq. 3), L359-361 (Eq. 13), L126-128 (Eq. 8)
# ----------------------------------------------------------------------------------------------------
def viscosity(U, nu, dt, dx):
    """Eq. 3: Uhat = (I - nu dt/dx^2 G^T G) Utilde, "for each axis, the Laplacian of the corresponding velocity
    component ... on grid points": per component, the 7-point operator G^T G of that component's own lattice, G
    = forward differences between lattice neighbours with nothing outside the lattice (reading R23: the paper is
    silent on the boundary rows; this is the form that keeps G^T G symmetric, which Eq. 8 relies on when it applies
    the same matrix in the backward pass).  Every face is updated (closed ones are overwritten by the projection,
    as with advection, R14).  Self-adjoint: the backward pass calls this same function on dJ/dUhat (Eq. 8)."""
    k = nu * dt / (dx * dx)
    out = []
    for f in U:
        f = np.asarray(f, dtype=np.float64)
        gtg = np.zeros_like(f)
        for ax in range(3):
            if f.shape[ax] < 2:
                continue
            d = np.diff(f, axis=ax)                     # G along this axis: f[i+1] - f[i]
            lo = [slice(None)] * 3; hi = [slice(None)] * 3
            lo[ax] = slice(0, -1); hi[ax] = slice(1, None)
            gtg[tuple(lo)] -= d                          # G^T: -d at the lower point, +d at the upper
            gtg[tuple(hi)] += d
        out.append(f - k * gtg)
    return out


def max_speed(U):
    """max over all faces of |u|, |v|, |w| -- the quantity of the CFL condition (R24)."""
    return max(float(np.max(np.abs(np.asarray(a, dtype=np.float64)))) for a in U)


# ----------------------------------------------------------------------------------------------------
# full steps forward and backward        PAPER.md:L78 (advection, projection), L111-141 (backward pass)
# ----------------------------------------------------------------------------------------------------
def rollout(U0, solid_fn, nsteps, dt, dx, dt_over_rho, bc, loss_fn, tol=1e-12, advect_on=True, nu=0.0):
    """N steps "advect -> geometry at t^{n+1} -> project" (R15) and the backward pass that "mirrors the
    forward simulation in a reversed order", per-step state stored instead of a graph (L236).

    solid_fn(step) -> (phi, us, dphi_dtheta, dus_dtheta) for step = 1..N, one scalar parameter theta;
    loss_fn(U) -> (J, dJ/dU) on the final velocity.
    Returns (J, dJ/dtheta, dJ/dU0).  dJ/dtheta = sum_n <dJ/dphi^n, dphi^n/dtheta> + <dJ/dU_s^n, dU_s^n/dtheta>
    with dJ/dphi from dJ/dS (Eq. 9a) through the weight builder (L141) and dJ/dU_s from Eq. 9b (R9, R10)."""
    U = [np.asarray(a, dtype=np.float64) for a in U0]
    tape = []
    for n in range(1, nsteps + 1):
        Uprev = U
        Ut = advect(U, dt, dx) if advect_on else [a.copy() for a in U]
        if nu != 0.0:
            Ut = viscosity(Ut, nu, dt, dx)               # L78: advection, viscosity, projection
        phi, us, dphi, dus = solid_fn(n)
        alpha = face_weights(phi, bc)
        U, p = project(Ut, alpha, us, dx, dt_over_rho, bc, tol=tol)
        tape.append((Uprev, Ut, phi, us, dphi, dus, alpha, p))
    J, g = loss_fn(U)
    g = [np.asarray(a, dtype=np.float64) for a in g]
    dtheta = 0.0
    for n in range(nsteps, 0, -1):
        Uprev, Ut, phi, us, dphi, dus, alpha, p = tape[n - 1]
        g_ut, g_alpha, g_us, _ = project_adjoint(g, alpha, p, Ut, us, dx, dt_over_rho, bc, tol=tol)
        g_phi = weights_adjoint(phi, g_alpha[0], g_alpha[1], g_alpha[2], bc)
        dtheta += float(np.sum(g_phi * dphi)) + sum(float(np.sum(a * b)) for a, b in zip(g_us, dus))
        if nu != 0.0:
            g_ut = viscosity(g_ut, nu, dt, dx)           # Eq. 8: the same symmetric matrix
        g = advect_adjoint(Uprev, g_ut, dt, dx) if advect_on else g_ut
    return J, dtheta, g


def loss_sum_u2(lo, hi):
    """BASELINE.json configs[1]: J = sum of u^2 over the u-faces with i, j, k in [lo, hi)."""
    def fn(U):
        g = [np.zeros_like(np.asarray(a, dtype=np.float64)) for a in U]
        blk = np.asarray(U[0], dtype=np.float64)[lo:hi, lo:hi, lo:hi]
        g[0][lo:hi, lo:hi, lo:hi] = 2.0 * blk
        return float(np.sum(blk * blk)), g
    return fn


def cfl_dt(U, t_left, dx, cfl, max_substeps=64):
    """Sub-step size under the CFL condition the paper says it adopts ("adopts CFL condition", L403-410
    Table 4: the steps simulated exceed the frames; no constant or formula is given -- reading R24): the remaining
    frame time t_left is cut into n equal sub-steps, n the smallest integer with dt = t_left / n <= cfl dx / max|U|
    (at most max_substeps); re-evaluated after every sub-step because the velocity changes."""
    vmax = max_speed(U)
    if not (vmax > 0.0) or not np.isfinite(vmax):
        return t_left
    n = max(1, min(max_substeps, int(np.ceil(t_left * vmax / (cfl * dx) - 1e-9))))
    return t_left / n


def rollout_substepped(U0, solid_fn_t, nframes, dt_frame, dx, rho, bc, loss_fn, cfl=1.0, dts=None, tol=1e-12,
                       advect_on=True, nu=0.0, max_substeps=64):
    """N frames of length dt_frame, each advanced by CFL sub-steps (cfl_dt, R24): per sub-step of size dt
    "advect -> viscosity -> geometry at the sub-step's end time -> project" with dt/rho in Eqs. 4-5 (PAPER.md:L78, L103,
    L151), and the backward pass in reversed order over the SUB-steps (L111); dt is a constant of the backward pass
    (R24: the sub-step sizes are not differentiated).

    solid_fn_t(t) -> (phi, us, dphi_dtheta, dus_dtheta) at physical time t; loss_fn(U) -> (J, dJ/dU).
    dts: replay these sub-step sizes (a list of lists, one per frame) instead of choosing them -- what a
    finite-difference check of the gradient needs, and what the CUDA path is compared on.
    Returns (J, dJ/dtheta, dJ/dU0, dts_used)."""
    U = [np.asarray(a, dtype=np.float64) for a in U0]
    tape, used = [], []
    for f in range(nframes):
        t, t_end = f * dt_frame, (f + 1) * dt_frame
        frame_dts = []
        k = 0
        while t_end - t > 1e-12 * dt_frame:
            dt = dts[f][k] if dts is not None else cfl_dt(U, t_end - t, dx, cfl, max_substeps)
            Uprev = U
            Ut = advect(U, dt, dx) if advect_on else [a.copy() for a in U]
            if nu != 0.0:
                Ut = viscosity(Ut, nu, dt, dx)
            t = t + dt
            phi, us, dphi, dus = solid_fn_t(t)
            alpha = face_weights(phi, bc)
            U, p = project(Ut, alpha, us, dx, dt / rho, bc, tol=tol)
            tape.append((Uprev, Ut, phi, us, dphi, dus, alpha, p, dt))
            frame_dts.append(dt)
            k += 1
            if dts is not None and k >= len(dts[f]):
                break
        used.append(frame_dts)
    J, g = loss_fn(U)
    g = [np.asarray(a, dtype=np.float64) for a in g]
    dtheta = 0.0
    for Uprev, Ut, phi, us, dphi, dus, alpha, p, dt in reversed(tape):
        g_ut, g_alpha, g_us, _ = project_adjoint(g, alpha, p, Ut, us, dx, dt / rho, bc, tol=tol)
        g_phi = weights_adjoint(phi, g_alpha[0], g_alpha[1], g_alpha[2], bc)
        dtheta += float(np.sum(g_phi * dphi)) + sum(float(np.sum(a * b)) for a, b in zip(g_us, dus))
        if nu != 0.0:
            g_ut = viscosity(g_ut, nu, dt, dx)
        g = advect_adjoint(Uprev, g_ut, dt, dx) if advect_on else g_ut
    return J, dtheta, g, used
