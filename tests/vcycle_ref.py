"""Test helper: the library's multigrid V-cycle preconditioner z = M^{-1} r written out in plain NumPy fp64.

NOT the oracle (the paper defines the projection's RESULT, not the preconditioner: every multigrid parameter is this
library's own choice, DESIGN.md section 6 / R13) -- a slow third implementation of that documented choice, used to
check the CUDA V-cycle kernels (fused 4-launch levels, cooperative coarse kernel with its packed per-cell phases,
shared-memory tail) against something that carries no fp32 rounding: V(nu, nu) with nu chosen per level (the finest
level, level 1, every level below: 1, 1, 1 by default -- the library's choice for grids below 3 M cells; 1, 2, 3
from there on), red-black Gauss-Seidel (pre: red then black, the first sweep from a zero
guess; post: black then red), piecewise-constant prolongation P, restriction P^T / 8,
rediscretised coarse operators with c_l = c / 4^l on weights that are the mean of the four coincident fine face
weights (absent fine faces of an odd edge count as closed), extents halving -- rounding up -- while they stay >= 4
(>= 2 while the level has more than 128 cells), coarsest level (<= 128 cells): exact solve (the
pseudo-inverse in the complement of the constant on singular systems); a larger coarsest level: 2 * (largest extent)
symmetric sweeps (red-black from zero, then black-red).
3-D grids only."""
import numpy as np


def _coarsen(a):
    """Coarse face weights in float32 with the library's summation order (so both hierarchies hold identical numbers).
    Extents halve rounding up: fine faces beyond an odd extent do not exist and count as closed, and the coarse
    boundary face of an odd axis coincides with the fine boundary face."""
    au, av, aw = [x.astype(np.float32) for x in a]
    nz, ny, nx = au.shape[0], au.shape[1], au.shape[2] - 1
    ez, ey, ex = nz + (nz & 1), ny + (ny & 1), nx + (nx & 1)
    q = np.float32(0.25)
    xi = list(range(0, nx, 2)) + [nx]   # fine x-faces under the coarse ones (the last one: the boundary face)
    yi = list(range(0, ny, 2)) + [ny]
    zi = list(range(0, nz, 2)) + [nz]
    pu = np.zeros((ez, ey, nx + 1), np.float32); pu[:nz, :ny] = au
    pu = pu[:, :, xi]
    cu = q * ((pu[0::2, 0::2] + pu[0::2, 1::2]) + (pu[1::2, 0::2] + pu[1::2, 1::2]))
    pv = np.zeros((ez, ny + 1, ex), np.float32); pv[:nz, :, :nx] = av
    pv = pv[:, yi, :]
    cv = q * ((pv[0::2, :, 0::2] + pv[0::2, :, 1::2]) + (pv[1::2, :, 0::2] + pv[1::2, :, 1::2]))
    pw = np.zeros((nz + 1, ey, ex), np.float32); pw[:, :ny, :nx] = aw
    pw = pw[zi]
    cw = q * ((pw[:, 0::2, 0::2] + pw[:, 0::2, 1::2]) + (pw[:, 1::2, 0::2] + pw[:, 1::2, 1::2]))
    return [cu, cv, cw]


def hierarchy(alpha):
    """[fine, ..., coarsest] face-weight triples (float32), by the library's halving rule."""
    lv = [[np.asarray(x, dtype=np.float32) for x in alpha]]
    while True:
        nz, ny, nx = lv[-1][0].shape[0], lv[-1][0].shape[1], lv[-1][0].shape[2] - 1
        lim = 2 if nx * ny * nz > 128 else 4
        h = [(nx + 1) // 2, (ny + 1) // 2, (nz + 1) // 2]
        if min(h) < lim or h == [nx, ny, nz]:
            break
        lv.append(_coarsen(lv[-1]))
    return lv


def _nbsum(z, a):
    au, av, aw = a
    s = np.zeros_like(z)
    s[:, :, 1:] += au[:, :, 1:-1] * z[:, :, :-1]
    s[:, :, :-1] += au[:, :, 1:-1] * z[:, :, 1:]
    s[:, 1:, :] += av[:, 1:-1, :] * z[:, :-1, :]
    s[:, :-1, :] += av[:, 1:-1, :] * z[:, 1:, :]
    s[1:] += aw[1:-1] * z[:-1]
    s[:-1] += aw[1:-1] * z[1:]
    return s


def _diag(a):
    au, av, aw = a
    return au[:, :, :-1] + au[:, :, 1:] + av[:, :-1, :] + av[:, 1:, :] + aw[:-1] + aw[1:]


def vcycle(r, alpha, c, singular, nu_fine=1, nu_l1=1, nu_deep=1, omega_deep=1.4):
    """nu_fine / nu_l1 / nu_deep: red-black sweeps before and after the coarse correction on the finest level / on
    level 1 / on every level below that (the library's defaults: nf_set_solver_options, nf_set_coarse_sweeps);
    omega_deep: over-relaxation factor of the sweeps on every level below the finest (nf_set_coarse_relaxation)."""
    levels = [[x.astype(np.float64) for x in a] for a in hierarchy(alpha)]

    def rec(l, r, c):
        a = levels[l]
        d = c * _diag(a)
        act = d > 0
        dinv = np.where(act, 1.0 / np.where(act, d, 1.0), 0.0)
        nz, ny, nx = r.shape
        k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij", sparse=True)
        red = ((i + j + k) & 1) == 0
        z = np.zeros_like(r)

        om = omega_deep if l >= 1 else 1.0   # over-relaxation of the sweeps on every level below the finest (SOR)

        def half(mask):
            zn = (1.0 - om) * z + om * (r + c * _nbsum(z, a)) * dinv
            z[mask & act] = zn[mask & act]
            z[mask & ~act] = 0.0

        if l == len(levels) - 1:
            if singular:
                r = np.where(act, r - r[act].sum() / max(int(act.sum()), 1), r)
            if r.size <= 128:  # direct solve with the (pseudo-)inverse of the coarsest operator on the active cells
                n = r.size
                A = np.zeros((n, n))
                for col in range(n):
                    e = np.zeros(n); e[col] = 1.0
                    e3 = e.reshape(r.shape)
                    A[:, col] = (d * e3 - c * _nbsum(e3, a)).ravel()
                ia = np.flatnonzero(act.ravel())
                sol = np.zeros(n)
                if ia.size:
                    sol[ia] = np.linalg.pinv(A[np.ix_(ia, ia)], hermitian=True) @ r.ravel()[ia] if singular else \
                        np.linalg.solve(A[np.ix_(ia, ia)], r.ravel()[ia])
                z = sol.reshape(r.shape)
            else:
                sweeps = 2 * max(nx, ny, nz)
                for _ in range(sweeps):
                    half(red); half(~red)
                for _ in range(sweeps):
                    half(~red); half(red)
            if singular:
                z = np.where(act, z - z[act].sum() / max(int(act.sum()), 1), z)
            return z
        nu = nu_fine if l == 0 else (nu_l1 if l == 1 else nu_deep)
        for _ in range(nu):
            half(red); half(~red)
        res = np.where(act, r - (d * z - c * _nbsum(z, a)), 0.0)
        ez, ey, ex = nz + (nz & 1), ny + (ny & 1), nx + (nx & 1)
        rp = np.zeros((ez, ey, ex)); rp[:nz, :ny, :nx] = res          # (absent children of an odd edge contribute 0)
        rc = 0.125 * rp.reshape(ez // 2, 2, ey // 2, 2, ex // 2, 2).sum(axis=(1, 3, 5))
        zc = rec(l + 1, rc, 0.25 * c)
        z += np.repeat(np.repeat(np.repeat(zc, 2, axis=0), 2, axis=1), 2, axis=2)[:nz, :ny, :nx]
        for _ in range(nu):
            half(~red); half(red)
        return z

    return rec(0, np.asarray(r, dtype=np.float64), float(c))
