"""Test helper: the library's multigrid V-cycle preconditioner z = M^{-1} r written out in plain NumPy fp64.

NOT the oracle (the paper defines the projection's RESULT, not the preconditioner: every multigrid parameter is this
library's own choice, DESIGN.md section 6 / R13) -- a slow third implementation of that documented choice, used to
check the CUDA V-cycle kernels (fused 4-launch levels, cooperative coarse kernel with its packed per-cell phases,
shared-memory tail) against something that carries no fp32 rounding: V(1,1), red-black Gauss-Seidel (pre: red then
black from a zero guess; post: black then red), piecewise-constant prolongation P, restriction P^T / 8,
rediscretised coarse operators with c_l = c / 4^l on weights that are the mean of the four coincident fine face
weights, levels halving while every extent is even and stays >= 4 (>= 2 while the level has more than 128 cells), coarsest level (<= 128 cells): exact solve (the
pseudo-inverse in the complement of the constant on singular systems); a larger coarsest level: 2 * (largest extent)
symmetric sweeps (red-black from zero, then black-red).
3-D grids only."""
import numpy as np


def _coarsen(a):
    """Coarse face weights in float32 with the library's summation order (so both hierarchies hold identical numbers)."""
    au, av, aw = [x.astype(np.float32) for x in a]
    q = np.float32(0.25)
    cu = q * ((au[0::2, 0::2, 0::2] + au[0::2, 1::2, 0::2]) + (au[1::2, 0::2, 0::2] + au[1::2, 1::2, 0::2]))
    cv = q * ((av[0::2, 0::2, 0::2] + av[0::2, 0::2, 1::2]) + (av[1::2, 0::2, 0::2] + av[1::2, 0::2, 1::2]))
    cw = q * ((aw[0::2, 0::2, 0::2] + aw[0::2, 0::2, 1::2]) + (aw[0::2, 1::2, 0::2] + aw[0::2, 1::2, 1::2]))
    return [cu, cv, cw]


def hierarchy(alpha):
    """[fine, ..., coarsest] face-weight triples (float32), by the library's halving rule."""
    lv = [[np.asarray(x, dtype=np.float32) for x in alpha]]
    while True:
        nz, ny, nx = lv[-1][0].shape[0], lv[-1][0].shape[1], lv[-1][0].shape[2] - 1
        if (nx | ny | nz) & 1 or min(nx, ny, nz) // 2 < (2 if nx * ny * nz > 128 else 4):
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


def vcycle(r, alpha, c, singular):
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

        def half(mask):
            zn = (r + c * _nbsum(z, a)) * dinv
            z[mask] = zn[mask]

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
        half(red); half(~red)
        res = np.where(act, r - (d * z - c * _nbsum(z, a)), 0.0)
        rc = 0.125 * res.reshape(nz // 2, 2, ny // 2, 2, nx // 2, 2).sum(axis=(1, 3, 5))
        zc = rec(l + 1, rc, 0.25 * c)
        z += np.repeat(np.repeat(np.repeat(zc, 2, axis=0), 2, axis=1), 2, axis=2)
        half(~red); half(red)
        return z

    return rec(0, np.asarray(r, dtype=np.float64), float(c))
