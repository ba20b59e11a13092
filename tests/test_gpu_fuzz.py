"""Robustness sweep of the solver: seeded random blob fields (1 .. 80 solid spheres: open domains, pockets, several
singular components), random Dirichlet / closed domain faces (every third case all closed), grid shapes from 32^3 to
192^3 incl. odd hierarchies, flat boxes and 2-D mode, velocities over four decades, default sweeps / V(1,1) / (2,3):
forward and adjoint projection must converge to 1e-6 in at most 60 iterations with finite results.  (No oracle here:
parity is tests/test_gpu_parity*.py's job; this guards the iteration-level machinery -- look-ahead, in-flight residual
replacement and its rejection, residual compatibility on singular systems, per-component gauges -- against stalls.)"""
import warnings

import numpy as np
import pytest

from paper_2405_14903_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SHAPES = [(32, 32, 32), (48, 40, 36), (64, 64, 64), (96, 64, 48), (100, 100, 100), (128, 128, 128), (160, 160, 160),
          (72, 90, 54), (256, 128, 64), (192, 192, 192), (50, 30, 22), (256, 192, 1), (120, 120, 120)]


def _blob_sdf(nx, ny, nz, seed, nblobs):
    rng = np.random.default_rng(seed)
    x, y, z = wl.node_coords(nx, ny, nz)
    phi = np.full((nz + 1, ny + 1, nx + 1), 1e9)
    for _ in range(nblobs):
        c = rng.uniform(0.15, 0.85, 3) * np.array([nx, ny, nz])
        r = rng.uniform(0.06, 0.2) * min(nx, ny, max(nz, 8))
        phi = np.minimum(phi, np.sqrt((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2) - r)
    return phi.astype(np.float32)


def test_random_geometries_converge_at_every_sweep_setting():
    import torch
    from paper_2405_14903_b200 import api
    api.load_library()
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    rng = np.random.default_rng(123)
    torch.manual_seed(5)
    bad = []
    for case in range(39):
        nx, ny, nz = SHAPES[case % len(SHAPES)]
        bt = tuple(int(v) for v in (rng.random(6) < (0.3 if case % 3 else 0.0)))
        if nz == 1:
            bt = bt[:4] + (0, 0)
        g = api.Grid(nx, ny, nz, 1.0 / nx)
        g.set_dt_rho(float(rng.uniform(0.2, 2.0)))
        for f in range(6):
            g.set_domain_bc(f, bt[f], float(rng.normal()) if bt[f] else 0.0)
        g.set_solid(d(_blob_sdf(nx, ny, nz, 1000 + case, int(rng.integers(1, 80)))))
        for nu in (None, (1, 1), (2, 3)):
            if nu:
                g.set_coarse_sweeps(*nu)
            scale = float(10 ** rng.uniform(-2, 2))
            U = [torch.randn(s, device="cuda") * scale for s in (g.shape_u, g.shape_v, g.shape_w)]
            p = torch.zeros(g.shape_p, device="cuda")
            with warnings.catch_warnings():
                warnings.simplefilter("ignore")
                rc = g.project(*U, p, tol=1e-6, maxit=200)
                fi = g.last_solve_info()
                G = [torch.randn_like(a) for a in U]
                rc2 = g.project_adjoint(*G, tol=1e-6, maxit=200)
                ai = g.last_solve_info()
            ok = rc == 0 and rc2 == 0 and fi["iters"] <= 60 and ai["iters"] <= 60 and bool(torch.isfinite(p).all()) \
                and all(bool(torch.isfinite(a).all()) for a in U + G)
            if not ok:
                bad.append((case, (nx, ny, nz), bt, g.components(), nu, rc, fi, rc2, ai))
        g.close()
    assert not bad, bad
