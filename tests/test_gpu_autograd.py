"""torch.autograd wrappers (paper_2405_14903_b200/autograd.py) against the fp64 oracle: a simulation written as plain
torch code back-propagates through the library's adjoints to the initial velocity, the shape parameters and a scalar
that scales the solid velocity; north_star's tolerances (1e-4 loss, 1e-3 gradients)."""
import numpy as np
import pytest

from oracle import nf_geom_oracle as G
from oracle import nf_oracle as orc
from paper_2405_14903_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


@pytest.fixture(scope="module")
def api():
    from paper_2405_14903_b200 import api as a
    a.load_library()
    return a


def make_grid(api, n, dx, bc_t, bc_v):
    g = api.Grid(n, n, n, dx)
    for f in range(6):
        g.set_domain_bc(f, bc_t[f], bc_v[f])
    return g


def test_shape_gradient_through_autograd_matches_oracle(torch, api):
    from paper_2405_14903_b200 import autograd as ag
    n, dx, nsteps = 20, float(np.float32(1.0 / 20)), 2
    dt = 0.4 * dx
    bc_t, bc_v = (1, 1, 0, 0, 0, 0), (1.0, 0.0, 0, 0, 0, 0)
    K, N, M = 2, 4, 8
    p0 = wl.geom_random_params(61, K, N, 0.2, 0.8, (0.5, 0.5), 0.2)
    rng = np.random.default_rng(9)
    U0 = [(0.2 * rng.standard_normal(s)).astype(np.float32) for s in wl.face_shapes(n, n, n)]
    g = make_grid(api, n, dx, bc_t, bc_v)
    params = torch.tensor(p0, dtype=torch.float64, requires_grad=True)           # a CPU leaf, like an optimiser's
    U = [torch.from_numpy(a).cuda().requires_grad_(True) for a in U0]
    cur = U
    for _ in range(nsteps):
        cur = ag.advect(g, *cur, dt)
        phi = ag.geom_sdf(g, params, K, N, M)
        cur = ag.project(g, *cur, phi, tol=1e-7, maxit=400)[:3]
    J = 0.5 * sum((a.double() ** 2).sum() for a in cur)
    J.backward()

    def loss_ref(V):
        return 0.5 * sum(float(np.sum(a * a)) for a in V), [a.copy() for a in V]
    Jr, gr, gU0r = G.rollout_parametric(U0, lambda s: [(p0.astype(np.float64), None, K, N, M)], nsteps, dt, dx, 1.0,
                                        orc.BC(bc_t, bc_v), loss_ref)
    gp = sum(s[0][0] for s in gr)
    assert abs(float(J.detach()) - Jr) < 1e-4 * Jr
    assert params.grad.dtype == torch.float64 and params.grad.device.type == "cpu"
    assert np.max(np.abs(params.grad.numpy() - gp)) < 1e-3 * np.max(np.abs(gp))
    num = np.sqrt(sum(float(((a.grad.cpu().numpy() - b) ** 2).sum()) for a, b in zip(U, gU0r)))
    assert num < 1e-3 * np.sqrt(sum(float((b ** 2).sum()) for b in gU0r))
    g.close()


def test_control_gradient_with_viscosity_through_autograd_matches_oracle(torch, api):
    """U_s = theta * basis built with torch ops from a CUDA scalar; advect -> viscosity -> project for 2 steps."""
    from paper_2405_14903_b200 import autograd as ag
    n, dx, nsteps, nu = 16, float(np.float32(1.0 / 16)), 2, 0.02
    dt = 0.5 * dx
    bc_t, bc_v = (1, 1, 0, 0, 0, 0), (0.5, 0.0, 0, 0, 0, 0)
    bc = orc.BC(bc_t, bc_v)
    i, j, k = wl.node_coords(n, n, n)
    phi = wl.sdf_sphere(i, j, k, (8.3, 7.6, 8.1), 4.2).astype(np.float32)
    rng = np.random.default_rng(10)
    basis = [rng.standard_normal(s).astype(np.float32) for s in wl.face_shapes(n, n, n)]
    U0 = [(0.2 * rng.standard_normal(s)).astype(np.float32) for s in wl.face_shapes(n, n, n)]
    theta0 = 0.3
    g = make_grid(api, n, dx, bc_t, bc_v)
    theta = torch.tensor(theta0, dtype=torch.float32, device="cuda", requires_grad=True)
    B = [torch.from_numpy(a).cuda() for a in basis]
    phid = torch.from_numpy(phi).cuda()
    cur = [torch.from_numpy(a).cuda() for a in U0]
    for _ in range(nsteps):
        cur = ag.advect(g, *cur, dt)
        cur = ag.viscosity(g, *cur, nu, dt)
        cur = ag.project(g, *cur, phid, *[theta * b for b in B], tol=1e-7, maxit=400)[:3]
    J = 0.5 * sum((a.double() ** 2).sum() for a in cur)
    J.backward()

    def loss_ref(V):
        return 0.5 * sum(float(np.sum(a * a)) for a in V), [a.copy() for a in V]
    us64 = [np.float32(theta0) * b for b in basis]          # fp32 product, like the device's theta * basis
    Jr, dth, _ = orc.rollout(U0, lambda s: (phi, us64, np.zeros_like(phi, dtype=np.float64), basis), nsteps, dt, dx, 1.0,
                             bc, loss_ref, nu=nu)
    assert abs(float(J.detach()) - Jr) < 1e-4 * Jr
    assert abs(float(theta.grad) - dth) < 1e-3 * abs(dth)
    g.close()
