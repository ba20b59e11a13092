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


def test_vectorised_env_rewards_and_action_gradients_match_oracle(torch, api):
    """FluidVecEnv (gym-style reset / step over the batched C-ABI calls): three environments with different control
    amplitudes run two steps; every environment's reward and its gradient w.r.t. its action equal the oracle's rollout
    (loss 1e-4, gradient 1e-3) -- the action enters through the solid velocity (Eq. 9b) with the shape frozen."""
    from paper_2405_14903_b200 import env as envmod
    n, nsteps = 24, 2
    P = wl.config2_params(n)
    bc = orc.BC(P["bc_types"], P["bc_values"])
    lo, hi = P["loss_lo"], P["loss_hi"]
    thetas = [0.3, 0.5, -0.8]
    rng = np.random.default_rng(5)
    U0 = [[(0.2 * rng.standard_normal(s)).astype(np.float32) for s in wl.face_shapes(n, n, n)] for _ in thetas]
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    frozen = {s: wl.config2_solid(P, s, 0.5) for s in range(1, nsteps + 1)}       # shape of theta = 0.5, frozen
    unit = {s: [d(a) for a in wl.config2_solid(P, s, 1.0)[1]] for s in frozen}     # u_s per unit amplitude
    phid = {s: d(v[0]) for s, v in frozen.items()}

    def geometry(e, t, action):
        s = int(round(t / P["dt"]))
        return phid[s], tuple(action * a for a in unit[s])

    def reward(e, U):
        blk = U[0][lo:hi, lo:hi, lo:hi].double()
        return (blk * blk).sum()

    venv = envmod.FluidVecEnv(len(thetas), n, n, n, P["dx"], P["dt"], geometry, reward, rho=P["dt"] / P["dt_over_rho"],
                              horizon=nsteps, bc_types=P["bc_types"], bc_values=P["bc_values"], tol=1e-6, maxit=200)
    acts = [torch.tensor(th, dtype=torch.float32, device="cuda", requires_grad=True) for th in thetas]
    venv.reset([[d(a) for a in U] for U in U0])
    for _ in range(nsteps):
        obs, rew, done, info = venv.step(acts)
    assert done == [True] * len(thetas) and len(info["iters"]) == len(thetas)
    sum(rew).backward()
    for e, th in enumerate(thetas):
        def sf(step, th=th):
            phi = frozen[step][0]
            _, us, _, dus = wl.config2_solid(P, step, th)
            return phi, us, np.zeros(phi.shape), dus
        Jo, dJo, _ = orc.rollout(U0[e], sf, nsteps, P["dt"], P["dx"], P["dt_over_rho"], bc, orc.loss_sum_u2(lo, hi))
        assert abs(float(rew[e].detach()) - Jo) <= 1e-4 * abs(Jo), (e, float(rew[e].detach()), Jo)
        assert abs(float(acts[e].grad) - dJo) <= 1e-3 * abs(dJo), (e, float(acts[e].grad), dJo)
    venv.close()
