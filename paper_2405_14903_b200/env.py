"""Gym-style vectorised environment over the batched C-ABI calls ("gym-like ...
PyTorch", L147-160: the paper's control tasks are 40^3-48^3 grids with 10-180 frames).  E equally sized simulations
advance together: one time step is  nf_advect -> [nf_viscosity] -> nf_set_solid(geometry of the action) ->
nf_project_batch  (one launch per solver pass for all environments), written with the torch.autograd wrappers of
autograd.py so that a reward computed from the returned velocities back-propagates to the actions through the library's
hand-written adjoints -- `reward.sum().backward()` after a rollout gives dJ/d(actions).

The task itself (geometry, reward, observation) is the caller's: the paper's six tasks are not reproducible from its
text, so this module holds the protocol and the stepping only -- no method arithmetic."""
import torch

from . import api, autograd


class FluidVecEnv:
    """reset() -> observations;  step(actions) -> (observations, rewards, dones, info).

    geometry_fn(env_index, t, action) -> (phi, (us, vs, ws) or None): the solid at physical time t for that action, as
        torch tensors on the device (phi on the nodes, > 0 in the fluid; differentiable w.r.t. `action` if gradients
        are wanted).
    reward_fn(env_index, (u, v, w)) -> scalar tensor;  observe_fn(env_index, (u, v, w)) -> tensor (default: u, v, w).
    """

    def __init__(self, n_envs, nx, ny, nz, dx, dt, geometry_fn, reward_fn, rho=1.0, horizon=10, nu=0.0,
                 bc_types=(0,) * 6, bc_values=(0.0,) * 6, observe_fn=None, tol=1e-6, maxit=400, device=None):
        self.grids = [api.Grid(nx, ny, nz, dx, device) for _ in range(int(n_envs))]
        for g in self.grids:
            g.set_dt_rho(dt / rho)
            for f in range(6):
                g.set_domain_bc(f, bc_types[f], bc_values[f])
        self.device = self.grids[0].device
        self.dt, self.nu, self.horizon, self.tol, self.maxit = float(dt), float(nu), int(horizon), tol, maxit
        self.geometry_fn, self.reward_fn = geometry_fn, reward_fn
        self.observe_fn = observe_fn or (lambda e, U: U)
        self.U, self.t = None, 0

    def __len__(self):
        return len(self.grids)

    def reset(self, U0=None):
        """U0: list of (u, v, w) per environment, or None for a fluid at rest."""
        g = self.grids[0]
        z = lambda: tuple(torch.zeros(s, dtype=torch.float32, device=self.device) for s in (g.shape_u, g.shape_v, g.shape_w))
        self.U = [z() if U0 is None else tuple(a.clone() for a in U0[e]) for e in range(len(self.grids))]
        self.t = 0
        return [self.observe_fn(e, U) for e, U in enumerate(self.U)]

    def step(self, actions):
        if self.U is None:
            raise RuntimeError("call reset() first")
        t1 = (self.t + 1) * self.dt
        Ut, phis, solids = [], [], []
        for e, (g, U) in enumerate(zip(self.grids, self.U)):
            V = autograd.advect(g, *U, self.dt)
            if self.nu != 0.0:
                V = autograd.viscosity(g, *V, self.nu, self.dt)
            phi, us = self.geometry_fn(e, t1, actions[e])
            Ut.append(V); phis.append(phi); solids.append(us)
        Un, ps = autograd.project_batch(self.grids, Ut, phis, solids, tol=self.tol, maxit=self.maxit)
        self.U = Un
        self.t += 1
        obs = [self.observe_fn(e, U) for e, U in enumerate(Un)]
        rew = [self.reward_fn(e, U) for e, U in enumerate(Un)]
        done = [self.t >= self.horizon] * len(self.grids)
        info = {"iters": [g.last_solve_info()["iters"] for g in self.grids], "pressure": ps, "t": t1}
        return obs, rew, done, info

    def detach(self):
        """Cut the autograd history at the current state (truncated back-propagation through time)."""
        self.U = [tuple(a.detach() for a in U) for U in self.U]

    def close(self):
        for g in self.grids:
            g.close()
        self.grids = []
