"""torch.autograd wrappers around the C ABI ("a torch.autograd.Function wrapper"), so that a
simulation written as ordinary torch code -- a controller network producing solid velocities, a loss on the final
velocity -- back-propagates through the library's hand-written adjoints (per-step state
instead of a graph of kernels).  Sequencing of C-ABI calls and tensor bookkeeping only: every step of the path runs in
the library's kernels, and each backward() is the matching adjoint entry point of include/nf.h.

    U = advect(grid, *U, dt)                       # nf_advect            / nf_advect_adjoint
    U = viscosity(grid, *U, nu, dt)                # nf_viscosity         / the same call (symmetric, Eq. 8)
    phi = geom_sdf(grid, params, K, N, M)          # nf_geom_sdf          / nf_geom_sdf_adjoint
    u, v, w, p = project(grid, *U, phi, us, vs, ws, tol, maxit)   # nf_set_solid + nf_project / nf_project_adjoint +
                                                                  # nf_weights_adjoint

A handle holds one geometry at a time: project() installs its phi / U_s again in backward().  The pressure output is
not differentiable (the paper's backward pass starts from dJ/dU, Eq. 6)."""
import torch


class _Advect(torch.autograd.Function):
    @staticmethod
    def forward(ctx, grid, dt, u, v, w):
        ctx.grid, ctx.dt = grid, float(dt)
        ctx.save_for_backward(u, v, w)
        out = [a.detach().clone() for a in (u, v, w)]
        grid.advect(*out, ctx.dt)
        return tuple(out)

    @staticmethod
    def backward(ctx, gu, gv, gw):
        u0, v0, w0 = ctx.saved_tensors
        g = [_dense(a, b) for a, b in zip((gu, gv, gw), (u0, v0, w0))]
        ctx.grid.advect_adjoint(u0, v0, w0, *g, ctx.dt)
        return (None, None) + tuple(g)


class _Viscosity(torch.autograd.Function):
    @staticmethod
    def forward(ctx, grid, nu, dt, u, v, w):
        ctx.grid, ctx.nu, ctx.dt = grid, float(nu), float(dt)
        out = [a.detach().clone() for a in (u, v, w)]
        grid.viscosity(*out, ctx.nu, ctx.dt)
        return tuple(out)

    @staticmethod
    def backward(ctx, gu, gv, gw):
        g = [a.contiguous().clone() for a in (gu, gv, gw)]
        ctx.grid.viscosity(*g, ctx.nu, ctx.dt)
        return (None, None, None) + tuple(g)


class _Project(torch.autograd.Function):
    @staticmethod
    def forward(ctx, grid, tol, maxit, u, v, w, phi, us, vs, ws):
        ctx.grid, ctx.tol, ctx.maxit = grid, float(tol), int(maxit)
        solid = [None if a is None else a.detach().contiguous() for a in (us, vs, ws)]
        phi_c = phi.detach().contiguous()
        grid.set_solid(phi_c, *solid)
        uhat = [a.detach().contiguous() for a in (u, v, w)]
        out = [a.clone() for a in uhat]
        p = torch.zeros(grid.shape_p, dtype=torch.float32, device=out[0].device)  # (a valid guess under warm start)
        grid.project(*out, p, tol=ctx.tol, maxit=ctx.maxit)
        ctx.has_us = [a is not None for a in solid]
        ctx.save_for_backward(p, phi_c, *uhat, *[a for a in solid if a is not None])
        ctx.mark_non_differentiable(p)
        return out[0], out[1], out[2], p

    @staticmethod
    def backward(ctx, gu, gv, gw, _gp):
        saved = list(ctx.saved_tensors)
        p, phi, uhat, rest = saved[0], saved[1], saved[2:5], saved[5:]
        solid = [rest.pop(0) if h else None for h in ctx.has_us]
        grid = ctx.grid
        grid.set_solid(phi, *solid)  # the hierarchy of this step
        g = [_dense(a, b) for a, b in zip((gu, gv, gw), uhat)]
        ga = [torch.empty_like(a) for a in uhat]
        gs = [torch.empty_like(a) for a in uhat]
        grid.project_adjoint(*g, p_saved=p, uhat=uhat, galpha=ga, gus=gs, tol=ctx.tol, maxit=ctx.maxit)
        gphi = torch.empty_like(phi)
        grid.weights_adjoint(*ga, gphi)
        gsolid = [b if h else None for b, h in zip(gs, ctx.has_us)]
        return (None, None, None) + tuple(g) + (gphi,) + tuple(gsolid)


class _GeomSdf(torch.autograd.Function):
    @staticmethod
    def forward(ctx, grid, K, N, M, complement, params):
        ctx.grid, ctx.cfg = grid, (int(K), int(N), int(M), bool(complement))
        ctx.par = params.detach().to("cpu", torch.float32).contiguous().numpy().copy()
        ctx.like = params
        phi = torch.empty(grid.shape_sdf, dtype=torch.float32, device=grid.device)
        grid.geom_sdf(ctx.par, K, N, M, phi, complement)
        return phi

    @staticmethod
    def backward(ctx, gphi):
        K, N, M, complement = ctx.cfg
        g = ctx.grid.geom_sdf_adjoint(ctx.par, K, N, M, gphi.contiguous(), complement)
        return (None, None, None, None, None, torch.from_numpy(g).to(device=ctx.like.device, dtype=ctx.like.dtype))


def _dense(g, like):
    """The incoming gradient as a fresh contiguous tensor (the adjoint entry points work in place); None -> zeros."""
    return torch.zeros_like(like) if g is None else g.contiguous().clone()


def advect(grid, u, v, w, dt):
    return _Advect.apply(grid, dt, u, v, w)


def viscosity(grid, u, v, w, nu, dt):
    return _Viscosity.apply(grid, nu, dt, u, v, w)


def project(grid, u, v, w, phi, us=None, vs=None, ws=None, tol=1e-6, maxit=400):
    """-> (u, v, w, p); differentiable w.r.t. u, v, w (Eq. 7), phi (Eq. 9a through the weight builder, L141) and the
    solid velocity (Eq. 9b)."""
    return _Project.apply(grid, tol, maxit, u, v, w, phi, us, vs, ws)


def geom_sdf(grid, params, K, N, M, complement=False):
    """phi on the nodes from a parameter tensor (any device; the gradient comes back on the same device / dtype)."""
    return _GeomSdf.apply(grid, K, N, M, complement, params)


class _ProjectBatch(torch.autograd.Function):
    """nf_set_solid per environment + nf_project_batch; backward: nf_project_adjoint_batch + nf_weights_adjoint.
    Flat argument list: for every environment u, v, w, phi, us, vs, ws (the solid velocities may be None)."""

    @staticmethod
    def forward(ctx, grids, tol, maxit, *flat):
        from . import api
        n = len(grids)
        ctx.grids, ctx.tol, ctx.maxit = grids, float(tol), int(maxit)
        envs = [flat[7 * e: 7 * e + 7] for e in range(n)]
        outs, ps, saved, has_us = [], [], [], []
        for g, (u, v, w, phi, us, vs, ws) in zip(grids, envs):
            solid = [None if a is None else a.detach().contiguous() for a in (us, vs, ws)]
            phi_c = phi.detach().contiguous()
            g.set_solid(phi_c, *solid)
            uhat = [a.detach().contiguous() for a in (u, v, w)]
            outs.append([a.clone() for a in uhat])
            ps.append(torch.zeros(g.shape_p, dtype=torch.float32, device=uhat[0].device))
            has_us.append([a is not None for a in solid])
            saved += [phi_c] + uhat + [a for a in solid if a is not None]
        api.project_batch(grids, outs, ps, tol=ctx.tol, maxit=ctx.maxit)
        ctx.has_us = has_us
        ctx.save_for_backward(*(ps + saved))
        ctx.mark_non_differentiable(*ps)
        return tuple(a for o in outs for a in o) + tuple(ps)

    @staticmethod
    def backward(ctx, *grads):
        from . import api
        grids, n = ctx.grids, len(ctx.grids)
        saved = list(ctx.saved_tensors)
        ps, rest = saved[:n], saved[n:]
        phis, uhats, solids = [], [], []
        for e in range(n):
            phis.append(rest.pop(0))
            uhats.append([rest.pop(0) for _ in range(3)])
            solids.append([rest.pop(0) if h else None for h in ctx.has_us[e]])
        G, ga, gs, ys = [], [], [], []
        for e, g in enumerate(grids):
            g.set_solid(phis[e], *solids[e])  # (a handle holds one geometry at a time: the one of this step)
            G.append([_dense(grads[3 * e + c], uhats[e][c]) for c in range(3)])
            ga.append([torch.empty_like(a) for a in uhats[e]])
            gs.append([torch.empty_like(a) for a in uhats[e]])
            ys.append(torch.zeros_like(ps[e]))
        api.project_adjoint_batch(grids, G, ys, p_saved=ps, uhat=uhats, galpha=ga, gus=gs, tol=ctx.tol, maxit=ctx.maxit)
        out = []
        for e, g in enumerate(grids):
            gphi = torch.empty_like(phis[e])
            g.weights_adjoint(*ga[e], gphi)
            out += G[e] + [gphi] + [b if h else None for b, h in zip(gs[e], ctx.has_us[e])]
        return (None, None, None) + tuple(out)


def project_batch(grids, U, phi, us=None, tol=1e-6, maxit=400):
    """Batched projection of n environments (include/nf.h nf_project_batch): U = list of (u, v, w), phi = list of node
    SDFs, us = list of (us, vs, ws) triples / None.  -> (list of (u, v, w), list of p); differentiable like project()."""
    n = len(grids)
    flat = []
    for e in range(n):
        s = (None, None, None) if us is None or us[e] is None else tuple(us[e])
        flat += list(U[e]) + [phi[e]] + list(s)
    out = _ProjectBatch.apply(list(grids), tol, maxit, *flat)
    return [tuple(out[3 * e: 3 * e + 3]) for e in range(n)], list(out[3 * n:])
