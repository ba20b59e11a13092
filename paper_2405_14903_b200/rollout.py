"""Full time steps forward and backward through the C ABI (PAPER.md:L78 forward order, L111-141 backward pass):
per step  nf_advect -> nf_set_solid(phi^{n+1}, u_s^{n+1}) -> nf_project,  and in reverse
nf_project_adjoint -> nf_weights_adjoint -> nf_advect_adjoint, with the per-step state (U^n, Uhat, p) kept by the
caller instead of an autodiff graph.  Argument marshalling and the two inner products of the geometry
chain rule only: every step of the path runs in the library's kernels."""
import torch


def rollout(grid, U0, solid_fn, nsteps, dt, loss_fn, tol=1e-6, maxit=400, advect_on=True, nu=0.0, stats=None):
    """solid_fn(step) -> (phi, (us, vs, ws), dphi_dtheta, (dus, dvs, dws)) as CUDA float32 tensors (the derivative
    tensors may be None); loss_fn(U) -> (J tensor, [dJ/du, dJ/dv, dJ/dw]).
    Several control parameters on which U_s depends linearly (BASELINE.json configs[2]: 16 bump amplitudes): pass
    dus = {"basis": [(bu, bv, bw) per parameter], "scale": s} -- dJ/dtheta then is a list, dJ/dtheta_k = sum over the
    steps of s <dJ/dU_s, basis_k> (Eq. 9b in the derived form R10).
    stats (optional dict): filled with the PCG iteration counts per step ("iters_fwd", "iters_adj"; synchronises).
    Returns (J, dJ/dtheta, dJ/dU0) -- J and dJ/dtheta as Python floats."""
    g = grid
    U = [a.clone() for a in U0]
    tape = []
    if stats is not None:
        stats["iters_fwd"], stats["iters_adj"] = [], []
    dvec = None
    for n in range(1, nsteps + 1):
        Uprev = [a.clone() for a in U]
        if advect_on:
            g.advect(*U, dt)
        if nu != 0.0:
            g.viscosity(*U, nu, dt)  # advection, viscosity, projection
        phi, us, dphi, dus = solid_fn(n)
        g.set_solid(phi, *us)
        Uhat = [a.clone() for a in U]
        p = torch.zeros(g.shape_p, dtype=torch.float32, device=U[0].device)  # (zeros: a valid guess under the warm-start option)
        g.project(*U, p, tol=tol, maxit=maxit)
        if stats is not None:
            stats["iters_fwd"].append(g.last_solve_info()["iters"])
        tape.append((Uprev, Uhat, p, phi, us, dphi, dus))
    J, G = loss_fn(U)
    G = [a.clone() for a in G]
    dtheta = torch.zeros((), dtype=torch.float64, device=U[0].device)
    ga = [torch.empty_like(a) for a in U]
    gs = [torch.empty_like(a) for a in U]
    gphi = torch.empty(g.shape_sdf, dtype=torch.float32, device=U[0].device)
    for n in range(nsteps, 0, -1):
        Uprev, Uhat, p, phi, us, dphi, dus = tape[n - 1]
        g.set_solid(phi, *us)  # the hierarchy of step n (the handle holds one geometry at a time)
        g.project_adjoint(*G, p_saved=p, uhat=Uhat, galpha=ga, gus=gs, tol=tol, maxit=maxit)
        if stats is not None:
            stats["iters_adj"].append(g.last_solve_info()["iters"])
        if dphi is not None:
            g.weights_adjoint(*ga, gphi)
            dtheta += (gphi.double() * dphi.double()).sum()
        if isinstance(dus, dict):
            if dvec is None:
                dvec = torch.zeros(len(dus["basis"]), dtype=torch.float64, device=U[0].device)
            for k, bk in enumerate(dus["basis"]):
                dvec[k] += dus["scale"] * sum((a.double() * b.double()).sum() for a, b in zip(gs, bk))
        elif dus is not None:
            for a, b in zip(gs, dus):
                if b is not None:
                    dtheta += (a.double() * b.double()).sum()
        if nu != 0.0:
            g.viscosity(*G, nu, dt)  # Eq. 8: the same symmetric matrix
        if advect_on:
            g.advect_adjoint(*Uprev, *G, dt)
    if dvec is not None:
        return float(J), [float(x) for x in dvec.cpu()], G
    return float(J), float(dtheta), G


def cfl_substeps(grid, U, dt_frame, cfl=1.0, max_substeps=64):
    """Sub-step sizes that advance one frame of length dt_frame under the CFL condition the paper says it adopts
    (its constant is not given -- R24: dt <= cfl * dx / max|U|): the first sub-step's dt from the
    current velocity, and the number of equal sub-steps that would cover the frame at that dt.  The caller re-evaluates
    after every sub-step (the velocity changes).  Returns (dt_sub, n_left)."""
    import math
    vmax = grid.max_speed(*U)
    if not (vmax > 0.0) or math.isinf(vmax):
        return dt_frame, 1
    n = max(1, min(max_substeps, int(math.ceil(dt_frame * vmax / (cfl * grid.dx) - 1e-9))))
    return dt_frame / n, n


def rollout_substepped(grid, U0, solid_fn_t, nframes, dt_frame, rho, loss_fn, cfl=1.0, dts=None, tol=1e-6, maxit=400,
                       advect_on=True, nu=0.0, max_substeps=64):
    """N frames of length dt_frame, each advanced by CFL sub-steps ("adopts CFL condition", L403-410
    Table 4: 11 / 54 / 58 solver steps per cycle; R24): per sub-step of size dt  nf_set_dt_rho(dt / rho) -> nf_advect ->
    [nf_viscosity] -> nf_set_solid(geometry at the sub-step's end time) -> nf_project, and the backward pass over the
    sub-steps in reverse with the same dt (a constant of the backward pass).  dt comes from cfl_substeps (nf_max_speed
    on the device) unless `dts` (one list of sub-step sizes per frame) is given, which replays them.
    solid_fn_t(t) -> (phi, (us, vs, ws), dphi_dtheta, (dus, dvs, dws)) at physical time t, CUDA float32 tensors.
    Returns (J, dJ/dtheta, dJ/dU0, dts_used).  Sequencing of C-ABI calls only."""
    g = grid
    U = [a.clone() for a in U0]
    tape, used = [], []
    for f in range(nframes):
        t, t_end = f * dt_frame, (f + 1) * dt_frame
        frame, k = [], 0
        while t_end - t > 1e-12 * dt_frame:
            dt = dts[f][k] if dts is not None else cfl_substeps(g, U, t_end - t, cfl, max_substeps)[0]
            Uprev = [a.clone() for a in U]
            g.set_dt_rho(dt / rho)
            if advect_on:
                g.advect(*U, dt)
            if nu != 0.0:
                g.viscosity(*U, nu, dt)
            t = t + dt
            phi, us, dphi, dus = solid_fn_t(t)
            g.set_solid(phi, *us)
            Uhat = [a.clone() for a in U]
            p = torch.zeros(g.shape_p, dtype=torch.float32, device=U[0].device)
            g.project(*U, p, tol=tol, maxit=maxit)
            tape.append((Uprev, Uhat, p, phi, us, dphi, dus, dt))
            frame.append(dt)
            k += 1
            if dts is not None and k >= len(dts[f]):
                break
        used.append(frame)
    J, G = loss_fn(U)
    G = [a.clone() for a in G]
    dtheta = torch.zeros((), dtype=torch.float64, device=U[0].device)
    ga = [torch.empty_like(a) for a in U]
    gs = [torch.empty_like(a) for a in U]
    gphi = torch.empty(g.shape_sdf, dtype=torch.float32, device=U[0].device)
    for Uprev, Uhat, p, phi, us, dphi, dus, dt in reversed(tape):
        g.set_dt_rho(dt / rho)
        g.set_solid(phi, *us)
        g.project_adjoint(*G, p_saved=p, uhat=Uhat, galpha=ga, gus=gs, tol=tol, maxit=maxit)
        g.weights_adjoint(*ga, gphi)
        if dphi is not None:
            dtheta += (gphi.double() * dphi.double()).sum()
        if dus is not None:
            for a, b in zip(gs, dus):
                if b is not None:
                    dtheta += (a.double() * b.double()).sum()
        if nu != 0.0:
            g.viscosity(*G, nu, dt)
        if advect_on:
            g.advect_adjoint(*Uprev, *G, dt)
    return float(J), float(dtheta), G, used


def tape_bytes(grid, nsteps):
    """Device memory of the per-step state kept for the backward pass instead of an autodiff graph:
    U^n, Uhat (3 face arrays each) and p per step, float32."""
    nu_, nv_, nw_ = [int(torch.tensor(s).prod()) for s in (grid.shape_u, grid.shape_v, grid.shape_w)]
    np_ = int(torch.tensor(grid.shape_p).prod())
    return 4 * nsteps * (2 * (nu_ + nv_ + nw_) + np_)


def rollout_parametric(grid, U0, prims_fn, nsteps, dt, loss_fn, tol=1e-6, maxit=400, advect_on=True, band=float("inf")):
    """The co-design loop: like rollout(), with the solid of step n given by
    parametric primitives: prims_fn(step) -> list of (params, pdot or None, K, N, M) (host vectors, layout of
    include/nf.h).  The solid is the union of the primitives; one with pdot moves and supplies U_s on the faces
    within `band` of it, in list order.  Backward: nf_project_adjoint -> nf_weights_adjoint -> nf_geom_csg_adjoint ->
    nf_geom_sdf_adjoint (dJ/dparams, through phi) and nf_geom_velocity_adjoint (dJ/dpdot).
    Returns (J, grads, dJ/dU0), grads[step-1][i] = (dJ/dparams, dJ/dpdot or None) as float64 NumPy vectors."""
    import numpy as np
    import warnings
    g = grid
    dev = U0[0].device
    if any(pd is not None for (_p, pd, _K, _N, _M) in prims_fn(1)):
        # R31: U_s is differentiated w.r.t. pdot only.  For a primitive that moves, dJ/dparams below holds the part
        # through phi (the shape at t^{n+1}) and NOT the part through U_s(params) (closest point and normal).
        warnings.warn("rollout_parametric: dJ/dparams of a moving primitive (pdot given) omits d U_s / d params "
                      "(DESIGN.md R31); dJ/dpdot and the gradients of static primitives are complete", RuntimeWarning,
                      stacklevel=2)
    new_nodes = lambda: torch.empty(g.shape_sdf, dtype=torch.float32, device=dev)
    U = [a.clone() for a in U0]
    tape = []
    for n in range(1, nsteps + 1):
        Uprev = [a.clone() for a in U]
        if advect_on:
            g.advect(*U, dt)
        prims = prims_fn(n)
        phis, partial = [], []
        for i, (p, pd, K, N, M) in enumerate(prims):
            f = new_nodes()
            g.geom_sdf(p, K, N, M, f)
            phis.append(f)
            if i == 0:
                partial.append(f)
            else:
                u = new_nodes()
                g.geom_csg("union", partial[-1], f, u)
                partial.append(u)
        us = None
        for (p, pd, K, N, M) in prims:
            if pd is not None:
                if us is None:
                    us = [torch.zeros(s, dtype=torch.float32, device=dev) for s in (g.shape_u, g.shape_v, g.shape_w)]
                g.geom_velocity(p, pd, K, N, M, *us, band=band)
        g.set_solid(partial[-1], *(us if us is not None else (None, None, None)))
        Uhat = [a.clone() for a in U]
        pr = torch.zeros(g.shape_p, dtype=torch.float32, device=dev)
        g.project(*U, pr, tol=tol, maxit=maxit)
        tape.append((Uprev, Uhat, pr, prims, phis, partial, us))
    J, G = loss_fn(U)
    G = [a.clone() for a in G]
    ga = [torch.empty_like(a) for a in U]
    gs = [torch.empty_like(a) for a in U]
    grads = [None] * nsteps
    for n in range(nsteps, 0, -1):
        Uprev, Uhat, pr, prims, phis, partial, us = tape[n - 1]
        g.set_solid(partial[-1], *(us if us is not None else (None, None, None)))
        g.project_adjoint(*G, p_saved=pr, uhat=Uhat, galpha=ga, gus=gs, tol=tol, maxit=maxit)
        gphi = new_nodes()
        g.weights_adjoint(*ga, gphi)
        gphis = [None] * len(prims)
        for i in range(len(prims) - 1, 0, -1):
            ga_i, gb_i = new_nodes(), new_nodes()
            g.geom_csg_adjoint("union", partial[i - 1], phis[i], gphi, ga_i, gb_i)
            gphi, gphis[i] = ga_i, gb_i
        gphis[0] = gphi
        out = [None] * len(prims)
        for i in range(len(prims) - 1, -1, -1):
            p, pd, K, N, M = prims[i]
            gp = g.geom_sdf_adjoint(p, K, N, M, gphis[i])
            gd = None
            if pd is not None:
                gd = g.geom_velocity_adjoint(p, K, N, M, *gs, band=band)
                # the faces this primitive owns are taken: its velocity map with pdot = 0 writes 0 exactly there
                g.geom_velocity(p, np.zeros_like(np.asarray(p, dtype=np.float32)), K, N, M, *gs, band=band)
            out[i] = (gp, gd)
        grads[n - 1] = out
        if advect_on:
            g.advect_adjoint(*Uprev, *G, dt)
    return float(J), grads, G
