/* nf.h -- C ABI of the B200-native NeuralFluid pressure projection (forward + adjoint), MGPCG solver,
 * face-weight builder and semi-Lagrangian advection.
 *
 * Paper: arXiv 2405.14903 (NeuralFluid); cited below as PAPER.md:Lnnn.  Readings of silent / garbled
 * passages are listed in DESIGN.md section 3 and cited as R<n>.
 *
 * Conventions ("pressures stored at cell centers and velocities at cell faces"):
 *   - All field arrays are float32, C-ordered [k][j][i] with x (i) fastest.
 *       p   : cells  nz * ny * nx
 *       u   : x-faces nz * ny * (nx+1)      u[k][j][i] is the face between cells i-1 and i
 *       v   : y-faces nz * (ny+1) * nx
 *       w   : z-faces (nz+1) * ny * nx
 *       sdf : nodes  (nz+1) * (ny+1) * (nx+1), > 0 in fluid (R1, R2)
 *   - G  (cells -> faces): (G p)_u[i] = p[i] - p[i-1];  G^T f = f_u[i]-f_u[i+1] + f_v[j]-f_v[j+1] + f_w[k]-f_w[k+1];
 *     -(1/dx) G^T is the divergence.  S = diag(alpha), c = dt_over_rho/dx, A = c G^T S G
 *     (Eq. 4).
 *   - Domain faces are numbered 0..5 = -x,+x,-y,+y,-z,+z.
 *
 * Pointers: unless a function name ends in `_host`, EVERY array pointer is a DEVICE pointer owned by the
 * caller (e.g. a contiguous float32 torch tensor).  The library never frees or retains a caller pointer
 * after the call returns; it copies what it needs.  `_host` entry points take HOST pointers (pageable or
 * pinned) and perform the host<->device copies themselves on the handle's stream.
 *
 * Execution: all kernels are enqueued on the handle's stream (nf_set_stream).  Calls that contain a
 * solve (nf_solve, nf_project, nf_project_adjoint) return once the iteration count is known (the host
 * polls a mapped status word; it never calls cudaDeviceSynchronize); results are ordered on the stream.
 * Every other call only enqueues work.  There is NO CPU fallback: every step runs in CUDA kernels.
 *
 * Threads: a handle is used by one host thread at a time; different handles are independent (no shared mutable
 * state in the library), so several small grids can be driven concurrently, one handle + stream + thread each
 * (paper_2405_14903_b200/envs.py; the cooperative coarse kernel is sized for its level so that they overlap).
 *
 * Errors: functions return an int status.  Negative = error, nothing useful written; NF_NOT_CONVERGED = the
 * best iterate was written but maxit was hit.  No exceptions, no exit(), no stdout.
 */
#ifndef NF_H_
#define NF_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nf_grid nf_grid; /* opaque: owns face weights, multigrid hierarchy, solver scratch */

enum {
  NF_OK = 0,
  NF_NOT_CONVERGED = 1,
  NF_ERR_INVALID = -1, /* NULL handle / pointer, non-positive size, bad enum value          */
  NF_ERR_ALLOC = -2,   /* device or host allocation failed                                   */
  NF_ERR_CUDA = -3,    /* a CUDA runtime call failed; see nf_last_error                      */
  NF_ERR_STATE = -4    /* weights not set yet (call nf_set_solid or nf_set_weights first)    */
};

enum { NF_BC_CLOSED = 0, NF_BC_DIRICHLET = 1 };

/* Library version string, e.g. "nf-b200 0.1 (sm_100a)". */
const char *nf_version(void);

/* Create a handle for an nx*ny*nz MAC grid with spacing dx.  Allocates the multigrid
 * hierarchy ("hierarchical grid data structure") and all solver scratch on the current
 * CUDA device.  Defaults: six closed walls, dt_over_rho = 1, stream 0.  nz == 1 selects 2-D mode (the hierarchy
 * coarsens x and y only; the two z-walls stay closed).  Arrays are addressed with 32-bit
 * offsets: (nx+8)(ny+1)(nz+1) must stay below 2^32 (about 1600^3), and nf_advect below 2^31 nodes; larger
 * grids return NF_ERR_INVALID. */
int nf_grid_create(int nx, int ny, int nz, float dx, nf_grid **out);
void nf_grid_destroy(nf_grid *g);

/* cuda_stream is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = legacy stream 0. */
int nf_set_stream(nf_grid *g, void *cuda_stream);

/* Delta t / rho of Eqs. 4-5 (R5).  c = dt_over_rho/dx. */
int nf_set_dt_rho(nf_grid *g, float dt_over_rho);

/* Domain boundary condition of face 0..5 (R6, R19): NF_BC_CLOSED = wall at rest, alpha forced to 0;
 * NF_BC_DIRICHLET = a ghost cell one dx outside holds p_value (Eq. 15a generalised).
 * Must be called BEFORE nf_set_solid / nf_set_weights; changing it afterwards invalidates the weights. */
int nf_set_domain_bc(nf_grid *g, int face, int type, float p_value);

/* Solver options (PAPER.md:L230 names only "MGPCG"; every parameter is this library's choice, R13):
 *   nu_pre / nu_post: red-black Gauss-Seidel sweeps before / after the coarse correction on the FINEST level
 *     (default 1, 1; PCG needs a symmetric preconditioner, i.e. nu_pre == nu_post -- unequal values are accepted for
 *     stand-alone V-cycles and run the generic kernels).  The levels below take nf_set_coarse_sweeps;
 *   flags: bit 0 = reserved,
 *          bit 1 = test hook: force the generic kernels (fp32 weights, one colour per launch) on every level,
 *          bit 2 = switch OFF the true-residual refresh.  By default a solve with tol < 3e-4 runs PCG to 30 tol,
 *                  re-evaluates r = b - A x in fp64 (the fp32 recursion r -= a q drifts: at 256^3 a recursive 1e-6
 *                  was a true 4e-5), and runs PCG on that residual for a correction down to tol; the true residual
 *                  then sits at the storage rounding of the fp32 pressure.  Where the fused
 *                  kernels run, the refresh happens IN FLIGHT instead: PCG runs straight to tol, one iteration
 *                  evaluates b - A x in fp64 once the residual is below sqrt(tol) and -- if that differs from the
 *                  recursive residual by no more than 10 % (decided on the device) -- continues from it with the
 *                  search direction kept and the later updates in a separate correction; otherwise as above,
 *          bit 3 = warm start: the solution array the caller passes (p of nf_project / nf_solve, y_out of
 *                  nf_project_adjoint) holds the initial guess on entry, e.g. the pressure of the previous time
 *                  step (the paper is silent on x0, R11; default x0 = 0).  The stopping criterion stays relative to
 *                  ||b||.  Never applied to the library's internal scratch (adjoint without y_out). */
int nf_set_solver_options(nf_grid *g, int nu_pre, int nu_post, int flags);

/* Red-black Gauss-Seidel sweeps before AND after the coarse correction on level 1 (the first level below the finest
 * one) and on every level below that (1..8 each; R13: the paper names only "MGPCG").  Default: 2 and 3 on grids of
 * 3 M cells and more, 1 and 1 below.  Those levels hold 1/8 + 1/64 + ... of the cells and run inside one cooperative
 * kernel: at 256^3 the extra sweeps double that kernel's time (+ 27 % on a PCG iteration) and save 45 % of the
 * iterations on the channel-gate workload.  May be called at any time between solves; handles
 * solved together by the *_batch calls must agree. */
int nf_set_coarse_sweeps(nf_grid *g, int nu_level1, int nu_deeper);
/* The smoothing sweeps in force: finest level before / after the coarse correction, level 1, every deeper level
 * (the defaults depend on the grid size: nf_grid_create picks 1, 1 and 1, 1 below 3 M cells, 2, 3 from there on).
 * Any pointer may be NULL. */
int nf_get_sweeps(nf_grid *g, int *nu_fine_pre, int *nu_fine_post, int *nu_level1, int *nu_deeper);
/* Over-relaxation factor omega of the red-black sweeps on every level below the finest (SOR: z <- (1 - omega) z +
 * omega GS(z); 1 <= omega < 2, NF_ERR_INVALID otherwise; 1 = Gauss-Seidel).  Pre- and post-smoother use the same factor
 * in mirrored order, so the V-cycle stays symmetric positive definite for PCG.  Costs no phase and no pass: those
 * levels' bodies carry the old value and restrict the full residual of all eight children (the finest level's fused
 * kernels are plain Gauss-Seidel whatever this says; 2-D grids ignore it).  Default 1.4 (measured on the channel-gate,
 * sphere-field and chamber workloads).  May be called at any time between solves; handles solved
 * together by the *_batch calls must agree. */
int nf_set_coarse_relaxation(nf_grid *g, float omega);
float nf_get_coarse_relaxation(nf_grid *g);

/* The low-order part of the pressure.  A solve to 1e-6 ends with a correction e
 * of a fp32 pressure x = O(1): rounding x + e back to fp32 alone leaves a TRUE residual of ~7e-6 at 256^3 (the storage
 * floor of p).  With a cell array installed here, nf_solve / nf_project / nf_project_adjoint also write
 * lo = (x + e) - fl(x + e), evaluated in fp64: the solution is p + lo (its fp64 true residual is the 1e-6 the
 * solver stopped at), and nf_project subtracts the gradient of p + lo.  lo is zeroed when a solve needs no correction.
 * NULL (the default) switches it off.  The array must stay valid until it is replaced. */
int nf_set_pressure_lo(nf_grid *g, float *lo_cells);

/* a-1  Face weights from the solid SDF: per face, the fluid area fraction alpha from
 * the 4 node values at its corners (marching-squares area; the printed one-fluid-corner formula
 * 1/2 * phi_A/(phi_A-phi_B) * phi_A/(phi_A-phi_D) and its companions, R3; alpha < 1e-4 -> 0, R4); closed
 * domain walls get 0 (R19).  Builds the coarse-level weights of the hierarchy.  us/vs/ws: solid velocity
 * on faces (same layout as u/v/w), any of them NULL = zero.  Copied; closed-wall faces are at rest. */
int nf_set_solid(nf_grid *g, const float *sdf_nodes, const float *us, const float *vs, const float *ws);

/* Test / power-user hook: install face weights directly (MAC face layout), bypassing the builder.
 * Closed-wall faces are forced to 0.  The solid velocity is kept (zero if never set). */
int nf_set_weights(nf_grid *g, const float *au, const float *av, const float *aw);
int nf_get_weights(nf_grid *g, float *au, float *av, float *aw);
/* Install only the solid velocity (NULL = zero), keeping the weights. */
int nf_set_solid_velocity(nf_grid *g, const float *us, const float *vs, const float *ws);

/* a-3..a-5  Solve A p = rhs with MGPCG, A = c G^T S G with homogeneous ghosts.
 * Convergence (R11): ||r||_2 <= tol ||rhs||_2, x0 = 0.  rhs is taken as 0 on inactive cells (sum of the 6
 * face weights = 0), where p = 0.  On every fluid component without an open Dirichlet face the system is
 * singular (R12): the mean of rhs over that component is removed and p has zero mean over it.
 * rhs is not modified.  p may not alias rhs. */
int nf_solve(nf_grid *g, const float *rhs, float *p, float tol, int maxit);

/* a-2, a-3..5, a-6  Pressure projection (Eqs. 4-5).  In: u,v,w = Uhat.  Out: u,v,w =
 * U^{n+1} = Uhat - c G p on faces with alpha > 0 and = U_s on faces with alpha = 0 (R7, R19); p = P^{n+1}
 * (scaled by dt_over_rho as set).  b = G^T (S Uhat + (I-S) U_s) + c alpha p_D on Dirichlet ghosts. */
int nf_project(nf_grid *g, float *u, float *v, float *w, float *p, float tol, int maxit);

/* a-7  Adjoint projection (Eqs. 6-7; L134-139 Eq. 9 in the derived forms R9, R10).
 * In: gu,gv,gw = dJ/dU^{n+1}; p_saved = P^{n+1}; uhat_* = the projection's input velocity.
 * Solves A y = -c G^T (M g), M = [alpha > 0], with the same hierarchy.
 * Out: gu,gv,gw (in place) = dJ/dUhat = M g + S G y;
 *      galpha_* (may be NULL) = dJ/dalpha_f = (G y)_f [ (Uhat - U_s)_f - c (G p)_f ];
 *      gus_*    (may be NULL) = dJ/dU_s = (I-M) g + (I-S) G y;  both 0 on closed walls (R19);
 *      y_out    (may be NULL) = the adjoint variable y (cell array). */
int nf_project_adjoint(nf_grid *g, float *gu, float *gv, float *gw, const float *p_saved,
                       const float *uhat_u, const float *uhat_v, const float *uhat_w,
                       float *galpha_u, float *galpha_v, float *galpha_w,
                       float *gus_u, float *gus_v, float *gus_w, float *y_out, float tol, int maxit);

/* ---- NEXT-4  Batched small grids (Table 1: the paper's tasks are 40^3-48^3 grids,
 * far too small to fill a B200 one at a time; L145 "gym-like" environments) --------------------------------------------
 * n handles of EQUAL extents on ONE stream, each with its own solid, boundary values and fields: nf_solve /
 * nf_project / nf_project_adjoint for all of them, with every pass of a PCG iteration issued as ONE kernel launch for
 * the whole batch (blockIdx.z = environment x z-chunk; one cooperative coarse-level launch, barriers per environment).
 * The PCG scalars, the convergence test (R11, relative to each environment's own ||b||) and the early exit stay per
 * environment; the host loop ends when all have converged.  x0 = 0, single-phase PCG on the recursive residual (no
 * fp64 refresh: these grids are far above the fp32 storage floor of DESIGN.md section 7).  Handles the batched kernels
 * cannot take (unequal extents, ragged levels, test hooks, more cooperative CTAs than SMs) are solved one at a time
 * inside the same call -- same results.  Arguments are HOST arrays of n device pointers, meanings as in the
 * single-handle calls; y (the adjoint variable, n cell arrays) is required.  status (may be NULL): NF_OK /
 * NF_NOT_CONVERGED per environment; the return value is the worst of them, or a negative error. */
int nf_solve_batch(nf_grid *const *g, int n, const float *const *rhs, float *const *p, float tol, int maxit, int *status);
int nf_project_batch(nf_grid *const *g, int n, float *const *u, float *const *v, float *const *w, float *const *p,
                     float tol, int maxit, int *status);
int nf_project_adjoint_batch(nf_grid *const *g, int n, float *const *gu, float *const *gv, float *const *gw,
                             const float *const *p_saved, const float *const *uhat_u, const float *const *uhat_v,
                             const float *const *uhat_w, float *const *galpha_u, float *const *galpha_v,
                             float *const *galpha_w, float *const *gus_u, float *const *gus_v, float *const *gus_w,
                             float *const *y, float tol, int maxit, int *status);

/* a-8  Semi-Lagrangian advection (Eq. 2; L353-357 Eqs. 11-12; R14, R20): for every face
 * position x of component c: v0 = U(x); x_m = x - dt/2 v0; v_m = U(x_m); x_b = x - dt v_m;
 * out_c = U_c(x_b), U(.) = per-component trilinear interpolation, positions clamped to the lattice.
 * In place (the library reads from an internal copy). */
int nf_advect(nf_grid *g, float *u, float *v, float *w, float dt);

/* NEXT-1  Explicit viscosity step (Eq. 3; L359-361 Eq. 13):
 * Uhat = (I - nu dt/dx^2 G^T G) Utilde, per component on that component's own lattice, 7-point, nothing outside
 * the lattice (R23: the symmetric form).  In place (the library reads from an internal copy).  Every face is
 * updated; closed ones are overwritten by the projection.  The operator is symmetric: the backward pass (Eq. 8)
 * is THIS call applied to dJ/dUhat -- there is no separate adjoint entry point.  Explicit: stable for
 * nu dt/dx^2 <= 1/6 (the caller's responsibility).  nu < 0 or dt < 0: NF_ERR_INVALID. */
int nf_viscosity(nf_grid *g, float *u, float *v, float *w, float nu, float dt);

/* NEXT-1  CFL sub-stepping support (the simulator "adopts CFL condition",
 * the steps simulated exceed the frames; the constant is not given, R24): *max_abs_host = max over all faces of
 * |u|, |v|, |w| (device reduction; HOST pointer; this call synchronises the stream).  The policy
 * dt = min(dt_frame_left, C dx / max) and the loop over sub-steps belong to the caller
 * (paper_2405_14903_b200/rollout.py: cfl_substeps); dt is a constant of the backward pass. */
int nf_max_speed(nf_grid *g, const float *u, const float *v, const float *w, float *max_abs_host);

/* a-9  Adjoint of nf_advect (Eq. 8).  u0,v0,w0 = the saved pre-advection U^n;
 * in: gu,gv,gw = dJ/dUtilde; out (in place): dJ/dU^n. */
int nf_advect_adjoint(nf_grid *g, const float *u0, const float *v0, const float *w0,
                      float *gu, float *gv, float *gw, float dt);

/* a-10  dJ/dalpha -> dJ/dphi at nodes, for the sdf last given to nf_set_solid.
 * gsdf_nodes is overwritten. */
int nf_weights_adjoint(nf_grid *g, const float *galpha_u, const float *galpha_v, const float *galpha_w,
                       float *gsdf_nodes);

/* ---- NEXT-2  Differentiable parametric geometry (section 2.2; L337-347 appendix A) ----
 * One primitive = one "closed 3-D surface": K key cross-sections, evenly spaced on [z0, z1] along the z axis, each a
 * closed curve of N cubic Bezier curves in the polar frame of its centre (L339-343).  Parameter vector (HOST pointer,
 * float32, physical units; node (i,j,k) sits at (i dx, j dx, k dx)):
 *     params = [z0, z1,  then for key k = 0..K-1:  cx_k, cy_k, rho1_k[0..N-1], rho2_k[0..N-1]]     2 + K (2 + 2N) floats
 * Curve i of a section spans the polar angles [theta_i, theta_{i+1}], theta_i = 2 pi i / N; its inner control points
 * sit at radius rho1_i, angle theta_i + 2 pi/(3N), and radius rho2_i, angle theta_{i+1} - 2 pi/(3N) (L341); the shared
 * endpoint on the ray theta_{i+1} is collinear with its two neighbours: radius 2 cos(2 pi/(3N)) rho2_i rho1_{i+1} /
 * (rho2_i + rho1_{i+1}) (R25).  Between key sections centre and radii are interpolated piecewise linearly in
 * s = clamp((z - z0)/(z1 - z0), 0, 1) (Eq. 10 is garbled: R27).  The curve is sampled at M points per Bezier curve and
 * the distance is the exact signed distance d2 to that closed polygon of N M edges (R26).
 * Limits: 1 <= K <= 64, 2 <= N <= 64, N M <= 2048, z1 > z0, all radii > 0 (NF_ERR_INVALID otherwise).
 * params_host / pdot_host / g*_host are HOST arrays (copied before the call returns); every field is a DEVICE array. */
enum { NF_GEOM_COMPLEMENT = 1 }; /* flags: the primitive is fluid INSIDE its surface (a chamber): phi = -d */
enum { NF_CSG_UNION = 0, NF_CSG_INTERSECTION = 1 };

/* phi at the nodes (layout of nf_set_solid's sdf_nodes; > 0 in the fluid): phi = d = max(d2(x, y; section(z)),
 * z0 - z, z - z1), the cross-section intersected with the slab z0 <= z <= z1 (R28); -d with NF_GEOM_COMPLEMENT.
 * Overwrites sdf_nodes.  Only enqueues work. */
int nf_geom_sdf(nf_grid *g, const float *params_host, int K, int N, int M, int flags, float *sdf_nodes);

/* gparams_host[a] = sum over nodes of gsdf_nodes * d phi / d params[a] ("back-propagating dJ/dS first
 * through the SDF phi then through the distance computation"): the reverse of nf_geom_sdf, gsdf_nodes e.g. from
 * nf_weights_adjoint.  2 + K (2 + 2N) doubles, overwritten.  Synchronises the stream. */
int nf_geom_sdf_adjoint(nf_grid *g, const float *params_host, int K, int N, int M, int flags, const float *gsdf_nodes,
                        double *gparams_host);

/* CSG on solids ("Union and intersection"; phi > 0 = fluid, so the union of two solids is min(a, b), the
 * intersection max(a, b): R29).  Node arrays; out may alias a or b.  The adjoint routes gout to the operand that
 * supplied the value (ties: a) and writes 0 to the other; ga, gb may alias gout but not each other. */
int nf_geom_csg(nf_grid *g, int op, const float *a, const float *b, float *out);
int nf_geom_csg_adjoint(nf_grid *g, int op, const float *a, const float *b, const float *gout, float *ga, float *gb);

/* Solid velocity of the moving geometry params(t), d params / dt = pdot ("SDF phi^{n+1} and velocity
 * u_s^{n+1} can be derived from the solid geometry", L132): at every face centre of each family, the velocity of the
 * closest point q of the section's polygon at that height -- q's edge and edge parameter held fixed -- along the
 * in-plane unit normal nh: U_s = (nh . qdot) nh (x and y components; w = 0); where the slab term of R28 is the active
 * one the surface is a cap moving at (0, 0, z0dot) or (0, 0, z1dot) (R30).  Only faces with d <= band (physical
 * units; INFINITY = all) are written, the others keep their values: several moving parts = one call each.
 * us / vs / ws: MAC face layout, any may be NULL (skipped).  Only enqueues work. */
int nf_geom_velocity(nf_grid *g, const float *params_host, const float *pdot_host, int K, int N, int M, float band,
                     float *us, float *vs, float *ws);

/* gpdot_host = J^T (gus, gvs, gws), J = d U_s / d pdot of nf_geom_velocity with the same band (U_s is linear in
 * pdot; its dependence on params through q and nh is not differentiated: R31).  gus / gvs / gws may be NULL (= 0),
 * e.g. from nf_project_adjoint's gus_*.  2 + K (2 + 2N) doubles, overwritten.  Synchronises the stream. */
int nf_geom_velocity_adjoint(nf_grid *g, const float *params_host, int K, int N, int M, float band, const float *gus,
                             const float *gvs, const float *gws, double *gpdot_host);

/* Apply A to a cell array (q = A p, homogeneous ghosts) -- exposed for tests and kernel benchmarks. */
int nf_apply_A(nf_grid *g, const float *p, float *q);
/* One V-cycle z = M^{-1} r (zero initial guess) -- exposed for tests and kernel benchmarks. */
int nf_vcycle(nf_grid *g, const float *r, float *z);

/* Host-buffer variants: the same operations through HOST pointers; the host->device and device->host
 * copies run on the handle's stream inside the call, which returns after the results are in host memory. */
int nf_project_host(nf_grid *g, float *u, float *v, float *w, float *p, float tol, int maxit);
int nf_project_adjoint_host(nf_grid *g, float *gu, float *gv, float *gw, const float *p_saved,
                            const float *uhat_u, const float *uhat_v, const float *uhat_w, float tol, int maxit);

/* The *_host calls copy H2D on one stream, compute on the handle's stream and copy D2H on a third, ordered by
 * events.  By default they return when the host arrays hold the results.  nf_set_host_async(g, 1): they return as
 * soon as the work is enqueued (the solve itself still ends before the return: the host drives it), so the D2H of one
 * call overlaps the H2D and the kernels of the next; the host arrays are valid after nf_host_sync(g), which waits
 * for every stream of the handle. */
int nf_set_host_async(nf_grid *g, int on);
int nf_host_sync(nf_grid *g);

/* Info about the last solve on this handle.  Synchronises the handle's stream.
 * relres = ||r||_2/||rhs||_2 as tracked by the solver; ms = device time of the solve (CUDA events). */
int nf_last_solve_info(nf_grid *g, int *iters, float *relres, float *ms);
/* Number of multigrid levels; number of active cells; 1 if no Dirichlet domain face carries an open weight (every
 * component is then singular, R12; nf_grid_components gives the per-component count). */
int nf_grid_info(nf_grid *g, int *levels, long long *active_cells, int *singular);
/* Fluid components of the current weights (R12): A = c G^T S G is block diagonal over the connected components of the
 * active cells (cells joined by faces with alpha > 0; found on the device by nf_set_solid / nf_set_weights).  A
 * component without an open face on a Dirichlet domain boundary is singular: every solve removes the mean of the
 * right-hand side over it (compatibility) and returns a pressure with zero mean over it (gauge) -- the paper is silent;
 * SURVEY.md 8c.1.  *components = number of components, *singular_components = those that are singular. */
int nf_grid_components(nf_grid *g, int *components, int *singular_components);
/* Per-kernel-class device timing (CUDA events around every launch on the handle's stream; adds launch overhead, so
 * use it on extra steps, not on timed ones).  nf_profile_enable(g,1) clears the counters and starts recording;
 * nf_profile_get synchronises the stream and returns the accumulated milliseconds and launch count of class idx
 * (0 <= idx < number of classes; NF_ERR_INVALID beyond).  *name points to static storage. */
int nf_profile_enable(nf_grid *g, int on);
int nf_profile_get(nf_grid *g, int idx, const char **name, double *ms, long long *launches);
/* Kernels launched by this handle since creation (for bench.py's gpu_launches). */
long long nf_launch_count(nf_grid *g);
/* Last error message of this handle (static storage inside the handle; "" if none). */
const char *nf_last_error(nf_grid *g);

/* The reduction of nf_max_speed (R24) for callers that must not allocate -- code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No handle (nf_grid_create allocates), no
 * cudaMalloc / cudaFree / allocating library call, no stream synchronisation: two kernels are enqueued on cuda_stream
 * (a cudaStream_t; NULL = legacy stream 0) of the CURRENT device and *max_abs_dev -- a DEVICE pointer to one float,
 * owned by the caller -- receives max over all faces of |u|, |v|, |w| (a NaN propagates) when they have run.
 * u, v, w: DEVICE arrays in the MAC layout of this header, (nx+1) ny nz, nx (ny+1) nz, nx ny (nz+1) floats, read only.
 * Scratch: a fixed 64 KB array in the library's device image (one per GPU that loads the library, held until the
 * process exits): one partial maximum per 16384 faces, so u + v + w faces <= 268 435 456 (cubes up to about 440^3;
 * 256^3 uses 3 084 of the 16 384 partials).  Larger grids, NULL pointers and non-positive extents return
 * NF_ERR_INVALID; NF_ERR_CUDA if the array's address cannot be resolved or a launch fails; nf_static_last_error()
 * (thread-local static storage) says which.  The array's address is resolved on the first call on each device
 * (cudaGetSymbolAddress: make that call outside a capture).  All calls on a device SHARE the array and it keeps the
 * last call's contents: nothing in it needs clearing (a call reads only the partials it has just written), calls on
 * one stream are ordered, but calls that OVERLAP on the GPU -- different streams, concurrently replayed graphs -- race
 * on it and must be serialised by the caller. */
int nf_max_speed_static(const float *u, const float *v, const float *w, int nx, int ny, int nz, void *cuda_stream,
                        float *max_abs_dev);
const char *nf_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* NF_H_ */
