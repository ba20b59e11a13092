// nf_api.cu -- the C ABI (include/nf.h): handle management, argument checking, and the composition of the
// hot-path calls from the kernels in nf_weights.cu / nf_solver.cu / nf_project.cu / nf_advect.cu.
#include <algorithm>
#include <new>

#include "nf_internal.cuh"

#define NF_CHECK_HANDLE(g) \
  do {                     \
    if (!(g)) return NF_ERR_INVALID; \
    (g)->err.clear();      \
  } while (0)

extern "C" const char *nf_version(void) { return "nf-b200 0.1 (sm_100a)"; }

template <typename T>
static cudaError_t dalloc(T **p, size_t n) {
  return cudaMalloc((void **)p, (n ? n : 1) * sizeof(T));
}

static void free_all(nf_grid *g) {
  for (int l = 0; l < NF_MAX_LEVELS; ++l) {
    NfLevel &L = g->lv[l];
    cudaFree(L.ax); cudaFree(L.ay); cudaFree(L.az); cudaFree(L.code); cudaFree(L.idg); cudaFree(L.pk); cudaFree(L.z); cudaFree(L.r);
  }
  cudaFree(g->us); cudaFree(g->vs); cudaFree(g->ws); cudaFree(g->sdf);
  cudaFree(g->p); cudaFree(g->q); cudaFree(g->xtmp); cudaFree(g->p2); cudaFree(g->b0); cudaFree(g->ecorr); cudaFree(g->rtrue); cudaFree(g->r_alt); cudaFree(g->tailpack); cudaFree(g->tailinv);
  cudaFree(g->fu); cudaFree(g->fv); cudaFree(g->fw);
  cudaFree(g->st); cudaFree(g->d_counts); cudaFree(g->geom_par); cudaFree(g->geom_grad);
  nf_components_free(g);
  nf_mg_free_batch(g);
  if (g->hst) cudaFreeHost((void *)g->hst);
  if (g->h_counts) cudaFreeHost(g->h_counts);
  if (g->ev0) cudaEventDestroy(g->ev0);
  if (g->ev1) cudaEventDestroy(g->ev1);
  if (g->ev_meta) cudaEventDestroy(g->ev_meta);
  for (cudaEvent_t e : g->prof_pool) cudaEventDestroy(e);
  if (g->hs_u) {
    cudaStreamDestroy(g->s_h2d); cudaStreamDestroy(g->s_d2h);
    cudaEventDestroy(g->ev_in); cudaEventDestroy(g->ev_comp); cudaEventDestroy(g->ev_out_proj); cudaEventDestroy(g->ev_out_adj);
  }
  cudaFree(g->hs_u); cudaFree(g->hs_v); cudaFree(g->hs_w); cudaFree(g->hs_p);
  cudaFree(g->hs_a); cudaFree(g->hs_b); cudaFree(g->hs_c); cudaFree(g->hs_d);
}

extern "C" int nf_grid_create(int nx, int ny, int nz, float dx, nf_grid **out) {
  if (!out) return NF_ERR_INVALID;
  *out = nullptr;
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0.0f)) return NF_ERR_INVALID;
  // every array is addressed with 32-bit offsets (x rows padded to a multiple of 4): < 2^32 slots
  if ((long long)(nx + 8) * (ny + 1) * (long long)(nz + 1) >= (1LL << 32)) return NF_ERR_INVALID;
  nf_grid *g = new (std::nothrow) nf_grid();
  if (!g) return NF_ERR_ALLOC;
  g->nx = nx; g->ny = ny; g->nz = nz; g->dx = dx; g->dt_over_rho = 1.0f;
  for (int f = 0; f < 6; ++f) { g->bc_type[f] = NF_BC_CLOSED; g->bc_val[f] = 0.0f; }
  g->stream = 0;
  g->nu_pre = 1; g->nu_post = 1;
  // Sweeps on the coarse levels (nf_set_coarse_sweeps overrides): chosen from measurements.  The
  // extra sweeps run as phases of the cooperative coarse kernel, whose cost is latency and does not shrink with the
  // grid, while the fine level's cost does: only large grids afford them.  Forward + adjoint solve, ms, sweeps on
  // (level 1, the levels below):
  //   channel-gate 256^3: (1,1) 22.8  (1,2) 18.1  (2,2) 17.7  (2,3) 16.5  (3,3) 16.9;  sphere field 384^3 / 512^3: -10 % / -8 %
  //   channel-gate 128^3: (1,1) 4.94  (1,2) 4.68;  64^3: 2.58 / 2.63;  but chamber 128^3 x 50 steps 7.09 -> 7.44 ms per
  //   step, plates 64^3 2.75 -> 3.05, sphere field 64^3 / 128^3 + 10 % / + 13 % with (1,2): small grids keep V(1,1)
  //   channel-gate 128^3 / 160^3 / 192^3 (final kernels): (1,1) 4.26 / 7.08 / 10.15, (2,3) 4.78 / 6.78 / 8.57: the switch sits at 3 M cells
  {
    const bool large = (long long)nx * ny * nz >= 3000000LL;
    g->nu_l1 = large ? 2 : 1;
    g->nu_deep = large ? 3 : 1;
  }
  // Over-relaxation of the sweeps on every level below the finest (nf_set_coarse_relaxation overrides): free of phases
  // and passes.  Forward + adjoint solve, ms, omega = 1 / 1.3 / 1.4 / 1.5 / 1.6 on the levels from 2 down (level 1 added later): channel-gate 256^3 15.7 / 15.5 / 14.3 / 14.3 /
  // 15.0, 128^3 4.36 / 4.20 / 4.09 / 3.96 / 3.96, 64^3 2.42 / 2.32 / 2.30 / 2.18 / 2.23; sphere field 128^3 2.34 / 2.25 / 2.26 /
  // 2.42 / 2.57 (256^3: 6.1 throughout); chamber 128^3 4.01 / 4.05 / 3.91 / 4.17 / 4.30.
  g->omega_deep = 1.4f;
  g->force_generic = false; g->refresh = true; g->warm = false; g->host_async = false;
  g->weights_set = g->have_sdf = g->have_us = false;
  g->singular = 1; g->singular_info = 1; g->nact = 0; g->ncomp = 0; g->nsing = 0; g->gauge_mode = 1;
  g->plo = nullptr; g->lo_valid = false;
  g->d_coarse = nullptr; g->h_coarse = nullptr; g->cbar = nullptr; g->cbar_count = 0; g->meta_pending = false;
  g->comp = nullptr; g->cc_cnt = nullptr; g->cc_regular = nullptr; g->cc_sums = nullptr; g->cc_meta = nullptr; g->h_cc_meta = nullptr;
  g->last_iters = 0; g->last_relres = 0.0f; g->last_timed = false; g->launches = 0;
  g->prof_on = false;
  for (int c = 0; c < NFK_COUNT; ++c) { g->prof_ms[c] = 0.0; g->prof_n[c] = 0; }
  for (int l = 0; l < NF_MAX_LEVELS; ++l) g->lv[l] = NfLevel{};
  // hierarchy: halve while every extent is even and stays >= 4
  int lx = nx, ly = ny, lz = nz, nl = 0;
  float c = g->dt_over_rho / dx;
  bool ok = true;
  for (;;) {
    NfLevel &L = g->lv[nl];
    L.nx = lx; L.ny = ly; L.nz = lz;
    L.pax = (lx + 1 + 3) & ~3;
    L.ncell = (long long)lx * ly * lz;
    L.c = c;
    ok = ok && dalloc(&L.ax, (size_t)lz * ly * L.pax) == cudaSuccess;
    ok = ok && dalloc(&L.ay, (size_t)lz * (ly + 1) * lx) == cudaSuccess;
    ok = ok && dalloc(&L.az, (size_t)(lz + 1) * ly * lx) == cudaSuccess;
    ok = ok && dalloc(&L.code, (size_t)L.ncell + 16) == cudaSuccess;
    ok = ok && dalloc(&L.idg, (size_t)L.ncell) == cudaSuccess;
    ok = ok && dalloc(&L.z, (size_t)L.ncell) == cudaSuccess;
    ok = ok && dalloc(&L.r, (size_t)L.ncell) == cudaSuccess;
    if (ok) ok = cudaMemset(L.ax, 0, (size_t)lz * ly * L.pax * sizeof(float)) == cudaSuccess;
    ++nl;
    if (!ok || nl >= NF_MAX_LEVELS) break;
    // 2-D mode (nz == 1): x and y coarsen, z stays one layer
    const bool flat = nz == 1;
    L.fz = flat ? 1 : 2;
    // Extents halve, rounding UP (a coarse cell at an odd edge has one child along that axis; the absent children
    // count as solid), while every coarse extent stays >= 4 -- except that a level with more than 128 cells (too many
    // for the direct coarsest solve of nf_mg.cu) is halved once more if it can be: 48^3 ends at 3^3 instead of 6^3,
    // 256^3 at 4^3, 250^3 goes 125, 63, 32, 16, 8, 4 (before: it stopped at 125^3 and needed 175 iterations).
    const int lim = L.ncell > 128 ? 2 : 4;
    const int hx = (lx + 1) / 2, hy = (ly + 1) / 2, hz = flat ? 1 : (lz + 1) / 2;
    if (hx < lim || hy < lim || (!flat && hz < lim)) break;
    if (hx == lx && hy == ly && hz == lz) break;
    lx = hx; ly = hy; lz = hz;
    c *= 0.25f;
  }
  g->nlev = nl;
  nf_mg_plan(g);
  // (2-D mode runs the 4-cell bodies on every level above the tail: the packed per-cell phases assume 2x2x2 children)
  for (int l = 2; l < g->tail && l < nl && nz != 1; ++l) ok = ok && dalloc(&g->lv[l].pk, 8 * (size_t)g->lv[l].ncell) == cudaSuccess;
  {
    size_t tc = 0;
    for (int l = g->tail; l < nl; ++l) tc += (size_t)g->lv[l].ncell;
    ok = ok && dalloc(&g->tailpack, 8 * tc) == cudaSuccess;
    ok = ok && dalloc(&g->tailinv, 128 * 128 + 4 + 136) == cudaSuccess;  // the inverse + component labels (nf_mg.cu)
  }
  const size_t nc = nf_nc(g);
  ok = ok && dalloc(&g->us, nf_nu(g)) == cudaSuccess && dalloc(&g->vs, nf_nv(g)) == cudaSuccess &&
       dalloc(&g->ws, nf_nw(g)) == cudaSuccess && dalloc(&g->sdf, nf_nn(g)) == cudaSuccess;
  ok = ok && dalloc(&g->p, nc) == cudaSuccess && dalloc(&g->q, nc) == cudaSuccess &&
       dalloc(&g->xtmp, nc) == cudaSuccess && dalloc(&g->p2, nc) == cudaSuccess &&
       dalloc(&g->b0, nc) == cudaSuccess && dalloc(&g->ecorr, nc) == cudaSuccess && dalloc(&g->rtrue, nc) == cudaSuccess && dalloc(&g->r_alt, nc) == cudaSuccess;
  ok = ok && dalloc(&g->fu, nf_nu(g)) == cudaSuccess && dalloc(&g->fv, nf_nv(g)) == cudaSuccess &&
       dalloc(&g->fw, nf_nw(g)) == cudaSuccess;
  ok = ok && dalloc(&g->st, 1) == cudaSuccess && dalloc(&g->d_counts, 2) == cudaSuccess;
  ok = ok && nf_components_alloc(g) == NF_OK;
  ok = ok && dalloc(&g->geom_par, 2 * (size_t)NF_GEOM_MAXP) == cudaSuccess && dalloc(&g->geom_grad, (size_t)NF_GEOM_MAXP) == cudaSuccess;
  ok = ok && cudaHostAlloc((void **)&g->hst, NF_RING * sizeof(NfHostStatus), cudaHostAllocMapped) == cudaSuccess;
  ok = ok && cudaHostGetDevicePointer((void **)&g->hst_dev, (void *)g->hst, 0) == cudaSuccess;
  ok = ok && cudaHostAlloc((void **)&g->h_counts, 2 * sizeof(double), cudaHostAllocDefault) == cudaSuccess;
  ok = ok && cudaEventCreate(&g->ev0) == cudaSuccess && cudaEventCreate(&g->ev1) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&g->ev_meta, cudaEventDisableTiming) == cudaSuccess;
  if (ok) {
    for (int s = 0; s < NF_RING; ++s) { g->hst[s].seq = 0; g->hst[s].done = 0; g->hst[s].converged = 0; }
    ok = nf_solver_init(g) == NF_OK;
  }
  if (!ok) {
    cudaGetLastError();
    free_all(g);
    delete g;
    return NF_ERR_ALLOC;
  }
  *out = g;
  return NF_OK;
}

extern "C" void nf_grid_destroy(nf_grid *g) {
  if (!g) return;
  cudaStreamSynchronize(g->stream);
  free_all(g);
  delete g;
}

extern "C" int nf_set_stream(nf_grid *g, void *cuda_stream) {
  NF_CHECK_HANDLE(g);
  g->stream = (cudaStream_t)cuda_stream;
  return NF_OK;
}

extern "C" int nf_set_dt_rho(nf_grid *g, float dt_over_rho) {
  NF_CHECK_HANDLE(g);
  if (!(dt_over_rho > 0.0f)) return NF_ERR_INVALID;
  g->dt_over_rho = dt_over_rho;
  float c = dt_over_rho / g->dx;
  bool changed = false;
  for (int l = 0; l < g->nlev; ++l) { changed = changed || g->lv[l].c != c; g->lv[l].c = c; c *= 0.25f; }
  // the inverse diagonals and the packed tail operator carry c: rebuild them from the current weights
  if (changed && g->weights_set) return nf_build_hierarchy(g);
  return NF_OK;
}

extern "C" int nf_set_domain_bc(nf_grid *g, int face, int type, float p_value) {
  NF_CHECK_HANDLE(g);
  if (face < 0 || face > 5 || (type != NF_BC_CLOSED && type != NF_BC_DIRICHLET)) return NF_ERR_INVALID;
  g->bc_type[face] = type;
  g->bc_val[face] = p_value;
  g->weights_set = false;  // closed walls force alpha = 0: the weights must be rebuilt
  return NF_OK;
}

extern "C" int nf_set_solver_options(nf_grid *g, int nu_pre, int nu_post, int flags) {
  NF_CHECK_HANDLE(g);
  if (nu_pre < 1 || nu_post < 1 || nu_pre > 8 || nu_post > 8 || flags < 0 || flags > 15) return NF_ERR_INVALID;
  g->nu_pre = nu_pre; g->nu_post = nu_post; g->force_generic = (flags & 2) != 0; g->refresh = (flags & 4) == 0; g->warm = (flags & 8) != 0;
  return NF_OK;
}

extern "C" int nf_set_coarse_sweeps(nf_grid *g, int nu_level1, int nu_deeper) {
  NF_CHECK_HANDLE(g);
  if (nu_level1 < 1 || nu_level1 > 8 || nu_deeper < 1 || nu_deeper > 8) return NF_ERR_INVALID;
  g->nu_l1 = nu_level1; g->nu_deep = nu_deeper;
  return g->weights_set ? nf_mg_upload_coarse(g) : NF_OK;  // (the batched kernel reads the sweep count from the device table)
}

extern "C" int nf_set_pressure_lo(nf_grid *g, float *lo_cells) {
  NF_CHECK_HANDLE(g);
  g->plo = lo_cells;
  g->lo_valid = false;
  return NF_OK;
}

extern "C" int nf_set_solid(nf_grid *g, const float *sdf_nodes, const float *us, const float *vs, const float *ws) {
  NF_CHECK_HANDLE(g);
  if (!sdf_nodes) return NF_ERR_INVALID;
  NF_TRY(nf_weights_from_sdf(g, sdf_nodes));
  NF_TRY(nf_store_solid_velocity(g, us, vs, ws));
  return nf_build_hierarchy(g);
}

extern "C" int nf_set_weights(nf_grid *g, const float *au, const float *av, const float *aw) {
  NF_CHECK_HANDLE(g);
  if (!au || !av || !aw) return NF_ERR_INVALID;
  NF_TRY(nf_weights_from_user(g, au, av, aw));
  return nf_build_hierarchy(g);
}

extern "C" int nf_get_weights(nf_grid *g, float *au, float *av, float *aw) {
  NF_CHECK_HANDLE(g);
  if (!g->weights_set) return NF_ERR_STATE;
  return nf_weights_to_user(g, au, av, aw);
}

extern "C" int nf_set_solid_velocity(nf_grid *g, const float *us, const float *vs, const float *ws) {
  NF_CHECK_HANDLE(g);
  return nf_store_solid_velocity(g, us, vs, ws);
}

static int solve_timed(nf_grid *g, const float *src, float *x, float tol, int maxit, bool warm) {
  if (!(tol > 0.0f) || maxit < 1) return NF_ERR_INVALID;
  NF_TRY(nf_meta_sync(g));
  NF_CUDA(g, cudaEventRecord(g->ev0, g->stream));
  NF_TRY(nf_solve_prepare_from(g, src, tol, maxit));
  int rc = nf_solve_run(g, x, tol, maxit, warm);
  if (rc < 0) return rc;
  NF_CUDA(g, cudaEventRecord(g->ev1, g->stream));
  g->last_timed = true;
  return rc;
}

extern "C" int nf_solve(nf_grid *g, const float *rhs, float *p, float tol, int maxit) {
  NF_CHECK_HANDLE(g);
  if (!rhs || !p || rhs == p) return NF_ERR_INVALID;
  if (!g->weights_set) return NF_ERR_STATE;
  return solve_timed(g, rhs, p, tol, maxit, g->warm);
}

extern "C" int nf_project(nf_grid *g, float *u, float *v, float *w, float *p, float tol, int maxit) {
  NF_CHECK_HANDLE(g);
  if (!u || !v || !w || !p) return NF_ERR_INVALID;
  if (!g->weights_set) return NF_ERR_STATE;
  NF_TRY(nf_rhs_impl(g, u, v, w));
  int rc = solve_timed(g, nullptr, p, tol, maxit, g->warm);
  if (rc < 0) return rc;
  NF_TRY(nf_grad_subtract_impl(g, u, v, w, p));
  return rc;
}

extern "C" int nf_project_adjoint(nf_grid *g, float *gu, float *gv, float *gw, const float *p_saved,
                                  const float *uhat_u, const float *uhat_v, const float *uhat_w, float *galpha_u,
                                  float *galpha_v, float *galpha_w, float *gus_u, float *gus_v, float *gus_w,
                                  float *y_out, float tol, int maxit) {
  NF_CHECK_HANDLE(g);
  if (!gu || !gv || !gw) return NF_ERR_INVALID;
  const bool want_ga = galpha_u || galpha_v || galpha_w;
  if (want_ga && !(galpha_u && galpha_v && galpha_w && p_saved && uhat_u && uhat_v && uhat_w)) return NF_ERR_INVALID;
  const bool want_gs = gus_u || gus_v || gus_w;
  if (want_gs && !(gus_u && gus_v && gus_w)) return NF_ERR_INVALID;
  if (!g->weights_set) return NF_ERR_STATE;
  float *y = y_out ? y_out : g->xtmp;
  NF_TRY(nf_adjoint_rhs_impl(g, gu, gv, gw));
  int rc = solve_timed(g, nullptr, y, tol, maxit, g->warm && y_out != nullptr);  // (never from internal scratch)
  if (rc < 0) return rc;
  NF_TRY(nf_adjoint_finish_impl(g, gu, gv, gw, y, p_saved, uhat_u, uhat_v, uhat_w, galpha_u, galpha_v, galpha_w,
                                gus_u, gus_v, gus_w));
  return rc;
}

// ---- batched entry points ------------------------------------------------------------------
// Groups of environments the batched kernels can take (equal extents, one stream, fused path, cooperative grid resident);
// anything else is solved one handle at a time -- the results are the same, only the number of launches differs.
template <class PRE, class POST>
static int batch_drive(nf_grid *const *gs, int n, float *const *x, float tol, int maxit, int *status, PRE pre, POST post) {
  if (!gs || n < 1 || !x || !(tol > 0.0f) || maxit < 1) return NF_ERR_INVALID;
  for (int e = 0; e < n; ++e) {
    if (!gs[e] || !x[e]) return NF_ERR_INVALID;
    gs[e]->err.clear();
    if (!gs[e]->weights_set) return NF_ERR_STATE;
  }
  for (int e = 0; e < n; ++e) NF_TRY(nf_meta_sync(gs[e]));
  int worst = NF_OK;
  int sms = 148, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  int e0 = 0;
  while (e0 < n) {
    int cnt = std::min(n - e0, NF_BATCH_MAX);
    if (gs[e0]->coarse_ctas > 0) cnt = std::min(cnt, std::max(1, sms / gs[e0]->coarse_ctas));
    nf_grid *G[NF_BATCH_MAX];
    float *X[NF_BATCH_MAX];
    int st[NF_BATCH_MAX];
    for (int e = 0; e < cnt; ++e) { G[e] = gs[e0 + e]; X[e] = x[e0 + e]; st[e] = NF_OK; }
    for (int e = 0; e < cnt; ++e) NF_TRY(pre(e0 + e));  // right-hand sides into lv[0].r
    if (cnt > 1 && nf_batch_ok(G, cnt)) {
      NF_TRY(nf_solve_batch_impl(G, cnt, nullptr, X, tol, maxit, st));
    } else {
      for (int e = 0; e < cnt; ++e) {
        NF_TRY(nf_solve_prepare_from(G[e], nullptr, tol, maxit));
        int rc = nf_solve_run(G[e], X[e], tol, maxit, false);
        if (rc < 0) return rc;
        st[e] = rc;
      }
    }
    for (int e = 0; e < cnt; ++e) {
      NF_TRY(post(e0 + e));
      if (status) status[e0 + e] = st[e];
      worst = std::max(worst, st[e]);
    }
    e0 += cnt;
  }
  return worst;
}

extern "C" int nf_solve_batch(nf_grid *const *g, int n, const float *const *rhs, float *const *p, float tol, int maxit,
                              int *status) {
  if (!rhs) return NF_ERR_INVALID;
  return batch_drive(g, n, p, tol, maxit, status,
                     [&](int e) -> int {
                       if (!rhs[e] || rhs[e] == p[e]) return NF_ERR_INVALID;
                       nf_grid *h = g[e];
                       NF_CUDA(h, cudaMemcpyAsync(h->lv[0].r, rhs[e], nf_nc(h) * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
                       return NF_OK;
                     },
                     [&](int) -> int { return NF_OK; });
}

extern "C" int nf_project_batch(nf_grid *const *g, int n, float *const *u, float *const *v, float *const *w,
                                float *const *p, float tol, int maxit, int *status) {
  if (!u || !v || !w) return NF_ERR_INVALID;
  return batch_drive(g, n, p, tol, maxit, status,
                     [&](int e) -> int {
                       if (!u[e] || !v[e] || !w[e]) return NF_ERR_INVALID;
                       return nf_rhs_impl(g[e], u[e], v[e], w[e]);
                     },
                     [&](int e) -> int { return nf_grad_subtract_impl(g[e], u[e], v[e], w[e], p[e]); });
}

extern "C" int nf_project_adjoint_batch(nf_grid *const *g, int n, float *const *gu, float *const *gv, float *const *gw,
                                        const float *const *p_saved, const float *const *uhat_u,
                                        const float *const *uhat_v, const float *const *uhat_w, float *const *galpha_u,
                                        float *const *galpha_v, float *const *galpha_w, float *const *gus_u,
                                        float *const *gus_v, float *const *gus_w, float *const *y, float tol, int maxit,
                                        int *status) {
  if (!gu || !gv || !gw || !y) return NF_ERR_INVALID;
  const bool want_ga = galpha_u || galpha_v || galpha_w;
  if (want_ga && !(galpha_u && galpha_v && galpha_w && p_saved && uhat_u && uhat_v && uhat_w)) return NF_ERR_INVALID;
  const bool want_gs = gus_u || gus_v || gus_w;
  if (want_gs && !(gus_u && gus_v && gus_w)) return NF_ERR_INVALID;
  return batch_drive(g, n, y, tol, maxit, status,
                     [&](int e) -> int {
                       if (!gu[e] || !gv[e] || !gw[e]) return NF_ERR_INVALID;
                       return nf_adjoint_rhs_impl(g[e], gu[e], gv[e], gw[e]);
                     },
                     [&](int e) -> int {
                       return nf_adjoint_finish_impl(g[e], gu[e], gv[e], gw[e], y[e], want_ga ? p_saved[e] : nullptr,
                                                     want_ga ? uhat_u[e] : nullptr, want_ga ? uhat_v[e] : nullptr,
                                                     want_ga ? uhat_w[e] : nullptr, want_ga ? galpha_u[e] : nullptr,
                                                     want_ga ? galpha_v[e] : nullptr, want_ga ? galpha_w[e] : nullptr,
                                                     want_gs ? gus_u[e] : nullptr, want_gs ? gus_v[e] : nullptr,
                                                     want_gs ? gus_w[e] : nullptr);
                     });
}

extern "C" int nf_viscosity(nf_grid *g, float *u, float *v, float *w, float nu, float dt) {
  NF_CHECK_HANDLE(g);
  if (!u || !v || !w || !(nu >= 0.0f) || !(dt >= 0.0f)) return NF_ERR_INVALID;
  return nf_viscosity_impl(g, u, v, w, nu, dt);
}

extern "C" int nf_max_speed(nf_grid *g, const float *u, const float *v, const float *w, float *max_abs_host) {
  NF_CHECK_HANDLE(g);
  if (!u || !v || !w || !max_abs_host) return NF_ERR_INVALID;
  return nf_max_speed_impl(g, u, v, w, max_abs_host);
}

// ---- NEXT-2: parametric geometry (nf_geom.cu) ---------------------------------------------------------------------
extern "C" int nf_geom_sdf(nf_grid *g, const float *params_host, int K, int N, int M, int flags, float *sdf_nodes) {
  NF_CHECK_HANDLE(g);
  if (!sdf_nodes || (flags & ~NF_GEOM_COMPLEMENT)) return NF_ERR_INVALID;
  return nf_geom_sdf_impl(g, params_host, K, N, M, flags, sdf_nodes);
}

extern "C" int nf_geom_sdf_adjoint(nf_grid *g, const float *params_host, int K, int N, int M, int flags,
                                   const float *gsdf_nodes, double *gparams_host) {
  NF_CHECK_HANDLE(g);
  if (!gsdf_nodes || !gparams_host || (flags & ~NF_GEOM_COMPLEMENT)) return NF_ERR_INVALID;
  return nf_geom_sdf_adjoint_impl(g, params_host, K, N, M, flags, gsdf_nodes, gparams_host);
}

extern "C" int nf_geom_velocity(nf_grid *g, const float *params_host, const float *pdot_host, int K, int N, int M,
                                float band, float *us, float *vs, float *ws) {
  NF_CHECK_HANDLE(g);
  if (!pdot_host || band != band) return NF_ERR_INVALID;
  return nf_geom_velocity_impl(g, params_host, pdot_host, K, N, M, band, us, vs, ws);
}

extern "C" int nf_geom_velocity_adjoint(nf_grid *g, const float *params_host, int K, int N, int M, float band,
                                        const float *gus, const float *gvs, const float *gws, double *gpdot_host) {
  NF_CHECK_HANDLE(g);
  if (!gpdot_host || band != band) return NF_ERR_INVALID;
  return nf_geom_velocity_adjoint_impl(g, params_host, K, N, M, band, gus, gvs, gws, gpdot_host);
}

extern "C" int nf_geom_csg(nf_grid *g, int op, const float *a, const float *b, float *out) {
  NF_CHECK_HANDLE(g);
  if (!a || !b || !out || (op != NF_CSG_UNION && op != NF_CSG_INTERSECTION)) return NF_ERR_INVALID;
  return nf_geom_csg_impl(g, op, a, b, out);
}

extern "C" int nf_geom_csg_adjoint(nf_grid *g, int op, const float *a, const float *b, const float *gout, float *ga,
                                   float *gb) {
  NF_CHECK_HANDLE(g);
  if (!a || !b || !gout || !ga || !gb || ga == gb || (op != NF_CSG_UNION && op != NF_CSG_INTERSECTION)) return NF_ERR_INVALID;
  return nf_geom_csg_adjoint_impl(g, op, a, b, gout, ga, gb);
}

extern "C" int nf_advect(nf_grid *g, float *u, float *v, float *w, float dt) {
  NF_CHECK_HANDLE(g);
  if (!u || !v || !w) return NF_ERR_INVALID;
  return nf_advect_impl(g, u, v, w, dt);
}

extern "C" int nf_advect_adjoint(nf_grid *g, const float *u0, const float *v0, const float *w0, float *gu, float *gv,
                                 float *gw, float dt) {
  NF_CHECK_HANDLE(g);
  if (!u0 || !v0 || !w0 || !gu || !gv || !gw) return NF_ERR_INVALID;
  return nf_advect_adjoint_impl(g, u0, v0, w0, gu, gv, gw, dt);
}

extern "C" int nf_weights_adjoint(nf_grid *g, const float *galpha_u, const float *galpha_v, const float *galpha_w,
                                  float *gsdf_nodes) {
  NF_CHECK_HANDLE(g);
  if (!galpha_u || !galpha_v || !galpha_w || !gsdf_nodes) return NF_ERR_INVALID;
  if (!g->have_sdf) return NF_ERR_STATE;
  return nf_weights_adjoint_impl(g, galpha_u, galpha_v, galpha_w, gsdf_nodes);
}

extern "C" int nf_apply_A(nf_grid *g, const float *p, float *q) {
  NF_CHECK_HANDLE(g);
  if (!p || !q || p == q) return NF_ERR_INVALID;
  if (!g->weights_set) return NF_ERR_STATE;
  return nf_apply_A_impl(g, p, q);
}

extern "C" int nf_vcycle(nf_grid *g, const float *r, float *z) {
  NF_CHECK_HANDLE(g);
  if (!r || !z) return NF_ERR_INVALID;
  if (!g->weights_set) return NF_ERR_STATE;
  NF_TRY(nf_meta_sync(g));
  const size_t bytes = nf_nc(g) * sizeof(float);
  NF_CUDA(g, cudaMemcpyAsync(g->lv[0].r, r, bytes, cudaMemcpyDeviceToDevice, g->stream));
  NF_TRY(nf_vcycle_impl(g, false, 0));
  NF_CUDA(g, cudaMemcpyAsync(z, g->lv[0].z, bytes, cudaMemcpyDeviceToDevice, g->stream));
  return NF_OK;
}

// ---- host-buffer variants ------------------------------------------------------------------------------------
static int ensure_host_staging(nf_grid *g) {
  if (g->hs_u) return NF_OK;
  // device staging for the host entry points (the caller's arrays live in host memory)
  if (dalloc(&g->hs_u, nf_nu(g)) != cudaSuccess || dalloc(&g->hs_v, nf_nv(g)) != cudaSuccess ||
      dalloc(&g->hs_w, nf_nw(g)) != cudaSuccess || dalloc(&g->hs_p, nf_nc(g)) != cudaSuccess ||
      dalloc(&g->hs_a, nf_nu(g)) != cudaSuccess || dalloc(&g->hs_b, nf_nv(g)) != cudaSuccess ||
      dalloc(&g->hs_c, nf_nw(g)) != cudaSuccess || dalloc(&g->hs_d, nf_nc(g)) != cudaSuccess) {
    g->err = "host-variant staging allocation failed";
    return NF_ERR_ALLOC;
  }
  NF_CUDA(g, cudaStreamCreateWithFlags(&g->s_h2d, cudaStreamNonBlocking));
  NF_CUDA(g, cudaStreamCreateWithFlags(&g->s_d2h, cudaStreamNonBlocking));
  NF_CUDA(g, cudaEventCreateWithFlags(&g->ev_in, cudaEventDisableTiming));
  NF_CUDA(g, cudaEventCreateWithFlags(&g->ev_comp, cudaEventDisableTiming));
  NF_CUDA(g, cudaEventCreateWithFlags(&g->ev_out_proj, cudaEventDisableTiming));
  NF_CUDA(g, cudaEventCreateWithFlags(&g->ev_out_adj, cudaEventDisableTiming));
  return NF_OK;
}

extern "C" int nf_set_host_async(nf_grid *g, int on) {
  NF_CHECK_HANDLE(g);
  g->host_async = on != 0;
  return NF_OK;
}

extern "C" int nf_host_sync(nf_grid *g) {
  NF_CHECK_HANDLE(g);
  if (g->hs_u) {
    NF_CUDA(g, cudaStreamSynchronize(g->s_d2h));
    NF_CUDA(g, cudaStreamSynchronize(g->s_h2d));
  }
  NF_CUDA(g, cudaStreamSynchronize(g->stream));
  return NF_OK;
}

// H2D on its own stream (after the previous D2H out of the same staging buffers), compute on the handle's stream,
// D2H on a third: the two copy directions and the kernels of neighbouring calls overlap.
extern "C" int nf_project_host(nf_grid *g, float *u, float *v, float *w, float *p, float tol, int maxit) {
  NF_CHECK_HANDLE(g);
  if (!u || !v || !w || !p) return NF_ERR_INVALID;
  if (!g->weights_set) return NF_ERR_STATE;
  NF_TRY(ensure_host_staging(g));
  const size_t bu = nf_nu(g) * sizeof(float), bv = nf_nv(g) * sizeof(float), bw = nf_nw(g) * sizeof(float);
  NF_CUDA(g, cudaStreamWaitEvent(g->s_h2d, g->ev_out_proj, 0));
  NF_CUDA(g, cudaMemcpyAsync(g->hs_u, u, bu, cudaMemcpyHostToDevice, g->s_h2d));
  NF_CUDA(g, cudaMemcpyAsync(g->hs_v, v, bv, cudaMemcpyHostToDevice, g->s_h2d));
  NF_CUDA(g, cudaMemcpyAsync(g->hs_w, w, bw, cudaMemcpyHostToDevice, g->s_h2d));
  NF_CUDA(g, cudaEventRecord(g->ev_in, g->s_h2d));
  NF_CUDA(g, cudaStreamWaitEvent(g->stream, g->ev_in, 0));
  int rc = nf_project(g, g->hs_u, g->hs_v, g->hs_w, g->hs_p, tol, maxit);
  if (rc < 0) return rc;
  NF_CUDA(g, cudaEventRecord(g->ev_comp, g->stream));
  NF_CUDA(g, cudaStreamWaitEvent(g->s_d2h, g->ev_comp, 0));
  NF_CUDA(g, cudaMemcpyAsync(p, g->hs_p, nf_nc(g) * sizeof(float), cudaMemcpyDeviceToHost, g->s_d2h));
  NF_CUDA(g, cudaMemcpyAsync(u, g->hs_u, bu, cudaMemcpyDeviceToHost, g->s_d2h));
  NF_CUDA(g, cudaMemcpyAsync(v, g->hs_v, bv, cudaMemcpyDeviceToHost, g->s_d2h));
  NF_CUDA(g, cudaMemcpyAsync(w, g->hs_w, bw, cudaMemcpyDeviceToHost, g->s_d2h));
  NF_CUDA(g, cudaEventRecord(g->ev_out_proj, g->s_d2h));
  if (!g->host_async) NF_CUDA(g, cudaStreamSynchronize(g->s_d2h));
  return rc;
}

extern "C" int nf_project_adjoint_host(nf_grid *g, float *gu, float *gv, float *gw, const float *p_saved,
                                       const float *uhat_u, const float *uhat_v, const float *uhat_w, float tol,
                                       int maxit) {
  NF_CHECK_HANDLE(g);
  (void)p_saved; (void)uhat_u; (void)uhat_v; (void)uhat_w;  // only needed for dJ/dalpha, not produced here
  if (!gu || !gv || !gw) return NF_ERR_INVALID;
  if (!g->weights_set) return NF_ERR_STATE;
  NF_TRY(ensure_host_staging(g));
  const size_t bu = nf_nu(g) * sizeof(float), bv = nf_nv(g) * sizeof(float), bw = nf_nw(g) * sizeof(float);
  NF_CUDA(g, cudaStreamWaitEvent(g->s_h2d, g->ev_out_adj, 0));
  NF_CUDA(g, cudaMemcpyAsync(g->hs_a, gu, bu, cudaMemcpyHostToDevice, g->s_h2d));
  NF_CUDA(g, cudaMemcpyAsync(g->hs_b, gv, bv, cudaMemcpyHostToDevice, g->s_h2d));
  NF_CUDA(g, cudaMemcpyAsync(g->hs_c, gw, bw, cudaMemcpyHostToDevice, g->s_h2d));
  NF_CUDA(g, cudaEventRecord(g->ev_in, g->s_h2d));
  NF_CUDA(g, cudaStreamWaitEvent(g->stream, g->ev_in, 0));
  int rc = nf_project_adjoint(g, g->hs_a, g->hs_b, g->hs_c, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
                              nullptr, nullptr, nullptr, nullptr, nullptr, tol, maxit);
  if (rc < 0) return rc;
  NF_CUDA(g, cudaEventRecord(g->ev_comp, g->stream));
  NF_CUDA(g, cudaStreamWaitEvent(g->s_d2h, g->ev_comp, 0));
  NF_CUDA(g, cudaMemcpyAsync(gu, g->hs_a, bu, cudaMemcpyDeviceToHost, g->s_d2h));
  NF_CUDA(g, cudaMemcpyAsync(gv, g->hs_b, bv, cudaMemcpyDeviceToHost, g->s_d2h));
  NF_CUDA(g, cudaMemcpyAsync(gw, g->hs_c, bw, cudaMemcpyDeviceToHost, g->s_d2h));
  NF_CUDA(g, cudaEventRecord(g->ev_out_adj, g->s_d2h));
  if (!g->host_async) NF_CUDA(g, cudaStreamSynchronize(g->s_d2h));
  return rc;
}

extern "C" int nf_last_solve_info(nf_grid *g, int *iters, float *relres, float *ms) {
  NF_CHECK_HANDLE(g);
  float t = 0.0f;
  if (g->last_timed) {
    NF_CUDA(g, cudaEventSynchronize(g->ev1));
    NF_CUDA(g, cudaEventElapsedTime(&t, g->ev0, g->ev1));
  }
  if (iters) *iters = g->last_iters;
  if (relres) *relres = g->last_relres;
  if (ms) *ms = t;
  return NF_OK;
}

extern "C" int nf_grid_info(nf_grid *g, int *levels, long long *active_cells, int *singular) {
  NF_CHECK_HANDLE(g);
  if (g->weights_set) NF_TRY(nf_meta_sync(g));
  if (levels) *levels = g->nlev;
  if (active_cells) *active_cells = g->weights_set ? g->nact : -1;
  if (singular) *singular = g->weights_set ? g->singular_info : -1;
  return NF_OK;
}

extern "C" int nf_set_coarse_relaxation(nf_grid *g, float omega) {
  NF_CHECK_HANDLE(g);
  if (!(omega >= 1.0f && omega < 2.0f)) return NF_ERR_INVALID;
  g->omega_deep = omega;
  return g->weights_set ? nf_mg_upload_coarse(g) : NF_OK;
}
extern "C" float nf_get_coarse_relaxation(nf_grid *g) { return g ? g->omega_deep : 0.0f; }

extern "C" int nf_get_sweeps(nf_grid *g, int *nu_fine_pre, int *nu_fine_post, int *nu_level1, int *nu_deeper) {
  NF_CHECK_HANDLE(g);
  if (nu_fine_pre) *nu_fine_pre = g->nu_pre;
  if (nu_fine_post) *nu_fine_post = g->nu_post;
  if (nu_level1) *nu_level1 = g->nu_l1;
  if (nu_deeper) *nu_deeper = g->nu_deep;
  return NF_OK;
}

extern "C" int nf_grid_components(nf_grid *g, int *components, int *singular_components) {
  NF_CHECK_HANDLE(g);
  if (!g->weights_set) return NF_ERR_STATE;
  NF_TRY(nf_meta_sync(g));
  if (components) *components = g->ncomp;
  if (singular_components) *singular_components = g->nsing;
  return NF_OK;
}

// ---- per-class kernel timing -------------------------------------------------------------------------------------
static const char *kClassNames[NFK_COUNT] = {
    "apply_A", "cg_update", "cg_check", "cg_pupdate", "down1_fine", "down2_fine", "up1_fine", "up2_fine", "vec_coarse",
    "rbgs_fine", "rbgs_coarse", "restrict_fine", "restrict_coarse", "prolong_fine", "prolong_coarse", "tail",
    "solve_setup", "rhs", "grad_subtract", "adjoint_rhs", "adjoint_finish", "weights", "coarsen", "encode", "store_us",
    "advect", "advect_adjoint", "weights_adjoint", "geometry", "misc", "sweep_fine"};

void nf_prof_begin(nf_grid *g, int cls) {
  const size_t r = g->prof_cls.size();
  if (g->prof_pool.size() < 2 * (r + 1)) {
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { g->prof_on = false; return; }
    g->prof_pool.push_back(a);
    g->prof_pool.push_back(b);
  }
  g->prof_cls.push_back(cls);
  cudaEventRecord(g->prof_pool[2 * r], g->stream);
}
void nf_prof_end(nf_grid *g) {
  const size_t r = g->prof_cls.size() - 1;
  cudaEventRecord(g->prof_pool[2 * r + 1], g->stream);
}
static void prof_collect(nf_grid *g) {
  if (g->prof_cls.empty()) return;
  cudaStreamSynchronize(g->stream);
  for (size_t r = 0; r < g->prof_cls.size(); ++r) {
    float ms = 0.0f;
    if (cudaEventElapsedTime(&ms, g->prof_pool[2 * r], g->prof_pool[2 * r + 1]) == cudaSuccess) {
      g->prof_ms[g->prof_cls[r]] += ms;
      g->prof_n[g->prof_cls[r]] += 1;
    }
  }
  g->prof_cls.clear();
}

extern "C" int nf_profile_enable(nf_grid *g, int on) {
  NF_CHECK_HANDLE(g);
  prof_collect(g);
  if (on) {
    for (int c = 0; c < NFK_COUNT; ++c) { g->prof_ms[c] = 0.0; g->prof_n[c] = 0; }
  }
  g->prof_on = on != 0;
  return NF_OK;
}

extern "C" int nf_profile_get(nf_grid *g, int idx, const char **name, double *ms, long long *launches) {
  NF_CHECK_HANDLE(g);
  if (idx < 0 || idx >= NFK_COUNT) return NF_ERR_INVALID;
  prof_collect(g);
  if (name) *name = kClassNames[idx];
  if (ms) *ms = g->prof_ms[idx];
  if (launches) *launches = g->prof_n[idx];
  return NF_OK;
}

extern "C" long long nf_launch_count(nf_grid *g) { return g ? g->launches : 0; }

extern "C" const char *nf_last_error(nf_grid *g) { return g ? g->err.c_str() : "null handle"; }
