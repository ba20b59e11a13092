// nf_project.cu -- a-2 right-hand side / divergence (Eq. 4), a-6 pressure-gradient subtract
// (Eq. 5) and the two face passes of a-7, the adjoint projection (Eqs. 6-7,
// L134-139 Eq. 9 in the derived forms R9 / R10).
#include "nf_internal.cuh"

struct NfBcv {
  int t[6];
  float v[6];  // ghost pressure (0 for closed walls)
};
static NfBcv bcv(const nf_grid *g) {
  NfBcv b;
  for (int f = 0; f < 6; ++f) {
    b.t[f] = g->bc_type[f];
    b.v[f] = g->bc_type[f] == NF_BC_DIRICHLET ? g->bc_val[f] : 0.0f;
  }
  return b;
}

// b = G^T (S Uhat + (I - S) U_s) + c alpha_f p_D on Dirichlet ghost neighbours.  One thread per cell.
__global__ void __launch_bounds__(256) k_rhs(const float *__restrict__ u, const float *__restrict__ v,
                                             const float *__restrict__ w, const float *__restrict__ us,
                                             const float *__restrict__ vs, const float *__restrict__ ws,
                                             const float *__restrict__ ax, const float *__restrict__ ay,
                                             const float *__restrict__ az, float *__restrict__ b, float c, int nx,
                                             int ny, int nz, int pax, NfBcv bc) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= nx || j >= ny || k >= nz) return;
  const size_t iu = ((size_t)k * ny + j) * (nx + 1) + i;
  const size_t ia = ((size_t)k * ny + j) * pax + i;
  const size_t iv = ((size_t)k * (ny + 1) + j) * nx + i;
  const size_t iw = ((size_t)k * ny + j) * nx + i;
  const size_t sw = (size_t)ny * nx;
  const float axl = ax[ia], axh = ax[ia + 1], ayl = ay[iv], ayh = ay[iv + nx], azl = az[iw], azh = az[iw + sw];
  float ful = axl * u[iu], fuh = axh * u[iu + 1];
  float fvl = ayl * v[iv], fvh = ayh * v[iv + nx];
  float fwl = azl * w[iw], fwh = azh * w[iw + sw];
  if (us) {
    ful += (1.0f - axl) * us[iu];
    fuh += (1.0f - axh) * us[iu + 1];
    fvl += (1.0f - ayl) * vs[iv];
    fvh += (1.0f - ayh) * vs[iv + nx];
    fwl += (1.0f - azl) * ws[iw];
    fwh += (1.0f - azh) * ws[iw + sw];
  }
  float r = ((ful - fuh) + (fvl - fvh)) + (fwl - fwh);
  if (i == 0) r += c * axl * bc.v[0];
  if (i == nx - 1) r += c * axh * bc.v[1];
  if (j == 0) r += c * ayl * bc.v[2];
  if (j == ny - 1) r += c * ayh * bc.v[3];
  if (k == 0) r += c * azl * bc.v[4];
  if (k == nz - 1) r += c * azh * bc.v[5];
  b[iw] = r;
}

// (G p) on the face between cell index `lo` side and `hi` side along one axis, with ghost values outside.
__device__ __forceinline__ float nf_face_grad(const float *__restrict__ p, size_t id_hi, size_t stride, int cidx, int n,
                                              float ghost_lo, float ghost_hi) {
  // cidx = face index along the axis in [0, n]; cell cidx is on the high side, cidx-1 on the low side
  const float ph = cidx < n ? p[id_hi] : ghost_hi;
  const float pl = cidx > 0 ? p[id_hi - stride] : ghost_lo;
  return ph - pl;
}

// U = Uhat - c G p on open faces, U = U_s on closed faces (R7, R19).  One thread per extended cell; it owns the
// low x-, y- and z-face of that cell.
__global__ void __launch_bounds__(256) k_grad_subtract(float *__restrict__ u, float *__restrict__ v,
                                                       float *__restrict__ w, const float *__restrict__ p,
                                                       const float *__restrict__ us, const float *__restrict__ vs,
                                                       const float *__restrict__ ws, const float *__restrict__ ax,
                                                       const float *__restrict__ ay, const float *__restrict__ az,
                                                       float c, int nx, int ny, int nz, int pax, NfBcv bc,
                                                       const float *__restrict__ plo) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i > nx || j > ny || k > nz) return;
  const size_t sy = nx, sz = (size_t)nx * ny;
  // cell id of (i,j,k) clipped into range is only dereferenced when the corresponding index is in range
  const size_t idc = ((size_t)k * ny + j) * nx + i;
  // (plo: the low-order part of the pressure, nf_set_pressure_lo -- the pressure is p + plo, the ghosts belong to p)
  if (j < ny && k < nz) {
    const size_t f = ((size_t)k * ny + j) * (nx + 1) + i;
    const float a = ax[((size_t)k * ny + j) * pax + i];
    if (a > 0.0f)
      u[f] = u[f] - c * (nf_face_grad(p, idc, 1, i, nx, bc.v[0], bc.v[1]) + (plo ? nf_face_grad(plo, idc, 1, i, nx, 0.0f, 0.0f) : 0.0f));
    else
      u[f] = us ? us[f] : 0.0f;
  }
  if (i < nx && k < nz) {
    const size_t f = ((size_t)k * (ny + 1) + j) * nx + i;
    const float a = ay[f];
    if (a > 0.0f)
      v[f] = v[f] - c * (nf_face_grad(p, idc, sy, j, ny, bc.v[2], bc.v[3]) + (plo ? nf_face_grad(plo, idc, sy, j, ny, 0.0f, 0.0f) : 0.0f));
    else
      v[f] = vs ? vs[f] : 0.0f;
  }
  if (i < nx && j < ny) {
    const size_t f = ((size_t)k * ny + j) * nx + i;
    const float a = az[f];
    if (a > 0.0f)
      w[f] = w[f] - c * (nf_face_grad(p, idc, sz, k, nz, bc.v[4], bc.v[5]) + (plo ? nf_face_grad(plo, idc, sz, k, nz, 0.0f, 0.0f) : 0.0f));
    else
      w[f] = ws ? ws[f] : 0.0f;
  }
}

// Eq. 6 (column form, R8): dJ/dP = -c G^T (M g), M = [alpha > 0].  One thread per cell.
__global__ void __launch_bounds__(256) k_adjoint_rhs(const float *__restrict__ gu, const float *__restrict__ gv,
                                                     const float *__restrict__ gw, const float *__restrict__ ax,
                                                     const float *__restrict__ ay, const float *__restrict__ az,
                                                     float *__restrict__ b, float c, int nx, int ny, int nz, int pax) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= nx || j >= ny || k >= nz) return;
  const size_t iu = ((size_t)k * ny + j) * (nx + 1) + i;
  const size_t ia = ((size_t)k * ny + j) * pax + i;
  const size_t iv = ((size_t)k * (ny + 1) + j) * nx + i;
  const size_t iw = ((size_t)k * ny + j) * nx + i;
  const size_t sw = (size_t)ny * nx;
  const float ful = ax[ia] > 0.0f ? gu[iu] : 0.0f, fuh = ax[ia + 1] > 0.0f ? gu[iu + 1] : 0.0f;
  const float fvl = ay[iv] > 0.0f ? gv[iv] : 0.0f, fvh = ay[iv + nx] > 0.0f ? gv[iv + nx] : 0.0f;
  const float fwl = az[iw] > 0.0f ? gw[iw] : 0.0f, fwh = az[iw + sw] > 0.0f ? gw[iw + sw] : 0.0f;
  b[iw] = -c * (((ful - fuh) + (fvl - fvh)) + (fwl - fwh));
}

// One face of the adjoint finish.  g (in/out), optional galpha / gus outputs.
__device__ __forceinline__ void nf_adj_face(float *__restrict__ g, size_t f, float a, float Gy, float Gp, float uhat,
                                            float usv, float c, bool closed_wall, float *__restrict__ ga,
                                            float *__restrict__ gs) {
  const float gin = g[f];
  const float Mg = a > 0.0f ? gin : 0.0f;
  g[f] = Mg + a * Gy;                                        // Eq. 7
  if (ga) ga[f] = closed_wall ? 0.0f : Gy * ((uhat - usv) - c * Gp);   // Eq. 9a, derived sign (R9)
  if (gs) gs[f] = closed_wall ? 0.0f : (gin - Mg) + (1.0f - a) * Gy;   // Eq. 9b, derived form (R10)
}

__global__ void __launch_bounds__(256)
k_adjoint_finish(float *__restrict__ gu, float *__restrict__ gv, float *__restrict__ gw, const float *__restrict__ y,
                 const float *__restrict__ p, const float *__restrict__ uu, const float *__restrict__ uv,
                 const float *__restrict__ uw, const float *__restrict__ us, const float *__restrict__ vs,
                 const float *__restrict__ ws, const float *__restrict__ ax, const float *__restrict__ ay,
                 const float *__restrict__ az, float *__restrict__ gau, float *__restrict__ gav,
                 float *__restrict__ gaw, float *__restrict__ gsu, float *__restrict__ gsv, float *__restrict__ gsw,
                 float c, int nx, int ny, int nz, int pax, NfBcv bc) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i > nx || j > ny || k > nz) return;
  const size_t sy = nx, sz = (size_t)nx * ny;
  const size_t idc = ((size_t)k * ny + j) * nx + i;
  const bool need_p = (gau || gav || gaw);
  if (j < ny && k < nz) {
    const size_t f = ((size_t)k * ny + j) * (nx + 1) + i;
    const float a = ax[((size_t)k * ny + j) * pax + i];
    const float Gy = nf_face_grad(y, idc, 1, i, nx, 0.0f, 0.0f);  // ghost pressure is data, not an unknown
    const float Gp = need_p ? nf_face_grad(p, idc, 1, i, nx, bc.v[0], bc.v[1]) : 0.0f;
    const bool wall = (i == 0 && bc.t[0] == NF_BC_CLOSED) || (i == nx && bc.t[1] == NF_BC_CLOSED);
    nf_adj_face(gu, f, a, Gy, Gp, need_p ? uu[f] : 0.0f, us ? us[f] : 0.0f, c, wall, gau, gsu);
  }
  if (i < nx && k < nz) {
    const size_t f = ((size_t)k * (ny + 1) + j) * nx + i;
    const float a = ay[f];
    const float Gy = nf_face_grad(y, idc, sy, j, ny, 0.0f, 0.0f);
    const float Gp = need_p ? nf_face_grad(p, idc, sy, j, ny, bc.v[2], bc.v[3]) : 0.0f;
    const bool wall = (j == 0 && bc.t[2] == NF_BC_CLOSED) || (j == ny && bc.t[3] == NF_BC_CLOSED);
    nf_adj_face(gv, f, a, Gy, Gp, need_p ? uv[f] : 0.0f, vs ? vs[f] : 0.0f, c, wall, gav, gsv);
  }
  if (i < nx && j < ny) {
    const size_t f = ((size_t)k * ny + j) * nx + i;
    const float a = az[f];
    const float Gy = nf_face_grad(y, idc, sz, k, nz, 0.0f, 0.0f);
    const float Gp = need_p ? nf_face_grad(p, idc, sz, k, nz, bc.v[4], bc.v[5]) : 0.0f;
    const bool wall = (k == 0 && bc.t[4] == NF_BC_CLOSED) || (k == nz && bc.t[5] == NF_BC_CLOSED);
    nf_adj_face(gw, f, a, Gy, Gp, need_p ? uw[f] : 0.0f, ws ? ws[f] : 0.0f, c, wall, gaw, gsw);
  }
}

int nf_rhs_impl(nf_grid *g, const float *u, const float *v, const float *w) {
  NfLevel &L = g->lv[0];
  NfDims d = nf_dims(L.nx, L.ny, L.nz);
  const bool hu = g->have_us;
  NF_LAUNCH(g, NFK_RHS, k_rhs<<<d.grid, d.block, 0, g->stream>>>(u, v, w, hu ? g->us : nullptr, hu ? g->vs : nullptr, hu ? g->ws : nullptr,
                                           L.ax, L.ay, L.az, L.r, L.c, L.nx, L.ny, L.nz, L.pax, bcv(g)));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_grad_subtract_impl(nf_grid *g, float *u, float *v, float *w, const float *p) {
  NfLevel &L = g->lv[0];
  NfDims d = nf_dims(L.nx + 1, L.ny + 1, L.nz + 1);
  const bool hu = g->have_us;
  NF_LAUNCH(g, NFK_GRADSUB, k_grad_subtract<<<d.grid, d.block, 0, g->stream>>>(u, v, w, p, hu ? g->us : nullptr, hu ? g->vs : nullptr,
                                                     hu ? g->ws : nullptr, L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz,
                                                     L.pax, bcv(g), g->lo_valid ? g->plo : nullptr));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_adjoint_rhs_impl(nf_grid *g, const float *gu, const float *gv, const float *gw) {
  NfLevel &L = g->lv[0];
  NfDims d = nf_dims(L.nx, L.ny, L.nz);
  NF_LAUNCH(g, NFK_ADJ_RHS, k_adjoint_rhs<<<d.grid, d.block, 0, g->stream>>>(gu, gv, gw, L.ax, L.ay, L.az, L.r, L.c, L.nx, L.ny, L.nz, L.pax));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_adjoint_finish_impl(nf_grid *g, float *gu, float *gv, float *gw, const float *y, const float *p_saved,
                           const float *uu, const float *uv, const float *uw, float *gau, float *gav, float *gaw,
                           float *gsu, float *gsv, float *gsw) {
  NfLevel &L = g->lv[0];
  NfDims d = nf_dims(L.nx + 1, L.ny + 1, L.nz + 1);
  const bool hu = g->have_us;
  NF_LAUNCH(g, NFK_ADJ_FINISH, k_adjoint_finish<<<d.grid, d.block, 0, g->stream>>>(gu, gv, gw, y, p_saved, uu, uv, uw, hu ? g->us : nullptr,
                                                      hu ? g->vs : nullptr, hu ? g->ws : nullptr, L.ax, L.ay, L.az,
                                                      gau, gav, gaw, gsu, gsv, gsw, L.c, L.nx, L.ny, L.nz, L.pax,
                                                      bcv(g)));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}
