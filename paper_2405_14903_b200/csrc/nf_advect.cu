// nf_advect.cu -- a-8 semi-Lagrangian advection (Eq. 2; L353-357 Eqs. 11-12) and a-9 its adjoint
// (Eq. 8).  Two-stage (mid-point) back-trace evaluated pointwise at every face (R20), per-component
// trilinear interpolation on each component's own staggered lattice, positions clamped to the lattice (R14).
#include "nf_internal.cuh"

struct NfLat {  // the three staggered lattices
  const float *f[3];
  int ex[3], ey[3], ez[3];
};

struct NfLoc {
  int i0, i1;
  float fr;
  bool free_;
};
// lattice coordinate along one axis: t = pos - offset, clamped to [0, n-1]
__device__ __forceinline__ NfLoc nf_locate(float t, int n) {
  NfLoc L;
  const float hi = (float)(n - 1);
  const float tc = fminf(fmaxf(t, 0.0f), hi);
  int i0 = (int)floorf(tc);
  if (i0 > n - 2) i0 = n - 2;
  if (i0 < 0) i0 = 0;
  L.i0 = i0;
  L.i1 = i0 + 1 < n ? i0 + 1 : n - 1;
  L.fr = tc - (float)i0;
  L.free_ = (t >= 0.0f) && (t <= hi);
  return L;
}

__device__ __forceinline__ void nf_comp_offsets(int comp, float &ox, float &oy, float &oz) {
  ox = comp == 0 ? 0.0f : 0.5f;
  oy = comp == 1 ? 0.0f : 0.5f;
  oz = comp == 2 ? 0.0f : 0.5f;
}

// trilinear interpolation of component `comp` at (x, y, z) in cell units
__device__ __forceinline__ float nf_interp(const NfLat &U, int comp, float x, float y, float z) {
  float ox, oy, oz;
  nf_comp_offsets(comp, ox, oy, oz);
  const int ex = U.ex[comp], ey = U.ey[comp], ez = U.ez[comp];
  const NfLoc X = nf_locate(x - ox, ex), Y = nf_locate(y - oy, ey), Z = nf_locate(z - oz, ez);
  const float *f = U.f[comp];
  const size_t r00 = ((size_t)Z.i0 * ey + Y.i0) * ex, r01 = ((size_t)Z.i0 * ey + Y.i1) * ex;
  const size_t r10 = ((size_t)Z.i1 * ey + Y.i0) * ex, r11 = ((size_t)Z.i1 * ey + Y.i1) * ex;
  const float wx1 = X.fr, wx0 = 1.0f - X.fr;
  const float a00 = wx0 * __ldg(f + r00 + X.i0) + wx1 * __ldg(f + r00 + X.i1);
  const float a01 = wx0 * __ldg(f + r01 + X.i0) + wx1 * __ldg(f + r01 + X.i1);
  const float a10 = wx0 * __ldg(f + r10 + X.i0) + wx1 * __ldg(f + r10 + X.i1);
  const float a11 = wx0 * __ldg(f + r11 + X.i0) + wx1 * __ldg(f + r11 + X.i1);
  const float b0 = (1.0f - Y.fr) * a00 + Y.fr * a01;
  const float b1 = (1.0f - Y.fr) * a10 + Y.fr * a11;
  return (1.0f - Z.fr) * b0 + Z.fr * b1;
}

// reverse of nf_interp: scatter gbar * weight into gf (atomics) and return gbar * d(out)/d(pos) (0 on clamped axes)
__device__ __forceinline__ void nf_interp_adjoint(const NfLat &U, int comp, float x, float y, float z, float gbar,
                                                  float *__restrict__ gf, float &gx, float &gy, float &gz) {
  float ox, oy, oz;
  nf_comp_offsets(comp, ox, oy, oz);
  const int ex = U.ex[comp], ey = U.ey[comp], ez = U.ez[comp];
  const NfLoc X = nf_locate(x - ox, ex), Y = nf_locate(y - oy, ey), Z = nf_locate(z - oz, ez);
  const float *f = U.f[comp];
  gx = gy = gz = 0.0f;
  if (gbar == 0.0f) return;
#pragma unroll
  for (int dz = 0; dz < 2; ++dz)
#pragma unroll
    for (int dy = 0; dy < 2; ++dy)
#pragma unroll
      for (int dx = 0; dx < 2; ++dx) {
        const float wx = dx ? X.fr : 1.0f - X.fr, wy = dy ? Y.fr : 1.0f - Y.fr, wz = dz ? Z.fr : 1.0f - Z.fr;
        const size_t id = ((size_t)(dz ? Z.i1 : Z.i0) * ey + (dy ? Y.i1 : Y.i0)) * ex + (dx ? X.i1 : X.i0);
        const float wgt = wx * wy * wz;
        if (wgt != 0.0f) atomicAdd(gf + id, gbar * wgt);
        const float val = __ldg(f + id);
        gx += gbar * val * (dx ? 1.0f : -1.0f) * wy * wz;
        gy += gbar * val * wx * (dy ? 1.0f : -1.0f) * wz;
        gz += gbar * val * wx * wy * (dz ? 1.0f : -1.0f);
      }
  if (!X.free_) gx = 0.0f;
  if (!Y.free_) gy = 0.0f;
  if (!Z.free_) gz = 0.0f;
}

__device__ __forceinline__ float nf_advect_face(const NfLat &U, int comp, float x, float y, float z, float s) {
  const float v0x = nf_interp(U, 0, x, y, z), v0y = nf_interp(U, 1, x, y, z), v0z = nf_interp(U, 2, x, y, z);
  const float xm = x - 0.5f * s * v0x, ym = y - 0.5f * s * v0y, zm = z - 0.5f * s * v0z;  // Eq. 11
  const float vmx = nf_interp(U, 0, xm, ym, zm), vmy = nf_interp(U, 1, xm, ym, zm), vmz = nf_interp(U, 2, xm, ym, zm);
  const float xb = x - s * vmx, yb = y - s * vmy, zb = z - s * vmz;  // Eq. 12
  return nf_interp(U, comp, xb, yb, zb);
}

// one thread per extended cell; it owns the low x-, y- and z-face of that cell
__global__ void __launch_bounds__(256) k_advect(NfLat U, float *__restrict__ ou, float *__restrict__ ov,
                                                float *__restrict__ ow, int nx, int ny, int nz, float s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i > nx || j > ny || k > nz) return;
  const float fi = (float)i, fj = (float)j, fk = (float)k;
  if (j < ny && k < nz) ou[((size_t)k * ny + j) * (nx + 1) + i] = nf_advect_face(U, 0, fi, fj + 0.5f, fk + 0.5f, s);
  if (i < nx && k < nz) ov[((size_t)k * (ny + 1) + j) * nx + i] = nf_advect_face(U, 1, fi + 0.5f, fj, fk + 0.5f, s);
  if (i < nx && j < ny) ow[((size_t)k * ny + j) * nx + i] = nf_advect_face(U, 2, fi + 0.5f, fj + 0.5f, fk, s);
}

struct NfGrad3 {
  float *g[3];
};

__device__ __forceinline__ void nf_advect_face_adjoint(const NfLat &U, const NfGrad3 &G, int comp, float x, float y,
                                                       float z, float s, float gout) {
  if (gout == 0.0f) return;
  const float v0x = nf_interp(U, 0, x, y, z), v0y = nf_interp(U, 1, x, y, z), v0z = nf_interp(U, 2, x, y, z);
  const float xm = x - 0.5f * s * v0x, ym = y - 0.5f * s * v0y, zm = z - 0.5f * s * v0z;
  const float vmx = nf_interp(U, 0, xm, ym, zm), vmy = nf_interp(U, 1, xm, ym, zm), vmz = nf_interp(U, 2, xm, ym, zm);
  const float xb = x - s * vmx, yb = y - s * vmy, zb = z - s * vmz;
  float gbx, gby, gbz;  // dJ/dx_b
  nf_interp_adjoint(U, comp, xb, yb, zb, gout, G.g[comp], gbx, gby, gbz);
  const float gvm[3] = {-s * gbx, -s * gby, -s * gbz};
  float gmx = 0.0f, gmy = 0.0f, gmz = 0.0f;  // dJ/dx_m
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    float tx, ty, tz;
    nf_interp_adjoint(U, d, xm, ym, zm, gvm[d], G.g[d], tx, ty, tz);
    gmx += tx; gmy += ty; gmz += tz;
  }
  const float gv0[3] = {-0.5f * s * gmx, -0.5f * s * gmy, -0.5f * s * gmz};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    float tx, ty, tz;
    nf_interp_adjoint(U, d, x, y, z, gv0[d], G.g[d], tx, ty, tz);
  }
}

__global__ void __launch_bounds__(256) k_advect_adjoint(NfLat U, NfGrad3 G, const float *__restrict__ gou,
                                                        const float *__restrict__ gov, const float *__restrict__ gow,
                                                        int nx, int ny, int nz, float s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i > nx || j > ny || k > nz) return;
  const float fi = (float)i, fj = (float)j, fk = (float)k;
  if (j < ny && k < nz)
    nf_advect_face_adjoint(U, G, 0, fi, fj + 0.5f, fk + 0.5f, s, gou[((size_t)k * ny + j) * (nx + 1) + i]);
  if (i < nx && k < nz)
    nf_advect_face_adjoint(U, G, 1, fi + 0.5f, fj, fk + 0.5f, s, gov[((size_t)k * (ny + 1) + j) * nx + i]);
  if (i < nx && j < ny)
    nf_advect_face_adjoint(U, G, 2, fi + 0.5f, fj + 0.5f, fk, s, gow[((size_t)k * ny + j) * nx + i]);
}

static NfLat make_lat(const nf_grid *g, const float *u, const float *v, const float *w) {
  NfLat U;
  U.f[0] = u; U.f[1] = v; U.f[2] = w;
  U.ex[0] = g->nx + 1; U.ey[0] = g->ny;     U.ez[0] = g->nz;
  U.ex[1] = g->nx;     U.ey[1] = g->ny + 1; U.ez[1] = g->nz;
  U.ex[2] = g->nx;     U.ey[2] = g->ny;     U.ez[2] = g->nz + 1;
  return U;
}

int nf_advect_impl(nf_grid *g, float *u, float *v, float *w, float dt) {
  NF_CUDA(g, cudaMemcpyAsync(g->fu, u, nf_nu(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fv, v, nf_nv(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fw, w, nf_nw(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NfDims d = nf_dims(g->nx + 1, g->ny + 1, g->nz + 1);
  NF_LAUNCH(g, NFK_ADVECT, k_advect<<<d.grid, d.block, 0, g->stream>>>(make_lat(g, g->fu, g->fv, g->fw), u, v, w, g->nx, g->ny, g->nz,
                                              dt / g->dx));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_advect_adjoint_impl(nf_grid *g, const float *u0, const float *v0, const float *w0, float *gu, float *gv,
                           float *gw, float dt) {
  NF_CUDA(g, cudaMemcpyAsync(g->fu, gu, nf_nu(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fv, gv, nf_nv(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fw, gw, nf_nw(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemsetAsync(gu, 0, nf_nu(g) * sizeof(float), g->stream));
  NF_CUDA(g, cudaMemsetAsync(gv, 0, nf_nv(g) * sizeof(float), g->stream));
  NF_CUDA(g, cudaMemsetAsync(gw, 0, nf_nw(g) * sizeof(float), g->stream));
  NfGrad3 G;
  G.g[0] = gu; G.g[1] = gv; G.g[2] = gw;
  NfDims d = nf_dims(g->nx + 1, g->ny + 1, g->nz + 1);
  NF_LAUNCH(g, NFK_ADVECT_ADJ, k_advect_adjoint<<<d.grid, d.block, 0, g->stream>>>(make_lat(g, u0, v0, w0), G, g->fu, g->fv, g->fw, g->nx, g->ny,
                                                      g->nz, dt / g->dx));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}
