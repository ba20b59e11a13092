// nf_advect.cu -- a-8 semi-Lagrangian advection (Eq. 2; L353-357 Eqs. 11-12) and a-9 its adjoint
// (Eq. 8).  Two-stage (mid-point) back-trace evaluated pointwise at every face (R20), per-component
// trilinear interpolation on each component's own staggered lattice, positions clamped to the lattice (R14).
//
// Both kernels are instruction-bound, not bandwidth-bound (ncu, profiles/): 7 trilinear interpolations per face.  So:
// one launch per face family (template parameter C: small kernels, high occupancy, compile-time lattice offsets);
// the first stage U(x) at the face's own position is lattice-aligned and is evaluated as the fixed 1- and 4-point
// stencils it reduces to (same clamping as the general interpolation) instead of three general interpolations;
// 32-bit index arithmetic throughout (lattices have < 2^31 points).
#include <cstring>

#include "nf_internal.cuh"
#ifndef NF_ADJ_MINB
#define NF_ADJ_MINB 4
#endif

struct NfLat {  // the three staggered lattices: extents and data
  const float *f[3];
  int ex[3], ey[3], ez[3];
};
struct NfGrad3 {
  float *g[3];
};

struct NfLoc {
  int i0;      // lower lattice index (upper = i0 + step)
  int step;    // 1, or 0 on a one-layer lattice
  float fr;    // weight of the upper index
  bool free_;  // position inside the lattice (not clamped): it carries a position gradient
};
// lattice coordinate along one axis: t = pos - offset, clamped to [0, n-1]
__device__ __forceinline__ NfLoc nf_locate(float t, int n) {
  NfLoc L;
  const float hi = (float)(n - 1);
  const float tc = fminf(fmaxf(t, 0.0f), hi);
  const int i0 = max(min((int)tc, n - 2), 0);  // (tc >= 0: truncation = floor)
  L.i0 = i0;
  L.step = n > 1 ? 1 : 0;
  L.fr = tc - (float)i0;
  L.free_ = (t >= 0.0f) && (t <= hi);
  return L;
}

// trilinear interpolation of component D at (x, y, z) in cell units
template <int D>
__device__ __forceinline__ float nf_interp(const NfLat &U, float x, float y, float z) {
  const int ex = U.ex[D], ey = U.ey[D], ez = U.ez[D];
  const NfLoc X = nf_locate(x - (D == 0 ? 0.0f : 0.5f), ex), Y = nf_locate(y - (D == 1 ? 0.0f : 0.5f), ey),
              Z = nf_locate(z - (D == 2 ? 0.0f : 0.5f), ez);
  const float *f = U.f[D] + ((Z.i0 * ey + Y.i0) * ex + X.i0);
  const int sx = X.step, sy = Y.step * ex, sz = Z.step * ex * ey;
  const float a00 = f[0] + X.fr * (f[sx] - f[0]);
  const float a01 = f[sy] + X.fr * (f[sy + sx] - f[sy]);
  const float a10 = f[sz] + X.fr * (f[sz + sx] - f[sz]);
  const float a11 = f[sz + sy] + X.fr * (f[sz + sy + sx] - f[sz + sy]);
  const float b0 = a00 + Y.fr * (a01 - a00);
  const float b1 = a10 + Y.fr * (a11 - a10);
  return b0 + Z.fr * (b1 - b0);
}

// Component D at the position of face (i, j, k) of family C (Eq. 11's u^n(x)).  D == C: the face value itself.
// D != C: the position is lattice-aligned along the third axis, half-way between two layers along C and along D,
// so the interpolation is the mean of four values; along C the two layers are i_C - 1 and i_C clamped to the
// lattice (which reproduces nf_locate's clamping exactly: both collapse onto the boundary layer).
// Returns the four lattice offsets in o[] as well (the adjoint scatters to them).
template <int C, int D>
__device__ __forceinline__ float nf_self(const NfLat &U, int i, int j, int k, int o[4]) {
  const int ex = U.ex[D], ey = U.ey[D];
  const int st[3] = {1, ex, ex * ey};
  const int idx[3] = {i, j, k};
  if (C == D) {
    o[0] = o[1] = o[2] = o[3] = (k * ey + j) * ex + i;
    return U.f[D][o[0]];
  }
  const int nC = C == 0 ? ex : (C == 1 ? ey : U.ez[D]);  // extent of lattice D along axis C
  const int lo = max(idx[C] - 1, 0), hi = min(idx[C], nC - 1);
  int base = 0;
#pragma unroll
  for (int a = 0; a < 3; ++a)
    if (a != C) base += idx[a] * st[a];
  o[0] = base + lo * st[C];
  o[1] = base + hi * st[C];
  o[2] = o[0] + st[D];
  o[3] = o[1] + st[D];
  const float *f = U.f[D];
  return 0.5f * (0.5f * (f[o[0]] + f[o[1]]) + 0.5f * (f[o[2]] + f[o[3]]));
}

// position of face (i, j, k) of family C in cell units
template <int C>
__device__ __forceinline__ void nf_face_pos(int i, int j, int k, float &x, float &y, float &z) {
  x = (float)i + (C == 0 ? 0.0f : 0.5f);
  y = (float)j + (C == 1 ? 0.0f : 0.5f);
  z = (float)k + (C == 2 ? 0.0f : 0.5f);
}

// a-8: one thread per face of family C.  s = dt / dx.
template <int C>
__global__ void __launch_bounds__(256) k_advect(NfLat U, float *__restrict__ out, float s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= U.ex[C] || j >= U.ey[C] || k >= U.ez[C]) return;
  float x, y, z;
  nf_face_pos<C>(i, j, k, x, y, z);
  int o[4];
  const float v0x = nf_self<C, 0>(U, i, j, k, o), v0y = nf_self<C, 1>(U, i, j, k, o), v0z = nf_self<C, 2>(U, i, j, k, o);
  const float xm = x - 0.5f * s * v0x, ym = y - 0.5f * s * v0y, zm = z - 0.5f * s * v0z;  // Eq. 11
  const float vmx = nf_interp<0>(U, xm, ym, zm), vmy = nf_interp<1>(U, xm, ym, zm), vmz = nf_interp<2>(U, xm, ym, zm);
  const float xb = x - s * vmx, yb = y - s * vmy, zb = z - s * vmz;  // Eq. 12
  out[(k * U.ey[C] + j) * U.ex[C] + i] = nf_interp<C>(U, xb, yb, zb);
}

// reverse of nf_interp: scatter gbar * weight into gf (atomics) and return gbar * d(out)/d(pos) (0 on clamped axes)
template <int D>
__device__ __forceinline__ void nf_interp_adjoint(const NfLat &U, float x, float y, float z, float gbar,
                                                  float *__restrict__ gf, float &gx, float &gy, float &gz) {
  gx = gy = gz = 0.0f;
  if (gbar == 0.0f) return;
  const int ex = U.ex[D], ey = U.ey[D], ez = U.ez[D];
  const NfLoc X = nf_locate(x - (D == 0 ? 0.0f : 0.5f), ex), Y = nf_locate(y - (D == 1 ? 0.0f : 0.5f), ey),
              Z = nf_locate(z - (D == 2 ? 0.0f : 0.5f), ez);
  const int base = (Z.i0 * ey + Y.i0) * ex + X.i0;
  const float *f = U.f[D] + base;
  float *g = gf + base;
  const int sx = X.step, sy = Y.step * ex, sz = Z.step * ex * ey;
#pragma unroll
  for (int dz = 0; dz < 2; ++dz)
#pragma unroll
    for (int dy = 0; dy < 2; ++dy) {
      const float wy = dy ? Y.fr : 1.0f - Y.fr, wz = dz ? Z.fr : 1.0f - Z.fr;
      const int row = (dz ? sz : 0) + (dy ? sy : 0);
      const float gw = gbar * wy * wz;
      const float v0 = gw * (1.0f - X.fr), v1 = gw * X.fr;
      if (v0 != 0.0f) atomicAdd(g + row, v0);
      if (v1 != 0.0f) atomicAdd(g + row + sx, v1);
      const float f0 = f[row], f1 = f[row + sx];
      gx += gw * (f1 - f0);
      const float fx = f0 + X.fr * (f1 - f0);
      gy += gbar * fx * (dy ? 1.0f : -1.0f) * wz;
      gz += gbar * fx * wy * (dz ? 1.0f : -1.0f);
    }
  if (!X.free_) gx = 0.0f;
  if (!Y.free_) gy = 0.0f;
  if (!Z.free_) gz = 0.0f;
}

// reverse of nf_self
template <int C, int D>
__device__ __forceinline__ void nf_self_adjoint(float *__restrict__ g, const int o[4], float gbar) {
  if (gbar == 0.0f) return;
  if (C == D) {
    atomicAdd(g + o[0], gbar);
  } else {
    const float q = 0.25f * gbar;
#pragma unroll
    for (int t = 0; t < 4; ++t) atomicAdd(g + o[t], q);
  }
}

// a-9: one thread per face of family C; gin = dJ/d(advected field) of that family; G accumulates dJ/dU^n.
template <int C>
__global__ void __launch_bounds__(256, NF_ADJ_MINB) k_advect_adjoint(NfLat U, NfGrad3 G, const float *__restrict__ gin, float s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= U.ex[C] || j >= U.ey[C] || k >= U.ez[C]) return;
  const float gout = gin[(k * U.ey[C] + j) * U.ex[C] + i];
  if (gout == 0.0f) return;
  float x, y, z;
  nf_face_pos<C>(i, j, k, x, y, z);
  int o0[4], o1[4], o2[4];
  const float v0x = nf_self<C, 0>(U, i, j, k, o0), v0y = nf_self<C, 1>(U, i, j, k, o1), v0z = nf_self<C, 2>(U, i, j, k, o2);
  const float xm = x - 0.5f * s * v0x, ym = y - 0.5f * s * v0y, zm = z - 0.5f * s * v0z;
  const float vmx = nf_interp<0>(U, xm, ym, zm), vmy = nf_interp<1>(U, xm, ym, zm), vmz = nf_interp<2>(U, xm, ym, zm);
  const float xb = x - s * vmx, yb = y - s * vmy, zb = z - s * vmz;
  float gbx, gby, gbz;  // dJ/dx_b
  nf_interp_adjoint<C>(U, xb, yb, zb, gout, G.g[C], gbx, gby, gbz);
  float gmx, gmy, gmz, tx, ty, tz;  // dJ/dx_m
  nf_interp_adjoint<0>(U, xm, ym, zm, -s * gbx, G.g[0], gmx, gmy, gmz);
  nf_interp_adjoint<1>(U, xm, ym, zm, -s * gby, G.g[1], tx, ty, tz);
  gmx += tx; gmy += ty; gmz += tz;
  nf_interp_adjoint<2>(U, xm, ym, zm, -s * gbz, G.g[2], tx, ty, tz);
  gmx += tx; gmy += ty; gmz += tz;
  nf_self_adjoint<C, 0>(G.g[0], o0, -0.5f * s * gmx);
  nf_self_adjoint<C, 1>(G.g[1], o1, -0.5f * s * gmy);
  nf_self_adjoint<C, 2>(G.g[2], o2, -0.5f * s * gmz);
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
  if (nf_nn(g) >= (size_t)1 << 31) {
    g->err = "nf_advect: grid too large for 32-bit lattice indices";
    return NF_ERR_INVALID;
  }
  NF_CUDA(g, cudaMemcpyAsync(g->fu, u, nf_nu(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fv, v, nf_nv(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fw, w, nf_nw(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  const NfLat U = make_lat(g, g->fu, g->fv, g->fw);
  const float s = dt / g->dx;
  NfDims d0 = nf_dims(U.ex[0], U.ey[0], U.ez[0]), d1 = nf_dims(U.ex[1], U.ey[1], U.ez[1]),
         d2 = nf_dims(U.ex[2], U.ey[2], U.ez[2]);
  NF_LAUNCH(g, NFK_ADVECT, k_advect<0><<<d0.grid, d0.block, 0, g->stream>>>(U, u, s));
  NF_LAUNCH(g, NFK_ADVECT, k_advect<1><<<d1.grid, d1.block, 0, g->stream>>>(U, v, s));
  NF_LAUNCH(g, NFK_ADVECT, k_advect<2><<<d2.grid, d2.block, 0, g->stream>>>(U, w, s));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_advect_adjoint_impl(nf_grid *g, const float *u0, const float *v0, const float *w0, float *gu, float *gv,
                           float *gw, float dt) {
  if (nf_nn(g) >= (size_t)1 << 31) {
    g->err = "nf_advect_adjoint: grid too large for 32-bit lattice indices";
    return NF_ERR_INVALID;
  }
  NF_CUDA(g, cudaMemcpyAsync(g->fu, gu, nf_nu(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fv, gv, nf_nv(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fw, gw, nf_nw(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemsetAsync(gu, 0, nf_nu(g) * sizeof(float), g->stream));
  NF_CUDA(g, cudaMemsetAsync(gv, 0, nf_nv(g) * sizeof(float), g->stream));
  NF_CUDA(g, cudaMemsetAsync(gw, 0, nf_nw(g) * sizeof(float), g->stream));
  NfGrad3 G;
  G.g[0] = gu; G.g[1] = gv; G.g[2] = gw;
  const NfLat U = make_lat(g, u0, v0, w0);
  const float s = dt / g->dx;
  NfDims d0 = nf_dims(U.ex[0], U.ey[0], U.ez[0]), d1 = nf_dims(U.ex[1], U.ey[1], U.ez[1]),
         d2 = nf_dims(U.ex[2], U.ey[2], U.ez[2]);
  NF_LAUNCH(g, NFK_ADVECT_ADJ, k_advect_adjoint<0><<<d0.grid, d0.block, 0, g->stream>>>(U, G, g->fu, s));
  NF_LAUNCH(g, NFK_ADVECT_ADJ, k_advect_adjoint<1><<<d1.grid, d1.block, 0, g->stream>>>(U, G, g->fv, s));
  NF_LAUNCH(g, NFK_ADVECT_ADJ, k_advect_adjoint<2><<<d2.grid, d2.block, 0, g->stream>>>(U, G, g->fw, s));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

// ------------------------------------------------------------------------------------------------------------
// NEXT-1: explicit viscosity  Uhat = (I - nu dt/dx^2 G^T G) Utilde   (Eq. 3, L359-361 Eq. 13)
// ------------------------------------------------------------------------------------------------------------
// Per component, the 7-point operator of that component's own lattice with nothing outside it (R23: keeps G^T G
// symmetric, so the backward pass -- Eq. 8 -- is this same kernel applied to the gradient).  One thread per lattice
// point; neighbours through L1 (24 B/point algorithmic: read + write once).
__global__ void __launch_bounds__(256) k_viscosity(const float *__restrict__ f, float *__restrict__ out, int ex, int ey,
                                                   int ez, float kk) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= ex || j >= ey || k >= ez) return;
  const int id = (k * ey + j) * ex + i, sy = ex, sz = ex * ey;
  const float c = f[id];
  float gtg = 0.0f;  // (G^T G f) at this point = sum over existing neighbours of (f - f_nb)
  if (i > 0) gtg += c - f[id - 1];
  if (i + 1 < ex) gtg += c - f[id + 1];
  if (j > 0) gtg += c - f[id - sy];
  if (j + 1 < ey) gtg += c - f[id + sy];
  if (k > 0) gtg += c - f[id - sz];
  if (k + 1 < ez) gtg += c - f[id + sz];
  out[id] = c - kk * gtg;
}

int nf_viscosity_impl(nf_grid *g, float *u, float *v, float *w, float nu, float dt) {
  if (nf_nn(g) >= (size_t)1 << 31) {
    g->err = "nf_viscosity: grid too large for 32-bit lattice indices";
    return NF_ERR_INVALID;
  }
  NF_CUDA(g, cudaMemcpyAsync(g->fu, u, nf_nu(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fv, v, nf_nv(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaMemcpyAsync(g->fw, w, nf_nw(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  const NfLat U = make_lat(g, g->fu, g->fv, g->fw);
  const float kk = nu * dt / (g->dx * g->dx);
  float *outs[3] = {u, v, w};
  for (int c = 0; c < 3; ++c) {
    NfDims d = nf_dims(U.ex[c], U.ey[c], U.ez[c]);
    NF_LAUNCH(g, NFK_ADVECT, k_viscosity<<<d.grid, d.block, 0, g->stream>>>(U.f[c], outs[c], U.ex[c], U.ey[c], U.ez[c], kk));
  }
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

// ------------------------------------------------------------------------------------------------------------
// NEXT-1: CFL sub-stepping support ("adopts CFL condition ... the actual steps simulated are
// higher than # Frames"; the condition's constant is not given, R24) -- max over all faces of |velocity|.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_max_abs(const float *__restrict__ f, size_t n, unsigned *out) {
  float m = 0.0f;
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  for (size_t t = tid; t < n; t += nth) {
    const float v = fabsf(f[t]);
    m = (v > m || v != v) ? v : m;  // (a NaN propagates)
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float t = __shfl_xor_sync(0xffffffffu, m, o);
    m = (t > m || t != t) ? t : m;
  }
  // non-negative floats order like their bit patterns (NaN patterns sort above every finite value)
  if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(m));
}

int nf_max_speed_impl(nf_grid *g, const float *u, const float *v, const float *w, float *out_host) {
  unsigned *d = reinterpret_cast<unsigned *>(g->d_counts);  // (scratch: two doubles, rewritten by every hierarchy build)
  NF_CUDA(g, cudaMemsetAsync(d, 0, sizeof(unsigned), g->stream));
  const float *f[3] = {u, v, w};
  const size_t n[3] = {nf_nu(g), nf_nv(g), nf_nw(g)};
  for (int c = 0; c < 3; ++c)
    NF_LAUNCH(g, NFK_MISC, k_max_abs<<<148 * 8, 256, 0, g->stream>>>(f[c], n[c], d));
  unsigned bits = 0;
  NF_CUDA(g, cudaMemcpyAsync(&bits, d, sizeof(unsigned), cudaMemcpyDeviceToHost, g->stream));
  NF_CUDA(g, cudaStreamSynchronize(g->stream));
  float r;
  memcpy(&r, &bits, sizeof(float));
  *out_host = r;
  return NF_OK;
}
