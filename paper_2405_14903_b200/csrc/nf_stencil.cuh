// nf_stencil.cuh -- device helpers shared by the stencil kernels of the solver (a-3, a-5): the six face weights of
// a cell from the fp32 arrays or from the 1-byte cell code, and 16-byte row loads with
// homogeneous ghosts.  A = c G^T S G (Eq. 4).
#pragma once
#include "nf_internal.cuh"

// 32-bit cell / face offsets in the stencil kernels (levels with >= 2^32 face slots do not take the vec path: nf_mg_plan)
typedef unsigned int nf_idx;

struct NfW6 {
  float xl, xh, yl, yh, zl, zh;
};

__device__ __forceinline__ NfW6 nf_load_w6(const float *__restrict__ ax, const float *__restrict__ ay,
                                           const float *__restrict__ az, int i, int j, int k, int nx, int ny, int pax) {
  NfW6 w;
  const nf_idx rx = ((nf_idx)k * ny + j) * pax + i;
  w.xl = __ldg(ax + rx);
  w.xh = __ldg(ax + rx + 1);
  const nf_idx ry = ((nf_idx)k * (ny + 1) + j) * nx + i;
  w.yl = __ldg(ay + ry);
  w.yh = __ldg(ay + ry + nx);
  const nf_idx rz = ((nf_idx)k * ny + j) * nx + i;
  w.zl = __ldg(az + rz);
  w.zh = __ldg(az + rz + (nf_idx)ny * nx);
  return w;
}
__device__ __forceinline__ float nf_w6_sum(const NfW6 &w) { return ((w.xl + w.xh) + (w.yl + w.yh)) + (w.zl + w.zh); }

// sum over the six neighbours of alpha_f * v_nb with homogeneous ghosts (v = 0 outside the grid)
__device__ __forceinline__ float nf_nb_sum(const float *__restrict__ v, const NfW6 &w, int i, int j, int k, int nx,
                                           int ny, int nz) {
  const nf_idx id = ((nf_idx)k * ny + j) * nx + i;
  const nf_idx sy = nx, sz = (nf_idx)nx * ny;
  float s = 0.0f;
  if (i > 0) s += w.xl * v[id - 1];
  if (i + 1 < nx) s += w.xh * v[id + 1];
  if (j > 0) s += w.yl * v[id - sy];
  if (j + 1 < ny) s += w.yh * v[id + sy];
  if (k > 0) s += w.zl * v[id - sz];
  if (k + 1 < nz) s += w.zh * v[id + sz];
  return s;
}

// sum over the six faces of alpha_f * (pc - v_nb) with homogeneous ghosts
__device__ __forceinline__ float nf_nb_diff(const float *__restrict__ v, const NfW6 &w, float pc, int i, int j, int k,
                                            int nx, int ny, int nz) {
  const nf_idx id = ((nf_idx)k * ny + j) * nx + i;
  const nf_idx sy = nx, sz = (nf_idx)nx * ny;
  float s = w.xl * (pc - (i > 0 ? v[id - 1] : 0.0f));
  s += w.xh * (pc - (i + 1 < nx ? v[id + 1] : 0.0f));
  s += w.yl * (pc - (j > 0 ? v[id - sy] : 0.0f));
  s += w.yh * (pc - (j + 1 < ny ? v[id + sy] : 0.0f));
  s += w.zl * (pc - (k > 0 ? v[id - sz] : 0.0f));
  s += w.zh * (pc - (k + 1 < nz ? v[id + sz] : 0.0f));
  return s;
}

// ---- cell-code path ------------------------------------------------------------------------------------------
// The six weights of cell (i,j,k) whose code is `code`: exactly 0.0f / 1.0f from the bits of a pure cell, the fp32
// arrays for a mixed cell (rare: O(n^2) cells).
__device__ __forceinline__ NfW6 nf_code_w6(const NfLvK &L, unsigned code, int i, int j, int k) {
  if (code & NF_CODE_MIXED) return nf_load_w6(L.ax, L.ay, L.az, i, j, k, L.nx, L.ny, L.pax);
  NfW6 w;
  w.xl = (code & 1u) ? 1.0f : 0.0f;
  w.xh = (code & 2u) ? 1.0f : 0.0f;
  w.yl = (code & 4u) ? 1.0f : 0.0f;
  w.yh = (code & 8u) ? 1.0f : 0.0f;
  w.zl = (code & 16u) ? 1.0f : 0.0f;
  w.zh = (code & 32u) ? 1.0f : 0.0f;
  return w;
}
// 1 / (c * sum of the six weights), 0 on an inactive cell.  Pure cells: (1/c) * (1/d), d = number of open faces.
static __constant__ float nf_c_inv_count[8] = {0.0f, 1.0f, 0.5f, 1.0f / 3.0f, 0.25f, 0.2f, 1.0f / 6.0f, 0.0f};
__device__ __forceinline__ float nf_code_idiag(const NfLvK &L, unsigned code, int i, int j, int k) {
  if (code & NF_CODE_MIXED) {
    const float d = nf_w6_sum(nf_load_w6(L.ax, L.ay, L.az, i, j, k, L.nx, L.ny, L.pax));
    return d > 0.0f ? L.ic / d : 0.0f;
  }
  return L.ic * nf_c_inv_count[__popc(code & 63u)];
}
// sum of the six weights
__device__ __forceinline__ float nf_code_diag(const NfLvK &L, unsigned code, int i, int j, int k) {
  if (code & NF_CODE_MIXED) return nf_w6_sum(nf_load_w6(L.ax, L.ay, L.az, i, j, k, L.nx, L.ny, L.pax));
  return (float)__popc(code & 63u);
}

// Row loads for the 4-cells-per-thread kernels (rows are 16-byte aligned: nx % 4 == 0).  `ok` false = the row lies
// outside the grid: homogeneous ghost values.
// (plain loads, no __restrict__ / __ldg: inside the persistent coarse kernel these arrays are written by other CTAs
// in earlier phases, so they must not take the non-coherent path)
__device__ __forceinline__ float4 nf_ld4(const float *p, nf_idx id, bool ok) {
  return ok ? *reinterpret_cast<const float4 *>(p + id) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
}
__device__ __forceinline__ unsigned nf_ldc4(const uint8_t *__restrict__ c, nf_idx id, bool ok) {
  return ok ? __ldg(reinterpret_cast<const unsigned *>(c + id)) : 0u;
}
__device__ __forceinline__ float nf_ld1(const float *p, nf_idx id, bool ok) { return ok ? p[id] : 0.0f; }
__device__ __forceinline__ unsigned nf_ldc1(const uint8_t *__restrict__ c, nf_idx id, bool ok) {
  return ok ? (unsigned)__ldg(c + id) : 0u;
}
__device__ __forceinline__ void nf_unpack4(const float4 v, float o[4]) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }
__device__ __forceinline__ unsigned nf_code_at(unsigned c4, int q) { return (c4 >> (8 * q)) & 255u; }
