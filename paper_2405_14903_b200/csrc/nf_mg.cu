// nf_mg.cu -- a-5 the multigrid V-cycle preconditioner z = M^{-1} r of MGPCG ("MGPCG ... hierarchical
// grid data structure, with custom CUDA kernels for prolongation and restriction").  Everything the paper leaves
// open (R13) is this library's choice: V(1,1), red-black Gauss-Seidel (pre: red->black from a
// zero guess, post: black->red), piecewise-constant prolongation P, restriction P^T/8, rediscretised coarse operators.
//
// Three families of kernels:
//   * "vec" kernels (levels with nx % 4 == 0): 4 cells per thread, float4 rows, weights from the 1-byte cell code.
//     One level of the V-cycle is 4 launches, none of them a single-colour pass over the arrays:
//       k_down1  z = pre-smooth(r)            red: z = r/diag;  black: z = (r + c sum a z_red)/diag, red values
//                                             recomputed on the fly from r (no second pass, no halo exchange)
//       k_down2  r_coarse = P^T/8 (r - A z)   only the red children contribute (the residual is zero on the cells
//                                             the last half sweep updated); for them r - A z = c sum a z_black
//       k_up1    black half sweep of the post-smoother on z + P z_coarse, prolongation evaluated on the fly
//       k_up2    red half sweep (+ r.z on level 0)
//   * generic kernels (any extents): one colour per launch, fp32 weights -- the v1 path, kept for ragged levels.
//   * k_tail: all levels that fit one CTA's shared memory (<= 5632 cells in total), whole sub-V-cycle in one launch.
#include <cooperative_groups.h>
#include <algorithm>
#include <cstring>

#include "nf_stencil.cuh"

namespace cg = cooperative_groups;

#define NF_VEC_BLOCKS (148 * 8)
#define NF_TAIL_MAX_CELLS 2048  // largest level of the shared-memory tail: a 12^3 level is cheaper inside the one-CTA tail, a 16^3 level as four grid phases (measured)
#define NF_TAIL_THREADS 1024

// ------------------------------------------------------------------------------------------------------------
// vec kernels
// ------------------------------------------------------------------------------------------------------------
struct NfRow4 {  // one row segment of 4 cells: values and codes, with the idiag-scaled value on demand
  float v[4];
  unsigned c4;
};
__device__ __forceinline__ NfRow4 nf_row(const float *f, const uint8_t *__restrict__ code, nf_idx id,
                                         bool ok) {
  NfRow4 R;
  nf_unpack4(nf_ld4(f, id, ok), R.v);
  R.c4 = nf_ldc4(code, id, ok);
  return R;
}

// PAR = (i0 + j + k) & 1 = colour of the first of the 4 cells; cell q is red iff ((q + PAR) & 1) == 0.
// R4(at, ok) / R1(at, ok): the right-hand side r on a row of 4 cells / one cell (0 when !ok).  k_down1 reads it from
// memory; k_update_down1 evaluates r - a q on the fly.  Returns the row of r of the thread's own 4 cells.
template <int PAR, class F4, class F1>
__device__ __forceinline__ float4 nf_down1_core(const NfLvK &L, F4 R4, F1 R1, float *z, int i0, int j, int k,
                                                unsigned *c4_out = nullptr) {
  const int nx = L.nx, ny = L.ny, nz = L.nz;
  const nf_idx sy = nx, sz = (nf_idx)nx * ny;
  const nf_idx id = ((nf_idx)k * ny + j) * nx + i0;
  // every load of r is issued before the branch on the code (one round trip for the common, deep path)
  NfRow4 C;
  const float4 crow = R4(id, true);
  nf_unpack4(crow, C.v);
  C.c4 = nf_ldc4(L.code, id, true);
  if (c4_out) *c4_out = C.c4;
  float out[4], yl[4], yh[4], zl[4], zh[4];
  nf_unpack4(R4(id - sy, j > 0), yl);
  nf_unpack4(R4(id + sy, j + 1 < ny), yh);
  nf_unpack4(R4(id - sz, k > 0), zl);
  nf_unpack4(R4(id + sz, k + 1 < nz), zh);
  const float re = PAR ? R1(id - 1, i0 > 0) : R1(id + 4, i0 + 4 < nx);
  if ((C.c4 & 0x80808080u) == 0x80808080u) {
    // all four cells are deep interior (NF_CODE_DEEP): every diagonal involved is 6c, every weight is 1, and no
    // neighbour code is needed
    // (L.om: over-relaxation, 1 on the finest level -- from the zero guess a red cell gets om r / diag, a black one
    // om (r + c sum of those) / diag)
    const float g6 = L.om * (L.ic * (1.0f / 6.0f));
    const float te = re;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (((q + PAR) & 1) == 0) {
        out[q] = C.v[q] * g6;
      } else {
        const float tl = q > 0 ? C.v[q - 1] : te, th = q < 3 ? C.v[q + 1] : te;
        const float sum = ((tl + th) + (yl[q] + yh[q])) + (zl[q] + zh[q]);
        out[q] = (C.v[q] + (L.om * (1.0f / 6.0f)) * sum) * g6;
      }
    }
    *reinterpret_cast<float4 *>(z + id) = make_float4(out[0], out[1], out[2], out[3]);
    return crow;
  }
  // general path: the red neighbours' values r/diag from the inverse-diagonal rows (one more round trip, no
  // dependence on the codes), the six weights of a black cell from its code
  float gyl[4], gyh[4], gzl[4], gzh[4], idg[4], t[4];
  nf_unpack4(nf_ld4(L.idg, id - sy, j > 0), gyl);
  nf_unpack4(nf_ld4(L.idg, id + sy, j + 1 < ny), gyh);
  nf_unpack4(nf_ld4(L.idg, id - sz, k > 0), gzl);
  nf_unpack4(nf_ld4(L.idg, id + sz, k + 1 < nz), gzh);
  nf_unpack4(nf_ld4(L.idg, id, true), idg);
#pragma unroll
  for (int q = 0; q < 4; ++q) t[q] = L.om * (C.v[q] * idg[q]);
  // the x-neighbour outside the segment that a black cell needs: left of q = 0 (PAR = 1) or right of q = 3 (PAR = 0)
  const float te = L.om * (re * (PAR ? nf_ld1(L.idg, id - 1, i0 > 0) : nf_ld1(L.idg, id + 4, i0 + 4 < nx)));
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (((q + PAR) & 1) == 0) {
      out[q] = t[q];  // red: z = r / diag
    } else {          // black: its six neighbours are red
      const NfW6 w = nf_code_w6(L, nf_code_at(C.c4, q), i0 + q, j, k);
      const float tl = q > 0 ? t[q - 1] : te, th = q < 3 ? t[q + 1] : te;
      float s = w.xl * tl + w.xh * th;
      s += w.yl * (L.om * (yl[q] * gyl[q]));
      s += w.yh * (L.om * (yh[q] * gyh[q]));
      s += w.zl * (L.om * (zl[q] * gzl[q]));
      s += w.zh * (L.om * (zh[q] * gzh[q]));
      out[q] = L.om * ((C.v[q] + L.c * s) * idg[q]);
    }
  }
  *reinterpret_cast<float4 *>(z + id) = make_float4(out[0], out[1], out[2], out[3]);
  return crow;
}
template <int PAR>
__device__ __forceinline__ void nf_down1_body(const NfLvK &L, const float *r, float *z, int i0, int j, int k) {
  nf_down1_core<PAR>(L, [&](nf_idx at, bool ok) { return nf_ld4(r, at, ok); },
                     [&](nf_idx at, bool ok) { return nf_ld1(r, at, ok); }, z, i0, j, k);
}

// a-4 + a-5 fused: the residual update r' = r - a q (a = rz / pq from device memory) evaluated on the fly for the row
// and its neighbour rows, ||r'||^2, and the pre-smoother z = smooth(r') in the same pass: 17 B/cell (r, q, code in;
// r', z out) instead of 12 + 9, and one kernel's fixed cost less per iteration.  r' goes to a second buffer (the
// neighbours' threads still read r).  The last CTA to finish runs the convergence check (nf_cg_check).
// (bz, nzc: this CTA's z-chunk and the number of z-chunks of ITS grid -- blockIdx.z / gridDim.z, or the environment's
// share of them in a batched launch)
__device__ __forceinline__ void nf_update_down1_body(const NfLvK &L, const float *rold,
                                                     const float *__restrict__ q, float *__restrict__ rnew,
                                                     float *__restrict__ z, int kch, NfSolveState *st, int slot,
                                                     NfHostStatus *hs, int seq, int bz, int nzc,
                                                     const float *rtrue = nullptr) {
  if (st->done) {  // (uniform: done is only ever set by the last CTA of an earlier launch)
    if (blockIdx.x == 0 && blockIdx.y == 0 && bz == 0 && threadIdx.x == 0 && threadIdx.y == 0)
      nf_cg_check(st, slot, hs, seq);
    return;
  }
  // (an accepted in-flight replacement: this iteration reads the true residual instead of the recursive one)
  if (rtrue && st->switched == 1) rold = rtrue;
  const double pq = st->pq[slot];
  const float a = (pq > 0.0) ? (float)(st->rz[slot] / pq) : 0.0f;
  // singular system: mu = mean of the residual being read (measured when it was written), taken off on the fly, so
  // that the residual stays compatible while it shrinks (NfSolveState::inv_nact; 0 = off)
  const bool proj = st->inv_nact != 0.0;
  const float mu = proj ? (float)(st->sr[1 - slot] * st->inv_nact) : 0.0f;
  const int i0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  float part = 0.0f;
  double sum = 0.0;
  if (i0 < L.nx && j < L.ny) {
    // (rows outside the grid: ghosts, 0.  Inactive cells inside it get -mu here; every use of a neighbour's value
    // multiplies it by that cell's inverse diagonal -- 0 when inactive -- or sits on the all-open fast path.)
    auto R4 = [&](nf_idx at, bool ok) {
      float4 v = nf_ld4(rold, at, ok);
      const float4 w = nf_ld4(q, at, ok);
      const float m = ok ? mu : 0.0f;
      v.x = (v.x - m) - a * w.x; v.y = (v.y - m) - a * w.y; v.z = (v.z - m) - a * w.z; v.w = (v.w - m) - a * w.w;
      return v;
    };
    auto R1 = [&](nf_idx at, bool ok) { return (nf_ld1(rold, at, ok) - (ok ? mu : 0.0f)) - a * nf_ld1(q, at, ok); };
    const int k0 = bz * kch, k1 = min(k0 + kch, L.nz);
    for (int k = k0; k < k1; ++k) {
      unsigned c4;
      float4 c = ((j + k) & 1) ? nf_down1_core<1>(L, R4, R1, z, i0, j, k, &c4) : nf_down1_core<0>(L, R4, R1, z, i0, j, k, &c4);
      if (proj) {  // the residual of an inactive cell stays 0
        c.x = (c4 & 0xffu) ? c.x : 0.0f; c.y = (c4 & 0xff00u) ? c.y : 0.0f;
        c.z = (c4 & 0xff0000u) ? c.z : 0.0f; c.w = (c4 & 0xff000000u) ? c.w : 0.0f;
        sum += (double)((c.x + c.y) + (c.z + c.w));
      }
      *reinterpret_cast<float4 *>(rnew + ((nf_idx)k * L.ny + j) * L.nx + i0) = c;
      part += (c.x * c.x + c.y * c.y) + (c.z * c.z + c.w * c.w);
    }
  }
  nf_block_atomic_add((double)part, &st->rr[slot]);
  if (proj) nf_block_atomic_add(sum, &st->sr[slot]);
  if (threadIdx.x == 0 && threadIdx.y == 0) {
    __threadfence();
    const unsigned total = gridDim.x * gridDim.y * (unsigned)nzc;
    const unsigned t = atomicAdd(&st->ticket, 1u);
    if (t == total - 1) {
      st->ticket = 0;
      __threadfence();
      nf_cg_check(st, slot, hs, seq);
    }
  }
}
__global__ void __launch_bounds__(256, 4) k_update_down1(NfLvK L, const float *__restrict__ rold,
                                                      const float *__restrict__ q, float *__restrict__ rnew,
                                                      float *__restrict__ z, int kch, NfSolveState *st, int slot,
                                                      NfHostStatus *hs, int seq, const float *rtrue) {
  nf_pdl_enter();
  nf_update_down1_body(L, rold, q, rnew, z, kch, st, slot, hs, seq, (int)blockIdx.z, (int)gridDim.z, rtrue);
}
// Batched launches: blockIdx.z = env * nzc + z-chunk; see k_papply4_b (nf_solver.cu)
__global__ void __launch_bounds__(256, 4) k_update_down1_b(const __grid_constant__ NfBatchK B, int kch, int slot,
                                                        int seq) {
  nf_pdl_enter();
  const int e = (int)blockIdx.z / B.nzc, bz = (int)blockIdx.z - e * B.nzc;
  const NfEnvK &E = B.e[e];
  nf_update_down1_body(E.L, E.r[0], E.q, E.r[1], E.z, kch, E.st, slot, E.hs, seq, bz, B.nzc);
}

__global__ void __launch_bounds__(256, 4) k_down1(NfLvK L, const float *__restrict__ r, float *__restrict__ z, int kch,
                                               const NfSolveState *st) {
  nf_pdl_enter();
  if (st && st->done) return;
  const int i0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  if (i0 >= L.nx || j >= L.ny) return;
  const int k0 = blockIdx.z * kch, k1 = min(k0 + kch, L.nz);
  for (int k = k0; k < k1; ++k) {
    if ((j + k) & 1)
      nf_down1_body<1>(L, r, z, i0, j, k);
    else
      nf_down1_body<0>(L, r, z, i0, j, k);
  }
}

// One thread per pair of coarse cells (I0, I0+1) = fine cells i0..i0+3 of the rows (2J+dj, FZ K+dk).  FZ = 2, or 1 in
// 2-D mode (one layer: 2 x 2 x 1 children, R = P^T / 4).
// GEN: the pre-smoother ran more than one sweep, so a red cell no longer holds z = r / diag: its residual is
// (r - diag z) + c sum a z_black (r is read as well).
template <int FZ, bool GEN = false>
__device__ __forceinline__ void nf_down2_body(const NfLvK &L, const float *z, float *rc, int cnx, int cny, int i0,
                                              int J, int K, const float *r = nullptr) {
  const int nx = L.nx, ny = L.ny, nz = L.nz;
  const nf_idx sy = nx, sz = (nf_idx)nx * ny;
  const int j0 = 2 * J, k0 = FZ * K;
  float zc[FZ][2][4];  // [dk][dj][q]
  unsigned cc[FZ][2];
#pragma unroll
  for (int dk = 0; dk < FZ; ++dk)
#pragma unroll
    for (int dj = 0; dj < 2; ++dj) {
      const nf_idx id = ((nf_idx)(k0 + dk) * ny + (j0 + dj)) * nx + i0;
      nf_unpack4(nf_ld4(z, id, true), zc[dk][dj]);
      cc[dk][dj] = nf_ldc4(L.code, id, true);
    }
  float acc0 = 0.0f, acc1 = 0.0f;
#pragma unroll
  for (int dk = 0; dk < FZ; ++dk)
#pragma unroll
    for (int dj = 0; dj < 2; ++dj) {
      const int j = j0 + dj, k = k0 + dk;
      const nf_idx id = ((nf_idx)k * ny + j) * nx + i0;
      const int par = (dj + dk) & 1;  // colour of q = 0 in this row (i0, j0, k0 are even)
      // the y / z neighbour rows: inside the 2x2 block or one row outside it
      float yo[4], zo[4];
      nf_unpack4(dj == 0 ? nf_ld4(z, id - sy, j > 0) : nf_ld4(z, id + sy, j + 1 < ny), yo);
      if (FZ == 2)
        nf_unpack4(dk == 0 ? nf_ld4(z, id - sz, k > 0) : nf_ld4(z, id + sz, k + 1 < nz), zo);
      else
        zo[0] = zo[1] = zo[2] = zo[3] = 0.0f;  // (one layer between closed walls: both z neighbours are ghosts)
      // (over-relaxed level, L.om != 1: the black children carry a residual too -- all four cells, both x-edges)
      const bool allc = GEN && L.om != 1.0f;
      float xel, xer;
      if (allc) {
        xel = nf_ld1(z, id - 1, i0 > 0);
        xer = nf_ld1(z, id + 4, i0 + 4 < nx);
      } else {
        xel = xer = par == 0 ? nf_ld1(z, id - 1, i0 > 0) : nf_ld1(z, id + 4, i0 + 4 < nx);
      }
      const bool open4 = (cc[dk][dj] & 0x7f7f7f7fu) == 0x3f3f3f3fu;  // all four cells: six open faces
      float rr[4];
      if (GEN) nf_unpack4(nf_ld4(r, id, true), rr);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        if (!allc && ((q + par) & 1) != 0) continue;  // red children only
        const float xl = q > 0 ? zc[dk][dj][q - 1] : xel, xh = q < 3 ? zc[dk][dj][q + 1] : xer;
        const float yl = dj == 0 ? yo[q] : zc[dk][0][q], yh = dj == 0 ? zc[dk][1][q] : yo[q];
        const float zl = dk == 0 ? zo[q] : zc[0][dj][q], zh = (FZ == 2 && dk == 0) ? zc[FZ - 1][dj][q] : zo[q];
        float s;
        if (open4) {
          s = ((xl + xh) + (yl + yh)) + (zl + zh);
          if (GEN) s += rr[q] * L.ic - 6.0f * zc[dk][dj][q];
        } else {
          const NfW6 w = nf_code_w6(L, nf_code_at(cc[dk][dj], q), i0 + q, j, k);
          s = ((w.xl * xl + w.xh * xh) + (w.yl * yl + w.yh * yh)) + (w.zl * zl + w.zh * zh);
          if (GEN) {
            const float d = nf_w6_sum(w);
            s = d > 0.0f ? s + (rr[q] * L.ic - d * zc[dk][dj][q]) : 0.0f;
          }
        }
        if (q < 2) acc0 += s; else acc1 += s;
      }
    }
  const float f = (FZ == 2 ? 0.125f : 0.25f) * L.c;
  *reinterpret_cast<float2 *>(rc + ((nf_idx)K * cny + J) * cnx + (i0 >> 1)) = make_float2(f * acc0, f * acc1);
}

// (r != nullptr: the general residual, after more than one pre-smoothing sweep)
__global__ void __launch_bounds__(256, 4) k_down2(NfLvK L, const float *__restrict__ z, float *__restrict__ rc, int cnx,
                                               int cny, int cnz, int kch, const NfSolveState *st,
                                               const float *__restrict__ r) {
  nf_pdl_enter();
  if (st && st->done) return;
  const int i0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int J = blockIdx.y * blockDim.y + threadIdx.y;
  if (i0 >= L.nx || J >= cny) return;
  const int K0 = blockIdx.z * kch, K1 = min(K0 + kch, cnz);
  if (r) {
    if (L.fz == 2) {
      for (int K = K0; K < K1; ++K) nf_down2_body<2, true>(L, z, rc, cnx, cny, i0, J, K, r);
    } else {
      for (int K = K0; K < K1; ++K) nf_down2_body<1, true>(L, z, rc, cnx, cny, i0, J, K, r);
    }
  } else if (L.fz == 2) {
    for (int K = K0; K < K1; ++K) nf_down2_body<2>(L, z, rc, cnx, cny, i0, J, K);
  } else {
    for (int K = K0; K < K1; ++K) nf_down2_body<1>(L, z, rc, cnx, cny, i0, J, K);
  }
}

__global__ void __launch_bounds__(256, 4) k_down2_b(const __grid_constant__ NfBatchK B) {
  nf_pdl_enter();
  const int e = (int)blockIdx.z / B.nzc, K = (int)blockIdx.z - e * B.nzc;  // (one coarse plane per CTA: nzc = cnz)
  const NfEnvK &E = B.e[e];
  if (E.st->done) return;
  const int i0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int J = blockIdx.y * blockDim.y + threadIdx.y;
  if (i0 >= E.L.nx || J >= B.cny) return;
  if (B.gen) {
    if (E.L.fz == 2) nf_down2_body<2, true>(E.L, E.z, E.rc, B.cnx, B.cny, i0, J, K, E.r[0]);
    else nf_down2_body<1, true>(E.L, E.z, E.rc, B.cnx, B.cny, i0, J, K, E.r[0]);
  } else if (E.L.fz == 2) nf_down2_body<2>(E.L, E.z, E.rc, B.cnx, B.cny, i0, J, K);
  else nf_down2_body<1>(E.L, E.z, E.rc, B.cnx, B.cny, i0, J, K);
}

// z + P z_coarse on a row of 4 fine cells
__device__ __forceinline__ void nf_row_prolonged(const float *z, const float *zc, nf_idx id, nf_idx cid, bool ok,
                                                 float o[4]) {
  if (ok) {
    const float4 a = *reinterpret_cast<const float4 *>(z + id);
    const float2 b = *reinterpret_cast<const float2 *>(zc + cid);
    o[0] = a.x + b.x; o[1] = a.y + b.x; o[2] = a.z + b.y; o[3] = a.w + b.y;
  } else {
    o[0] = o[1] = o[2] = o[3] = 0.0f;
  }
}

// Black half sweep on z + P zc (in place: only black cells change; red cells keep the un-prolonged value, which
// k_up2 overwrites without reading).
template <int PAR, int FZ>
__device__ __forceinline__ void nf_up1_body(const NfLvK &L, float *z, const float *r, const float *zc, int cnx,
                                            int cny, int i0, int j, int k) {
  const int nx = L.nx, ny = L.ny, nz = L.nz;
  const nf_idx sy = nx, sz = (nf_idx)nx * ny;
  const nf_idx id = ((nf_idx)k * ny + j) * nx + i0;
  const nf_idx scy = cnx, scz = (nf_idx)cnx * cny;
  const nf_idx cid = ((nf_idx)(k >> (FZ - 1)) * cny + (j >> 1)) * cnx + (i0 >> 1);  // (FZ == 1: nz == 1, no z rows)
  const float4 zold = *reinterpret_cast<const float4 *>(z + id);
  float zp[4], yl[4], yh[4], zl[4], zh[4], rr[4], out[4];
  {
    const float2 b = *reinterpret_cast<const float2 *>(zc + cid);
    zp[0] = zold.x + b.x; zp[1] = zold.y + b.x; zp[2] = zold.z + b.y; zp[3] = zold.w + b.y;
  }
  // parent row of j-1 is the same as j's iff j is odd; of j+1 iff j is even (same in z)
  nf_row_prolonged(z, zc, id - sy, (j & 1) ? cid : cid - scy, j > 0, yl);
  nf_row_prolonged(z, zc, id + sy, (j & 1) ? cid + scy : cid, j + 1 < ny, yh);
  nf_row_prolonged(z, zc, id - sz, (k & 1) ? cid : cid - scz, k > 0, zl);
  nf_row_prolonged(z, zc, id + sz, (k & 1) ? cid + scz : cid, k + 1 < nz, zh);
  nf_unpack4(nf_ld4(r, id, true), rr);
  const unsigned c4 = nf_ldc4(L.code, id, true);
  float xe;
  if (PAR) {
    const bool ok = i0 > 0;
    xe = ok ? z[id - 1] + zc[cid - 1] : 0.0f;
  } else {
    const bool ok = i0 + 4 < nx;
    xe = ok ? z[id + 4] + zc[cid + 2] : 0.0f;
  }
  out[0] = zold.x; out[1] = zold.y; out[2] = zold.z; out[3] = zold.w;
  const bool open4 = (c4 & 0x7f7f7f7fu) == 0x3f3f3f3fu;
  const float g6 = L.ic * (1.0f / 6.0f);
  float ig[4];
  nf_unpack4(nf_ld4(L.idg, id, !open4), ig);
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (((q + PAR) & 1) == 0) continue;
    const float xl = q > 0 ? zp[q - 1] : xe, xh = q < 3 ? zp[q + 1] : xe;
    // (over-relaxed, L.om != 1: the old value is the PROLONGED one; an inactive cell stays 0)
    if (open4) {
      const float s = ((xl + xh) + (yl[q] + yh[q])) + (zl[q] + zh[q]);
      out[q] = (rr[q] + L.c * s) * g6;
      if (L.om != 1.0f) out[q] = (1.0f - L.om) * zp[q] + L.om * out[q];
    } else {
      const unsigned code = nf_code_at(c4, q);
      const NfW6 w = nf_code_w6(L, code, i0 + q, j, k);
      const float s = ((w.xl * xl + w.xh * xh) + (w.yl * yl[q] + w.yh * yh[q])) + (w.zl * zl[q] + w.zh * zh[q]);
      out[q] = (rr[q] + L.c * s) * ig[q];
      if (L.om != 1.0f) out[q] = ig[q] > 0.0f ? (1.0f - L.om) * zp[q] + L.om * out[q] : 0.0f;
    }
  }
  *reinterpret_cast<float4 *>(z + id) = make_float4(out[0], out[1], out[2], out[3]);
}

__global__ void __launch_bounds__(256, 4) k_up1(NfLvK L, float *z, const float *__restrict__ r,
                                             const float *__restrict__ zc, int cnx, int cny, int kch,
                                             const NfSolveState *st) {
  nf_pdl_enter();
  if (st && st->done) return;
  const int i0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  if (i0 >= L.nx || j >= L.ny) return;
  const int k0 = blockIdx.z * kch, k1 = min(k0 + kch, L.nz);
  for (int k = k0; k < k1; ++k) {
    if (L.fz == 2) {
      if ((j + k) & 1)
        nf_up1_body<1, 2>(L, z, r, zc, cnx, cny, i0, j, k);
      else
        nf_up1_body<0, 2>(L, z, r, zc, cnx, cny, i0, j, k);
    } else {
      if ((j + k) & 1)
        nf_up1_body<1, 1>(L, z, r, zc, cnx, cny, i0, j, k);
      else
        nf_up1_body<0, 1>(L, z, r, zc, cnx, cny, i0, j, k);
    }
  }
}

__global__ void __launch_bounds__(256, 4) k_up1_b(const __grid_constant__ NfBatchK B, int kch) {
  nf_pdl_enter();
  const int e = (int)blockIdx.z / B.nzc, bz = (int)blockIdx.z - e * B.nzc;
  const NfEnvK &E = B.e[e];
  if (E.st->done) return;
  const NfLvK &L = E.L;
  const int i0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  if (i0 >= L.nx || j >= L.ny) return;
  const int k0 = bz * kch, k1 = min(k0 + kch, L.nz);
  for (int k = k0; k < k1; ++k) {
    if (L.fz == 2) {
      if ((j + k) & 1) nf_up1_body<1, 2>(L, E.z, E.r[0], E.zc, B.cnx, B.cny, i0, j, k);
      else nf_up1_body<0, 2>(L, E.z, E.r[0], E.zc, B.cnx, B.cny, i0, j, k);
    } else {
      if ((j + k) & 1) nf_up1_body<1, 1>(L, E.z, E.r[0], E.zc, B.cnx, B.cny, i0, j, k);
      else nf_up1_body<0, 1>(L, E.z, E.r[0], E.zc, B.cnx, B.cny, i0, j, k);
    }
  }
}

// Red half sweep in place (black neighbours are final); returns r.z over the 4 cells.
// zcp != nullptr (over-relaxed levels only): the cells' old values have not been prolonged yet -- the first red half sweep
// after nf_up1_body, which leaves the red cells alone; cnx, cny: the coarse level's extents.
template <int PAR>
__device__ __forceinline__ float nf_up2_body(const NfLvK &L, float *z, const float *r, int i0, int j, int k,
                                             const float *zcp = nullptr, int cnx = 0, int cny = 0) {
  const int nx = L.nx, ny = L.ny, nz = L.nz;
  const nf_idx sy = nx, sz = (nf_idx)nx * ny;
  const nf_idx id = ((nf_idx)k * ny + j) * nx + i0;
  float zc[4], yl[4], yh[4], zl[4], zh[4], rr[4];
  nf_unpack4(nf_ld4(z, id, true), zc);
  nf_unpack4(nf_ld4(z, id - sy, j > 0), yl);
  nf_unpack4(nf_ld4(z, id + sy, j + 1 < ny), yh);
  nf_unpack4(nf_ld4(z, id - sz, k > 0), zl);
  nf_unpack4(nf_ld4(z, id + sz, k + 1 < nz), zh);
  nf_unpack4(nf_ld4(r, id, true), rr);
  const unsigned c4 = nf_ldc4(L.code, id, true);
  // red q = 0 needs its left neighbour (PAR = 0), red q = 3 its right neighbour (PAR = 1)
  const float xe = PAR == 0 ? nf_ld1(z, id - 1, i0 > 0) : nf_ld1(z, id + 4, i0 + 4 < nx);
  float dot = 0.0f;
  const bool open4 = (c4 & 0x7f7f7f7fu) == 0x3f3f3f3fu;
  const float g6 = L.ic * (1.0f / 6.0f);
  float ig[4];
  nf_unpack4(nf_ld4(L.idg, id, !open4), ig);
  float pz[2] = {0.0f, 0.0f};  // the coarse values under cells 0,1 / 2,3 (over-relaxed first red sweep)
  if (zcp) {
    const float2 b = *reinterpret_cast<const float2 *>(zcp + ((nf_idx)(L.fz == 2 ? k >> 1 : k) * cny + (j >> 1)) * cnx + (i0 >> 1));
    pz[0] = b.x; pz[1] = b.y;
  }
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (((q + PAR) & 1) == 0) {
      const float xl = q > 0 ? zc[q - 1] : xe, xh = q < 3 ? zc[q + 1] : xe;
      const float zo = zc[q] + pz[q >> 1];
      if (open4) {
        const float s = ((xl + xh) + (yl[q] + yh[q])) + (zl[q] + zh[q]);
        zc[q] = (rr[q] + L.c * s) * g6;
        if (L.om != 1.0f) zc[q] = (1.0f - L.om) * zo + L.om * zc[q];
      } else {
        const unsigned code = nf_code_at(c4, q);
        const NfW6 w = nf_code_w6(L, code, i0 + q, j, k);
        const float s = ((w.xl * xl + w.xh * xh) + (w.yl * yl[q] + w.yh * yh[q])) + (w.zl * zl[q] + w.zh * zh[q]);
        zc[q] = (rr[q] + L.c * s) * ig[q];
        if (L.om != 1.0f) zc[q] = ig[q] > 0.0f ? (1.0f - L.om) * zo + L.om * zc[q] : 0.0f;
      }
    }
  }
#pragma unroll
  for (int q = 0; q < 4; ++q) dot += rr[q] * zc[q];
  *reinterpret_cast<float4 *>(z + id) = make_float4(zc[0], zc[1], zc[2], zc[3]);
  return dot;
}

// flip = 0: the red half sweep; 1: the black one (the same body on the other colour of every row)
template <bool DOT>
__global__ void __launch_bounds__(256, 4) k_up2(NfLvK L, float *z, const float *__restrict__ r, int kch,
                                             NfSolveState *st, int slot, int flip) {
  nf_pdl_enter();
  if (st && st->done) return;
  const int i0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  float dot = 0.0f;
  if (i0 < L.nx && j < L.ny) {
    const int k0 = blockIdx.z * kch, k1 = min(k0 + kch, L.nz);
    for (int k = k0; k < k1; ++k)
      dot += ((j + k + flip) & 1) ? nf_up2_body<1>(L, z, r, i0, j, k) : nf_up2_body<0>(L, z, r, i0, j, k);
  }
  if (DOT) nf_block_atomic_add((double)dot, &st->rz[slot]);
}
// (slot < 0: no r.z)
__global__ void __launch_bounds__(256, 4) k_up2_b(const __grid_constant__ NfBatchK B, int kch, int slot, int flip) {
  nf_pdl_enter();
  const int e = (int)blockIdx.z / B.nzc, bz = (int)blockIdx.z - e * B.nzc;
  const NfEnvK &E = B.e[e];
  if (E.st->done) return;  // (uniform over the environment's CTAs)
  const NfLvK &L = E.L;
  const int i0 = 4 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  float dot = 0.0f;
  if (i0 < L.nx && j < L.ny) {
    const int k0 = bz * kch, k1 = min(k0 + kch, L.nz);
    for (int k = k0; k < k1; ++k)
      dot += ((j + k + flip) & 1) ? nf_up2_body<1>(L, E.z, E.r[0], i0, j, k) : nf_up2_body<0>(L, E.z, E.r[0], i0, j, k);
  }
  if (slot >= 0) nf_block_atomic_add((double)dot, &E.st->rz[slot]);
}

// ------------------------------------------------------------------------------------------------------------
// generic kernels (any extents, fp32 weights, one colour per launch)
// ------------------------------------------------------------------------------------------------------------
// Red-black Gauss-Seidel half sweep on the cells with (i+j+k) % 2 == color.  One thread per x-pair of cells.
// ZERO: the initial guess is zero (neighbours are not read).  DOT: also accumulate r.z over BOTH cells of the pair
// (used on the last half sweep of the V-cycle on level 0, where z is final).
template <bool ZERO, bool DOT>
__global__ void __launch_bounds__(256) k_rbgs(float *__restrict__ z, const float *__restrict__ r,
                                              const float *__restrict__ ax, const float *__restrict__ ay,
                                              const float *__restrict__ az, float c, int nx, int ny, int nz, int pax,
                                              int color, NfSolveState *st, int slot, float om = 1.0f,
                                              int old_is_zero = 0) {
  if (st && st->done) return;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  double part = 0.0;
  if (j < ny && k < nz) {
    const int par = (j + k + color) & 1;
    const int i = 2 * t + par;
    if (i < nx) {
      const NfW6 w = nf_load_w6(ax, ay, az, i, j, k, nx, ny, pax);
      const size_t id = ((size_t)k * ny + j) * nx + i;
      const float d = nf_w6_sum(w);
      float zn = 0.0f;
      const float rv = r[id];
      if (d > 0.0f) {
        float s = rv;
        if (!ZERO) s += c * nf_nb_sum(z, w, i, j, k, nx, ny, nz);
        zn = s / (c * d);
        // over-relaxation (om = 1: plain Gauss-Seidel).  ZERO / old_is_zero: the cell's old value is the zero guess --
        // the array itself still holds the previous cycle's result on the cells no sweep has written yet
        if (om != 1.0f) zn = (ZERO || old_is_zero) ? om * zn : (1.0f - om) * z[id] + om * zn;
      }
      z[id] = zn;
      if (DOT) part = (double)rv * (double)zn;
    }
    if (DOT) {
      const int io = 2 * t + 1 - par;
      if (io < nx) {
        const size_t ido = ((size_t)k * ny + j) * nx + io;
        part += (double)r[ido] * (double)z[ido];
      }
    }
  }
  if (DOT) nf_block_atomic_add(part, &st->rz[slot]);
}

// r_c = (1/8) sum over the 8 children of (r_f - A_f z_f)   (R = P^T / 8, P = piecewise-constant prolongation)
__global__ void __launch_bounds__(256) k_residual_restrict(const float *__restrict__ z, const float *__restrict__ r,
                                                           const float *__restrict__ ax, const float *__restrict__ ay,
                                                           const float *__restrict__ az, float c, int nx, int ny,
                                                           int nz, int pax, float *__restrict__ rc, int cnx, int cny,
                                                           int cnz, int fz, const NfSolveState *st) {
  if (st && st->done) return;
  const int I = blockIdx.x * blockDim.x + threadIdx.x;
  const int J = blockIdx.y * blockDim.y + threadIdx.y;
  const int K = blockIdx.z * blockDim.z + threadIdx.z;
  if (I >= cnx || J >= cny || K >= cnz) return;
  float acc = 0.0f;
#pragma unroll
  for (int dk = 0; dk < 2; ++dk)
#pragma unroll
    for (int dj = 0; dj < 2; ++dj)
#pragma unroll
      for (int di = 0; di < 2; ++di) {
        if (dk >= fz) continue;  // (2-D mode: the children are the 2 x 2 x 1 cells)
        const int i = 2 * I + di, j = 2 * J + dj, k = fz * K + dk;
        if (i >= nx || j >= ny || k >= nz) continue;  // (odd extent: this child does not exist)
        const NfW6 w = nf_load_w6(ax, ay, az, i, j, k, nx, ny, pax);
        const size_t id = ((size_t)k * ny + j) * nx + i;
        acc += r[id] - c * (nf_w6_sum(w) * z[id] - nf_nb_sum(z, w, i, j, k, nx, ny, nz));
      }
  rc[((size_t)K * cny + J) * cnx + I] = (fz == 2 ? 0.125f : 0.25f) * acc;
}

// z_f += z_c[parent]   (piecewise-constant prolongation)
__global__ void __launch_bounds__(256) k_prolong_add(float *__restrict__ z, const float *__restrict__ zc, int nx,
                                                     int ny, int nz, int cnx, int cny, int fz, const NfSolveState *st) {
  if (st && st->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= nx || j >= ny || k >= nz) return;
  z[((size_t)k * ny + j) * nx + i] += __ldg(zc + ((size_t)(fz == 2 ? k >> 1 : k) * cny + (j >> 1)) * cnx + (i >> 1));
}

__global__ void __launch_bounds__(256) k_dot_rz(const float *__restrict__ a, const float *__restrict__ b, size_t n,
                                                double *dst, const NfSolveState *st) {
  if (st && st->done) return;
  double part = 0.0;
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  for (size_t t = tid; t < n; t += nth) part += (double)a[t] * (double)b[t];
  nf_block_atomic_add(part, dst);
}

// ------------------------------------------------------------------------------------------------------------
// tail: levels tail .. nlev-1 inside one CTA, everything in shared memory
// ------------------------------------------------------------------------------------------------------------
// Per level the hierarchy build packs (k_tail_pack): idg[n] = 1/(c diag) (0 inactive), wg[f][n] = c alpha_f with
// faces towards the outside of the grid zeroed, col[n] = (i+j+k) & 1 as float.  8n floats per level.
// The coarsest level (<= NF_DIRECT_MAX cells: the hierarchy halves down to extents of 2 or 3) is solved DIRECTLY with
// the inverse of its operator, computed in fp64 when the weights change (k_coarse_inverse) -- one small matrix-vector
// product instead of 2 x 8 symmetric Gauss-Seidel sweeps by one warp (measured: 6.8 us of a 20 us tail at 256^3, 9.8 us
// of 15 us at 48^3, whose coarsest level was 6^3).
#define NF_DIRECT_MAX 128
struct NfTailK {
  int nlev, sweeps;
  int npre[NF_MAX_LEVELS], npost[NF_MAX_LEVELS];  // red-black sweeps before / after the coarse correction, per level
  float om[NF_MAX_LEVELS];  // over-relaxation factor of the sweeps, per level (1 = Gauss-Seidel)
  int singular;  // the system has the constant null vector (R12): the coarsest solve works in its complement
  int direct;    // 1: the coarsest level is solved with the precomputed inverse
  int n[NF_MAX_LEVELS], nx[NF_MAX_LEVELS], ny[NF_MAX_LEVELS], nz[NF_MAX_LEVELS];
  int np[NF_MAX_LEVELS];    // n rounded up to a multiple of 4 (16-byte alignment of every block in shared memory)
  int soff[NF_MAX_LEVELS];  // float offset of the level in shared memory: z[np], r[np], pack[8 n]
  int goff[NF_MAX_LEVELS];  // float offset of the level's pack in the global pack array
  int fz[NF_MAX_LEVELS];    // z-coarsening factor towards the next level (1 in 2-D mode)
  int minv_soff;            // float offset of the coarsest inverse (n^2 floats, padded to a multiple of 4)
  int scratch_soff;         // 1024 floats of scratch (partial sums of the matrix-vector product)
  int total_floats;         // dynamic shared memory, in floats
};

__global__ void __launch_bounds__(256) k_tail_pack(const float *__restrict__ ax, const float *__restrict__ ay,
                                                   const float *__restrict__ az, float c, int nx, int ny, int nz,
                                                   int pax, float *__restrict__ pack) {
  const int n = nx * ny * nz;
  const int id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= n) return;
  const int i = id % nx, j = (id / nx) % ny, k = id / (nx * ny);
  const NfW6 w = nf_load_w6(ax, ay, az, i, j, k, nx, ny, pax);
  const float d = nf_w6_sum(w);
  pack[id] = d > 0.0f ? 1.0f / (c * d) : 0.0f;
  pack[1 * n + id] = i > 0 ? c * w.xl : 0.0f;
  pack[2 * n + id] = i + 1 < nx ? c * w.xh : 0.0f;
  pack[3 * n + id] = j > 0 ? c * w.yl : 0.0f;
  pack[4 * n + id] = j + 1 < ny ? c * w.yh : 0.0f;
  pack[5 * n + id] = k > 0 ? c * w.zl : 0.0f;
  pack[6 * n + id] = k + 1 < nz ? c * w.zh : 0.0f;
  pack[7 * n + id] = (float)((i + j + k) & 1);
}

// Inverse of the coarsest operator A_c (n <= NF_DIRECT_MAX cells) from its pack, in fp64, by in-place Gauss-Jordan
// elimination without pivoting (A_c is symmetric positive definite on the active cells; inactive cells are decoupled
// identity rows whose rows / columns of the result are zeroed).  Null spaces (R12, per component): the coarse cells
// are labelled by connected component (min-label propagation in shared memory); a component none of whose cells has an
// open face on a Dirichlet domain boundary has the constant null vector u = e / sqrt(#cells): A_c + sigma u u^T is
// inverted instead and (1/sigma) u u^T subtracted again, which leaves the pseudo-inverse.  Behind the n^2 floats of the
// inverse the kernel writes, as ints, the singular-component number of every cell (-1: none) and their count: the
// tail projects its right-hand side and its result on the complement of those null vectors.  One CTA; runs when the
// weights change (nf_build_hierarchy).
struct NfDir6 {
  int dir[6];
};
__global__ void __launch_bounds__(1024) k_coarse_inverse(const float *__restrict__ pack, int n, NfLvK Lc, NfDir6 bc,
                                                          float *__restrict__ minv) {
  extern __shared__ double sa[];
  double *a = sa, *rowk = sa + n * n, *colk = rowk + n;
  __shared__ double s_pivot, s_sig[NF_DIRECT_MAX];
  __shared__ int s_lab[NF_DIRECT_MAX], s_reg[NF_DIRECT_MAX], s_cnt[NF_DIRECT_MAX], s_id[NF_DIRECT_MAX], s_kc;
  const int nx = Lc.nx, ny = Lc.ny, nz = Lc.nz;
  const int tid = threadIdx.x, nthr = blockDim.x;
  const int off[6] = {-1, 1, -nx, nx, -nx * ny, nx * ny};
  for (int e = tid; e < n * n; e += nthr) a[e] = 0.0;
  for (int i = tid; i < n; i += nthr) {
    s_lab[i] = pack[i] > 0.0f ? i : -1;
    s_reg[i] = 0;
    s_cnt[i] = 0;
    s_sig[i] = 0.0;
    s_id[i] = -1;
  }
  __syncthreads();
  for (int i = tid; i < n; i += nthr) {
    const float idg = pack[i];
    if (idg > 0.0f) {
      a[i * n + i] = 1.0 / (double)idg;
      for (int f = 0; f < 6; ++f) {
        const float w = pack[(1 + f) * n + i];
        if (w != 0.0f) a[i * n + i + off[f]] = -(double)w;
      }
    } else {
      a[i * n + i] = 1.0;
    }
  }
  // components: min-label propagation through the open faces
  for (;;) {
    int changed = 0;
    for (int i = tid; i < n; i += nthr) {
      int m = s_lab[i];
      if (m < 0) continue;
      for (int f = 0; f < 6; ++f)
        if (pack[(1 + f) * n + i] != 0.0f) m = min(m, s_lab[i + off[f]]);
      if (m < s_lab[i]) { s_lab[i] = m; changed = 1; }
    }
    if (!__syncthreads_or(changed)) break;
  }
  // a component with an open face on a Dirichlet domain boundary is regular
  for (int i = tid; i < n; i += nthr) {
    if (s_lab[i] < 0) continue;
    const int ci = i % nx, cj = (i / nx) % ny, ck = i / (nx * ny);
    const bool edge = (ci == 0 && bc.dir[0]) || (ci == nx - 1 && bc.dir[1]) || (cj == 0 && bc.dir[2]) ||
                      (cj == ny - 1 && bc.dir[3]) || (ck == 0 && bc.dir[4]) || (ck == nz - 1 && bc.dir[5]);
    if (edge) {
      const NfW6 w = nf_load_w6(Lc.ax, Lc.ay, Lc.az, ci, cj, ck, nx, ny, Lc.pax);
      const bool open = (ci == 0 && bc.dir[0] && w.xl > 0.0f) || (ci == nx - 1 && bc.dir[1] && w.xh > 0.0f) ||
                        (cj == 0 && bc.dir[2] && w.yl > 0.0f) || (cj == ny - 1 && bc.dir[3] && w.yh > 0.0f) ||
                        (ck == 0 && bc.dir[4] && w.zl > 0.0f) || (ck == nz - 1 && bc.dir[5] && w.zh > 0.0f);
      if (open) s_reg[s_lab[i]] = 1;
    }
  }
  __syncthreads();
  if (tid == 0) {  // number the singular components; sigma = mean diagonal of the component
    int kc = 0;
    for (int i = 0; i < n; ++i) {
      const int r = s_lab[i];
      if (r < 0 || s_reg[r]) continue;
      if (s_id[r] < 0) s_id[r] = kc++;
      s_cnt[r] += 1;
      s_sig[r] += 1.0 / (double)pack[i];
    }
    for (int r = 0; r < n; ++r)
      if (s_cnt[r] > 0) s_sig[r] /= s_cnt[r];
    s_kc = kc;
  }
  __syncthreads();
  if (s_kc > 0) {
    for (int e = tid; e < n * n; e += nthr) {
      const int i = e / n, j = e - i * n;
      const int r = s_lab[i];
      if (r >= 0 && r == s_lab[j] && s_id[r] >= 0) a[e] += s_sig[r] / s_cnt[r];
    }
    __syncthreads();
  }
  for (int k = 0; k < n; ++k) {
    if (tid == 0) s_pivot = a[k * n + k];
    __syncthreads();
    const double ip = 1.0 / s_pivot;
    for (int j = tid; j < n; j += nthr) {
      rowk[j] = (j == k ? 1.0 : a[k * n + j]) * ip;
      colk[j] = a[j * n + k];
    }
    __syncthreads();
    for (int e = tid; e < n * n; e += nthr) {
      const int i = e / n, j = e - i * n;
      if (i == k) a[e] = rowk[j];
      else a[e] = (j == k ? 0.0 : a[e]) - colk[i] * rowk[j];
    }
    __syncthreads();
  }
  for (int e = tid; e < n * n; e += nthr) {
    const int i = e / n, j = e - i * n;
    const int r = s_lab[i];
    const bool act = r >= 0 && s_lab[j] >= 0;
    double v = 0.5 * (a[e] + a[j * n + i]);
    if (act && r == s_lab[j] && s_id[r] >= 0) v -= 1.0 / (s_sig[r] * s_cnt[r]);
    minv[e] = act ? (float)v : 0.0f;
  }
  int *lab_out = reinterpret_cast<int *>(minv + ((n * n + 3) & ~3));
  for (int i = tid; i < n; i += nthr) lab_out[i] = s_lab[i] >= 0 ? s_id[s_lab[i]] : -1;
  if (tid == 0) lab_out[n] = s_kc;
}

// smem per level (float offset soff[l]): z[np], r[np], pack[8n]
__device__ __forceinline__ void nf_tail_half(float *__restrict__ z, const float *__restrict__ r,
                                             const float *__restrict__ pk, int n, int nx, int sy, int sz, float color,
                                             bool zero, float om = 1.0f) {
  // nx even: the cells 2h, 2h+1 lie in one row and have different colours -- every thread updates one cell of the
  // wanted colour (no idle half); nx odd: scan all cells
  const bool pairs = (nx & 1) == 0;
  const int cnt = pairs ? (n >> 1) : n;
  for (int h = threadIdx.x; h < cnt; h += blockDim.x) {
    int id = h;
    if (pairs) {
      id = 2 * h;
      if (pk[7 * n + id] != color) id += 1;
    } else if (pk[7 * n + id] != color) {
      continue;
    }
    float a = r[id];
    if (!zero) {
      a += pk[1 * n + id] * z[max(id - 1, 0)];
      a += pk[2 * n + id] * z[min(id + 1, n - 1)];
      a += pk[3 * n + id] * z[max(id - sy, 0)];
      a += pk[4 * n + id] * z[min(id + sy, n - 1)];
      a += pk[5 * n + id] * z[max(id - sz, 0)];
      a += pk[6 * n + id] * z[min(id + sz, n - 1)];
    }
    // (over-relaxed: z = (1 - om) z + om GS; an inactive cell -- pk[id] = 0 -- stays 0 whatever the prolongation left)
    const float g = pk[id];
    z[id] = g > 0.0f ? (zero ? om * (a * g) : (1.0f - om) * z[id] + om * (a * g)) : 0.0f;
  }
  __syncthreads();
}

// v -= mean of v over the active cells (pk[id] > 0), on the active cells.  Warp 0 only; caller syncs around it.
__device__ __forceinline__ void nf_tail_project_warp(float *v, const float *pk, int n) {
  const int lane = threadIdx.x;
  float s = 0.0f, c = 0.0f;
  for (int id = lane; id < n; id += 32)
    if (pk[id] > 0.0f) {
      s += v[id];
      c += 1.0f;
    }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    s += __shfl_xor_sync(0xffffffffu, s, o);
    c += __shfl_xor_sync(0xffffffffu, c, o);
  }
  const float m = c > 0.0f ? s / c : 0.0f;
  for (int id = lane; id < n; id += 32)
    if (pk[id] > 0.0f) v[id] -= m;
  __syncwarp();
}

// v -= its mean over every singular component of the coarsest level (clab[id] = component number or -1; kc of them).
// Warp 0 only; caller syncs around it.
__device__ __forceinline__ void nf_tail_project_comps(float *v, const int *clab, int n, int kc) {
  const int lane = threadIdx.x;
  for (int c = 0; c < kc; ++c) {
    float s = 0.0f, m = 0.0f;
    for (int id = lane; id < n; id += 32)
      if (clab[id] == c) {
        s += v[id];
        m += 1.0f;
      }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      s += __shfl_xor_sync(0xffffffffu, s, o);
      m += __shfl_xor_sync(0xffffffffu, m, o);
    }
    const float mean = m > 0.0f ? s / m : 0.0f;
    for (int id = lane; id < n; id += 32)
      if (clab[id] == c) v[id] -= mean;
  }
  __syncwarp();
}

// Packed operator of the tail levels (and the coarsest inverse), global -> shared, by the bulk-copy engine
// (cp.async.bulk + mbarrier): one thread issues it, no registers are staged, and in k_vcoarse it overlaps the whole
// down sweep of the levels above.  Every block is 16-byte aligned on both sides (np, goff: NfTailK).
__device__ __forceinline__ void nf_tail_bulk(unsigned dst, const char *src, unsigned bytes, unsigned bar) {
  for (unsigned o = 0; o < bytes; o += 32768u) {
    const unsigned b = min(32768u, bytes - o);
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst + o),
                 "l"(src + o), "r"(b), "r"(bar)
                 : "memory");
  }
}
__device__ __forceinline__ void nf_tail_prefetch(const NfTailK &T, const float *__restrict__ pack_g,
                                                 const float *__restrict__ minv_g, float *sm,
                                                 unsigned long long *mbar) {  // called by ONE thread
  const unsigned bar = (unsigned)__cvta_generic_to_shared(mbar);
  asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  const int nc = T.n[T.nlev - 1];
  const unsigned mbytes = T.direct ? 4u * (unsigned)(((nc * nc + 3) & ~3) + ((nc + 1 + 3) & ~3)) : 0u;
  unsigned total = mbytes;
  for (int l = 0; l < T.nlev; ++l) total += 32u * (unsigned)T.n[l];
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(total) : "memory");
  for (int l = 0; l < T.nlev; ++l)
    nf_tail_bulk((unsigned)__cvta_generic_to_shared(sm + T.soff[l] + 2 * T.np[l]), (const char *)(pack_g + T.goff[l]),
                 32u * (unsigned)T.n[l], bar);
  if (mbytes) nf_tail_bulk((unsigned)__cvta_generic_to_shared(sm + T.minv_soff), (const char *)minv_g, mbytes, bar);
}
__device__ __forceinline__ void nf_tail_wait(unsigned long long *mbar) {
  const unsigned bar = (unsigned)__cvta_generic_to_shared(mbar);
  unsigned done = 0;
  while (!done) {
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\nselp.u32 %0, 1, 0, p;\n}"
        : "=r"(done)
        : "r"(bar)
        : "memory");
  }
}

// The sub-V-cycle of the tail levels by ONE CTA (all of its threads must call it); rg / zg: right-hand side and
// result of the first tail level in global memory (plain loads: rg may have been written in this very kernel).
// mbar != nullptr: the packs are arriving through nf_tail_prefetch -- wait for them instead of loading.
__device__ __forceinline__ void nf_tail_run(const NfTailK &T, const float *__restrict__ pack_g,
                                            const float *__restrict__ minv_g, const float *rg, float *zg, float *sm,
                                            unsigned long long *mbar) {
  const int nl = T.nlev;
  // the first level's right-hand side, zero every z (and the packs unless prefetched)
  for (int l = 0; l < nl; ++l) {
    const int n = T.n[l], np = T.np[l];
    float *base = sm + T.soff[l];
    if (!mbar) {
      const float *src = pack_g + T.goff[l];
      for (int t = threadIdx.x; t < 8 * n; t += blockDim.x) base[2 * np + t] = src[t];
    }
    for (int t = threadIdx.x; t < n; t += blockDim.x) {
      base[t] = 0.0f;
      base[np + t] = l == 0 ? rg[t] : 0.0f;
    }
  }
  if (!mbar && T.direct) {
    const int nc = T.n[nl - 1];
    const int mfl = ((nc * nc + 3) & ~3) + ((nc + 1 + 3) & ~3);  // the inverse and, behind it, the component labels
    for (int t = threadIdx.x; t < mfl; t += blockDim.x) sm[T.minv_soff + t] = minv_g[t];
  }
  if (mbar) nf_tail_wait(mbar);
  __syncthreads();
  // down
  for (int l = 0; l + 1 < nl; ++l) {
    const int n = T.n[l], nx = T.nx[l], ny = T.ny[l];
    float *z = sm + T.soff[l], *r = z + T.np[l], *pk = z + 2 * T.np[l];
    const float om = T.om[l];
    nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 0.0f, true, om);
    nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 1.0f, false, om);
    for (int s = 1; s < T.npre[l]; ++s) {
      nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 0.0f, false, om);
      nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 1.0f, false, om);
    }
    // (plain Gauss-Seidel, one sweep: the black residual is zero and a red cell holds r / diag exactly; several sweeps:
    // the red residual needs the full expression; over-relaxed: so does every child)
    const bool first_only = T.npre[l] == 1 && om == 1.0f, allc = om != 1.0f;
    // residual + restriction: r_c = 1/8 sum children (r - A z), A z = z/idg - sum wg z_nb on active cells
    const int cn = T.n[l + 1], cnx = T.nx[l + 1], cny = T.ny[l + 1], fz = T.fz[l];
    float *rc = sm + T.soff[l + 1] + T.np[l + 1];
    const int sy = nx, sz = nx * ny;
    for (int cidx = threadIdx.x; cidx < cn; cidx += blockDim.x) {
      const int I = cidx % cnx, J = (cidx / cnx) % cny, K = cidx / (cnx * cny);
      float acc = 0.0f;
#pragma unroll
      for (int dk = 0; dk < 2; ++dk)
#pragma unroll
        for (int dj = 0; dj < 2; ++dj)
#pragma unroll
          for (int di = 0; di < 2; ++di) {
            // (the residual is zero on the black cells: the black half sweep has just solved their equations)
            if ((!allc && ((di + dj + dk) & 1)) || dk >= fz) continue;
            if (2 * I + di >= nx || 2 * J + dj >= ny || fz * K + dk >= T.nz[l]) continue;  // (odd extent: no such child)
            const int id = ((fz * K + dk) * ny + (2 * J + dj)) * nx + 2 * I + di;
            const float s = pk[1 * n + id] * z[max(id - 1, 0)] + pk[2 * n + id] * z[min(id + 1, n - 1)] +
                      pk[3 * n + id] * z[max(id - sy, 0)] + pk[4 * n + id] * z[min(id + sy, n - 1)] +
                      pk[5 * n + id] * z[max(id - sz, 0)] + pk[6 * n + id] * z[min(id + sz, n - 1)];
            // (after ONE sweep a red cell holds z = r idg exactly, so r - A z = c sum alpha z_nb there; inactive:
            // weights 0.  After more sweeps the red value has been updated: the full expression)
            const float g = pk[id];
            acc += first_only ? s : (g > 0.0f ? s + (r[id] - z[id] / g) : 0.0f);
          }
      rc[cidx] = (fz == 2 ? 0.125f : 0.25f) * acc;
    }
    __syncthreads();
  }
  // coarsest level
  {
    const int l = nl - 1;
    const int n = T.n[l], nx = T.nx[l], ny = T.ny[l];
    float *z = sm + T.soff[l], *r = z + T.np[l], *pk = z + 2 * T.np[l];
    // Singular system: the restricted residual is compatible (zero sum over the active cells) only up to rounding,
    // and an (almost) exact solve would amplify what is left into a huge constant in z (which, prolonged, ends up
    // dominating the search direction: PCG then stalls near 1e-5 and diverges).  Solve in the complement of the
    // constant: project r before and z after (P M_c P stays symmetric).
    const int *clab = reinterpret_cast<const int *>(sm + T.minv_soff + ((n * n + 3) & ~3));
    const int kc = T.direct ? clab[n] : 0;  // singular components of the coarsest level (k_coarse_inverse)
    if (T.direct ? kc > 0 : T.singular != 0) {
      if (threadIdx.x < 32) {
        if (T.direct) nf_tail_project_comps(r, clab, n, kc);
        else nf_tail_project_warp(r, pk, n);
      }
      __syncthreads();
    }
    if (T.direct) {
      // z = A_c^{-1} r with the precomputed (symmetric) inverse: thread (part, i) sums a slice of column i -- read as
      // row-major mi[j n + i], conflict-free across i -- and the slices are added through the scratch block
      const float *mi = sm + T.minv_soff;
      float *scr = sm + T.scratch_soff;
      const int parts = min((int)blockDim.x / n, 8);
      const int part = threadIdx.x / n, i = threadIdx.x - part * n;
      if (part < parts) {
        const int j0 = part * n / parts, j1 = (part + 1) * n / parts;
        float acc = 0.0f;
        for (int j = j0; j < j1; ++j) acc += mi[j * n + i] * r[j];
        scr[part * n + i] = acc;
      }
      __syncthreads();
      if (threadIdx.x < n) {
        float acc = 0.0f;
        for (int p = 0; p < parts; ++p) acc += scr[p * n + threadIdx.x];
        z[threadIdx.x] = acc;
      }
      __syncthreads();
    } else {  // (a coarsest level with more than NF_DIRECT_MAX cells -- odd extents high up: symmetric sweeps)
      for (int s = 0; s < T.sweeps; ++s) {
        nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 0.0f, s == 0);
        nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 1.0f, false);
      }
      for (int s = 0; s < T.sweeps; ++s) {
        nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 1.0f, false);
        nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 0.0f, false);
      }
    }
    if (T.direct ? kc > 0 : T.singular != 0) {
      if (threadIdx.x < 32) {
        if (T.direct) nf_tail_project_comps(z, clab, n, kc);
        else nf_tail_project_warp(z, pk, n);
      }
      __syncthreads();
    }
  }
  // up
  for (int l = nl - 2; l >= 0; --l) {
    const int n = T.n[l], nx = T.nx[l], ny = T.ny[l];
    float *z = sm + T.soff[l], *r = z + T.np[l], *pk = z + 2 * T.np[l];
    const int cnx = T.nx[l + 1], cny = T.ny[l + 1], fz = T.fz[l];
    const float *zc = sm + T.soff[l + 1];
    for (int id = threadIdx.x; id < n; id += blockDim.x) {
      const int i = id % nx, j = (id / nx) % ny, k = id / (nx * ny);
      z[id] += zc[((fz == 2 ? k >> 1 : k) * cny + (j >> 1)) * cnx + (i >> 1)];
    }
    __syncthreads();
    for (int s = 0; s < T.npost[l]; ++s) {
      nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 1.0f, false, T.om[l]);
      nf_tail_half(z, r, pk, n, nx, nx, nx * ny, 0.0f, false, T.om[l]);
    }
  }
  for (int t = threadIdx.x; t < T.n[0]; t += blockDim.x) zg[t] = sm[T.soff[0] + t];
}

__global__ void __launch_bounds__(NF_TAIL_THREADS) k_tail(NfTailK T, const float *__restrict__ pack_g,
                                                           const float *__restrict__ minv_g,
                                                           const float *__restrict__ rg, float *__restrict__ zg,
                                                           const NfSolveState *st) {
  if (st && st->done) return;
  extern __shared__ __align__(16) float sm[];
  __shared__ unsigned long long mbar;
  if (threadIdx.x == 0) nf_tail_prefetch(T, pack_g, minv_g, sm, &mbar);
  __syncthreads();
  nf_tail_run(T, pack_g, minv_g, rg, zg, sm, &mbar);
}

// ------------------------------------------------------------------------------------------------------------
// persistent coarse part of the V-cycle: every level below the finest one in ONE cooperative launch
// ------------------------------------------------------------------------------------------------------------
// Levels first .. nb-1 run the vec bodies with grid-stride loops over the (4-cell row, j, k) tasks; phases are
// separated by grid barriers instead of kernel boundaries (all of these levels are L2-resident at 256^3: 128^3 and
// below), and CTA 0 runs the shared-memory tail between the down and the up sweep.
// Per-cell ("dense") phases for the small levels (64^3 and below): one thread per cell, operator from the level's pack
// (pk[0] = 1/(c diag), pk[1..6] = c alpha_f with faces towards the outside zeroed), every load issued up front -- ONE
// round trip per phase.  (The 4-cells-per-thread code path costs two to three dependent round trips around a cut cell
// -- code, then inverse diagonals, then fp32 weights -- and a grid-synchronised phase lasts as long as its slowest warp.)
// Same arithmetic as the tail (nf_tail_half) and, up to rounding order, as the vec bodies.
struct NfDenseLv {
  const float *pk;
  float *z, *r;
  int nx, ny, nz, n;
};
__device__ __forceinline__ void nf_dense_nb(const NfDenseLv &D, int id, int nb[6]) {
  const int sy = D.nx, sz = D.nx * D.ny;
  nb[0] = max(id - 1, 0); nb[1] = min(id + 1, D.n - 1);
  nb[2] = max(id - sy, 0); nb[3] = min(id + sy, D.n - 1);
  nb[4] = max(id - sz, 0); nb[5] = min(id + sz, D.n - 1);
}
// pre-smooth from a zero guess, both colours in one phase: red z = r idg; black from its red neighbours' r idg
// (om: over-relaxation factor; from the zero guess both colours are om times the Gauss-Seidel value)
__device__ __forceinline__ void nf_dense_down1(const NfDenseLv &D, int id, float om) {
  const int i = id % D.nx, j = (id / D.nx) % D.ny, k = id / (D.nx * D.ny);
  const float idg = D.pk[id], rv = D.r[id];
  float a = rv;
  if ((i + j + k) & 1) {
    int nb[6];
    nf_dense_nb(D, id, nb);
#pragma unroll
    for (int f = 0; f < 6; ++f) a += D.pk[(1 + f) * D.n + id] * (om * (D.r[nb[f]] * D.pk[nb[f]]));
  }
  D.z[id] = om * (a * idg);
}
// residual + restriction of the coarse cell cid: red children only (the black residual is zero)
// (allc: over-relaxed sweeps leave a residual on the black cells too -- all eight children, full expression)
__device__ __forceinline__ void nf_dense_down2(const NfDenseLv &D, float *rc, int cnx, int cny, int cid, bool gen,
                                               bool allc = false) {
  const int I = cid % cnx, J = (cid / cnx) % cny, K = cid / (cnx * cny);
  float acc = 0.0f;
#pragma unroll
  for (int dk = 0; dk < 2; ++dk)
#pragma unroll
    for (int dj = 0; dj < 2; ++dj)
#pragma unroll
      for (int di = 0; di < 2; ++di) {
        if (!allc && ((di + dj + dk) & 1)) continue;
        const int id = ((2 * K + dk) * D.ny + (2 * J + dj)) * D.nx + 2 * I + di;
        int nb[6];
        nf_dense_nb(D, id, nb);
        float s = 0.0f;
#pragma unroll
        for (int f = 0; f < 6; ++f) s += D.pk[(1 + f) * D.n + id] * D.z[nb[f]];
        // (after ONE sweep r - A z = c sum alpha z_nb on a red cell: z = r / diag there; after more, the full expression)
        const float g = D.pk[id];
        if (g > 0.0f) acc += gen ? s + (D.r[id] - D.z[id] / g) : s;
      }
  rc[cid] = 0.125f * acc;
}
// black half sweep on z + P zc (red cells keep the un-prolonged value; the red sweep does not read it)
__device__ __forceinline__ void nf_dense_up1(const NfDenseLv &D, const float *zc, int cnx, int cny, int id, float om) {
  const int i = id % D.nx, j = (id / D.nx) % D.ny, k = id / (D.nx * D.ny);
  if (((i + j + k) & 1) == 0) return;
  int nb[6];
  nf_dense_nb(D, id, nb);
  const int di[6] = {-1, 1, 0, 0, 0, 0}, dj[6] = {0, 0, -1, 1, 0, 0}, dk[6] = {0, 0, 0, 0, -1, 1};
  float a = D.r[id];
#pragma unroll
  for (int f = 0; f < 6; ++f) {
    const int ii = min(max(i + di[f], 0), D.nx - 1), jj = min(max(j + dj[f], 0), D.ny - 1),
              kk = min(max(k + dk[f], 0), D.nz - 1);
    a += D.pk[(1 + f) * D.n + id] * (D.z[nb[f]] + zc[((kk >> 1) * cny + (jj >> 1)) * cnx + (ii >> 1)]);
  }
  const float g = D.pk[id];
  // (over-relaxed: the old value is the PROLONGED one; an inactive cell stays 0)
  const float zo = om != 1.0f ? D.z[id] + zc[((k >> 1) * cny + (j >> 1)) * cnx + (i >> 1)] : 0.0f;
  D.z[id] = g > 0.0f ? (1.0f - om) * zo + om * (a * g) : 0.0f;
}
// half sweep on the cells of one colour (0 = red, 1 = black)
// (om: over-relaxation; zc != nullptr: the cell's old value has not been prolonged yet -- the first red half sweep
// after nf_dense_up1, which leaves the red cells alone)
__device__ __forceinline__ void nf_dense_up2(const NfDenseLv &D, int id, int color, float om, const float *zc, int cnx,
                                             int cny) {
  const int i = id % D.nx, j = (id / D.nx) % D.ny, k = id / (D.nx * D.ny);
  if (((i + j + k) & 1) != color) return;
  int nb[6];
  nf_dense_nb(D, id, nb);
  float a = D.r[id];
#pragma unroll
  for (int f = 0; f < 6; ++f) a += D.pk[(1 + f) * D.n + id] * D.z[nb[f]];
  const float g = D.pk[id];
  float zo = 0.0f;
  if (om != 1.0f) zo = D.z[id] + (zc ? zc[((k >> 1) * cny + (j >> 1)) * cnx + (i >> 1)] : 0.0f);
  D.z[id] = g > 0.0f ? (1.0f - om) * zo + om * (a * g) : 0.0f;
}

struct NfCoarseK {
  int first, nb, has_tail;
  int dense_from;  // levels >= dense_from (and < nb) run the per-cell phases
  int nu[NF_MAX_LEVELS];  // red-black sweeps before and after the coarse correction, per level
  float om[NF_MAX_LEVELS];  // over-relaxation factor of the per-cell (dense) levels' sweeps; 1 elsewhere
  const float *pk[NF_MAX_LEVELS];
  NfLvK lv[NF_MAX_LEVELS];
  float *z[NF_MAX_LEVELS], *r[NF_MAX_LEVELS];
  NfTailK T;
  const float *pack;
  const float *minv;  // inverse of the coarsest operator (k_coarse_inverse)
};

// The body: `cta` of `nctas` CTAs work on one environment's coarse levels; SYNC() is the barrier among exactly those.
// MODE 2: some level runs more than one sweep (P.nu).  MODE 1: one sweep everywhere, but over-relaxed on the per-cell
// levels (general residual of all children, no sweep loops).  MODE 0: V(1,1) Gauss-Seidel, which carries none of that
// code: unused, it still cost 2 - 8 us per launch (register allocation and a colder instruction cache: 91 -> 99 us at
// 256^3, 53 -> 57 at 128^3; the over-relaxed V(1,1) of a 128^3 grid ran 14 us slower inside the MODE 2 instance).
// FLAT: 2-D mode (nz == 1: 2 x 2 x 1 children); the 3-D instance carries none of those bodies either.
template <int MODE, bool FLAT, class SYNC>
__device__ __forceinline__ void nf_vcoarse_body(const NfCoarseK &P, int cta, int nctas, float *sm,
                                                unsigned long long *mbar, SYNC sync) {
  if (P.has_tail && cta == 0 && threadIdx.x == 0) nf_tail_prefetch(P.T, P.pack, P.minv, sm, mbar);
  // task index: warps are dealt round-robin over the CTAs so that a small level still spreads over every SM
  const int gn = nctas * blockDim.x;  // (tasks < 2^31)
  const int gt = ((threadIdx.x >> 5) * nctas + cta) * 32 + (threadIdx.x & 31);
  // The static data of the small levels (codes, inverse diagonals, fp32 weights) was evicted from L2 by the fine
  // level's streaming passes: pull it back with L2 prefetches now, off the critical path of the phases below.
  for (int l = P.first; l < P.nb; ++l) {
    const NfLvK &L = P.lv[l];
    const size_t nc = (size_t)L.nx * L.ny * L.nz;
    for (size_t o = (size_t)gt * 128; o < nc; o += (size_t)gn * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(L.code + o));
    if (l >= P.dense_from) {
      for (size_t o = (size_t)gt * 32; o < 8 * nc; o += (size_t)gn * 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(P.pk[l] + o));
    } else if (l >= 2) {
      const size_t nxf = (size_t)L.nz * L.ny * L.pax, nyf = (size_t)L.nz * (L.ny + 1) * L.nx, nzf = (size_t)(L.nz + 1) * L.ny * L.nx;
      for (size_t o = (size_t)gt * 32; o < nc; o += (size_t)gn * 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(L.idg + o));
      for (size_t o = (size_t)gt * 32; o < nxf; o += (size_t)gn * 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(L.ax + o));
      for (size_t o = (size_t)gt * 32; o < nyf; o += (size_t)gn * 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(L.ay + o));
      for (size_t o = (size_t)gt * 32; o < nzf; o += (size_t)gn * 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(L.az + o));
    }
  }
  // one half sweep of level l as a phase: color 0 = red, 1 = black
  auto half = [&](int l, int color, const float *zcp) {
    const NfLvK &L = P.lv[l];
    if (l >= P.dense_from) {
      NfDenseLv D;
      D.pk = P.pk[l]; D.z = P.z[l]; D.r = P.r[l]; D.nx = L.nx; D.ny = L.ny; D.nz = L.nz; D.n = L.nx * L.ny * L.nz;
      for (int t = gt; t < D.n; t += gn) nf_dense_up2(D, t, color, P.om[l], zcp, P.lv[l + 1].nx, P.lv[l + 1].ny);
    } else {
      const int nx4 = L.nx >> 2, ny = L.ny, nz = L.nz;
      for (int t = gt; t < nx4 * ny * nz; t += gn) {
        const int i0 = 4 * (t % nx4), j = (t / nx4) % ny, k = t / (nx4 * ny);
        if ((j + k + color) & 1)
          nf_up2_body<1>(L, P.z[l], P.r[l], i0, j, k, zcp, P.lv[l + 1].nx, P.lv[l + 1].ny);
        else
          nf_up2_body<0>(L, P.z[l], P.r[l], i0, j, k, zcp, P.lv[l + 1].nx, P.lv[l + 1].ny);
      }
    }
  };
  for (int l = P.first; l < P.nb; ++l) {
    const NfLvK &L = P.lv[l];
    const int nx4 = L.nx >> 2, ny = L.ny, nz = L.nz;
    const int cnx = P.lv[l + 1].nx, cny = P.lv[l + 1].ny, cnz = P.lv[l + 1].nz;
    const bool dense = l >= P.dense_from;
    NfDenseLv D;
    D.pk = P.pk[l]; D.z = P.z[l]; D.r = P.r[l]; D.nx = L.nx; D.ny = ny; D.nz = nz; D.n = L.nx * ny * nz;
    if (dense) {
      for (int t = gt; t < D.n; t += gn) nf_dense_down1(D, t, P.om[l]);
    } else {
      for (int t = gt; t < nx4 * ny * nz; t += gn) {
        const int i0 = 4 * (t % nx4), j = (t / nx4) % ny, k = t / (nx4 * ny);
        if ((j + k) & 1)
          nf_down1_body<1>(L, P.r[l], P.z[l], i0, j, k);
        else
          nf_down1_body<0>(L, P.r[l], P.z[l], i0, j, k);
      }
    }
    sync();
    if (MODE == 2) {  // further pre-smoothing sweeps: red, black, red, ... (one call site: one copy of the code)
      for (int q = 0; q < 2 * (P.nu[l] - 1); ++q) {
        half(l, q & 1, nullptr);
        sync();
      }
    }
    // (the general residual is right after one sweep as well -- r - diag z is then a rounding zero on the red cells --
    // so the MODE 1 / 2 instances carry that form only)
    const bool gen = MODE != 0;
    if (dense) {
      for (int t = gt; t < cnx * cny * cnz; t += gn) nf_dense_down2(D, P.r[l + 1], cnx, cny, t, gen, MODE != 0 && P.om[l] != 1.0f);
    } else {
      for (int t = gt; t < nx4 * cny * cnz; t += gn) {
        const int i0 = 4 * (t % nx4), J = (t / nx4) % cny, K = t / (nx4 * cny);
        nf_down2_body<FLAT ? 1 : 2, MODE != 0>(L, P.z[l], P.r[l + 1], cnx, cny, i0, J, K, P.r[l]);
      }
    }
    sync();
  }
  if (P.has_tail) {
    if (cta == 0) nf_tail_run(P.T, P.pack, P.minv, P.r[P.nb], P.z[P.nb], sm, mbar);
    sync();
  }
  for (int l = P.nb - 1; l >= P.first; --l) {
    const NfLvK &L = P.lv[l];
    const int nx4 = L.nx >> 2, ny = L.ny, nz = L.nz;
    const int cnx = P.lv[l + 1].nx, cny = P.lv[l + 1].ny;
    const bool dense = l >= P.dense_from;
    NfDenseLv D;
    D.pk = P.pk[l]; D.z = P.z[l]; D.r = P.r[l]; D.nx = L.nx; D.ny = ny; D.nz = nz; D.n = L.nx * ny * nz;
    if (dense) {
      for (int t = gt; t < D.n; t += gn) nf_dense_up1(D, P.z[l + 1], cnx, cny, t, P.om[l]);
    } else {
      for (int t = gt; t < nx4 * ny * nz; t += gn) {
        const int i0 = 4 * (t % nx4), j = (t / nx4) % ny, k = t / (nx4 * ny);
        // (explicit branches: selecting the body through a conditional expression made it an indirect call --
        // un-inlined, with a stack frame; this phase took 15 us at the 128^3 level against 5 us for k_up2's)
        if ((j + k) & 1)
          nf_up1_body<1, FLAT ? 1 : 2>(L, P.z[l], P.r[l], P.z[l + 1], cnx, cny, i0, j, k);
        else
          nf_up1_body<0, FLAT ? 1 : 2>(L, P.z[l], P.r[l], P.z[l + 1], cnx, cny, i0, j, k);
      }
    }
    sync();
    // the red half sweep, then (black, red) once more per further sweep -- one call site
    for (int q = 0; q < (MODE == 2 ? 2 * P.nu[l] - 1 : 1); ++q) {
      if (q) sync();
      half(l, q & 1, q == 0 ? P.z[l + 1] : nullptr);  // (the first red half sweep prolongs its own old value)
    }
    if (l > P.first) sync();
  }
}

template <int MODE, bool FLAT>
__global__ void __launch_bounds__(NF_TAIL_THREADS, 1) k_vcoarse(const __grid_constant__ NfCoarseK P,
                                                                 const NfSolveState *st) {
  if (st && st->done) return;  // (uniform over the grid: written by an earlier kernel)
  extern __shared__ __align__(16) float sm[];
  __shared__ unsigned long long mbar;
  cg::grid_group grid = cg::this_grid();
  nf_vcoarse_body<MODE, FLAT>(P, (int)blockIdx.x, (int)gridDim.x, sm, &mbar, [&]() { grid.sync(); });
}

// Batched: ONE cooperative launch runs the coarse levels of up to NF_BATCH_MAX equally sized
// environments, `nctas` CTAs each (CTA = env * nctas + cta).  The barrier is per environment: an epoch counter in the
// environment's own word (arrive with one atomic, spin until all nctas have): environments never wait for one another,
// and one that has converged leaves at once -- after adding the arrivals it skips, so that the counter stays in step
// with the host's count of barriers per launch.
struct NfCoarseBatchK {
  int n, nctas, nbar;  // environments, CTAs per environment, barriers of one launch
  unsigned base[NF_BATCH_MAX];  // value of the environment's counter when the launch starts
  unsigned *bar[NF_BATCH_MAX];
  const NfSolveState *st[NF_BATCH_MAX];
  const NfCoarseK *P[NF_BATCH_MAX];  // (device copies: one NfCoarseK is ~1.7 KB, sixteen would not fit the parameters)
};
template <int MODE>
__global__ void __launch_bounds__(NF_TAIL_THREADS, 1) k_vcoarse_b(const __grid_constant__ NfCoarseBatchK B) {
  const int e = (int)blockIdx.x / B.nctas, cta = (int)blockIdx.x - e * B.nctas;
  unsigned *bar = B.bar[e];
  if (B.st[e] && B.st[e]->done) {
    if (threadIdx.x == 0) atomicAdd(bar, (unsigned)B.nbar);
    return;
  }
  extern __shared__ __align__(16) float sm[];
  __shared__ unsigned long long mbar;
  __shared__ NfCoarseK sP;
  {  // the environment's level table: global -> shared (one round trip)
    const int *src = reinterpret_cast<const int *>(B.P[e]);
    int *dst = reinterpret_cast<int *>(&sP);
    for (int t = threadIdx.x; t < (int)(sizeof(NfCoarseK) / sizeof(int)); t += blockDim.x) dst[t] = src[t];
  }
  __syncthreads();
  unsigned target = B.base[e];
  const unsigned nctas = (unsigned)B.nctas;
  nf_vcoarse_body<MODE, false>(sP, cta, B.nctas, sm, &mbar, [&]() {
    __syncthreads();
    if (threadIdx.x == 0) {
      __threadfence();
      atomicAdd(bar, 1u);
      target += nctas;
      while ((int)(*reinterpret_cast<volatile unsigned *>(bar) - target) < 0) {
      }
      __threadfence();
    }
    __syncthreads();
  });
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
static inline int nf_nu_coarse(const nf_grid *g, int l) { return l <= 1 ? g->nu_l1 : g->nu_deep; }
// over-relaxation of the red-black sweeps: every level below the finest (their bodies carry the old value and the full
// residual; the finest level's fused kernels are plain Gauss-Seidel), never in 2-D mode
static inline float nf_omega(const nf_grid *g, int l) { return (l >= 1 && g->nz != 1) ? g->omega_deep : 1.0f; }
// some grid-phase level of the coarse kernel runs more than one sweep
static inline int nf_coarse_mode(const nf_grid *g) {  // the instance of the coarse kernel (nf_vcoarse_body's MODE)
  if (g->nu_l1 > 1 || (g->nu_deep > 1 && g->tail > 2)) return 2;
  return (g->omega_deep != 1.0f && g->nz != 1) ? 1 : 0;
}
#define NF_TAIL_SMEM_MAX 231424  // dynamic shared memory of k_tail / k_vcoarse (226 KB of the 227 KB a CTA may use)

// Shared-memory layout of a tail that starts at level `first` (NfTailK); T.total_floats is what it needs.
static void tail_desc(const nf_grid *g, int first, NfTailK *T) {
  const int nl = g->nlev;
  T->nlev = nl - first;
  int so = 0, go = 0, m = 1;
  for (int l = first; l < nl; ++l) {
    const NfLevel &L = g->lv[l];
    const int t = l - first, n = (int)L.ncell, np = (n + 3) & ~3;
    T->n[t] = n; T->np[t] = np; T->nx[t] = L.nx; T->ny[t] = L.ny; T->nz[t] = L.nz; T->fz[t] = L.fz;
    T->soff[t] = so; T->goff[t] = go;
    so += 2 * np + 8 * n;
    so = (so + 3) & ~3;
    go += 8 * n;
    if (l == nl - 1) m = std::max(L.nx, std::max(L.ny, L.nz));
  }
  const int nc = nl > first ? (int)g->lv[nl - 1].ncell : 0;
  T->direct = (nc > 0 && nc <= NF_DIRECT_MAX) ? 1 : 0;
  T->minv_soff = so;
  if (T->direct) so += ((nc * nc + 3) & ~3) + ((nc + 1 + 3) & ~3);
  T->scratch_soff = so;
  so += 1024;
  T->total_floats = so;
  T->sweeps = 2 * m;
  for (int l = first; l < nl; ++l) {
    T->npre[l - first] = l == 0 ? g->nu_pre : nf_nu_coarse(g, l);
    T->npost[l - first] = l == 0 ? g->nu_post : nf_nu_coarse(g, l);
    T->om[l - first] = nf_omega(g, l);
  }
  T->singular = g->singular_info;  // (only read when the coarsest level is too large for the direct solve)
}
static size_t tail_smem_bytes(const nf_grid *g) {
  NfTailK T;
  tail_desc(g, g->tail, &T);
  return (size_t)T.total_floats * sizeof(float);
}

// Decide which levels form the shared-memory tail and which run the vec kernels (called from nf_grid_create).
void nf_mg_plan(nf_grid *g) {
  const int nl = g->nlev;
  int tail = nl;
  for (int l = nl - 1; l >= 0; --l) {
    if (g->lv[l].ncell > NF_TAIL_MAX_CELLS) break;
    NfTailK T;
    tail_desc(g, l, &T);
    if ((size_t)T.total_floats * sizeof(float) > NF_TAIL_SMEM_MAX) break;
    tail = l;
  }
  g->tail = tail;
  const int nb = tail < nl ? tail : nl - 1;  // levels [0, nb) have a coarser level below them
  for (int l = 0; l < nl; ++l) {
    const NfLevel &L = g->lv[l];
    const double slots = (double)(L.nz + 1) * (L.ny + 1) * (L.pax + 4);  // largest face array of the level
    g->lv[l].vec_idx32 = slots < 4.0e9 ? 1 : 0;
    // (the 4-cells-per-thread kernels work on whole 2 x 2 x 2 families: every extent even, x a multiple of 4)
    g->lv[l].vec = (l < nb && (L.nx & 3) == 0 && (L.ny & 1) == 0 && (L.fz == 1 || (L.nz & 1) == 0) && g->lv[l].vec_idx32) ? 1 : 0;
  }
}

int nf_mg_init(nf_grid *g) {
  const int smem = NF_TAIL_SMEM_MAX;
  NF_CUDA(g, cudaFuncSetAttribute(k_tail, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  NF_CUDA(g, cudaFuncSetAttribute(k_vcoarse<0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  NF_CUDA(g, cudaFuncSetAttribute(k_vcoarse<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  NF_CUDA(g, cudaFuncSetAttribute(k_vcoarse<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  NF_CUDA(g, cudaFuncSetAttribute(k_vcoarse<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  NF_CUDA(g, cudaFuncSetAttribute(k_vcoarse<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  NF_CUDA(g, cudaFuncSetAttribute(k_vcoarse_b<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem - 4096));
  NF_CUDA(g, cudaFuncSetAttribute(k_vcoarse_b<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem - 4096));
  NF_CUDA(g, cudaFuncSetAttribute(k_vcoarse_b<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem - 4096));
  NF_CUDA(g, cudaFuncSetAttribute(k_coarse_inverse, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (NF_DIRECT_MAX * NF_DIRECT_MAX + 2 * NF_DIRECT_MAX) * (int)sizeof(double)));
  // the cooperative coarse kernel: one CTA per SM; needs a tail, at least one vec level below the finest one, and
  // every level between the finest one and the tail to be a vec level
  g->coarse_ctas = 0;
  const int nl = g->nlev;
  if (g->tail < nl && g->tail >= 2) {
    bool all_vec = true;
    for (int l = 1; l < g->tail; ++l) all_vec = all_vec && g->lv[l].vec;
    int dev = 0, sms = 0, coop = 0, per_sm = 0;
    NF_CUDA(g, cudaGetDevice(&dev));
    NF_CUDA(g, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    NF_CUDA(g, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    NF_CUDA(g, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_vcoarse<2, false>, NF_TAIL_THREADS, tail_smem_bytes(g)));
    if (all_vec && coop && per_sm >= 1) {
      // One CTA per 4096 cells of the first coarse level, at least 8, at most one per SM.  A cooperative grid is
      // resident as a whole: sized for the level instead of for the machine, the coarse kernels of several small
      // grids (the paper's 40^3-64^3 environments, one handle + stream each) run side by side on disjoint SMs --
      // 8 concurrent 48^3 environments: 636 -> 1770 projection steps/s -- and the barrier is cheaper; grids with a
      // first coarse level of >= 148 x 4096 cells (>= 170^3 fine cells) keep one CTA per SM.
      const long long want = (g->lv[1].ncell + 4095) / 4096;
      g->coarse_ctas = (int)std::min<long long>(sms, std::max<long long>(8, want));
    }
  }
  return NF_OK;
}

// (re)build the packed tail arrays from the current weights
int nf_mg_pack_tail(nf_grid *g) {
  for (int l = 2; l < g->tail && l < g->nlev; ++l) {  // the per-cell levels of k_vcoarse
    NfLevel &L = g->lv[l];
    if (!L.pk) continue;
    const int n = (int)L.ncell;
    NF_LAUNCH(g, NFK_COARSEN, k_tail_pack<<<(n + 255) / 256, 256, 0, g->stream>>>(L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax, L.pk));
  }
  size_t off = 0;
  for (int l = g->tail; l < g->nlev; ++l) {
    NfLevel &L = g->lv[l];
    const int n = (int)L.ncell;
    NF_LAUNCH(g, NFK_COARSEN, k_tail_pack<<<(n + 255) / 256, 256, 0, g->stream>>>(L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax, g->tailpack + 8 * off));
    if (l == g->nlev - 1 && n <= NF_DIRECT_MAX)  // the coarsest operator's inverse (fp64 Gauss-Jordan, one CTA)
    {
      NfDir6 bc;
      for (int f = 0; f < 6; ++f) bc.dir[f] = g->bc_type[f] == NF_BC_DIRICHLET ? 1 : 0;
      NF_LAUNCH(g, NFK_COARSEN, k_coarse_inverse<<<1, 1024, (size_t)(n * n + 2 * n) * sizeof(double), g->stream>>>(g->tailpack + 8 * off, n, nf_lvk(L), bc, g->tailinv));
    }
    off += (size_t)n;
  }
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

static void smooth_half(nf_grid *g, NfLevel &L, int color, bool zero, bool dot, NfSolveState *st, int slot,
                        bool old_is_zero = false) {
  const float om = nf_omega(g, (int)(&L - &g->lv[0]));
  const int oz = old_is_zero ? 1 : 0;
  NfDims d = nf_dims((L.nx + 1) / 2, L.ny, L.nz);
  const int cls = (&L == &g->lv[0]) ? NFK_RBGS0 : NFK_RBGS_C;
  if (zero)
    NF_LAUNCH(g, cls, k_rbgs<true, false><<<d.grid, d.block, 0, g->stream>>>(L.z, L.r, L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax, color, st, slot, om, oz));
  else if (dot)
    NF_LAUNCH(g, cls, k_rbgs<false, true><<<d.grid, d.block, 0, g->stream>>>(L.z, L.r, L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax, color, st, slot, om, oz));
  else
    NF_LAUNCH(g, cls, k_rbgs<false, false><<<d.grid, d.block, 0, g->stream>>>(L.z, L.r, L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax, color, st, slot, om, oz));
}

// The level table of the cooperative coarse kernel (levels 1 .. tail-1 as grid phases, then the tail)
static void fill_coarse(const nf_grid *g, NfCoarseK *P) {
  const int nl = g->nlev, nb = g->tail < nl ? g->tail : nl - 1;
  memset(P, 0, sizeof(*P));
  P->first = 1; P->nb = nb; P->has_tail = 1;
  for (int l = 0; l < NF_MAX_LEVELS; ++l) {
    P->nu[l] = nf_nu_coarse(g, l);
    P->om[l] = nf_omega(g, l);
  }
  P->dense_from = NF_MAX_LEVELS;
  for (int l = 0; l < nl; ++l) {
    P->lv[l] = nf_lvk(g->lv[l]);
    P->lv[l].om = P->om[l];  // (the 4-cell bodies of level 1 read it from the level's own table)
    P->z[l] = g->lv[l].z;
    P->r[l] = g->lv[l].r;
    P->pk[l] = g->lv[l].pk;
    if (l >= 2 && l < nb && g->lv[l].pk && P->dense_from == NF_MAX_LEVELS) P->dense_from = l;
  }
  tail_desc(g, g->tail, &P->T);
  P->minv = g->tailinv;
  P->pack = g->tailpack;
}
// Device copy of that table for the batched kernel (k_vcoarse_b); refreshed whenever the hierarchy is rebuilt.
int nf_mg_upload_coarse(nf_grid *g) {
  if (g->coarse_ctas <= 0) return NF_OK;
  if (!g->d_coarse) NF_CUDA(g, cudaMalloc((void **)&g->d_coarse, sizeof(NfCoarseK)));
  if (!g->cbar) {
    NF_CUDA(g, cudaMalloc((void **)&g->cbar, 128));
    NF_CUDA(g, cudaMemset(g->cbar, 0, 128));
    g->cbar_count = 0;
  }
  if (!g->h_coarse) {
    NF_CUDA(g, cudaHostAlloc((void **)&g->h_coarse, sizeof(NfCoarseK), cudaHostAllocDefault));
    NF_CUDA(g, cudaEventCreateWithFlags(&g->ev_coarse, cudaEventDisableTiming));
  } else {
    NF_CUDA(g, cudaEventSynchronize(g->ev_coarse));  // (the previous upload has read the pinned buffer)
  }
  NfCoarseK *P = static_cast<NfCoarseK *>(g->h_coarse);
  // (the table's only host-read input is the global "singular" flag of a tail too large for the direct coarsest solve)
  if (!(g->lv[g->nlev - 1].ncell <= NF_DIRECT_MAX)) NF_TRY(nf_meta_sync(g));
  fill_coarse(g, P);
  NF_CUDA(g, cudaMemcpyAsync(g->d_coarse, P, sizeof(*P), cudaMemcpyHostToDevice, g->stream));
  NF_CUDA(g, cudaEventRecord(g->ev_coarse, g->stream));
  return NF_OK;
}
void nf_mg_free_batch(nf_grid *g) {
  cudaFree(g->d_coarse);
  cudaFree(g->cbar);
  if (g->h_coarse) {
    cudaFreeHost(g->h_coarse);
    cudaEventDestroy(g->ev_coarse);
  }
}

// One batched PCG iteration's V-cycle part for n environments (equal extents, same stream; checked by the caller):
// k_down2_b, k_vcoarse_b, k_up1_b, k_up2_b -- four launches for all of them.  B: filled by the caller (r[0] = the
// current residual).  slot: parity slot that receives r.z.
int nf_vcycle_batch(nf_grid **G, int n, const NfBatchK &Bin, int slot) {
  nf_grid *g = G[0];
  NfLevel &L = g->lv[0], &C = g->lv[1];
  NfBatchK B = Bin;
  const int kch = nf_kch(L.nx / 4, L.ny, L.nz, NF_KCH_MG);
  NfDims d = nf_vdims(L.nx / 4, L.ny, L.nz, kch);
  NfDims d2 = nf_vdims(L.nx / 4, C.ny, C.nz, 1);
  B.nzc = (int)d2.grid.z;
  d2.grid.z *= n;
  B.gen = g->nu_pre > 1 ? 1 : 0;
  if (g->nu_pre > 1) {  // further pre-smoothing sweeps on the finest level: red, black
    B.nzc = (int)d.grid.z;
    dim3 gs = d.grid;
    gs.z *= n;
    for (int s = 1; s < g->nu_pre; ++s)
      for (int color = 0; color < 2; ++color)
        NF_LAUNCH(g, NFK_SWEEP_0, nf_launch_pdl(k_up2_b, gs, d.block, g->stream, B, kch, -1, color));
    B.nzc = (int)(d2.grid.z / n);
  }
  NF_LAUNCH(g, NFK_DOWN2_0, nf_launch_pdl(k_down2_b, d2.grid, d2.block, g->stream, B));
  {
    NfCoarseBatchK CB;
    memset(&CB, 0, sizeof(CB));
    CB.n = n; CB.nctas = g->coarse_ctas;
    const int nb = g->tail;
    CB.nbar = 0;  // 4 nu phases per level 1 .. nb-1 (no barrier after the last), one after the tail
    for (int l = 1; l < nb; ++l) CB.nbar += 4 * nf_nu_coarse(g, l);
    for (int e = 0; e < n; ++e) {
      CB.base[e] = G[e]->cbar_count;
      CB.bar[e] = G[e]->cbar;
      CB.st[e] = G[e]->st;
      CB.P[e] = static_cast<const NfCoarseK *>(G[e]->d_coarse);
    }
    for (int e = 0; e < n; ++e) G[e]->cbar_count += (unsigned)(CB.nbar * CB.nctas);
    void *args[] = {(void *)&CB};
    NF_LAUNCH(g, NFK_VEC_C, cudaLaunchCooperativeKernel(nf_coarse_mode(g) == 2 ? (void *)k_vcoarse_b<2> : (nf_coarse_mode(g) == 1 ? (void *)k_vcoarse_b<1> : (void *)k_vcoarse_b<0>), dim3(n * g->coarse_ctas), dim3(NF_TAIL_THREADS), args, tail_smem_bytes(g), g->stream));
  }
  B.nzc = (int)d.grid.z;
  dim3 gb = d.grid;
  gb.z *= n;
  NF_LAUNCH(g, NFK_UP1_0, nf_launch_pdl(k_up1_b, gb, d.block, g->stream, B, kch));
  for (int s = 1; s < g->nu_post; ++s)
    for (int color = 0; color < 2; ++color)
      NF_LAUNCH(g, NFK_SWEEP_0, nf_launch_pdl(k_up2_b, gb, d.block, g->stream, B, kch, -1, color));
  NF_LAUNCH(g, NFK_UP2_0, nf_launch_pdl(k_up2_b, gb, d.block, g->stream, B, kch, slot, 0));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}
int nf_update_down1_batch(nf_grid **G, int n, const NfBatchK &Bin, int slot, int seq) {
  nf_grid *g = G[0];
  NfLevel &L = g->lv[0];
  NfBatchK B = Bin;
  const int kch = nf_kch(L.nx / 4, L.ny, L.nz, NF_KCH_MG);
  NfDims d = nf_vdims(L.nx / 4, L.ny, L.nz, kch);
  B.nzc = (int)d.grid.z;
  d.grid.z *= n;
  NF_LAUNCH(g, NFK_UPDATE, nf_launch_pdl(k_update_down1_b, d.grid, d.block, g->stream, B, kch, slot, seq));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

// z = M^{-1} r on level 0 (lv[0].r -> lv[0].z).  with_dot: accumulate r.z into st->rz[slot] and honour st->done.
bool nf_update_down1_ok(const nf_grid *g) {
  return g->nu_pre == g->nu_post && !g->force_generic && g->lv[0].vec && g->nlev > 1;
}
int nf_update_down1(nf_grid *g, int slot, NfHostStatus *hs, int seq, const float *rtrue) {
  NfLevel &L = g->lv[0];
  const int kch = nf_kch(L.nx / 4, L.ny, L.nz, NF_KCH_MG);
  NfDims d = nf_vdims(L.nx / 4, L.ny, L.nz, kch);
  NF_LAUNCH(g, NFK_UPDATE, nf_launch_pdl(k_update_down1, d.grid, d.block, g->stream, nf_lvk(L), (const float *)L.r, (const float *)g->q, g->r_alt, L.z, kch, g->st, slot, hs, seq, rtrue));
  float *t = L.r;
  L.r = g->r_alt;
  g->r_alt = t;
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_vcycle_impl(nf_grid *g, bool with_dot, int slot, bool skip_down1) {
  NfSolveState *st = with_dot ? g->st : nullptr;
  const int nl = g->nlev;
  const bool has_tail = g->tail < nl;
  const int nb = has_tail ? g->tail : nl - 1;
  const bool fused = g->nu_pre == g->nu_post && !g->force_generic;
  bool dot_done = false;
  const bool coop = fused && g->coarse_ctas > 0 && g->lv[0].vec;
  for (int l = 0; l < (coop ? 1 : nb); ++l) {
    NfLevel &L = g->lv[l], &C = g->lv[l + 1];
    // (the 4-cell bodies are plain Gauss-Seidel: an over-relaxed level outside the cooperative kernel runs the generic ones)
    if (L.vec && fused && nf_omega(g, l) == 1.0f) {
      const int kch = nf_kch(L.nx / 4, L.ny, L.nz, NF_KCH_MG);
      NfDims d = nf_vdims(L.nx / 4, L.ny, L.nz, kch);
      const int nu = l == 0 ? g->nu_pre : nf_nu_coarse(g, l);
      if (!(l == 0 && skip_down1))
        NF_LAUNCH(g, (l == 0 ? NFK_DOWN1_0 : NFK_VEC_C), nf_launch_pdl(k_down1, d.grid, d.block, g->stream, nf_lvk(L), L.r, L.z, kch, (const NfSolveState *)st));
      for (int s = 1; s < nu; ++s)  // further sweeps: red, black
        for (int color = 0; color < 2; ++color)
          NF_LAUNCH(g, (l == 0 ? NFK_SWEEP_0 : NFK_VEC_C), nf_launch_pdl(k_up2<false>, d.grid, d.block, g->stream, nf_lvk(L), L.z, (const float *)L.r, kch, st, slot, color));
      NfDims d2 = nf_vdims(L.nx / 4, C.ny, C.nz, 1);
      NF_LAUNCH(g, (l == 0 ? NFK_DOWN2_0 : NFK_VEC_C), nf_launch_pdl(k_down2, d2.grid, d2.block, g->stream, nf_lvk(L), L.z, C.r, C.nx, C.ny, C.nz, 1, (const NfSolveState *)st, (const float *)(nu > 1 ? L.r : nullptr)));
    } else {
      for (int s = 0; s < (l == 0 ? g->nu_pre : nf_nu_coarse(g, l)); ++s) {
        smooth_half(g, L, 0, s == 0, false, st, slot);
        smooth_half(g, L, 1, false, false, st, slot, s == 0);  // (first black half sweep: its own old value is the zero guess)
      }
      NfDims d = nf_dims(C.nx, C.ny, C.nz);
      NF_LAUNCH(g, (l == 0 ? NFK_RESTRICT0 : NFK_RESTRICT_C), k_residual_restrict<<<d.grid, d.block, 0, g->stream>>>(L.z, L.r, L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax, C.r, C.nx, C.ny, C.nz, L.fz, st));
    }
  }
  if (coop) {
    NfCoarseK P;
    fill_coarse(g, &P);
    const NfSolveState *stc = st;
    void *args[] = {(void *)&P, (void *)&stc};
    const int mode = nf_coarse_mode(g);
    const bool flat = g->nz == 1;  // (2-D grids are never over-relaxed: mode 0 or 2)
    void *kfun = flat ? (mode == 2 ? (void *)k_vcoarse<2, true> : (void *)k_vcoarse<0, true>)
                      : (mode == 2 ? (void *)k_vcoarse<2, false>
                                   : (mode == 1 ? (void *)k_vcoarse<1, false> : (void *)k_vcoarse<0, false>));
    NF_LAUNCH(g, NFK_VEC_C, cudaLaunchCooperativeKernel(kfun, dim3(g->coarse_ctas), dim3(NF_TAIL_THREADS), args, tail_smem_bytes(g), g->stream));
  } else if (has_tail) {
    NfTailK T;
    tail_desc(g, g->tail, &T);
    NfLevel &F = g->lv[g->tail];
    NF_LAUNCH(g, NFK_BOTTOM, k_tail<<<1, NF_TAIL_THREADS, tail_smem_bytes(g), g->stream>>>(T, g->tailpack, g->tailinv, F.r, F.z, st));
  } else {  // coarsest level too large for one CTA (odd extents): a few symmetric sweeps in global memory
    NfLevel &B = g->lv[nl - 1];
    const int nsw = 4;
    for (int s = 0; s < nsw; ++s) {
      smooth_half(g, B, 0, s == 0, false, st, slot);
      smooth_half(g, B, 1, false, false, st, slot);
    }
    for (int s = 0; s < nsw; ++s) {
      smooth_half(g, B, 1, false, false, st, slot);
      smooth_half(g, B, 0, false, false, st, slot);
    }
  }
  for (int l = (coop ? 0 : nb - 1); l >= 0; --l) {
    NfLevel &L = g->lv[l], &C = g->lv[l + 1];
    if (L.vec && fused && nf_omega(g, l) == 1.0f) {
      const int kch = nf_kch(L.nx / 4, L.ny, L.nz, NF_KCH_MG);
      NfDims d = nf_vdims(L.nx / 4, L.ny, L.nz, kch);
      const int nu = l == 0 ? g->nu_post : nf_nu_coarse(g, l);
      NF_LAUNCH(g, (l == 0 ? NFK_UP1_0 : NFK_VEC_C), nf_launch_pdl(k_up1, d.grid, d.block, g->stream, nf_lvk(L), L.z, L.r, C.z, C.nx, C.ny, kch, (const NfSolveState *)st));
      for (int s = 1; s < nu; ++s)  // (up1 was the first black half sweep) red, then the next black one
        for (int color = 0; color < 2; ++color)
          NF_LAUNCH(g, (l == 0 ? NFK_SWEEP_0 : NFK_VEC_C), nf_launch_pdl(k_up2<false>, d.grid, d.block, g->stream, nf_lvk(L), L.z, (const float *)L.r, kch, st, slot, color));
      if (l == 0 && with_dot) {
        NF_LAUNCH(g, NFK_UP2_0, nf_launch_pdl(k_up2<true>, d.grid, d.block, g->stream, nf_lvk(L), L.z, (const float *)L.r, kch, g->st, slot, 0));
        dot_done = true;
      } else {
        NF_LAUNCH(g, (l == 0 ? NFK_UP2_0 : NFK_VEC_C), nf_launch_pdl(k_up2<false>, d.grid, d.block, g->stream, nf_lvk(L), L.z, (const float *)L.r, kch, st, slot, 0));
      }
    } else {
      NfDims d = nf_dims(L.nx, L.ny, L.nz);
      NF_LAUNCH(g, (l == 0 ? NFK_PROLONG0 : NFK_PROLONG_C), k_prolong_add<<<d.grid, d.block, 0, g->stream>>>(L.z, C.z, L.nx, L.ny, L.nz, C.nx, C.ny, L.fz, st));
      const int nu = l == 0 ? g->nu_post : nf_nu_coarse(g, l);
      for (int s = 0; s < nu; ++s) {
        const bool dot = with_dot && l == 0 && s == nu - 1;
        smooth_half(g, L, 1, false, false, st, slot);
        smooth_half(g, L, 0, false, dot, st, slot);
        dot_done = dot_done || dot;
      }
    }
  }
  if (with_dot && !dot_done) {
    NfLevel &L = g->lv[0];
    NF_LAUNCH(g, NFK_MISC, k_dot_rz<<<NF_VEC_BLOCKS, 256, 0, g->stream>>>(L.r, L.z, (size_t)L.ncell, &g->st->rz[slot], st));
  }
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}
