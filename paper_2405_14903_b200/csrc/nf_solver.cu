// nf_solver.cu -- a-3 weighted 7-point Laplacian apply, a-4 CG vector ops with device-resident scalars,
// a-5 multigrid V-cycle preconditioner, and the host loop of MGPCG.
// Everything the paper leaves open (smoother, transfers, coarse weights, coarse solve; R13) is described in
// DESIGN.md section 6.
#include <chrono>
#include <thread>

#include "nf_internal.cuh"

#define NF_VEC_BLOCKS (148 * 8)
#define NF_BOTTOM_MAX_CELLS 4096
#define NF_LOOKAHEAD 2

// ------------------------------------------------------------------------------------------------------------
// cell-local helpers
// ------------------------------------------------------------------------------------------------------------
struct NfW6 {
  float xl, xh, yl, yh, zl, zh;
};
__device__ __forceinline__ NfW6 nf_load_w6(const float *__restrict__ ax, const float *__restrict__ ay,
                                           const float *__restrict__ az, int i, int j, int k, int nx, int ny, int pax) {
  NfW6 w;
  const size_t rx = ((size_t)k * ny + j) * pax + i;
  w.xl = __ldg(ax + rx);
  w.xh = __ldg(ax + rx + 1);
  const size_t ry = ((size_t)k * (ny + 1) + j) * nx + i;
  w.yl = __ldg(ay + ry);
  w.yh = __ldg(ay + ry + nx);
  const size_t rz = ((size_t)k * ny + j) * nx + i;
  w.zl = __ldg(az + rz);
  w.zh = __ldg(az + rz + (size_t)ny * nx);
  return w;
}
// sum over the six neighbours of alpha_f * v_nb with homogeneous ghosts (v = 0 outside the grid)
__device__ __forceinline__ float nf_nb_sum(const float *__restrict__ v, const NfW6 &w, int i, int j, int k, int nx,
                                           int ny, int nz) {
  const size_t id = ((size_t)k * ny + j) * nx + i;
  const size_t sy = nx, sz = (size_t)nx * ny;
  float s = 0.0f;
  if (i > 0) s += w.xl * v[id - 1];
  if (i + 1 < nx) s += w.xh * v[id + 1];
  if (j > 0) s += w.yl * v[id - sy];
  if (j + 1 < ny) s += w.yh * v[id + sy];
  if (k > 0) s += w.zl * v[id - sz];
  if (k + 1 < nz) s += w.zh * v[id + sz];
  return s;
}

// ------------------------------------------------------------------------------------------------------------
// a-3  q = A p = c (sum_f alpha_f (p - p_nb)), fused p.q partial sums
// ------------------------------------------------------------------------------------------------------------
template <bool DOT>
__global__ void __launch_bounds__(256) k_apply_A(const float *__restrict__ p, const float *__restrict__ ax,
                                                 const float *__restrict__ ay, const float *__restrict__ az,
                                                 float *__restrict__ q, float c, int nx, int ny, int nz, int pax,
                                                 NfSolveState *st, int slot) {
  if (DOT && st->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  double part = 0.0;
  if (i < nx && j < ny && k < nz) {
    const NfW6 w = nf_load_w6(ax, ay, az, i, j, k, nx, ny, pax);
    const size_t id = ((size_t)k * ny + j) * nx + i;
    const float pc = p[id];
    const float d = ((w.xl + w.xh) + (w.yl + w.yh)) + (w.zl + w.zh);
    const float qv = c * (d * pc - nf_nb_sum(p, w, i, j, k, nx, ny, nz));
    q[id] = qv;
    part = (double)pc * (double)qv;
  }
  if (DOT) nf_block_atomic_add(part, &st->pq[slot]);
}

// ------------------------------------------------------------------------------------------------------------
// a-4  CG vector ops
// ------------------------------------------------------------------------------------------------------------
// x += a p ; r -= a q ; rr += r.r      a = rz/pq read from device memory
__global__ void __launch_bounds__(256) k_cg_update(float *__restrict__ x, float *__restrict__ r,
                                                   const float *__restrict__ p, const float *__restrict__ q, size_t n,
                                                   int vec4, NfSolveState *st, int slot) {
  if (st->done) return;
  const double pq = st->pq[slot];
  const float a = (pq > 0.0) ? (float)(st->rz[slot] / pq) : 0.0f;
  double part = 0.0;
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  if (vec4) {
    const size_t n4 = n >> 2;
    float4 *x4 = (float4 *)x, *r4 = (float4 *)r;
    const float4 *p4 = (const float4 *)p, *q4 = (const float4 *)q;
    for (size_t t = tid; t < n4; t += nth) {
      float4 xv = x4[t], rv = r4[t];
      const float4 pv = p4[t], qv = q4[t];
      xv.x += a * pv.x; xv.y += a * pv.y; xv.z += a * pv.z; xv.w += a * pv.w;
      rv.x -= a * qv.x; rv.y -= a * qv.y; rv.z -= a * qv.z; rv.w -= a * qv.w;
      x4[t] = xv;
      r4[t] = rv;
      part += ((double)rv.x * rv.x + (double)rv.y * rv.y) + ((double)rv.z * rv.z + (double)rv.w * rv.w);
    }
  } else {
    for (size_t t = tid; t < n; t += nth) {
      const float rv = r[t] - a * q[t];
      x[t] += a * p[t];
      r[t] = rv;
      part += (double)rv * rv;
    }
  }
  nf_block_atomic_add(part, &st->rr[slot]);
}

// One thread: advance the iteration counter, decide convergence (R11), publish the status to the mapped host
// ring, and clear the accumulators of the other parity slot.
__global__ void k_cg_check(NfSolveState *st, int slot, NfHostStatus *hs, int seq) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  if (!st->done) {
    st->iter += 1;
    const double rr = st->rr[slot];
    if (!(rr == rr) || rr <= st->tol2 * st->bb) {
      st->done = 1;
      st->converged = (rr == rr) ? 1 : 0;
    } else if (st->iter >= st->maxit) {
      st->done = 1;
      st->converged = 0;
    }
    st->pq[1 - slot] = 0.0;
    st->rr[1 - slot] = 0.0;
    st->rz[1 - slot] = 0.0;
    st->relres = st->bb > 0.0 ? sqrt(rr / st->bb) : 0.0;
  }
  hs->relres = (float)st->relres;
  hs->iter = st->iter;
  hs->done = st->done;
  hs->converged = st->converged;
  __threadfence_system();
  hs->seq = seq;
  __threadfence_system();
}

// p = z + beta p,  beta = rz_new/rz_old (first: p = z)
__global__ void __launch_bounds__(256) k_cg_pupdate(float *__restrict__ p, const float *__restrict__ z, size_t n,
                                                    int vec4, const NfSolveState *st, int slot, int first) {
  if (st->done) return;
  float beta = 0.0f;
  if (!first) {
    const double rz_old = st->rz[slot];
    beta = rz_old != 0.0 ? (float)(st->rz[1 - slot] / rz_old) : 0.0f;
  }
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  if (vec4) {
    const size_t n4 = n >> 2;
    float4 *p4 = (float4 *)p;
    const float4 *z4 = (const float4 *)z;
    for (size_t t = tid; t < n4; t += nth) {
      const float4 zv = z4[t];
      float4 pv = zv;
      if (!first) {  // (p is uninitialised on the first call: do not read it)
        pv = p4[t];
        pv.x = zv.x + beta * pv.x; pv.y = zv.y + beta * pv.y; pv.z = zv.z + beta * pv.z; pv.w = zv.w + beta * pv.w;
      }
      p4[t] = pv;
    }
  } else {
    for (size_t t = tid; t < n; t += nth) p[t] = first ? z[t] : z[t] + beta * p[t];
  }
}

__global__ void __launch_bounds__(256) k_dot(const float *__restrict__ a, const float *__restrict__ b, size_t n,
                                             double *dst, const NfSolveState *st) {
  if (st && st->done) return;
  double part = 0.0;
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  for (size_t t = tid; t < n; t += nth) part += (double)a[t] * (double)b[t];
  nf_block_atomic_add(part, dst);
}

// ------------------------------------------------------------------------------------------------------------
// solve set-up: r = mask(src), sum over active cells; then mean removal (singular, R12) and bb = ||r||^2
// ------------------------------------------------------------------------------------------------------------
// (src may alias r)
__global__ void __launch_bounds__(256) k_mask_sum(const float *src, float *r,
                                                  const float *__restrict__ ax, const float *__restrict__ ay,
                                                  const float *__restrict__ az, int nx, int ny, int nz, int pax,
                                                  double *sum) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  double part = 0.0;
  if (i < nx && j < ny && k < nz) {
    const NfW6 w = nf_load_w6(ax, ay, az, i, j, k, nx, ny, pax);
    const size_t id = ((size_t)k * ny + j) * nx + i;
    const float d = ((w.xl + w.xh) + (w.yl + w.yh)) + (w.zl + w.zh);
    const float v = d > 0.0f ? src[id] : 0.0f;
    r[id] = v;
    part = v;
  }
  nf_block_atomic_add(part, sum);
}

// r -= mean on active cells (if singular); accumulates ||r||^2 into *sq (may be null)
__global__ void __launch_bounds__(256) k_sub_mean(float *__restrict__ r, const float *__restrict__ ax,
                                                  const float *__restrict__ ay, const float *__restrict__ az, int nx,
                                                  int ny, int nz, int pax, const double *sum, double inv_nact,
                                                  int singular, double *sq) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  double part = 0.0;
  if (i < nx && j < ny && k < nz) {
    const size_t id = ((size_t)k * ny + j) * nx + i;
    float v = r[id];
    if (singular) {
      const NfW6 w = nf_load_w6(ax, ay, az, i, j, k, nx, ny, pax);
      const float d = ((w.xl + w.xh) + (w.yl + w.yh)) + (w.zl + w.zh);
      if (d > 0.0f) {
        v = (float)((double)v - (*sum) * inv_nact);
        r[id] = v;
      }
    }
    part = (double)v * v;
  }
  if (sq) nf_block_atomic_add(part, sq);
}

__global__ void k_init_state(NfSolveState *st, double tol, int maxit) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  st->pq[0] = st->pq[1] = 0.0;
  st->rr[0] = st->rr[1] = 0.0;
  st->rz[0] = st->rz[1] = 0.0;
  st->bb = 0.0;
  st->sum = 0.0;
  st->tol2 = tol * tol;
  st->relres = 0.0;
  st->iter = 0;
  st->maxit = maxit;
  st->done = 0;
  st->converged = 0;
}
// after bb is known: a zero (or NaN) right-hand side is "converged at iteration 0" with x = 0 (R11)
__global__ void k_start_state(NfSolveState *st) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  st->sum = 0.0;
  if (!(st->bb > 0.0)) {
    st->done = 1;
    st->converged = (st->bb == 0.0) ? 1 : 0;
  }
}

// ------------------------------------------------------------------------------------------------------------
// a-5  V-cycle pieces
// ------------------------------------------------------------------------------------------------------------
// Red-black Gauss-Seidel half sweep on the cells with (i+j+k) % 2 == color.  One thread per x-pair of cells.
// ZERO: the initial guess is zero (neighbours are not read).  DOT: also accumulate r.z over BOTH cells of the pair
// (used on the last half sweep of the V-cycle on level 0, where z is final).
template <bool ZERO, bool DOT>
__global__ void __launch_bounds__(256) k_rbgs(float *__restrict__ z, const float *__restrict__ r,
                                              const float *__restrict__ ax, const float *__restrict__ ay,
                                              const float *__restrict__ az, float c, int nx, int ny, int nz, int pax,
                                              int color, NfSolveState *st, int slot) {
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
      const float d = ((w.xl + w.xh) + (w.yl + w.yh)) + (w.zl + w.zh);
      float zn = 0.0f;
      const float rv = r[id];
      if (d > 0.0f) {
        float s = rv;
        if (!ZERO) s += c * nf_nb_sum(z, w, i, j, k, nx, ny, nz);
        zn = s / (c * d);
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
                                                           int cnz, const NfSolveState *st) {
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
        const int i = 2 * I + di, j = 2 * J + dj, k = 2 * K + dk;
        const NfW6 w = nf_load_w6(ax, ay, az, i, j, k, nx, ny, pax);
        const size_t id = ((size_t)k * ny + j) * nx + i;
        const float d = ((w.xl + w.xh) + (w.yl + w.yh)) + (w.zl + w.zh);
        acc += r[id] - c * (d * z[id] - nf_nb_sum(z, w, i, j, k, nx, ny, nz));
      }
  rc[((size_t)K * cny + J) * cnx + I] = 0.125f * acc;
}

// z_f += z_c[parent]   (piecewise-constant prolongation)
__global__ void __launch_bounds__(256) k_prolong_add(float *__restrict__ z, const float *__restrict__ zc, int nx,
                                                     int ny, int nz, int cnx, int cny, const NfSolveState *st) {
  if (st && st->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= nx || j >= ny || k >= nz) return;
  z[((size_t)k * ny + j) * nx + i] += __ldg(zc + ((size_t)(k >> 1) * cny + (j >> 1)) * cnx + (i >> 1));
}

// Coarsest level in ONE CTA, all data in shared memory: `sweeps` red->black sweeps from a zero guess followed by
// `sweeps` black->red sweeps (a symmetric positive semi-definite approximate inverse).
// smem layout: z[n], r[n], idiag[n], wgt[6][n]
__global__ void __launch_bounds__(256) k_bottom(float *__restrict__ zg, const float *__restrict__ rg,
                                                const float *__restrict__ ax, const float *__restrict__ ay,
                                                const float *__restrict__ az, float c, int nx, int ny, int nz, int pax,
                                                int sweeps, const NfSolveState *st) {
  if (st && st->done) return;
  extern __shared__ float sm[];
  const int n = nx * ny * nz;
  float *z = sm, *r = sm + n, *idg = sm + 2 * n, *wg = sm + 3 * n;
  const int sy = nx, sz = nx * ny;
  for (int id = threadIdx.x; id < n; id += blockDim.x) {
    const int i = id % nx, j = (id / nx) % ny, k = id / sz;
    const NfW6 w = nf_load_w6(ax, ay, az, i, j, k, nx, ny, pax);
    const float d = ((w.xl + w.xh) + (w.yl + w.yh)) + (w.zl + w.zh);
    idg[id] = d > 0.0f ? 1.0f / (c * d) : 0.0f;
    wg[0 * n + id] = i > 0 ? c * w.xl : 0.0f;
    wg[1 * n + id] = i + 1 < nx ? c * w.xh : 0.0f;
    wg[2 * n + id] = j > 0 ? c * w.yl : 0.0f;
    wg[3 * n + id] = j + 1 < ny ? c * w.yh : 0.0f;
    wg[4 * n + id] = k > 0 ? c * w.zl : 0.0f;
    wg[5 * n + id] = k + 1 < nz ? c * w.zh : 0.0f;
    r[id] = rg[id];
    z[id] = 0.0f;
  }
  __syncthreads();
  for (int s = 0; s < 4 * sweeps; ++s) {
    // half sweeps: forward part = red, black, red, black ...; backward part = black, red, ...
    const int half = s & 1;
    const int color = (s < 2 * sweeps) ? half : 1 - half;
    for (int id = threadIdx.x; id < n; id += blockDim.x) {
      const int i = id % nx, j = (id / nx) % ny, k = id / sz;
      if (((i + j + k) & 1) != color) continue;
      float a = r[id];
      a += wg[0 * n + id] * z[i > 0 ? id - 1 : id];
      a += wg[1 * n + id] * z[i + 1 < nx ? id + 1 : id];
      a += wg[2 * n + id] * z[j > 0 ? id - sy : id];
      a += wg[3 * n + id] * z[j + 1 < ny ? id + sy : id];
      a += wg[4 * n + id] * z[k > 0 ? id - sz : id];
      a += wg[5 * n + id] * z[k + 1 < nz ? id + sz : id];
      z[id] = a * idg[id];
    }
    __syncthreads();
  }
  for (int id = threadIdx.x; id < n; id += blockDim.x) zg[id] = z[id];
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
static inline int vec_ok(const void *a, const void *b, const void *c, const void *d, size_t n) {
  const uintptr_t m = (uintptr_t)a | (uintptr_t)b | (uintptr_t)c | (uintptr_t)d;
  return ((m & 15) == 0 && (n & 3) == 0) ? 1 : 0;
}

int nf_solver_init(nf_grid *g) {
  NF_CUDA(g, cudaFuncSetAttribute(k_bottom, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  9 * NF_BOTTOM_MAX_CELLS * (int)sizeof(float)));
  return NF_OK;
}

int nf_apply_A_impl(nf_grid *g, const float *p, float *q) {
  NfLevel &L = g->lv[0];
  NfDims d = nf_dims(L.nx, L.ny, L.nz);
  NF_LAUNCH(g, NFK_APPLY, k_apply_A<false><<<d.grid, d.block, 0, g->stream>>>(p, L.ax, L.ay, L.az, q, L.c, L.nx, L.ny, L.nz, L.pax, nullptr, 0));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

static void smooth_half(nf_grid *g, NfLevel &L, int color, bool zero, bool dot, NfSolveState *st, int slot) {
  NfDims d = nf_dims((L.nx + 1) / 2, L.ny, L.nz);
  const bool lvl0 = (&L == &g->lv[0]);
  if (zero)
    NF_LAUNCH(g, (lvl0 ? NFK_RBGS0 : NFK_RBGS_C), k_rbgs<true, false><<<d.grid, d.block, 0, g->stream>>>(L.z, L.r, L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax,
                                                           color, st, slot));
  else if (dot)
    NF_LAUNCH(g, (lvl0 ? NFK_RBGS0 : NFK_RBGS_C), k_rbgs<false, true><<<d.grid, d.block, 0, g->stream>>>(L.z, L.r, L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax,
                                                           color, st, slot));
  else
    NF_LAUNCH(g, (lvl0 ? NFK_RBGS0 : NFK_RBGS_C), k_rbgs<false, false><<<d.grid, d.block, 0, g->stream>>>(L.z, L.r, L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax,
                                                            color, st, slot));
}

static int bottom_sweeps(const NfLevel &L) {
  int m = L.nx > L.ny ? L.nx : L.ny;
  m = m > L.nz ? m : L.nz;
  return 4 * m;
}

// z = M^{-1} r on level 0 (lv[0].r -> lv[0].z).  st may be null (no early exit, no dot).
int nf_vcycle_impl(nf_grid *g, bool with_dot, int slot) {
  NfSolveState *st = with_dot ? g->st : nullptr;
  const int nl = g->nlev;
  for (int l = 0; l + 1 < nl; ++l) {
    NfLevel &L = g->lv[l], &C = g->lv[l + 1];
    for (int s = 0; s < g->nu_pre; ++s) {
      smooth_half(g, L, 0, s == 0, false, st, slot);
      smooth_half(g, L, 1, false, false, st, slot);
    }
    NfDims d = nf_dims(C.nx, C.ny, C.nz);
    NF_LAUNCH(g, (l == 0 ? NFK_RESTRICT0 : NFK_RESTRICT_C), k_residual_restrict<<<d.grid, d.block, 0, g->stream>>>(L.z, L.r, L.ax, L.ay, L.az, L.c, L.nx, L.ny, L.nz, L.pax,
                                                           C.r, C.nx, C.ny, C.nz, st));
  }
  {
    NfLevel &B = g->lv[nl - 1];
    if (B.ncell <= NF_BOTTOM_MAX_CELLS) {
      const size_t smem = (size_t)9 * B.ncell * sizeof(float);
      NF_LAUNCH(g, NFK_BOTTOM, k_bottom<<<1, 256, smem, g->stream>>>(B.z, B.r, B.ax, B.ay, B.az, B.c, B.nx, B.ny, B.nz, B.pax, bottom_sweeps(B),
                                            st));
    } else {  // coarsest level too large for one CTA (odd sizes): a few symmetric sweeps in global memory
      const int nb = 4;
      for (int s = 0; s < nb; ++s) {
        smooth_half(g, B, 0, s == 0, false, st, slot);
        smooth_half(g, B, 1, false, false, st, slot);
      }
      for (int s = 0; s < nb; ++s) {
        smooth_half(g, B, 1, false, false, st, slot);
        smooth_half(g, B, 0, false, false, st, slot);
      }
    }
    if (nl == 1 && with_dot) {
      NF_LAUNCH(g, NFK_MISC, k_dot<<<NF_VEC_BLOCKS, 256, 0, g->stream>>>(B.r, B.z, (size_t)B.ncell, &g->st->rz[slot], st));
    }
  }
  for (int l = nl - 2; l >= 0; --l) {
    NfLevel &L = g->lv[l], &C = g->lv[l + 1];
    NfDims d = nf_dims(L.nx, L.ny, L.nz);
    NF_LAUNCH(g, (l == 0 ? NFK_PROLONG0 : NFK_PROLONG_C), k_prolong_add<<<d.grid, d.block, 0, g->stream>>>(L.z, C.z, L.nx, L.ny, L.nz, C.nx, C.ny, st));
    for (int s = 0; s < g->nu_post; ++s) {
      smooth_half(g, L, 1, false, false, st, slot);
      smooth_half(g, L, 0, false, with_dot && l == 0 && s == g->nu_post - 1, st, slot);
    }
  }
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

// lv[0].r holds the raw right-hand side (src == nullptr) or is filled from src.  Masks inactive cells, removes
// the mean over active cells if the system is singular (R12) and computes bb.
int nf_solve_prepare_from(nf_grid *g, const float *src, float tol, int maxit) {
  NfLevel &L = g->lv[0];
  NfDims d = nf_dims(L.nx, L.ny, L.nz);
  NF_LAUNCH(g, NFK_SETUP, k_init_state<<<1, 32, 0, g->stream>>>(g->st, (double)tol, maxit));
  NF_LAUNCH(g, NFK_SETUP, k_mask_sum<<<d.grid, d.block, 0, g->stream>>>(src ? src : L.r, L.r, L.ax, L.ay, L.az, L.nx, L.ny, L.nz, L.pax,
                                                &g->st->sum));
  const double inv = g->nact > 0 ? 1.0 / (double)g->nact : 0.0;
  NF_LAUNCH(g, NFK_SETUP, k_sub_mean<<<d.grid, d.block, 0, g->stream>>>(L.r, L.ax, L.ay, L.az, L.nx, L.ny, L.nz, L.pax, &g->st->sum, inv,
                                                g->singular, &g->st->bb));
  NF_LAUNCH(g, NFK_SETUP, k_start_state<<<1, 32, 0, g->stream>>>(g->st));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}
int nf_solve_prepare(nf_grid *g, float tol, int maxit) { return nf_solve_prepare_from(g, nullptr, tol, maxit); }

static int wait_seq(nf_grid *g, int idx, int expect) {
  NfHostStatus *h = &g->hst[idx & (NF_RING - 1)];
  auto t0 = std::chrono::steady_clock::now();
  unsigned spins = 0;
  while (h->seq != expect) {
    if ((++spins & 0x3ff) == 0) {
      cudaError_t e = cudaStreamQuery(g->stream);
      if (e != cudaSuccess && e != cudaErrorNotReady) {
        g->err = std::string("solver stream failed: ") + cudaGetErrorString(e);
        return NF_ERR_CUDA;
      }
      if (e == cudaSuccess && h->seq != expect) {
        g->err = "solver status never arrived (stream idle)";
        return NF_ERR_CUDA;
      }
      if (std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count() > 120.0) {
        g->err = "solver watchdog: no progress for 120 s";
        return NF_ERR_CUDA;
      }
      std::this_thread::yield();
    }
  }
  return NF_OK;
}

// MGPCG on A x = lv[0].r (prepared).  x is overwritten.
int nf_solve_run(nf_grid *g, float *x, float tol, int maxit) {
  (void)tol;
  NfLevel &L = g->lv[0];
  const size_t n = (size_t)L.ncell;
  NfDims dc = nf_dims(L.nx, L.ny, L.nz);
  const int v4 = vec_ok(x, L.r, g->p, g->q, n) && vec_ok(L.z, L.z, L.z, L.z, n);
  for (int s = 0; s < NF_RING; ++s) g->hst[s].seq = 0;
  NF_CUDA(g, cudaMemsetAsync(x, 0, n * sizeof(float), g->stream));
  int rc = nf_vcycle_impl(g, true, 0);
  if (rc != NF_OK) return rc;
  NF_LAUNCH(g, NFK_PUPDATE, k_cg_pupdate<<<NF_VEC_BLOCKS, 256, 0, g->stream>>>(g->p, L.z, n, v4, g->st, 0, 1));
  int it = 0, last_seen = -1, done = 0, converged = 0;
  float relres = 0.0f;
  if (maxit < 1) maxit = 1;
  for (it = 0; it < maxit && !done; ++it) {
    const int slot = it & 1;
    NF_LAUNCH(g, NFK_APPLY, k_apply_A<true><<<dc.grid, dc.block, 0, g->stream>>>(g->p, L.ax, L.ay, L.az, g->q, L.c, L.nx, L.ny, L.nz, L.pax,
                                                         g->st, slot));
    NF_LAUNCH(g, NFK_UPDATE, k_cg_update<<<NF_VEC_BLOCKS, 256, 0, g->stream>>>(x, L.r, g->p, g->q, n, v4, g->st, slot));
    NF_LAUNCH(g, NFK_CHECK, k_cg_check<<<1, 32, 0, g->stream>>>(g->st, slot, &g->hst_dev[it & (NF_RING - 1)], it + 1));
    if (it + 1 < maxit) {
      rc = nf_vcycle_impl(g, true, 1 - slot);
      if (rc != NF_OK) return rc;
      NF_LAUNCH(g, NFK_PUPDATE, k_cg_pupdate<<<NF_VEC_BLOCKS, 256, 0, g->stream>>>(g->p, L.z, n, v4, g->st, slot, 0));
    }
    NF_CUDA(g, cudaGetLastError());
    const int look = it - NF_LOOKAHEAD;
    if (look >= 0) {
      rc = wait_seq(g, look, look + 1);
      if (rc != NF_OK) return rc;
      NfHostStatus *h = &g->hst[look & (NF_RING - 1)];
      last_seen = look;
      if (h->done) done = 1;
      // the ring slot can be reused NF_RING iterations later; clear it now that it has been consumed
      h->seq = 0;
    }
  }
  // drain: every enqueued check kernel must have reported before the ring is reused
  const int enq = it;  // checks enqueued: 0 .. enq-1
  for (int s = last_seen + 1; s < enq; ++s) {
    rc = wait_seq(g, s, s + 1);
    if (rc != NF_OK) return rc;
  }
  {
    NfHostStatus *h = &g->hst[(enq - 1) & (NF_RING - 1)];
    converged = h->converged;
    relres = h->relres;
    g->last_iters = h->iter;
  }
  // gauge: zero mean over active cells on a singular system (R12)
  if (g->singular) {
    NF_LAUNCH(g, NFK_SETUP, k_mask_sum<<<dc.grid, dc.block, 0, g->stream>>>(x, x, L.ax, L.ay, L.az, L.nx, L.ny, L.nz, L.pax, &g->st->sum));
    const double inv = g->nact > 0 ? 1.0 / (double)g->nact : 0.0;
    NF_LAUNCH(g, NFK_SETUP, k_sub_mean<<<dc.grid, dc.block, 0, g->stream>>>(x, L.ax, L.ay, L.az, L.nx, L.ny, L.nz, L.pax, &g->st->sum, inv, 1,
                                                    nullptr));
  }
  NF_CUDA(g, cudaGetLastError());
  // iteration count: read back from the device state lazily in nf_last_solve_info; keep the host view here
  g->last_relres = relres;
  return converged ? NF_OK : NF_NOT_CONVERGED;
}
