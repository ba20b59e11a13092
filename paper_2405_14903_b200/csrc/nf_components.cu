// nf_components.cu -- fluid components of the active cells and the per-component null-space handling (reading R12 in
// the per-component form of SURVEY.md 8c.1 / 8c.3 item 12; the paper is silent on singular systems).
//
// A = c G^T S G (Eq. 4) is block diagonal over the connected components of the active cells (two cells
// are connected when the face between them is open, alpha > 0).  A component that touches no open face of a Dirichlet
// domain boundary has the constant null vector: its right-hand side must have zero mean over the component
// (compatibility) and the pressure is fixed by zero mean over the component (gauge).  nf_set_solid alone therefore has
// to find the components -- a gate that closes a channel, cavities cut off during shape optimisation, the pockets of
// BASELINE.json configs[4] at 64^3.
//
// Labelling: union-find on the grid graph (ECL-CC style: hook the larger root under the smaller with atomicCAS, path
// halving in find), started from x-runs found with one warp ballot, merged along y and z, then flattened.  Grids with a
// single component (every headline workload) stop after the flatten pass: no label is ever read in a solve.
#include <algorithm>

#include "nf_stencil.cuh"

#define NF_COMP_CAP 65536  // components with per-component statistics (more: the rest is treated as regular)

// comp[] while labelling: parent index (self = root), 0xffffffff on inactive cells.
// comp[] afterwards:      -2 - slot on active cells (slot = dense component number), -1 on inactive cells.
__device__ __forceinline__ unsigned nf_cc_find(unsigned *p, unsigned x) {
  for (;;) {
    const unsigned px = *reinterpret_cast<volatile unsigned *>(p + x);
    if (px == x) return x;
    const unsigned ppx = *reinterpret_cast<volatile unsigned *>(p + px);
    if (ppx != px) p[x] = ppx;  // path halving (parents only ever decrease: a benign race)
    x = px;
  }
}
__device__ __forceinline__ void nf_cc_unite(unsigned *p, unsigned a, unsigned b) {
  for (;;) {
    a = nf_cc_find(p, a);
    b = nf_cc_find(p, b);
    if (a == b) return;
    if (a < b) { const unsigned t = a; a = b; b = t; }
    if (atomicCAS(p + a, a, b) == a) return;  // a was still a root: now it hangs under the smaller root b
  }
}

// One thread per cell, consecutive ids in a warp: every cell starts under the first cell of its x-run inside the warp
// (lane 0 under its left neighbour when the run continues from the previous warp).
__global__ void __launch_bounds__(256) k_cc_init(NfLvK L, unsigned *__restrict__ comp, unsigned n) {
  const unsigned id = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned lane = threadIdx.x & 31u;
  bool active = false, link = false;
  if (id < n) {
    const int i = (int)(id % (unsigned)L.nx), j = (int)((id / (unsigned)L.nx) % (unsigned)L.ny),
              k = (int)(id / ((unsigned)L.nx * (unsigned)L.ny));
    const unsigned code = L.code[id];
    active = code != 0;
    if (active && i > 0) link = nf_code_w6(L, code, i, j, k).xl > 0.0f;
  }
  const unsigned links = __ballot_sync(0xffffffffu, link);
  if (id >= n) return;
  unsigned parent = 0xffffffffu;
  if (active) {
    const unsigned breaks = ~links & (0xffffffffu >> (31u - lane));  // lanes <= mine whose run starts there
    if (breaks) {
      parent = id - (lane - (31u - (unsigned)__clz(breaks)));
    } else {  // the run reaches back beyond lane 0
      parent = lane == 0 ? id - 1 : id - lane;
    }
  }
  comp[id] = parent;
}

// "is the low x- / y- / z-face of this cell open": one bit of a pure cell's code, the fp32 weight of a mixed cell
__device__ __forceinline__ bool nf_cc_open_lo(const NfLvK &L, unsigned code, int axis, int i, int j, int k) {
  if (!(code & NF_CODE_MIXED)) return (code >> (2 * axis)) & 1u;
  if (axis == 0) return __ldg(L.ax + ((nf_idx)k * L.ny + j) * L.pax + i) > 0.0f;
  if (axis == 1) return __ldg(L.ay + ((nf_idx)k * (L.ny + 1) + j) * L.nx + i) > 0.0f;
  return __ldg(L.az + ((nf_idx)k * L.ny + j) * L.nx + i) > 0.0f;
}
// Unions along y and z.  A cell whose left neighbour is x-linked to it and makes the same union one cell to the left
// (the two cells below / behind being x-linked as well) skips its own: one union per overlap of two x-runs instead of
// one per cell -- in open fluid that is 1/nx of them, and the kernel is a pass over the codes.
__global__ void __launch_bounds__(256) k_cc_merge(NfLvK L, unsigned *comp, unsigned n) {
  const unsigned id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= n) return;
  const unsigned code = L.code[id];
  if (code == 0) return;
  const int nx = L.nx, ny = L.ny;
  const int i = (int)(id % (unsigned)nx), j = (int)((id / (unsigned)nx) % (unsigned)ny),
            k = (int)(id / ((unsigned)nx * (unsigned)ny));
  const bool linked = i > 0 && nf_cc_open_lo(L, code, 0, i, j, k);
  const unsigned cleft = linked ? L.code[id - 1] : 0u;
#pragma unroll
  for (int axis = 1; axis <= 2; ++axis) {
    const unsigned step = axis == 1 ? (unsigned)nx : (unsigned)nx * (unsigned)ny;
    if ((axis == 1 ? j : k) == 0 || !nf_cc_open_lo(L, code, axis, i, j, k)) continue;
    if (linked && nf_cc_open_lo(L, cleft, axis, i - 1, j, k)) {
      const unsigned cb = L.code[id - step];
      if (nf_cc_open_lo(L, cb, 0, i, axis == 1 ? j - 1 : j, axis == 2 ? k - 1 : k)) continue;  // made by the left cell
    }
    nf_cc_unite(comp, id, id - step);
  }
}

// comp[id] = root of id; counts the roots in meta[0].  The walk to the root is READ-ONLY here: with path halving a
// thread passing through cell x could overwrite the root x's own thread has just stored with an intermediate parent it
// read earlier, and the labelling pass below relies on every entry pointing at a root.  (A stale read of comp[x] by
// a passing thread is harmless: old parent and root are both ancestors.)
__global__ void __launch_bounds__(256) k_cc_flatten(unsigned *comp, unsigned n, int *meta) {
  const unsigned id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= n) return;
  if (comp[id] == 0xffffffffu) return;
  unsigned r = id;
  for (;;) {
    const unsigned pr = *reinterpret_cast<volatile unsigned *>(comp + r);
    if (pr == r) break;
    r = pr;
  }
  comp[id] = r;
  if (r == id) atomicAdd(meta, 1);
}

// More than one component: number the roots (slot = order of arrival) ...
__global__ void __launch_bounds__(256) k_cc_number(int *comp, unsigned n, int *meta) {
  if (meta[0] <= 1) return;
  const unsigned id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= n) return;
  if (comp[id] == (int)id) comp[id] = -2 - atomicAdd(meta + 1, 1);
}
// ... hand the number to every cell of the component, count the cells and mark the components with an open face on a
// Dirichlet domain boundary
struct NfBc6c {
  int dir[6];
};
__global__ void __launch_bounds__(256) k_cc_label(NfLvK L, int *comp, unsigned n, const int *meta, NfBc6c bc,
                                                  int *__restrict__ cnt, int *__restrict__ regular) {
  if (meta[0] <= 1) return;
  const unsigned id = blockIdx.x * blockDim.x + threadIdx.x;
  int v = -1;
  if (id < n) {
    v = comp[id];
    if (v >= 0) {  // a non-root cell: its root holds the number already (roots are not written in this kernel)
      v = comp[v];
      comp[id] = v;
    }
  }
  // cells per component: one atomic per CTA when the whole CTA lies in one component (the common case)
  __shared__ int s_first, s_cnt;
  if (threadIdx.x == 0) { s_first = -1; s_cnt = 0; }
  __syncthreads();
  if (v < -1) atomicCAS(&s_first, -1, v);
  __syncthreads();
  const int first = s_first;
  const bool uniform = __syncthreads_and(v >= -1 || v == first);
  const int slot = -2 - v;
  if (uniform) {
    if (v < -1) atomicAdd(&s_cnt, 1);
    __syncthreads();
    if (threadIdx.x == 0 && first < -1 && -2 - first < NF_COMP_CAP) atomicAdd(cnt + (-2 - first), s_cnt);
  } else if (v < -1 && slot < NF_COMP_CAP) {
    atomicAdd(cnt + slot, 1);
  }
  if (v < -1 && slot < NF_COMP_CAP) {
    const int i = (int)(id % (unsigned)L.nx), j = (int)((id / (unsigned)L.nx) % (unsigned)L.ny),
              k = (int)(id / ((unsigned)L.nx * (unsigned)L.ny));
    const bool edge = (i == 0 && bc.dir[0]) || (i == L.nx - 1 && bc.dir[1]) || (j == 0 && bc.dir[2]) ||
                      (j == L.ny - 1 && bc.dir[3]) || (k == 0 && bc.dir[4]) || (k == L.nz - 1 && bc.dir[5]);
    if (edge) {
      const NfW6 w = nf_code_w6(L, L.code[id], i, j, k);
      const bool open = (i == 0 && bc.dir[0] && w.xl > 0.0f) || (i == L.nx - 1 && bc.dir[1] && w.xh > 0.0f) ||
                        (j == 0 && bc.dir[2] && w.yl > 0.0f) || (j == L.ny - 1 && bc.dir[3] && w.yh > 0.0f) ||
                        (k == 0 && bc.dir[4] && w.zl > 0.0f) || (k == L.nz - 1 && bc.dir[5] && w.zh > 0.0f);
      if (open) regular[slot] = 1;
    }
  }
}
// meta[2] = number of singular components among the first NF_COMP_CAP
__global__ void __launch_bounds__(256) k_cc_finish(int *meta, const int *__restrict__ regular) {
  if (meta[0] <= 1) return;
  const int K = min(meta[0], NF_COMP_CAP);
  int s = 0;
  for (int c = threadIdx.x; c < K; c += blockDim.x) s += regular[c] ? 0 : 1;
  atomicAdd(meta + 2, s);
}

// ------------------------------------------------------------------------------------------------------------
// per-component compatibility / gauge (only on systems with several components, one of them singular)
// ------------------------------------------------------------------------------------------------------------
// sums[slot] += x over the cells of every singular component
__global__ void __launch_bounds__(256) k_cc_sum(const float *__restrict__ x, const int *__restrict__ comp, unsigned n,
                                                const int *__restrict__ regular, double *__restrict__ sums) {
  const unsigned id = blockIdx.x * blockDim.x + threadIdx.x;
  int slot = -1;
  double v = 0.0;
  if (id < n) {
    const int c = comp[id];
    if (c < -1 && -2 - c < NF_COMP_CAP && !regular[-2 - c]) {
      slot = -2 - c;
      v = (double)x[id];
    }
  }
  __shared__ int s_first;
  if (threadIdx.x == 0) s_first = -1;
  __syncthreads();
  if (slot >= 0) atomicCAS(&s_first, -1, slot);
  __syncthreads();
  const int first = s_first;
  if (__syncthreads_and(slot < 0 || slot == first)) {
    if (first >= 0) nf_block_atomic_add(v, sums + first);  // (uniform over the CTA: every thread takes this branch)
  } else if (slot >= 0) {
    atomicAdd(sums + slot, v);
  }
}
// x -= mean of its component on the cells of singular components (also into dst2); sq += sum of the new x^2
__global__ void __launch_bounds__(256) k_cc_center(float *__restrict__ x, float *__restrict__ dst2,
                                                   const int *__restrict__ comp, unsigned n,
                                                   const int *__restrict__ regular, const int *__restrict__ cnt,
                                                   const double *__restrict__ sums, double *sq) {
  const unsigned id = blockIdx.x * blockDim.x + threadIdx.x;
  double part = 0.0;
  if (id < n) {
    float v = x[id];
    const int c = comp[id];
    if (c < -1 && -2 - c < NF_COMP_CAP && !regular[-2 - c]) {
      const int slot = -2 - c;
      v = (float)((double)v - sums[slot] / (double)max(cnt[slot], 1));
      x[id] = v;
    }
    if (dst2) dst2[id] = v;
    part = (double)v * v;
  }
  if (sq) nf_block_atomic_add(part, sq);
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
int nf_components_alloc(nf_grid *g) {
  g->comp = nullptr; g->cc_cnt = nullptr; g->cc_regular = nullptr; g->cc_sums = nullptr; g->cc_meta = nullptr;
  g->h_cc_meta = nullptr;
  if (g->lv[0].ncell >= 0x7ffffff0LL) return NF_OK;  // labels are 32-bit signed: beyond that the global reading of R12
  if (cudaMalloc((void **)&g->comp, (size_t)g->lv[0].ncell * sizeof(int)) != cudaSuccess ||
      cudaMalloc((void **)&g->cc_cnt, NF_COMP_CAP * sizeof(int)) != cudaSuccess ||
      cudaMalloc((void **)&g->cc_regular, NF_COMP_CAP * sizeof(int)) != cudaSuccess ||
      cudaMalloc((void **)&g->cc_sums, NF_COMP_CAP * sizeof(double)) != cudaSuccess ||
      cudaMalloc((void **)&g->cc_meta, 4 * sizeof(int)) != cudaSuccess ||
      cudaHostAlloc((void **)&g->h_cc_meta, 4 * sizeof(int), cudaHostAllocDefault) != cudaSuccess)
    return NF_ERR_ALLOC;
  return NF_OK;
}
void nf_components_free(nf_grid *g) {
  cudaFree(g->comp); cudaFree(g->cc_cnt); cudaFree(g->cc_regular); cudaFree(g->cc_sums); cudaFree(g->cc_meta);
  if (g->h_cc_meta) cudaFreeHost(g->h_cc_meta);
}

// Label the components of level 0 from its cell codes (enqueued; the counts land in g->h_cc_meta, read by
// nf_build_hierarchy after its synchronisation).
int nf_components_build(nf_grid *g) {
  if (!g->comp) return NF_OK;
  NfLevel &L = g->lv[0];
  const unsigned n = (unsigned)L.ncell, nb = (n + 255u) / 256u;
  unsigned *comp = reinterpret_cast<unsigned *>(g->comp);
  NF_CUDA(g, cudaMemsetAsync(g->cc_meta, 0, 4 * sizeof(int), g->stream));
  NF_CUDA(g, cudaMemsetAsync(g->cc_cnt, 0, NF_COMP_CAP * sizeof(int), g->stream));
  NF_CUDA(g, cudaMemsetAsync(g->cc_regular, 0, NF_COMP_CAP * sizeof(int), g->stream));
  NfBc6c bc;
  for (int f = 0; f < 6; ++f) bc.dir[f] = g->bc_type[f] == NF_BC_DIRICHLET ? 1 : 0;
  NF_LAUNCH(g, NFK_CLASSIFY, k_cc_init<<<nb, 256, 0, g->stream>>>(nf_lvk(L), comp, n));
  NF_LAUNCH(g, NFK_CLASSIFY, k_cc_merge<<<nb, 256, 0, g->stream>>>(nf_lvk(L), comp, n));
  NF_LAUNCH(g, NFK_CLASSIFY, k_cc_flatten<<<nb, 256, 0, g->stream>>>(comp, n, g->cc_meta));
  NF_LAUNCH(g, NFK_CLASSIFY, k_cc_number<<<nb, 256, 0, g->stream>>>(g->comp, n, g->cc_meta));
  NF_LAUNCH(g, NFK_CLASSIFY, k_cc_label<<<nb, 256, 0, g->stream>>>(nf_lvk(L), g->comp, n, g->cc_meta, bc, g->cc_cnt, g->cc_regular));
  NF_LAUNCH(g, NFK_CLASSIFY, k_cc_finish<<<1, 256, 0, g->stream>>>(g->cc_meta, g->cc_regular));
  NF_CUDA(g, cudaMemcpyAsync(g->h_cc_meta, g->cc_meta, 4 * sizeof(int), cudaMemcpyDeviceToHost, g->stream));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

// x -= the mean over its component, on every singular component (compatibility of b / gauge of p, R12); dst2
// (optional) receives a copy; sq (optional, device) accumulates the sum of squares of the result.
int nf_components_center(nf_grid *g, float *x, float *dst2, double *sq) {
  const unsigned n = (unsigned)g->lv[0].ncell, nb = (n + 255u) / 256u;
  NF_CUDA(g, cudaMemsetAsync(g->cc_sums, 0, (size_t)std::min(g->ncomp, NF_COMP_CAP) * sizeof(double), g->stream));
  NF_LAUNCH(g, NFK_SETUP, k_cc_sum<<<nb, 256, 0, g->stream>>>(x, g->comp, n, g->cc_regular, g->cc_sums));
  NF_LAUNCH(g, NFK_SETUP, k_cc_center<<<nb, 256, 0, g->stream>>>(x, dst2, g->comp, n, g->cc_regular, g->cc_cnt, g->cc_sums, sq));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}
