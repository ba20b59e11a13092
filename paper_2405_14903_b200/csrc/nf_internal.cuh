// nf_internal.cuh -- internal declarations of the CUDA path (sm_100a).  Not part of the C ABI (include/nf.h).
// Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "nf.h"

#define NF_MAX_LEVELS 12
#define NF_RING 64          // mapped host status ring (power of two)
#define NF_ALPHA_EPS 1e-4f  // R4: alpha < 1e-4 -> 0

// One multigrid level ("hierarchical grid data structure").  Level 0 is the simulation grid.
// Face weights are stored per level in MAC face layout, except that x-face rows are padded to a multiple of
// 4 floats (pax) so that every row of every array starts 16-byte aligned:
//   ax[(k*ny + j)*pax + i], i in [0, nx]   weight of the x-face between cells i-1 and i
//   ay[(k*(ny+1) + j)*nx + i], j in [0, ny]
//   az[(k*ny + j)*nx + i], k in [0, nz]
//
// Cell code (one byte per cell): bits 0..5 = face -x,+x,-y,+y,-z,+z has alpha == 1 exactly,
// bit 6 (NF_CODE_MIXED) = some face of the cell is fractional (0 < alpha < 1), in which case the six fp32 weights
// are read instead.  code == 0  <=>  the cell is inactive (sum of its six weights is 0).
#define NF_CODE_MIXED 64u
// bit 7 (NF_CODE_DEEP): the cell has six fully open faces and so has each of its six neighbours that lies inside the
// grid -- the pre-smoother's fast path needs no neighbour code (every diagonal involved is 6c).
#define NF_CODE_DEEP 128u
struct NfLevel {
  int nx, ny, nz, pax;
  long long ncell;
  float c;  // c_l = (dt_over_rho/dx) / 4^l  (rediscretised operator on spacing 2^l dx)
  float *ax, *ay, *az;
  uint8_t *code;
  float *idg;    // 1 / (c_l * sum of the six weights), 0 on inactive cells (written with the codes)
  float *z, *r;  // level 0: CG vectors z and r; level > 0: coarse correction and restricted residual
  float *pk;     // levels 2 .. tail-1 (k_vcoarse's per-cell phases): idg[n], c*alpha_f[6][n] (0 towards outside), unused[n]
  int fz;         // z-coarsening factor towards the next level: 2, or 1 in 2-D mode (nz == 1: x and y coarsen only)
  int vec_idx32;  // 1: every array of the level has < 2^32 slots (32-bit offsets in the stencil kernels)
  int vec;       // 1: nx % 4 == 0 and a coarser level exists -> the float4 / code kernels run on this level
};

// Kernel-side view of a level (passed by value).  ic = 1/c.
struct NfLvK {
  const float *ax, *ay, *az;
  const uint8_t *code;
  const float *idg;
  float c, ic;
  int nx, ny, nz, pax;
  int fz;  // z coarsening factor towards the next level: 2, or 1 in 2-D mode (nz == 1)
  float om;  // over-relaxation factor of the level's sweeps in the 4-cell bodies (1 outside the cooperative kernel)
};
static inline NfLvK nf_lvk(const NfLevel &L) {
  NfLvK K;
  K.ax = L.ax; K.ay = L.ay; K.az = L.az; K.code = L.code; K.idg = L.idg;
  K.c = L.c; K.ic = 1.0f / L.c; K.nx = L.nx; K.ny = L.ny; K.nz = L.nz; K.pax = L.pax;
  K.fz = L.fz;
  K.om = 1.0f;
  return K;
}

// Device-resident PCG scalars.  Slots [2] alternate with the iteration parity so that no kernel has to
// reset a value another kernel of the same iteration still reads.  The control words every CTA reads on entry
// (done) live in their own 128-byte line, and each accumulator pair in its own line, so that the fp64 atomics of
// the CTAs that finish do not queue in front of the flag reads of the CTAs that start.
struct alignas(128) NfSolveState {
  int iter, maxit, done, converged;
  unsigned ticket;  // CTAs of k_cg_update that have finished (the last one runs the convergence check)
  int last_slot;    // parity slot of the last executed iteration of the current phase (-1: none)
  double bb;    // ||b||^2 after masking / mean removal
  double tol2;  // (tolerance of the current phase)^2
  double relres;  // sqrt(rr/bb) at the last executed iteration
  // Singular system with ONE fluid component (gauge mode 1): the residual is kept compatible -- zero mean over the
  // active cells -- in every iteration (k_update_down1), not only at the start: fp32 cannot remove a mean of 5e-9 |b|
  // from b itself (it is below the rounding of the entries), the mean stays while the residual falls by 1e-6, and
  // the V-cycle amplifies the constant mode: PCG then stalled near 1e-6 and DIVERGED.
  // in-flight residual replacement (nf_solver.cu: run_pcg_phase): 0 not tried, 1 accepted (the iteration read the true
  // residual, later x updates go to the correction array), -1 rejected (the true residual differed from the recursive
  // one by more than 10 % of its norm: PCG goes on undisturbed to the phase-1 tolerance and the solve restarts on the
  // true residual as in round 1)
  int switched;
  double dev2, rrt, srt;  // ||r_true - r||^2, ||r_true||^2, sum r_true of the attempt
  double inv_nact;  // 1 / #active cells when that projection is on, else 0
  double sb;        // sum of the prepared right-hand side b0 as stored (what the true residual's mean is)
  alignas(128) double pq[2];
  alignas(128) double rr[2];
  alignas(128) double rz[2];
  alignas(128) double sr[2];  // sum of the residual written in iteration parity s (or sr[1]: at the start of a phase)
  alignas(128) double sum;   // scratch: sum over active cells
};

struct NfHostStatus {  // written by the device into mapped pinned memory
  volatile int seq;    // iteration number + 1 once written (0 = not yet)
  volatile int iter;   // iterations actually executed so far
  volatile int done;
  volatile int converged;
  volatile float relres;
  volatile int switched;  // NfSolveState::switched
};

// One environment of a batched PCG iteration (nf_solver.cu: nf_solve_batch_run): the level-0
// operator, its CG vectors and scalars, and the first coarse level's r / z.  p[s], r[s]: the buffer that iteration
// parity s WRITES (the search direction and the residual ping-pong between two buffers each).
#define NF_BATCH_MAX 16
struct NfEnvK {
  NfLvK L;
  float *z, *q, *x;
  float *p[2], *r[2];
  float *rc, *zc;
  NfSolveState *st;
  NfHostStatus *hs;
};
struct NfBatchK {
  int n;    // environments in this launch (<= NF_BATCH_MAX)
  int nzc;  // z-chunks (CTAs along blockIdx.z) per environment
  int cnx, cny, cnz;  // extents of the first coarse level
  int gen;  // k_down2_b: general residual (the pre-smoother ran more than one sweep)
  NfEnvK e[NF_BATCH_MAX];
};

// limits of the parametric geometry (nf_geom.cu): K key sections, N curves per section, N*M polygon edges
#define NF_GEOM_MAXK 64
#define NF_GEOM_MAXN 64
#define NF_GEOM_MAXNM 2048
#define NF_GEOM_MAXP (2 + NF_GEOM_MAXK * (2 + 2 * NF_GEOM_MAXN))

// Kernel classes for the per-class device timing of nf_profile_* (bench.py's roofline leg).
enum {
  NFK_APPLY = 0, NFK_UPDATE, NFK_CHECK, NFK_PUPDATE, NFK_DOWN1_0, NFK_DOWN2_0, NFK_UP1_0, NFK_UP2_0, NFK_VEC_C,
  NFK_RBGS0, NFK_RBGS_C, NFK_RESTRICT0, NFK_RESTRICT_C, NFK_PROLONG0, NFK_PROLONG_C, NFK_BOTTOM, NFK_SETUP, NFK_RHS,
  NFK_GRADSUB, NFK_ADJ_RHS, NFK_ADJ_FINISH, NFK_WEIGHTS, NFK_COARSEN, NFK_CLASSIFY, NFK_STORE_US, NFK_ADVECT,
  NFK_ADVECT_ADJ, NFK_WEIGHTS_ADJ, NFK_GEOM, NFK_MISC, NFK_SWEEP_0, NFK_COUNT
};

struct nf_grid {
  int nx, ny, nz;
  float dx, dt_over_rho;
  int bc_type[6];
  float bc_val[6];
  cudaStream_t stream;
  int nlev;
  int coarse_ctas;  // > 0: CTAs of the cooperative coarse kernel k_vcoarse (nf_mg.cu); 0 = per-level launches
  int tail;  // first level of the shared-memory tail of the V-cycle (levels tail .. nlev-1 run in one CTA); nlev if none
  NfLevel lv[NF_MAX_LEVELS];
  bool weights_set, have_sdf, have_us;
  int singular;  // 1: ONE component and it is singular -- the global mean is removed (R12); see gauge_mode
  int singular_info;  // no open face on any Dirichlet domain boundary (what nf_grid_info reports)
  // fluid components (nf_components.cu): labels, per-component cell counts / "has a Dirichlet face" flags / sums
  int *comp, *cc_cnt, *cc_regular, *cc_meta, *h_cc_meta;
  double *cc_sums;
  int ncomp, nsing;  // components of the current weights; those without an open Dirichlet face
  int gauge_mode;    // 0: no singular component; 1: a single, singular component (global path); 2: per component
  long long nact;
  int nu_pre, nu_post;  // red-black sweeps before / after the coarse correction on the FINEST level
  int nu_l1, nu_deep;   // ... on level 1 / on every level below that (pre = post; nf_set_coarse_sweeps)
  float omega_deep;     // over-relaxation factor of the sweeps on every level below the finest (nf_set_coarse_relaxation)
  bool warm;     // flag 8 of nf_set_solver_options: caller-provided solution arrays hold the initial guess
  bool refresh;  // true-residual refresh between two PCG phases (default on; flag 4 of nf_set_solver_options: off)
  bool force_generic;  // test hook: run the generic (fp32-weight, one colour per launch) kernels everywhere
  // solid velocity (MAC layout, closed walls at rest) and the last SDF
  float *us, *vs, *ws, *sdf;
  // CG vectors on level 0 (r and z live in lv[0])
  float *r_alt;  // the residual ping-pongs between lv[0].r and this buffer (k_update_down1); both owned by the handle
  float *ecorr;  // correction vector of the second PCG phase / after an in-flight replacement
  float *rtrue;  // the true residual of an in-flight replacement attempt (read by ONE k_update_down1 if accepted)
  float *b0;  // the prepared right-hand side (kept for the true-residual refresh, nf_solver.cu)
  float *p, *p2, *q, *xtmp;  // p / p2: the search direction ping-pongs between two buffers (k_papply4)
  float *tailpack;  // 8 floats per cell of the tail levels (nf_mg.cu)
  float *plo;      // caller's array for the low-order part of the next solutions (nf_set_pressure_lo), or NULL
  bool lo_valid;   // the last solve wrote it
  bool meta_pending;     // the counts of the last hierarchy build have not been read yet (nf_meta_sync)
  cudaEvent_t ev_meta, ev_coarse;
  void *h_coarse;        // pinned staging of d_coarse
  void *d_coarse;        // device copy of the coarse kernel's level table (batched launches, nf_mg.cu)
  unsigned *cbar;        // per-environment barrier counter of k_vcoarse_b
  unsigned cbar_count;   // its value after everything enqueued so far
  float *tailinv;   // inverse of the coarsest level's operator (n <= 128 cells: n^2 floats; k_coarse_inverse)
  // scratch face arrays (advection copy / adjoint staging)
  float *fu, *fv, *fw;
  NfSolveState *st;      // device
  NfHostStatus *hst;     // mapped pinned host ring
  NfHostStatus *hst_dev; // device alias of hst
  // parametric geometry (nf_geom.cu): device copies of params / pdot (2 x NF_GEOM_MAXP floats), the parameter gradient
  float *geom_par;
  double *geom_grad;
  double *d_counts;      // device: [0] active cells, [1] open faces on Dirichlet domain faces
  double *h_counts;      // pinned host copy
  cudaEvent_t ev0, ev1;
  int last_iters;
  float last_relres;
  bool last_timed;
  long long launches;
  std::string err;
  // per-class kernel timing (off by default)
  bool prof_on;
  std::vector<cudaEvent_t> prof_pool;  // event pairs: [2*r], [2*r+1]
  std::vector<int> prof_cls;           // class of record r
  double prof_ms[NFK_COUNT];
  long long prof_n[NFK_COUNT];
  // host staging for the *_host entry points
  float *hs_u, *hs_v, *hs_w, *hs_p, *hs_a, *hs_b, *hs_c, *hs_d;
  // copy streams of the *_host entry points (H2D and D2H run on their own streams, ordered by events)
  cudaStream_t s_h2d, s_d2h;
  cudaEvent_t ev_in, ev_comp, ev_out_proj, ev_out_adj;
  bool host_async;  // nf_set_host_async: *_host calls return before their D2H copies finish (nf_host_sync waits)
};

void nf_prof_begin(nf_grid *g, int cls);
void nf_prof_end(nf_grid *g);
// Every kernel launch of the library goes through this macro: it counts the launch and, when profiling is on,
// brackets it with CUDA events on the handle's stream.
#define NF_LAUNCH(g, cls, ...)              \
  do {                                      \
    if ((g)->prof_on) nf_prof_begin(g, cls); \
    __VA_ARGS__;                            \
    if ((g)->prof_on) nf_prof_end(g);       \
    (g)->launches += 1;                     \
  } while (0)

#define NF_CUDA(g, call)                                                            \
  do {                                                                              \
    cudaError_t e_ = (call);                                                        \
    if (e_ != cudaSuccess) {                                                        \
      (g)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                \
      return NF_ERR_CUDA;                                                           \
    }                                                                               \
  } while (0)

#define NF_TRY(expr)            \
  do {                          \
    int rc_ = (expr);           \
    if (rc_ < 0) return rc_;    \
  } while (0)

static inline size_t nf_nu(const nf_grid *g) { return (size_t)g->nz * g->ny * (g->nx + 1); }
static inline size_t nf_nv(const nf_grid *g) { return (size_t)g->nz * (g->ny + 1) * g->nx; }
static inline size_t nf_nw(const nf_grid *g) { return (size_t)(g->nz + 1) * g->ny * g->nx; }
static inline size_t nf_nc(const nf_grid *g) { return (size_t)g->nz * g->ny * g->nx; }
static inline size_t nf_nn(const nf_grid *g) { return (size_t)(g->nz + 1) * (g->ny + 1) * (g->nx + 1); }

// Launch geometry for a logical (tx, ty, tz) thread lattice: 256 threads per block, x fastest.
struct NfDims {
  dim3 grid, block;
};
static inline NfDims nf_dims(int tx, int ty, int tz) {
  int bx = 4;
  while (bx < tx && bx < 128) bx <<= 1;
  int by = 1;
  while (by < ty && bx * by < 256) by <<= 1;
  int bz = 1;
  while (bz < tz && bx * by * bz < 256) bz <<= 1;
  NfDims d;
  d.block = dim3(bx, by, bz);
  d.grid = dim3((tx + bx - 1) / bx, (ty + by - 1) / by, (tz + bz - 1) / bz);
  return d;
}

// Launch geometry of the 4-cells-per-thread ("vec") stencil kernels: thread lattice (nx/4, rows_y), CTAs of up to
// 64 x 4 threads, and every CTA marches through `kch` consecutive z-planes (blockIdx.z = chunk): 8x fewer CTAs (and
// reduction atomics) than one plane per CTA, and the z-neighbour rows of one plane are the L1-resident centre rows
// of the next.
#define NF_KCH_MG 8  // planes per CTA: V-cycle kernels (measured in situ at 256^3: 1 -> 4 saves 10-20 % per kernel, 4 -> 8 another 1-4 %)
#define NF_KCH_AP 8  // planes per CTA: A-apply (z-neighbour rows rotate through registers)
static inline NfDims nf_vdims(int tx, int ty, int tz, int kch) {
  int bx = 1;
  while (bx < tx && bx < 64) bx <<= 1;  // whole 256-cell rows per CTA: contiguous DRAM segments beat square tiles
  int by = 1;
  while (by < ty && bx * by < 256) by <<= 1;
  NfDims d;
  d.block = dim3(bx, by, 1);
  d.grid = dim3((tx + bx - 1) / bx, (ty + by - 1) / by, (tz + kch - 1) / kch);
  return d;
}

// Planes per CTA for a level: the full chunk (kmax) only where that still leaves >= 4 CTAs per SM; small grids (the
// paper's 40^3-64^3 tasks) march less and spread over more CTAs instead -- at 48^3 eight planes per CTA meant 18 CTAs
// on 148 SMs.
static inline int nf_kch(int tx, int ty, int tz, int kmax) {
  const NfDims d = nf_vdims(tx, ty, tz, 1);
  const long long ctas = (long long)d.grid.x * d.grid.y * tz;
  const long long k = ctas / (148 * 4);  // (measured 48^3 .. 192^3: 2, 4, 8, 16, 32 CTAs per SM; 4 is best at 128^3)
  return (int)(k < 1 ? 1 : (k > kmax ? kmax : k));
}

// ---- kernels / host launchers implemented across the .cu files -------------------------------------------
// nf_weights.cu
int nf_weights_from_sdf(nf_grid *g, const float *sdf);
int nf_weights_from_user(nf_grid *g, const float *au, const float *av, const float *aw);
int nf_weights_to_user(nf_grid *g, float *au, float *av, float *aw);
int nf_build_hierarchy(nf_grid *g);  // coarse weights + active count + singular flag
int nf_meta_sync(nf_grid *g);        // wait for / read the counts of the last hierarchy build
int nf_store_solid_velocity(nf_grid *g, const float *us, const float *vs, const float *ws);
int nf_weights_adjoint_impl(nf_grid *g, const float *gau, const float *gav, const float *gaw, float *gsdf);
// nf_components.cu
int nf_components_alloc(nf_grid *g);
void nf_components_free(nf_grid *g);
int nf_components_build(nf_grid *g);
int nf_components_center(nf_grid *g, float *x, float *dst2, double *sq);
// nf_solver.cu
int nf_apply_A_impl(nf_grid *g, const float *p, float *q);
// nf_mg.cu
void nf_mg_plan(nf_grid *g);      // choose the shared-memory tail and the vec levels (after the level extents are known)
int nf_mg_init(nf_grid *g);       // kernel attributes
int nf_mg_pack_tail(nf_grid *g);  // packed operator of the tail levels from the current weights
int nf_mg_upload_coarse(nf_grid *g);  // device copy of the coarse kernel's level table (after every hierarchy build)
void nf_mg_free_batch(nf_grid *g);
int nf_vcycle_batch(nf_grid **G, int n, const NfBatchK &B, int slot);
int nf_update_down1_batch(nf_grid **G, int n, const NfBatchK &B, int slot, int seq);
int nf_vcycle_impl(nf_grid *g, bool with_dot, int slot, bool skip_down1 = false);  // z = M^{-1} r on lv[0].r -> lv[0].z
// fused r' = r - a q + pre-smoother of level 0 (r' into g->r_alt, then the two buffers swap); false if not applicable
bool nf_update_down1_ok(const nf_grid *g);
int nf_update_down1(nf_grid *g, int slot, NfHostStatus *hs, int seq, const float *rtrue = nullptr);
// Solve A x = lv[0].r (already masked; mean removed if singular; st->bb set by nf_solve_prepare).
int nf_solver_init(nf_grid *g);                          // kernel attributes (once per process)
int nf_solve_prepare(nf_grid *g, float tol, int maxit);  // from lv[0].r: mask, mean removal, bb
int nf_solve_prepare_from(nf_grid *g, const float *src, float tol, int maxit);
int nf_solve_run(nf_grid *g, float *x, float tol, int maxit, bool warm);  // warm: x holds the initial guess
bool nf_batch_ok(nf_grid **G, int n);  // the n handles can be solved by the batched kernels
int nf_solve_batch_impl(nf_grid **G, int n, const float *const *src, float *const *x, float tol, int maxit, int *status);
// nf_project.cu
int nf_rhs_impl(nf_grid *g, const float *u, const float *v, const float *w);  // -> lv[0].r
int nf_grad_subtract_impl(nf_grid *g, float *u, float *v, float *w, const float *p);
int nf_adjoint_rhs_impl(nf_grid *g, const float *gu, const float *gv, const float *gw);  // -> lv[0].r
int nf_adjoint_finish_impl(nf_grid *g, float *gu, float *gv, float *gw, const float *y, const float *p_saved,
                           const float *uu, const float *uv, const float *uw, float *gau, float *gav, float *gaw,
                           float *gsu, float *gsv, float *gsw);
// nf_advect.cu
int nf_advect_impl(nf_grid *g, float *u, float *v, float *w, float dt);
int nf_viscosity_impl(nf_grid *g, float *u, float *v, float *w, float nu, float dt);
int nf_max_speed_impl(nf_grid *g, const float *u, const float *v, const float *w, float *out_host);
int nf_advect_adjoint_impl(nf_grid *g, const float *u0, const float *v0, const float *w0, float *gu, float *gv,
                           float *gw, float dt);
// nf_geom.cu
int nf_geom_sdf_impl(nf_grid *g, const float *params, int K, int N, int M, int flags, float *sdf_nodes);
int nf_geom_sdf_adjoint_impl(nf_grid *g, const float *params, int K, int N, int M, int flags, const float *gsdf_nodes,
                             double *gparams_host);
int nf_geom_velocity_impl(nf_grid *g, const float *params, const float *pdot, int K, int N, int M, float band,
                          float *us, float *vs, float *ws);
int nf_geom_velocity_adjoint_impl(nf_grid *g, const float *params, int K, int N, int M, float band, const float *gus,
                                  const float *gvs, const float *gws, double *gpdot_host);
int nf_geom_csg_impl(nf_grid *g, int op, const float *a, const float *b, float *out);
int nf_geom_csg_adjoint_impl(nf_grid *g, int op, const float *a, const float *b, const float *gout, float *ga, float *gb);

// Programmatic dependent launch (PDL): the kernels of one PCG iteration are launched with the programmatic stream
// serialisation attribute and start with nf_pdl_enter() -- "my dependents may be scheduled" + "wait until the grids
// I depend on have completed and flushed".  The next kernel's CTAs are then already resident (launch latency, CTA
// scheduling and prologue behind them) when the previous kernel's last wave drains: each of the 7 kernels of an
// iteration otherwise pays a fixed ~15 us of ramp-up and tail on top of its bytes.
#ifdef __CUDACC__
template <typename... KArgs, typename... Args>
static inline cudaError_t nf_launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, cudaStream_t stream, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = 0;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
__device__ __forceinline__ void nf_pdl_enter() {
  asm volatile("griddepcontrol.launch_dependents;");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}
#endif

// ---- device helpers ---------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ double nf_warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}
// Block reduction (warp shuffles, then one warp over the per-warp partials) followed by ONE fp64 atomicAdd
// per block.  Every thread of the block must call it.  blockDim total <= 1024.
__device__ __forceinline__ void nf_block_atomic_add(double v, double *dst) {
  __shared__ double s_part[32];
  const int tid = (threadIdx.z * blockDim.y + threadIdx.y) * blockDim.x + threadIdx.x;
  const int nthr = blockDim.x * blockDim.y * blockDim.z;
  const int lane = tid & 31, wid = tid >> 5;
  v = nf_warp_sum(v);
  if (lane == 0) s_part[wid] = v;
  __syncthreads();
  if (wid == 0) {
    const int nw = (nthr + 31) >> 5;
    double t = lane < nw ? s_part[lane] : 0.0;
    t = nf_warp_sum(t);
    if (lane == 0) atomicAdd(dst, t);
  }
  __syncthreads();
}
// Advance the iteration counter, decide convergence (R11), publish the status to the mapped host ring, and clear
// the accumulators of the other parity slot.  One thread, after rr[slot] is complete.
__device__ __forceinline__ void nf_cg_check(NfSolveState *st, int slot, NfHostStatus *hs, int seq) {
  if (!st->done) {
    st->iter += 1;
    st->last_slot = slot;
    const double rr = *(volatile double *)&st->rr[slot];
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
    st->sr[1 - slot] = 0.0;
    st->relres = st->bb > 0.0 ? sqrt(rr / st->bb) : 0.0;
  }
  hs->relres = (float)st->relres;
  hs->iter = st->iter;
  hs->done = st->done;
  hs->converged = st->converged;
  hs->switched = st->switched;
  __threadfence_system();
  hs->seq = seq;
  __threadfence_system();
}

#endif
