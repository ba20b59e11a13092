// nf_weights.cu -- a-1 face-weight builder, coarse-level weights of the hierarchy
// (PAPER.md:L230), active-cell / singularity classification (R12) and a-10 the weights adjoint.
#include "nf_internal.cuh"

// ------------------------------------------------------------------------------------------------------------
// Marching-squares fluid area fraction of a unit face with corner SDF values P[0..3] in cyclic order.
// phi > 0 is fluid, phi == 0 counts as solid (R1).  If GRAD, d[q] = d alpha / d P[q].
// tri(a; b, d) = 1/2 * a/(a-b) * a/(a-d): the paper's printed one-fluid-corner formula.
// ------------------------------------------------------------------------------------------------------------
template <bool GRAD>
__device__ __forceinline__ float nf_tri(float a, float b, float d, float &da, float &db, float &dd) {
  const float iab = 1.0f / (a - b), iad = 1.0f / (a - d);
  const float fb = a / (a - b), fd = a / (a - d);  // (true divisions: x / (x - 0) must be exactly 1)
  if (GRAD) {
    const float fb_a = -b * iab * iab, fb_b = a * iab * iab;
    const float fd_a = -d * iad * iad, fd_d = a * iad * iad;
    da = 0.5f * (fb_a * fd + fb * fd_a);
    db = 0.5f * fb_b * fd;
    dd = 0.5f * fb * fd_d;
  }
  return 0.5f * fb * fd;
}

template <bool GRAD>
__device__ __forceinline__ float nf_area_fraction(const float P0, const float P1, const float P2, const float P3,
                                                  float *d /*[4] if GRAD*/) {
  const float P[4] = {P0, P1, P2, P3};
  const bool F[4] = {P0 > 0.0f, P1 > 0.0f, P2 > 0.0f, P3 > 0.0f};
  const int s = (int)F[0] + (int)F[1] + (int)F[2] + (int)F[3];
  float out = 0.0f;
  float g[4] = {0.0f, 0.0f, 0.0f, 0.0f};
  if (s == 4) {
    out = 1.0f;
  } else if (s == 1 || s == 3) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int qb = (q + 1) & 3, qd = (q + 3) & 3;
      const bool hit = (s == 1) ? F[q] : !F[q];
      if (hit) {
        float da, db, dd;
        const float t = nf_tri<GRAD>(P[q], P[qb], P[qd], da, db, dd);
        if (s == 1) {
          out = t;
          if (GRAD) { g[q] = da; g[qb] = db; g[qd] = dd; }
        } else {
          out = 1.0f - t;
          if (GRAD) { g[q] = -da; g[qb] = -db; g[qd] = -dd; }
        }
      }
    }
  } else if (s == 2) {
    bool adjacent = false;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int q1 = (q + 1) & 3, q2 = (q + 2) & 3, q3 = (q + 3) & 3;
      if (F[q] && F[q1]) {  // fluid corners q, q+1; solid neighbours q-1 (of q) and q+2 (of q+1)
        adjacent = true;
        const float A = P[q], B = P[q1], C = P[q2], D = P[q3];
        const float iad = 1.0f / (A - D), ibc = 1.0f / (B - C);
        out = 0.5f * (A / (A - D) + B / (B - C));
        if (GRAD) {
          g[q] = 0.5f * (-D * iad * iad);
          g[q3] = 0.5f * (A * iad * iad);
          g[q1] = 0.5f * (-C * ibc * ibc);
          g[q2] = 0.5f * (B * ibc * ibc);
        }
      }
    }
    if (!adjacent) {  // diagonal: tie-break on the mean of the four values (R3)
      const float mean = 0.25f * (P[0] + P[1] + P[2] + P[3]);
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const int q1 = q + 1, q2 = (q + 2) & 3, q3 = (q + 3) & 3;
        if (F[q] && F[q2]) {
          const float A = P[q], B = P[q1], C = P[q2], D = P[q3];
          float a1, b1, c1, a2, b2, c2;
          if (mean > 0.0f) {  // fluid joined: 1 - two solid triangles at B and D
            const float t1 = nf_tri<GRAD>(B, C, A, a1, b1, c1);  // corner B, neighbours C and A
            const float t2 = nf_tri<GRAD>(D, A, C, a2, b2, c2);  // corner D, neighbours A and C
            out = 1.0f - t1 - t2;
            if (GRAD) {
              g[q1] = -a1; g[q2] = -b1 - c2; g[q] = -c1 - b2; g[q3] = -a2;
            }
          } else {  // fluid separated: two fluid triangles at A and C
            const float t1 = nf_tri<GRAD>(A, B, D, a1, b1, c1);
            const float t2 = nf_tri<GRAD>(C, D, B, a2, b2, c2);
            out = t1 + t2;
            if (GRAD) {
              g[q] = a1; g[q1] = b1 + c2; g[q3] = c1 + b2; g[q2] = a2;
            }
          }
        }
      }
    }
  }
  if (out < NF_ALPHA_EPS) {  // R4
    out = 0.0f;
    if (GRAD) { g[0] = g[1] = g[2] = g[3] = 0.0f; }
  }
  if (GRAD) { d[0] = g[0]; d[1] = g[1]; d[2] = g[2]; d[3] = g[3]; }
  return out;
}

struct NfBc6 {
  int t[6];
};

// One thread per "extended cell" (i <= nx, j <= ny, k <= nz): it owns the low x-, y- and z-face of that cell.
__global__ void __launch_bounds__(256) k_weights_from_sdf(const float *__restrict__ phi, float *__restrict__ ax,
                                                          float *__restrict__ ay, float *__restrict__ az, int nx,
                                                          int ny, int nz, int pax, NfBc6 bc) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i > nx || j > ny || k > nz) return;
  const size_t sx = 1, sy = (size_t)nx + 1, sz = (size_t)(nx + 1) * (ny + 1);
  const size_t n0 = (size_t)k * sz + (size_t)j * sy + i;
  const bool hi = i < nx, hj = j < ny, hk = k < nz;
  const float p000 = __ldg(phi + n0);
  const float p001 = hi ? __ldg(phi + n0 + sx) : 0.0f;
  const float p010 = hj ? __ldg(phi + n0 + sy) : 0.0f;
  const float p100 = hk ? __ldg(phi + n0 + sz) : 0.0f;
  if (hj && hk) {  // x-face: corners (k,j),(k,j+1),(k+1,j+1),(k+1,j) at node column i
    const float p110 = __ldg(phi + n0 + sy + sz);
    float a = nf_area_fraction<false>(p000, p010, p110, p100, nullptr);
    if ((i == 0 && bc.t[0] == NF_BC_CLOSED) || (i == nx && bc.t[1] == NF_BC_CLOSED)) a = 0.0f;
    ax[((size_t)k * ny + j) * pax + i] = a;
  }
  if (hi && hk) {  // y-face: corners (k,i),(k,i+1),(k+1,i+1),(k+1,i)
    const float p101 = __ldg(phi + n0 + sx + sz);
    float a = nf_area_fraction<false>(p000, p001, p101, p100, nullptr);
    if ((j == 0 && bc.t[2] == NF_BC_CLOSED) || (j == ny && bc.t[3] == NF_BC_CLOSED)) a = 0.0f;
    ay[((size_t)k * (ny + 1) + j) * nx + i] = a;
  }
  if (hi && hj) {  // z-face: corners (j,i),(j,i+1),(j+1,i+1),(j+1,i)
    const float p011 = __ldg(phi + n0 + sx + sy);
    float a = nf_area_fraction<false>(p000, p001, p011, p010, nullptr);
    if ((k == 0 && bc.t[4] == NF_BC_CLOSED) || (k == nz && bc.t[5] == NF_BC_CLOSED)) a = 0.0f;
    az[((size_t)k * ny + j) * nx + i] = a;
  }
}

// a-10: scatter dJ/dalpha * d alpha/d phi to the four corner nodes of every face.
__global__ void __launch_bounds__(256) k_weights_adjoint(const float *__restrict__ phi, const float *__restrict__ gau,
                                                         const float *__restrict__ gav, const float *__restrict__ gaw,
                                                         float *__restrict__ gphi, int nx, int ny, int nz, NfBc6 bc) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i > nx || j > ny || k > nz) return;
  const size_t sx = 1, sy = (size_t)nx + 1, sz = (size_t)(nx + 1) * (ny + 1);
  const size_t n0 = (size_t)k * sz + (size_t)j * sy + i;
  const bool hi = i < nx, hj = j < ny, hk = k < nz;
  const float p000 = __ldg(phi + n0);
  const float p001 = hi ? __ldg(phi + n0 + sx) : 0.0f;
  const float p010 = hj ? __ldg(phi + n0 + sy) : 0.0f;
  const float p100 = hk ? __ldg(phi + n0 + sz) : 0.0f;
  float d[4];
  if (hj && hk && !((i == 0 && bc.t[0] == NF_BC_CLOSED) || (i == nx && bc.t[1] == NF_BC_CLOSED))) {
    const float p110 = __ldg(phi + n0 + sy + sz);
    const bool any = (p000 > 0) | (p010 > 0) | (p110 > 0) | (p100 > 0);
    const bool all = (p000 > 0) & (p010 > 0) & (p110 > 0) & (p100 > 0);
    if (any && !all) {
      nf_area_fraction<true>(p000, p010, p110, p100, d);
      const float ga = __ldg(gau + ((size_t)k * ny + j) * (nx + 1) + i);
      if (d[0] != 0.0f) atomicAdd(gphi + n0, ga * d[0]);
      if (d[1] != 0.0f) atomicAdd(gphi + n0 + sy, ga * d[1]);
      if (d[2] != 0.0f) atomicAdd(gphi + n0 + sy + sz, ga * d[2]);
      if (d[3] != 0.0f) atomicAdd(gphi + n0 + sz, ga * d[3]);
    }
  }
  if (hi && hk && !((j == 0 && bc.t[2] == NF_BC_CLOSED) || (j == ny && bc.t[3] == NF_BC_CLOSED))) {
    const float p101 = __ldg(phi + n0 + sx + sz);
    const bool any = (p000 > 0) | (p001 > 0) | (p101 > 0) | (p100 > 0);
    const bool all = (p000 > 0) & (p001 > 0) & (p101 > 0) & (p100 > 0);
    if (any && !all) {
      nf_area_fraction<true>(p000, p001, p101, p100, d);
      const float ga = __ldg(gav + ((size_t)k * (ny + 1) + j) * nx + i);
      if (d[0] != 0.0f) atomicAdd(gphi + n0, ga * d[0]);
      if (d[1] != 0.0f) atomicAdd(gphi + n0 + sx, ga * d[1]);
      if (d[2] != 0.0f) atomicAdd(gphi + n0 + sx + sz, ga * d[2]);
      if (d[3] != 0.0f) atomicAdd(gphi + n0 + sz, ga * d[3]);
    }
  }
  if (hi && hj && !((k == 0 && bc.t[4] == NF_BC_CLOSED) || (k == nz && bc.t[5] == NF_BC_CLOSED))) {
    const float p011 = __ldg(phi + n0 + sx + sy);
    const bool any = (p000 > 0) | (p001 > 0) | (p011 > 0) | (p010 > 0);
    const bool all = (p000 > 0) & (p001 > 0) & (p011 > 0) & (p010 > 0);
    if (any && !all) {
      nf_area_fraction<true>(p000, p001, p011, p010, d);
      const float ga = __ldg(gaw + ((size_t)k * ny + j) * nx + i);
      if (d[0] != 0.0f) atomicAdd(gphi + n0, ga * d[0]);
      if (d[1] != 0.0f) atomicAdd(gphi + n0 + sx, ga * d[1]);
      if (d[2] != 0.0f) atomicAdd(gphi + n0 + sx + sy, ga * d[2]);
      if (d[3] != 0.0f) atomicAdd(gphi + n0 + sy, ga * d[3]);
    }
  }
}

// Copy user MAC-layout weights into the internal layout (x rows padded to pax), forcing closed walls to 0.
__global__ void __launch_bounds__(256) k_weights_import(const float *__restrict__ au, const float *__restrict__ av,
                                                        const float *__restrict__ aw, float *__restrict__ ax,
                                                        float *__restrict__ ay, float *__restrict__ az, int nx, int ny,
                                                        int nz, int pax, NfBc6 bc) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i > nx || j > ny || k > nz) return;
  if (j < ny && k < nz) {
    float a = au[((size_t)k * ny + j) * (nx + 1) + i];
    if ((i == 0 && bc.t[0] == NF_BC_CLOSED) || (i == nx && bc.t[1] == NF_BC_CLOSED)) a = 0.0f;
    ax[((size_t)k * ny + j) * pax + i] = a;
  }
  if (i < nx && k < nz) {
    float a = av[((size_t)k * (ny + 1) + j) * nx + i];
    if ((j == 0 && bc.t[2] == NF_BC_CLOSED) || (j == ny && bc.t[3] == NF_BC_CLOSED)) a = 0.0f;
    ay[((size_t)k * (ny + 1) + j) * nx + i] = a;
  }
  if (i < nx && j < ny) {
    float a = aw[((size_t)k * ny + j) * nx + i];
    if ((k == 0 && bc.t[4] == NF_BC_CLOSED) || (k == nz && bc.t[5] == NF_BC_CLOSED)) a = 0.0f;
    az[((size_t)k * ny + j) * nx + i] = a;
  }
}

__global__ void __launch_bounds__(256) k_weights_export(const float *__restrict__ ax, float *__restrict__ au, int nx,
                                                        int ny, int nz, int pax) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i > nx || j >= ny || k >= nz) return;
  au[((size_t)k * ny + j) * (nx + 1) + i] = ax[((size_t)k * ny + j) * pax + i];
}

// Coarse face weight = arithmetic mean of the coincident fine face weights (R13): four of them,
// or -- in 2-D mode, fz == 1, where z does not coarsen -- the two of an x- or y-face and the four of a z-face.
__global__ void __launch_bounds__(256) k_coarsen_weights(const float *__restrict__ fax, const float *__restrict__ fay,
                                                         const float *__restrict__ faz, float *__restrict__ cax,
                                                         float *__restrict__ cay, float *__restrict__ caz, int fnx,
                                                         int fny, int fnz, int fpax, int cnx, int cny, int cnz,
                                                         int cpax, int fz) {
  const int I = blockIdx.x * blockDim.x + threadIdx.x;
  const int J = blockIdx.y * blockDim.y + threadIdx.y;
  const int K = blockIdx.z * blockDim.z + threadIdx.z;
  if (I > cnx || J > cny || K > cnz) return;
  // Coarse face weight = mean of the (up to) four coincident fine faces; fine faces beyond an odd extent do not exist
  // and count as closed.  The coarse boundary face of an odd axis coincides with the fine boundary face.
  const int i = 2 * I, j = 2 * J, k = fz * K;
  auto fx = [&](int ii, int jj, int kk) -> float {
    return (jj < fny && kk < fnz) ? fax[((size_t)kk * fny + jj) * fpax + min(ii, fnx)] : 0.0f;
  };
  auto fy = [&](int ii, int jj, int kk) -> float {
    return (ii < fnx && kk < fnz) ? fay[((size_t)kk * (fny + 1) + min(jj, fny)) * fnx + ii] : 0.0f;
  };
  auto fzf = [&](int ii, int jj, int kk) -> float {
    return (ii < fnx && jj < fny) ? faz[((size_t)min(kk, fnz) * fny + jj) * fnx + ii] : 0.0f;
  };
  if (J < cny && K < cnz)
    cax[((size_t)K * cny + J) * cpax + I] = fz == 2 ? 0.25f * ((fx(i, j, k) + fx(i, j + 1, k)) + (fx(i, j, k + 1) + fx(i, j + 1, k + 1)))
                                                    : 0.5f * (fx(i, j, k) + fx(i, j + 1, k));
  if (I < cnx && K < cnz)
    cay[((size_t)K * (cny + 1) + J) * cnx + I] = fz == 2 ? 0.25f * ((fy(i, j, k) + fy(i + 1, j, k)) + (fy(i, j, k + 1) + fy(i + 1, j, k + 1)))
                                                         : 0.5f * (fy(i, j, k) + fy(i + 1, j, k));
  if (I < cnx && J < cny)
    caz[((size_t)K * cny + J) * cnx + I] = 0.25f * ((fzf(i, j, k) + fzf(i + 1, j, k)) + (fzf(i, j + 1, k) + fzf(i + 1, j + 1, k)));
}

// Cell codes of one level from its fp32 weights: bits 0..5 = face is fully open, bit 6 = the
// cell has a fractional face.  With counts != nullptr (level 0) also: counts[0] += active cells (sum of six
// weights > 0); counts[1] += open faces on Dirichlet domain faces (R12).
#define NF_ENC_KCH 8
__global__ void __launch_bounds__(256) k_encode(const float *__restrict__ ax, const float *__restrict__ ay,
                                                const float *__restrict__ az, uint8_t *__restrict__ code,
                                                float *__restrict__ idg, float ic, int nx, int ny, int nz, int pax,
                                                NfBc6 bc, double *__restrict__ counts) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  double act = 0.0, dir = 0.0;
  // (each CTA marches through NF_ENC_KCH planes: 8x fewer same-address fp64 atomics for the two counts)
  for (int k = blockIdx.z * NF_ENC_KCH; k < min((int)(blockIdx.z + 1) * NF_ENC_KCH, nz); ++k)
  if (i < nx && j < ny) {
    float w[6];
    w[0] = ax[((size_t)k * ny + j) * pax + i];
    w[1] = ax[((size_t)k * ny + j) * pax + i + 1];
    w[2] = ay[((size_t)k * (ny + 1) + j) * nx + i];
    w[3] = ay[((size_t)k * (ny + 1) + j + 1) * nx + i];
    w[4] = az[((size_t)k * ny + j) * nx + i];
    w[5] = az[((size_t)(k + 1) * ny + j) * nx + i];
    unsigned c = 0;
    bool mixed = false;
#pragma unroll
    for (int f = 0; f < 6; ++f) {
      if (w[f] == 1.0f) c |= 1u << f;
      else if (w[f] != 0.0f) mixed = true;
    }
    if (mixed) c |= NF_CODE_MIXED;
    code[((size_t)k * ny + j) * nx + i] = (uint8_t)c;
    {  // the smoother's inverse diagonal, in the arithmetic of nf_code_idiag (nf_stencil.cuh)
      const float d = ((w[0] + w[1]) + (w[2] + w[3])) + (w[4] + w[5]);
      const float inv_count[8] = {0.0f, 1.0f, 0.5f, 1.0f / 3.0f, 0.25f, 0.2f, 1.0f / 6.0f, 0.0f};
      idg[((size_t)k * ny + j) * nx + i] = mixed ? (d > 0.0f ? ic / d : 0.0f) : ic * inv_count[__popc(c & 63u)];
    }
    if (counts) {
      if (w[0] + w[1] + w[2] + w[3] + w[4] + w[5] > 0.0f) act += 1.0;
      if (i == 0 && bc.t[0] == NF_BC_DIRICHLET && w[0] > 0.0f) dir += 1.0;
      if (i == nx - 1 && bc.t[1] == NF_BC_DIRICHLET && w[1] > 0.0f) dir += 1.0;
      if (j == 0 && bc.t[2] == NF_BC_DIRICHLET && w[2] > 0.0f) dir += 1.0;
      if (j == ny - 1 && bc.t[3] == NF_BC_DIRICHLET && w[3] > 0.0f) dir += 1.0;
      if (k == 0 && bc.t[4] == NF_BC_DIRICHLET && w[4] > 0.0f) dir += 1.0;
      if (k == nz - 1 && bc.t[5] == NF_BC_DIRICHLET && w[5] > 0.0f) dir += 1.0;
    }
  }
  if (counts) {
    nf_block_atomic_add(act, counts + 0);
    nf_block_atomic_add(dir, counts + 1);
  }
}

// Second pass of the encoding: set NF_CODE_DEEP (in place: the bit is not an input of this kernel).
__global__ void __launch_bounds__(256) k_encode_deep(uint8_t *code, int nx, int ny, int nz) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= nx || j >= ny || k >= nz) return;
  const size_t id = ((size_t)k * ny + j) * nx + i, sy = nx, sz = (size_t)nx * ny;
  const unsigned full = 63u, m = 127u;
  bool deep = (code[id] & m) == full;
  deep = deep && (i == 0 || (code[id - 1] & m) == full) && (i + 1 == nx || (code[id + 1] & m) == full);
  deep = deep && (j == 0 || (code[id - sy] & m) == full) && (j + 1 == ny || (code[id + sy] & m) == full);
  deep = deep && (k == 0 || (code[id - sz] & m) == full) && (k + 1 == nz || (code[id + sz] & m) == full);
  if (deep) code[id] = (uint8_t)(full | NF_CODE_DEEP);
}

// Copy a MAC face array (or zero it when src == nullptr) and put closed walls at rest (R19).
__global__ void __launch_bounds__(256) k_store_us(const float *__restrict__ src, float *__restrict__ dst, int ex, int ey,
                                                  int ez, int axis, int closed_lo, int closed_hi) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z * blockDim.z + threadIdx.z;
  if (i >= ex || j >= ey || k >= ez) return;
  const size_t id = ((size_t)k * ey + j) * ex + i;
  float v = src ? src[id] : 0.0f;
  const int c = axis == 0 ? i : (axis == 1 ? j : k);
  const int e = axis == 0 ? ex : (axis == 1 ? ey : ez);
  if ((c == 0 && closed_lo) || (c == e - 1 && closed_hi)) v = 0.0f;
  dst[id] = v;
}

static NfBc6 bc6(const nf_grid *g) {
  NfBc6 b;
  for (int f = 0; f < 6; ++f) b.t[f] = g->bc_type[f];
  return b;
}

int nf_weights_from_sdf(nf_grid *g, const float *sdf) {
  NfLevel &L = g->lv[0];
  NfDims d = nf_dims(g->nx + 1, g->ny + 1, g->nz + 1);
  NF_CUDA(g, cudaMemcpyAsync(g->sdf, sdf, nf_nn(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_LAUNCH(g, NFK_WEIGHTS, k_weights_from_sdf<<<d.grid, d.block, 0, g->stream>>>(g->sdf, L.ax, L.ay, L.az, g->nx, g->ny, g->nz, L.pax, bc6(g)));
  g->have_sdf = true;
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_weights_from_user(nf_grid *g, const float *au, const float *av, const float *aw) {
  NfLevel &L = g->lv[0];
  NfDims d = nf_dims(g->nx + 1, g->ny + 1, g->nz + 1);
  NF_LAUNCH(g, NFK_WEIGHTS, k_weights_import<<<d.grid, d.block, 0, g->stream>>>(au, av, aw, L.ax, L.ay, L.az, g->nx, g->ny, g->nz, L.pax, bc6(g)));
  g->have_sdf = false;
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_weights_to_user(nf_grid *g, float *au, float *av, float *aw) {
  NfLevel &L = g->lv[0];
  if (au) {
    NfDims d = nf_dims(g->nx + 1, g->ny, g->nz);
    NF_LAUNCH(g, NFK_MISC, k_weights_export<<<d.grid, d.block, 0, g->stream>>>(L.ax, au, g->nx, g->ny, g->nz, L.pax));
  }
  if (av) NF_CUDA(g, cudaMemcpyAsync(av, L.ay, nf_nv(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  if (aw) NF_CUDA(g, cudaMemcpyAsync(aw, L.az, nf_nw(g) * sizeof(float), cudaMemcpyDeviceToDevice, g->stream));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_build_hierarchy(nf_grid *g) {
  for (int l = 0; l + 1 < g->nlev; ++l) {
    NfLevel &F = g->lv[l], &C = g->lv[l + 1];
    NfDims d = nf_dims(C.nx + 1, C.ny + 1, C.nz + 1);
    NF_LAUNCH(g, NFK_COARSEN, k_coarsen_weights<<<d.grid, d.block, 0, g->stream>>>(F.ax, F.ay, F.az, C.ax, C.ay, C.az, F.nx, F.ny, F.nz, F.pax,
                                                         C.nx, C.ny, C.nz, C.pax, F.fz));
  }
  double *cnt = g->d_counts;
  NF_CUDA(g, cudaMemsetAsync(cnt, 0, 2 * sizeof(double), g->stream));
  for (int l = 0; l < g->nlev; ++l) {
    NfLevel &L = g->lv[l];
    NfDims d = nf_dims(L.nx, L.ny, L.nz);
    NfDims de = nf_dims(L.nx, L.ny, 1);
    de.grid.z = (L.nz + NF_ENC_KCH - 1) / NF_ENC_KCH;
    NF_LAUNCH(g, NFK_CLASSIFY, k_encode<<<de.grid, de.block, 0, g->stream>>>(L.ax, L.ay, L.az, L.code, L.idg, 1.0f / L.c, L.nx, L.ny, L.nz, L.pax, bc6(g), l == 0 ? cnt : nullptr));
    if (L.vec) NF_LAUNCH(g, NFK_CLASSIFY, k_encode_deep<<<d.grid, d.block, 0, g->stream>>>(L.code, L.nx, L.ny, L.nz));
  }
  NF_CUDA(g, cudaGetLastError());
  NF_TRY(nf_components_build(g));  // fluid components of level 0 (R12 per component, nf_components.cu)
  {
    int rc = nf_mg_pack_tail(g);
    if (rc != NF_OK) return rc;
  }
  NF_CUDA(g, cudaMemcpyAsync(g->h_counts, cnt, 2 * sizeof(double), cudaMemcpyDeviceToHost, g->stream));
  // The counts (active cells, Dirichlet faces, components) are read lazily: nf_meta_sync waits for this event the
  // first time a call needs them, so that nf_set_solid itself does not drain the stream (many small environments on
  // one stream: their hierarchy builds queue up back to back).
  NF_CUDA(g, cudaEventRecord(g->ev_meta, g->stream));
  g->meta_pending = true;
  g->weights_set = true;
  return nf_mg_upload_coarse(g);
}

// Host copies of the device-side counts of the last hierarchy build (blocks until that build has run).
int nf_meta_sync(nf_grid *g) {
  if (!g->meta_pending) return NF_OK;
  NF_CUDA(g, cudaEventSynchronize(g->ev_meta));
  g->meta_pending = false;
  const double *hc = g->h_counts;
  g->nact = (long long)hc[0];
  g->singular_info = hc[1] > 0.0 ? 0 : 1;
  // null-space handling (R12): none / one global mean / per component
  if (g->comp && g->h_cc_meta[0] > 1) {
    g->ncomp = g->h_cc_meta[0];
    g->nsing = g->h_cc_meta[2];
    g->gauge_mode = g->nsing > 0 ? 2 : 0;
  } else {
    g->ncomp = g->nact > 0 ? 1 : 0;
    g->nsing = g->singular_info ? g->ncomp : 0;
    g->gauge_mode = g->singular_info ? 1 : 0;
  }
  g->singular = g->gauge_mode == 1 ? 1 : 0;
  return NF_OK;
}

int nf_store_solid_velocity(nf_grid *g, const float *us, const float *vs, const float *ws) {
  g->have_us = (us || vs || ws);
  if (!g->have_us) return NF_OK;  // kernels treat U_s as identically zero
  const int cl[6] = {g->bc_type[0] == NF_BC_CLOSED, g->bc_type[1] == NF_BC_CLOSED, g->bc_type[2] == NF_BC_CLOSED,
                     g->bc_type[3] == NF_BC_CLOSED, g->bc_type[4] == NF_BC_CLOSED, g->bc_type[5] == NF_BC_CLOSED};
  NfDims d = nf_dims(g->nx + 1, g->ny, g->nz);
  NF_LAUNCH(g, NFK_STORE_US, k_store_us<<<d.grid, d.block, 0, g->stream>>>(us, g->us, g->nx + 1, g->ny, g->nz, 0, cl[0], cl[1]));
  d = nf_dims(g->nx, g->ny + 1, g->nz);
  NF_LAUNCH(g, NFK_STORE_US, k_store_us<<<d.grid, d.block, 0, g->stream>>>(vs, g->vs, g->nx, g->ny + 1, g->nz, 1, cl[2], cl[3]));
  d = nf_dims(g->nx, g->ny, g->nz + 1);
  NF_LAUNCH(g, NFK_STORE_US, k_store_us<<<d.grid, d.block, 0, g->stream>>>(ws, g->ws, g->nx, g->ny, g->nz + 1, 2, cl[4], cl[5]));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_weights_adjoint_impl(nf_grid *g, const float *gau, const float *gav, const float *gaw, float *gsdf) {
  NF_CUDA(g, cudaMemsetAsync(gsdf, 0, nf_nn(g) * sizeof(float), g->stream));
  NfDims d = nf_dims(g->nx + 1, g->ny + 1, g->nz + 1);
  NF_LAUNCH(g, NFK_WEIGHTS_ADJ, k_weights_adjoint<<<d.grid, d.block, 0, g->stream>>>(g->sdf, gau, gav, gaw, gsdf, g->nx, g->ny, g->nz, bc6(g)));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}
