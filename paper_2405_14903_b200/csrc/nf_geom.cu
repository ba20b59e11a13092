// nf_geom.cu -- SURVEY.md 8f NEXT-2: the differentiable parametric geometry of PAPER.md:L55-67 (section 2.2) and
// L337-347 (appendix A) on the device: polar-Bezier cross-sections, key sections along z, the node SDF phi, its
// adjoint to the parameters (L141), CSG (L67) and the solid velocity of a moving geometry (L89, L132).
// Readings R25-R31.
//
// One CTA = 1024 consecutive points (x fastest) of ONE z-plane.  Every point of a plane sees the same cross-section, so
// the CTA first builds it in shared memory -- the interpolated section, the N M vertices of the sampled Bezier curves (fp64,
// N M <= 2048 values: noise), one 6-float record per polygon edge -- and then every thread scans the N M edges for
// 4 points (distance, closest edge, parity of the +x ray).  ALU-bound: ~20 fp32 instructions per (point, edge).
// The reverse kernels redo the scan, scatter into per-CTA vertex gradients (shared-memory atomics; only cut-cell
// nodes carry a gradient in practice) and chain vertices -> control points -> section -> key sections in the CTA,
// ending in a handful of fp64 atomics on the parameter gradient.
#include "nf_internal.cuh"

#define NF_GEOM_NT 256  // threads per CTA
#define NF_GEOM_PPT 4   // points per thread: plane offsets base + tid + 256 q (no tile edges: a plane of 257 x 257 nodes
                        // wastes 0.8 % of the lanes, a 64 x 16 tiling 20 %)

struct NfGeomK {
  const float *par;   // device: [z0, z1, K x (cx, cy, rho1[N], rho2[N])]
  const float *pdot;  // device: same layout (velocity kernels), else nullptr
  int K, N, M;
  float dx;
};

struct NfGeomPlane {
  double z, z0, z1, lam;
  int k0, k1;    // key sections bracketing the plane
  bool clamped;  // the section does not depend on z0 / z1 here
  int cap;       // which cap the slab term max(z0 - z, z - z1) refers to
  float slab;
};

// shared-memory carve-up (nf_geom_smem_bytes must agree)
struct NfGeomSm {
  double *sec, *secd, *gsec;  // W = 2 + 2N each: section, its time derivative, its gradient
  double *cur;                // 16 per curve: cos[4], sin[4] of the control directions, radii[4], their rates[4]
  float *seg;                 // 6 per edge: ax, ay, ex, ey, 1/|e|^2, ex/ey
  float *V, *Vd, *gV;         // 2 per vertex: position, velocity, gradient
  float *ctrl;                // 8 per curve: gradient w.r.t. e0, p0, p1, e1
  float *gsl;                 // [2]: gradient w.r.t. the caps; [2] = "any point of the CTA carried a gradient"
  int *bb;                    // [4]: bounding box of the polygon as order-preserving ints (velocity kernels' band cull)
};
static size_t nf_geom_smem_bytes(int N, int M) {
  const size_t W = 2 + 2 * (size_t)N, NM = (size_t)N * M;
  return (3 * W + 16 * (size_t)N) * sizeof(double) + (6 * NM + 3 * 2 * NM + 8 * (size_t)N + 8) * sizeof(float);
}
__device__ __forceinline__ NfGeomSm nf_geom_carve(unsigned char *raw, int N, int M) {
  const int W = 2 + 2 * N, NM = N * M;
  NfGeomSm s;
  s.sec = reinterpret_cast<double *>(raw);
  s.secd = s.sec + W;
  s.gsec = s.secd + W;
  s.cur = s.gsec + W;
  s.seg = reinterpret_cast<float *>(s.cur + 16 * N);
  s.V = s.seg + 6 * NM;
  s.Vd = s.V + 2 * NM;
  s.gV = s.Vd + 2 * NM;
  s.ctrl = s.gV + 2 * NM;
  s.gsl = s.ctrl + 8 * N;
  s.bb = reinterpret_cast<int *>(s.gsl + 4);
  return s;
}

// R27: K key sections evenly spaced on [z0, z1], piecewise-linear in s = clamp((z - z0)/(z1 - z0), 0, 1)
__device__ __forceinline__ NfGeomPlane nf_geom_plane(const NfGeomK &G, double z) {
  NfGeomPlane P;
  P.z = z;
  P.z0 = (double)G.par[0];
  P.z1 = (double)G.par[1];
  const double sr = (z - P.z0) / (P.z1 - P.z0);
  const double s = fmin(fmax(sr, 0.0), 1.0);
  P.clamped = !(sr > 0.0 && sr < 1.0) || G.K == 1;
  if (G.K == 1) {
    P.k0 = P.k1 = 0;
    P.lam = 0.0;
  } else {
    const double t = s * (double)(G.K - 1);
    P.k0 = min((int)floor(t), G.K - 2);
    P.k1 = P.k0 + 1;
    P.lam = t - (double)P.k0;
  }
  P.cap = (P.z0 - z >= z - P.z1) ? 0 : 1;
  P.slab = (float)fmax(P.z0 - z, z - P.z1);
  return P;
}

__device__ __forceinline__ void nf_bernstein3(double t, double B[4]) {
  const double u = 1.0 - t;
  B[0] = u * u * u;
  B[1] = 3.0 * u * u * t;
  B[2] = 3.0 * u * t * t;
  B[3] = t * t * t;
}

// The four control directions of curve i (appendix A): e0 at theta_i, p0 at theta_i + delta, p1 at
// theta_{i+1} - delta, e1 at theta_{i+1}; theta_i = 2 pi i / N, delta = 2 pi / (3N).
__device__ __forceinline__ void nf_curve_dirs(int i, int N, double cs[4], double sn[4]) {
  const double inv = 1.0 / (3.0 * (double)N);
  sincospi((double)(6 * i) * inv, &sn[0], &cs[0]);
  sincospi((double)(6 * i + 2) * inv, &sn[1], &cs[1]);
  sincospi((double)(6 * i + 4) * inv, &sn[2], &cs[2]);
  sincospi((double)(6 * i + 6) * inv, &sn[3], &cs[3]);
}

// Builds the plane's cross-section in shared memory.  All threads of the CTA call it.
__device__ void nf_geom_setup(const NfGeomK &G, const NfGeomPlane &P, const NfGeomSm &S, bool zero_grad) {
  const int tid = threadIdx.x, nth = blockDim.x;
  const int N = G.N, M = G.M, W = 2 + 2 * N, NM = N * M;
  const float *k0 = G.par + 2 + (size_t)P.k0 * W, *k1 = G.par + 2 + (size_t)P.k1 * W;
  double sdot = 0.0;
  if (G.pdot && !P.clamped) {
    const double L = P.z1 - P.z0;
    sdot = ((double)G.pdot[0] * (P.z - P.z1) - (double)G.pdot[1] * (P.z - P.z0)) / (L * L);
  }
  for (int t = tid; t < W; t += nth) {
    const double a = (double)k0[t], b = (double)k1[t];
    S.sec[t] = (1.0 - P.lam) * a + P.lam * b;
    if (G.pdot) {
      const float *d0 = G.pdot + 2 + (size_t)P.k0 * W, *d1 = G.pdot + 2 + (size_t)P.k1 * W;
      S.secd[t] = (1.0 - P.lam) * (double)d0[t] + P.lam * (double)d1[t] + sdot * (double)(G.K - 1) * (b - a);
    }
    S.gsec[t] = 0.0;
  }
  if (tid < 3) S.gsl[tid] = 0.0f;
  __syncthreads();
  // per curve: the four control directions, the four radii (R25: endpoint radius 2 cos(delta) a b / (a + b), a = rho2 of
  // the curve before the endpoint, b = rho1 of the curve after it) and their rates
  {
    const double cdl = cospi(2.0 / (3.0 * (double)N));
    const double *r1 = S.sec + 2, *r2 = S.sec + 2 + N, *r1d = S.secd + 2, *r2d = S.secd + 2 + N;
    for (int i = tid; i < N; i += nth) {
      const int im = (i + N - 1) % N, ip = (i + 1) % N;
      double *c = S.cur + 16 * i;
      nf_curve_dirs(i, N, c, c + 4);
      const double a0 = r2[im], b0 = r1[i], a1 = r2[i], b1 = r1[ip];
      c[8] = 2.0 * cdl * a0 * b0 / (a0 + b0);
      c[9] = r1[i];
      c[10] = r2[i];
      c[11] = 2.0 * cdl * a1 * b1 / (a1 + b1);
      if (G.pdot) {
        c[12] = 2.0 * cdl * (b0 * b0 * r2d[im] + a0 * a0 * r1d[i]) / ((a0 + b0) * (a0 + b0));
        c[13] = r1d[i];
        c[14] = r2d[i];
        c[15] = 2.0 * cdl * (b1 * b1 * r2d[i] + a1 * a1 * r1d[ip]) / ((a1 + b1) * (a1 + b1));
      }
    }
  }
  __syncthreads();
  for (int v = tid; v < NM; v += nth) {
    const int i = v / M, m = v - i * M;
    const double *c = S.cur + 16 * i;
    double B[4];
    nf_bernstein3((double)m / (double)M, B);
    double x = S.sec[0], y = S.sec[1];
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      x += B[b] * c[8 + b] * c[b];
      y += B[b] * c[8 + b] * c[4 + b];
    }
    S.V[2 * v] = (float)x;
    S.V[2 * v + 1] = (float)y;
    if (G.pdot) {
      double xd = S.secd[0], yd = S.secd[1];
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        xd += B[b] * c[12 + b] * c[b];
        yd += B[b] * c[12 + b] * c[4 + b];
      }
      S.Vd[2 * v] = (float)xd;
      S.Vd[2 * v + 1] = (float)yd;
    }
    if (zero_grad) S.gV[2 * v] = S.gV[2 * v + 1] = 0.0f;
  }
  __syncthreads();
  for (int v = tid; v < NM; v += nth) {
    const int w = v + 1 == NM ? 0 : v + 1;
    const float ax = S.V[2 * v], ay = S.V[2 * v + 1];
    const float ex = S.V[2 * w] - ax, ey = S.V[2 * w + 1] - ay;
    const float l2 = ex * ex + ey * ey;
    float *sg = S.seg + 6 * v;
    sg[0] = ax; sg[1] = ay; sg[2] = ex; sg[3] = ey;
    sg[4] = l2 > 0.0f ? 1.0f / l2 : 0.0f;
    sg[5] = ey != 0.0f ? ex / ey : 0.0f;
  }
  __syncthreads();
}

// R26: exact distance of NF_GEOM_PPT points to the closed polygon, the closest edge and the parameter on it, and the
// even-odd parity of the ray towards +x.
template <bool TRACK>
__device__ __forceinline__ void nf_geom_scan(const float *__restrict__ seg, int NM, const float (&X)[NF_GEOM_PPT],
                                             const float (&Y)[NF_GEOM_PPT],
                                             float (&d2)[NF_GEOM_PPT], int (&kb)[NF_GEOM_PPT],
                                             float (&tb)[NF_GEOM_PPT], unsigned &inside) {
#pragma unroll
  for (int q = 0; q < NF_GEOM_PPT; ++q) { d2[q] = INFINITY; kb[q] = 0; tb[q] = 0.0f; }
  inside = 0u;
  for (int k = 0; k < NM; ++k) {
    const float2 a = *reinterpret_cast<const float2 *>(seg + 6 * k);
    const float2 e = *reinterpret_cast<const float2 *>(seg + 6 * k + 2);
    const float2 c = *reinterpret_cast<const float2 *>(seg + 6 * k + 4);
    const float by = a.y + e.y;
#pragma unroll
    for (int q = 0; q < NF_GEOM_PPT; ++q) {
      const float dxp = X[q] - a.x, dyp = Y[q] - a.y;
      const float tau = __saturatef((dxp * e.x + dyp * e.y) * c.x);
      const float rx = dxp - tau * e.x, ry = dyp - tau * e.y;
      const float d = rx * rx + ry * ry;
      if (d < d2[q]) {
        d2[q] = d;
        if (TRACK) { kb[q] = k; tb[q] = tau; }
      }
      const bool strad = (a.y > Y[q]) != (by > Y[q]);
      inside ^= (strad && dxp < dyp * c.y) ? (1u << q) : 0u;
    }
  }
}

// vertices -> control points -> (c, rho1, rho2) of the section -> key sections, z0, z1.  All threads call it.
__device__ void nf_geom_chain(const NfGeomK &G, const NfGeomPlane &P, const NfGeomSm &S, double *gout) {
  __syncthreads();
  if (S.gsl[2] == 0.0f) return;  // (uniform: read after the barrier)
  const int tid = threadIdx.x, nth = blockDim.x;
  const int N = G.N, M = G.M, W = 2 + 2 * N;
  for (int i = tid; i < N; i += nth) {
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int m = 0; m < M; ++m) {
      double B[4];
      nf_bernstein3((double)m / (double)M, B);
      const double gx = S.gV[2 * (i * M + m)], gy = S.gV[2 * (i * M + m) + 1];
#pragma unroll
      for (int c = 0; c < 4; ++c) { acc[2 * c] += B[c] * gx; acc[2 * c + 1] += B[c] * gy; }
    }
#pragma unroll
    for (int c = 0; c < 8; ++c) S.ctrl[8 * i + c] = (float)acc[c];
  }
  __syncthreads();
  const double cdl = cospi(2.0 / (3.0 * (double)N));
  const double *r1 = S.sec + 2, *r2 = S.sec + 2 + N;
  for (int i = tid; i < N; i += nth) {
    const int im = (i + N - 1) % N, ip = (i + 1) % N;
    const double *cs = S.cur + 16 * i, *sn = cs + 4;
    const float *ci = S.ctrl + 8 * i, *cm = S.ctrl + 8 * im, *cp = S.ctrl + 8 * ip;
    // endpoint at theta_i (e1 of the curve before = e0 of this one) and at theta_{i+1}
    const double ge0 = ((double)cm[6] + ci[0]) * cs[0] + ((double)cm[7] + ci[1]) * sn[0];
    const double ge1 = ((double)ci[6] + cp[0]) * cs[3] + ((double)ci[7] + cp[1]) * sn[3];
    const double a0 = r2[im], b0 = r1[i], a1 = r2[i], b1 = r1[ip];
    S.gsec[2 + i] = ci[2] * cs[1] + ci[3] * sn[1] + ge0 * 2.0 * cdl * a0 * a0 / ((a0 + b0) * (a0 + b0));
    S.gsec[2 + N + i] = ci[4] * cs[2] + ci[5] * sn[2] + ge1 * 2.0 * cdl * b1 * b1 / ((a1 + b1) * (a1 + b1));
  }
  if (tid < 2) {
    double s = 0.0;
    for (int i = 0; i < N; ++i) s += (double)S.ctrl[8 * i + tid] + S.ctrl[8 * i + 2 + tid] + S.ctrl[8 * i + 4 + tid] +
                                     S.ctrl[8 * i + 6 + tid];
    S.gsec[tid] = s;
  }
  __syncthreads();
  const float *k0 = G.par + 2 + (size_t)P.k0 * W, *k1 = G.par + 2 + (size_t)P.k1 * W;
  for (int t = tid; t < W; t += nth) {
    const double gs = S.gsec[t];
    if (gs != 0.0) {
      atomicAdd(gout + 2 + (size_t)P.k0 * W + t, (1.0 - P.lam) * gs);
      if (G.K > 1) atomicAdd(gout + 2 + (size_t)P.k1 * W + t, P.lam * gs);
    }
  }
  if (tid == 0) {
    double gs = 0.0;
    if (!P.clamped)
      for (int t = 0; t < W; ++t) gs += S.gsec[t] * (double)(G.K - 1) * ((double)k1[t] - (double)k0[t]);
    const double L = P.z1 - P.z0;
    const double g0 = (double)S.gsl[0] + gs * (P.z - P.z1) / (L * L);
    const double g1 = (double)S.gsl[1] - gs * (P.z - P.z0) / (L * L);
    if (g0 != 0.0) atomicAdd(gout + 0, g0);
    if (g1 != 0.0) atomicAdd(gout + 1, g1);
  }
}

// ------------------------------------------------------------------------------------------------------------
// phi on the nodes (R28): d = max(d2(x, y; section(z)), z0 - z, z - z1), phi = sign * d
// ------------------------------------------------------------------------------------------------------------
// Points of a plane, x fastest: thread t of CTA b owns the offsets 1024 b + t + 256 q.
struct NfGeomPts {
  int i[NF_GEOM_PPT], j[NF_GEOM_PPT];
  bool ok[NF_GEOM_PPT];
};
__device__ __forceinline__ NfGeomPts nf_geom_points(int npx, int npy) {
  NfGeomPts p;
#pragma unroll
  for (int q = 0; q < NF_GEOM_PPT; ++q) {
    const int id = (blockIdx.x * NF_GEOM_PPT + q) * NF_GEOM_NT + threadIdx.x;
    p.j[q] = id / npx;
    p.i[q] = id - p.j[q] * npx;
    p.ok[q] = id < npx * npy;
  }
  return p;
}

__global__ void __launch_bounds__(NF_GEOM_NT) k_geom_sdf(NfGeomK G, int nxn, int nyn, float sign, float *__restrict__ out) {
  extern __shared__ __align__(16) unsigned char nf_geom_raw[];
  const NfGeomSm S = nf_geom_carve(nf_geom_raw, G.N, G.M);
  const NfGeomPlane P = nf_geom_plane(G, (double)blockIdx.z * (double)G.dx);
  nf_geom_setup(G, P, S, false);
  const NfGeomPts pt = nf_geom_points(nxn, nyn);
  float X[NF_GEOM_PPT], Y[NF_GEOM_PPT], d2[NF_GEOM_PPT], tb[NF_GEOM_PPT];
  int kb[NF_GEOM_PPT];
  unsigned inside;
#pragma unroll
  for (int q = 0; q < NF_GEOM_PPT; ++q) { X[q] = (float)pt.i[q] * G.dx; Y[q] = (float)pt.j[q] * G.dx; }
  nf_geom_scan<false>(S.seg, G.N * G.M, X, Y, d2, kb, tb, inside);
#pragma unroll
  for (int q = 0; q < NF_GEOM_PPT; ++q) {
    if (pt.ok[q]) {
      const float sd = ((inside >> q) & 1u) ? -sqrtf(d2[q]) : sqrtf(d2[q]);
      out[((size_t)blockIdx.z * nyn + pt.j[q]) * nxn + pt.i[q]] = sign * fmaxf(sd, P.slab);
    }
  }
}

// dJ/dphi -> dJ/dparams (L141)
__global__ void __launch_bounds__(NF_GEOM_NT) k_geom_sdf_adjoint(NfGeomK G, int nxn, int nyn, float sign,
                                                                 const float *__restrict__ gphi, double *__restrict__ gout) {
  extern __shared__ __align__(16) unsigned char nf_geom_raw[];
  const NfGeomSm S = nf_geom_carve(nf_geom_raw, G.N, G.M);
  const NfGeomPlane P = nf_geom_plane(G, (double)blockIdx.z * (double)G.dx);
  nf_geom_setup(G, P, S, true);
  const int NM = G.N * G.M;
  const NfGeomPts pt = nf_geom_points(nxn, nyn);
  float g[NF_GEOM_PPT];
  bool work = false;
#pragma unroll
  for (int q = 0; q < NF_GEOM_PPT; ++q) {
    g[q] = pt.ok[q] ? sign * gphi[((size_t)blockIdx.z * nyn + pt.j[q]) * nxn + pt.i[q]] : 0.0f;
    work = work || g[q] != 0.0f;
  }
  if (work) {
    S.gsl[2] = 1.0f;
    float X[NF_GEOM_PPT], Y[NF_GEOM_PPT], d2[NF_GEOM_PPT], tb[NF_GEOM_PPT];
    int kb[NF_GEOM_PPT];
    unsigned inside;
#pragma unroll
    for (int q = 0; q < NF_GEOM_PPT; ++q) { X[q] = (float)pt.i[q] * G.dx; Y[q] = (float)pt.j[q] * G.dx; }
    nf_geom_scan<true>(S.seg, NM, X, Y, d2, kb, tb, inside);
#pragma unroll
    for (int q = 0; q < NF_GEOM_PPT; ++q) {
      if (g[q] == 0.0f) continue;
      const float dist = sqrtf(d2[q]);
      const float sgn = ((inside >> q) & 1u) ? -1.0f : 1.0f;
      if (P.slab > sgn * dist) {
        atomicAdd(&S.gsl[P.cap], P.cap == 0 ? g[q] : -g[q]);
      } else if (dist > 0.0f) {
        const float *sg = S.seg + 6 * kb[q];
        const float qx = sg[0] + tb[q] * sg[2], qy = sg[1] + tb[q] * sg[3];
        const float sc = -sgn * g[q] / dist;
        const float gx = sc * (X[q] - qx), gy = sc * (Y[q] - qy);
        const int k1 = kb[q] + 1 == NM ? 0 : kb[q] + 1;
        atomicAdd(&S.gV[2 * kb[q]], (1.0f - tb[q]) * gx);
        atomicAdd(&S.gV[2 * kb[q] + 1], (1.0f - tb[q]) * gy);
        atomicAdd(&S.gV[2 * k1], tb[q] * gx);
        atomicAdd(&S.gV[2 * k1 + 1], tb[q] * gy);
      }
    }
  }
  nf_geom_chain(G, P, S, gout);
}

// ------------------------------------------------------------------------------------------------------------
// U_s on the faces of family C (R30): the closest surface point's velocity along the in-plane normal, caps move in z
// ------------------------------------------------------------------------------------------------------------
// order-preserving float <-> int (for shared-memory atomicMin / atomicMax on coordinates)
__device__ __forceinline__ int nf_f2o(float f) {
  const int i = __float_as_int(f);
  return i ^ ((i >> 31) & 0x7fffffff);
}
__device__ __forceinline__ float nf_o2f(int i) { return __int_as_float(i ^ ((i >> 31) & 0x7fffffff)); }

template <int C, bool ADJ>
__global__ void __launch_bounds__(NF_GEOM_NT) k_geom_velocity(NfGeomK G, int nxf, int nyf, float band,
                                                              float *__restrict__ out, const float *__restrict__ gin,
                                                              double *__restrict__ gout) {
  extern __shared__ __align__(16) unsigned char nf_geom_raw[];
  const NfGeomSm S = nf_geom_carve(nf_geom_raw, G.N, G.M);
  const double z = (C == 2) ? (double)blockIdx.z * (double)G.dx : ((double)blockIdx.z + 0.5) * (double)G.dx;
  const NfGeomPlane P = nf_geom_plane(G, z);
  // Band cull (exact): d = max(d2, slab) >= slab, and d2 >= the distance to the polygon's bounding box; a plane
  // farther than the band from the slab, or a point farther than the band from the box, is not written.
  if (P.slab > band) return;  // (uniform over the CTA; nothing of this plane is within the band)
  nf_geom_setup(G, P, S, ADJ);
  const int NM = G.N * G.M;
  if (threadIdx.x < 4) S.bb[threadIdx.x] = (threadIdx.x & 1) ? nf_f2o(-INFINITY) : nf_f2o(INFINITY);
  __syncthreads();
  for (int v = threadIdx.x; v < NM; v += blockDim.x) {
    atomicMin(&S.bb[0], nf_f2o(S.V[2 * v]));
    atomicMax(&S.bb[1], nf_f2o(S.V[2 * v]));
    atomicMin(&S.bb[2], nf_f2o(S.V[2 * v + 1]));
    atomicMax(&S.bb[3], nf_f2o(S.V[2 * v + 1]));
  }
  __syncthreads();
  const float bx0 = nf_o2f(S.bb[0]) - band, bx1 = nf_o2f(S.bb[1]) + band;
  const float by0 = nf_o2f(S.bb[2]) - band, by1 = nf_o2f(S.bb[3]) + band;
  NfGeomPts pt = nf_geom_points(nxf, nyf);
  float X[NF_GEOM_PPT], Y[NF_GEOM_PPT], g[NF_GEOM_PPT];
  bool work = false;
#pragma unroll
  for (int q = 0; q < NF_GEOM_PPT; ++q) {
    X[q] = (C == 0) ? (float)pt.i[q] * G.dx : ((float)pt.i[q] + 0.5f) * G.dx;
    Y[q] = (C == 1) ? (float)pt.j[q] * G.dx : ((float)pt.j[q] + 0.5f) * G.dx;
    // (written with negations so that band = +inf, where the box is (-inf, +inf), keeps every point)
    pt.ok[q] = pt.ok[q] && !(X[q] < bx0) && !(X[q] > bx1) && !(Y[q] < by0) && !(Y[q] > by1);
    g[q] = (ADJ && pt.ok[q]) ? gin[((size_t)blockIdx.z * nyf + pt.j[q]) * nxf + pt.i[q]] : 0.0f;
    work = work || (ADJ ? g[q] != 0.0f : pt.ok[q]);
  }
  if (work) {
    float d2[NF_GEOM_PPT], tb[NF_GEOM_PPT];
    int kb[NF_GEOM_PPT];
    unsigned inside;
    nf_geom_scan<true>(S.seg, NM, X, Y, d2, kb, tb, inside);
    const float zcap = ADJ ? 0.0f : G.pdot[P.cap];
#pragma unroll
    for (int q = 0; q < NF_GEOM_PPT; ++q) {
      if (!pt.ok[q] || (ADJ && g[q] == 0.0f)) continue;
      const float dist = sqrtf(d2[q]);
      const float sd = ((inside >> q) & 1u) ? -dist : dist;
      if (!(fmaxf(sd, P.slab) <= band)) continue;
      const bool cap = P.slab > sd;
      const float *sg = S.seg + 6 * kb[q];
      const int k1 = kb[q] + 1 == NM ? 0 : kb[q] + 1;
      const float inv = dist > 0.0f ? 1.0f / dist : 0.0f;
      const float nx_ = (X[q] - (sg[0] + tb[q] * sg[2])) * inv, ny_ = (Y[q] - (sg[1] + tb[q] * sg[3])) * inv;
      const float nc = C == 0 ? nx_ : ny_;
      if (!ADJ) {
        float val = 0.0f;
        if (cap) {
          val = C == 2 ? zcap : 0.0f;
        } else if (C < 2) {
          const float qdx = (1.0f - tb[q]) * S.Vd[2 * kb[q]] + tb[q] * S.Vd[2 * k1];
          const float qdy = (1.0f - tb[q]) * S.Vd[2 * kb[q] + 1] + tb[q] * S.Vd[2 * k1 + 1];
          val = (nx_ * qdx + ny_ * qdy) * nc;
        }
        out[((size_t)blockIdx.z * nyf + pt.j[q]) * nxf + pt.i[q]] = val;
      } else {
        if (cap) {
          if (C == 2) { S.gsl[2] = 1.0f; atomicAdd(&S.gsl[P.cap], g[q]); }
        } else if (C < 2) {
          S.gsl[2] = 1.0f;
          const float gx = g[q] * nc * nx_, gy = g[q] * nc * ny_;
          atomicAdd(&S.gV[2 * kb[q]], (1.0f - tb[q]) * gx);
          atomicAdd(&S.gV[2 * kb[q] + 1], (1.0f - tb[q]) * gy);
          atomicAdd(&S.gV[2 * k1], tb[q] * gx);
          atomicAdd(&S.gV[2 * k1 + 1], tb[q] * gy);
        }
      }
    }
  }
  if (ADJ) nf_geom_chain(G, P, S, gout);
}

// ------------------------------------------------------------------------------------------------------------
// CSG on solids, phi > 0 = fluid (R29): union = min, intersection = max; the reverse routes to the operand that won
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_geom_csg(int op, const float *a, const float *b, float *out, size_t n) {
  const size_t nth = (size_t)gridDim.x * blockDim.x;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += nth)
    out[t] = op == NF_CSG_UNION ? fminf(a[t], b[t]) : fmaxf(a[t], b[t]);
}
__global__ void __launch_bounds__(256) k_geom_csg_adjoint(int op, const float *__restrict__ a, const float *__restrict__ b,
                                                          const float *gout, float *ga, float *gb, size_t n) {
  const size_t nth = (size_t)gridDim.x * blockDim.x;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += nth) {
    const bool ta = op == NF_CSG_UNION ? a[t] <= b[t] : a[t] >= b[t];
    const float g = gout[t];
    ga[t] = ta ? g : 0.0f;
    gb[t] = ta ? 0.0f : g;
  }
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
static int geom_check(nf_grid *g, const float *params, int K, int N, int M, const char *who) {
  if (!params || K < 1 || N < 2 || M < 1 || K > NF_GEOM_MAXK || N > NF_GEOM_MAXN || (long long)N * M > NF_GEOM_MAXNM) {
    g->err = std::string(who) + ": need 1 <= K <= 64, 2 <= N <= 64, 1 <= M, N M <= 2048";
    return NF_ERR_INVALID;
  }
  if (!(params[1] > params[0])) {
    g->err = std::string(who) + ": need z1 > z0";
    return NF_ERR_INVALID;
  }
  const int W = 2 + 2 * N;
  for (int k = 0; k < K; ++k)
    for (int t = 2; t < W; ++t)
      if (!(params[2 + k * W + t] > 0.0f)) {
        g->err = std::string(who) + ": control radii must be positive";
        return NF_ERR_INVALID;
      }
  return NF_OK;
}

static int geom_upload(nf_grid *g, const float *params, const float *pdot, int K, int N, NfGeomK *G, int M) {
  const size_t P = 2 + (size_t)K * (2 + 2 * N);
  // (pageable source: the copy is staged before the call returns, so the caller's array may change afterwards)
  NF_CUDA(g, cudaMemcpyAsync(g->geom_par, params, P * sizeof(float), cudaMemcpyHostToDevice, g->stream));
  if (pdot) NF_CUDA(g, cudaMemcpyAsync(g->geom_par + NF_GEOM_MAXP, pdot, P * sizeof(float), cudaMemcpyHostToDevice, g->stream));
  G->par = g->geom_par;
  G->pdot = pdot ? g->geom_par + NF_GEOM_MAXP : nullptr;
  G->K = K; G->N = N; G->M = M; G->dx = g->dx;
  return NF_OK;
}

template <typename Kern>
static int geom_smem(nf_grid *g, Kern kern, int N, int M, size_t *bytes) {
  *bytes = nf_geom_smem_bytes(N, M);
  if (*bytes > 48 * 1024) NF_CUDA(g, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*bytes));
  return NF_OK;
}

static dim3 geom_grid(int npx, int npy, int npz) {
  const long long per = (long long)NF_GEOM_NT * NF_GEOM_PPT;
  return dim3((unsigned)(((long long)npx * npy + per - 1) / per), 1, npz);
}

static int geom_download(nf_grid *g, int K, int N, double *gout_host) {
  const size_t P = 2 + (size_t)K * (2 + 2 * N);
  NF_CUDA(g, cudaMemcpyAsync(gout_host, g->geom_grad, P * sizeof(double), cudaMemcpyDeviceToHost, g->stream));
  NF_CUDA(g, cudaStreamSynchronize(g->stream));
  return NF_OK;
}

int nf_geom_sdf_impl(nf_grid *g, const float *params, int K, int N, int M, int flags, float *sdf_nodes) {
  NF_TRY(geom_check(g, params, K, N, M, "nf_geom_sdf"));
  NfGeomK G;
  NF_TRY(geom_upload(g, params, nullptr, K, N, &G, M));
  size_t sm;
  NF_TRY(geom_smem(g, k_geom_sdf, N, M, &sm));
  const dim3 block(NF_GEOM_NT);
  NF_LAUNCH(g, NFK_GEOM, k_geom_sdf<<<geom_grid(g->nx + 1, g->ny + 1, g->nz + 1), block, sm, g->stream>>>(
                             G, g->nx + 1, g->ny + 1, (flags & NF_GEOM_COMPLEMENT) ? -1.0f : 1.0f, sdf_nodes));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_geom_sdf_adjoint_impl(nf_grid *g, const float *params, int K, int N, int M, int flags, const float *gsdf_nodes,
                             double *gparams_host) {
  NF_TRY(geom_check(g, params, K, N, M, "nf_geom_sdf_adjoint"));
  NfGeomK G;
  NF_TRY(geom_upload(g, params, nullptr, K, N, &G, M));
  size_t sm;
  NF_TRY(geom_smem(g, k_geom_sdf_adjoint, N, M, &sm));
  NF_CUDA(g, cudaMemsetAsync(g->geom_grad, 0, NF_GEOM_MAXP * sizeof(double), g->stream));
  const dim3 block(NF_GEOM_NT);
  NF_LAUNCH(g, NFK_GEOM, k_geom_sdf_adjoint<<<geom_grid(g->nx + 1, g->ny + 1, g->nz + 1), block, sm, g->stream>>>(
                             G, g->nx + 1, g->ny + 1, (flags & NF_GEOM_COMPLEMENT) ? -1.0f : 1.0f, gsdf_nodes, g->geom_grad));
  NF_CUDA(g, cudaGetLastError());
  return geom_download(g, K, N, gparams_host);
}

template <bool ADJ>
static int geom_velocity_launch(nf_grid *g, const NfGeomK &G, float band, float *us, float *vs, float *ws,
                                const float *gus, const float *gvs, const float *gws) {
  size_t sm;
  NF_TRY(geom_smem(g, k_geom_velocity<0, ADJ>, G.N, G.M, &sm));
  NF_TRY(geom_smem(g, k_geom_velocity<1, ADJ>, G.N, G.M, &sm));
  NF_TRY(geom_smem(g, k_geom_velocity<2, ADJ>, G.N, G.M, &sm));
  const dim3 block(NF_GEOM_NT);
  const int nx = g->nx, ny = g->ny, nz = g->nz;
  if (ADJ ? gus != nullptr : us != nullptr)
    NF_LAUNCH(g, NFK_GEOM, k_geom_velocity<0, ADJ><<<geom_grid(nx + 1, ny, nz), block, sm, g->stream>>>(
                               G, nx + 1, ny, band, us, gus, g->geom_grad));
  if (ADJ ? gvs != nullptr : vs != nullptr)
    NF_LAUNCH(g, NFK_GEOM, k_geom_velocity<1, ADJ><<<geom_grid(nx, ny + 1, nz), block, sm, g->stream>>>(
                               G, nx, ny + 1, band, vs, gvs, g->geom_grad));
  if (ADJ ? gws != nullptr : ws != nullptr)
    NF_LAUNCH(g, NFK_GEOM, k_geom_velocity<2, ADJ><<<geom_grid(nx, ny, nz + 1), block, sm, g->stream>>>(
                               G, nx, ny, band, ws, gws, g->geom_grad));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_geom_velocity_impl(nf_grid *g, const float *params, const float *pdot, int K, int N, int M, float band,
                          float *us, float *vs, float *ws) {
  NF_TRY(geom_check(g, params, K, N, M, "nf_geom_velocity"));
  NfGeomK G;
  NF_TRY(geom_upload(g, params, pdot, K, N, &G, M));
  return geom_velocity_launch<false>(g, G, band, us, vs, ws, nullptr, nullptr, nullptr);
}

int nf_geom_velocity_adjoint_impl(nf_grid *g, const float *params, int K, int N, int M, float band, const float *gus,
                                  const float *gvs, const float *gws, double *gpdot_host) {
  NF_TRY(geom_check(g, params, K, N, M, "nf_geom_velocity_adjoint"));
  NfGeomK G;
  NF_TRY(geom_upload(g, params, nullptr, K, N, &G, M));
  NF_CUDA(g, cudaMemsetAsync(g->geom_grad, 0, NF_GEOM_MAXP * sizeof(double), g->stream));
  NF_TRY(geom_velocity_launch<true>(g, G, band, nullptr, nullptr, nullptr, gus, gvs, gws));
  return geom_download(g, K, N, gpdot_host);
}

int nf_geom_csg_impl(nf_grid *g, int op, const float *a, const float *b, float *out) {
  NF_LAUNCH(g, NFK_GEOM, k_geom_csg<<<148 * 8, 256, 0, g->stream>>>(op, a, b, out, nf_nn(g)));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}

int nf_geom_csg_adjoint_impl(nf_grid *g, int op, const float *a, const float *b, const float *gout, float *ga, float *gb) {
  NF_LAUNCH(g, NFK_GEOM, k_geom_csg_adjoint<<<148 * 8, 256, 0, g->stream>>>(op, a, b, gout, ga, gb, nf_nn(g)));
  NF_CUDA(g, cudaGetLastError());
  return NF_OK;
}
