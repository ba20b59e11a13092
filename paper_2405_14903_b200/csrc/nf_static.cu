// nf_static.cu -- nf_max_speed_static: the CFL reduction of nf_max_speed (R24) for callers that
// must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// It needs no nf_grid handle (creating one allocates) and calls no cudaMalloc / cudaFree / allocating library routine:
// the scratch of the two-stage reduction -- one partial maximum per segment of NF_STATIC_SEG faces -- lives in a
// file-scope __device__ array of NF_STATIC_MAX_PARTIALS floats (64 KB; every GPU that loads the library holds it until
// the process exits).  Sizes whose partials would not fit are rejected (NF_ERR_INVALID, nf_static_last_error says why).
//
// The array's name is a host-side stand-in in host code, not a device address: its address is taken ONCE PER DEVICE,
// with that device current, by cudaGetSymbolAddress (static_scratch below) and passed to the kernels.
//
// Every call, from every thread and stream, shares the one array per device, and the array keeps the last call's
// contents.  Nothing in it has to start at zero: stage 1 writes exactly the partials that stage 2 of the same call reads
// (stale partials beyond them are never read).  Two calls that OVERLAP on the GPU (different streams, or graphs
// replayed concurrently) race on it; calls on one stream are ordered and safe.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "nf.h"

#define NF_STATIC_SEG 16384            // faces per CTA of stage 1 (256 threads x 64 faces)
#define NF_STATIC_MAX_PARTIALS 16384   // floats of scratch: 64 KB; u + v + w faces <= ~2.68e8 (cubes up to ~440^3)
#define NF_STATIC_MAX_DEVICES 64

static __device__ __align__(256) float nf_static_scratch[NF_STATIC_MAX_PARTIALS];

static thread_local char t_err[256] = "";

// max of |v|, a NaN propagating (the rule of k_max_abs, nf_advect.cu)
__device__ __forceinline__ float nf_static_absmax(float m, float v) { return (v > m || v != v) ? v : m; }

// stage 1: CTA b reduces the faces [b SEG, (b+1) SEG) of its component to part[b]
__global__ void __launch_bounds__(256) k_max_abs_partials(const float *__restrict__ u, const float *__restrict__ v,
                                                          const float *__restrict__ w, unsigned long long nu,
                                                          unsigned long long nv, unsigned long long nw, unsigned bu,
                                                          unsigned bv, float *__restrict__ part) {
  const unsigned b = blockIdx.x;
  const float *f;
  unsigned long long n, first;
  if (b < bu) { f = u; n = nu; first = (unsigned long long)b * NF_STATIC_SEG; }
  else if (b < bu + bv) { f = v; n = nv; first = (unsigned long long)(b - bu) * NF_STATIC_SEG; }
  else { f = w; n = nw; first = (unsigned long long)(b - bu - bv) * NF_STATIC_SEG; }
  const unsigned long long last = first + NF_STATIC_SEG < n ? first + NF_STATIC_SEG : n;
  float m = 0.0f;
  for (unsigned long long t = first + threadIdx.x; t < last; t += 256) m = nf_static_absmax(m, fabsf(f[t]));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = nf_static_absmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  __shared__ float s[8];
  if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < 8; ++i) m = nf_static_absmax(m, s[i]);
    part[b] = m;
  }
}
// stage 2: one CTA reduces the nb partials of THIS call into the caller's output
__global__ void __launch_bounds__(1024) k_max_abs_final(const float *__restrict__ part, unsigned nb,
                                                        float *__restrict__ out) {
  float m = 0.0f;
  for (unsigned t = threadIdx.x; t < nb; t += 1024) m = nf_static_absmax(m, part[t]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = nf_static_absmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  __shared__ float s[32];
  if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < 32; ++i) m = nf_static_absmax(m, s[i]);
    *out = m;
  }
}

// Device address of the scratch array on the CURRENT device: resolved once per device, cached.
static int static_scratch(float **ptr) {
  static std::mutex mu;
  static float *addr[NF_STATIC_MAX_DEVICES] = {nullptr};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= NF_STATIC_MAX_DEVICES) {
    snprintf(t_err, sizeof(t_err), "nf_max_speed_static: cudaGetDevice failed or device index %d out of range (%s)", dev,
             cudaGetErrorString(e));
    return NF_ERR_CUDA;
  }
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    float *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, nf_static_scratch);
    if (e != cudaSuccess || !p) {
      snprintf(t_err, sizeof(t_err), "nf_max_speed_static: cudaGetSymbolAddress failed on device %d: %s", dev,
               cudaGetErrorString(e));
      return NF_ERR_CUDA;
    }
    addr[dev] = p;
  }
  *ptr = addr[dev];
  return NF_OK;
}

extern "C" const char *nf_static_last_error(void) { return t_err; }

extern "C" int nf_max_speed_static(const float *u, const float *v, const float *w, int nx, int ny, int nz,
                                   void *cuda_stream, float *max_abs_dev) {
  t_err[0] = 0;
  if (!u || !v || !w || !max_abs_dev || nx < 1 || ny < 1 || nz < 1) {
    snprintf(t_err, sizeof(t_err), "nf_max_speed_static: NULL pointer or non-positive extent");
    return NF_ERR_INVALID;
  }
  const unsigned long long nu = (unsigned long long)(nx + 1) * ny * nz, nv = (unsigned long long)nx * (ny + 1) * nz,
                           nw = (unsigned long long)nx * ny * (nz + 1);
  const unsigned long long bu = (nu + NF_STATIC_SEG - 1) / NF_STATIC_SEG, bv = (nv + NF_STATIC_SEG - 1) / NF_STATIC_SEG,
                           bw = (nw + NF_STATIC_SEG - 1) / NF_STATIC_SEG;
  if (bu + bv + bw > NF_STATIC_MAX_PARTIALS) {
    snprintf(t_err, sizeof(t_err),
             "nf_max_speed_static: %d x %d x %d needs %llu partial maxima, the static scratch holds %d (u + v + w faces "
             "<= %llu); use nf_max_speed",
             nx, ny, nz, bu + bv + bw, NF_STATIC_MAX_PARTIALS, (unsigned long long)NF_STATIC_MAX_PARTIALS * NF_STATIC_SEG);
    return NF_ERR_INVALID;
  }
  float *part = nullptr;
  const int rc = static_scratch(&part);
  if (rc != NF_OK) return rc;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const unsigned nb = (unsigned)(bu + bv + bw);
  k_max_abs_partials<<<nb, 256, 0, s>>>(u, v, w, nu, nv, nw, (unsigned)bu, (unsigned)bv, part);
  k_max_abs_final<<<1, 1024, 0, s>>>(part, nb, max_abs_dev);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(t_err, sizeof(t_err), "nf_max_speed_static: launch failed: %s", cudaGetErrorString(e));
    return NF_ERR_CUDA;
  }
  return NF_OK;
}
