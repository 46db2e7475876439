// Diagnostics of PAPER.md section 5: density tracing ("simple observation", section 5.10) and the error metrics of
// section 5.1 (TSRE, mean-TSRE over the cube and over its l-b and l-v images, TAM).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace iris {

// Density tracing: every cell adds its column density n_H2 h to the channel that contains its line-of-sight velocity,
// divided by the channel width (reading S28).  One thread per pixel marches its column (lanes along x:
// coalesced field reads) and adds into its own spectrum, which must be zero on entry.  The channel decision is taken
// in double, with the expression the definition uses, so that it cannot differ from a float64 evaluation.
__global__ void __launch_bounds__(128)
density_trace_kernel(const float* __restrict__ nH2, const float* __restrict__ vlos, int npix, int nz, int nv, double v0,
                     double dv, float scale /* h / dv */, float* __restrict__ cube) {
  const int pix = blockIdx.x * blockDim.x + threadIdx.x;
  if (pix >= npix) return;
  float* row = cube + (int64_t)pix * nv;
  for (int k = 0; k < nz; ++k) {
    const int64_t cell = (int64_t)k * npix + pix;
    const double fl = floor(((double)vlos[cell] - v0) / dv + 0.5);
    if (fl < 0.0 || fl >= (double)nv) continue;
    row[(int)fl] += nH2[cell] * scale;
  }
}

// ---- metrics.  acc[0..8] (double, zero on entry except the maxima = -inf):
//   0 sum TSRE over voxels, 1 sum TSRE over l-b pixels, 2 sum TSRE over l-v pixels, 3 sum T1 active, 4 sum T2 active,
//   5 max T1, 6 max T2, 7 active(T1), 8 active(T2)
__device__ __forceinline__ double tsre_of(double a, double b, double Tmin) {
  const double fa = fabs(a), fb = fabs(b);
  return (fa > Tmin && fb > Tmin) ? 2.0 * fabs(a - b) / (fa + fb) : 0.0;
}

__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__device__ __forceinline__ void atomic_max_double(double* addr, double v) {
  unsigned long long* a = reinterpret_cast<unsigned long long*>(addr);
  unsigned long long old = *a;
  while (__longlong_as_double((long long)old) < v) {
    const unsigned long long seen = atomicCAS(a, old, (unsigned long long)__double_as_longlong(v));
    if (seen == old) break;
    old = seen;
  }
}

// voxel-wise part (Eq. 5.1.1 - 5.1.2, 5.1.4 - 5.1.5) and, per pixel, the l-b image part: one warp per pixel
__global__ void __launch_bounds__(256)
metrics_pixel_kernel(const float* __restrict__ T1, const float* __restrict__ T2, int npix, int nv, double Tmin,
                     double* __restrict__ acc) {
  const int lane = threadIdx.x & 31;
  const int pix = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (pix >= npix) return;
  const float* a = T1 + (int64_t)pix * nv;
  const float* b = T2 + (int64_t)pix * nv;
  double s = 0.0, s1 = 0.0, s2 = 0.0, n1 = 0.0, n2 = 0.0, m1 = -INFINITY, m2 = -INFINITY, sa = 0.0, sb = 0.0;
  for (int v = lane; v < nv; v += 32) {
    const double x = (double)a[v], y = (double)b[v];
    s += tsre_of(x, y, Tmin);
    if (fabs(x) > Tmin) { s1 += x; n1 += 1.0; }
    if (fabs(y) > Tmin) { s2 += y; n2 += 1.0; }
    m1 = fmax(m1, x); m2 = fmax(m2, y);
    sa += x; sb += y;
  }
  s = warp_sum_d(s); s1 = warp_sum_d(s1); s2 = warp_sum_d(s2); n1 = warp_sum_d(n1); n2 = warp_sum_d(n2);
  sa = warp_sum_d(sa); sb = warp_sum_d(sb);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    m1 = fmax(m1, __shfl_xor_sync(0xffffffffu, m1, o));
    m2 = fmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
  }
  if (lane == 0) {
    atomicAdd(acc + 0, s);
    atomicAdd(acc + 1, tsre_of(sa / nv, sb / nv, Tmin));
    atomicAdd(acc + 3, s1); atomicAdd(acc + 4, s2);
    atomicAdd(acc + 7, n1); atomicAdd(acc + 8, n2);
    atomic_max_double(acc + 5, m1); atomic_max_double(acc + 6, m2);
  }
}

// l-v image part (Eq. 5.1.3): one thread per (x, v), mean over y (lanes along v: coalesced)
__global__ void __launch_bounds__(256)
metrics_lv_kernel(const float* __restrict__ T1, const float* __restrict__ T2, int ny, int nx, int nv, double Tmin,
                  double* __restrict__ acc) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double r = 0.0;
  if (t < (int64_t)nx * nv) {
    double sa = 0.0, sb = 0.0;
    for (int y = 0; y < ny; ++y) {
      sa += (double)T1[(int64_t)y * nx * nv + t];
      sb += (double)T2[(int64_t)y * nx * nv + t];
    }
    r = tsre_of(sa / ny, sb / ny, Tmin);
  }
  r = warp_sum_d(r);
  if ((threadIdx.x & 31) == 0 && r != 0.0) atomicAdd(acc + 2, r);
}

}  // namespace iris
