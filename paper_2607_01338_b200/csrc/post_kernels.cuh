// K6 (separable Gaussian beam) and K7 (seeded noise, Eq. 4.12.1).
#pragma once
#include "iris_math.cuh"

namespace iris {

constexpr int kMaxBeamRadius = 32;

struct BeamConsts {
  int R;                              // radius ceil(4 sigma)
  float g[2 * kMaxBeamRadius + 1];    // 1-D weights, sum 1
};

struct NoiseConsts {
  uint32_t k0, k1;     // Philox key = seed
  float mu, sigma;     // already multiplied by gamma
  int on;
};

// z ~ N(0,1) of voxel `idx`: Box-Muller on the first two words of Philox4x32-10(key, counter = idx).
// The uniforms use the top 24 bits, so they are exact in fp32 and identical to the float64 definition.
__device__ __forceinline__ float voxel_normal(const NoiseConsts& nc, uint64_t idx) {
  uint32_t r[4];
  philox4x32_10(nc.k0, nc.k1, (uint32_t)idx, (uint32_t)(idx >> 32), 0u, 0u, r);
  const float u1 = ((float)(r[0] >> 8) + 0.5f) * (1.0f / 16777216.0f);
  const float u2 = ((float)(r[1] >> 8) + 0.5f) * (1.0f / 16777216.0f);
  return sqrtf(-2.0f * logf(u1)) * cospif(2.0f * u2);
}

// One 1-D pass of the beam along a spatial axis "a" of a cube laid out with the channel fastest.
//   out[a, b, v] = sum_d g[d] in[a + d, b, v],  zero outside [0, na)
// A CTA owns TA consecutive positions along a, one b, 32 consecutive channels; the (TA + 2R) x 32 input
// tile is staged once in shared memory (each input element is read from L2/HBM (TA+2R)/TA times).
// Lanes run along v, so global accesses are 128-byte coalesced and shared accesses conflict-free.
// If nc.on, the noise of K7 is added in the same pass (epilogue of the second pass).
constexpr int kBeamTA = 32;

__global__ void __launch_bounds__(256)
beam_pass_kernel(BeamConsts bc, NoiseConsts nc, const float* __restrict__ in, float* __restrict__ out, int na, int nb,
                 int nv, int64_t stride_a, int64_t stride_b) {
  __shared__ float tile[kBeamTA + 2 * kMaxBeamRadius][32];
  const int lane = threadIdx.x, w = threadIdx.y;          // 32 x 8
  const int v = blockIdx.x * 32 + lane;
  const int a0 = blockIdx.y * kBeamTA;
  const int b = blockIdx.z;
  const int R = bc.R;
  const int64_t base = (int64_t)b * stride_b + v;
  for (int r = w; r < kBeamTA + 2 * R; r += 8) {
    const int a = a0 - R + r;
    float val = 0.0f;
    if (v < nv && a >= 0 && a < na) val = in[base + (int64_t)a * stride_a];
    tile[r][lane] = val;
  }
  __syncthreads();
  if (v >= nv) return;
  for (int i = w; i < kBeamTA; i += 8) {
    const int a = a0 + i;
    if (a >= na) break;
    float acc = 0.0f;
    for (int d = 0; d <= 2 * R; ++d) acc = fmaf(bc.g[d], tile[i + d][lane], acc);
    const int64_t idx = base + (int64_t)a * stride_a;
    if (nc.on) acc += fmaf(nc.sigma, voxel_normal(nc, (uint64_t)idx), nc.mu);
    out[idx] = acc;
  }
}

// K7 alone (no beam configured): in-place.
__global__ void __launch_bounds__(256) noise_kernel(NoiseConsts nc, float* __restrict__ cube, int64_t nvox) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nvox) return;
  cube[i] += fmaf(nc.sigma, voxel_normal(nc, (uint64_t)i), nc.mu);
}

}  // namespace iris
