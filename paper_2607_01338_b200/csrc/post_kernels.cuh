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

// z ~ N(0,1) per voxel (reading S10): one Philox4x32-10(key, counter = voxel / 4) call serves four
// consecutive voxels; words (r0, r1) the voxels 4c, 4c+1, words (r2, r3) the voxels 4c+2, 4c+3; a word pair gives
// u1, u2 and the two Box-Muller deviates sqrt(-2 ln u1) cos(2 pi u2) (even voxel), sqrt(-2 ln u1) sin(2 pi u2) (odd).
// The uniforms use the top 24 bits: k + 1/2 is exact in fp32 for k < 2^23 only; above, it rounds to k or k + 1.  For the
// radius that matters where u1 is close to 1 (ln u1 = -(1 - u1): a rounding of 2^-25 in u1 is an absolute error of 3e-8 in
// ln u1, i.e. 1e-5 in a deviate of 1e-3, and u1 = 1 - 2^-25 rounds to 1, R = 0), so the known residual
// (k + 1/2) - fl(k + 1/2) in {0, +-1/2} is put back to first order: ln u1 = ln(u~) + (u1 - u~) / u~ (the next term is 1e-15).
// For the angle the rounding of u2 moves a deviate by 2e-7 R.
__device__ __forceinline__ void box_muller_pair(uint32_t ra, uint32_t rb, float& z_even, float& z_odd) {
  const float kf = (float)(ra >> 8);                      // exact
  const float t = kf + 0.5f;                              // rounded above 2^23
  const float resid = (kf - t) + 0.5f;                    // exact: 0 below 2^23, +-1/2 above
  const float u1 = t * (1.0f / 16777216.0f);
  const float ln_u1 = fmaf(resid * (1.0f / 16777216.0f), rcp_approx(u1), logf(u1));
  const float u2 = ((float)(rb >> 8) + 0.5f) * (1.0f / 16777216.0f);
  float R;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(R) : "f"(-2.0f * ln_u1));      // 2^-22 relative
  // MUFU.SIN / COS: absolute error 2^-21.4 on [0, 2 pi), plus 4e-7 for the rounding of the angle: <= 1e-6 R in a deviate
  float sn, cs;
  __sincosf(6.283185307179586f * u2, &sn, &cs);
  z_even = R * cs;
  z_odd = R * sn;
}

// the deviates of the voxel pair (idx, idx + 1), idx even
__device__ __forceinline__ void voxel_normal_pair(const NoiseConsts& nc, uint64_t idx, float& z0, float& z1) {
  uint32_t r[4];
  const uint64_t c = idx >> 2;
  philox4x32_10(nc.k0, nc.k1, (uint32_t)c, (uint32_t)(c >> 32), 0u, 0u, r);
  const bool hi = (idx >> 1) & 1;
  box_muller_pair(hi ? r[2] : r[0], hi ? r[3] : r[1], z0, z1);
}

__device__ __forceinline__ float voxel_normal(const NoiseConsts& nc, uint64_t idx) {
  float z0, z1;
  voxel_normal_pair(nc, idx & ~1ull, z0, z1);
  return (idx & 1) ? z1 : z0;
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

// Register formulation of the same pass (even nv, R <= 16): a thread owns a PAIR of channels and TA consecutive
// positions along a; it streams the TA + 2 RB input rows once (8-byte loads, a warp reads 256 contiguous bytes per
// row) and scatters each row into the TA packed accumulators it contributes to (fma.rn.f32x2), so every loaded
// value feeds up to 2 RB + 1 outputs of the same thread and no shared memory is involved: 2 RB + 1 packed FMAs + 2
// loads + 1 store per pair of outputs, against 13 LDS + 13 FFMA + addressing per single output of the tiled kernel.
// RB is the compile-time radius class (taps beyond the configured radius are zero).
template <int RB>
struct BeamTaps { float w[2 * RB + 1]; };

template <int RB, int TA>
__global__ void __launch_bounds__(128)
beam_pass_reg_kernel(BeamTaps<RB> taps, NoiseConsts nc, const float* __restrict__ in, float* __restrict__ out, int na,
                     int nb, int nv, int64_t stride_a, int64_t stride_b) {
  const int vp = blockIdx.x * 32 + threadIdx.x;            // channel pair
  const int a0 = (blockIdx.y * blockDim.y + threadIdx.y) * TA;
  const int b = blockIdx.z;
  if (2 * vp >= nv || a0 >= na) return;
  const int64_t base = (int64_t)b * stride_b + 2 * vp;
  unsigned long long acc[TA];
#pragma unroll
  for (int i = 0; i < TA; ++i) acc[i] = 0ull;
#pragma unroll
  for (int r = 0; r < TA + 2 * RB; ++r) {
    const int a = a0 - RB + r;
    float2 v = make_float2(0.0f, 0.0f);
    if (a >= 0 && a < na) v = *reinterpret_cast<const float2*>(in + base + (int64_t)a * stride_a);
    unsigned long long vv;
    asm("mov.b64 %0, {%1, %2};" : "=l"(vv) : "f"(v.x), "f"(v.y));
#pragma unroll
    for (int i = 0; i < TA; ++i) {
      const int k = r - i;                                  // tap index of input row r for output i
      if (k >= 0 && k <= 2 * RB) {
        unsigned long long ww;
        asm("mov.b64 %0, {%1, %1};" : "=l"(ww) : "f"(taps.w[k]));
        asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[i]) : "l"(ww), "l"(vv));
      }
    }
  }
#pragma unroll
  for (int i = 0; i < TA; ++i) {
    const int a = a0 + i;
    if (a < na) {
      float2 o;
      asm("mov.b64 {%0, %1}, %2;" : "=f"(o.x), "=f"(o.y) : "l"(acc[i]));
      const int64_t idx = base + (int64_t)a * stride_a;
      if (nc.on) {                 // idx is even: the two channels of the thread share one Box-Muller pair
        float z0, z1;
        voxel_normal_pair(nc, (uint64_t)idx, z0, z1);
        o.x += fmaf(nc.sigma, z0, nc.mu);
        o.y += fmaf(nc.sigma, z1, nc.mu);
      }
      *reinterpret_cast<float2*>(out + idx) = o;
    }
  }
}

template <int RB>
inline void launch_beam_pass_reg(const BeamConsts& bc, const NoiseConsts& nc, const float* in, float* out, int na, int nb,
                                 int nv, int64_t stride_a, int64_t stride_b, cudaStream_t st) {
  constexpr int TA = 16;
  BeamTaps<RB> taps;
  for (int k = 0; k <= 2 * RB; ++k) {
    const int d = k - (RB - bc.R);
    taps.w[k] = (d >= 0 && d <= 2 * bc.R) ? bc.g[d] : 0.0f;
  }
  const int tiles = (na + TA - 1) / TA;
  dim3 block(32, 4), grid((nv / 2 + 31) / 32, (tiles + 3) / 4, nb);
  beam_pass_reg_kernel<RB, TA><<<grid, block, 0, st>>>(taps, nc, in, out, na, nb, nv, stride_a, stride_b);
}

// One pass with the best kernel for (R, nv): register formulation when nv is even and R <= 16, tiled otherwise.
inline void launch_beam_pass(const BeamConsts& bc, const NoiseConsts& nc, const float* in, float* out, int na, int nb,
                             int nv, int64_t stride_a, int64_t stride_b, cudaStream_t st) {
  const bool aligned = (nv % 2 == 0) && ((reinterpret_cast<uintptr_t>(in) | reinterpret_cast<uintptr_t>(out)) % 8 == 0);
  if (aligned && bc.R <= 4) return launch_beam_pass_reg<4>(bc, nc, in, out, na, nb, nv, stride_a, stride_b, st);
  if (aligned && bc.R <= 8) return launch_beam_pass_reg<8>(bc, nc, in, out, na, nb, nv, stride_a, stride_b, st);
  if (aligned && bc.R <= 16) return launch_beam_pass_reg<16>(bc, nc, in, out, na, nb, nv, stride_a, stride_b, st);
  dim3 block(32, 8), grid((nv + 31) / 32, (na + kBeamTA - 1) / kBeamTA, nb);
  beam_pass_kernel<<<grid, block, 0, st>>>(bc, nc, in, out, na, nb, nv, stride_a, stride_b);
}

// K7 alone (no beam configured): in-place, four consecutive voxels (one Philox call) per thread.
__global__ void __launch_bounds__(256) noise_kernel(NoiseConsts nc, float* __restrict__ cube, int64_t nvox) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t i0 = 4 * c;
  if (i0 >= nvox) return;
  uint32_t r[4];
  philox4x32_10(nc.k0, nc.k1, (uint32_t)c, (uint32_t)((uint64_t)c >> 32), 0u, 0u, r);
  float z[4];
  box_muller_pair(r[0], r[1], z[0], z[1]);
  box_muller_pair(r[2], r[3], z[2], z[3]);
#pragma unroll
  for (int k = 0; k < 4; ++k)
    if (i0 + k < nvox) cube[i0 + k] += fmaf(nc.sigma, z[k], nc.mu);
}

}  // namespace iris
