// K3 (line-window formulation, narrow channels) as a FLAT SEGMENT STREAM: the production LOS transfer kernel.
//
// Same recurrence, the same line window and the same arithmetic per (cell, channel) update as transfer_series.cuh
// (difference form D = I^[T] - I^[C], Dt = D * exp(sum tau_d), profile from the channel centre, base-2 units, packed
// f32x2 updates of channel pairs); what changes is how the updates are handed to the lanes.  The series kernel gives
// the 8 lanes of a pixel one cell at a time: a window of 17 - 21 channel pairs costs 3 passes of 8 pairs, a third of
// the lanes idle, and every lane repeats the per-cell set-up.  Here
//
// 1. the window of every (cell, pixel) is cut into SEGMENTS of 4 consecutive channel pairs (8 channels), and the
//    segments of the warp's 4 pixels, cell after cell, form one stream; a PASS hands 32 consecutive segments of the
//    stream to the 32 lanes, whatever cells they belong to.  Only the last segment of a window can be partly outside it
//    (its channels lie beyond |x| = X_w, where the update is below the window threshold anyway): 92 % of the lane-slots
//    do algorithmic work on the BASELINE cubes, against 65 - 75 %.
// 2. Everything that depends on the cell only is worked out ONCE per (cell, pixel) in phase A, including the factors
//    that depend on the march so far: the continuum C before the cell and the accumulated dust attenuation G are
//    prefix "sums" along the 8 cells of a chunk (an affine scan and a product scan over the lanes), so a record holds
//    the final operands of the update and phase B has no per-cell prologue at all.
// 3. A lane fetches the record of its segment (a gather of four LDS.128) and computes, for its 4 pairs, the update as
//    an affine map  Dt' = alpha Dt + beta  WITHOUT touching the spectrum: (alpha, beta) do not depend on Dt, so all
//    segments of a pass are computed at once although several of them (consecutive cells of one pixel) act on the
//    same channels.  The maps are then applied to the spectrum in shared memory in cell order: one short step per
//    cell row present in the pass (about three), each a predicated LDS.64 / FFMA2 / STS.64 per pair.
// 4. Four independent pairs per lane give the dependent MUFU -> FMA chains of the update the instruction-level
//    parallelism that the resident warps alone (the spectra of 4 pixels per warp fill the shared memory) do not.
//
// Stream bookkeeping.  Segments are numbered along the whole march (spos .. send are pending).  owner[] (a ring of
// bytes) maps a segment to the slot of its record; records live in a ring of 64 slots (at most 31 pending + 32 new
// ones).  A chunk whose segments do not fit the ring is published in batches.  Pending segments (< 32) are carried into
// the next chunk, so only the very last pass of a pixel column is partly filled.
//
// Dust attenuation can take G = exp(sum tau_d) out of the fp32 range: a chunk with a cell of tau_d > kFlatSlowTau is
// marched one cell row at a time, and whenever G passes kFoldG the pending segments are flushed and G is folded back
// into the stored spectra (transfer_common.cuh).
#pragma once
#include "transfer_common.cuh"
#include "transfer_window.cuh"
#include "transfer_series.cuh"      // packed f32x2 helpers, kSeriesMaxS / kSeriesDeg3MaxS

namespace iris {

constexpr int kFlatPPW = 4;              // pixels per warp
constexpr int kFlatRows = 32 / kFlatPPW; // cell rows per chunk: one record per lane
constexpr int kFlatSeg = 4;              // channel pairs per segment
constexpr int kFlatRecSlots = 64;        // record ring
constexpr int kFlatRecBytes = 4 * kFlatRecSlots * (int)sizeof(float4);
constexpr float kFlatSlowTau = 7.0f;     // 8 cells of tau_d <= 7 on top of G <= kFoldG stay inside the fp32 range

// pairs of a spectrum incl. padding: the last segment of a window may reach 3 pairs beyond it
__host__ __device__ inline int flat_padded_pairs(int npts) { return (((npts + 1) / 2 + (kFlatSeg - 1)) + 3) / 4 * 4; }
// owner ring: a power of two that holds 32 pending segments, the largest single window and some slack
__host__ __device__ inline int flat_ring_size(int npts) {
  const int need = 64 + ((npts + 1) / 2 + kFlatSeg - 1) / kFlatSeg + 1;
  int r = 256;
  while (r < need) r <<= 1;
  return r;
}
inline size_t flat_smem_per_warp(int npts) {
  return (size_t)kFlatRecBytes + (size_t)flat_ring_size(npts) + (size_t)kFlatPPW * flat_padded_pairs(npts) * sizeof(float2);
}

// Record of one (cell, pixel), 4 float4 in the ring (field-major: rec[f * 64 + slot]):
//   f0 = { x0, xs, bits(qlo | nq << 16), bits(segstart & 0xffff | g << 16 | (row & 0x3fff) << 18) }   row: running
//        count of the cell rows that have segments (consecutive rows of a pass differ by one: at most 32 apply steps)
//   f1 = { pA0, pA1, pA2, pA3 }                          polA(u') = As' pol(u') (see transfer_series.cuh)
//   f2 = { Pn, -Qn, -Rn, C G }   (dust)                  operands of the update, already scaled by G' = G exp(tau_d)
//        { C - S_L, -, -, - }    (no dust)
//   f3 = { tau_d log2(e) + 1e-30, pA4, -, - }
template <bool DUST, int DEG>
__global__ void __launch_bounds__(128)
transfer_flat_kernel(MarchConsts mc, const float* __restrict__ coef, int64_t ncell, int npix, int nz, int nv, int npp,
                     int ring, float* __restrict__ out, float* __restrict__ out_cont) {
  extern __shared__ float4 smem4[];
  constexpr unsigned FULL = 0xffffffffu;
  constexpr int PPW = kFlatPPW, ROWS = kFlatRows, SEG = kFlatSeg, SLOTS = kFlatRecSlots;
  constexpr float LOG2E = 1.4426950408889634f;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int pix0 = (blockIdx.x * wpc + warp) * PPW;
  const size_t warp_bytes = (size_t)kFlatRecBytes + (size_t)ring + (size_t)PPW * npp * sizeof(float2);
  char* base = reinterpret_cast<char*>(smem4) + (size_t)warp * warp_bytes;
  float4* rec = reinterpret_cast<float4*>(base);
  unsigned char* owner = reinterpret_cast<unsigned char*>(base + kFlatRecBytes);
  float2* spec = reinterpret_cast<float2*>(base + kFlatRecBytes + ring);      // pair q of pixel g: spec[g * npp + q]
  const unsigned ring_mask = (unsigned)ring - 1u;
  for (int k = lane; k < PPW * npp; k += 32) spec[k] = make_float2(0.0f, 0.0f);
  __syncwarp();

  // phase A: lane L makes the record of (cell row L / PPW, pixel L % PPW) of the chunk
  const int ja = lane / PPW, ga = lane % PPW;
  float C_run = mc.T_bg;      // continuum before the next chunk, of pixel ga
  float G_run = 1.0f;         // exp(dust optical depth so far) since the last fold, of pixel ga
  unsigned spos = 0u, send = 0u;      // pending segments of the stream: [spos, send)
  unsigned nrec = 0u;                 // records made so far (slot = count mod 64)

  const float* p = coef + min(pix0 + ga, npix - 1) + (int64_t)ja * npix;
  float l_e = 0.0f, l_a = 0.0f, l_c = 0.0f, l_s = 1.0f, l_td = 0.0f, l_sd = 0.0f;
  if (ja < nz) {
    l_e = p[0]; l_a = p[ncell]; l_c = p[2 * ncell]; l_s = p[3 * ncell];
    if (DUST) { l_td = p[4 * ncell]; l_sd = p[5 * ncell]; }
  }

  // ---- phase B: passes over the pending segments (all full passes; with flush also the last, partly filled one)
  auto run_passes = [&](bool flush) {
    const f32x2 ONE = pk1(1.0f), NEG1 = pk1(-1.0f);
    constexpr float L1 = 0.6931471805599453f, L2 = L1 * L1, L3 = L2 * L1, L4 = L2 * L2;
    const f32x2 C4 = pk1(L4 / 24.0f), C3 = pk1(-L3 / 6.0f), C2 = pk1(L2 / 2.0f), C1 = pk1(-L1);   // -(1 - 2^-t) / t
    while ((int)(send - spos) >= 32 || (flush && send != spos)) {
      const unsigned s = spos + (unsigned)lane;
      const bool valid = (int)(send - s) > 0;
      const int slot = owner[s & ring_mask] & (SLOTS - 1);
      const float4 r0 = rec[slot], r1 = rec[SLOTS + slot], r2 = rec[2 * SLOTS + slot], r3 = rec[3 * SLOTS + slot];
      const unsigned w2 = (unsigned)__float_as_int(r0.z), w3 = (unsigned)__float_as_int(r0.w);
      const int k = (int)((s - w3) & 0xffffu);                     // segment of the window
      const int q = (int)(w2 & 0xffffu) + SEG * k;                   // its first pair
      const int g = (int)((w3 >> 16) & 3u);
      const int rowid = (int)(w3 >> 18);
      const float xs = r0.y;
      const float x = fmaf((float)(2 * SEG * k), xs, r0.x);
      float2* d = spec + g * npp + q;
      const f32x2 p0 = pk1(r1.x), p1 = pk1(r1.y), p2 = pk1(r1.z), p3 = pk1(r1.w), p4 = pk1(r3.y);
      f32x2 al[SEG], be[SEG], u[SEG], pol[SEG], t[SEG], qq[SEG], mn[SEG];
      {
        f32x2 xx = pk(x, x + xs);
        const f32x2 step2 = pk1(2.0f * xs);
#pragma unroll
        for (int i = 0; i < SEG; ++i) { u[i] = mul2(xx, xx); xx = add2(xx, step2); }
      }
#pragma unroll
      for (int i = 0; i < SEG; ++i) pol[i] = DEG > 3 ? fma2(fma2(p4, u[i], p3), u[i], p2) : fma2(p3, u[i], p2);
#pragma unroll
      for (int i = 0; i < SEG; ++i) pol[i] = fma2(pol[i], u[i], p1);
#pragma unroll
      for (int i = 0; i < SEG; ++i) pol[i] = fma2(pol[i], u[i], p0);
#pragma unroll
      for (int i = 0; i < SEG; ++i) {
        float u0, u1;
        upk(u[i], u0, u1);
        t[i] = mul2(pk(ex2_approx(-u0), ex2_approx(-u1)), pol[i]);            // tau_L log2(e)
      }
      float t0[SEG], t1[SEG], f0[SEG], f1[SEG];
#pragma unroll
      for (int i = 0; i < SEG; ++i) {
        upk(t[i], t0[i], t1[i]);
        f0[i] = ex2_approx(-t0[i]);
        f1[i] = ex2_approx(-t1[i]);
        qq[i] = fma2(t[i], C4, C3);
      }
#pragma unroll
      for (int i = 0; i < SEG; ++i) qq[i] = fma2(qq[i], t[i], C2);
#pragma unroll
      for (int i = 0; i < SEG; ++i) qq[i] = fma2(qq[i], t[i], C1);
#pragma unroll
      for (int i = 0; i < SEG; ++i) {
        // mn = -(1 - exp(-tau_L)) = 2^-t - 1; Taylor below tau_L = 0.08
        const f32x2 sm = mul2(qq[i], t[i]);
        const f32x2 bg = add2(pk(f0[i], f1[i]), NEG1);
        float s0, s1, b0, b1;
        upk(sm, s0, s1);
        upk(bg, b0, b1);
        mn[i] = pk(fabsf(t0[i]) < 0.115f ? s0 : b0, fabsf(t1[i]) < 0.115f ? s1 : b1);
      }
      if (DUST) {
        // Dt' = Dt + (Dt + C G) mn + [t P + mn (-Q t - R)] / (t + tau_d')  =  alpha Dt + beta
        const f32x2 Pn = pk1(r2.x), nQn = pk1(r2.y), nRn = pk1(r2.z), CG = pk1(r2.w), tdp = pk1(r3.x);
        f32x2 rr[SEG], num[SEG];
#pragma unroll
        for (int i = 0; i < SEG; ++i) {
          const f32x2 tt = add2(t[i], tdp);
          float a0, a1;
          upk(tt, a0, a1);
          rr[i] = pk(rcp_approx(a0), rcp_approx(a1));
          num[i] = fma2(nQn, t[i], nRn);
        }
#pragma unroll
        for (int i = 0; i < SEG; ++i) {
          num[i] = fma2(mn[i], num[i], mul2(t[i], Pn));
          al[i] = add2(mn[i], ONE);
        }
#pragma unroll
        for (int i = 0; i < SEG; ++i) be[i] = fma2(rr[i], num[i], mul2(CG, mn[i]));
      } else {
        // Dt' = Dt + (Dt + C - S_L) mn
        const f32x2 nsc = pk1(r2.x);
#pragma unroll
        for (int i = 0; i < SEG; ++i) { al[i] = add2(mn[i], ONE); be[i] = mul2(nsc, mn[i]); }
      }
      // ---- apply in cell order: one step per cell row present in the pass
      const int row_first = __shfl_sync(FULL, rowid, 0);
      const int nvalid = min(32, (int)(send - spos));
      const int row_last = __shfl_sync(FULL, rowid, nvalid - 1);
      const int myrank = valid ? ((rowid - row_first) & 0x3fff) : -1;
      const int nrank = ((row_last - row_first) & 0x3fff) + 1;
      for (int r = 0; r < nrank; ++r) {
        if (myrank == r) {
#pragma unroll
          for (int i = 0; i < SEG; ++i) {
            const float2 v = d[i];
            const f32x2 nv2 = fma2(al[i], pk(v.x, v.y), be[i]);
            float2 w;
            upk(nv2, w.x, w.y);
            d[i] = w;
          }
        }
        __syncwarp();
      }
      spos += 32u;
      if ((int)(send - spos) < 0) spos = send;
    }
  };

  // ---- phase A + phase B for the cell rows [jlo, jhi) of the chunk that starts at cell z0
  unsigned nrow = 0u;                 // cell rows with segments so far
  for (int z0 = 0; z0 < nz; z0 += ROWS) {
    // a chunk with an opaque cell is marched one cell row at a time (G is folded in between)
    const int step = (DUST && __any_sync(FULL, l_td > kFlatSlowTau)) ? 1 : ROWS;
    for (int jlo = 0; jlo < ROWS; jlo += step) {
      const int jhi = jlo + step;
      const bool last_group = jhi >= ROWS;
      const bool mine = ja >= jlo && ja < jhi && z0 + ja < nz;
      // window
      int klo = 0, khi = -1;
      int nq = 0, qlo = 0;
      if (mine && line_window(l_e, l_a, l_c, l_s, nv, klo, khi) > 0) { qlo = klo >> 1; nq = (khi >> 1) - qlo + 1; }
      const int nseg = (nq + SEG - 1) / SEG;
      // dust factors of the cell and the march so far: product scan of exp(tau_d), affine scan of the continuum step
      float E_d = 1.0f, m_d = 0.0f, Eg = 1.0f;
      if (DUST && mine) {
        const float td_e = fminf(l_td, kMaxTauDCell);
        E_d = exp_neg(td_e);
        m_d = one_minus_exp_neg(td_e);
        Eg = ex2_approx(td_e * LOG2E);
      }
      float Gpre = 1.0f, Cj = C_run;
      if (DUST) {
        float P = Eg, A = E_d, B = mine ? l_sd * m_d : 0.0f;
#pragma unroll
        for (int dlt = PPW; dlt < 32; dlt <<= 1) {
          const float Pp = __shfl_up_sync(FULL, P, dlt), Ap = __shfl_up_sync(FULL, A, dlt), Bp = __shfl_up_sync(FULL, B, dlt);
          if (lane >= dlt) { P *= Pp; B = fmaf(A, Bp, B); A *= Ap; }       // (A, B) after (Ap, Bp): x -> A (Ap x + Bp) + B
        }
        float Pex = __shfl_up_sync(FULL, P, PPW), Aex = __shfl_up_sync(FULL, A, PPW), Bex = __shfl_up_sync(FULL, B, PPW);
        if (lane < PPW) { Pex = 1.0f; Aex = 1.0f; Bex = 0.0f; }
        Gpre = G_run * Pex;
        Cj = fmaf(C_run, Aex, Bex);
        // the march after these rows, from the last cell row
        const float Pl = __shfl_sync(FULL, P, 32 - PPW + ga), Al = __shfl_sync(FULL, A, 32 - PPW + ga),
                    Bl = __shfl_sync(FULL, B, 32 - PPW + ga);
        G_run *= Pl;
        C_run = fmaf(C_run, Al, Bl);
      }
      // stream positions, record slot, row id
      int incl = nseg;
#pragma unroll
      for (int dlt = 1; dlt < 32; dlt <<= 1) {
        const int v = __shfl_up_sync(FULL, incl, dlt);
        if (lane >= dlt) incl += v;
      }
      const unsigned segstart = send + (unsigned)(incl - nseg);
      const unsigned total_end = send + (unsigned)__shfl_sync(FULL, incl, 31);
      const unsigned has = __ballot_sync(FULL, nseg > 0);
      const int slot = (int)((nrec + (unsigned)__popc(has & ((1u << lane) - 1u))) & (SLOTS - 1));
      nrec += (unsigned)__popc(has);
      unsigned rows_with = has | (has >> 1);
      rows_with = (rows_with | (rows_with >> 2)) & 0x11111111u;          // bit 4 j: row j has a segment
      const unsigned rowid = nrow + (unsigned)__popc(rows_with & ((1u << (PPW * ja)) - 1u));
      nrow += (unsigned)__popc(rows_with);
      if (nseg > 0) {
        // polynomial of the channel integral from the channel centre (transfer_series.cuh), scaled by
        // As' = a_c (2 s / sqrt(pi)) log2(e)
        const float sc = l_s;
        const float a_min = fmaxf(1.0e-10f * l_e, 1.0e-30f);
        const float a_safe = fabsf(l_a) < a_min ? a_min : l_a;
        const float sp = 1.1283791670955126f * sc;
        const float As = a_safe * sp, Es = l_e * sp;
        const float Asp = As * LOG2E;
        const float xs = 1.2011224087864498f * sc;
        const float s2 = sc * sc, s4 = s2 * s2, s6 = s4 * s2, s8 = s4 * s4;
        const float c0 = 1.0f - s2 * (1.0f / 12.0f) + s4 * (1.0f / 160.0f) - s6 * (1.0f / 2688.0f) + s8 * (1.0f / 55296.0f);
        const float c1 = s2 * (1.0f / 6.0f) - s4 * (1.0f / 40.0f) + s6 * (1.0f / 448.0f) - s8 * (1.0f / 6912.0f);
        const float c2 = s4 * (1.0f / 120.0f) - s6 * (1.0f / 672.0f) + s8 * (1.0f / 6912.0f);
        const float c3 = s6 * (1.0f / 5040.0f) - s8 * (1.0f / 25920.0f);
        const float c4 = s8 * (1.0f / 362880.0f);
        constexpr float L1 = 0.6931471805599453f, L2 = L1 * L1, L3 = L2 * L1, L4 = L2 * L2;
        float4 f0, f2, f3;
        f0.x = ((float)(2 * qlo) + 0.5f - l_c) * xs;
        f0.y = xs;
        f0.z = __int_as_float(qlo | (nq << 16));
        f0.w = __int_as_float((int)((segstart & 0xffffu) | ((unsigned)ga << 16) | ((rowid & 0x3fffu) << 18)));
        if (DUST) {
          const float Gn = Gpre * Eg;
          const float iA = LOG2E * rcp_approx(Asp);
          f2.x = m_d * fmaf(-l_sd, As, Es) * iA * Gn;
          f2.y = -E_d * Es * iA * Gn;
          f2.z = -E_d * l_sd * l_td * LOG2E * Gn;
          f2.w = Cj * Gpre;
          f3.x = fmaf(l_td, LOG2E, 1.0e-30f);
        } else {
          f2 = make_float4(mc.T_bg - Es * rcp_approx(As), 0.0f, 0.0f, 0.0f);
          f3.x = 0.0f;
        }
        f3.y = DEG > 3 ? Asp * (c4 * L4) : 0.0f;
        f3.z = 0.0f; f3.w = 0.0f;
        rec[slot] = f0;
        rec[SLOTS + slot] = make_float4(Asp * c0, Asp * (c1 * L1), Asp * (c2 * L2), Asp * (c3 * L3));
        rec[2 * SLOTS + slot] = f2;
        rec[3 * SLOTS + slot] = f3;
      }
      // the next chunk's coefficients, requested before the passes of this one
      if (last_group) {
        const int zn = z0 + ROWS + ja;
        l_e = 0.0f; l_a = 0.0f; l_td = 0.0f;
        if (zn < nz) {
          p += (int64_t)ROWS * npix;
          l_e = p[0]; l_a = p[ncell]; l_c = p[2 * ncell]; l_s = p[3 * ncell];
          if (DUST) { l_td = p[4 * ncell]; l_sd = p[5 * ncell]; }
        }
      }
      // publish the segments (in batches if the ring is too small for all of them) and run the full passes; everything
      // pending is flushed at the end of the march and before G is folded back into the spectra (the pending
      // segments were built for the old scale)
      const bool fold = DUST && __any_sync(FULL, G_run > kFoldG);
      const bool flush_after = fold || (last_group && z0 + ROWS >= nz);
      const int mx = __reduce_max_sync(FULL, nseg);
      int done = 0;                                    // segments of this lane already published
      for (;;) {
        const unsigned lim = spos + (unsigned)ring;   // segments below lim fit the ring
        for (int k = 0; k < mx; ++k) {
          const unsigned sk = segstart + (unsigned)k;
          if (k >= done && k < nseg && (int)(lim - sk) > 0) owner[sk & ring_mask] = (unsigned char)slot;
        }
        done = max(done, min(nseg, (int)(lim - segstart)));           // (negative when the window starts beyond lim)
        const bool all = (int)(lim - total_end) >= 0;
        send = all ? total_end : lim;
        __syncwarp();
        run_passes(flush_after && all);
        if (all) break;
      }
      if (fold) {
        for (int g = 0; g < PPW; ++g) {
          const float Gg = __shfl_sync(FULL, G_run, g);
          if (Gg > kFoldG) {
            const float inv = 1.0f / Gg;
            float2* sg = spec + g * npp;
            for (int q = lane; q < npp; q += 32) { float2 v = sg[q]; v.x *= inv; v.y *= inv; sg[q] = v; }
            if (ga == g) G_run = 1.0f;
          }
        }
        __syncwarp();
      }
    }
  }
  __syncwarp();

  // ---- K5: subtraction / conversion, one pixel at a time, 32 lanes along the channels
  for (int g = 0; g < PPW; ++g) {
    const int pix = pix0 + g;
    const float Cg = __shfl_sync(FULL, C_run, g), invG = 1.0f / __shfl_sync(FULL, G_run, g);
    if (pix >= npix) break;
    const float* sg = reinterpret_cast<const float*>(spec + g * npp);
    if (out != nullptr) {
      float* o = out + (int64_t)pix * nv;
      for (int c = lane; c < nv; c += 32) o[c] = convert_out(sg[c] * invG, Cg, mc);
    }
    if (out_cont != nullptr && lane == 0) out_cont[pix] = Cg * mc.inv_KRJ;
  }
}

template <bool DUST, int DEG>
inline cudaError_t launch_transfer_flat_t(const MarchConsts& mc, const float* coef, int64_t ncell, int npix, int nz, int nv,
                                          float* out, float* out_cont, cudaStream_t st) {
  const int npp = flat_padded_pairs(nv), ring = flat_ring_size(nv);
  const size_t per_warp = flat_smem_per_warp(nv);
  // warps per CTA: the count that leaves most warps resident in the 227 KB of an SM (ties: the larger CTA)
  int wpc = 1, best = 0;
  for (int w = 4; w >= 1; w >>= 1) {
    const size_t per_cta = w * per_warp + 1024;
    const int resident = per_cta <= 227 * 1024 ? (int)((227 * 1024) / per_cta) * w : 0;
    if (resident > best) { best = resident; wpc = w; }
  }
  if (best == 0) return cudaErrorInvalidConfiguration;
  const size_t smem = wpc * per_warp;
  const int ppc = wpc * kFlatPPW;
  const unsigned grid = (unsigned)((npix + ppc - 1) / ppc);
  cudaError_t e = cudaFuncSetAttribute(transfer_flat_kernel<DUST, DEG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  transfer_flat_kernel<DUST, DEG><<<grid, wpc * 32, smem, st>>>(mc, coef, ncell, npix, nz, nv, npp, ring, out, out_cont);
  return cudaGetLastError();
}

// s_max: upper bound of dv / b over all cells (dv / microturbulence); selects the polynomial degree.
inline cudaError_t launch_transfer_flat(const MarchConsts& mc, const float* coef, int64_t ncell, int npix, int nz, int nv,
                                        bool dust, float s_max, float* out, float* out_cont, cudaStream_t st) {
  const bool deg3 = s_max <= kSeriesDeg3MaxS;
  if (dust) return deg3 ? launch_transfer_flat_t<true, 3>(mc, coef, ncell, npix, nz, nv, out, out_cont, st)
                        : launch_transfer_flat_t<true, 4>(mc, coef, ncell, npix, nz, nv, out, out_cont, st);
  return deg3 ? launch_transfer_flat_t<false, 3>(mc, coef, ncell, npix, nz, nv, out, out_cont, st)
              : launch_transfer_flat_t<false, 4>(mc, coef, ncell, npix, nz, nv, out, out_cont, st);
}

}  // namespace iris
