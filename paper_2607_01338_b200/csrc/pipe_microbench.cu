// Issue-rate microbenchmarks of the sm_100a pipes the LOS transfer kernel lives on (FP32 FMA, packed
// FFMA2, MUFU ex2 / rcp, ALU, warp shuffle, shared memory).  They supply the measured denominators of the
// "alu" roofline in DESIGN.md (MEASURED_PEAKS.json holds only HBM and bf16 tensor peaks).
//
// Stand-alone program (not part of libiris_so.so):  python -m paper_2607_01338_b200.microbench
// Every kernel runs ITER iterations of an unrolled body of CHAINS independent dependency chains on
// 148 x 8 CTAs of 256 threads.  Each CTA records %smid and clock64() at its start and end; the host takes,
// per SM, the warp instructions of the CTAs that ran there over (latest end - earliest start) and reports the
// median over SMs, and independently the whole-grid figure from the CUDA-event time at the given SM clock.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_)); exit(1); } } while (0)

constexpr int ITER = 8192;
constexpr int CHAINS = 8;

enum Op { FFMA_RRR, FFMA_IMM, FFMA2, FMUL2, MUFU_EX2, MUFU_RCP, ALU_LOP, FMNMX, SHFL, LDS, STS_LDS, MIX_FMA_MUFU, MIX_FMA_ALU, MIX_FFMA2_MUFU, NOPS };

static const char* kNames[NOPS] = {"ffma_rrr", "ffma_imm", "ffma2", "fmul2", "mufu_ex2", "mufu_rcp_fadd", "alu_lop3", "fmnmx", "shfl",
                                   "lds_chase", "sts_lds", "mix_8ffma_1mufu", "mix_1ffma_1alu", "mix_4ffma2_1mufu"};
// warp instructions per chain step, and of those how many FP32 multiply-adds per lane (for the FMA/clk figure)
static const int kInstrPerStep[NOPS] = {1, 1, 1, 1, 1, 2, 1, 1, 1, 1, 2, 9, 2, 5};
static const int kFmaPerStep[NOPS] = {1, 1, 2, 2, 0, 0, 0, 0, 0, 0, 0, 8, 1, 8};

__device__ __forceinline__ unsigned long long pack2(float a, float b) {
  unsigned long long r;
  asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b));
  return r;
}

template <int OP>
__global__ void __launch_bounds__(256) bench_kernel(float* out, const float* in, long long* cycles, int iters) {
  __shared__ float sm[256 * 2];
  float x[CHAINS];
  unsigned long long p[CHAINS];
  const float b = in[0], c = in[1];
  const unsigned long long bb = pack2(b, in[2]), cc = pack2(c, in[3]);
#pragma unroll
  for (int i = 0; i < CHAINS; ++i) { x[i] = in[4 + i] + threadIdx.x; p[i] = pack2(x[i], x[i] + 1.0f); }
  unsigned q[CHAINS];
  if (OP == LDS) {   // every word holds the shared-memory address of the word 32 further on (conflict-free chase)
    const unsigned base = (unsigned)__cvta_generic_to_shared(sm);
    ((unsigned*)sm)[threadIdx.x] = base + 4u * ((threadIdx.x + 32) & 511);
    ((unsigned*)sm)[threadIdx.x + 256] = base + 4u * ((threadIdx.x + 256 + 32) & 511);
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) q[i] = base + 4u * ((threadIdx.x + 32 * i) & 511);
  } else {
    sm[threadIdx.x] = x[0]; sm[threadIdx.x + 256] = x[1];
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) q[i] = 0u;
  }
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) {
      if (OP == FFMA_RRR) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(b), "f"(c));
      if (OP == FFMA_IMM) asm volatile("fma.rn.f32 %0, %0, %1, 0f3F8CCCCD;" : "+f"(x[i]) : "f"(b));
      if (OP == FFMA2) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[i]) : "l"(bb), "l"(cc));
      if (OP == FMUL2) asm volatile("mul.rn.f32x2 %0, %0, %1;" : "+l"(p[i]) : "l"(bb));
      if (OP == MUFU_EX2) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
      if (OP == MUFU_RCP) {   // rcp alone is folded (rcp(rcp(x)) = x): pair it with an add
        asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
        asm volatile("add.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(b));
      }
      if (OP == ALU_LOP) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(*(unsigned*)&x[i]) : "r"(__float_as_uint(b)), "r"(__float_as_uint(c)));
      if (OP == FMNMX) asm volatile("min.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(b));
      if (OP == SHFL) asm volatile("shfl.sync.idx.b32 %0, %0, %1, 0x1f, 0xffffffff;" : "+f"(x[i]) : "r"((threadIdx.x + 1) & 31));
      if (OP == LDS) asm volatile("ld.shared.b32 %0, [%0];" : "+r"(q[i]) :: "memory");   // address chase
      if (OP == STS_LDS) {
        asm volatile("st.shared.f32 [%1], %0;" :: "f"(x[i]), "r"((unsigned)__cvta_generic_to_shared(&sm[(threadIdx.x + i * 32) & 511])) : "memory");
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x[i]) : "r"((unsigned)__cvta_generic_to_shared(&sm[(threadIdx.x + i * 32 + 32) & 511])) : "memory");
      }
      if (OP == MIX_FMA_MUFU) {
        float y = x[i];
#pragma unroll
        for (int k = 0; k < 8; ++k) asm volatile("fma.rn.f32 %0, %0, %1, 0f3F8CCCCD;" : "+f"(y) : "f"(b));
        asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(y));
        x[i] = y;
      }
      if (OP == MIX_FMA_ALU) {
        asm volatile("fma.rn.f32 %0, %0, %1, 0f3F8CCCCD;" : "+f"(x[i]) : "f"(b));
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(*(unsigned*)&x[i]) : "r"(__float_as_uint(b)), "r"(__float_as_uint(c)));
      }
      if (OP == MIX_FFMA2_MUFU) {
        unsigned long long q = p[i];
#pragma unroll
        for (int k = 0; k < 4; ++k) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(q) : "l"(bb), "l"(cc));
        p[i] = q;
        asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
      }
    }
  }
  const long long t1 = clock64();
  float s = 0.0f;
#pragma unroll
  for (int i = 0; i < CHAINS; ++i) {
    float lo, hi;
    asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p[i]));
    s += x[i] + lo + hi + (float)q[i];
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
  if (threadIdx.x == 0) {
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    cycles[3 * blockIdx.x] = t0; cycles[3 * blockIdx.x + 1] = t1; cycles[3 * blockIdx.x + 2] = smid;
  }
}

typedef void (*kern_t)(float*, const float*, long long*, int);
static kern_t kKernels[NOPS] = {bench_kernel<0>, bench_kernel<1>, bench_kernel<2>, bench_kernel<3>, bench_kernel<4>,
                                bench_kernel<5>, bench_kernel<6>, bench_kernel<7>, bench_kernel<8>, bench_kernel<9>,
                                bench_kernel<10>, bench_kernel<11>, bench_kernel<12>, bench_kernel<13>};

int main(int argc, char** argv) {
  double sm_mhz = argc > 1 ? atof(argv[1]) : 1965.0;   // SM clock under load, for the event-time figure
  int dev = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int ctas_per_sm = 8, threads = 256, grid = sms * ctas_per_sm;
  float *d_out, *d_in; long long* d_cyc;
  CK(cudaMalloc(&d_out, sizeof(float) * grid * threads));
  CK(cudaMalloc(&d_in, sizeof(float) * 64));
  CK(cudaMalloc(&d_cyc, sizeof(long long) * 3 * grid));
  std::vector<float> h_in(64);
  for (int i = 0; i < 64; ++i) h_in[i] = 0.999f + 1e-4f * i;
  CK(cudaMemcpy(d_in, h_in.data(), sizeof(float) * 64, cudaMemcpyHostToDevice));
  cudaEvent_t a, b;
  CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
  printf("{\"sm_count\": %d, \"assumed_sm_mhz\": %.0f, \"ctas_per_sm\": %d, \"threads_per_cta\": %d, \"pipes\": {", sms, sm_mhz, ctas_per_sm, threads);
  for (int op = 0; op < NOPS; ++op) {
    kKernels[op]<<<grid, threads>>>(d_out, d_in, d_cyc, 64);   // warm-up
    CK(cudaDeviceSynchronize());
    CK(cudaEventRecord(a));
    kKernels[op]<<<grid, threads>>>(d_out, d_in, d_cyc, ITER);
    CK(cudaEventRecord(b));
    CK(cudaDeviceSynchronize());
    CK(cudaGetLastError());
    float ms = 0.0f;
    CK(cudaEventElapsedTime(&ms, a, b));
    std::vector<long long> cyc(3 * grid);
    CK(cudaMemcpy(cyc.data(), d_cyc, sizeof(long long) * 3 * grid, cudaMemcpyDeviceToHost));
    const double winstr_cta = (double)(threads / 32) * ITER * CHAINS * kInstrPerStep[op];
    std::vector<long long> first(1024, -1), last(1024, -1);
    std::vector<int> nctas(1024, 0);
    for (int g = 0; g < grid; ++g) {
      const int s = (int)cyc[3 * g + 2];
      if (first[s] < 0 || cyc[3 * g] < first[s]) first[s] = cyc[3 * g];
      if (cyc[3 * g + 1] > last[s]) last[s] = cyc[3 * g + 1];
      nctas[s]++;
    }
    std::vector<double> ipcs;
    for (int s = 0; s < 1024; ++s)
      if (nctas[s]) ipcs.push_back(nctas[s] * winstr_cta / (double)(last[s] - first[s]));
    std::sort(ipcs.begin(), ipcs.end());
    const double ipc_clock = ipcs[ipcs.size() / 2];
    const double ipc_event = winstr_cta * grid / sms / (ms * 1e-3 * sm_mhz * 1e6);
    const double fma_clk = ipc_clock * 32.0 * kFmaPerStep[op] / kInstrPerStep[op];
    printf("%s\"%s\": {\"warp_instr_per_clk_per_sm\": %.3f, \"by_event_time\": %.3f, \"fp32_fma_per_clk_per_sm\": %.1f, \"ms\": %.4f}",
           op ? ", " : "", kNames[op], ipc_clock, ipc_event, fma_clk, ms);
  }
  printf("}}\n");
  return 0;
}
