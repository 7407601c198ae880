// Pipe-rate microbenchmarks for the ALU roofline of the tracer (SURVEY.md 8(d) asks for
// them): how many SMSP clocks one warp instruction of each class occupies its pipe on this B200, measured with
// many independent chains per thread and full occupancy, so that latency is hidden and the pipe is the limit.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o microbench microbench.cu && ./microbench
//
// Prints one line per class: SMSP clocks per warp instruction (at the clock given by SM_MHZ, default 1965).
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>

constexpr int CHAINS = 8;
constexpr int UNROLL = 32;

enum { K_FFMA, K_IMAD, K_IMAD_WIDE, K_LOP3, K_DFMA, K_MUFU_RCP, K_PHILOX, K_FFMA2, N_KINDS };
static const char* NAMES[N_KINDS] = {"FFMA (fp32 fused multiply-add)", "IMAD (32-bit integer multiply-add)",
                                     "IMAD.WIDE.U32 (32x32->64 multiply)", "LOP3 (integer logic)",
                                     "DFMA (fp64 fused multiply-add)", "MUFU.RCP (special function)",
                                     "Philox4x32-10 block (20 wide multiplies + 20 LOP3)",
                                     "FFMA2 (packed fp32 fused multiply-add, two per lane)"};
static const double INSTR_PER_STEP[N_KINDS] = {1, 1, 1, 1, 1, 1, 1, 1};

template <int KIND>
__global__ void __launch_bounds__(256, 4) bench(int iters, uint32_t seed, uint32_t* out) {
  uint32_t id = blockIdx.x * blockDim.x + threadIdx.x + seed;
  float f[CHAINS]; double d[CHAINS]; uint32_t u[CHAINS]; unsigned long long w[CHAINS]; float2 f2[CHAINS];
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) { f[c] = 1.0f + id * 1e-9f + c; d[c] = 1.0 + id * 1e-12 + c; u[c] = id * 2654435761u + c; w[c] = u[c]; f2[c] = make_float2(f[c], f[c] + 0.5f); }
  const float fa = 1.0000001f, fb = 1e-7f;
  const double da = 1.0000000001, db = 1e-10;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < UNROLL; ++k) {
#pragma unroll
      for (int c = 0; c < CHAINS; ++c) {
        if (KIND == K_FFMA) f[c] = fmaf(f[c], fa, fb);
        if (KIND == K_IMAD) u[c] = u[c] * u[(c + 1) % CHAINS] + id;
        if (KIND == K_IMAD_WIDE) w[c] = (unsigned long long)(uint32_t)(w[c] ^ (w[c] >> 32)) * 0xD2511F53ull;
        if (KIND == K_LOP3) u[c] = u[c] ^ u[(c + 1) % CHAINS] ^ (id + k);
        if (KIND == K_DFMA) d[c] = fma(d[c], da, db);
        if (KIND == K_FFMA2) f2[c] = __ffma2_rn(f2[c], make_float2(fa, fa), make_float2(fb, fb));
        if (KIND == K_MUFU_RCP) { asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(f[c])); f[c] += fb; }  // + one FADD on the FMA pipe
      }
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) acc ^= __float_as_uint(f[c]) ^ (uint32_t)__double2loint(d[c]) ^ u[c] ^ (uint32_t)w[c] ^ (uint32_t)(w[c] >> 32) ^ __float_as_uint(f2[c].x) ^ __float_as_uint(f2[c].y);
  if (acc == 0x12345678u) out[id & 1023] = acc;
}

struct Keys { uint32_t k0[10], k1[10]; };
__global__ void __launch_bounds__(256, 4) bench_philox(const __grid_constant__ Keys pk, int iters, uint32_t* out) {
  uint32_t id = blockIdx.x * blockDim.x + threadIdx.x, acc = 0;
  for (int i = 0; i < iters; ++i) {
    uint32_t r[3][4];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      uint32_t c0 = id + c * 77777u + i * 131u, c1 = 0, c2 = 0, c3 = 0;
#pragma unroll
      for (int rd = 0; rd < 10; ++rd) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ pk.k0[rd], n2 = hi0 ^ c3 ^ pk.k1[rd];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
      }
      r[c][0] = c0; r[c][1] = c1; r[c][2] = c2; r[c][3] = c3;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) acc += r[c][0] ^ r[c][1] ^ r[c][2] ^ r[c][3];
  }
  if (acc == 0x12345678u) out[id & 1023] = acc;
}

// IMAD.WIDE chains with NL extra independent LOP3 per multiply (each chain step is one LOP3 + one wide multiply,
// as in a Philox round): how the integer multiplier and the logic pipe share the sub-partition
template <int NL>
__global__ void __launch_bounds__(256, 4) bench_mix(int iters, uint32_t seed, uint32_t* out) {
  constexpr int CH = 6;
  uint32_t id = blockIdx.x * blockDim.x + threadIdx.x + seed;
  unsigned long long w[CH]; uint32_t u[CH][4];
#pragma unroll
  for (int c = 0; c < CH; ++c) { w[c] = id * 2654435761u + c; for (int j = 0; j < 4; ++j) u[c][j] = id + 17 * c + j; }
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 16; ++r) {
#pragma unroll
      for (int c = 0; c < CH; ++c) {
        unsigned long long p; const uint32_t x = (uint32_t)w[c] ^ (uint32_t)(w[c] >> 32) ^ seed;
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(x), "r"(0xD2511F53u));
        w[c] = p;
#pragma unroll
        for (int j = 0; j < NL; ++j) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[c][j]) : "r"(id), "r"(seed));
      }
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int c = 0; c < CH; ++c) { acc ^= (uint32_t)w[c] ^ (uint32_t)(w[c] >> 32); for (int j = 0; j < 4; ++j) acc ^= u[c][j]; }
  if (acc == 0x12345678u) out[id & 1023] = acc;
}

// The arithmetic core of the tracer's stage A for one row of 32 neutron ids: words 0 and 1 of Philox block 0 of
// (id, id_hi, 0, exp) -- the compiler drops what the unused words 2, 3 would need -- and the two window compares,
// three rows in flight; no compaction, no stores.  What this loop costs is what stage A cannot go below.
__global__ void __launch_bounds__(256, 4) bench_stage_a(const __grid_constant__ Keys pk, int iters, uint32_t id_hi, uint32_t expw,
                                                        uint32_t lo0, uint32_t d0, uint32_t lo1, uint32_t d1, uint32_t* out) {
  uint32_t id = blockIdx.x * blockDim.x + threadIdx.x, acc = 0;
  for (int i = 0; i < iters; ++i) {
    uint32_t w0[3], w1[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      uint32_t c0 = id + k * 77777u + i * 131u, c1 = id_hi, c2 = 0u, c3 = expw;
#pragma unroll
      for (int rd = 0; rd < 9; ++rd) {
        unsigned long long p0, p1;
        asm("mul.wide.u32 %0, %1, %2;" : "=l"(p0) : "r"(0xD2511F53u), "r"(c0));
        asm("mul.wide.u32 %0, %1, %2;" : "=l"(p1) : "r"(0xCD9E8D57u), "r"(c2));
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ pk.k0[rd], n2 = (uint32_t)(p0 >> 32) ^ c3 ^ pk.k1[rd];
        c0 = n0; c1 = (uint32_t)p1; c2 = n2; c3 = (uint32_t)p0;
      }
      w0[k] = __umulhi(0xCD9E8D57u, c2) ^ c1 ^ pk.k0[9];
      w1[k] = 0xCD9E8D57u * c2;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) acc += ((w0[k] - lo0 <= d0) && (w1[k] - lo1 <= d1)) ? 1u : 0u;
  }
  if (acc == 0x12345678u) out[id & 1023] = acc;
}

template <int KIND>
static double run(double mhz) {
  uint32_t* d; cudaMalloc(&d, 4096);
  int n_sm = 0; cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, 0);
  const int grid = n_sm * 4, iters = 400;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0);
    bench<KIND><<<grid, 256>>>(iters, rep, d);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  const double warp_instr_per_smsp = (double)grid * 8 / (n_sm * 4) * iters * UNROLL * CHAINS * INSTR_PER_STEP[KIND];
  cudaFree(d);
  return best * 1e-3 * mhz * 1e6 / warp_instr_per_smsp;
}

static double run_philox(double mhz) {
  uint32_t* d; cudaMalloc(&d, 4096);
  int n_sm = 0; cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, 0);
  Keys pk; for (int r = 0; r < 10; ++r) { pk.k0[r] = 1234u + r * 0x9E3779B9u; pk.k1[r] = 99u + r * 0xBB67AE85u; }
  const int grid = n_sm * 4, iters = 4000;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0);
    bench_philox<<<grid, 256>>>(pk, iters, d);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  const double warp_blocks_per_smsp = (double)grid * 8 / (n_sm * 4) * iters * 3;
  cudaFree(d);
  return best * 1e-3 * mhz * 1e6 / warp_blocks_per_smsp;
}

template <int NL>
static double run_mix(double mhz) {
  uint32_t* d; cudaMalloc(&d, 4096);
  int n_sm = 0; cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, 0);
  const int grid = n_sm * 4, iters = 300;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0);
    bench_mix<NL><<<grid, 256>>>(iters, rep, d);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaFree(d);
  return best * 1e-3 * mhz * 1e6 / ((double)grid * 8 / (n_sm * 4) * iters * 16 * 6);   // clocks per (multiply + its LOP3 + NL LOP3)
}

static double run_stage_a(double mhz) {
  uint32_t* d; cudaMalloc(&d, 4096);
  int n_sm = 0; cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, 0);
  Keys pk; for (int r = 0; r < 10; ++r) { pk.k0[r] = 1234u + r * 0x9E3779B9u; pk.k1[r] = 99u + r * 0xBB67AE85u; }
  const int grid = n_sm * 4, iters = 4000;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0);
    bench_stage_a<<<grid, 256>>>(pk, iters, 7u, 3u, 0x40000000u, 0x7FFFFFFFu, 0x40000000u, 0x7FFFFFFFu, d);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaFree(d);
  return best * 1e-3 * mhz * 1e6 / ((double)grid * 8 / (n_sm * 4) * iters * 3);   // clocks per row of 32 ids
}

// What a CUDA-event pair around one launch reads for a kernel that does nothing: the floor under every per-launch
// "kernel time" the library reports and under every per-step event pair of bench.py.
__global__ void __launch_bounds__(640, 1) null_kernel(int* out, int never) {
  if (never == 12345) out[0] = 1;
}
static double event_floor_us() {
  int* d = nullptr;
  cudaMalloc(&d, 4);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best = 1e30;
  for (int r = 0; r < 60; ++r) {
    cudaEventRecord(e0);
    null_kernel<<<148, 640>>>(d, 0);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (r >= 10 && (double)ms * 1e3 < best) best = (double)ms * 1e3;
  }
  cudaFree(d);
  return best;
}

int main() {
  const char* env = getenv("SM_MHZ");
  const double mhz = env ? atof(env) : 1965.0;
  double v[N_KINDS];
  v[K_FFMA] = run<K_FFMA>(mhz); v[K_IMAD] = run<K_IMAD>(mhz); v[K_IMAD_WIDE] = run<K_IMAD_WIDE>(mhz);
  v[K_LOP3] = run<K_LOP3>(mhz); v[K_DFMA] = run<K_DFMA>(mhz); v[K_MUFU_RCP] = run<K_MUFU_RCP>(mhz);
  v[K_PHILOX] = run_philox(mhz);
  v[K_FFMA2] = run<K_FFMA2>(mhz);
  printf("SMSP clocks per warp instruction at %.0f MHz (32 resident warps per SM, %d independent chains per thread)\n", mhz, CHAINS);
  for (int k = 0; k < N_KINDS; ++k) printf("  %-52s %7.2f\n", NAMES[k], v[k]);
  const double m0 = run_mix<0>(mhz), m1 = run_mix<1>(mhz), m2 = run_mix<2>(mhz), m3 = run_mix<3>(mhz), sa = run_stage_a(mhz);
  printf("  %-52s %7.2f %7.2f %7.2f %7.2f\n", "wide multiply + (1 + NL) LOP3, NL = 0..3", m0, m1, m2, m3);
  printf("  %-52s %7.2f\n", "stage-A core: Philox words 0,1 + window test, per row", sa);
  const double fl = event_floor_us();
  printf("  %-52s %7.2f us\n", "event pair around a kernel that does nothing", fl);
  // one machine-readable line for bench.py
  printf("{\"sm_mhz\": %.0f, \"ffma\": %.4f, \"imad\": %.4f, \"imad_wide\": %.4f, \"lop3\": %.4f, \"dfma\": %.4f, \"mufu\": %.4f, "
         "\"philox_block\": %.3f, \"wide_lop3\": [%.4f, %.4f, %.4f, %.4f], \"stage_a_core_row\": %.3f, \"event_floor_us\": %.2f, \"ffma2\": %.4f}\n",
         mhz, v[K_FFMA], v[K_IMAD], v[K_IMAD_WIDE], v[K_LOP3], v[K_DFMA], v[K_MUFU_RCP], v[K_PHILOX], m0, m1, m2, m3, sa, fl, v[K_FFMA2]);
  return 0;
}
