// Instrumentation: the ALU rooflines of the blend kernels, MEASURED ("the builder measures them with
// two dependent-free micro-kernels and records them").  MEASURED_PEAKS.json holds only the HBM copy rate and the
// bf16 tensor rate; the blend kernels (S3 / S4a) are bound by FP32-pipe issue and by the MUFU (XU) pipe, so their
// denominators are taken here, on the device the bench runs on, at the clock it runs at:
//   [0] FFMA      three-register fma.rn.f32, 16 independent chains per thread          lane-instructions / s
//   [1] FFMA2     packed fma.rn.f32x2 (sm_100), 8 independent chains of pairs          lane-instructions / s (2 flops x 2)
//   [2] MUFU.EX2  ex2.approx.ftz.f32, 8 independent chains                             lane-ops / s
//   [3] MUFU.COS  cos.approx.ftz.f32 (range multiply + MUFU.COS), 8 chains             lane-ops / s
//   [4] MIX       4 FFMA : 1 MUFU.EX2 per chain step (the blend's mix), all instructions  lane-instructions / s
//   [5] IADD      add.s32 on the ALU pipe, 16 chains (the other half of the issue budget) lane-instructions / s
// [8..13] the same six per SM per clock (rate / (SMs x [6])), [6] = SM clock in Hz seen by the kernels (clock64 ticks per
// %globaltimer ns of CTA 0), [7] = number of SMs.  Nothing here is used to render.
#include "common.cuh"

namespace gabsplat {
namespace {

constexpr int kPeakThreads = 256;
constexpr int kPeakCtasPerSm = 8;   // 64 warps per SM: every scheduler has 16 warps to pick from
constexpr int kPeakIters = 2048;     // chain steps per thread
constexpr int kUnroll = 8;           // chain steps per loop iteration (128 instructions per branch)

__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}

template <int MODE>
__global__ void __launch_bounds__(kPeakThreads) peak_kernel(int iters, float seed, float* sink, long long* cycles) {
  const unsigned long long n0 = global_ns();
  const long long t0 = clock64();
  float r = 0.f;
  if (MODE == 0) {
    float a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = seed + (float)(threadIdx.x + i);
    const float m = 0.999f + seed, c = 1e-3f + seed;
#pragma unroll 1
    for (int it = 0; it < iters; it += kUnroll) {
#pragma unroll
      for (int r8 = 0; r8 < kUnroll; ++r8)
#pragma unroll
        for (int i = 0; i < 16; ++i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(m), "f"(c));
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) r += a[i];
  } else if (MODE == 1) {
    float2 a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = make_float2(seed + (float)(threadIdx.x + i), seed - (float)i);
    const float2 m = make_float2(0.999f + seed, 0.998f + seed), c = make_float2(1e-3f + seed, 2e-3f + seed);
#pragma unroll 1
    for (int it = 0; it < iters; it += kUnroll) {
#pragma unroll
      for (int r8 = 0; r8 < kUnroll; ++r8)
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        unsigned long long& x = reinterpret_cast<unsigned long long&>(a[i]);
        asm volatile("fma.rn.f32x2 %0, %0, %1, %2;"
                     : "+l"(x)
                     : "l"(reinterpret_cast<const unsigned long long&>(m)), "l"(reinterpret_cast<const unsigned long long&>(c)));
      }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) r += a[i].x + a[i].y;
  } else if (MODE == 2) {
    float a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = seed - 0.1f * (float)((threadIdx.x + i) & 7);
#pragma unroll 1
    for (int it = 0; it < iters; it += kUnroll) {
#pragma unroll
      for (int r8 = 0; r8 < kUnroll; ++r8)
#pragma unroll
        for (int i = 0; i < 8; ++i) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[i]));   // overflows to +inf: same rate
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) r += a[i];
  } else if (MODE == 3) {
    float a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = seed + 0.1f * (float)((threadIdx.x + i) & 7);
#pragma unroll 1
    for (int it = 0; it < iters; it += kUnroll) {
#pragma unroll
      for (int r8 = 0; r8 < kUnroll; ++r8)
#pragma unroll
        for (int i = 0; i < 8; ++i) asm volatile("cos.approx.ftz.f32 %0, %0;" : "+f"(a[i]));
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) r += a[i];
  } else if (MODE == 4) {
    // the blend's mix, dependency-free: per step 4 FFMA on four accumulators of their own and one MUFU.EX2 on a fifth
    float a[4][4], b[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      b[i] = seed - 0.1f * (float)((threadIdx.x + i) & 7);
#pragma unroll
      for (int j = 0; j < 4; ++j) a[i][j] = seed + 0.01f * (float)((threadIdx.x + i + j) & 7);
    }
    const float m = 0.5f + seed, c = 1e-3f + seed;
#pragma unroll 1
    for (int it = 0; it < iters; it += kUnroll) {
#pragma unroll
      for (int r8 = 0; r8 < 2 * kUnroll; ++r8)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
#pragma unroll
          for (int j = 0; j < 4; ++j) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i][j]) : "f"(m), "f"(c));
          asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(b[i]));
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) r += a[i][0] + a[i][1] + a[i][2] + a[i][3] + b[i];
  } else {
    int a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = (int)threadIdx.x + i;
    const int c = (int)seed + 3;
#pragma unroll 1
    for (int it = 0; it < iters; it += kUnroll) {
#pragma unroll
      for (int r8 = 0; r8 < kUnroll; ++r8)
#pragma unroll
        for (int i = 0; i < 16; ++i) asm volatile("add.s32 %0, %0, %1;" : "+r"(a[i]) : "r"(c));
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) r += (float)a[i];
  }
  const long long t1 = clock64();
  const unsigned long long n1 = global_ns();
  if (r == 123456.789f) sink[0] = r;  // never true: keeps the chains alive
  if (blockIdx.x == 0 && threadIdx.x == 0) { cycles[0] = t1 - t0; cycles[1] = (long long)(n1 - n0); }
}

// warp instructions per chain step of each mode, and what is counted as the result
constexpr int kInstrPerIter[6] = {16, 8, 8, 8, 40, 16};  // MIX: 2 x 4 x (4 FFMA + 1 MUFU)

}  // namespace

// results: 16 floats (see the header of this file).  Synchronises.  scratch: >= 64 bytes of device memory.
cudaError_t measure_peaks(float* results_host, void* scratch, cudaStream_t st) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  float* sink = reinterpret_cast<float*>(scratch);
  long long* cycles = reinterpret_cast<long long*>(reinterpret_cast<char*>(scratch) + 16);
  cudaEvent_t a, b;
  if ((e = cudaEventCreate(&a)) != cudaSuccess) return e;
  if ((e = cudaEventCreate(&b)) != cudaSuccess) { cudaEventDestroy(a); return e; }
  const int grid = sms * kPeakCtasPerSm;
  for (int i = 0; i < 16; ++i) results_host[i] = 0.f;
  double clock_hz = 0.0;
  for (int mode = 0; mode < 6 && e == cudaSuccess; ++mode) {
    double best_rate = 0.0, best_per_clk = 0.0;
    for (int rep = 0; rep < 4; ++rep) {  // rep 0 warms up
      cudaEventRecord(a, st);
      switch (mode) {
        case 0: peak_kernel<0><<<grid, kPeakThreads, 0, st>>>(kPeakIters, 0.f, sink, cycles); break;
        case 1: peak_kernel<1><<<grid, kPeakThreads, 0, st>>>(kPeakIters, 0.f, sink, cycles); break;
        case 2: peak_kernel<2><<<grid, kPeakThreads, 0, st>>>(kPeakIters, 0.f, sink, cycles); break;
        case 3: peak_kernel<3><<<grid, kPeakThreads, 0, st>>>(kPeakIters, 0.f, sink, cycles); break;
        case 4: peak_kernel<4><<<grid, kPeakThreads, 0, st>>>(kPeakIters, 0.f, sink, cycles); break;
        default: peak_kernel<5><<<grid, kPeakThreads, 0, st>>>(kPeakIters, 0.f, sink, cycles); break;
      }
      launched();
      cudaEventRecord(b, st);
      e = cudaEventSynchronize(b);
      if (e != cudaSuccess) break;
      float ms = 0.f;
      cudaEventElapsedTime(&ms, a, b);
      long long cn[2] = {0, 0};
      e = cudaMemcpy(cn, cycles, sizeof(cn), cudaMemcpyDeviceToHost);
      if (e != cudaSuccess) break;
      const long long cyc = cn[0];
      if (rep == 0) continue;
      const double lane_instr = (double)grid * kPeakThreads * (double)kPeakIters * kInstrPerIter[mode];
      const double rate = lane_instr / (ms * 1e-3);
      // per SM and clock: the device-wide rate over (SMs x the SM clock CTA 0 saw: clock64 ticks per %globaltimer ns)
      const double hz = cn[1] > 0 ? (double)cyc / ((double)cn[1] * 1e-9) : 0.0;
      const double per_clk = hz > 0.0 ? rate / ((double)sms * hz) : 0.0;
      if (rate > best_rate) { best_rate = rate; best_per_clk = per_clk; clock_hz = hz; }
    }
    results_host[mode] = (float)best_rate;
    results_host[8 + mode] = (float)best_per_clk;
    if (mode == 0) results_host[6] = (float)clock_hz;
  }
  results_host[7] = (float)sms;
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  return e;
}

}  // namespace gabsplat
