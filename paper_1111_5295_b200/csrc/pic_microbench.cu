// pic_microbench.cu — the paper's micro-benchmark method ("we measure the peak performance
// of individual operations with micro-benchmarks") for the instruction classes the mover is made
// of, on the device at hand: thread-operations per clock and SM for FFMA, packed FFMA2, FMNMX
// (ALU pipe), MUFU.RSQ, DFMA, and the FFMA2 + FMNMX mix that shows the issue-slot saving of the
// packed form.  SURVEY.md 8(d) "Also measure".  Not on the hot path.
#include <cuda_runtime.h>

#include <algorithm>

#include "../../include/pic.h"

namespace {

__device__ __forceinline__ float ffma1(float a, float b, float c) {
  float d; asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c)); return d; }
__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b,
                                                    unsigned long long c) {
  unsigned long long d;
  asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ float fmax1(float a, float b) {
  float d; asm volatile("max.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b)); return d; }
__device__ __forceinline__ float rsq1(float a) {
  float d; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(d) : "f"(a)); return d; }
__device__ __forceinline__ double dfma1(double a, double b, double c) {
  double d; asm volatile("fma.rn.f64 %0, %1, %2, %3;" : "=d"(d) : "d"(a), "d"(b), "d"(c)); return d; }

constexpr int kThreads = 256, kBlocksPerSm = 8, kChains = 8;

// WHICH: 0 FFMA, 1 FFMA2, 2 FMNMX, 3 MUFU.RSQ, 4 DFMA, 5 FFMA2 + FMNMX (4 + 4 per iteration).
// kChains independent dependent chains per thread; 64 warps per SM hide the latencies.
template <int WHICH>
__global__ void __launch_bounds__(kThreads) ubench_kernel(int iters, float s, float* sink) {
  float a[kChains];
  double q[kChains];
  unsigned long long p[kChains / 2];
#pragma unroll
  for (int i = 0; i < kChains; ++i) { a[i] = s * (float)(threadIdx.x + i); q[i] = (double)a[i]; }
#pragma unroll
  for (int i = 0; i < kChains / 2; ++i)
    p[i] = ((unsigned long long)__float_as_uint(a[2 * i]) << 32) | __float_as_uint(a[2 * i + 1]);
  const float b = 1.0f + s, c = s;
  const unsigned long long pb = ((unsigned long long)__float_as_uint(b) << 32) | __float_as_uint(b);
  const unsigned long long pc = ((unsigned long long)__float_as_uint(c) << 32) | __float_as_uint(c);
  const double qb = 1.0 + (double)s, qc = (double)s;
  for (int it = 0; it < iters; ++it) {
    if (WHICH == 0) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) a[i] = ffma1(a[i], b, c);
    } else if (WHICH == 1) {
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) p[i] = ffma2(p[i], pb, pc);
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) p[i] = ffma2(p[i], pb, pc);
    } else if (WHICH == 2) {
      // max then min, so that consecutive operations of a chain cannot be merged into FMNMX3
#pragma unroll
      for (int i = 0; i < kChains; ++i) a[i] = (it & 1) ? fmax1(a[i], c) : -fmax1(-a[i], -b);
    } else if (WHICH == 3) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) a[i] = rsq1(a[i]);
    } else if (WHICH == 4) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) q[i] = dfma1(q[i], qb, qc);
    } else if (WHICH == 5) {
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) p[i] = ffma2(p[i], pb, pc);
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) a[i] = (it & 1) ? fmax1(a[i], c) : -fmax1(-a[i], -b);
    } else if (WHICH == 6) {
      // 8 scalar FFMA + 4 FMNMX: the same FMA work as mix 5 in scalar form
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) {
        p[i] = ((unsigned long long)__float_as_uint(ffma1(__uint_as_float((unsigned)(p[i] >> 32)), b, c)) << 32) |
               __float_as_uint(ffma1(__uint_as_float((unsigned)p[i]), b, c));
      }
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) a[i] = (it & 1) ? fmax1(a[i], c) : -fmax1(-a[i], -b);
    } else if (WHICH == 7) {
      // 4 scalar FFMA + 4 FMNMX
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) a[i + kChains / 2] = ffma1(a[i + kChains / 2], b, c);
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) a[i] = (it & 1) ? fmax1(a[i], c) : -fmax1(-a[i], -b);
    } else if (WHICH == 8) {
      // 2 FFMA2 + 4 scalar FFMA + 4 FMNMX
      p[0] = ffma2(p[0], pb, pc);
      p[1] = ffma2(p[1], pb, pc);
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) a[i + kChains / 2] = ffma1(a[i + kChains / 2], b, c);
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) a[i] = (it & 1) ? fmax1(a[i], c) : -fmax1(-a[i], -b);
    } else {
      // 4 FFMA2 + 2 MUFU.RSQ
#pragma unroll
      for (int i = 0; i < kChains / 2; ++i) p[i] = ffma2(p[i], pb, pc);
      a[0] = rsq1(a[0]);
      a[1] = rsq1(a[1]);
    }
  }
  float r = 0.0f;
#pragma unroll
  for (int i = 0; i < kChains; ++i) r += a[i] + (float)q[i];
#pragma unroll
  for (int i = 0; i < kChains / 2; ++i)
    r += __uint_as_float((unsigned)p[i]) + __uint_as_float((unsigned)(p[i] >> 32));
  sink[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

template <int WHICH>
cudaError_t run(int blocks, int iters, float* sink, cudaEvent_t e0, cudaEvent_t e1) {
  ubench_kernel<WHICH><<<blocks, kThreads>>>(std::max(iters / 50, 1), 1e-9f, sink);  // warm-up
  cudaEventRecord(e0);
  ubench_kernel<WHICH><<<blocks, kThreads>>>(iters, 1e-9f, sink);
  cudaEventRecord(e1);
  return cudaEventSynchronize(e1);
}

}  // namespace

extern "C" int pic_microbench(int which, int iters, double* thread_gops, int* n_sm) {
  if (which < 0 || which > 9 || iters < 1 || !thread_gops) return PIC_ERR_ARG;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
    cudaGetLastError();
    return PIC_ERR_CUDA;
  }
  const int blocks = sms * kBlocksPerSm;
  float* sink = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaError_t e = cudaMalloc(&sink, sizeof(float) * (size_t)blocks * kThreads);
  if (e == cudaSuccess) e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  if (e == cudaSuccess) {
    switch (which) {
      case 0: e = run<0>(blocks, iters, sink, e0, e1); break;
      case 1: e = run<1>(blocks, iters, sink, e0, e1); break;
      case 2: e = run<2>(blocks, iters, sink, e0, e1); break;
      case 3: e = run<3>(blocks, iters, sink, e0, e1); break;
      case 4: e = run<4>(blocks, iters, sink, e0, e1); break;
      case 5: e = run<5>(blocks, iters, sink, e0, e1); break;
      case 6: e = run<6>(blocks, iters, sink, e0, e1); break;
      case 7: e = run<7>(blocks, iters, sink, e0, e1); break;
      case 8: e = run<8>(blocks, iters, sink, e0, e1); break;
      default: e = run<9>(blocks, iters, sink, e0, e1); break;
    }
  }
  float ms = 0.0f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(sink);
  if (e != cudaSuccess || !(ms > 0.0f)) { cudaGetLastError(); return PIC_ERR_CUDA; }
  // thread-operations of the launch: blocks x kThreads x iters x kChains (FFMA2 counts as two
  // thread-operations; the mix has kChains/2 FFMA2 + kChains/2 FMNMX per iteration)
  // mixes 6-9: thread-operations per iteration = 8+4, 4+4, 4+4+4, 8+2 (FFMA2 counts two)
  const double per_iter = which == 1 ? 2.0 * kChains : which == 5 ? 1.5 * kChains
                        : which == 6 ? 12.0 : which == 7 ? 8.0 : which == 8 ? 12.0
                        : which == 9 ? 10.0 : kChains;
  *thread_gops = (double)blocks * kThreads * (double)iters * per_iter / ((double)ms * 1e6);
  if (n_sm) *n_sm = sms;
  return PIC_OK;
}
