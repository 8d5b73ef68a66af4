// dfp_microbench.cu - libdfp_bench.so (include/dfp_bench.h): measured denominators for the roofline of the projector
// kernels.  A PROBE, not part of the method and not part of libdfp.so: bench.py and one GPU test load it.
// Measured denominators for the roofline of the projector kernels ("micro-benchmarks
// as denominators").  The projector kernels are bound by the SM-side pipes, not by HBM:
//   * the shared-memory / LSU pipe: how many warp-wide, bank-conflict-free LDS.32 one SM retires per clock - the
//     gradient kernel needs 32 of them per warp-sample (dfp_fwd_tma.cuh), the back-projection gradient 12 per
//     voxel-view;
//   * the fp32 pipe: lane-operations per clock per SM for streams of FADD, FFMA and packed FFMA2 - the forward
//     kernels are issue-bound.
// Each kernel runs as one resident wave (blocks_per_sm blocks on every SM) timed by the host with CUDA events
// (dfp_microbench below); the per-block clock64() counts are written out for inspection only.
#include <cuda_runtime.h>

#include "../../include/dfp_bench.h"

namespace dfp {

constexpr int kMbThreads = 256;
constexpr int kMbLdsPerIter = 32;          // LDS per thread per iteration, as one gradient sample
constexpr int kMbChains = 8;               // independent dependency chains per thread (ALU kernels)

// Warp-wide LDS.32 at lane-consecutive words (bank = lane: conflict-free), 32 loads at immediate offsets from one
// index per iteration - the addressing of the staged gradient kernel.
__global__ void __launch_bounds__(kMbThreads) mb_lds_kernel(int iters, int stride, float* sink, long long* cycles) {
  __shared__ float buf[4096];
  for (int i = threadIdx.x; i < 4096; i += kMbThreads) buf[i] = (float)(i & 7);
  __syncthreads();
  unsigned idx = threadIdx.x;
  float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
    const float* c = buf + idx;
#pragma unroll
    for (int j = 0; j < kMbLdsPerIter; j += 4) {
      a0 += c[32 * j];
      a1 += c[32 * j + 32];
      a2 += c[32 * j + 64];
      a3 += c[32 * j + 96];
    }
    idx = (idx + (unsigned)stride) & 2047u;            // stride is a multiple of 32: the bank stays the lane
  }
  const long long t1 = clock64();
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
  sink[(size_t)blockIdx.x * kMbThreads + threadIdx.x] = (a0 + a1) + (a2 + a3);
}

// KIND 0: FADD (two source registers), 1: FFMA (three), 2: packed FFMA2 (two results per instruction).
template <int KIND>
__global__ void __launch_bounds__(kMbThreads) mb_alu_kernel(int iters, float a, float b, float* sink, long long* cycles) {
  float2 x[kMbChains];
#pragma unroll
  for (int i = 0; i < kMbChains; ++i) x[i] = make_float2(threadIdx.x * 1e-3f + i, i * 0.5f);
  const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int i = 0; i < kMbChains; ++i) {
        if (KIND == 0) x[i].x = x[i].x + b;
        else if (KIND == 1) x[i].x = fmaf(x[i].x, a, b);
        else x[i] = __ffma2_rn(x[i], a2, b2);
      }
    }
  }
  const long long t1 = clock64();
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < kMbChains; ++i) s += x[i].x + x[i].y;
  sink[(size_t)blockIdx.x * kMbThreads + threadIdx.x] = s;
}

}  // namespace dfp

// One resident wave of a micro-benchmark kernel, timed with CUDA events on the default stream (the kernels' own
// clock64() counts are kept for inspection only: on B200 that counter does not tick at the SM clock).
extern "C" int dfp_microbench(int kind, double* per_second) {
  using namespace dfp;
  if (!per_second) return DFP_BENCH_ERR_NULL;
  if (kind < DFP_MB_LDS || kind > DFP_MB_FFMA2) return DFP_BENCH_ERR_KIND;
  int dev = 0, n_sm = 0, R = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return DFP_BENCH_ERR_CUDA;
  if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return DFP_BENCH_ERR_CUDA;
  const void* fn = kind == DFP_MB_LDS    ? (const void*)mb_lds_kernel
                   : kind == DFP_MB_FADD ? (const void*)mb_alu_kernel<0>
                   : kind == DFP_MB_FFMA ? (const void*)mb_alu_kernel<1>
                                         : (const void*)mb_alu_kernel<2>;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&R, fn, kMbThreads, 0) != cudaSuccess) return DFP_BENCH_ERR_CUDA;
  if (R < 1 || n_sm < 1) return DFP_BENCH_ERR_CUDA;
  const int grid = n_sm * R;
  float* sink = nullptr;
  long long* cyc = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (cudaMalloc(&sink, sizeof(float) * (size_t)grid * kMbThreads) != cudaSuccess) return DFP_BENCH_ERR_CUDA;
  if (cudaMalloc(&cyc, sizeof(long long) * grid) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess ||
      cudaEventCreate(&e1) != cudaSuccess) {
    cudaFree(sink); cudaFree(cyc);
    if (e0) cudaEventDestroy(e0);
    return DFP_BENCH_ERR_CUDA;
  }
  double work = 0;        // whole grid: warp-instructions (LDS) or fp32 results (ALU)
  for (int pass = 0; pass < 2; ++pass) {                 // warm-up, then the measured wave
    const int iters = pass ? 8000 : 50;
    if (pass) cudaEventRecord(e0, 0);
    if (kind == DFP_MB_LDS) {
      mb_lds_kernel<<<grid, kMbThreads>>>(iters, 96, sink, cyc);
      work = (double)grid * iters * kMbLdsPerIter * (kMbThreads / 32);
    } else {
      if (kind == DFP_MB_FADD) mb_alu_kernel<0><<<grid, kMbThreads>>>(iters, 1.0001f, 1e-3f, sink, cyc);
      else if (kind == DFP_MB_FFMA) mb_alu_kernel<1><<<grid, kMbThreads>>>(iters, 1.0001f, 1e-3f, sink, cyc);
      else mb_alu_kernel<2><<<grid, kMbThreads>>>(iters, 1.0001f, 1e-3f, sink, cyc);
      work = (double)grid * iters * 4 * kMbChains * kMbThreads * (kind == DFP_MB_FFMA2 ? 2 : 1);
    }
    if (pass) cudaEventRecord(e1, 0);
  }
  float ms = 0.f;
  cudaError_t e = cudaEventSynchronize(e1);
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  cudaFree(sink); cudaFree(cyc);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (e != cudaSuccess || !(ms > 0.f)) return DFP_BENCH_ERR_CUDA;
  *per_second = work / ((double)ms * 1e-3);
  return DFP_BENCH_OK;
}
