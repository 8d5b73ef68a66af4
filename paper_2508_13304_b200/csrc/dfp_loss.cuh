// dfp_loss.cuh - the loss of the paper's 2D/3D registration task on the device (Eq.25 :230-235):
// normalised cross-correlation of each view's projection l with its measured image b, and its pose gradient from the
// three moments of dfp_forward_fused_moments.  dNCC/dl_i = alpha + beta l_i + gamma b_i with
//   gamma = 1 / (|l~| |b~|),  beta = -NCC / |l~|^2,  alpha = -gamma mean(b) - beta mean(l)      (l~ = l - mean(l)),
// so dNCC/dtheta = alpha m0 + beta m1 + gamma m2 (Eq.20 :185 with that upstream).  Sums in fp64, fixed order.
#pragma once
#include <cuda_runtime.h>

namespace dfp {

constexpr int kNccThreads = 256;
constexpr int kNccBlocks = 64;           // partial sums per view

// partial[view][block][5] = sums of l, b, l l, b b, l b over the block's grid-stride share of the view's pixels
__global__ void __launch_bounds__(kNccThreads) ncc_partial_kernel(size_t npix, const float* __restrict__ proj,
                                                                  const float* __restrict__ target,
                                                                  double* __restrict__ partial) {
  const int view = blockIdx.y;
  const float* l = proj + (size_t)view * npix;
  const float* b = target + (size_t)view * npix;
  double s[5] = {0, 0, 0, 0, 0};
  for (size_t i = (size_t)blockIdx.x * kNccThreads + threadIdx.x; i < npix; i += (size_t)gridDim.x * kNccThreads) {
    const double x = (double)__ldg(l + i), y = (double)__ldg(b + i);
    s[0] += x; s[1] += y; s[2] = fma(x, x, s[2]); s[3] = fma(y, y, s[3]); s[4] = fma(x, y, s[4]);
  }
  __shared__ double sh[kNccThreads / 32][5];
#pragma unroll
  for (int q = 0; q < 5; ++q)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s[q] += __shfl_xor_sync(0xffffffffu, s[q], o);
  if ((threadIdx.x & 31) == 0)
#pragma unroll
    for (int q = 0; q < 5; ++q) sh[threadIdx.x >> 5][q] = s[q];
  __syncthreads();
  if (threadIdx.x < 5) {
    double t = 0;
    for (int w = 0; w < kNccThreads / 32; ++w) t += sh[w][threadIdx.x];
    partial[((size_t)view * gridDim.x + blockIdx.x) * 5 + threadIdx.x] = t;
  }
}

// one warp per view: finish the sums, NCC, coefficients, gradient
__global__ void __launch_bounds__(32) ncc_finish_kernel(size_t npix, int nblk, const double* __restrict__ partial,
                                                        const float* __restrict__ moments, float* __restrict__ ncc,
                                                        float* __restrict__ grad) {
  const int view = blockIdx.x, lane = threadIdx.x;
  double s[5] = {0, 0, 0, 0, 0};
  for (int b = lane; b < nblk; b += 32)
#pragma unroll
    for (int q = 0; q < 5; ++q) s[q] += partial[((size_t)view * nblk + b) * 5 + q];
#pragma unroll
  for (int q = 0; q < 5; ++q)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s[q] += __shfl_xor_sync(0xffffffffu, s[q], o);
  const double n = (double)npix, ml = s[0] / n, mb = s[1] / n;
  const double vl = s[2] - n * ml * ml, vb = s[3] - n * mb * mb, cov = s[4] - n * ml * mb;   // |l~|^2, |b~|^2, l~.b~
  const bool ok = vl > 0.0 && vb > 0.0;
  const double sa = sqrt(vl), sb = sqrt(vb);
  const double c = ok ? cov / (sa * sb) : 0.0;
  const double gam = ok ? 1.0 / (sa * sb) : 0.0, bet = ok ? -c / vl : 0.0, alp = -gam * mb - bet * ml;
  if (lane == 0) ncc[view] = (float)c;
  if (lane < 6) {
    const float* m = moments + (size_t)view * 18;
    grad[view * 6 + lane] = (float)(alp * (double)m[lane] + bet * (double)m[6 + lane] + gam * (double)m[12 + lane]);
  }
}

}  // namespace dfp
