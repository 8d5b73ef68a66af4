// dfp_joseph.cuh - forward projection and its pose gradient with JOSEPH weights (DFP_FLAG_JOSEPH).
//
// Joseph's projector (BASELINE.json north_star: "trilinear or Joseph interpolation"): the ray is stepped from
// voxel-centre plane to voxel-centre plane along its DRIVING axis a* = argmax_a |e'_a| (object frame); in each plane
// the volume is interpolated bilinearly (zero-extended) at the intersection point and every plane carries the path
// length between consecutive planes, v_a* / |e'_a*|:   a^ij = (v_a* / |e'_a*|) x bilinear weight of voxel j.
// The gradient follows the paper's discretisation literally, as the Siddon kernels do (Eq.19-20 :179-191, :189):
// g_j = central differences of the zero-extended voxel values, lever arm at the voxel centre r'_j, on grid voxels;
//   A_i = sum_j a^ij g_j,  B_i = sum_j a^ij r'_j x g_j   -> six running sums per ray, then the common reduction.
//
// One thread per ray; per-ray set-up in fp64 (driving axis, plane range with t > 0 and the bilinear support inside
// reach, start and increment of the two in-plane coordinates), planes marched in fp32 on centred indices.  Values
// are read straight from the caller's volume through L1 with bound predicates: a first, plain kernel for the
// "next" row.  The body is instantiated per driving axis so that every index is static.
#pragma once
#include <cuda_runtime.h>

#include "dfp_kernels.cuh"

namespace dfp {

struct JosephRay {
  int axis;                 // driving axis a*
  int k0, k1;               // planes k0..k1 (inclusive) can contribute; k1 < k0: none
  float pb0, dpb, pd0, dpd; // in-plane continuous indices, CENTRED (minus (n-1)/2): p(k) = p0 + k dp
  float wlen;               // v_a* / |e'_a*|
};

__device__ __forceinline__ JosephRay joseph_setup(const FwdGeom& G, const FwdView& V, int iu, int iv) {
  const double dx = V.d0[0] + iu * V.du[0] + iv * V.dv[0];
  const double dy = V.d0[1] + iu * V.du[1] + iv * V.dv[1];
  const double dz = V.d0[2] + iu * V.du[2] + iv * V.dv[2];
  const double inv = 1.0 / sqrt(dx * dx + dy * dy + dz * dz);
  const double e[3] = {dx * inv, dy * inv, dz * inv};
  const int n[3] = {G.L.nx, G.L.ny, G.L.nz};
  const double v[3] = {(double)G.vx, (double)G.vy, (double)G.vz}, c[3] = {(double)G.cx, (double)G.cy, (double)G.cz};
  int a = 0;
  if (fabs(e[1]) > fabs(e[a])) a = 1;
  if (fabs(e[2]) > fabs(e[a])) a = 2;
  const int b = (a + 1) % 3, d = (a + 2) % 3;
  JosephRay r;
  r.axis = a;
  r.wlen = (float)(v[a] / fabs(e[a]));
  const double x0 = c[a] - 0.5 * (n[a] - 1) * v[a];             // plane k = 0
  const double t0 = (x0 - V.src[a]) / e[a], dt = v[a] / e[a];   // t_k = t0 + k dt
  double klo = 0.0, khi = (double)(n[a] - 1);
  // t_k > 0
  if (dt > 0) klo = fmax(klo, floor(-t0 / dt) + 1.0); else khi = fmin(khi, ceil(-t0 / dt) - 1.0);
  // in-plane coordinate inside the support of the zero-extended bilinear interpolant: -1 < p < n
  double p0[2], dp[2];
  const int ax2[2] = {b, d};
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    const int m = ax2[q];
    p0[q] = (V.src[m] + t0 * e[m] - c[m]) / v[m];               // centred index at k = 0
    dp[q] = dt * e[m] / v[m];
    const double lo = -0.5 * (n[m] - 1) - 1.0, hi = 0.5 * (n[m] - 1) + 1.0;
    if (fabs(dp[q]) > 1e-300) {
      double ka = (lo - p0[q]) / dp[q], kb = (hi - p0[q]) / dp[q];
      if (ka > kb) { const double s = ka; ka = kb; kb = s; }
      klo = fmax(klo, ceil(ka));
      khi = fmin(khi, floor(kb));
    } else if (p0[q] <= lo || p0[q] >= hi) {
      khi = -1.0; klo = 0.0;
    }
  }
  r.k0 = (int)klo;
  r.k1 = khi >= klo ? (int)khi : (int)klo - 1;
  r.pb0 = (float)p0[0]; r.dpb = (float)dp[0];
  r.pd0 = (float)p0[1]; r.dpd = (float)dp[1];
  return r;
}

// voxel value with zero extension along the two in-plane axes (the driving-axis index is always in range)
__device__ __forceinline__ float jload(const float* __restrict__ vol, long long off, bool ok) {
  return ok ? __ldg(vol + off) : 0.f;
}

// A = driving axis; B = (A+1)%3, D = (A+2)%3.  GRAD = false: returns the projection in acc[0].
template <int A, bool GRAD>
__device__ __forceinline__ void joseph_march(const FwdGeom& G, const JosephRay& r, const float* __restrict__ vol,
                                             float* acc) {
  constexpr int B = (A + 1) % 3, D = (A + 2) % 3;
  const int n[3] = {G.L.nx, G.L.ny, G.L.nz};
  const long long S[3] = {1, G.L.nx, (long long)G.L.nx * G.L.ny};
  const float vv[3] = {G.vx, G.vy, G.vz}, cc[3] = {G.cx, G.cy, G.cz}, sg[3] = {G.sgx, G.sgy, G.sgz};
  const float hb = 0.5f * (float)(n[B] - 1), hd = 0.5f * (float)(n[D] - 1), ha = 0.5f * (float)(n[A] - 1);
  float sum = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f, b0 = 0.f, b1 = 0.f, b2 = 0.f;
  for (int k = r.k0; k <= r.k1; ++k) {
    const float kf = (float)k;
    const float qb = fmaf(kf, r.dpb, r.pb0) + hb, qd = fmaf(kf, r.dpd, r.pd0) + hd;     // continuous indices
    const float fb = floorf(qb), fd = floorf(qd);
    const float wb1 = qb - fb, wd1 = qd - fd, wb0 = 1.f - wb1, wd0 = 1.f - wd1;
    const int ib = (int)fb, id = (int)fd;
    const long long base = (long long)k * S[A] + (long long)ib * S[B] + (long long)id * S[D];
    const bool okb0 = (unsigned)ib < (unsigned)n[B], okb1 = (unsigned)(ib + 1) < (unsigned)n[B];
    const bool okd0 = (unsigned)id < (unsigned)n[D], okd1 = (unsigned)(id + 1) < (unsigned)n[D];
    if (!GRAD) {
      const float v00 = jload(vol, base, okb0 && okd0), v10 = jload(vol, base + S[B], okb1 && okd0);
      const float v01 = jload(vol, base + S[D], okb0 && okd1), v11 = jload(vol, base + S[B] + S[D], okb1 && okd1);
      sum += wd0 * (wb0 * v00 + wb1 * v10) + wd1 * (wb0 * v01 + wb1 * v11);
    } else {
      // the in-plane 4 x 4 neighbourhood without its corners (12 voxels) and the 2 x 2 block in planes k-1, k+1
      // (8 voxels), each loaded once; zero extension by predicate
      const bool okbm = (unsigned)(ib - 1) < (unsigned)n[B], okb2 = (unsigned)(ib + 2) < (unsigned)n[B];
      const bool okdm = (unsigned)(id - 1) < (unsigned)n[D], okd2 = (unsigned)(id + 2) < (unsigned)n[D];
      const bool okam = k > 0, okap = k + 1 < n[A];
      const bool okb[4] = {okbm, okb0, okb1, okb2}, okd[4] = {okdm, okd0, okd1, okd2};
      float P[4][4];                                   // P[jd+1][jb+1] = voxel (ib+jb, id+jd), jb, jd in -1..2
#pragma unroll
      for (int jd = 0; jd < 4; ++jd)
#pragma unroll
        for (int jb = 0; jb < 4; ++jb) {
          const bool corner = (jd == 0 || jd == 3) && (jb == 0 || jb == 3);
          P[jd][jb] = corner ? 0.f : jload(vol, base + (jb - 1) * S[B] + (jd - 1) * S[D], okb[jb] && okd[jd]);
        }
#pragma unroll
      for (int jd = 0; jd < 2; ++jd)
#pragma unroll
        for (int jb = 0; jb < 2; ++jb) {
          const bool ok = okb[jb + 1] && okd[jd + 1];
          const float w = ok ? (jb ? wb1 : wb0) * (jd ? wd1 : wd0) : 0.f;       // grid voxels only (O13)
          const long long o = base + jb * S[B] + jd * S[D];
          const float ga = jload(vol, o + S[A], ok && okap) - jload(vol, o - S[A], ok && okam);
          const float gb = P[jd + 1][jb + 2] - P[jd + 1][jb];
          const float gd = P[jd + 2][jb + 1] - P[jd][jb + 1];
          float g3[3], r3[3];
          g3[A] = w * ga * sg[A]; g3[B] = w * gb * sg[B]; g3[D] = w * gd * sg[D];
          r3[A] = fmaf(kf - ha, vv[A], cc[A]);
          r3[B] = fmaf((float)(ib + jb) - hb, vv[B], cc[B]);
          r3[D] = fmaf((float)(id + jd) - hd, vv[D], cc[D]);
          a0 += g3[0]; a1 += g3[1]; a2 += g3[2];
          b0 += r3[1] * g3[2] - r3[2] * g3[1];
          b1 += r3[2] * g3[0] - r3[0] * g3[2];
          b2 += r3[0] * g3[1] - r3[1] * g3[0];
        }
    }
  }
  if (!GRAD) {
    acc[0] = r.wlen * sum;
  } else {
    acc[0] = r.wlen * a0; acc[1] = r.wlen * a1; acc[2] = r.wlen * a2;
    acc[3] = r.wlen * b0; acc[4] = r.wlen * b1; acc[5] = r.wlen * b2;
  }
}

template <bool GRAD>
__device__ __forceinline__ void joseph_ray(const FwdGeom& G, const JosephRay& r, const float* __restrict__ vol,
                                           float* acc) {
  if (r.axis == 0) joseph_march<0, GRAD>(G, r, vol, acc);
  else if (r.axis == 1) joseph_march<1, GRAD>(G, r, vol, acc);
  else joseph_march<2, GRAD>(G, r, vol, acc);
}

__global__ void __launch_bounds__(kFwdThreads) joseph_fwd_kernel(FwdGeom G, const FwdView* __restrict__ views,
                                                                 const float* __restrict__ vol,
                                                                 float* __restrict__ proj) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  if (iu >= G.nu || iv >= G.nv) return;
  const JosephRay r = joseph_setup(G, views[view], iu, iv);
  float acc[1] = {0.f};
  joseph_ray<false>(G, r, vol, acc);
  proj[((size_t)view * G.nv + iv) * G.nu + iu] = acc[0];
}

__global__ void __launch_bounds__(kFwdThreads) joseph_grad_kernel(FwdGeom G, const FwdView* __restrict__ views,
                                                                  const float* __restrict__ vol,
                                                                  const float* __restrict__ upstream,
                                                                  float* __restrict__ partials) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  const bool live = iu < G.nu && iv < G.nv;
  float out[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (live) {
    const JosephRay r = joseph_setup(G, views[view], iu, iv);
    joseph_ray<true>(G, r, vol, out);
    const float w = __ldg(upstream + ((size_t)view * G.nv + iv) * G.nu + iu);
#pragma unroll
    for (int q = 0; q < 6; ++q) out[q] *= w;
  }
  reduce6_to_partials<kFwdThreads>(out, partials, view);
}

}  // namespace dfp
