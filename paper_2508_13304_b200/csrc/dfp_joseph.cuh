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
// reach, start and increment of the two in-plane coordinates), planes marched in fp32 on centred indices.  The
// forward kernel reads the packed quad cells of the trilinear gather path (one or two 16-byte reads per plane, zero
// border instead of bound predicates); the gradient kernel reads g_j of the
// four voxels from the per-voxel gradient volume (dfp_kernels.cuh: grad_volume_kernel), one float4 each.  Kernels
// for the "next" row.  The body is instantiated per driving axis so that every index is static.
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

// A = driving axis; B = (A+1)%3, D = (A+2)%3.  GRAD = false: returns the projection in acc[0].
template <int A, bool GRAD>
__device__ __forceinline__ void joseph_march(const FwdGeom& G, const JosephRay& r, const float4* __restrict__ pvol,
                                             const float4* __restrict__ gvol, float* acc) {
  constexpr int B = (A + 1) % 3, D = (A + 2) % 3;
  const int n[3] = {G.L.nx, G.L.ny, G.L.nz};
  const float vv[3] = {G.vx, G.vy, G.vz}, cc[3] = {G.cx, G.cy, G.cz};
  const float hb = 0.5f * (float)(n[B] - 1), hd = 0.5f * (float)(n[D] - 1), ha = 0.5f * (float)(n[A] - 1);
  float sum = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f, b0 = 0.f, b1 = 0.f, b2 = 0.f;
  for (int k = r.k0; k <= r.k1; ++k) {
    const float kf = (float)k;
    const float qb = fmaf(kf, r.dpb, r.pb0) + hb, qd = fmaf(kf, r.dpd, r.pd0) + hd;     // continuous indices
    const float fb = floorf(qb), fd = floorf(qd);
    const float wb1 = qb - fb, wd1 = qd - fd, wb0 = 1.f - wb1, wd0 = 1.f - wd1;
    const int ib = (int)fb, id = (int)fd;
    const bool okb0 = (unsigned)ib < (unsigned)n[B], okb1 = (unsigned)(ib + 1) < (unsigned)n[B];
    const bool okd0 = (unsigned)id < (unsigned)n[D], okd1 = (unsigned)(id + 1) < (unsigned)n[D];
    if (!GRAD) {
      // the 2 x 2 in-plane voxels from the packed quad cells (pack_volume_kernel: cell (x,y,z) holds voxels
      // (x,y), (x+1,y), (x,y+1), (x+1,y+1) of slice z; zero border of kPad cells, so no bound predicates):
      // driving axis z: one cell; x or y: the cells of two consecutive slices, two of their four values each
      int x, y, z;
      if (A == 0) { x = k; y = ib; z = id; } else if (A == 1) { x = id; y = k; z = ib; } else { x = ib; y = id; z = k; }
      const unsigned X = (unsigned)(x + G.L.lx), Y = (unsigned)(y + G.L.ly), Z = (unsigned)(z + G.L.lz);
      const unsigned idx = X + 3u * (X & ~1u) + 2u * Y + G.L.by * (Y & ~1u) + 4u * Z + G.L.bz * (Z & ~1u);
      const float4 c0 = ldg4(pvol + idx);
      float v00, v10, v01, v11;                       // v[jb][jd]
      if (A == 2) {
        v00 = c0.x; v10 = c0.y; v01 = c0.z; v11 = c0.w;
      } else {
        const float4 c1 = ldg4(pvol + (idx + ((Z & 1u) ? 2u * G.L.bz + 4u : 4u)));      // slice z + 1
        if (A == 0) { v00 = c0.x; v10 = c0.z; v01 = c1.x; v11 = c1.z; }           // B = y, D = z
        else        { v00 = c0.x; v10 = c1.x; v01 = c0.y; v11 = c1.y; }           // B = z, D = x
      }
      sum += wd0 * (wb0 * v00 + wb1 * v10) + wd1 * (wb0 * v01 + wb1 * v11);
    } else {
      // g_j of the four voxels from the per-voxel gradient volume (grad_volume_kernel); grid voxels only (O13)
      const GradBricks Bk = GradBricks::make(G.L.nx, G.L.ny, G.L.nz);
      int FA, FB[2], FD[2];
      if (A == 0) { FA = Bk.FX(k); FB[0] = Bk.FY(ib); FB[1] = Bk.FY(ib + 1); FD[0] = Bk.FZ(id); FD[1] = Bk.FZ(id + 1); }
      else if (A == 1) { FA = Bk.FY(k); FB[0] = Bk.FZ(ib); FB[1] = Bk.FZ(ib + 1); FD[0] = Bk.FX(id); FD[1] = Bk.FX(id + 1); }
      else { FA = Bk.FZ(k); FB[0] = Bk.FX(ib); FB[1] = Bk.FX(ib + 1); FD[0] = Bk.FY(id); FD[1] = Bk.FY(id + 1); }
      const bool okb[2] = {okb0, okb1}, okd[2] = {okd0, okd1};
      float r3[3];
      r3[A] = fmaf(kf - ha, vv[A], cc[A]);
#pragma unroll
      for (int jd = 0; jd < 2; ++jd)
#pragma unroll
        for (int jb = 0; jb < 2; ++jb) {
          const bool ok = okb[jb] && okd[jd];
          const float w = (jb ? wb1 : wb0) * (jd ? wd1 : wd0);
          float4 g = make_float4(0.f, 0.f, 0.f, 0.f);
          if (ok) g = ldg4(gvol + (FA + FB[jb] + FD[jd]));
          const float g0 = w * g.x, g1 = w * g.y, g2 = w * g.z;
          r3[B] = fmaf((float)(ib + jb) - hb, vv[B], cc[B]);
          r3[D] = fmaf((float)(id + jd) - hd, vv[D], cc[D]);
          a0 += g0; a1 += g1; a2 += g2;
          b0 += r3[1] * g2 - r3[2] * g1;
          b1 += r3[2] * g0 - r3[0] * g2;
          b2 += r3[0] * g1 - r3[1] * g0;
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
__device__ __forceinline__ void joseph_ray(const FwdGeom& G, const JosephRay& r, const float4* __restrict__ pvol,
                                           const float4* __restrict__ gvol, float* acc) {
  if (r.axis == 0) joseph_march<0, GRAD>(G, r, pvol, gvol, acc);
  else if (r.axis == 1) joseph_march<1, GRAD>(G, r, pvol, gvol, acc);
  else joseph_march<2, GRAD>(G, r, pvol, gvol, acc);
}

__global__ void __launch_bounds__(kFwdThreads) joseph_fwd_kernel(FwdGeom G, const FwdView* __restrict__ views,
                                                                 const float4* __restrict__ pvol,
                                                                 float* __restrict__ proj) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  if (iu >= G.nu || iv >= G.nv) return;
  const JosephRay r = joseph_setup(G, views[view], iu, iv);
  float acc[1] = {0.f};
  joseph_ray<false>(G, r, pvol, nullptr, acc);
  proj[((size_t)view * G.nv + iv) * G.nu + iu] = acc[0];
}

__global__ void __launch_bounds__(kFwdThreads) joseph_grad_kernel(FwdGeom G, const FwdView* __restrict__ views,
                                                                  const float4* __restrict__ gvol,
                                                                  const float* __restrict__ upstream,
                                                                  float* __restrict__ partials) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  const bool live = iu < G.nu && iv < G.nv;
  float out[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (live) {
    const JosephRay r = joseph_setup(G, views[view], iu, iv);
    joseph_ray<true>(G, r, nullptr, gvol, out);
    const float w = __ldg(upstream + ((size_t)view * G.nv + iv) * G.nu + iu);
#pragma unroll
    for (int q = 0; q < 6; ++q) out[q] *= w;
  }
  reduce6_to_partials<kFwdThreads>(out, partials, view);
}

}  // namespace dfp
