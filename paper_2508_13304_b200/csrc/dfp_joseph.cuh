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
// floor() of the two in-plane coordinates by the magic-number addition of the trilinear kernels (no F2I / FRND):
// t = (q - 1/2) + 1.5 * 2^23 holds rint(q - 1/2) in its low mantissa bits, which is floor(q) except at integers,
// where either neighbour with weight 0 / 1 gives the same interpolant.
template <int A, bool GRAD>
__device__ __forceinline__ void joseph_march(const FwdGeom& G, const JosephRay& r, const float4* __restrict__ pvol,
                                             const float4* __restrict__ gvol, float* acc) {
  constexpr int B = (A + 1) % 3, D = (A + 2) % 3;
  const int n[3] = {G.L.nx, G.L.ny, G.L.nz};
  const float vv[3] = {G.vx, G.vy, G.vz}, cc[3] = {G.cx, G.cy, G.cz};
  const float hb = 0.5f * (float)(n[B] - 1), hd = 0.5f * (float)(n[D] - 1), ha = 0.5f * (float)(n[A] - 1);
  const float pb = r.pb0 + (hb - 0.5f), pd = r.pd0 + (hd - 0.5f);          // continuous index minus 1/2 at k = 0
  float sum = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f, b0 = 0.f, b1 = 0.f, b2 = 0.f;
  float kf = (float)r.k0;
  const GradBricks Bk = GradBricks::make(G.L.nx, G.L.ny, G.L.nz);
#pragma unroll(GRAD ? 1 : 4)
  for (int k = r.k0; k <= r.k1; ++k, kf += 1.0f) {
    const float qb = fmaf(kf, r.dpb, pb), qd = fmaf(kf, r.dpd, pd);
    const float tb = qb + kMagic, td = qd + kMagic;
    const float wb1 = (qb - (tb - kMagic)) + 0.5f, wd1 = (qd - (td - kMagic)) + 0.5f;
    const float wb0 = 1.f - wb1, wd0 = 1.f - wd1;
    const int ib = __float_as_int(tb) - kMagicBits, id = __float_as_int(td) - kMagicBits;
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
        const float4 c1 = ldg4(pvol + (idx + ((Z & 1u) ? 2u * G.L.bz + 4u : 4u)));  // slice z + 1
        if (A == 0) { v00 = c0.x; v10 = c0.z; v01 = c1.x; v11 = c1.z; }           // B = y, D = z
        else        { v00 = c0.x; v10 = c1.x; v01 = c0.y; v11 = c1.y; }           // B = z, D = x
      }
      sum += wd0 * (wb0 * v00 + wb1 * v10) + wd1 * (wb0 * v01 + wb1 * v11);
    } else {
      // g_j of the four voxels from the per-voxel gradient volume (grad_volume_kernel); grid voxels only (O13).
      // The four lever arms differ by one pitch along B and D:  sum_j w_j r'_j x g_j =
      //   r'_00 x S + v_B e_B x S_b + v_D e_D x S_d,   S = sum_j w_j g_j,  S_b / S_d = the jb = 1 / jd = 1 parts.
      const bool okb0 = (unsigned)ib < (unsigned)n[B], okb1 = (unsigned)(ib + 1) < (unsigned)n[B];
      const bool okd0 = (unsigned)id < (unsigned)n[D], okd1 = (unsigned)(id + 1) < (unsigned)n[D];
      int FA, FB0, FB1, FD0, FD1;
      if (A == 0) { FA = Bk.FX(k); FB0 = Bk.FY(ib); FB1 = Bk.FY(ib + 1); FD0 = Bk.FZ(id); FD1 = Bk.FZ(id + 1); }
      else if (A == 1) { FA = Bk.FY(k); FB0 = Bk.FZ(ib); FB1 = Bk.FZ(ib + 1); FD0 = Bk.FX(id); FD1 = Bk.FX(id + 1); }
      else { FA = Bk.FZ(k); FB0 = Bk.FX(ib); FB1 = Bk.FX(ib + 1); FD0 = Bk.FY(id); FD1 = Bk.FY(id + 1); }
      const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
      const float4 g00 = (okb0 && okd0) ? ldg4(gvol + (FA + FB0 + FD0)) : z4;
      const float4 g10 = (okb1 && okd0) ? ldg4(gvol + (FA + FB1 + FD0)) : z4;
      const float4 g01 = (okb0 && okd1) ? ldg4(gvol + (FA + FB0 + FD1)) : z4;
      const float4 g11 = (okb1 && okd1) ? ldg4(gvol + (FA + FB1 + FD1)) : z4;
      const float w00 = wb0 * wd0, w10 = wb1 * wd0, w01 = wb0 * wd1, w11 = wb1 * wd1;
      float S[3], Sb[3], Sd[3], r3[3];
      Sb[0] = fmaf(w10, g10.x, w11 * g11.x); Sb[1] = fmaf(w10, g10.y, w11 * g11.y); Sb[2] = fmaf(w10, g10.z, w11 * g11.z);
      Sd[0] = fmaf(w01, g01.x, w11 * g11.x); Sd[1] = fmaf(w01, g01.y, w11 * g11.y); Sd[2] = fmaf(w01, g01.z, w11 * g11.z);
      S[0] = fmaf(w00, g00.x, fmaf(w01, g01.x, Sb[0]));
      S[1] = fmaf(w00, g00.y, fmaf(w01, g01.y, Sb[1]));
      S[2] = fmaf(w00, g00.z, fmaf(w01, g01.z, Sb[2]));
      r3[A] = fmaf(kf - ha, vv[A], cc[A]);
      r3[B] = fmaf((float)ib - hb, vv[B], cc[B]);
      r3[D] = fmaf((float)id - hd, vv[D], cc[D]);
      float bq[3];
      bq[0] = r3[1] * S[2] - r3[2] * S[1];
      bq[1] = r3[2] * S[0] - r3[0] * S[2];
      bq[2] = r3[0] * S[1] - r3[1] * S[0];
      // (A, B, D) is a cyclic permutation of (x, y, z):  e_B x S = S_D e_A - S_A e_D,   e_D x S = S_A e_B - S_B e_A
      bq[A] = fmaf(vv[B], Sb[D], bq[A]);
      bq[D] = fmaf(-vv[B], Sb[A], bq[D]);
      bq[B] = fmaf(vv[D], Sd[A], bq[B]);
      bq[A] = fmaf(-vv[D], Sd[B], bq[A]);
      a0 += S[0]; a1 += S[1]; a2 += S[2];
      b0 += bq[0]; b1 += bq[1]; b2 += bq[2];
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
