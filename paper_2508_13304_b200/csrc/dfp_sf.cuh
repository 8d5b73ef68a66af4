// dfp_sf.cuh - the four operations with SEPARABLE-FOOTPRINT weights (DFP_FLAG_SF, PAPER.md :213 ref [29],
// Tables III / IV rows SF; reading DESIGN.md U16).  Voxel-driven, everything from Eq.13's Jacobian at the voxel centre:
//   (u_j, v_j) = p(r'_j),  J = d(u, v)/dr'  (pixel-index units per mm, P_eff = P [R | t]);
//   widths wu_k = |J_uk| v_k, wv_k = |J_vk| v_k;  T(u), R(v) = unit-area trapezoids from the two widest rects of each axis;
//   a^ij = v_x v_y v_z sqrt(det J J^T) * int_pixel T du * int_pixel R dv.
// One thread per voxel, the views inside (the footprint of a (voxel, view) is computed once and serves every pixel it
// covers; the volume is written once; per-view 6-vectors are reduced per block).  fp64 for the footprint (a weight is
// a difference of trapezoid integrals at u_j -+ a few pixels).
//   MODE 0  forward     l_i += a^ij mu_j         scatter with atomicAdd (fp32; the paper's own kernels accumulate with
//                                                atomics, :207) into the zeroed projections - the one non-deterministic
//                                                summation order of the library, at the 1e-7 level
//   MODE 1  back        mu_j = sum_i a^ij l_i    gather: the exact transpose
//   MODE 2  forward pose gradient  sum_j (A^T w)_j G_f^j, G_f^j per voxel (Eq.19-20): gather the upstream image
//   MODE 3  back pose gradient     sum_ij a^ij w_j (D_u^i J_u(r_j) + D_v^i J_v(r_j))   (Eq.22, per-pixel G_b^i)
#pragma once
#include <cuda_runtime.h>

#include "dfp_dd.cuh"

namespace dfp {

// int_{-inf}^{x} of the unit-area trapezoid centred at c with base b >= top t >= 0
__device__ __forceinline__ double sf_cdf(double c, double b, double t, double x) {
  const double h = 2.0 / (b + t);
  const double x0 = c - 0.5 * b, x1 = c - 0.5 * t, x2 = c + 0.5 * t, x3 = c + 0.5 * b;
  double s = h * (fmin(fmax(x, x1), x2) - x1);
  if (x1 > x0) { const double r = fmin(fmax(x, x0), x1) - x0; s += h * r * r / (2.0 * (x1 - x0)); }
  if (x3 > x2) { const double r = fmin(fmax(x, x2), x3) - x2; s += h * (r - r * r / (2.0 * (x3 - x2))); }
  return s;
}
__device__ __forceinline__ void sf_two_widest(double a, double b, double c, double* base, double* top) {
  const double hi = fmax(a, fmax(b, c)), lo = fmin(a, fmin(b, c)), mid = a + b + c - hi - lo;
  *base = hi + mid; *top = hi - mid;
}

struct SfFoot {                 // footprint of one (voxel, view)
  double uj, vj, bu, tu, bv, tv, M;
  double Ju[3], Jv[3];
  int iu0, iu1, iv0, iv1;
  bool ok;
};
__device__ __forceinline__ SfFoot sf_footprint(const DdGeom& G, const double (*E)[4], const double* r) {
  SfFoot f;
  const double up = fma(E[0][0], r[0], fma(E[0][1], r[1], fma(E[0][2], r[2], E[0][3])));
  const double vp = fma(E[1][0], r[0], fma(E[1][1], r[1], fma(E[1][2], r[2], E[1][3])));
  const double wp = fma(E[2][0], r[0], fma(E[2][1], r[1], fma(E[2][2], r[2], E[2][3])));
  f.ok = wp > 0.0;
  const double rw = 1.0 / wp;
  f.uj = up * rw; f.vj = vp * rw;
  double wu[3], wv[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    f.Ju[k] = (E[0][k] - E[2][k] * f.uj) * rw;          // Eq.13: (P_1k w' - P_3k u') / w'^2
    f.Jv[k] = (E[1][k] - E[2][k] * f.vj) * rw;
    wu[k] = fabs(f.Ju[k]) * G.v[k]; wv[k] = fabs(f.Jv[k]) * G.v[k];
  }
  const double guu = f.Ju[0] * f.Ju[0] + f.Ju[1] * f.Ju[1] + f.Ju[2] * f.Ju[2];
  const double gvv = f.Jv[0] * f.Jv[0] + f.Jv[1] * f.Jv[1] + f.Jv[2] * f.Jv[2];
  const double guv = f.Ju[0] * f.Jv[0] + f.Ju[1] * f.Jv[1] + f.Ju[2] * f.Jv[2];
  f.M = G.v[0] * G.v[1] * G.v[2] * sqrt(fmax(guu * gvv - guv * guv, 0.0));
  sf_two_widest(wu[0], wu[1], wu[2], &f.bu, &f.tu);
  sf_two_widest(wv[0], wv[1], wv[2], &f.bv, &f.tv);
  if (!(f.bu > 0.0) || !(f.bv > 0.0) || !(f.M > 0.0) || !(f.bu < 1e6) || !(f.bv < 1e6)) f.ok = false;
  if (f.ok) {
    f.iu0 = max((int)floor(f.uj - 0.5 * f.bu + 0.5), 0); f.iu1 = min((int)floor(f.uj + 0.5 * f.bu + 0.5), G.nu - 1);
    f.iv0 = max((int)floor(f.vj - 0.5 * f.bv + 0.5), 0); f.iv1 = min((int)floor(f.vj + 0.5 * f.bv + 0.5), G.nv - 1);
  } else {
    f.iu0 = f.iv0 = 0; f.iu1 = f.iv1 = -1;
  }
  return f;
}

constexpr int kSfThreads = 256;
template <int MODE>
__global__ void __launch_bounds__(kSfThreads) sf_kernel(DdGeom G, int n_views, int accumulate,
                                                        const DdView* __restrict__ views,
                                                        const float* __restrict__ vol,      // MODE 0, 2: the volume
                                                        const float* __restrict__ img,      // MODE 1, 3: projections; 2: upstream
                                                        const float* __restrict__ upvol,    // MODE 3: upstream volume
                                                        float* __restrict__ out) {
  const size_t nvox = (size_t)G.n[0] * G.n[1] * G.n[2];
  const size_t j = (size_t)blockIdx.x * kSfThreads + threadIdx.x;
  const bool live = j < nvox;
  int xyz[3] = {0, 0, 0};
  if (live) { xyz[0] = (int)(j % G.n[0]); xyz[1] = (int)((j / G.n[0]) % G.n[1]); xyz[2] = (int)(j / ((size_t)G.n[0] * G.n[1])); }
  __shared__ double E[3][4];
  __shared__ float red[kSfThreads / 32][6];
  double r[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) r[k] = G.c[k] + ((double)xyz[k] - G.h[k]) * G.v[k];
  const float rx = (float)r[0], ry = (float)r[1], rz = (float)r[2];
  float mu = 0.f, gx = 0.f, gy = 0.f, gz = 0.f, wj = 0.f;
  if (live && (MODE == 0 || MODE == 2)) {
    const size_t sy = (size_t)G.n[0], sz = (size_t)G.n[0] * G.n[1];
    mu = __ldg(vol + j);
    if (MODE == 2) {          // g_j: central differences of the zero-extended voxel values (:183)
      gx = ((xyz[0] + 1 < G.n[0] ? __ldg(vol + j + 1) : 0.f) - (xyz[0] > 0 ? __ldg(vol + j - 1) : 0.f)) / (2.f * G.vx);
      gy = ((xyz[1] + 1 < G.n[1] ? __ldg(vol + j + sy) : 0.f) - (xyz[1] > 0 ? __ldg(vol + j - sy) : 0.f)) / (2.f * G.vy);
      gz = ((xyz[2] + 1 < G.n[2] ? __ldg(vol + j + sz) : 0.f) - (xyz[2] > 0 ? __ldg(vol + j - sz) : 0.f)) / (2.f * G.vz);
    }
  }
  if (live && MODE == 3) wj = __ldg(upvol + j);
  bool work = live;
  if (MODE == 0) work = live && mu != 0.f;
  if (MODE == 2) work = live && (gx != 0.f || gy != 0.f || gz != 0.f);
  if (MODE == 3) work = live && wj != 0.f;
  double acc = (MODE == 1 && accumulate && live) ? (double)out[j] : 0.0;
  for (int view = 0; view < n_views; ++view) {
    __syncthreads();
    if (threadIdx.x < 12) E[threadIdx.x >> 2][threadIdx.x & 3] = views[view].P[threadIdx.x >> 2][threadIdx.x & 3];
    __syncthreads();
    double s0 = 0.0, s1 = 0.0;
    SfFoot f;
    f.ok = false;
    if (work) {
      f = sf_footprint(G, E, r);
      const size_t base = (size_t)view * G.nu * G.nv;
      for (int iv = f.iv0; iv <= f.iv1; ++iv) {
        const double fv = sf_cdf(f.vj, f.bv, f.tv, iv + 0.5) - sf_cdf(f.vj, f.bv, f.tv, iv - 0.5);
        if (!(fv > 0.0)) continue;
        for (int iu = f.iu0; iu <= f.iu1; ++iu) {
          const double fu = sf_cdf(f.uj, f.bu, f.tu, iu + 0.5) - sf_cdf(f.uj, f.bu, f.tu, iu - 0.5);
          if (!(fu > 0.0)) continue;
          const double w = f.M * fu * fv;
          const size_t pix = base + (size_t)iv * G.nu + iu;
          if (MODE == 0) {
            atomicAdd(out + pix, (float)(w * (double)mu));
          } else if (MODE == 1 || MODE == 2) {
            s0 = fma(w, (double)__ldg(img + pix), s0);
          } else {
            const float* p = img + pix;
            const float lp = iu + 1 < G.nu ? __ldg(p + 1) : 0.f, lm = iu > 0 ? __ldg(p - 1) : 0.f;
            const float tp = iv + 1 < G.nv ? __ldg(p + G.nu) : 0.f, tm = iv > 0 ? __ldg(p - G.nu) : 0.f;
            s0 = fma(w, 0.5 * ((double)lp - (double)lm), s0);
            s1 = fma(w, 0.5 * ((double)tp - (double)tm), s1);
          }
        }
      }
    }
    if (MODE == 1) acc += s0;
    if (MODE == 2 || MODE == 3) {
      float s6[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      if (work && f.ok) {
        float qx, qy, qz;
        if (MODE == 2) {        // (A^T w)_j g_j
          const float s = (float)s0;
          qx = s * gx; qy = s * gy; qz = s * gz;
        } else {                // w_j (su J_u + sv J_v), object frame
          qx = wj * (float)(s0 * f.Ju[0] + s1 * f.Jv[0]);
          qy = wj * (float)(s0 * f.Ju[1] + s1 * f.Jv[1]);
          qz = wj * (float)(s0 * f.Ju[2] + s1 * f.Jv[2]);
        }
        s6[0] = qx; s6[1] = qy; s6[2] = qz;
        s6[3] = ry * qz - rz * qy; s6[4] = rz * qx - rx * qz; s6[5] = rx * qy - ry * qx;
      }
#pragma unroll
      for (int q = 0; q < 6; ++q) {
        float v = s6[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        s6[q] = v;
      }
      const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
      if (lane == 0) {
#pragma unroll
        for (int q = 0; q < 6; ++q) red[warp][q] = s6[q];
      }
      __syncthreads();
      if (threadIdx.x < 6) {
        float t = 0.f;
#pragma unroll
        for (int wI = 0; wI < kSfThreads / 32; ++wI) t += red[wI][threadIdx.x];
        // MODE 2: partials[view][block][6] (fwd_contract_kernel); MODE 3: partials[block][view][6] (bp_contract_kernel)
        const size_t at = MODE == 2 ? ((size_t)view * gridDim.x + blockIdx.x) : ((size_t)blockIdx.x * n_views + view);
        out[at * 6 + threadIdx.x] = t;
      }
    }
  }
  if (MODE == 1 && live) out[j] = (float)acc;
}

}  // namespace dfp
