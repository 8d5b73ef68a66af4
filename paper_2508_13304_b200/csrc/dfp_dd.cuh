// dfp_dd.cuh - the four operations with DISTANCE-DRIVEN weights (DFP_FLAG_DD, PAPER.md :213 ref [44],
// Tables III / IV rows DD; reading DESIGN.md U14).
//
// Per view (object frame): driving axis a = argmax |n'_a| of the direction source -> detector centre; the detector's
// u pairs with the in-plane axis along which the pixel step U' is longer.  Per plane k of voxel centres along a, the
// boundary mid-points (iu -+ 1/2, iv), (iu, iv -+ 1/2) of a pixel are projected from the source onto the plane; in
// continuous voxel indices they bound the pixel's footprint [B0, B1] x [D0, D1];
//   a^ij = L (|[B0,B1] n cell(jb)| / (B1 - B0)) (|[D0,D1] n cell(jd)| / (D1 - D0)),  L = v_a / |e'_a| (pixel-centre ray).
// A boundary position is AFFINE in the plane index k (position = s' + (x_a - s'_a) dir / dir_a), so a pixel carries
// four (start, increment) pairs in fp64 (a weight is a difference of positions of magnitude n/2: fp32 would leave 1e-5
// relative error per weight); per plane the four positions are re-based onto the first cell they touch and the overlaps
// are fp32 on numbers of order one.
// ALL FOUR operations are pixel-driven and share one traversal (dd_kernel<MODE>: one thread per pixel, the planes
// inside; a footprint narrower than a voxel - every BASELINE config - takes a loop-free 2 x 2 path):
//   MODE 0  l_i = sum_j a^ij mu_j
//   MODE 1  A_i = sum_j a^ij g_j, B_i = sum_j a^ij r'_j x g_j       per-voxel G_f^j (Eq.19-20), g_j from the per-voxel
//           gradient volume of grad_volume_kernel
//   MODE 2  mu_j = sum_i a^ij l_i, the EXACT transpose (Eq.21): the forward traversal with the read turned into a
//           SCATTER (the same a^ij by construction).  The scatter adds 64-bit FIXED-POINT integers (as the SF forward
//           projector, dfp_sf.cuh): integer sums do not depend on the order, so the call is deterministic; the scale
//           follows max|l| (found on the device) and a host bound on sum_i a^ij
//   MODE 3  sum_ij a^ij w_j (D_u^i J_u(r_j) + D_v^i J_v(r_j))       per-pixel G_b^i (Eq.22), D = central differences of
//           the zero-extended projection, J = Eq.13 at the voxel centre; a sum over (i, j) pairs, taken per pixel in
//           registers like MODE 1 - no scatter
#pragma once
#include <cuda_runtime.h>

#include "dfp_kernels.cuh"

namespace dfp {

struct DdGeom {
  int n[3];                // nx, ny, nz
  int nu, nv;
  double v[3], c[3], h[3]; // pitch, centre, (n - 1) / 2
  float cx, cy, cz, vx, vy, vz;
};
inline DdGeom make_dd_geom(const dfp_geometry& g) {
  DdGeom G;
  G.n[0] = g.nx; G.n[1] = g.ny; G.n[2] = g.nz; G.nu = g.nu; G.nv = g.nv;
  G.v[0] = g.vx; G.v[1] = g.vy; G.v[2] = g.vz; G.c[0] = g.cx; G.c[1] = g.cy; G.c[2] = g.cz;
  for (int a = 0; a < 3; ++a) G.h[a] = 0.5 * (G.n[a] - 1);
  G.cx = g.cx; G.cy = g.cy; G.cz = g.cz; G.vx = g.vx; G.vy = g.vy; G.vz = g.vz;
  return G;
}

// A pixel: the four boundary positions as affine functions of the plane index k.
struct DdPixel {
  double b0, db0, b1, db1, d0, dd0, d1, dd1;
  double L;
  bool ok;                 // the planes of this view are in front of the source along all five rays (for xa on the
                           // side `front_sign` of the source)
  double front_sign;
};
__device__ __forceinline__ DdPixel dd_pixel(const DdGeom& G, const DdView& W, int iu, int iv) {
  DdPixel p;
  const int a = W.a;
  const double us[5] = {(double)iu, iu - 0.5, iu + 0.5, (double)iu, (double)iu};
  const double vs[5] = {(double)iv, (double)iv, (double)iv, iv - 0.5, iv + 0.5};
  double inv[5], dax[5];
  p.ok = true;
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const double da = fma(us[q], W.Uo[a], fma(vs[q], W.Vo[a], W.X00[a])) - W.so[a];
    if (fabs(da) < 1e-300) p.ok = false;
    inv[q] = 1.0 / da;
    const int ax = q < 3 ? W.ub : W.vb;
    dax[q] = fma(us[q], W.Uo[ax], fma(vs[q], W.Vo[ax], W.X00[ax])) - W.so[ax];
  }
  // t_q = (xa - so_a) inv_q > 0 for all five rays: the inv_q share a sign, and xa lies on that side of the source
  p.front_sign = inv[0] > 0 ? 1.0 : -1.0;
#pragma unroll
  for (int q = 1; q < 5; ++q) if ((inv[q] > 0 ? 1.0 : -1.0) != p.front_sign) p.ok = false;
  {  // unit direction of the pixel-centre ray along a
    double n2 = 0;
#pragma unroll
    for (int x = 0; x < 3; ++x) {
      const double d = fma(us[0], W.Uo[x], fma(vs[0], W.Vo[x], W.X00[x])) - W.so[x];
      n2 = fma(d, d, n2);
    }
    p.L = G.v[a] * sqrt(n2) * fabs(inv[0]);
  }
  // index(k) = (so_ax - c_ax) / v_ax + h_ax + (xa(k) - so_a) inv dax / v_ax,  xa(k) = c_a + (k - h_a) v_a
  const double x0 = G.c[a] - G.h[a] * G.v[a] - W.so[a];
  auto affine = [&](int q, double* s0, double* s1) {
    const int ax = q < 3 ? W.ub : W.vb;
    const double m = inv[q] * dax[q] / G.v[ax];
    *s0 = (W.so[ax] - G.c[ax]) / G.v[ax] + G.h[ax] + x0 * m;
    *s1 = G.v[a] * m;
  };
  affine(1, &p.b0, &p.db0); affine(2, &p.b1, &p.db1); affine(3, &p.d0, &p.dd0); affine(4, &p.d1, &p.dd1);
  return p;
}

// ------------------------------------------------------------------------------------------------ the four operations
struct DdFixed { unsigned max_bits; unsigned pad; };     // largest |l| of the call as float bits (dd_maxabs_kernel)
__global__ void dd_maxabs_kernel(const float* __restrict__ x, size_t n, DdFixed* __restrict__ fx) {
  unsigned m = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    m = max(m, __float_as_uint(fabsf(__ldg(x + i))));            // |x| as bits: monotone, NaN above everything
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m) atomicMax(&fx->max_bits, m);
}
// Fixed-point exponent: |sum| < 2^eb 2^hb with max|l| < 2^eb and the host's bound sum_i a^ij <= 2^hb.
__device__ __forceinline__ int dd_fixed_exponent(unsigned max_bits, int hb) {
  int eb;
  frexpf(__uint_as_float(max_bits), &eb);
  return 61 - eb - hb;
}
__global__ void dd_fixed_to_float_kernel(const long long* __restrict__ acc, const DdFixed* __restrict__ fx, int hb,
                                         size_t n, int accumulate, float* __restrict__ out) {
  const unsigned mb = fx->max_bits;
  const bool bad = mb >= 0x7f800000u;                             // Inf / NaN in the projections
  const double inv = mb && !bad ? scalbn(1.0, -dd_fixed_exponent(mb, hb)) : 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const float v = bad ? __int_as_float(0x7fc00000) : (float)((double)acc[i] * inv);
    out[i] = accumulate ? out[i] + v : v;
  }
}

template <int MODE>
__global__ void __launch_bounds__(kFwdThreads) dd_kernel(DdGeom G, const DdView* __restrict__ views,
                                                        const float* __restrict__ vol,     // 0: volume; 3: upstream volume
                                                        const float4* __restrict__ gvol, GradBricks GB,   // 1
                                                        const float* __restrict__ img,     // 1: upstream; 2, 3: projections
                                                        const DdFixed* __restrict__ fx, int hb,            // 2
                                                        float* __restrict__ out) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  const bool live = iu < G.nu && iv < G.nv;
  __shared__ DdView W;
  __shared__ float Pf[3][4];
  for (int i = threadIdx.x; i < (int)(sizeof(DdView) / 4); i += blockDim.x)
    reinterpret_cast<int*>(&W)[i] = reinterpret_cast<const int*>(views + view)[i];
  __syncthreads();
  if (MODE == 3 && threadIdx.x < 12) Pf[threadIdx.x >> 2][threadIdx.x & 3] = (float)W.P[threadIdx.x >> 2][threadIdx.x & 3];
  if (MODE == 3) __syncthreads();
  const size_t pix = ((size_t)view * G.nv + iv) * G.nu + iu;
  double sum = 0.0;
  float A0 = 0.f, A1 = 0.f, A2 = 0.f, B0 = 0.f, B1 = 0.f, B2 = 0.f;
  // per-pixel inputs of the back-projection modes
  float li = 0.f, Du = 0.f, Dv = 0.f, T0 = 0.f, T1 = 0.f, T2 = 0.f;
  double fscale = 0.0;
  bool work = live;
  if (MODE == 2) {
    li = live ? __ldg(img + pix) : 0.f;
    const unsigned mb = fx->max_bits;
    if (mb && mb < 0x7f800000u) fscale = scalbn(1.0, dd_fixed_exponent(mb, hb));
    work = live && li != 0.f;
  }
  if (MODE == 3 && live) {     // central differences of the zero-extended projection (:202)
    const float* p = img + pix;
    Du = 0.5f * ((iu + 1 < G.nu ? __ldg(p + 1) : 0.f) - (iu > 0 ? __ldg(p - 1) : 0.f));
    Dv = 0.5f * ((iv + 1 < G.nv ? __ldg(p + G.nu) : 0.f) - (iv > 0 ? __ldg(p - G.nu) : 0.f));
    T0 = fmaf(Du, Pf[0][0], Dv * Pf[1][0]); T1 = fmaf(Du, Pf[0][1], Dv * Pf[1][1]); T2 = fmaf(Du, Pf[0][2], Dv * Pf[1][2]);
    work = Du != 0.f || Dv != 0.f;
  }
  if (work) {
    const DdPixel p = dd_pixel(G, W, iu, iv);
    const int a = W.a, nb = G.n[W.ub], nd = G.n[W.vb];
    const size_t sx = 1, sy = (size_t)G.n[0], sz = (size_t)G.n[0] * G.n[1];
    const size_t sa = a == 0 ? sx : (a == 1 ? sy : sz), sb = W.ub == 0 ? sx : (W.ub == 1 ? sy : sz),
                 sd = W.vb == 0 ? sx : (W.vb == 1 ? sy : sz);
    // planes in front of the source: (x_a(k) - s'_a) front_sign > 0, x_a(k) = c_a + (k - h_a) v_a - the bound on k once
    int k_lo = 0, k_hi = G.n[a] - 1;
    {
      const double kz = (W.so[a] - G.c[a]) / G.v[a] + G.h[a];          // plane index of the source
      if (p.front_sign > 0) k_lo = max(k_lo, (int)floor(kz) + 1); else k_hi = min(k_hi, (int)ceil(kz) - 1);
    }
    const float Lf = (float)p.L;
    for (int k = k_lo; p.ok && k <= k_hi; ++k) {
      const double kd = (double)k;
      double b0 = fma(kd, p.db0, p.b0), b1 = fma(kd, p.db1, p.b1), d0 = fma(kd, p.dd0, p.d0), d1 = fma(kd, p.dd1, p.d1);
      if (b0 > b1) { const double t = b0; b0 = b1; b1 = t; }
      if (d0 > d1) { const double t = d0; d0 = d1; d1 = t; }
      if (!(b1 > b0) || !(d1 > d0)) continue;
      // the first cell each interval touches becomes the origin: the overlaps are then fp32 on numbers of order one
      const double jbf = floor(b0 + 0.5), jdf = floor(d0 + 0.5);
      if (!(fabs(jbf) < 1e9) || !(fabs(jdf) < 1e9) || !(b1 - jbf < 1e6) || !(d1 - jdf < 1e6)) continue;
      const int jbo = (int)jbf, jdo = (int)jdf;
      const float fb0 = (float)(b0 - jbf), fb1 = (float)(b1 - jbf), fd0 = (float)(d0 - jdf), fd1 = (float)(d1 - jdf);
      const float wl = Lf * fast_rcp((fb1 - fb0) * (fd1 - fd0));
      float plane = 0.f;
      // one voxel of the plane: weight wf on voxel (k, jb, jd)
      auto add = [&](float wf, int jb, int jd) {
        const size_t lin = (size_t)k * sa + (size_t)jb * sb + (size_t)jd * sd;
        if (MODE == 0) {
          plane = fmaf(wf, __ldg(vol + lin), plane);
        } else if (MODE == 2) {
          const long long q = __double2ll_rn((double)(wf * li) * fscale);
          atomicAdd(reinterpret_cast<unsigned long long*>(out) + lin, (unsigned long long)q);
        } else {
          // (k, jb, jd) -> (x, y, z) by selects (an array indexed by W.a would live in local memory)
          const int X = a == 0 ? k : (W.ub == 0 ? jb : jd), Y = a == 1 ? k : (W.ub == 1 ? jb : jd),
                    Z = a == 2 ? k : (W.ub == 2 ? jb : jd);
          const float rx = G.cx + ((float)X - (float)G.h[0]) * G.vx, ry = G.cy + ((float)Y - (float)G.h[1]) * G.vy,
                      rz = G.cz + ((float)Z - (float)G.h[2]) * G.vz;
          float lx, ly, lz;
          if (MODE == 1) {
            const float4 g = ldg4(gvol + (GB.FX(X) + GB.FY(Y) + GB.FZ(Z)));
            lx = wf * g.x; ly = wf * g.y; lz = wf * g.z;
          } else {             // Eq.13 at the voxel centre: q = a^ij w_j (D_u J_u + D_v J_v)
            const float wj = __ldg(vol + lin);
            const float up = fmaf(Pf[0][0], rx, fmaf(Pf[0][1], ry, fmaf(Pf[0][2], rz, Pf[0][3])));
            const float vp = fmaf(Pf[1][0], rx, fmaf(Pf[1][1], ry, fmaf(Pf[1][2], rz, Pf[1][3])));
            const float wp = fmaf(Pf[2][0], rx, fmaf(Pf[2][1], ry, fmaf(Pf[2][2], rz, Pf[2][3])));
            const float rw = fast_rcp(wp);
            const float cc = fmaf(Du, up, Dv * vp) * rw;
            const float sc = wf * wj * rw;
            lx = sc * fmaf(-cc, Pf[2][0], T0); ly = sc * fmaf(-cc, Pf[2][1], T1); lz = sc * fmaf(-cc, Pf[2][2], T2);
          }
          A0 += lx; A1 += ly; A2 += lz;
          B0 += ry * lz - rz * ly;
          B1 += rz * lx - rx * lz;
          B2 += rx * ly - ry * lx;
        }
      };
      if (fb1 < 1.5f && fd1 < 1.5f) {
        // footprint narrower than a voxel (fine detectors: every BASELINE config): at most 2 x 2 cells, no loops
        const float ob[2] = {fminf(fb1, 0.5f) - fb0, fmaxf(fb1 - 0.5f, 0.f)};
        const float od[2] = {fminf(fd1, 0.5f) - fd0, fmaxf(fd1 - 0.5f, 0.f)};
#pragma unroll
        for (int qd = 0; qd < 2; ++qd) {
#pragma unroll
          for (int qb = 0; qb < 2; ++qb) {
            const int jb = jbo + qb, jd = jdo + qd;
            const float wf = wl * ob[qb] * od[qd];
            if (wf > 0.f && jb >= 0 && jb < nb && jd >= 0 && jd < nd) add(wf, jb, jd);
          }
        }
      } else {
        const int nbj = min((int)floorf(fb1 + 0.5f), nb - 1 - jbo), ndj = min((int)floorf(fd1 + 0.5f), nd - 1 - jdo);
        for (int qd = max(0, -jdo); qd <= ndj; ++qd) {
          const float od = fminf(fd1, (float)qd + 0.5f) - fmaxf(fd0, (float)qd - 0.5f);
          if (!(od > 0.f)) continue;
          for (int qb = max(0, -jbo); qb <= nbj; ++qb) {
            const float ob = fminf(fb1, (float)qb + 0.5f) - fmaxf(fb0, (float)qb - 0.5f);
            if (!(ob > 0.f)) continue;
            add(wl * ob * od, jbo + qb, jdo + qd);
          }
        }
      }
      if (MODE == 0) sum += (double)plane;
    }
  }
  if (MODE == 0) {
    if (live) out[pix] = (float)sum;
  } else if (MODE == 1) {
    float o6[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (live) {
      const float w = __ldg(img + pix);
      o6[0] = w * A0; o6[1] = w * A1; o6[2] = w * A2; o6[3] = w * B0; o6[4] = w * B1; o6[5] = w * B2;
    }
    reduce6_to_partials<kFwdThreads>(o6, out, view);
  } else if (MODE == 3) {
    // partials[tile][view][6] (S'_q, S'_c of dfp_kernels.cuh: bp_grad_kernel; bp_contract_kernel finishes the job)
    __shared__ float red[kFwdThreads / 32][6];
    float o6[6] = {A0, A1, A2, B0, B1, B2};
#pragma unroll
    for (int q = 0; q < 6; ++q) {
      float v = o6[q];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      o6[q] = v;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) {
#pragma unroll
      for (int q = 0; q < 6; ++q) red[warp][q] = o6[q];
    }
    __syncthreads();
    if (threadIdx.x < 6) {
      float s = 0.f;
#pragma unroll
      for (int wI = 0; wI < kFwdThreads / 32; ++wI) s += red[wI][threadIdx.x];
      const size_t tile = (size_t)blockIdx.y * gridDim.x + blockIdx.x;
      out[(tile * gridDim.z + view) * 6 + threadIdx.x] = s;
    }
  }
}

}  // namespace dfp
