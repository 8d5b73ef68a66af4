// dfp_dd.cuh - the four operations with DISTANCE-DRIVEN weights (DFP_FLAG_DD, PAPER.md :213 ref [44],
// Tables III / IV rows DD; reading DESIGN.md U14).
//
// Per view (object frame): driving axis a = argmax |n'_a| of the direction source -> detector centre; the detector's
// u pairs with the in-plane axis along which the pixel step U' is longer.  Per plane k of voxel centres along a, the
// boundary mid-points (iu -+ 1/2, iv), (iu, iv -+ 1/2) of a pixel are projected from the source onto the plane; in
// continuous voxel indices they bound the pixel's footprint [B0, B1] x [D0, D1];
//   a^ij = L (|[B0,B1] n cell(jb)| / (B1 - B0)) (|[D0,D1] n cell(jd)| / (D1 - D0)),  L = v_a / |e'_a| (pixel-centre ray).
// A boundary position is AFFINE in the plane index k (position = s' + (x_a - s'_a) dir / dir_a), so a pixel carries
// four (start, increment) pairs; they and the overlaps are taken in fp64 (a weight is a difference of positions of
// magnitude n/2: fp32 would leave 1e-5 relative error per weight) - the kernels of this "next" row are arithmetic-light
// per voxel read and are measured beside the trilinear ones in DESIGN.md.
//   dd_fwd_kernel        l_i = sum_j a^ij mu_j                                  one thread per pixel
//   dd_fwd_grad_kernel   A_i = sum_j a^ij g_j, B_i = sum_j a^ij r'_j x g_j      per-voxel G_f^j (Eq.19-20), g_j from the
//                        per-voxel gradient volume of grad_volume_kernel
//   dd_bp_kernel         mu_j = sum_i a^ij l_i, the EXACT transpose (Eq.21)     one thread per voxel: the pixels whose
//                        footprint can meet the voxel's cell are found by projecting the cell's corners onto the
//                        detector, each candidate's weight is then the forward formula
//   dd_bp_grad_kernel    sum_ij a^ij w_j (D_u^i J_u(r_j) + D_v^i J_v(r_j))      per-pixel G_b^i (Eq.22), D = central
//                        differences of the zero-extended projection, J = Eq.13 at the voxel centre
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

// Continuous voxel index, along axis `ax`, of the point where the ray source -> detector point (u, v) meets the plane
// x_a = xa; false if the plane is not in front of the source along that ray.
__device__ __forceinline__ bool dd_hit(const DdGeom& G, const DdView& W, double u, double v, double xa, int ax,
                                       double* idx) {
  const int a = W.a;
  const double da = fma(u, W.Uo[a], fma(v, W.Vo[a], W.X00[a])) - W.so[a];
  const double dx = fma(u, W.Uo[ax], fma(v, W.Vo[ax], W.X00[ax])) - W.so[ax];
  if (fabs(da) < 1e-300) return false;
  const double t = (xa - W.so[a]) / da;
  *idx = (fma(t, dx, W.so[ax]) - G.c[ax]) / G.v[ax] + G.h[ax];
  return t > 0.0;
}

// A pixel of the forward kernels: the four boundary positions as affine functions of the plane index k.
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

// Voxel offset of (plane k, in-plane indices jb along W.ub, jd along W.vb) in vol[z][y][x].
__device__ __forceinline__ void dd_voxel(const DdView& W, int k, int jb, int jd, int* xyz) {
  xyz[W.a] = k; xyz[W.ub] = jb; xyz[W.vb] = jd;
}

// ------------------------------------------------------------------------------------------------ forward
// GRAD 0: l_i = sum_j a^ij mu_j (reads the caller's volume); GRAD 1: the six sums of Eq.19-20 times the upstream weight.
template <int GRAD>
__global__ void __launch_bounds__(kFwdThreads) dd_fwd_kernel(DdGeom G, const DdView* __restrict__ views,
                                                            const float* __restrict__ vol,
                                                            const float4* __restrict__ gvol, GradBricks GB,
                                                            const float* __restrict__ upstream,
                                                            float* __restrict__ out) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  const bool live = iu < G.nu && iv < G.nv;
  __shared__ DdView W;
  for (int i = threadIdx.x; i < (int)(sizeof(DdView) / 4); i += blockDim.x)
    reinterpret_cast<int*>(&W)[i] = reinterpret_cast<const int*>(views + view)[i];
  __syncthreads();
  double sum = 0.0;
  float A0 = 0.f, A1 = 0.f, A2 = 0.f, B0 = 0.f, B1 = 0.f, B2 = 0.f;
  if (live) {
    const DdPixel p = dd_pixel(G, W, iu, iv);
    const int a = W.a, nb = G.n[W.ub], nd = G.n[W.vb];
    const size_t sx = 1, sy = (size_t)G.n[0], sz = (size_t)G.n[0] * G.n[1];
    const size_t st[3] = {sx, sy, sz};
    const size_t sa = st[a], sb = st[W.ub], sd = st[W.vb];
    for (int k = 0; p.ok && k < G.n[a]; ++k) {
      const double xa_rel = (G.c[a] + (k - G.h[a]) * G.v[a] - W.so[a]) * p.front_sign;
      if (!(xa_rel > 0.0)) continue;
      const double kd = (double)k;
      double b0 = fma(kd, p.db0, p.b0), b1 = fma(kd, p.db1, p.b1), d0 = fma(kd, p.dd0, p.d0), d1 = fma(kd, p.dd1, p.d1);
      if (b0 > b1) { const double t = b0; b0 = b1; b1 = t; }
      if (d0 > d1) { const double t = d0; d0 = d1; d1 = t; }
      if (!(b1 > b0) || !(d1 > d0)) continue;
      const int jb0 = max((int)floor(b0 + 0.5), 0), jb1 = min((int)floor(b1 + 0.5), nb - 1);
      const int jd0 = max((int)floor(d0 + 0.5), 0), jd1 = min((int)floor(d1 + 0.5), nd - 1);
      const double wl = p.L / ((b1 - b0) * (d1 - d0));
      for (int jd = jd0; jd <= jd1; ++jd) {
        const double od = fmin(d1, jd + 0.5) - fmax(d0, jd - 0.5);
        if (!(od > 0.0)) continue;
        for (int jb = jb0; jb <= jb1; ++jb) {
          const double ob = fmin(b1, jb + 0.5) - fmax(b0, jb - 0.5);
          if (!(ob > 0.0)) continue;
          const double wgt = wl * ob * od;
          if (!GRAD) {
            sum = fma(wgt, (double)__ldg(vol + (size_t)k * sa + (size_t)jb * sb + (size_t)jd * sd), sum);
          } else {
            int xyz[3];
            dd_voxel(W, k, jb, jd, xyz);
            const float4 g = ldg4(gvol + (GB.FX(xyz[0]) + GB.FY(xyz[1]) + GB.FZ(xyz[2])));
            const float wf = (float)wgt;
            const float rx = G.cx + ((float)xyz[0] - (float)G.h[0]) * G.vx, ry = G.cy + ((float)xyz[1] - (float)G.h[1]) * G.vy,
                        rz = G.cz + ((float)xyz[2] - (float)G.h[2]) * G.vz;
            const float lx = wf * g.x, ly = wf * g.y, lz = wf * g.z;
            A0 += lx; A1 += ly; A2 += lz;
            B0 += ry * lz - rz * ly;
            B1 += rz * lx - rx * lz;
            B2 += rx * ly - ry * lx;
          }
        }
      }
    }
  }
  if (!GRAD) {
    if (live) out[((size_t)view * G.nv + iv) * G.nu + iu] = (float)sum;
  } else {
    float o6[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (live) {
      const float w = __ldg(upstream + ((size_t)view * G.nv + iv) * G.nu + iu);
      o6[0] = w * A0; o6[1] = w * A1; o6[2] = w * A2; o6[3] = w * B0; o6[4] = w * B1; o6[5] = w * B2;
    }
    reduce6_to_partials<kFwdThreads>(o6, out, view);
  }
}

// ------------------------------------------------------------------------------------------------ back (transpose)
// Offsets, in voxels, from the voxel centre r (on the plane x_a = r_a) to the points where the rays source -> detector
// point (u, v) meet that plane:  off_x(u, v) = (D_x E_a - E_x D_a) / (D_a v_x),  D = X(u, v) - s' (affine in u, v),
// E = r - s'.  The 2 x 2 determinant of two nearly parallel vectors of ~1000 mm is a few hundred: it is expanded ONCE per
// (voxel, view), in fp64, about a reference pixel (uc, vc) inside the voxel's window -
//   det_x(u, v) = c_x + (u - uc) p_x + (v - vc) q_x,   D_a(u, v) = D_a(uc, vc) + (u - uc) U_a + (v - vc) V_a -
// and its three coefficients are small numbers without cancellation left in them, so every boundary of every
// candidate pixel is then two fp32 FMAs per function, a reciprocal and a product (no fp64 per pixel).
struct DdLocal {
  float Dc[3];            // D(uc, vc) along a, ub, vb
  float U[3], V[3];       // detector steps along a, ub, vb
  float cb, pb, qb;       // det along ub
  float cd, pd, qd;       // det along vb
  float Ea, ivb, ivd, va; // E_a; 1 / pitch along ub, vb; pitch along a
};
__device__ __forceinline__ DdLocal dd_local(const DdGeom& G, const DdView& W, const double* E, int uc, int vc) {
  DdLocal q;
  const int ax[3] = {W.a, W.ub, W.vb};
  double D[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    D[i] = fma((double)uc, W.Uo[ax[i]], fma((double)vc, W.Vo[ax[i]], W.X00[ax[i]])) - W.so[ax[i]];
    q.Dc[i] = (float)D[i]; q.U[i] = (float)W.Uo[ax[i]]; q.V[i] = (float)W.Vo[ax[i]];
  }
  const double Ea = E[W.a], Eb = E[W.ub], Ed = E[W.vb];
  q.cb = (float)fma(D[1], Ea, -Eb * D[0]);
  q.pb = (float)fma(W.Uo[W.ub], Ea, -Eb * W.Uo[W.a]);
  q.qb = (float)fma(W.Vo[W.ub], Ea, -Eb * W.Vo[W.a]);
  q.cd = (float)fma(D[2], Ea, -Ed * D[0]);
  q.pd = (float)fma(W.Uo[W.vb], Ea, -Ed * W.Uo[W.a]);
  q.qd = (float)fma(W.Vo[W.vb], Ea, -Ed * W.Vo[W.a]);
  q.Ea = (float)Ea; q.ivb = 1.0f / (float)G.v[W.ub]; q.ivd = 1.0f / (float)G.v[W.vb]; q.va = (float)G.v[W.a];
  return q;
}
// offset along ub (AXIS 0) or vb (AXIS 1) at the detector point (uc + du, vc + dv); *front: t = E_a / D_a > 0
template <int AXIS>
__device__ __forceinline__ float dd_off(const DdLocal& q, float du, float dv, bool* front) {
  const float Da = fmaf(du, q.U[0], fmaf(dv, q.V[0], q.Dc[0]));
  const float det = AXIS == 0 ? fmaf(du, q.pb, fmaf(dv, q.qb, q.cb)) : fmaf(du, q.pd, fmaf(dv, q.qd, q.cd));
  *front = q.Ea * Da > 0.f;
  return det * fast_rcp(Da) * (AXIS == 0 ? q.ivb : q.ivd);
}
// normalised overlap of the footprint [x0, x1] (either order) with the voxel's cell [-1/2, 1/2]; 0 if none
__device__ __forceinline__ float dd_cell_overlap(float x0, float x1) {
  const float lo = fminf(x0, x1), hi = fmaxf(x0, x1);
  const float o = fminf(hi, 0.5f) - fmaxf(lo, -0.5f);
  return (o > 0.f && hi > lo) ? o / (hi - lo) : 0.f;
}
// slab length v_a / |e_a| of the pixel-centre ray at (uc + du, vc + dv)
__device__ __forceinline__ float dd_slab_length(const DdLocal& q, float du, float dv) {
  const float d0 = fmaf(du, q.U[0], fmaf(dv, q.V[0], q.Dc[0])), d1 = fmaf(du, q.U[1], fmaf(dv, q.V[1], q.Dc[1])),
              d2 = fmaf(du, q.U[2], fmaf(dv, q.V[2], q.Dc[2]));
  return q.va * sqrtf(fmaf(d0, d0, fmaf(d1, d1, d2 * d2))) * fast_rcp(fabsf(d0));
}

// Candidate pixels of a voxel: the detector bounding box of its cell's four corners on the plane (fp32: the box gets
// one pixel of margin anyway - the footprints are taken on the pixels' mid-lines, which an in-plane rotation tilts by a
// fraction of a pixel).
struct DdWindow { int u0, u1, v0, v1; };
__device__ __forceinline__ DdWindow dd_window(const DdGeom& G, const DdView& W, const float* P, const float* r) {
  float umin = 3e38f, umax = -3e38f, vmin = 3e38f, vmax = -3e38f;
  bool ok = true;
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    float q[3] = {r[0], r[1], r[2]};
    q[W.ub] += ((c & 1) ? 0.5f : -0.5f) * (float)G.v[W.ub];
    q[W.vb] += ((c & 2) ? 0.5f : -0.5f) * (float)G.v[W.vb];
    const float wp = fmaf(P[8], q[0], fmaf(P[9], q[1], fmaf(P[10], q[2], P[11])));
    if (!(wp > 0.f)) ok = false;
    const float rw = 1.0f / wp;
    const float u = fmaf(P[0], q[0], fmaf(P[1], q[1], fmaf(P[2], q[2], P[3]))) * rw;
    const float v = fmaf(P[4], q[0], fmaf(P[5], q[1], fmaf(P[6], q[2], P[7]))) * rw;
    umin = fminf(umin, u); umax = fmaxf(umax, u); vmin = fminf(vmin, v); vmax = fmaxf(vmax, v);
  }
  DdWindow w;
  if (!ok || !(umax - umin < 1e6f) || !(vmax - vmin < 1e6f)) { w.u0 = w.v0 = 0; w.u1 = w.v1 = -1; return w; }
  w.u0 = max((int)floorf(umin + 0.5f) - 1, 0); w.u1 = min((int)floorf(umax + 0.5f) + 1, G.nu - 1);
  w.v0 = max((int)floorf(vmin + 0.5f) - 1, 0); w.v1 = min((int)floorf(vmax + 0.5f) + 1, G.nv - 1);
  return w;
}

constexpr int kDdBpThreads = 256;
// GRAD 0: vol[j] (+)= sum_views sum_i a^ij l_i.  One thread per voxel, x fastest; the view loop is inside the thread
// so that the volume is written once and the sum over views has a fixed order.
// GRAD 1: partials[tile][view][6] of sum_ij a^ij w_j (D_u^i J_u(r_j) + D_v^i J_v(r_j)) and its moment about the origin
// of the object frame (S'_q, S'_c of dfp_kernels.cuh: bp_grad_kernel; the same bp_contract_kernel finishes the job).
template <int GRAD>
__global__ void __launch_bounds__(kDdBpThreads) dd_bp_kernel(DdGeom G, int n_views, int accumulate,
                                                            const DdView* __restrict__ views,
                                                            const BpView* __restrict__ bviews,
                                                            const float* __restrict__ proj,
                                                            const float* __restrict__ upstream,
                                                            float* __restrict__ out) {
  const size_t nvox = (size_t)G.n[0] * G.n[1] * G.n[2];
  const size_t j = (size_t)blockIdx.x * kDdBpThreads + threadIdx.x;
  const bool live = j < nvox;
  int xyz[3] = {0, 0, 0};
  if (live) { xyz[0] = (int)(j % G.n[0]); xyz[1] = (int)((j / G.n[0]) % G.n[1]); xyz[2] = (int)(j / ((size_t)G.n[0] * G.n[1])); }
  __shared__ DdView W;
  __shared__ BpView BV;
  __shared__ float red[kDdBpThreads / 32][6];
  const float wj = (GRAD && live) ? __ldg(upstream + j) : 0.f;
  // object-frame mm of the voxel centre
  const float rx = G.cx + ((float)xyz[0] - (float)G.h[0]) * G.vx, ry = G.cy + ((float)xyz[1] - (float)G.h[1]) * G.vy,
              rz = G.cz + ((float)xyz[2] - (float)G.h[2]) * G.vz;
  double acc = (!GRAD && accumulate && live) ? (double)out[j] : 0.0;
  for (int view = 0; view < n_views; ++view) {
    __syncthreads();
    for (int i = threadIdx.x; i < (int)(sizeof(DdView) / 4); i += blockDim.x)
      reinterpret_cast<int*>(&W)[i] = reinterpret_cast<const int*>(views + view)[i];
    if (GRAD && threadIdx.x < (int)(sizeof(BpView) / 4))
      reinterpret_cast<float*>(&BV)[threadIdx.x] = reinterpret_cast<const float*>(bviews + view)[threadIdx.x];
    __syncthreads();
    double su = 0.0, sv = 0.0;
    if (live && (!GRAD || wj != 0.f)) {
      double E[3];
#pragma unroll
      for (int x = 0; x < 3; ++x) E[x] = G.c[x] + ((double)xyz[x] - G.h[x]) * G.v[x] - W.so[x];
      float Pl[12];
#pragma unroll
      for (int q = 0; q < 12; ++q) Pl[q] = (float)W.P[q >> 2][q & 3];
      const float rc[3] = {rx, ry, rz};
      const DdWindow win = dd_window(G, W, Pl, rc);
      const float* img = proj + (size_t)view * G.nu * G.nv;
      if (win.u0 <= win.u1 && win.v0 <= win.v1) {
        const int uc = (win.u0 + win.u1) >> 1, vc = (win.v0 + win.v1) >> 1;
        const DdLocal q = dd_local(G, W, E, uc, vc);
        for (int iv = win.v0; iv <= win.v1; ++iv) {
          const float dv = (float)(iv - vc);
          bool fl, fr, f2, f3;
          float bl = dd_off<0>(q, (float)(win.u0 - uc) - 0.5f, dv, &fl);      // the left boundary of the row's first pixel
          for (int iu = win.u0; iu <= win.u1; ++iu) {
            const float du = (float)(iu - uc);
            const float br = dd_off<0>(q, du + 0.5f, dv, &fr);                // shared with the next pixel
            const float ob = dd_cell_overlap(bl, br);
            const bool fb = fl && fr;
            bl = br; fl = fr;
            if (!(ob > 0.f) || !fb) continue;
            const float d0 = dd_off<1>(q, du, dv - 0.5f, &f2), d1 = dd_off<1>(q, du, dv + 0.5f, &f3);
            const float od = dd_cell_overlap(d0, d1);
            if (!(od > 0.f) || !(f2 && f3)) continue;
            const double wgt = (double)(dd_slab_length(q, du, dv) * ob * od);
            if (!GRAD) {
              acc = fma(wgt, (double)__ldg(img + (size_t)iv * G.nu + iu), acc);
            } else {
              const float lp = iu + 1 < G.nu ? __ldg(img + (size_t)iv * G.nu + iu + 1) : 0.f;
              const float lm = iu > 0 ? __ldg(img + (size_t)iv * G.nu + iu - 1) : 0.f;
              const float tp = iv + 1 < G.nv ? __ldg(img + (size_t)(iv + 1) * G.nu + iu) : 0.f;
              const float tm = iv > 0 ? __ldg(img + (size_t)(iv - 1) * G.nu + iu) : 0.f;
              su = fma(wgt, 0.5 * ((double)lp - (double)lm), su);
              sv = fma(wgt, 0.5 * ((double)tp - (double)tm), sv);
            }
          }
        }
      }
    }
    if (GRAD) {
      float s6[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      if (live && wj != 0.f) {
        // Eq.13 at the voxel centre from the folded P_eff rows of BpView (u, v in the rows' own shifted units)
        const float xf = (float)xyz[0] - (float)G.h[0], yf = (float)xyz[1] - (float)G.h[1], zf = (float)xyz[2] - (float)G.h[2];
        const float up = fmaf(BV.A[0][0], xf, fmaf(BV.A[0][1], yf, fmaf(BV.A[0][2], zf, BV.A[0][3])));
        const float vp = fmaf(BV.A[1][0], xf, fmaf(BV.A[1][1], yf, fmaf(BV.A[1][2], zf, BV.A[1][3])));
        const float wp = fmaf(BV.A[2][0], xf, fmaf(BV.A[2][1], yf, fmaf(BV.A[2][2], zf, BV.A[2][3])));
        const float rw = 1.0f / wp, uq = up * rw, vq = vp * rw;
        const float dlu = (float)su, dlv = (float)sv;
        const float cc = fmaf(dlu, uq, dlv * vq);
        const float sc = wj * rw;
        const float qx = sc * fmaf(dlu, BV.J[0][0], fmaf(dlv, BV.J[1][0], -cc * BV.J[2][0]));
        const float qy = sc * fmaf(dlu, BV.J[0][1], fmaf(dlv, BV.J[1][1], -cc * BV.J[2][1]));
        const float qz = sc * fmaf(dlu, BV.J[0][2], fmaf(dlv, BV.J[1][2], -cc * BV.J[2][2]));
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
        for (int wI = 0; wI < kDdBpThreads / 32; ++wI) t += red[wI][threadIdx.x];
        out[((size_t)blockIdx.x * n_views + view) * 6 + threadIdx.x] = t;
      }
    }
  }
  if (!GRAD && live) out[j] = (float)acc;
}

}  // namespace dfp
