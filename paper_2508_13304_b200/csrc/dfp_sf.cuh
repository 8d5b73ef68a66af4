// dfp_sf.cuh - the four operations with SEPARABLE-FOOTPRINT weights (DFP_FLAG_SF, PAPER.md :213 ref [29],
// Tables III / IV rows SF; reading DESIGN.md U16).  Voxel-driven, everything from Eq.13's Jacobian at the voxel centre:
//   (u_j, v_j) = p(r'_j),  J = d(u, v)/dr'  (pixel-index units per mm, P_eff = P [R | t]);
//   widths wu_k = |J_uk| v_k, wv_k = |J_vk| v_k;  T(u), R(v) = unit-area trapezoids from the two widest rects of each axis;
//   a^ij = v_x v_y v_z sqrt(det J J^T) * int_pixel T du * int_pixel R dv.
// One thread per voxel, the views inside (the footprint of a (voxel, view) is computed once and serves every pixel it
// covers; the volume is written once; per-view 6-vectors are reduced per block).  The projected centre is taken in
// fp64 and split into a reference pixel + an offset; the trapezoid integrals are fp32 about that origin.
//   MODE 0  forward     l_i += a^ij mu_j         scatter (the paper's own kernels accumulate with atomics, :207) as
//                                                64-bit FIXED-POINT integer atomics into a zeroed accumulator image:
//                                                integer sums do not depend on the order, so the call is deterministic
//                                                like the rest of the library; sf_fixed_to_float_kernel finishes it
//   MODE 1  back        mu_j = sum_i a^ij l_i    gather: the exact transpose
//   MODE 2  forward pose gradient  sum_j (A^T w)_j G_f^j, G_f^j per voxel (Eq.19-20): gather the upstream image
//   MODE 3  back pose gradient     sum_ij a^ij w_j (D_u^i J_u(r_j) + D_v^i J_v(r_j))   (Eq.22, per-pixel G_b^i)
#pragma once
#include <cuda_runtime.h>

#include "dfp_dd.cuh"

namespace dfp {

// Unit-area trapezoid with base b >= top t >= 0 about its centre: half widths, height 2 / (b + t), 1 / (b - t).
struct SfTrap { float hb, ht, h, rr; };
__device__ __forceinline__ SfTrap sf_trap(float w0, float w1, float w2) {
  // base = sum, top = difference of the two widest of the three rects' widths
  const float hi = fmaxf(w0, fmaxf(w1, w2)), lo = fminf(w0, fminf(w1, w2)), mid = (w0 + w1 + w2) - hi - lo;
  SfTrap T;
  T.hb = 0.5f * (hi + mid); T.ht = 0.5f * (hi - mid);
  T.h = fast_rcp(T.hb + T.ht);
  T.rr = mid > 0.f ? fast_rcp(2.f * mid) : 0.f;          // 1 / (2 (x1 - x0)) = 1 / (b - t), b - t = 2 mid
  return T;
}
// int_{-inf}^{x} of the trapezoid, x measured from its centre
__device__ __forceinline__ float sf_cdf(const SfTrap& T, float x) {
  const float c = fminf(fmaxf(x, -T.ht), T.ht) + T.ht;           // flat top
  const float r = fminf(fmaxf(x, -T.hb), -T.ht) + T.hb;          // rising ramp
  const float q = fminf(fmaxf(x, T.ht), T.hb) - T.ht;            // falling ramp
  return T.h * (c + fmaf(r * r, T.rr, fmaf(-q * q, T.rr, q)));
}

// Footprint of one (voxel, view).  The projected centre is taken in fp64 and kept as a reference pixel (uc, vc) plus
// an offset |.| <= 1/2 (a weight is a difference of trapezoid integrals a few pixels from the centre: with the centre
// as the origin everything after it is fp32 at ~1e-7 of the weight).
struct SfFoot {
  float du, dv;           // (u_j - uc, v_j - vc)
  int uc, vc;
  SfTrap Tu, Tv;
  float M;
  float Ju[3], Jv[3];
  int iu0, iu1, iv0, iv1;
  bool ok;
};
__device__ __forceinline__ SfFoot sf_footprint(const DdGeom& G, const double (*E)[4], const float (*Ef)[4], const double* r) {
  SfFoot f;
  const double up = fma(E[0][0], r[0], fma(E[0][1], r[1], fma(E[0][2], r[2], E[0][3])));
  const double vp = fma(E[1][0], r[0], fma(E[1][1], r[1], fma(E[1][2], r[2], E[1][3])));
  const double wp = fma(E[2][0], r[0], fma(E[2][1], r[1], fma(E[2][2], r[2], E[2][3])));
  const float wf = (float)wp;
  f.ok = wf > 0.f;
  const float rw = fast_rcp(wf);
  const float ucf = rintf((float)up * rw), vcf = rintf((float)vp * rw);
  f.ok = f.ok && fabsf(ucf) < 1e9f && fabsf(vcf) < 1e9f;
  f.uc = f.ok ? (int)ucf : 0; f.vc = f.ok ? (int)vcf : 0;
  f.du = (float)fma(-(double)f.uc, wp, up) * rw;
  f.dv = (float)fma(-(double)f.vc, wp, vp) * rw;
  const float uj = (float)f.uc + f.du, vj = (float)f.vc + f.dv;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    f.Ju[k] = (Ef[0][k] - Ef[2][k] * uj) * rw;          // Eq.13: (P_1k w' - P_3k u') / w'^2
    f.Jv[k] = (Ef[1][k] - Ef[2][k] * vj) * rw;
  }
  const float guu = f.Ju[0] * f.Ju[0] + f.Ju[1] * f.Ju[1] + f.Ju[2] * f.Ju[2];
  const float gvv = f.Jv[0] * f.Jv[0] + f.Jv[1] * f.Jv[1] + f.Jv[2] * f.Jv[2];
  const float guv = f.Ju[0] * f.Jv[0] + f.Ju[1] * f.Jv[1] + f.Ju[2] * f.Jv[2];
  f.M = G.vx * G.vy * G.vz * sqrtf(fmaxf(fmaf(guu, gvv, -guv * guv), 0.f));
  f.Tu = sf_trap(fabsf(f.Ju[0]) * G.vx, fabsf(f.Ju[1]) * G.vy, fabsf(f.Ju[2]) * G.vz);
  f.Tv = sf_trap(fabsf(f.Jv[0]) * G.vx, fabsf(f.Jv[1]) * G.vy, fabsf(f.Jv[2]) * G.vz);
  if (!(f.Tu.hb > 0.f) || !(f.Tv.hb > 0.f) || !(f.M > 0.f) || !(f.Tu.hb < 1e6f) || !(f.Tv.hb < 1e6f)) f.ok = false;
  if (f.ok) {
    f.iu0 = max(f.uc + (int)floorf(f.du - f.Tu.hb + 0.5f), 0); f.iu1 = min(f.uc + (int)floorf(f.du + f.Tu.hb + 0.5f), G.nu - 1);
    f.iv0 = max(f.vc + (int)floorf(f.dv - f.Tv.hb + 0.5f), 0); f.iv1 = min(f.vc + (int)floorf(f.dv + f.Tv.hb + 0.5f), G.nv - 1);
  } else {
    f.iu0 = f.iv0 = 0; f.iu1 = f.iv1 = -1;
  }
  return f;
}

// MODE 0 sums its projections as 64-bit FIXED-POINT integers (integer addition is associative: the result does not
// depend on the order the atomics land in, unlike an fp32 atomicAdd).  The scale 2^e is chosen on the device from the
// largest |mu| (sf_maxabs_kernel) and the longest chord of the grid so that no pixel can overflow:
//   |l_i| <= max|mu| sum_j a^ij,  sum_j a^ij ~ the chord of the pixel's ray <= the grid's diagonal (8x head-room).
struct SfFixed { unsigned max_bits; unsigned pad; };
__global__ void sf_maxabs_kernel(const float* __restrict__ vol, size_t n, SfFixed* __restrict__ fx) {
  unsigned m = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    m = max(m, __float_as_uint(fabsf(__ldg(vol + i))));          // |x| as bits: monotone, NaN above everything
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m) atomicMax(&fx->max_bits, m);
}
__device__ __forceinline__ int sf_fixed_exponent(const DdGeom& G, unsigned max_bits) {
  const float diag = sqrtf((float)G.n[0] * G.vx * (float)G.n[0] * G.vx + (float)G.n[1] * G.vy * (float)G.n[1] * G.vy +
                           (float)G.n[2] * G.vz * (float)G.n[2] * G.vz);
  int eb;
  frexpf(__uint_as_float(max_bits) * diag * 8.f, &eb);           // bound < 2^eb
  return 61 - eb;
}
__global__ void sf_fixed_to_float_kernel(DdGeom G, const long long* __restrict__ acc, const SfFixed* __restrict__ fx,
                                         size_t n, float* __restrict__ out) {
  const unsigned mb = fx->max_bits;
  const bool bad = mb >= 0x7f800000u;                             // Inf / NaN in the volume
  const double inv = mb && !bad ? scalbn(1.0, -sf_fixed_exponent(G, mb)) : 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    out[i] = bad ? __int_as_float(0x7fc00000) : (float)((double)acc[i] * inv);
}

constexpr int kSfThreads = 256, kSfBatch = 8;
template <int MODE>
__global__ void __launch_bounds__(kSfThreads) sf_kernel(DdGeom G, int n_views, int accumulate,
                                                        const DdView* __restrict__ views,
                                                        const float* __restrict__ vol,      // MODE 0, 2: the volume
                                                        const float* __restrict__ img,      // MODE 1, 3: projections; 2: upstream
                                                        const float* __restrict__ upvol,    // MODE 3: upstream volume
                                                        const SfFixed* __restrict__ fx,     // MODE 0: fixed-point scale
                                                        float* __restrict__ out) {
  const size_t nvox = (size_t)G.n[0] * G.n[1] * G.n[2];
  const size_t j = (size_t)blockIdx.x * kSfThreads + threadIdx.x;
  const bool live = j < nvox;
  int xyz[3] = {0, 0, 0};
  if (live) { xyz[0] = (int)(j % G.n[0]); xyz[1] = (int)((j / G.n[0]) % G.n[1]); xyz[2] = (int)(j / ((size_t)G.n[0] * G.n[1])); }
  // the views run in batches of kSfBatch: their matrices are staged together and the per-view block reductions of the
  // gradient modes wait for the end of the batch - three barriers per batch instead of three per view
  __shared__ double Eb[kSfBatch][3][4];
  __shared__ float Efb[kSfBatch][3][4];
  __shared__ float red[kSfBatch][kSfThreads / 32][6];
  double fscale = 0.0;
  if (MODE == 0) {
    const unsigned mb = fx->max_bits;
    if (mb && mb < 0x7f800000u) fscale = scalbn(1.0, sf_fixed_exponent(G, mb));
  }
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
  for (int view0 = 0; view0 < n_views; view0 += kSfBatch) {
   const int nb = min(kSfBatch, n_views - view0);
   __syncthreads();
   if (threadIdx.x < 12 * nb) {
     const int b = threadIdx.x / 12, q = threadIdx.x % 12;
     const double e = views[view0 + b].P[q >> 2][q & 3];
     Eb[b][q >> 2][q & 3] = e;
     Efb[b][q >> 2][q & 3] = (float)e;
   }
   __syncthreads();
   for (int vb = 0; vb < nb; ++vb) {
    const int view = view0 + vb;
    const double (*E)[4] = Eb[vb];
    const float (*Ef)[4] = Efb[vb];
    double s0 = 0.0, s1 = 0.0;
    SfFoot f;
    f.ok = false;
    if (work) {
      f = sf_footprint(G, E, Ef, r);
      const size_t base = (size_t)view * G.nu * G.nv;
      float cv0 = sf_cdf(f.Tv, (float)(f.iv0 - f.vc) - 0.5f - f.dv);          // rolling: the lower edge of the first row
      for (int iv = f.iv0; iv <= f.iv1; ++iv) {
        const float cv1 = sf_cdf(f.Tv, (float)(iv - f.vc) + 0.5f - f.dv);
        const float fv = cv1 - cv0;
        cv0 = cv1;
        if (!(fv > 0.f)) continue;
        const float mv = f.M * fv;
        float cu0 = sf_cdf(f.Tu, (float)(f.iu0 - f.uc) - 0.5f - f.du);
        for (int iu = f.iu0; iu <= f.iu1; ++iu) {
          const float cu1 = sf_cdf(f.Tu, (float)(iu - f.uc) + 0.5f - f.du);
          const float fu = cu1 - cu0;
          cu0 = cu1;
          if (!(fu > 0.f)) continue;
          const float w = mv * fu;
          const size_t pix = base + (size_t)iv * G.nu + iu;
          if (MODE == 0) {
            const long long q = __double2ll_rn((double)w * (double)mu * fscale);
            atomicAdd(reinterpret_cast<unsigned long long*>(out) + pix, (unsigned long long)q);
          } else if (MODE == 1 || MODE == 2) {
            s0 = fma((double)w, (double)__ldg(img + pix), s0);
          } else {
            const float* p = img + pix;
            const float lp = iu + 1 < G.nu ? __ldg(p + 1) : 0.f, lm = iu > 0 ? __ldg(p - 1) : 0.f;
            const float tp = iv + 1 < G.nv ? __ldg(p + G.nu) : 0.f, tm = iv > 0 ? __ldg(p - G.nu) : 0.f;
            s0 = fma((double)w, 0.5 * ((double)lp - (double)lm), s0);
            s1 = fma((double)w, 0.5 * ((double)tp - (double)tm), s1);
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
          const float a0 = (float)s0, a1 = (float)s1;
          qx = wj * fmaf(a0, f.Ju[0], a1 * f.Jv[0]);
          qy = wj * fmaf(a0, f.Ju[1], a1 * f.Jv[1]);
          qz = wj * fmaf(a0, f.Ju[2], a1 * f.Jv[2]);
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
        for (int q = 0; q < 6; ++q) red[vb][warp][q] = s6[q];
      }
    }
   }
   if (MODE == 2 || MODE == 3) {
     __syncthreads();
     if (threadIdx.x < 6 * nb) {
       const int vb = threadIdx.x / 6, q = threadIdx.x % 6, view = view0 + vb;
       float t = 0.f;
#pragma unroll
       for (int wI = 0; wI < kSfThreads / 32; ++wI) t += red[vb][wI][q];
       // MODE 2: partials[view][block][6] (fwd_contract_kernel); MODE 3: partials[block][view][6] (bp_contract_kernel)
       const size_t at = MODE == 2 ? ((size_t)view * gridDim.x + blockIdx.x) : ((size_t)blockIdx.x * n_views + view);
       out[at * 6 + q] = t;
     }
   }
  }
  if (MODE == 1 && live) out[j] = (float)acc;
}

}  // namespace dfp
