// dfp_kernels.cuh - sm_100a kernels of the dfp hot path.
//
//   pack_volume_kernel      vol -> zero-padded pair-packed copy  P[z][y][x] = (v[x], v[x+1])       (a3/a4 input)
//   fwd_project_kernel      a2 + a3: per-ray clip (fp64, once per ray) and fixed-step trilinear march (fp32)
//   fwd_grad_kernel         a2 + a4: fused gradient projection, 6 register accumulators per ray, warp-shuffle
//                           and block reduction into per-(view, block) partials
//   fwd_contract_kernel     a5: deterministic fp64 sum of the partials, dL/dt = -R S_A, dL/dgamma_k = -w_k.S_B
//   pack_proj_kernel        proj -> zero-padded quad-packed copy Q[v][u] = (l[v][u], l[v][u+1], l[v+1][u], l[v+1][u+1])
//   bp_kernel               a6: voxel-driven back-projection, one 128-bit fetch per (voxel, view)
//   bp_grad_kernel          a7: back-projection gradient, per-view 6-vector partials per voxel tile
//   bp_contract_kernel      a8: fp64 sum of the partials, dL/dt = R S'_q, dL/dgamma_k = (R^T a_k).S'_c
//   count_steps_kernel      ray-step count of the metric
//
// No kernel tests a volume / detector bound in its inner loop: the packed copies carry a zero border that
// realises the zero extension of f~ and b~ (U7), and the per-ray clip / per-sample clamp keeps every
// access inside that border.  floor() is taken with the 1.5*2^23 magic-number add (FADD + IADD on the FMA/ALU
// pipes) instead of F2I/FRND, which issue at 1/8 rate on sm_100.
#pragma once
#include <cuda_runtime.h>

#include "dfp_params.h"

namespace dfp {

constexpr float kMagic = 12582912.0f;        // 1.5 * 2^23: (x + kMagic) - kMagic == rint(x) for |x| < 2^22
constexpr int kMagicBits = 0x4B400000;       // __float_as_int(kMagic)

constexpr int kFwdTU = 16, kFwdTV = 16;      // block tile of detector pixels (8 warps, each an 8x4 pixel patch)
constexpr int kFwdThreads = kFwdTU * kFwdTV;
constexpr int kBpTX = 32, kBpTY = 8;         // block tile of voxels in (x, y)
constexpr int kBpThreads = kBpTX * kBpTY;
constexpr int kBpZ = 8;                      // voxels along z per thread in bp_kernel (register accumulators)

__device__ __forceinline__ float lerp(float a, float v0, float v1) { return fmaf(a, v1 - v0, v0); }

// 1 / w' for the perspective divide: MUFU.RCP plus one Newton step (relative error < 2^-23, no range check or
// slow path: w' is a source-to-voxel depth in mm, far inside the normal range).  __frcp_rn costs ~11 instructions.
__device__ __forceinline__ float fast_rcp(float w) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(w));
  return fmaf(r, fmaf(-w, r, 1.0f), r);
}

__device__ __forceinline__ float2 ldg2(const float2* p) { return __ldg(p); }
__device__ __forceinline__ float4 ldg4(const float4* p) { return __ldg(p); }

// ------------------------------------------------------------------------------------------------ packing
__global__ void __launch_bounds__(256) pack_volume_kernel(VolLayout L, const float* __restrict__ vol,
                                                          float4* __restrict__ pvol) {
  const size_t n = (size_t)L.px * L.py * L.pz;
  const unsigned nbxy = (unsigned)L.nbx * L.nby;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    // output order = memory order: brick-major, 8 cells per brick (x fastest, then y, then z)
    const unsigned within = (unsigned)(i & 7), brick = (unsigned)(i >> 3);
    const unsigned bz = brick / nbxy, rem = brick - bz * nbxy;
    const unsigned by = rem / L.nbx, bx = rem - by * L.nbx;
    const int x = (int)(2 * bx + (within & 1)) - L.lx;
    const int y = (int)(2 * by + ((within >> 1) & 1)) - L.ly;
    const int z = (int)(2 * bz + (within >> 2)) - L.lz;
    float4 c = make_float4(0.f, 0.f, 0.f, 0.f);
    if (z >= 0 && z < L.nz) {
      const float* sl = vol + (size_t)z * L.ny * L.nx;
      const bool x0 = x >= 0 && x < L.nx, x1 = x + 1 >= 0 && x + 1 < L.nx;
      const bool y0 = y >= 0 && y < L.ny, y1 = y + 1 >= 0 && y + 1 < L.ny;
      if (x0 && y0) c.x = __ldg(sl + (size_t)y * L.nx + x);
      if (x1 && y0) c.y = __ldg(sl + (size_t)y * L.nx + x + 1);
      if (x0 && y1) c.z = __ldg(sl + (size_t)(y + 1) * L.nx + x);
      if (x1 && y1) c.w = __ldg(sl + (size_t)(y + 1) * L.nx + x + 1);
    }
    pvol[i] = c;
  }
}

// Per-voxel gradient volume for the weight models that follow the paper's per-voxel G_f^j (Siddon, Joseph;
// PAPER.md :183, :189): g_j = central differences of the zero-extended voxel values times 1/(2 v_a), one float4
// (g_x, g_y, g_z, f_j) per GRID voxel, in 2 x 2 x 2 bricks of 128 B so that the rays of a warp, which spread over a
// few voxels in every direction, touch few lines.  GradBricks::index(x, y, z) = FX(x) + FY(y) + FZ(z).
struct GradBricks {
  int nx, ny, nz;
  int fy8, fz8;                  // 8 * nbx, 8 * nbx * nby
  __host__ __device__ static GradBricks make(int nx, int ny, int nz) {
    GradBricks b;
    b.nx = nx; b.ny = ny; b.nz = nz;
    b.fy8 = 8 * ((nx + 1) / 2);
    b.fz8 = b.fy8 * ((ny + 1) / 2);
    return b;
  }
  __host__ __device__ size_t cells() const { return (size_t)fz8 * ((nz + 1) / 2); }
  __device__ __forceinline__ int FX(int x) const { return ((x >> 1) << 3) + (x & 1); }
  __device__ __forceinline__ int FY(int y) const { return (y >> 1) * fy8 + ((y & 1) << 1); }
  __device__ __forceinline__ int FZ(int z) const { return (z >> 1) * fz8 + ((z & 1) << 2); }
};

__global__ void __launch_bounds__(256) grad_volume_kernel(GradBricks B, float sgx, float sgy, float sgz,
                                                          const float* __restrict__ vol, float4* __restrict__ gvol) {
  const size_t n = B.cells();
  const unsigned nbx = (unsigned)B.fy8 / 8u, nbxy = (unsigned)B.fz8 / 8u;
  const size_t sy = (size_t)B.nx, sz = (size_t)B.nx * B.ny;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const unsigned within = (unsigned)(i & 7), brick = (unsigned)(i >> 3);
    const unsigned bz = brick / nbxy, rem = brick - bz * nbxy;
    const unsigned by = rem / nbx, bx = rem - by * nbx;
    const int x = (int)(2 * bx + (within & 1)), y = (int)(2 * by + ((within >> 1) & 1)), z = (int)(2 * bz + (within >> 2));
    float4 g = make_float4(0.f, 0.f, 0.f, 0.f);
    if (x < B.nx && y < B.ny && z < B.nz) {
      const float* c = vol + (size_t)z * sz + (size_t)y * sy + x;
      g.x = sgx * ((x + 1 < B.nx ? __ldg(c + 1) : 0.f) - (x > 0 ? __ldg(c - 1) : 0.f));
      g.y = sgy * ((y + 1 < B.ny ? __ldg(c + sy) : 0.f) - (y > 0 ? __ldg(c - sy) : 0.f));
      g.z = sgz * ((z + 1 < B.nz ? __ldg(c + sz) : 0.f) - (z > 0 ? __ldg(c - sz) : 0.f));
      g.w = __ldg(c);
    }
    gvol[i] = g;
  }
}

__global__ void __launch_bounds__(256) pack_proj_kernel(int nu, int nv, int pu, int pv, size_t n_views,
                                                        const float* __restrict__ proj, float4* __restrict__ q) {
  const size_t per = (size_t)pu * pv, n = per * n_views;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t view = i / per;
    const int r = (int)(i - view * per);
    const int u = r % pu - kPadDet, v = r / pu - kPadDet;
    const float* img = proj + view * (size_t)nu * nv;
    const bool u0 = u >= 0 && u < nu, u1 = u + 1 >= 0 && u + 1 < nu;
    const bool v0 = v >= 0 && v < nv, v1 = v + 1 >= 0 && v + 1 < nv;
    float4 c;
    c.x = (u0 && v0) ? __ldg(img + (size_t)v * nu + u) : 0.f;
    c.y = (u1 && v0) ? __ldg(img + (size_t)v * nu + u + 1) : 0.f;
    c.z = (u0 && v1) ? __ldg(img + (size_t)(v + 1) * nu + u) : 0.f;
    c.w = (u1 && v1) ? __ldg(img + (size_t)(v + 1) * nu + u + 1) : 0.f;
    q[i] = c;
  }
}

// ------------------------------------------------------------------------------------------------ ray set-up
// a2 (Eq.2a :67-69: the delta selects the source->pixel line).  Runs once per ray in fp64 so that the
// fp32 march starts from correctly rounded constants: sample kappa sits at centred-index position
// pm + kappa*dp (+0.5, folded out for the magic floor), kappa = k - kref, tau_k = (k + 1/2) D.
// The march keeps the ray in DOUBLE (pm, dp: 12 registers, touched once per chunk / group of samples) and re-bases it
// every few samples onto a nearby integer origin, so that the fp32 position of a sample is a small number (|q| < 32)
// with an error of ~1e-6 voxel - instead of 3e-5 for a 512^3 volume if the fp32 position ran over the whole grid.
// The interpolation weights inherit that error; it is what the pose-gradient sums are most sensitive to.
struct Ray {
  double pm[3];            // centred-index position of sample kappa = 0, minus 0.5
  double dp[3];            // centred-index step per sample
  int k0, n;               // first kappa and sample count (n <= 0: the ray misses the clip box)
};

__device__ __forceinline__ Ray setup_ray(const FwdGeom& G, const FwdView& V, int iu, int iv, double* e_mm,
                                         double* ref_mm) {
  const double dx = V.d0[0] + iu * V.du[0] + iv * V.dv[0];
  const double dy = V.d0[1] + iu * V.du[1] + iv * V.dv[1];
  const double dz = V.d0[2] + iu * V.du[2] + iv * V.dv[2];
  const double inv = 1.0 / sqrt(dx * dx + dy * dy + dz * dz);
  const double e[3] = {dx * inv, dy * inv, dz * inv};
  const double iv3[3] = {1.0 / (double)G.vx, 1.0 / (double)G.vy, 1.0 / (double)G.vz};
  const double c3[3] = {G.cx, G.cy, G.cz};
  const double f3[3] = {G.L.fx, G.L.fy, G.L.fz};
  double ps[3], pe[3];
  double tmin = 0.0, tmax = 1e30;
  bool hit = true;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    ps[a] = (V.src[a] - c3[a]) * iv3[a] + f3[a];
    pe[a] = e[a] * iv3[a];
    const double lo = G.lo[a], hi = G.hi[a];
    if (fabs(pe[a]) > 1e-14) {
      double t0 = (lo - ps[a]) / pe[a], t1 = (hi - ps[a]) / pe[a];
      if (t0 > t1) { const double s = t0; t0 = t1; t1 = s; }
      tmin = fmax(tmin, t0);
      tmax = fmin(tmax, t1);
    } else if (ps[a] < lo || ps[a] > hi) {
      hit = false;
    }
  }
  const double D = G.step;
  Ray r;
  // tau_k = (k + 1/2) D in [tmin, tmax]
  const double kf0 = ceil(tmin / D - 0.5), kf1 = floor(tmax / D - 0.5);
  const int k0 = (int)fmax(kf0, 0.0);
  const int k1 = (int)fmin(kf1, 1.0e9);
  r.n = hit ? (k1 - k0 + 1) : 0;
  r.k0 = k0 - G.kref;
  const double tref = (G.kref + 0.5) * D;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    r.pm[a] = ps[a] + tref * pe[a] - 0.5;
    r.dp[a] = D * pe[a];
  }
  if (e_mm) {
#pragma unroll
    for (int a = 0; a < 3; ++a) { e_mm[a] = e[a]; ref_mm[a] = V.src[a] + tref * e[a]; }
  }
  return r;
}

// Re-based march of the gather kernels: groups of kRebase samples share an integer origin (the rounded position of the
// group's first sample); inside a group the position is fma(j, dp, b) with |b| <= 1/2, j < kRebase.
constexpr int kRebase = 16;
struct RayGroup {
  float bx, by, bz;        // position of the group's first sample minus the origin
  int ox, oy, oz;          // origin (centred index)
};
__device__ __forceinline__ RayGroup ray_group(const Ray& r, int kappa) {
  RayGroup g;
  const double k = (double)kappa;
  const double px = fma(k, r.dp[0], r.pm[0]), py = fma(k, r.dp[1], r.pm[1]), pz = fma(k, r.dp[2], r.pm[2]);
  const double rx = rint(px), ry = rint(py), rz = rint(pz);
  g.ox = (int)rx; g.oy = (int)ry; g.oz = (int)rz;
  g.bx = (float)(px - rx); g.by = (float)(py - ry); g.bz = (float)(pz - rz);
  return g;
}
// Exact cell and fractions of one sample (fp64): the slow path of the exact-interpolant gradient mode, whose
// integrand is discontinuous at cell faces - a sample within fp32 rounding of a face takes its cell from here.
__device__ __forceinline__ void exact_cell(const Ray& r, int kappa, int* cell, float* frac) {
  const double k = (double)kappa;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double p = fma(k, r.dp[a], r.pm[a]) + 0.5;        // centred-index position
    const double f = floor(p);
    cell[a] = (int)f;
    frac[a] = (float)(p - f);
  }
}
constexpr float kFaceEps = 6e-6f;      // |fraction - {0,1}| below this: the fp32 cell decision is not trusted

// pixel of this thread: warps are 8(u) x 4(v) patches, (kFwdTU/8) x (kFwdTV/4) warps per block
__device__ __forceinline__ void fwd_pixel(int& iu, int& iv) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  iu = blockIdx.x * kFwdTU + (warp % (kFwdTU / 8)) * 8 + (lane & 7);
  iv = blockIdx.y * kFwdTV + (warp / (kFwdTU / 8)) * 4 + (lane >> 3);
}

// ------------------------------------------------------------------------------------------------ a3 forward
// l_i = D sum_k f~(r'_k)  (Eq.18 :172-177 with a^ij = D * trilinear weight; U1).
// Cell index of the sample's base voxel from the magic-rounded coordinates (VolLayout): 3 LOP + 6 IMAD/LEA.
__device__ __forceinline__ unsigned brick_index(const VolLayout& L, unsigned X, unsigned Y, unsigned Z) {
  return X + 3u * (X & ~1u) + 2u * Y + L.by * (Y & ~1u) + 4u * Z + L.bz * (Z & ~1u) + L.c0;
}
// position, magic-rounded cell bits (kMagicBits + centred cell index) and fractions of sample j of a group
struct SamplePos {
  unsigned X, Y, Z;
  float ax, ay, az;
};
__device__ __forceinline__ SamplePos sample_pos(const RayGroup& g, float jf, float dpx, float dpy, float dpz) {
  SamplePos s;
  const float qx = fmaf(jf, dpx, g.bx), qy = fmaf(jf, dpy, g.by), qz = fmaf(jf, dpz, g.bz);
  const float tx = qx + kMagic, ty = qy + kMagic, tz = qz + kMagic;
  s.ax = (qx - (tx - kMagic)) + 0.5f; s.ay = (qy - (ty - kMagic)) + 0.5f; s.az = (qz - (tz - kMagic)) + 0.5f;
  s.X = (unsigned)(__float_as_int(tx) + g.ox); s.Y = (unsigned)(__float_as_int(ty) + g.oy);
  s.Z = (unsigned)(__float_as_int(tz) + g.oz);
  return s;
}

__global__ void __launch_bounds__(kFwdThreads) fwd_project_kernel(FwdGeom G, const FwdView* __restrict__ views,
                                                                  const float4* __restrict__ pvol,
                                                                  float* __restrict__ proj) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  if (iu >= G.nu || iv >= G.nv) return;
  const Ray r = setup_ray(G, views[view], iu, iv, nullptr, nullptr);
  const float dpx = (float)r.dp[0], dpy = (float)r.dp[1], dpz = (float)r.dp[2];
  const unsigned dz1 = 2u * G.L.bz + 4u;     // FZ(Z+1) - FZ(Z) for odd Z (4 for even Z)
  float sum = 0.f;
  for (int g0 = 0; g0 < r.n; g0 += kRebase) {
    const RayGroup grp = ray_group(r, r.k0 + g0);
    const int m = min(kRebase, r.n - g0);
    float jf = 0.f;
    for (int j = 0; j < m; ++j) {
      const SamplePos sp = sample_pos(grp, jf, dpx, dpy, dpz);
      const unsigned idx = brick_index(G.L, sp.X, sp.Y, sp.Z);
      const unsigned up = (sp.Z & 1u) ? dz1 : 4u;
      const float4 c0 = ldg4(pvol + idx), c1 = ldg4(pvol + (idx + up));
      const float r00 = lerp(sp.ax, c0.x, c0.y), r10 = lerp(sp.ax, c0.z, c0.w);
      const float r01 = lerp(sp.ax, c1.x, c1.y), r11 = lerp(sp.ax, c1.z, c1.w);
      sum += lerp(sp.az, lerp(sp.ay, r00, r10), lerp(sp.ay, r01, r11));
      jf += 1.0f;
    }
  }
  proj[((size_t)view * G.nv + iv) * G.nu + iu] = G.step * sum;
}

// a5, first stage, shared by the gradient kernels that keep one 6-vector per ray: warp shuffle, then across the
// block's warps through shared memory in fixed order -> partials[view][block][6] (deterministic, no atomics).
template <int NTHREADS>
__device__ __forceinline__ void reduce6_to_partials(float (&out)[6], float* __restrict__ partials, int view) {
  __shared__ float red[NTHREADS / 32][6];
#pragma unroll
  for (int q = 0; q < 6; ++q) {
    float v = out[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    out[q] = v;
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) {
#pragma unroll
    for (int q = 0; q < 6; ++q) red[warp][q] = out[q];
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    float s = 0.f;
#pragma unroll
    for (int wI = 0; wI < NTHREADS / 32; ++wI) s += red[wI][threadIdx.x];
    const size_t blk = (size_t)blockIdx.y * gridDim.x + blockIdx.x;
    const size_t nblk = (size_t)gridDim.x * gridDim.y;
    partials[((size_t)view * nblk + blk) * 6 + threadIdx.x] = s;
  }
}

// ------------------------------------------------------------------------------------------------ a4 gradient
// Per ray (Eq.7-8 :101-113, Eq.19 :179-183, on the fly per :207):
//   A_i = D sum_k g~(r'_k),  B_i = D sum_k r'_k x g~(r'_k),  g~_a = [f~(r'+v_a e_a) - f~(r'-v_a e_a)] / (2 v_a).
// Shifting by one voxel keeps the fractional weights, so each g~_a is ONE trilinear interpolation of voxel
// differences: 32 distinct voxels per sample, fetched as 16 float2 cells.  With r'_k = r_ref + kappa D e:
//   B_i = D [ r_ref x sum g + D e x sum kappa g ]     -> six running sums (sum g, sum kappa g) per ray.
// Block result: sum_i w_i A_i, sum_i w_i B_i over the block's rays -> partials[view][block][6]   (Eq.20 :185).
// MODE 0: central differences of f~ (the paper's, 32 voxels); MODE 1 (DFP_FLAG_GRAD_INTERP): exact derivative of the
// trilinear interpolant in the sample's cell (the forward kernel's 8 voxels; G.sg* = 1 / pitch instead of 1 / 2 pitch).
template <int MODE>
__global__ void __launch_bounds__(kFwdThreads) fwd_grad_kernel(FwdGeom G, const FwdView* __restrict__ views,
                                                               const float4* __restrict__ pvol,
                                                               const float* __restrict__ upstream,
                                                               float* __restrict__ partials) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  const bool live = iu < G.nu && iv < G.nv;
  float out[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (live) {
    double e_mm[3], ref_mm[3];
    const Ray r = setup_ray(G, views[view], iu, iv, e_mm, ref_mm);
    const float dpx = (float)r.dp[0], dpy = (float)r.dp[1], dpz = (float)r.dp[2];
    const unsigned by8 = 2u * G.L.by + 4u;          // 8*nbx:     FY(Y+2) - FY(Y)
    const unsigned bz8 = 2u * G.L.bz + 8u;          // 8*nbx*nby: FZ(Z+2) - FZ(Z)
    float gx = 0.f, gy = 0.f, gz = 0.f, hx = 0.f, hy = 0.f, hz = 0.f;
    for (int g0 = 0; g0 < r.n; g0 += kRebase) {
    const RayGroup grp = ray_group(r, r.k0 + g0);
    const int m = min(kRebase, r.n - g0);
    float jf = 0.f, kf = (float)(r.k0 + g0);
    for (int j = 0; j < m; ++j) {
      SamplePos sp = sample_pos(grp, jf, dpx, dpy, dpz);
      if (MODE == 1) {
        // the derivative of the interpolant jumps at cell faces: a sample within fp32 rounding of one takes its cell
        // (and fractions) from the fp64 position, as the oracle does
        const float mn = fminf(fminf(fminf(sp.ax, 1.f - sp.ax), fminf(sp.ay, 1.f - sp.ay)), fminf(sp.az, 1.f - sp.az));
        if (mn < kFaceEps) {
          int cell[3];
          float fr[3];
          exact_cell(r, r.k0 + g0 + j, cell, fr);
          sp.X = (unsigned)(kMagicBits + cell[0]); sp.Y = (unsigned)(kMagicBits + cell[1]); sp.Z = (unsigned)(kMagicBits + cell[2]);
          sp.ax = fr[0]; sp.ay = fr[1]; sp.az = fr[2];
        }
      }
      const float ax = sp.ax, ay = sp.ay, az = sp.az;
      const unsigned idx = brick_index(G.L, sp.X, sp.Y, sp.Z);
      float ddx, ddy, ddz;
      if (MODE == 1) {
        const unsigned up = (sp.Z & 1u) ? bz8 - 4u : 4u;                                  // FZ(Z+1) - FZ(Z)
        const float4 c0 = ldg4(pvol + idx), c1 = ldg4(pvol + (idx + up));                // slices z, z+1: rows y, y+1
        const float d00 = c0.y - c0.x, d10 = c0.w - c0.z, d01 = c1.y - c1.x, d11 = c1.w - c1.z;
        const float r00 = fmaf(ax, d00, c0.x), r10 = fmaf(ax, d10, c0.z);
        const float r01 = fmaf(ax, d01, c1.x), r11 = fmaf(ax, d11, c1.z);
        ddx = lerp(az, lerp(ay, d00, d10), lerp(ay, d01, d11));
        ddy = lerp(az, r10 - r00, r11 - r01);
        ddz = lerp(ay, r01, r11) - lerp(ay, r00, r10);
      } else {
      // neighbour cells: +-1 along an axis stays inside the brick or hops to the next one, by parity
      const unsigned ox = sp.X & 1u, oy = sp.Y & 1u, oz = sp.Z & 1u;
      const unsigned dxp = 1u + 6u * ox, dxm = dxp - 8u;
      const unsigned dyp = 2u + (by8 - 4u) * oy, dym = dyp - by8;
      const unsigned dzp = 4u + (bz8 - 8u) * oz, dzm = dzp - bz8;
      float rv[2][2], rdx[2][2], rym[2], ryp[2];
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const unsigned b = k ? idx + dzp : idx;
        const float4 A = ldg4(pvol + (b + dxm)), B = ldg4(pvol + (b + dxp));   // x-1,x | x+1,x+2 ; rows y, y+1
        const float4 C = ldg4(pvol + (b + dym)), D = ldg4(pvol + (b + dyp));   // x,x+1 ; rows y-1,y | y+1,y+2
        rv[0][k] = lerp(ax, A.y, B.x);
        rv[1][k] = lerp(ax, A.w, B.z);
        rdx[0][k] = lerp(ax, B.x - A.x, B.y - A.y);
        rdx[1][k] = lerp(ax, B.z - A.z, B.w - A.w);
        rym[k] = lerp(ax, C.x, C.y);
        ryp[k] = lerp(ax, D.z, D.w);
      }
      float rzm[2], rzp[2];
      {
        const float4 E = ldg4(pvol + (idx + dzm)), F = ldg4(pvol + (idx + bz8));  // slices z-1, z+2; rows y, y+1
        rzm[0] = lerp(ax, E.x, E.y); rzm[1] = lerp(ax, E.z, E.w);
        rzp[0] = lerp(ax, F.x, F.y); rzp[1] = lerp(ax, F.z, F.w);
      }
      ddx = lerp(az, lerp(ay, rdx[0][0], rdx[1][0]), lerp(ay, rdx[0][1], rdx[1][1]));
      const float dy0 = lerp(ay, rv[1][0] - rym[0], ryp[0] - rv[0][0]);
      const float dy1 = lerp(ay, rv[1][1] - rym[1], ryp[1] - rv[0][1]);
      ddy = lerp(az, dy0, dy1);
      const float dz0 = lerp(az, rv[0][1] - rzm[0], rzp[0] - rv[0][0]);
      const float dz1 = lerp(az, rv[1][1] - rzm[1], rzp[1] - rv[1][0]);
      ddz = lerp(ay, dz0, dz1);
      }
      gx += ddx; gy += ddy; gz += ddz;
      hx = fmaf(kf, ddx, hx); hy = fmaf(kf, ddy, hy); hz = fmaf(kf, ddz, hz);
      kf += 1.0f;
      jf += 1.0f;
    }
    }
    // per-ray epilogue (once per ray): scale to per-mm gradients, lever arm about the reference sample
    const float w = upstream ? __ldg(upstream + ((size_t)view * G.nv + iv) * G.nu + iu) : 1.f;   // null: unit weights
    const float D = G.step;
    const float sx = gx * G.sgx, sy = gy * G.sgy, sz = gz * G.sgz;            // sum g  (per mm)
    const float mx = hx * G.sgx * D, my = hy * G.sgy * D, mz = hz * G.sgz * D; // D sum kappa g
    const float ex = (float)e_mm[0], ey = (float)e_mm[1], ez = (float)e_mm[2];
    const float px = (float)ref_mm[0], py = (float)ref_mm[1], pz = (float)ref_mm[2];
    const float wd = w * D;
    out[0] = wd * sx; out[1] = wd * sy; out[2] = wd * sz;
    out[3] = wd * ((py * sz - pz * sy) + (ey * mz - ez * my));
    out[4] = wd * ((pz * sx - px * sz) + (ez * mx - ex * mz));
    out[5] = wd * ((px * sy - py * sx) + (ex * my - ey * mx));
  }
  reduce6_to_partials<kFwdThreads>(out, partials, view);
}

// a5, second stage: one block per view, fp64, fixed summation order (deterministic), then the 6x6 contraction
//   dL/dt = -R S_A,  dL/dgamma_k = -w_k . S_B          (PAPER.md :79: grad_theta = grad_theta M . grad_M)
__global__ void __launch_bounds__(256) fwd_contract_kernel(int nblk, const float* __restrict__ partials,
                                                           const FwdContract* __restrict__ con,
                                                           float* __restrict__ grad, int gstride = 6, int goff = 0) {
  const int view = blockIdx.x;
  __shared__ double sh[8][6];
  double acc[6] = {0, 0, 0, 0, 0, 0};
  const float* p = partials + (size_t)view * nblk * 6;
  for (int b = threadIdx.x; b < nblk; b += blockDim.x)
#pragma unroll
    for (int q = 0; q < 6; ++q) acc[q] += (double)p[(size_t)b * 6 + q];
#pragma unroll
  for (int q = 0; q < 6; ++q)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
  if ((threadIdx.x & 31) == 0)
#pragma unroll
    for (int q = 0; q < 6; ++q) sh[threadIdx.x >> 5][q] = acc[q];
  __syncthreads();
  if (threadIdx.x == 0) {
    double S[6];
    for (int q = 0; q < 6; ++q) {
      double s = 0;
      for (int wI = 0; wI < 8; ++wI) s += sh[wI][q];
      S[q] = s;
    }
    const FwdContract& C = con[view];
    for (int a = 0; a < 3; ++a) {
      grad[view * gstride + goff + a] = (float)(-(C.R[a * 3 + 0] * S[0] + C.R[a * 3 + 1] * S[1] + C.R[a * 3 + 2] * S[2]));
      grad[view * gstride + goff + 3 + a] =
          (float)(-(C.w[a * 3 + 0] * S[3] + C.w[a * 3 + 1] * S[4] + C.w[a * 3 + 2] * S[5]));
    }
  }
}

// ray-step count of the metric: samples whose position lies in the clip box, summed over all rays
__global__ void __launch_bounds__(kFwdThreads) count_steps_kernel(FwdGeom G, const FwdView* __restrict__ views,
                                                                  unsigned long long* __restrict__ total) {
  int iu, iv;
  fwd_pixel(iu, iv);
  long long n = 0;
  if (iu < G.nu && iv < G.nv) {
    const Ray r = setup_ray(G, views[blockIdx.z], iu, iv, nullptr, nullptr);
    n = r.n > 0 ? r.n : 0;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xffffffffu, n, o);
  if ((threadIdx.x & 31) == 0 && n) atomicAdd(total, (unsigned long long)n);
}

// ------------------------------------------------------------------------------------------------ a6 back
// mu_j = sum_v W b~_v(u, v),  (u', v', w') = P_eff,v (r'_j; 1)   (Eq.1 :60-63, Eq.21 :193-196).
// A[0], A[1] arrive with 0.5*A[2] already subtracted (u - 1/2 for the magic floor) - see bp_fold_half().
struct BpPix {
  float a, b;        // fractional weights along u, v
  unsigned idx;      // packed cell index of (floor u, floor v) within the view
  float rw;          // 1 / w'
  float uq, vq;      // clamped (u - 1/2), (v - 1/2) in CU/CV-centred pixel units
  bool front;        // w' > 0
};

__device__ __forceinline__ BpPix bp_locate(float up, float vp, float wp, float ulo, float uhi, float vlo, float vhi,
                                           unsigned pu, unsigned C0) {
  BpPix o;
  float r = fast_rcp(wp);
  o.front = wp > 0.f;
  o.rw = r;
  // fminf/fmaxf drop NaNs, so a degenerate w' cannot produce an out-of-range index
  o.uq = fminf(fmaxf(up * r, ulo), uhi);
  o.vq = fminf(fmaxf(vp * r, vlo), vhi);
  const float tu = o.uq + kMagic, tv = o.vq + kMagic;
  o.a = (o.uq - (tu - kMagic)) + 0.5f;
  o.b = (o.vq - (tv - kMagic)) + 0.5f;
  o.idx = (unsigned)__float_as_int(tv) * pu + (unsigned)__float_as_int(tu) + C0;
  return o;
}

template <int WEIGHT>
__global__ void __launch_bounds__(kBpThreads) bp_kernel(BpGeom G, int n_views, const BpView* __restrict__ views,
                                                        const float4* __restrict__ q, float* __restrict__ vol) {
  const int ix = blockIdx.x * kBpTX + (threadIdx.x & (kBpTX - 1));
  const int iy = blockIdx.y * kBpTY + threadIdx.x / kBpTX;
  const int z0 = blockIdx.z * kBpZ;
  __shared__ BpView sv;
  const float xf = (float)ix - G.hx, yf = (float)iy - G.hy, zf = (float)z0 - G.hz;
  // clamp range of (u - 1/2) in CU-centred units: u in [-1, nu]
  const float ulo = -1.5f - (float)G.CU, uhi = (float)(G.nu - G.CU) - 0.5f;
  const float vlo = -1.5f - (float)G.CV, vhi = (float)(G.nv - G.CV) - 0.5f;
  const unsigned pu = G.pu;
  const unsigned C0 = (unsigned)(G.CV + kPadDet) * pu + (unsigned)(G.CU + kPadDet) - (unsigned)kMagicBits * (pu + 1u);
  const size_t per = (size_t)G.pu * G.pv;
  float acc[kBpZ];
#pragma unroll
  for (int m = 0; m < kBpZ; ++m)   // DFP_FLAG_ACCUMULATE: start from the caller's volume (a slice of the views)
    acc[m] = ((G.flags & DFP_FLAG_ACCUMULATE) && ix < G.nx && iy < G.ny && z0 + m < G.nz)
                 ? vol[((size_t)(z0 + m) * G.ny + iy) * G.nx + ix] : 0.f;
  for (int view = 0; view < n_views; ++view) {
    __syncthreads();
    if (threadIdx.x < sizeof(BpView) / 4) ((float*)&sv)[threadIdx.x] = ((const float*)(views + view))[threadIdx.x];
    __syncthreads();
    const float ub = fmaf(sv.A[0][0], xf, fmaf(sv.A[0][1], yf, fmaf(sv.A[0][2], zf, sv.A[0][3])));
    const float vb = fmaf(sv.A[1][0], xf, fmaf(sv.A[1][1], yf, fmaf(sv.A[1][2], zf, sv.A[1][3])));
    const float wb = fmaf(sv.A[2][0], xf, fmaf(sv.A[2][1], yf, fmaf(sv.A[2][2], zf, sv.A[2][3])));
    const float4* img = q + (size_t)view * per;
#pragma unroll
    for (int m = 0; m < kBpZ; ++m) {
      const float mf = (float)m;
      const BpPix p = bp_locate(fmaf(mf, sv.A[0][2], ub), fmaf(mf, sv.A[1][2], vb), fmaf(mf, sv.A[2][2], wb), ulo,
                                uhi, vlo, vhi, pu, C0);
      const float4 c = ldg4(img + p.idx);
      const float val = lerp(p.b, lerp(p.a, c.x, c.y), lerp(p.a, c.z, c.w));
      float wgt = WEIGHT ? G.sad2 * p.rw * p.rw : 1.f;
      wgt = p.front ? wgt : 0.f;
      acc[m] = fmaf(wgt, val, acc[m]);
    }
  }
  if (ix < G.nx && iy < G.ny) {
#pragma unroll
    for (int m = 0; m < kBpZ; ++m)
      if (z0 + m < G.nz) vol[((size_t)(z0 + m) * G.ny + iy) * G.nx + ix] = acc[m];
  }
}

// ------------------------------------------------------------------------------------------------ a7 back gradient
// Per (voxel j, view) in the OBJECT frame (Eq.12-17 :139-168, Eq.22 :198-206):
//   q' = W [ d~_u l (J1 - u J3) + d~_v l (J2 - v J3) ] / w'   (+ b~ dW/dr' if DW),   J_r = P_eff[r][0:3]
//   S'_q += w_j q',  S'_c += w_j r'_j x q';   along the thread's z column r'_j = r'_0 + m vz e_z, so
//   S'_c = r'_0 x sum(w q') + vz e_z x sum(m w q')  -> six running sums per (thread, view).
// d~_u l = [b~(u+1,v) - b~(u-1,v)]/2 is ONE bilinear interpolation of pixel differences: 12 distinct pixels,
// fetched as 4 quad cells.  Result: partials[tile][view][6].
// MODE 1 (DFP_FLAG_GRAD_INTERP): d_u l, d_v l = exact derivatives of the bilinear interpolant (the 4 pixels of b~).
template <int WEIGHT, int DW, int MODE>
__global__ void __launch_bounds__(kBpThreads) bp_grad_kernel(BpGeom G, int n_views, int zchunk,
                                                             const BpView* __restrict__ views,
                                                             const BpViewD* __restrict__ viewsd,
                                                             const float4* __restrict__ q,
                                                             const float* __restrict__ upstream,
                                                             float* __restrict__ partials) {
  const int ix = blockIdx.x * kBpTX + (threadIdx.x & (kBpTX - 1));
  const int iy = blockIdx.y * kBpTY + threadIdx.x / kBpTX;
  const int z0 = blockIdx.z * zchunk;
  const int z1 = min(z0 + zchunk, G.nz);
  const bool live = ix < G.nx && iy < G.ny;
  __shared__ BpView sv;
  __shared__ float red[kBpThreads / 32][6];
  const float xf = (float)ix - G.hx, yf = (float)iy - G.hy, zf = (float)z0 - G.hz;
  // clamp range of (u - 1/2): u in [-2, nu+1] (support of the central difference of b~)
  const float ulo = -2.5f - (float)G.CU, uhi = (float)(G.nu - G.CU) + 0.5f;
  const float vlo = -2.5f - (float)G.CV, vhi = (float)(G.nv - G.CV) + 0.5f;
  const unsigned pu = G.pu;
  const unsigned C0 = (unsigned)(G.CV + kPadDet) * pu + (unsigned)(G.CU + kPadDet) - (unsigned)kMagicBits * (pu + 1u);
  const size_t per = (size_t)G.pu * G.pv;
  const size_t tile = ((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
  // object-frame mm of the column's first voxel
  const float rx = G.cx + xf * G.vx, ry = G.cy + yf * G.vy, rz = G.cz + zf * G.vz;
  const float* wcol = upstream + ((size_t)z0 * G.ny + (live ? iy : 0)) * G.nx + (live ? ix : 0);
  const size_t wstride = (size_t)G.ny * G.nx;
  for (int view = 0; view < n_views; ++view) {
    __syncthreads();
    if (threadIdx.x < sizeof(BpView) / 4) ((float*)&sv)[threadIdx.x] = ((const float*)(views + view))[threadIdx.x];
    __syncthreads();
    float s[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (live) {
      const float ub = fmaf(sv.A[0][0], xf, fmaf(sv.A[0][1], yf, fmaf(sv.A[0][2], zf, sv.A[0][3])));
      const float vb = fmaf(sv.A[1][0], xf, fmaf(sv.A[1][1], yf, fmaf(sv.A[1][2], zf, sv.A[1][3])));
      const float wb = fmaf(sv.A[2][0], xf, fmaf(sv.A[2][1], yf, fmaf(sv.A[2][2], zf, sv.A[2][3])));
      const float4* img = q + (size_t)view * per;
      float mf = 0.f;
      for (int z = z0; z < z1; ++z) {
        BpPix p = bp_locate(fmaf(mf, sv.A[0][2], ub), fmaf(mf, sv.A[1][2], vb), fmaf(mf, sv.A[2][2], wb), ulo,
                            uhi, vlo, vhi, pu, C0);
        if (MODE == 1 && fminf(fminf(p.a, 1.f - p.a), fminf(p.b, 1.f - p.b)) < 1e-4f) {
          // the derivative of the bilinear interpolant jumps at pixel boundaries: a voxel that projects within fp32
          // rounding of one (|u - c_u| <= n/2 pixels in fp32: up to 3e-5 pixel) takes its cell and fractions from the
          // fp64 rows, as the oracle does
          const double* Ad = reinterpret_cast<const double*>(viewsd + view);
          const double X = (double)xf, Y = (double)yf, Z = (double)zf + (double)mf;
          const double wd = fma(__ldg(Ad + 8), X, fma(__ldg(Ad + 9), Y, fma(__ldg(Ad + 10), Z, __ldg(Ad + 11))));
          double ud = fma(__ldg(Ad + 0), X, fma(__ldg(Ad + 1), Y, fma(__ldg(Ad + 2), Z, __ldg(Ad + 3)))) / wd;
          double vd = fma(__ldg(Ad + 4), X, fma(__ldg(Ad + 5), Y, fma(__ldg(Ad + 6), Z, __ldg(Ad + 7)))) / wd;
          ud = fmin(fmax(ud, (double)ulo), (double)uhi) + 0.5;
          vd = fmin(fmax(vd, (double)vlo), (double)vhi) + 0.5;
          const double fu = floor(ud), fv = floor(vd);
          p.a = (float)(ud - fu); p.b = (float)(vd - fv);
          p.idx = (unsigned)((int)fv + G.CV + kPadDet) * pu + (unsigned)((int)fu + G.CU + kPadDet);
        }
        const float4* c = img + p.idx;
        float dlu, dlv, b00, b01, b10, b11;            // (x2 for MODE 0) interpolated differences; the 4 pixels of b~
        if (MODE == 1) {
          const float4 q0 = ldg4(c);                   // l[v][u], l[v][u+1], l[v+1][u], l[v+1][u+1]
          dlu = lerp(p.b, q0.y - q0.x, q0.w - q0.z);
          dlv = lerp(p.a, q0.z - q0.x, q0.w - q0.y);
          b00 = q0.x; b01 = q0.y; b10 = q0.z; b11 = q0.w;
        } else {
          const float4 cl = ldg4(c - 1), cr = ldg4(c + 1);      // rows v, v+1; columns u-1,u | u+1,u+2
          const float4 cd = ldg4(c - pu), cu = ldg4(c + pu);    // columns u, u+1; rows v-1,v | v+1,v+2
          // d~_u l (x2): per row lerp_a(l[u+1]-l[u-1], l[u+2]-l[u]), then lerp_b over the two rows
          const float du0 = lerp(p.a, cr.x - cl.x, cr.y - cl.y);
          const float du1 = lerp(p.a, cr.z - cl.z, cr.w - cl.w);
          dlu = lerp(p.b, du0, du1);
          // d~_v l (x2): per column lerp_b(l[v+1]-l[v-1], l[v+2]-l[v]), then lerp_a over the two columns
          const float dv0 = lerp(p.b, cu.x - cd.x, cu.z - cd.z);
          const float dv1 = lerp(p.b, cu.y - cd.y, cu.w - cd.w);
          dlv = lerp(p.a, dv0, dv1);
          b00 = cl.y; b01 = cr.x; b10 = cl.w; b11 = cr.z;
        }
        const float wj = __ldg(wcol + (size_t)(z - z0) * wstride);
        float W = WEIGHT ? G.sad2 * p.rw * p.rw : 1.f;
        W = p.front ? W : 0.f;
        // u, v of Eq.13 in the same (CU-centred, minus 1/2) units as the folded rows J1, J2
        const float cc = fmaf(dlu, p.uq, dlv * p.vq);
        float qx = fmaf(dlu, sv.J[0][0], fmaf(dlv, sv.J[1][0], -cc * sv.J[2][0]));
        float qy = fmaf(dlu, sv.J[0][1], fmaf(dlv, sv.J[1][1], -cc * sv.J[2][1]));
        float qz = fmaf(dlu, sv.J[0][2], fmaf(dlv, sv.J[1][2], -cc * sv.J[2][2]));
        float sc = (MODE == 1 ? 1.0f : 0.5f) * W * p.rw * wj;
        if (DW) {
          // + b~ dW/dr',  dW/dr' = -2 W / w' * J3   (U8); b~ from the same cells
          const float b0 = lerp(p.a, b00, b01), b1 = lerp(p.a, b10, b11);
          const float bv = lerp(p.b, b0, b1);
          const float k = (MODE == 1 ? -2.f : -4.f) * bv;      // relative to the common factor (0.5) W / w'
          qx = fmaf(k, sv.J[2][0], qx); qy = fmaf(k, sv.J[2][1], qy); qz = fmaf(k, sv.J[2][2], qz);
        }
        s[0] = fmaf(sc, qx, s[0]); s[1] = fmaf(sc, qy, s[1]); s[2] = fmaf(sc, qz, s[2]);
        const float scm = sc * mf;
        s[3] = fmaf(scm, qx, s[3]); s[4] = fmaf(scm, qy, s[4]); s[5] = fmaf(scm, qz, s[5]);
        mf += 1.0f;
      }
      // S'_c of the column: r'_0 x sum(w q') + vz e_z x sum(m w q')
      const float mx = s[3] * G.vz, my = s[4] * G.vz;
      const float cx = ry * s[2] - rz * s[1] - my;
      const float cy = rz * s[0] - rx * s[2] + mx;
      const float cz = rx * s[1] - ry * s[0];
      s[3] = cx; s[4] = cy; s[5] = cz;
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      float v = s[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      s[k] = v;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) {
#pragma unroll
      for (int k = 0; k < 6; ++k) red[warp][k] = s[k];
    }
    __syncthreads();
    if (threadIdx.x < 6) {
      float t = 0.f;
#pragma unroll
      for (int wI = 0; wI < kBpThreads / 32; ++wI) t += red[wI][threadIdx.x];
      partials[(tile * n_views + view) * 6 + threadIdx.x] = t;
    }
  }
}

// a8: one block per view, fp64, fixed order; dL/dt = R S'_q, dL/dgamma_k = (R^T a_k) . S'_c
__global__ void __launch_bounds__(256) bp_contract_kernel(int n_tiles, int n_views, const float* __restrict__ partials,
                                                          const BpContract* __restrict__ con,
                                                          float* __restrict__ grad) {
  const int view = blockIdx.x;
  __shared__ double sh[8][6];
  double acc[6] = {0, 0, 0, 0, 0, 0};
  for (int t = threadIdx.x; t < n_tiles; t += blockDim.x)
#pragma unroll
    for (int k = 0; k < 6; ++k) acc[k] += (double)partials[((size_t)t * n_views + view) * 6 + k];
#pragma unroll
  for (int k = 0; k < 6; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], o);
  if ((threadIdx.x & 31) == 0)
#pragma unroll
    for (int k = 0; k < 6; ++k) sh[threadIdx.x >> 5][k] = acc[k];
  __syncthreads();
  if (threadIdx.x == 0) {
    double S[6];
    for (int k = 0; k < 6; ++k) {
      double s = 0;
      for (int wI = 0; wI < 8; ++wI) s += sh[wI][k];
      S[k] = s;
    }
    const BpContract& C = con[view];
    for (int a = 0; a < 3; ++a) {
      grad[view * 6 + a] = (float)(C.R[a * 3 + 0] * S[0] + C.R[a * 3 + 1] * S[1] + C.R[a * 3 + 2] * S[2]);
      grad[view * 6 + 3 + a] = (float)(C.a[a * 3 + 0] * S[3] + C.a[a * 3 + 1] * S[4] + C.a[a * 3 + 2] * S[5]);
    }
  }
}

}  // namespace dfp
