// dfp_siddon.cuh - forward projection and its pose gradient with SIDDON weights (DFP_FLAG_SIDDON).
//
// Siddon's exact radiological path [28] is the weight model of the paper's own ray-driven projector (PAPER.md :213,
// ref :395): a^ij = length of ray i inside voxel j, voxels being boxes of constant value (Eq.18 :172-177).  The
// gradient follows the paper's discretisation literally (Eq.19-20 :179-191, :189): per voxel j of the grid,
// g_j = central differences of the zero-extended voxel values (:183) and the lever arm at the voxel centre r'_j;
//   A_i = sum_j a^ij g_j,  B_i = sum_j a^ij r'_j x g_j   -> six running sums per ray, never the 12-element G_f^j,
// then the same per-view reduction / contraction as the trilinear kernels (dL/dt = -R S_A, dL/dgamma_k = -w_k.S_B).
//
// One thread per ray, incremental 3-D DDA over the voxel grid (the merged plane-crossing list of Siddon's paper,
// generated in order instead of sorted).  Crossing PARAMETERS reach ~1000 mm while a segment is ~1 voxel long, so a
// length taken as a difference of two fp32 parameters would carry 1e-4 relative error; the set-up therefore runs in
// fp64 and the loop tracks only the (small) distances to the next crossings.  Values are read straight from the caller's
// volume through L1 (forward: one voxel per segment); the gradient reads one float4 of the per-voxel gradient volume
// (dfp_kernels.cuh: grad_volume_kernel) per segment.  No shared-memory staging: kernels for the "next" row, measured
// beside the trilinear ones in DESIGN.md.
#pragma once
#include <cuda_runtime.h>

#include "dfp_kernels.cuh"

namespace dfp {

struct SiddonRay {
  double t, tmax;              // current parameter (mm from the source) and exit parameter
  double tn[3], dt[3];         // next crossing of each plane family, spacing of the crossings
  int i[3], step[3];           // current voxel index, +-1 per axis
  int nseg;                    // number of segments = plane crossings between entry and exit + 1
  bool hit;
};

// Per-ray set-up (fp64, once per ray): the half-line s' + t e', t >= 0, against the grid box.
__device__ __forceinline__ SiddonRay siddon_setup(const FwdGeom& G, const FwdView& V, int iu, int iv, double* e_out) {
  const double dx = V.d0[0] + iu * V.du[0] + iv * V.dv[0];
  const double dy = V.d0[1] + iu * V.du[1] + iv * V.dv[1];
  const double dz = V.d0[2] + iu * V.du[2] + iv * V.dv[2];
  const double inv = 1.0 / sqrt(dx * dx + dy * dy + dz * dz);
  const double e[3] = {dx * inv, dy * inv, dz * inv};
  const int n[3] = {G.L.nx, G.L.ny, G.L.nz};
  const double v[3] = {(double)G.vx, (double)G.vy, (double)G.vz}, c[3] = {(double)G.cx, (double)G.cy, (double)G.cz};
  SiddonRay r;
  r.hit = true;
  double tmin = 0.0, tmax = 1e300, lo[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    lo[a] = c[a] - 0.5 * n[a] * v[a];
    const double hi = c[a] + 0.5 * n[a] * v[a], o = V.src[a];
    if (fabs(e[a]) < 1e-300) {
      if (o <= lo[a] || o >= hi) r.hit = false;
    } else {
      double t0 = (lo[a] - o) / e[a], t1 = (hi - o) / e[a];
      if (t0 > t1) { const double s = t0; t0 = t1; t1 = s; }
      tmin = fmax(tmin, t0);
      tmax = fmin(tmax, t1);
    }
  }
  if (!(tmax > tmin)) r.hit = false;
  r.t = tmin;
  r.tmax = tmax;
  r.nseg = 1;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double p = V.src[a] + tmin * e[a];
    int i = (int)floor((p - lo[a]) / v[a]);
    i = min(max(i, 0), n[a] - 1);
    r.i[a] = i;
    // voxel of the exit point: every plane of family a between the two indices is crossed once
    int ie = (int)floor((V.src[a] + fmin(tmax, 1e30) * e[a] - lo[a]) / v[a]);
    ie = min(max(ie, 0), n[a] - 1);
    r.nseg += abs(ie - i);
    if (fabs(e[a]) < 1e-300) {
      r.step[a] = 0; r.dt[a] = 1e300; r.tn[a] = 1e300;
    } else {
      r.step[a] = e[a] > 0 ? 1 : -1;
      r.dt[a] = v[a] / fabs(e[a]);
      r.tn[a] = (lo[a] + (i + (e[a] > 0 ? 1 : 0)) * v[a] - V.src[a]) / e[a];
    }
    if (e_out) e_out[a] = e[a];
  }
  return r;
}

// One DDA step: returns the length of the segment inside the current voxel, then advances the voxel offset and the
// crossed family's distance.
// The state keeps, per family, the distance from the CURRENT point to the next crossing (fp32, at most one crossing
// spacing, a few mm): a segment length is then the minimum of three small numbers, known to ~1e-7 relative, and
// the subtraction r_a - len is exact or rounds at 1e-7 of a spacing - no fp64 and no large parameter in the loop
// (the per-ray set-up, which does subtract parameters of ~1000 mm, runs in fp64).
// The loop runs SiddonRay::nseg times (counted by the fp64 set-up from the entry and exit voxels).  Where two
// crossings coincide to within the fp32 drift of the distances (~1e-5 mm) the loop may take them in the other order
// or count one more / fewer than the set-up did; every segment this misplaces is that short, and the voxel offset
// is clamped to the volume (clamp_offset), so such a step reads a valid voxel with a ~1e-5 mm weight.
// Branch-free on purpose: the three families take turns within a warp, and an if / else form compiled to a
// divergent branch with a dozen register moves per step.
struct SiddonState {
  float rx, ry, rz, dtx, dty, dtz;       // distance to the next x / y / z plane; spacing of the crossings
  int idx, stx, sty, stz;                // offset of the voxel and its step per family: linear in the caller's volume
                                         // (forward); GradBricks index and the step of the NEXT crossing (gradient)
  int ttx, tty, ttz;                     // gradient: step of this crossing + step of the following one (they alternate
                                         // with the parity of the index: inside the brick, then to the next brick)
  float px, py, pz, dpx, dpy, dpz;       // gradient: voxel centre r'_j (mm) and its step per family
};
template <bool BRICK>
__device__ __forceinline__ SiddonState siddon_state(const SiddonRay& r, const FwdGeom& G) {
  const int nx = G.L.nx, ny = G.L.ny, nz = G.L.nz;
  SiddonState s;
  s.rx = (float)fmin(r.tn[0] - r.t, 1e30); s.ry = (float)fmin(r.tn[1] - r.t, 1e30); s.rz = (float)fmin(r.tn[2] - r.t, 1e30);
  s.dtx = (float)fmin(r.dt[0], 1e30); s.dty = (float)fmin(r.dt[1], 1e30); s.dtz = (float)fmin(r.dt[2], 1e30);
  const int ix = r.i[0], iy = r.i[1], iz = r.i[2], sx = r.step[0], sy = r.step[1], sz = r.step[2];
  if (!BRICK) {
    s.idx = (iz * ny + iy) * nx + ix;
    s.stx = sx; s.sty = sy * nx; s.stz = sz * nx * ny;
  } else {
    const GradBricks B = GradBricks::make(nx, ny, nz);
    s.idx = B.FX(ix) + B.FY(iy) + B.FZ(iz);
    s.stx = B.FX(ix + sx) - B.FX(ix); s.ttx = 8 * sx;
    s.sty = B.FY(iy + sy) - B.FY(iy); s.tty = B.fy8 * sy;
    s.stz = B.FZ(iz + sz) - B.FZ(iz); s.ttz = B.fz8 * sz;
    // voxel centre r'_j = c + (i - (n-1)/2) v, stepped in fp32 (a few hundred additions of a pitch: ~1e-5 mm)
    s.px = fmaf((float)ix - 0.5f * (float)(nx - 1), G.vx, G.cx); s.dpx = (float)sx * G.vx;
    s.py = fmaf((float)iy - 0.5f * (float)(ny - 1), G.vy, G.cy); s.dpy = (float)sy * G.vy;
    s.pz = fmaf((float)iz - 0.5f * (float)(nz - 1), G.vz, G.cz); s.dpz = (float)sz * G.vz;
  }
  return s;
}
// offset into [0, last]: a negative offset wraps to a large unsigned number and lands on `last`
__device__ __forceinline__ unsigned clamp_offset(int idx, unsigned last) { return min((unsigned)idx, last); }

template <bool BRICK>
__device__ __forceinline__ float siddon_step(SiddonState& s) {
  const bool cx = s.rx <= s.ry && s.rx <= s.rz;
  const bool cy = !cx && s.ry <= s.rz;
  const bool cz = !cx && !cy;
  const float len = fmaxf(cx ? s.rx : (cy ? s.ry : s.rz), 0.f);
  s.rx = cx ? s.dtx : s.rx - len;
  s.ry = cy ? s.dty : s.ry - len;
  s.rz = cz ? s.dtz : s.rz - len;
  s.idx += cx ? s.stx : (cy ? s.sty : s.stz);
  if (BRICK) {
    s.stx = cx ? s.ttx - s.stx : s.stx;
    s.sty = cy ? s.tty - s.sty : s.sty;
    s.stz = cz ? s.ttz - s.stz : s.stz;
    s.px += cx ? s.dpx : 0.f;
    s.py += cy ? s.dpy : 0.f;
    s.pz += cz ? s.dpz : 0.f;
  }
  return len;
}

// ------------------------------------------------------------------------------------------------ forward
__global__ void __launch_bounds__(kFwdThreads, 6) siddon_fwd_kernel(FwdGeom G, const FwdView* __restrict__ views,
                                                                 const float* __restrict__ vol,
                                                                 float* __restrict__ proj) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  if (iu >= G.nu || iv >= G.nv) return;
  const SiddonRay r = siddon_setup(G, views[view], iu, iv, nullptr);
  float sum = 0.f;
  if (r.hit) {
    SiddonState s = siddon_state<false>(r, G);
    const unsigned last = (unsigned)(G.L.nx * G.L.ny * G.L.nz) - 1u;
    for (int n = r.nseg; n > 0; --n) {
      const float val = __ldg(vol + clamp_offset(s.idx, last));
      const float len = siddon_step<false>(s);
      sum = fmaf(len, val, sum);
    }
  }
  proj[((size_t)view * G.nv + iv) * G.nu + iu] = sum;
}

// ------------------------------------------------------------------------------------------------ pose gradient
// g_j comes from the per-voxel gradient volume (grad_volume_kernel, written once per call): one 16-byte read per
// segment instead of six predicated scalar gathers - the first version, which differenced the caller's volume in the
// loop, was L1TEX-bound.
__global__ void __launch_bounds__(kFwdThreads, 5) siddon_grad_kernel(FwdGeom G, const FwdView* __restrict__ views,
                                                                  const float4* __restrict__ gvol,
                                                                  const float* __restrict__ upstream,
                                                                  float* __restrict__ partials) {
  int iu, iv;
  fwd_pixel(iu, iv);
  const int view = blockIdx.z;
  const bool live = iu < G.nu && iv < G.nv;
  float out[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (live) {
    const SiddonRay r = siddon_setup(G, views[view], iu, iv, nullptr);
    float ax_ = 0.f, ay_ = 0.f, az_ = 0.f, bx = 0.f, by = 0.f, bz = 0.f;     // A_i, B_i
    if (r.hit) {
      SiddonState s = siddon_state<true>(r, G);
      const unsigned last = (unsigned)GradBricks::make(G.L.nx, G.L.ny, G.L.nz).cells() - 1u;
      for (int n = r.nseg; n > 0; --n) {
        const float4 g = ldg4(gvol + clamp_offset(s.idx, last));
        const float rx = s.px, ry = s.py, rz = s.pz;
        const float len = siddon_step<true>(s);
        const float lx = len * g.x, ly = len * g.y, lz = len * g.z;          // a^ij g_j
        ax_ += lx; ay_ += ly; az_ += lz;
        bx += ry * lz - rz * ly;
        by += rz * lx - rx * lz;
        bz += rx * ly - ry * lx;
      }
    }
    const float w = __ldg(upstream + ((size_t)view * G.nv + iv) * G.nu + iu);
    out[0] = w * ax_; out[1] = w * ay_; out[2] = w * az_;
    out[3] = w * bx; out[4] = w * by; out[5] = w * bz;
  }
  reduce6_to_partials<kFwdThreads>(out, partials, view);
}

}  // namespace dfp
