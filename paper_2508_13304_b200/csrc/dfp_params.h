// dfp_params.h - device-visible parameter blocks and the host-side (fp64) per-view setup that fills them.
//
// Step a1 of the hot path: everything that depends only on (geometry, angle,
// pose) is computed ONCE per view on the host in double precision and rounded to fp32 at the end, so that
// the kernels start from correctly rounded constants:
//   * forward paths: source and detector frame rotated into the OBJECT frame (s' = R^T (s - t), e' = R^T e),
//     expressed in "centred index" coordinates of the volume;
//   * back paths: P_eff = P [R | t] with the integer part of the principal point folded in, so that the
//     perspective divide yields pixel coordinates centred within one pixel of 0.
// PAPER.md Eq.1 :60-63 (projection matrix), Table I :27-42 (M = [R | t], r' = R^T (r - t)).
#pragma once
#include <cmath>
#include <cstdint>

#include "../../include/dfp.h"

namespace dfp {

constexpr int kPad = 4;          // zero border (voxels / pixels) around the packed copies; see DESIGN.md
constexpr int kPadDet = 4;

// ---------------------------------------------------------------- geometry shared by all views of a call
// Packed volume: one float4 QUAD cell per padded voxel position (X,Y,Z) = (ix+lx, iy+ly, iz+lz),
//   cell = (v[ix][iy], v[ix+1][iy], v[ix][iy+1], v[ix+1][iy+1]) at slice iz   (out-of-range voxels = 0),
// stored in 2x2x2-cell BRICKS of 128 bytes (one L1 line):
//   cell index = FX(X) + FY(Y) + FZ(Z),  FX = (X>>1)*8 + (X&1),  FY = (Y>>1)*8*nbx + (Y&1)*2,
//                                        FZ = (Z>>1)*8*nbx*nby + (Z&1)*4
// so that the 32 rays of a warp (a compact patch perpendicular to the ray, whatever its direction) touch
// few distinct lines per load.
struct VolLayout {
  int nx, ny, nz;
  int px, py, pz;                // padded dims (all even)
  int nbx, nby;                  // bricks per row / per slab row
  int lx, ly, lz;                // low-side pad (kPad or kPad+1, chosen so that H_a + l_a is even)
  int hx, hy, hz;                // H_a = floor((n_a - 1)/2): integer part of the centre index
  float fx, fy, fz;              // (n_a-1)/2 - H_a  in {0, 0.5}
  unsigned by, bz;               // 4*nbx - 2, 4*nbx*nby - 4: multipliers of (Y & ~1), (Z & ~1)
  unsigned c0;                   // folds (H_a + l_a) and the magic-number bias into the cell index
};

struct FwdGeom {
  VolLayout L;
  int nu, nv;
  float ivx, ivy, ivz;           // 1 / voxel pitch
  float vx, vy, vz;              // voxel pitch (mm)
  float cx, cy, cz;              // volume centre (mm, object frame)
  float step;                    // D (mm)
  int kref;                      // reference sample index (samples are k = kref + kappa)
  float lo[3], hi[3];            // clip box in centred-index coordinates (value support / gradient support)
  float sgx, sgy, sgz;           // 1/(2 v_a): central-difference scale
};

// One view of the forward paths (object frame, mm).  Ray of pixel (iu,iv): from `src` towards
// src + d0 + iu*du + iv*dv.  pc(r') = (r' - c)/v + frac  are the centred-index coordinates.
struct FwdView {
  double src[3];                 // s' (mm) - fp64: the per-ray set-up runs in double (once per ray)
  double d0[3], du[3], dv[3];    // pixel (0,0) centre minus source; one-pixel steps along u and v (mm)
};

// Final contraction of the forward gradient (a5):  dL/dt = -R S_A,  dL/dgamma_k = -w_k . S_B.
struct FwdContract {
  double R[9];
  double w[9];                   // rows: w_x, w_y, w_z (axial vectors of R^T dR/dgamma_k)
};

struct BpGeom {
  int nx, ny, nz;
  int nu, nv;
  int pu, pv;                    // padded packed-projection dims
  int CU, CV;                    // integer principal-point offsets folded out of P_eff
  float hx, hy, hz;              // (n_a - 1)/2
  float vx, vy, vz, cx, cy, cz;
  float sad2;                    // SAD^2 (FDK weight numerator)
  int bp_weight, flags;
};

// One view of the back paths.  (u - CU) = A[0].(xf,yf,zf,1)/w', (v - CV) likewise, w' = A[2].(...),
// with (xf,yf,zf) = voxel index minus (n-1)/2.  J rows are P_eff[0:3] in OBJECT-frame mm (for Eq.13).
struct BpView {
  float A[3][4];
  float J[3][3];                 // P_eff rows (centred), spatial part, per mm in the object frame
};

// Final contraction of the back-projection gradient (a8): dL/dt = R S'_q, dL/dgamma_k = (R^T a_k) . S'_c.
struct BpContract {
  double R[9];
  double a[9];                   // rows: R^T a_x, R^T a_y, R^T a_z
};

// ---------------------------------------------------------------- small fp64 helpers (host only)
struct Mat3 { double m[3][3]; };

inline Mat3 mat_mul(const Mat3& a, const Mat3& b) {
  Mat3 c;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) c.m[i][j] = a.m[i][0] * b.m[0][j] + a.m[i][1] * b.m[1][j] + a.m[i][2] * b.m[2][j];
  return c;
}
inline Mat3 rot_x(double a) { return {{{1, 0, 0}, {0, std::cos(a), -std::sin(a)}, {0, std::sin(a), std::cos(a)}}}; }
inline Mat3 rot_y(double a) { return {{{std::cos(a), 0, std::sin(a)}, {0, 1, 0}, {-std::sin(a), 0, std::cos(a)}}}; }
inline Mat3 rot_z(double a) { return {{{std::cos(a), -std::sin(a), 0}, {std::sin(a), std::cos(a), 0}, {0, 0, 1}}}; }
// R = Rz(gz) Ry(gy) Rx(gx)  (U3)
inline Mat3 pose_rotation(const float* pose) { return mat_mul(rot_z(pose[5]), mat_mul(rot_y(pose[4]), rot_x(pose[3]))); }
inline void mulT(const Mat3& R, const double* v, double* out) {   // out = R^T v
  for (int j = 0; j < 3; ++j) out[j] = R.m[0][j] * v[0] + R.m[1][j] * v[1] + R.m[2][j] * v[2];
}

inline float step_of(const dfp_geometry& g) {
  return g.step_mm > 0.f ? g.step_mm : std::fmin(g.vx, std::fmin(g.vy, g.vz));
}

inline VolLayout make_layout(const dfp_geometry& g) {
  VolLayout L;
  L.nx = g.nx; L.ny = g.ny; L.nz = g.nz;
  L.hx = (g.nx - 1) / 2; L.hy = (g.ny - 1) / 2; L.hz = (g.nz - 1) / 2;
  L.lx = kPad + ((L.hx + kPad) & 1); L.ly = kPad + ((L.hy + kPad) & 1); L.lz = kPad + ((L.hz + kPad) & 1);
  L.px = (g.nx + L.lx + kPad + 1) & ~1;
  L.py = (g.ny + L.ly + kPad + 1) & ~1;
  L.pz = (g.nz + L.lz + kPad + 1) & ~1;
  L.nbx = L.px / 2; L.nby = L.py / 2;
  L.by = 4u * (unsigned)L.nbx - 2u;
  L.bz = 4u * (unsigned)L.nbx * (unsigned)L.nby - 4u;
  // index = sum_a [ w_a*T_a + b_a*(T_a & ~1) ] + c0 with T_a = float bits of the magic-rounded coordinate
  // = kMagicBits + i_a (i_a = centred index), X = i_a + H_a + l_a (even offset keeps the parity of T_a).
  {
    const unsigned mb = 0x4B400000u;
    const unsigned ox = (unsigned)(L.hx + L.lx) - mb, oy = (unsigned)(L.hy + L.ly) - mb, oz = (unsigned)(L.hz + L.lz) - mb;
    L.c0 = ox * 4u + oy * (2u + L.by) + oz * (4u + L.bz);
  }
  L.fx = (float)((g.nx - 1) * 0.5 - L.hx); L.fy = (float)((g.ny - 1) * 0.5 - L.hy);
  L.fz = (float)((g.nz - 1) * 0.5 - L.hz);
  return L;
}

// grad = false: support of f~ is (-1, n) per axis; grad = true: support of the central difference is (-2, n+1).
inline FwdGeom make_fwd_geom(const dfp_geometry& g, bool grad, bool interp = false) {
  FwdGeom G;
  G.L = make_layout(g);
  G.nu = g.nu; G.nv = g.nv;
  G.vx = g.vx; G.vy = g.vy; G.vz = g.vz;
  G.ivx = (float)(1.0 / g.vx); G.ivy = (float)(1.0 / g.vy); G.ivz = (float)(1.0 / g.vz);
  G.cx = g.cx; G.cy = g.cy; G.cz = g.cz;
  G.step = step_of(g);
  G.kref = (int)std::lround((double)g.sad / (double)G.step);
  const double margin = (grad ? 2.0 : 1.0) + 0.0625;      // superset of the support; inside the kPad border
  const int n[3] = {g.nx, g.ny, g.nz};
  const int H[3] = {G.L.hx, G.L.hy, G.L.hz};
  for (int a = 0; a < 3; ++a) {                           // centred index = index - H_a
    G.lo[a] = (float)(-margin - H[a]);
    G.hi[a] = (float)(n[a] - 1 + margin - H[a]);
  }
  // central differences over 2 voxels (O3), or the exact derivative of the interpolant per voxel (GRAD_INTERP)
  const double sg = interp ? 1.0 : 0.5;
  G.sgx = (float)(sg / g.vx); G.sgy = (float)(sg / g.vy); G.sgz = (float)(sg / g.vz);
  return G;
}

struct ViewFrame {      // world-frame scanner vectors of one view (O5)
  double n[3], s[3], dc[3], eu[3], ev[3], cu, cv;
};
inline ViewFrame make_frame(const dfp_geometry& g, double beta) {
  ViewFrame f;
  f.n[0] = std::cos(beta); f.n[1] = std::sin(beta); f.n[2] = 0;
  f.eu[0] = -std::sin(beta); f.eu[1] = std::cos(beta); f.eu[2] = 0;
  f.ev[0] = 0; f.ev[1] = 0; f.ev[2] = 1;
  for (int a = 0; a < 3; ++a) { f.s[a] = (double)g.sad * f.n[a]; f.dc[a] = -((double)g.sdd - (double)g.sad) * f.n[a]; }
  f.cu = (g.nu - 1) * 0.5 + (double)g.u0;
  f.cv = (g.nv - 1) * 0.5 + (double)g.v0;
  return f;
}

inline void make_fwd_view(const dfp_geometry& g, float angle, const float* pose, FwdView* V, FwdContract* C) {
  const ViewFrame f = make_frame(g, angle);
  const Mat3 R = pose_rotation(pose);
  const double t[3] = {pose[0], pose[1], pose[2]};
  double sw[3], p00[3], tmp[3];
  for (int a = 0; a < 3; ++a) {
    sw[a] = f.s[a] - t[a];
    p00[a] = f.dc[a] - f.cu * (double)g.du * f.eu[a] - f.cv * (double)g.dv * f.ev[a] - f.s[a];   // pixel(0,0) - s
  }
  mulT(R, sw, V->src);
  mulT(R, p00, V->d0);
  for (int a = 0; a < 3; ++a) tmp[a] = (double)g.du * f.eu[a];
  mulT(R, tmp, V->du);
  for (int a = 0; a < 3; ++a) tmp[a] = (double)g.dv * f.ev[a];
  mulT(R, tmp, V->dv);
  if (C) {
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) C->R[i * 3 + j] = R.m[i][j];
    // axial vectors of R^T dR/dgamma_k for R = Rz Ry Rx:  w_x = e_x, w_y = Rx^T e_y, w_z = (Ry Rx)^T e_z
    const Mat3 Rx = rot_x(pose[3]), RyRx = mat_mul(rot_y(pose[4]), Rx);
    const double ex[3] = {1, 0, 0}, ey[3] = {0, 1, 0}, ez[3] = {0, 0, 1};
    C->w[0] = ex[0]; C->w[1] = ex[1]; C->w[2] = ex[2];
    mulT(Rx, ey, C->w + 3);
    mulT(RyRx, ez, C->w + 6);
  }
}

inline BpGeom make_bp_geom(const dfp_geometry& g) {
  BpGeom G;
  G.nx = g.nx; G.ny = g.ny; G.nz = g.nz; G.nu = g.nu; G.nv = g.nv;
  G.pu = g.nu + 2 * kPadDet; G.pv = g.nv + 2 * kPadDet;
  const ViewFrame f = make_frame(g, 0.0);
  G.CU = (int)std::floor(f.cu); G.CV = (int)std::floor(f.cv);
  G.hx = (g.nx - 1) * 0.5f; G.hy = (g.ny - 1) * 0.5f; G.hz = (g.nz - 1) * 0.5f;
  G.vx = g.vx; G.vy = g.vy; G.vz = g.vz; G.cx = g.cx; G.cy = g.cy; G.cz = g.cz;
  G.sad2 = (float)((double)g.sad * (double)g.sad);
  G.bp_weight = g.bp_weight; G.flags = g.flags;
  return G;
}

inline void make_bp_view(const dfp_geometry& g, const BpGeom& G, float angle, const float* pose, BpView* V,
                         BpContract* C) {
  const ViewFrame f = make_frame(g, angle);
  const Mat3 R = pose_rotation(pose);
  const double t[3] = {pose[0], pose[1], pose[2]};
  // world projection matrix in pixel-index units (Eq.1), principal point's integer part removed:
  //   P3 = (-n | SAD),  P1 = (SDD/du)(e_u | 0) + (c_u - CU) P3,  P2 = (SDD/dv)(e_v | 0) + (c_v - CV) P3
  double P[3][4];
  for (int a = 0; a < 3; ++a) P[2][a] = -f.n[a];
  P[2][3] = g.sad;
  for (int a = 0; a < 4; ++a) {
    const double e1 = a < 3 ? f.eu[a] : 0.0, e2 = a < 3 ? f.ev[a] : 0.0;
    P[0][a] = ((double)g.sdd / (double)g.du) * e1 + (f.cu - G.CU) * P[2][a];
    P[1][a] = ((double)g.sdd / (double)g.dv) * e2 + (f.cv - G.CV) * P[2][a];
  }
  // P_eff = P [R | t; 0 0 0 1]  acting on object-frame mm
  double E[3][4];
  for (int r = 0; r < 3; ++r) {
    for (int c = 0; c < 3; ++c) E[r][c] = P[r][0] * R.m[0][c] + P[r][1] * R.m[1][c] + P[r][2] * R.m[2][c];
    E[r][3] = P[r][0] * t[0] + P[r][1] * t[1] + P[r][2] * t[2] + P[r][3];
  }
  // fold the -1/2 of the magic-number floor into the u and v rows: (E0 - E2/2).x / w' = u - CU - 1/2.
  // Eq.13's J_u = (P1 - u P3)/w' is unchanged by this shift as long as u is taken in the same units.
  for (int c = 0; c < 4; ++c) { E[0][c] -= 0.5 * E[2][c]; E[1][c] -= 0.5 * E[2][c]; }
  // acting on centred voxel indices: r' = c + (idx - h) * v
  for (int r = 0; r < 3; ++r) {
    V->A[r][0] = (float)(E[r][0] * (double)g.vx);
    V->A[r][1] = (float)(E[r][1] * (double)g.vy);
    V->A[r][2] = (float)(E[r][2] * (double)g.vz);
    V->A[r][3] = (float)(E[r][0] * (double)g.cx + E[r][1] * (double)g.cy + E[r][2] * (double)g.cz + E[r][3]);
    for (int c = 0; c < 3; ++c) V->J[r][c] = (float)E[r][c];
  }
  if (C) {
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) C->R[i * 3 + j] = R.m[i][j];
    // axial vectors of dR/dgamma_k R^T: a_x = R e_x, a_y = Rz e_y, a_z = e_z; stored as R^T a_k
    const Mat3 Rz = rot_z(pose[5]);
    const double ax[3] = {R.m[0][0], R.m[1][0], R.m[2][0]};
    const double ay[3] = {Rz.m[0][1], Rz.m[1][1], Rz.m[2][1]};
    const double az[3] = {0, 0, 1};
    mulT(R, ax, C->a);
    mulT(R, ay, C->a + 3);
    mulT(R, az, C->a + 6);
  }
}

}  // namespace dfp
