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

// The same rows in DOUBLE, for the TMA kernels' producer warp: per (voxel tile, view) it re-bases the rows onto the
// tile's first voxel and the staged patch's first pixel (fp64) and only then rounds to fp32, so that the consumers'
// fp32 (u, v) are patch-local numbers (< 100 pixels) with ~3e-6 pixel of error whatever the detector size.
struct BpViewD {
  double A[3][4];
  double J[3][3];
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

// World-frame scanner of one view.  Pixel (iu,iv) centre = dc + (iu - cu) U + (iv - cv) V; Eq.1 (PAPER.md :60-63)
// in pixel-index units is  u w' = pu.(r;1) + cu w',  v w' = pv.(r;1) + cv w',  w' = p3.(r;1) = depth from the source
// along the detector normal in mm.
struct ViewFrame {
  double s[3], dc[3], U[3], V[3], cu, cv;
  double pu[4], pv[4], p3[4];
  double sdd, ulen, vlen, udotv; // perpendicular source-detector distance; |U|, |V| (mm); U.V
  bool ok;                       // false: degenerate frame (U parallel to V, or the source in the detector plane)
};
inline int view_stride(const dfp_geometry& g) { return (g.flags & DFP_FLAG_VIEW_FRAMES) ? 12 : 1; }

// Circular orbit (O5): views[v] = gantry angle.
inline ViewFrame make_frame_circular(const dfp_geometry& g, double beta) {
  ViewFrame f;
  const double n[3] = {std::cos(beta), std::sin(beta), 0}, eu[3] = {-std::sin(beta), std::cos(beta), 0}, ev[3] = {0, 0, 1};
  for (int a = 0; a < 3; ++a) {
    f.s[a] = (double)g.sad * n[a]; f.dc[a] = -((double)g.sdd - (double)g.sad) * n[a];
    f.U[a] = (double)g.du * eu[a]; f.V[a] = (double)g.dv * ev[a];
    f.p3[a] = -n[a];
    f.pu[a] = ((double)g.sdd / (double)g.du) * eu[a];
    f.pv[a] = ((double)g.sdd / (double)g.dv) * ev[a];
  }
  f.p3[3] = g.sad; f.pu[3] = 0; f.pv[3] = 0;
  f.sdd = g.sdd; f.ulen = g.du; f.vlen = g.dv; f.udotv = 0;
  f.cu = (g.nu - 1) * 0.5 + (double)g.u0;
  f.cv = (g.nv - 1) * 0.5 + (double)g.v0;
  f.ok = true;
  return f;
}

// Explicit frame (DFP_FLAG_VIEW_FRAMES): views[12 v ..] = s, dc, U, V.  With q = r - s written in the basis
// (U, V, D = dc - s), q = a U + b V + k D, the point s + q / k of the line lies on the detector at dc + (a/k) U + (b/k) V:
// (a, b, k) = B^-1 q with B = [U V D] (columns), so the rows of B^-1, scaled by SDD_v = |det B| / |U x V| to make
// w' a depth in mm, are the spatial parts of pu, pv, p3.
inline ViewFrame make_frame_explicit(const dfp_geometry& g, const float* fr) {
  ViewFrame f;
  double D[3];
  for (int a = 0; a < 3; ++a) { f.s[a] = fr[a]; f.dc[a] = fr[3 + a]; f.U[a] = fr[6 + a]; f.V[a] = fr[9 + a]; D[a] = f.dc[a] - f.s[a]; }
  auto cross = [](const double* x, const double* y, double* o) {
    o[0] = x[1] * y[2] - x[2] * y[1]; o[1] = x[2] * y[0] - x[0] * y[2]; o[2] = x[0] * y[1] - x[1] * y[0];
  };
  double VxD[3], DxU[3], UxV[3];
  cross(f.V, D, VxD); cross(D, f.U, DxU); cross(f.U, f.V, UxV);
  const double det = f.U[0] * VxD[0] + f.U[1] * VxD[1] + f.U[2] * VxD[2];
  const double area = std::sqrt(UxV[0] * UxV[0] + UxV[1] * UxV[1] + UxV[2] * UxV[2]);
  f.ulen = std::sqrt(f.U[0] * f.U[0] + f.U[1] * f.U[1] + f.U[2] * f.U[2]);
  f.vlen = std::sqrt(f.V[0] * f.V[0] + f.V[1] * f.V[1] + f.V[2] * f.V[2]);
  f.udotv = f.U[0] * f.V[0] + f.U[1] * f.V[1] + f.U[2] * f.V[2];
  f.cu = (g.nu - 1) * 0.5 + (double)g.u0;
  f.cv = (g.nv - 1) * 0.5 + (double)g.v0;
  f.ok = std::isfinite(det) && std::isfinite(area) && area > 1e-12 * f.ulen * f.vlen && f.ulen > 0 && f.vlen > 0 &&
         std::fabs(det) > 1e-6 * area * std::sqrt(D[0] * D[0] + D[1] * D[1] + D[2] * D[2]);
  if (!f.ok) { f.sdd = 0; return f; }
  f.sdd = std::fabs(det) / area;
  const double k = f.sdd / det;                        // rows of B^-1 are (V x D, D x U, U x V) / det
  f.pu[3] = f.pv[3] = f.p3[3] = 0;
  for (int a = 0; a < 3; ++a) {
    f.pu[a] = k * VxD[a]; f.pv[a] = k * DxU[a]; f.p3[a] = k * UxV[a];
    f.pu[3] -= f.pu[a] * f.s[a]; f.pv[3] -= f.pv[a] * f.s[a]; f.p3[3] -= f.p3[a] * f.s[a];
  }
  return f;
}
inline ViewFrame make_frame(const dfp_geometry& g, const float* views, int v) {
  return (g.flags & DFP_FLAG_VIEW_FRAMES) ? make_frame_explicit(g, views + 12 * (size_t)v)
                                          : make_frame_circular(g, (double)views[v]);
}

inline void make_fwd_view(const ViewFrame& f, const float* pose, FwdView* V, FwdContract* C) {
  const Mat3 R = pose_rotation(pose);
  const double t[3] = {pose[0], pose[1], pose[2]};
  double sw[3], p00[3];
  for (int a = 0; a < 3; ++a) {
    sw[a] = f.s[a] - t[a];
    p00[a] = f.dc[a] - f.cu * f.U[a] - f.cv * f.V[a] - f.s[a];   // pixel(0,0) - s
  }
  mulT(R, sw, V->src);
  mulT(R, p00, V->d0);
  mulT(R, f.U, V->du);
  mulT(R, f.V, V->dv);
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

// One view of the distance-driven kernels (dfp_dd.cuh), object frame, mm, fp64: source, detector point of pixel index
// (0, 0), displacement of one pixel step along u and v; P maps an object-frame point to pixel indices,
// (u', v', w') = P (r'; 1), u = u'/w' (Eq.1 with the pose folded in; used to find the pixels a voxel cell can meet);
// a = driving axis of the view, ub / vb = the in-plane axes paired with the detector's u / v.
struct DdView {
  double so[3], X00[3], Uo[3], Vo[3];
  double P[3][4];
  int a, ub, vb, pad;
};
inline void make_dd_view(const dfp_geometry& g, const ViewFrame& f, const float* pose, DdView* D) {
  const Mat3 R = pose_rotation(pose);
  const double t[3] = {pose[0], pose[1], pose[2]};
  double sw[3], x00[3];
  for (int a = 0; a < 3; ++a) {
    sw[a] = f.s[a] - t[a];
    x00[a] = f.dc[a] - f.cu * f.U[a] - f.cv * f.V[a] - t[a];
  }
  mulT(R, sw, D->so);
  mulT(R, x00, D->X00);
  mulT(R, f.U, D->Uo);
  mulT(R, f.V, D->Vo);
  double n[3];
  for (int a = 0; a < 3; ++a)
    n[a] = D->X00[a] + 0.5 * (g.nu - 1) * D->Uo[a] + 0.5 * (g.nv - 1) * D->Vo[a] - D->so[a];
  int a = 0;
  for (int k = 1; k < 3; ++k) if (std::fabs(n[k]) > std::fabs(n[a])) a = k;
  const int b = (a + 1) % 3, d = (a + 2) % 3;
  const bool u_is_b = std::fabs(D->Uo[b]) >= std::fabs(D->Uo[d]);
  D->a = a; D->ub = u_is_b ? b : d; D->vb = u_is_b ? d : b; D->pad = 0;
  double P[3][4];
  for (int c = 0; c < 4; ++c) {
    P[2][c] = f.p3[c];
    P[0][c] = f.pu[c] + f.cu * f.p3[c];
    P[1][c] = f.pv[c] + f.cv * f.p3[c];
  }
  for (int r = 0; r < 3; ++r) {
    for (int c = 0; c < 3; ++c) D->P[r][c] = P[r][0] * R.m[0][c] + P[r][1] * R.m[1][c] + P[r][2] * R.m[2][c];
    D->P[r][3] = P[r][0] * t[0] + P[r][1] * t[1] + P[r][2] * t[2] + P[r][3];
  }
}

inline BpGeom make_bp_geom(const dfp_geometry& g) {
  BpGeom G;
  G.nx = g.nx; G.ny = g.ny; G.nz = g.nz; G.nu = g.nu; G.nv = g.nv;
  G.pu = g.nu + 2 * kPadDet; G.pv = g.nv + 2 * kPadDet;
  G.CU = (int)std::floor((g.nu - 1) * 0.5 + (double)g.u0); G.CV = (int)std::floor((g.nv - 1) * 0.5 + (double)g.v0);
  G.hx = (g.nx - 1) * 0.5f; G.hy = (g.ny - 1) * 0.5f; G.hz = (g.nz - 1) * 0.5f;
  G.vx = g.vx; G.vy = g.vy; G.vz = g.vz; G.cx = g.cx; G.cy = g.cy; G.cz = g.cz;
  G.sad2 = (float)((double)g.sad * (double)g.sad);
  G.bp_weight = g.bp_weight; G.flags = g.flags;
  return G;
}

inline void make_bp_view(const dfp_geometry& g, const BpGeom& G, const ViewFrame& f, const float* pose, BpView* V,
                         BpContract* C, BpViewD* VD = nullptr) {
  const Mat3 R = pose_rotation(pose);
  const double t[3] = {pose[0], pose[1], pose[2]};
  // world projection matrix in pixel-index units (Eq.1), principal point's integer part removed:
  //   circular orbit: P3 = (-n | SAD),  P1 = (SDD/du)(e_u | 0) + (c_u - CU) P3,  P2 = (SDD/dv)(e_v | 0) + (c_v - CV) P3
  double P[3][4];
  for (int a = 0; a < 4; ++a) {
    P[2][a] = f.p3[a];
    P[0][a] = f.pu[a] + (f.cu - G.CU) * P[2][a];
    P[1][a] = f.pv[a] + (f.cv - G.CV) * P[2][a];
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
    if (VD) {
      VD->A[r][0] = E[r][0] * (double)g.vx; VD->A[r][1] = E[r][1] * (double)g.vy; VD->A[r][2] = E[r][2] * (double)g.vz;
      VD->A[r][3] = E[r][0] * (double)g.cx + E[r][1] * (double)g.cy + E[r][2] * (double)g.cz + E[r][3];
      for (int c = 0; c < 3; ++c) VD->J[r][c] = E[r][c];
    }
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
