// dfp_oracle.cpp - TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, fp64 CPU statement of what the dfp hot path computes, written from
// /root/reference/PAPER.md (arXiv 2508.13304) and the readings in SURVEY.md §8(c) / DESIGN.md.
// It shares no code, header, table or helper with the CUDA path (paper_2508_13304_b200/csrc) and
// neither imports the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// `--impl reference` leg may load it.  OpenMP is used only to spread independent rays / voxels
// over cores; there is no blocking, fusion or reordering inside a ray or a voxel.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): closed-form ellipsoid and Gaussian line
// integrals, explicit-transpose adjointness, central finite differences in all six pose
// parameters, the translation invariant dL/dt = -R A[grad mu], 6-accumulator vs the paper's
// 12-element G route, stored-G literal algorithm on BOTH sides (forward: 12 stored G_f volumes projected;
// back: stored central-difference images back-projected, Eq.13, G_b contracted - at general
// non-integer (u,v)), brute-force back-projection on tiny grids;
// Siddon weights (O12, tests/test_oracle_siddon.py): chord of the grid box, brute-force clipping
// of the ray against every voxel's own box, explicit transpose, closed forms, the paper's literal
// stored-G algorithm, finite differences of closed-form projections; Joseph weights (O13,
// tests/test_oracle_joseph.py): hand formulas for constant and in-plane-linear volumes, explicit
// transpose, closed forms with second-order convergence on all three driving axes, stored-G,
// finite differences of closed-form projections; explicit view frames (O14,
// tests/test_oracle_view_frames.py): Eq.1 on the source -> pixel lines of tilted / skewed / shifted
// detectors, closed-form blobs under a general frame, the frame of a circular view against the
// circular path, scanner and object moved together, finite differences of the discrete projector /
// back-projector under a general frame.
// Distance-driven pair (O15, tests/test_oracle_dd.py) and separable-footprint pair (O16, tests/test_oracle_sf.py):
// textbook weights on the standard views, footprint mass vs the brute-force integral of exact chords, exact
// transposes, closed forms with convergence, stored-G on both sides, finite differences.
// No function here is "parity unpinned".
//
// Conventions:
//   vol[iz][iy][ix], x fastest; proj[view][iv][iu], u fastest; pose = (tx,ty,tz,gx,gy,gz) mm / rad.
//   O1  voxel centre r'_j = c + ((ix-(nx-1)/2)vx, (iy-(ny-1)/2)vy, (iz-(nz-1)/2)vz)
//   O2  f~ = trilinear interpolant between voxel centres, out-of-range voxels read as 0
//   O4  R = Rz(gz) Ry(gy) Rx(gx);  r = R r' + t;  r' = R^T (r - t)         (Table I :29-36)
//   O5  view angle b: n=(cos b, sin b,0); source s = SAD n; detector centre -(SDD-SAD) n;
//       e_u=(-sin b, cos b, 0); e_v=(0,0,1); P in pixel-index units         (Eq.1 :60-63)
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
struct ora_geom {
  int32_t nx, ny, nz;
  double vx, vy, vz;
  double cx, cy, cz;
  int32_t nu, nv;
  double du, dv, u0, v0;
  double sad, sdd;
  double step_mm;
  int32_t bp_weight;
  int32_t flags;
};
}

namespace {

struct V3 { double x, y, z; };
inline V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double comp(V3 a, int k) { return k == 0 ? a.x : (k == 1 ? a.y : a.z); }

struct M3 { double m[3][3]; };
inline M3 mul(const M3& a, const M3& b) {
  M3 c;
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    double s = 0; for (int k = 0; k < 3; ++k) s += a.m[i][k] * b.m[k][j]; c.m[i][j] = s; }
  return c;
}
inline V3 mul(const M3& a, V3 v) {
  return {a.m[0][0] * v.x + a.m[0][1] * v.y + a.m[0][2] * v.z,
          a.m[1][0] * v.x + a.m[1][1] * v.y + a.m[1][2] * v.z,
          a.m[2][0] * v.x + a.m[2][1] * v.y + a.m[2][2] * v.z};
}
inline V3 mulT(const M3& a, V3 v) {   // a^T v
  return {a.m[0][0] * v.x + a.m[1][0] * v.y + a.m[2][0] * v.z,
          a.m[0][1] * v.x + a.m[1][1] * v.y + a.m[2][1] * v.z,
          a.m[0][2] * v.x + a.m[1][2] * v.y + a.m[2][2] * v.z};
}
inline M3 Rx(double a) { double c = cos(a), s = sin(a); return {{{1, 0, 0}, {0, c, -s}, {0, s, c}}}; }
inline M3 Ry(double a) { double c = cos(a), s = sin(a); return {{{c, 0, s}, {0, 1, 0}, {-s, 0, c}}}; }
inline M3 Rz(double a) { double c = cos(a), s = sin(a); return {{{c, -s, 0}, {s, c, 0}, {0, 0, 1}}}; }
inline M3 dRx(double a) { double c = cos(a), s = sin(a); return {{{0, 0, 0}, {0, -s, -c}, {0, c, -s}}}; }
inline M3 dRy(double a) { double c = cos(a), s = sin(a); return {{{-s, 0, c}, {0, 0, 0}, {-c, 0, -s}}}; }
inline M3 dRz(double a) { double c = cos(a), s = sin(a); return {{{-s, -c, 0}, {c, -s, 0}, {0, 0, 0}}}; }

// O4 + U4: pose -> R, t and dR/dgamma_k (PAPER.md :79 "has an explicit expression").
struct Pose {
  M3 R; V3 t; M3 dR[3];
  explicit Pose(const double* th) {
    t = {th[0], th[1], th[2]};
    M3 rx = Rx(th[3]), ry = Ry(th[4]), rz = Rz(th[5]);
    R = mul(rz, mul(ry, rx));
    dR[0] = mul(rz, mul(ry, dRx(th[3])));
    dR[1] = mul(rz, mul(dRy(th[4]), rx));
    dR[2] = mul(dRz(th[5]), mul(ry, rx));
  }
};

// O5: one view of the scanner.  Default: circular cone-beam orbit, gantry angle `views[v]`.
// O14 (flags & 64, "view frames"; SURVEY.md 8b optional extension, PAPER.md :244 non-circular orbit): `views` holds
// 12 numbers per view, world frame, mm: source s, detector reference point c (where the pixel index is (c_u, c_v)),
// and the displacements U, V of one pixel step along u and along v (any flat detector; U, V need not be orthogonal).
//   pixel (iu,iv) centre = c + (iu - c_u) U + (iv - c_v) V                                       (definition)
//   P (Eq.1 :60-63, pixel-index units) follows from intersecting the line s -> r with the detector plane:
//   nh = unit normal of the plane on the far side of the source, w' = (r - s).nh (depth in mm, as in the circular
//   case), SDD_v = (c - s).nh, and with the dual vectors U* = (V x nh)/(U.(V x nh)), V* = (nh x U)/(V.(nh x U))
//   (U*.U = 1, U*.V = 0):  u = c_u + (x - c).U*  at  x = s + (SDD_v / w')(r - s), i.e.
//   P_3 = (nh | -nh.s),  P_1 = SDD_v (U* | -U*.s) + (c_u - (c - s).U*) P_3,  P_2 likewise with V*, c_v.
struct View {
  V3 s, dc, U, Vs; double P[3][4]; double cu, cv;
  View(const ora_geom& g, const double* views, int v) {
    cu = (g.nu - 1) / 2.0 + g.u0;
    cv = (g.nv - 1) / 2.0 + g.v0;
    if (g.flags & 64) {
      const double* f = views + 12 * (size_t)v;
      s = {f[0], f[1], f[2]}; dc = {f[3], f[4], f[5]}; U = {f[6], f[7], f[8]}; Vs = {f[9], f[10], f[11]};
      V3 nh = cross(U, Vs);
      nh = (1.0 / sqrt(dot(nh, nh))) * nh;
      if (dot(dc - s, nh) < 0) nh = -1.0 * nh;
      const double sddv = dot(dc - s, nh);
      V3 Ud = cross(Vs, nh); Ud = (1.0 / dot(U, Ud)) * Ud;
      V3 Vd = cross(nh, U); Vd = (1.0 / dot(Vs, Vd)) * Vd;
      double P3[4] = {nh.x, nh.y, nh.z, -dot(nh, s)};
      double e1[4] = {Ud.x, Ud.y, Ud.z, -dot(Ud, s)}, e2[4] = {Vd.x, Vd.y, Vd.z, -dot(Vd, s)};
      const double ou = cu - dot(dc - s, Ud), ov = cv - dot(dc - s, Vd);
      for (int k = 0; k < 4; ++k) {
        P[2][k] = P3[k];
        P[0][k] = sddv * e1[k] + ou * P3[k];
        P[1][k] = sddv * e2[k] + ov * P3[k];
      }
      return;
    }
    const double beta = views[v];
    V3 n = {cos(beta), sin(beta), 0.0};
    s = g.sad * n;
    dc = -(g.sdd - g.sad) * n;
    V3 eu = {-sin(beta), cos(beta), 0.0}, ev = {0.0, 0.0, 1.0};
    U = g.du * eu;
    Vs = g.dv * ev;
    double P3[4] = {-n.x, -n.y, -n.z, g.sad};
    double e1[4] = {eu.x, eu.y, eu.z, 0.0}, e2[4] = {ev.x, ev.y, ev.z, 0.0};
    for (int k = 0; k < 4; ++k) {
      P[2][k] = P3[k];
      P[0][k] = (g.sdd / g.du) * e1[k] + cu * P3[k];
      P[1][k] = (g.sdd / g.dv) * e2[k] + cv * P3[k];
    }
  }
  V3 pixel(const ora_geom& g, int iu, int iv) const {
    (void)g;
    return dc + (iu - cu) * U + (iv - cv) * Vs;
  }
};

inline double step_of(const ora_geom& g) {
  return g.step_mm > 0 ? g.step_mm : std::min(g.vx, std::min(g.vy, g.vz));
}

// O1: object-frame mm -> continuous voxel index.
inline V3 to_index(const ora_geom& g, V3 rp) {
  return {(rp.x - g.cx) / g.vx + (g.nx - 1) / 2.0, (rp.y - g.cy) / g.vy + (g.ny - 1) / 2.0,
          (rp.z - g.cz) / g.vz + (g.nz - 1) / 2.0};
}
inline V3 voxel_centre(const ora_geom& g, int ix, int iy, int iz) {
  return {g.cx + (ix - (g.nx - 1) / 2.0) * g.vx, g.cy + (iy - (g.ny - 1) / 2.0) * g.vy,
          g.cz + (iz - (g.nz - 1) / 2.0) * g.vz};
}

template <typename T>
struct Vol {
  const T* v; int nx, ny, nz;
  double at(long ix, long iy, long iz) const {
    if (ix < 0 || iy < 0 || iz < 0 || ix >= nx || iy >= ny || iz >= nz) return 0.0;
    return (double)v[((size_t)iz * ny + iy) * nx + ix];
  }
};

// O2: zero-extended trilinear interpolant at continuous index p.
template <typename T>
inline double trilin(const Vol<T>& V, V3 p) {
  double fx = floor(p.x), fy = floor(p.y), fz = floor(p.z);
  long ix = (long)fx, iy = (long)fy, iz = (long)fz;
  double ax = p.x - fx, ay = p.y - fy, az = p.z - fz;
  double s = 0.0;
  for (int dz = 0; dz < 2; ++dz) for (int dy = 0; dy < 2; ++dy) for (int dx = 0; dx < 2; ++dx) {
    double w = (dx ? ax : 1 - ax) * (dy ? ay : 1 - ay) * (dz ? az : 1 - az);
    s += w * V.at(ix + dx, iy + dy, iz + dz);
  }
  return s;
}

// O3: volume gradient at a sample (per mm).
//  mode 0 CENTRAL (the paper's "central finite difference", PAPER.md :183):
//         g_a = [f~(r' + v_a e_a) - f~(r' - v_a e_a)] / (2 v_a)
//  mode 1 INTERP: exact derivative of the trilinear interpolant (test aid).
template <typename T>
inline V3 vol_grad(const Vol<T>& V, const ora_geom& g, V3 p, int mode) {
  if (mode == 0) {
    V3 ex = {1, 0, 0}, ey = {0, 1, 0}, ez = {0, 0, 1};
    return {(trilin(V, p + ex) - trilin(V, p - ex)) / (2 * g.vx),
            (trilin(V, p + ey) - trilin(V, p - ey)) / (2 * g.vy),
            (trilin(V, p + ez) - trilin(V, p - ez)) / (2 * g.vz)};
  }
  double fx = floor(p.x), fy = floor(p.y), fz = floor(p.z);
  long ix = (long)fx, iy = (long)fy, iz = (long)fz;
  double a[3] = {p.x - fx, p.y - fy, p.z - fz};
  double gx = 0, gy = 0, gz = 0;
  for (int dz = 0; dz < 2; ++dz) for (int dy = 0; dy < 2; ++dy) for (int dx = 0; dx < 2; ++dx) {
    double val = V.at(ix + dx, iy + dy, iz + dz);
    double wx = dx ? a[0] : 1 - a[0], wy = dy ? a[1] : 1 - a[1], wz = dz ? a[2] : 1 - a[2];
    gx += (dx ? 1.0 : -1.0) * wy * wz * val;
    gy += wx * (dy ? 1.0 : -1.0) * wz * val;
    gz += wx * wy * (dz ? 1.0 : -1.0) * val;
  }
  return {gx / g.vx, gy / g.vy, gz / g.vz};
}

// Sample index range [k0,k1] that is a SUPERSET of the samples whose object-frame position can
// fall inside the volume padded by `pad` voxels (O6: "clipping the range never changes the value").
inline bool k_range(const ora_geom& g, V3 ps, V3 pe_per_mm, double step, double pad, long& k0, long& k1) {
  double lo = -1e300, hi = 1e300;
  double n[3] = {(double)g.nx, (double)g.ny, (double)g.nz};
  for (int a = 0; a < 3; ++a) {
    double o = comp(ps, a), d = comp(pe_per_mm, a);
    double bmin = -pad, bmax = n[a] - 1 + pad;
    if (fabs(d) < 1e-300) { if (o < bmin || o > bmax) return false; continue; }
    double t0 = (bmin - o) / d, t1 = (bmax - o) / d;
    if (t0 > t1) std::swap(t0, t1);
    lo = std::max(lo, t0); hi = std::min(hi, t1);
  }
  if (hi < lo || hi < 0) return false;
  k0 = (long)floor(lo / step) - 2; if (k0 < 0) k0 = 0;
  k1 = (long)ceil(hi / step) + 2;
  return true;
}
inline bool in_padded_box(const ora_geom& g, V3 p, double pad) {
  return p.x >= -pad && p.x <= g.nx - 1 + pad && p.y >= -pad && p.y <= g.ny - 1 + pad &&
         p.z >= -pad && p.z <= g.nz - 1 + pad;
}

// ------------------------------------------------------------------------------------------------
// O6: forward projection, Eq.2a :67-69 discretised as Eq.18 :172-177 with a fixed-step
// trilinear ray-march (reading U1):  l_i = D * sum_k f~(R^T (s + tau_k e - t)),  tau_k=(k+1/2) D.
template <typename T>
void forward_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                  double* proj, int64_t* ray_steps) {
  Vol<T> V{vol, g.nx, g.ny, g.nz};
  const double D = step_of(g);
  int64_t total_steps = 0;
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    int64_t steps_v = 0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : steps_v)
    for (int iv = 0; iv < g.nv; ++iv) {
      for (int iu = 0; iu < g.nu; ++iu) {
        V3 d = view.pixel(g, iu, iv) - view.s;
        V3 e = (1.0 / sqrt(dot(d, d))) * d;
        // range of k worth visiting (object-frame line: s' + tau e')
        V3 ps = to_index(g, mulT(pose.R, view.s - pose.t));
        V3 eo = mulT(pose.R, e);
        V3 pe = {eo.x / g.vx, eo.y / g.vy, eo.z / g.vz};
        long k0, k1;
        double sum = 0.0;
        if (k_range(g, ps, pe, D, 3.0, k0, k1)) {
          for (long k = k0; k <= k1; ++k) {
            double tau = (k + 0.5) * D;
            V3 r = view.s + tau * e;                 // world sample, fixed in the world
            V3 rp = mulT(pose.R, r - pose.t);        // r' = R^T (r - t)
            V3 p = to_index(g, rp);
            sum += trilin(V, p);
            if (in_padded_box(g, p, 2.0)) ++steps_v;
          }
        }
        proj[((size_t)v * g.nv + iv) * g.nu + iu] = D * sum;
      }
    }
    total_steps += steps_v;
  }
  if (ray_steps) *ray_steps = total_steps;
}

// O10: explicit transpose of the forward projector (adjointness pin only).
template <typename T>
void forward_T_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* y,
                    double* vol_out) {
  const double D = step_of(g);
  size_t nvox = (size_t)g.nx * g.ny * g.nz;
  for (size_t i = 0; i < nvox; ++i) vol_out[i] = 0.0;
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    for (int iv = 0; iv < g.nv; ++iv) for (int iu = 0; iu < g.nu; ++iu) {
      double yi = (double)y[((size_t)v * g.nv + iv) * g.nu + iu];
      V3 d = view.pixel(g, iu, iv) - view.s;
      V3 e = (1.0 / sqrt(dot(d, d))) * d;
      V3 ps = to_index(g, mulT(pose.R, view.s - pose.t));
      V3 eo = mulT(pose.R, e);
      V3 pe = {eo.x / g.vx, eo.y / g.vy, eo.z / g.vz};
      long k0, k1;
      if (!k_range(g, ps, pe, D, 3.0, k0, k1)) continue;
      for (long k = k0; k <= k1; ++k) {
        V3 p = to_index(g, mulT(pose.R, view.s + ((k + 0.5) * D) * e - pose.t));
        double fx = floor(p.x), fy = floor(p.y), fz = floor(p.z);
        long ix = (long)fx, iy = (long)fy, iz = (long)fz;
        double ax = p.x - fx, ay = p.y - fy, az = p.z - fz;
        for (int dz = 0; dz < 2; ++dz) for (int dy = 0; dy < 2; ++dy) for (int dx = 0; dx < 2; ++dx) {
          long X = ix + dx, Y = iy + dy, Z = iz + dz;
          if (X < 0 || Y < 0 || Z < 0 || X >= g.nx || Y >= g.ny || Z >= g.nz) continue;
          double w = (dx ? ax : 1 - ax) * (dy ? ay : 1 - ay) * (dz ? az : 1 - az);
          vol_out[((size_t)Z * g.ny + Y) * g.nx + X] += D * w * yi;
        }
      }
    }
  }
}

// dL/dtheta_k = sum_ab (dM_ab/dtheta_k) (grad_M L)_ab, M = [R | t]   (PAPER.md :79, reading U4).
inline void contract_M(const Pose& pose, const double GM[3][4], double* out6) {
  for (int k = 0; k < 3; ++k) out6[k] = GM[k][3];
  for (int k = 0; k < 3; ++k) {
    double s = 0;
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) s += pose.dR[k].m[a][b] * GM[a][b];
    out6[3 + k] = s;
  }
}

// ------------------------------------------------------------------------------------------------
// O7: forward pose gradient, Eq.3-8 :81-113 and Eq.19-20 :179-191.
//  lever_arm 0 SAMPLE: G_f evaluated at the interpolated sample (reading U2, default)
//            1 VOXEL : per-voxel G_f^j (central-difference gradient and lever arm at voxel centres,
//                      "Compute matrix G_f^j for each voxel", :189) projected with the weights a^ij
//  grad_mode 0 CENTRAL | 1 INTERP (SAMPLE only)
//  route 0: six accumulators  A_i = D sum g~,  B_i = D sum r' x g~;  dL/dt = -R S_A, dL/dgamma_k = -w_k.S_B
//        1: the paper's 12-element route  G_f = [ (r-t) g~^T | -R g~ ]  (Eq.6/8), contracted with dM/dtheta
template <typename T>
void forward_grad_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                       const float* upstream, double* grad, int lever_arm, int grad_mode, int route) {
  Vol<T> V{vol, g.nx, g.ny, g.nz};
  const double D = step_of(g);
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    // per-row partial sums, added in row order afterwards (deterministic)
    std::vector<double> rowacc((size_t)g.nv * 12, 0.0);
#pragma omp parallel for schedule(dynamic, 4)
    for (int iv = 0; iv < g.nv; ++iv) {
      double acc[12] = {0};
      for (int iu = 0; iu < g.nu; ++iu) {
        double w = (double)upstream[((size_t)v * g.nv + iv) * g.nu + iu];
        V3 d = view.pixel(g, iu, iv) - view.s;
        V3 e = (1.0 / sqrt(dot(d, d))) * d;
        V3 ps = to_index(g, mulT(pose.R, view.s - pose.t));
        V3 eo = mulT(pose.R, e);
        V3 pe = {eo.x / g.vx, eo.y / g.vy, eo.z / g.vz};
        long k0, k1;
        if (!k_range(g, ps, pe, D, 3.0, k0, k1)) continue;
        V3 A = {0, 0, 0}, B = {0, 0, 0};
        double GM[3][4] = {{0}};
        for (long k = k0; k <= k1; ++k) {
          V3 r = view.s + ((k + 0.5) * D) * e;
          V3 rp = mulT(pose.R, r - pose.t);
          V3 p = to_index(g, rp);
          if (lever_arm == 0) {
            V3 gr = vol_grad(V, g, p, grad_mode);
            if (route == 0) {
              A = A + gr;
              B = B + cross(rp, gr);
            } else {
              V3 lever = r - pose.t;              // (x-tx, y-ty, z-tz), Eq.6
              V3 Rg = mul(pose.R, gr);
              for (int a = 0; a < 3; ++a) {
                GM[a][0] += comp(lever, a) * gr.x;
                GM[a][1] += comp(lever, a) * gr.y;
                GM[a][2] += comp(lever, a) * gr.z;
                GM[a][3] += -comp(Rg, a);
              }
            }
          } else {
            // VOXEL: sum_j a^ij G_f^j, a^ij = trilinear weight of voxel j (including the one-voxel
            // ring where the central difference of the zero-extended volume is still non-zero).
            double fx = floor(p.x), fy = floor(p.y), fz = floor(p.z);
            long ix = (long)fx, iy = (long)fy, iz = (long)fz;
            double ax = p.x - fx, ay = p.y - fy, az = p.z - fz;
            for (int dz = 0; dz < 2; ++dz) for (int dy = 0; dy < 2; ++dy) for (int dx = 0; dx < 2; ++dx) {
              long X = ix + dx, Y = iy + dy, Z = iz + dz;
              double wt = (dx ? ax : 1 - ax) * (dy ? ay : 1 - ay) * (dz ? az : 1 - az);
              V3 gj = {(V.at(X + 1, Y, Z) - V.at(X - 1, Y, Z)) / (2 * g.vx),
                       (V.at(X, Y + 1, Z) - V.at(X, Y - 1, Z)) / (2 * g.vy),
                       (V.at(X, Y, Z + 1) - V.at(X, Y, Z - 1)) / (2 * g.vz)};
              V3 rj = voxel_centre(g, (int)X, (int)Y, (int)Z);   // r'_j
              V3 lever = mul(pose.R, rj);                          // r_j - t = R r'_j
              V3 Rg = mul(pose.R, gj);
              for (int a = 0; a < 3; ++a) {
                GM[a][0] += wt * comp(lever, a) * gj.x;
                GM[a][1] += wt * comp(lever, a) * gj.y;
                GM[a][2] += wt * comp(lever, a) * gj.z;
                GM[a][3] += -wt * comp(Rg, a);
              }
            }
          }
        }
        if (lever_arm == 0 && route == 0) {
          acc[0] += w * D * A.x; acc[1] += w * D * A.y; acc[2] += w * D * A.z;
          acc[3] += w * D * B.x; acc[4] += w * D * B.y; acc[5] += w * D * B.z;
        } else {
          for (int a = 0; a < 3; ++a) for (int b = 0; b < 4; ++b) acc[a * 4 + b] += w * D * GM[a][b];
        }
      }
      for (int q = 0; q < 12; ++q) rowacc[(size_t)iv * 12 + q] = acc[q];
    }
    double tot[12] = {0};
    for (int iv = 0; iv < g.nv; ++iv) for (int q = 0; q < 12; ++q) tot[q] += rowacc[(size_t)iv * 12 + q];
    double* out = grad + 6 * v;
    if (lever_arm == 0 && route == 0) {
      V3 SA = {tot[0], tot[1], tot[2]}, SB = {tot[3], tot[4], tot[5]};
      V3 dt = mul(pose.R, SA);
      out[0] = -dt.x; out[1] = -dt.y; out[2] = -dt.z;
      // axial vectors of R^T dR/dgamma_k:  w_x = e_x, w_y = Rx^T e_y, w_z = (Ry Rx)^T e_z
      const double* th = poses + 6 * v;
      V3 wx = {1, 0, 0};
      V3 wy = mulT(Rx(th[3]), V3{0, 1, 0});
      V3 wz = mulT(mul(Ry(th[4]), Rx(th[3])), V3{0, 0, 1});
      out[3] = -dot(wx, SB); out[4] = -dot(wy, SB); out[5] = -dot(wz, SB);
    } else {
      double GM[3][4];
      for (int a = 0; a < 3; ++a) for (int b = 0; b < 4; ++b) GM[a][b] = tot[a * 4 + b];
      contract_M(pose, GM, out);
    }
  }
}

// zero-extended bilinear interpolant of one projection at pixel-index coordinates (u,v).  O8.
struct Img {
  const float* p; int nu, nv;
  double at(long iu, long iv) const {
    if (iu < 0 || iv < 0 || iu >= nu || iv >= nv) return 0.0;
    return (double)p[(size_t)iv * nu + iu];
  }
};
inline double bilin(const Img& I, double u, double v) {
  double fu = floor(u), fv = floor(v);
  long iu = (long)fu, iv = (long)fv;
  double a = u - fu, b = v - fv;
  return (1 - b) * ((1 - a) * I.at(iu, iv) + a * I.at(iu + 1, iv)) +
         b * ((1 - a) * I.at(iu, iv + 1) + a * I.at(iu + 1, iv + 1));
}

// ------------------------------------------------------------------------------------------------
// O8: voxel-driven back-projection, Eq.2b :71-75 / Eq.21 :193-196.
//   r_j = R_v r'_j + t_v; (u',v',w') = P_v (r_j;1); mu_j = sum_v W b~_v(u'/w', v'/w'); W = 1 | (SAD/w')^2.
void backproject_impl(const ora_geom& g, int n_views, const double* angles, const double* poses,
                      const float* proj, double* vol_out, int iz0, int iz1) {
  std::vector<View> views; std::vector<Pose> ps;
  for (int v = 0; v < n_views; ++v) { views.emplace_back(g, angles, v); ps.emplace_back(poses + 6 * v); }
#pragma omp parallel for schedule(dynamic, 1) collapse(2)
  for (int iz = iz0; iz < iz1; ++iz) for (int iy = 0; iy < g.ny; ++iy) for (int ix = 0; ix < g.nx; ++ix) {
    V3 rp = voxel_centre(g, ix, iy, iz);
    double s = 0.0;
    for (int v = 0; v < n_views; ++v) {
      V3 r = mul(ps[v].R, rp) + ps[v].t;
      const double(*P)[4] = views[v].P;
      double up = P[0][0] * r.x + P[0][1] * r.y + P[0][2] * r.z + P[0][3];
      double vp = P[1][0] * r.x + P[1][1] * r.y + P[1][2] * r.z + P[1][3];
      double wp = P[2][0] * r.x + P[2][1] * r.y + P[2][2] * r.z + P[2][3];
      if (wp <= 0) continue;
      Img I{proj + (size_t)v * g.nu * g.nv, g.nu, g.nv};
      double W = g.bp_weight ? (g.sad / wp) * (g.sad / wp) : 1.0;
      s += W * bilin(I, up / wp, vp / wp);
    }
    vol_out[((size_t)(iz - iz0) * g.ny + iy) * g.nx + ix] = s;
  }
}

// O10: explicit transpose of the back-projector (splat), adjointness pin only.
void backproject_T_impl(const ora_geom& g, int n_views, const double* angles, const double* poses,
                        const double* x, double* proj_out) {
  size_t np = (size_t)n_views * g.nu * g.nv;
  for (size_t i = 0; i < np; ++i) proj_out[i] = 0.0;
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v); Pose pose(poses + 6 * v);
    double* out = proj_out + (size_t)v * g.nu * g.nv;
    for (int iz = 0; iz < g.nz; ++iz) for (int iy = 0; iy < g.ny; ++iy) for (int ix = 0; ix < g.nx; ++ix) {
      V3 r = mul(pose.R, voxel_centre(g, ix, iy, iz)) + pose.t;
      const double(*P)[4] = view.P;
      double up = P[0][0] * r.x + P[0][1] * r.y + P[0][2] * r.z + P[0][3];
      double vp = P[1][0] * r.x + P[1][1] * r.y + P[1][2] * r.z + P[1][3];
      double wp = P[2][0] * r.x + P[2][1] * r.y + P[2][2] * r.z + P[2][3];
      if (wp <= 0) continue;
      double W = g.bp_weight ? (g.sad / wp) * (g.sad / wp) : 1.0;
      double u = up / wp, vv = vp / wp;
      double fu = floor(u), fv = floor(vv);
      long iu = (long)fu, iw = (long)fv;
      double a = u - fu, b = vv - fv;
      double xv = x[((size_t)iz * g.ny + iy) * g.nx + ix] * W;
      for (int dv = 0; dv < 2; ++dv) for (int du = 0; du < 2; ++du) {
        long U = iu + du, Vv = iw + dv;
        if (U < 0 || Vv < 0 || U >= g.nu || Vv >= g.nv) continue;
        out[(size_t)Vv * g.nu + U] += (du ? a : 1 - a) * (dv ? b : 1 - b) * xv;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// O9: back-projection pose gradient, Eq.9-17 :115-168 and Eq.22 :198-206.
//  d~_u l = [b~(u+1,v) - b~(u-1,v)]/2 (central difference in pixel units, :202); J from Eq.13 :143-146;
//  q = W (d~_u l J_u + d~_v l J_v)  [+ b~ dW/dr, dW/dr = -2 W/w' P_3[0:3], if flags&1];
//  route 0: S_q = sum_j w_j q_j, S_c = sum_j w_j (r_j - t) x q_j; dL/dt = S_q; dL/dgamma_k = a_k . S_c,
//           a_x = R e_x, a_y = Rz e_y, a_z = e_z  (axial vectors of dR/dgamma_k R^T)
//  route 1: the paper's 12-element  G_b = q^T (x) (x',y',z',1)  (Eq.15/17) contracted with dM/dtheta.
//  grad_mode 0 CENTRAL | 1 INTERP (exact derivative of the bilinear interpolant; test aid)
void backproject_grad_impl(const ora_geom& g, int n_views, const double* angles, const double* poses,
                           const float* proj, const float* upstream, double* grad, int grad_mode, int route) {
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v); Pose pose(poses + 6 * v);
    Img I{proj + (size_t)v * g.nu * g.nv, g.nu, g.nv};
    const double(*P)[4] = view.P;
    std::vector<double> slab((size_t)g.nz * 12, 0.0);
#pragma omp parallel for schedule(dynamic, 1)
    for (int iz = 0; iz < g.nz; ++iz) {
      double acc[12] = {0};
      for (int iy = 0; iy < g.ny; ++iy) for (int ix = 0; ix < g.nx; ++ix) {
        double wj = (double)upstream[((size_t)iz * g.ny + iy) * g.nx + ix];
        V3 rp = voxel_centre(g, ix, iy, iz);
        V3 r = mul(pose.R, rp) + pose.t;
        double up = P[0][0] * r.x + P[0][1] * r.y + P[0][2] * r.z + P[0][3];
        double vp = P[1][0] * r.x + P[1][1] * r.y + P[1][2] * r.z + P[1][3];
        double wp = P[2][0] * r.x + P[2][1] * r.y + P[2][2] * r.z + P[2][3];
        if (wp <= 0) continue;
        double u = up / wp, vv = vp / wp;
        double W = g.bp_weight ? (g.sad / wp) * (g.sad / wp) : 1.0;
        double dlu, dlv;
        if (grad_mode == 0) {
          dlu = 0.5 * (bilin(I, u + 1, vv) - bilin(I, u - 1, vv));
          dlv = 0.5 * (bilin(I, u, vv + 1) - bilin(I, u, vv - 1));
        } else {
          double fu = floor(u), fv = floor(vv);
          long iu = (long)fu, iw = (long)fv;
          double a = u - fu, b = vv - fv;
          dlu = (1 - b) * (I.at(iu + 1, iw) - I.at(iu, iw)) + b * (I.at(iu + 1, iw + 1) - I.at(iu, iw + 1));
          dlv = (1 - a) * (I.at(iu, iw + 1) - I.at(iu, iw)) + a * (I.at(iu + 1, iw + 1) - I.at(iu + 1, iw));
        }
        V3 Ju = {(P[0][0] * wp - P[2][0] * up) / (wp * wp), (P[0][1] * wp - P[2][1] * up) / (wp * wp),
                 (P[0][2] * wp - P[2][2] * up) / (wp * wp)};
        V3 Jv = {(P[1][0] * wp - P[2][0] * vp) / (wp * wp), (P[1][1] * wp - P[2][1] * vp) / (wp * wp),
                 (P[1][2] * wp - P[2][2] * vp) / (wp * wp)};
        V3 q = W * ((dlu * Ju) + (dlv * Jv));
        if ((g.flags & 1) && g.bp_weight) {
          V3 dW = (-2.0 * W / wp) * V3{P[2][0], P[2][1], P[2][2]};
          q = q + bilin(I, u, vv) * dW;
        }
        if (route == 0) {
          V3 c = cross(r - pose.t, q);
          acc[0] += wj * q.x; acc[1] += wj * q.y; acc[2] += wj * q.z;
          acc[3] += wj * c.x; acc[4] += wj * c.y; acc[5] += wj * c.z;
        } else {
          double h[4] = {rp.x, rp.y, rp.z, 1.0};
          for (int a = 0; a < 3; ++a) for (int b = 0; b < 4; ++b) acc[a * 4 + b] += wj * comp(q, a) * h[b];
        }
      }
      for (int k = 0; k < 12; ++k) slab[(size_t)iz * 12 + k] = acc[k];
    }
    double tot[12] = {0};
    for (int iz = 0; iz < g.nz; ++iz) for (int k = 0; k < 12; ++k) tot[k] += slab[(size_t)iz * 12 + k];
    double* out = grad + 6 * v;
    if (route == 0) {
      const double* th = poses + 6 * v;
      V3 Sq = {tot[0], tot[1], tot[2]}, Sc = {tot[3], tot[4], tot[5]};
      V3 ax = mul(pose.R, V3{1, 0, 0});
      V3 ay = mul(Rz(th[5]), V3{0, 1, 0});
      V3 az = {0, 0, 1};
      out[0] = Sq.x; out[1] = Sq.y; out[2] = Sq.z;
      out[3] = dot(ax, Sc); out[4] = dot(ay, Sc); out[5] = dot(az, Sc);
    } else {
      double GM[3][4];
      for (int a = 0; a < 3; ++a) for (int b = 0; b < 4; ++b) GM[a][b] = tot[a * 4 + b];
      contract_M(pose, GM, out);
    }
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// O12: Siddon's exact radiological path [28] - the weights of the paper's own ray-driven
// projector (PAPER.md :213, ref :395): a^ij = length of the intersection of ray i with voxel j, voxels being boxes
// of constant value mu_j (Eq.18 :172-177, "projection path length" :177).
// Following Siddon's formulation: the parameters at which the half-line s' + t e' (t >= 0, object frame, mm)
// crosses the planes of the three families that bound the voxels are merged into ONE sorted list; two consecutive
// parameters delimit a segment that lies in one voxel, identified by the segment's midpoint.
struct Seg { double len; long ix, iy, iz; };
inline void siddon_segments(const ora_geom& g, V3 so, V3 eo, std::vector<double>& ts, std::vector<Seg>& out) {
  out.clear(); ts.clear();
  const double n[3] = {(double)g.nx, (double)g.ny, (double)g.nz}, v[3] = {g.vx, g.vy, g.vz}, c[3] = {g.cx, g.cy, g.cz};
  double lo[3], tmin = 0.0, tmax = 1e300;
  for (int a = 0; a < 3; ++a) {
    lo[a] = c[a] - 0.5 * n[a] * v[a];
    const double hi = c[a] + 0.5 * n[a] * v[a], o = comp(so, a), d = comp(eo, a);
    if (fabs(d) < 1e-300) { if (o <= lo[a] || o >= hi) return; continue; }
    double t0 = (lo[a] - o) / d, t1 = (hi - o) / d;
    if (t0 > t1) std::swap(t0, t1);
    tmin = std::max(tmin, t0); tmax = std::min(tmax, t1);
  }
  if (!(tmax > tmin)) return;
  ts.push_back(tmin); ts.push_back(tmax);
  for (int a = 0; a < 3; ++a) {
    const double o = comp(so, a), d = comp(eo, a);
    if (fabs(d) < 1e-300) continue;
    for (long i = 0; i <= (long)n[a]; ++i) {
      const double t = (lo[a] + i * v[a] - o) / d;
      if (t > tmin && t < tmax) ts.push_back(t);
    }
  }
  std::sort(ts.begin(), ts.end());
  for (size_t m = 0; m + 1 < ts.size(); ++m) {
    const double len = ts[m + 1] - ts[m];
    if (!(len > 0)) continue;
    const V3 mid = so + (0.5 * (ts[m] + ts[m + 1])) * eo;
    long idx[3];
    for (int a = 0; a < 3; ++a) {
      idx[a] = (long)floor((comp(mid, a) - lo[a]) / v[a]);
      idx[a] = std::min(std::max(idx[a], 0L), (long)n[a] - 1);
    }
    out.push_back({len, idx[0], idx[1], idx[2]});
  }
}

// l_i = sum_j a^ij mu_j.  (transpose = true: the explicit transpose, vol_out += a^ij y_i; adjointness pin only.)
template <typename T>
void forward_siddon_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                         double* proj, const double* y_in, double* vol_out) {
  Vol<T> V{vol, g.nx, g.ny, g.nz};
  const bool transpose = vol_out != nullptr;
  if (transpose) for (size_t i = 0; i < (size_t)g.nx * g.ny * g.nz; ++i) vol_out[i] = 0.0;
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    const V3 so = mulT(pose.R, view.s - pose.t);
#pragma omp parallel for schedule(dynamic, 4) if (!transpose)
    for (int iv = 0; iv < g.nv; ++iv) {
      std::vector<double> ts; std::vector<Seg> segs;
      for (int iu = 0; iu < g.nu; ++iu) {
        V3 d = view.pixel(g, iu, iv) - view.s;
        V3 eo = mulT(pose.R, (1.0 / sqrt(dot(d, d))) * d);
        siddon_segments(g, so, eo, ts, segs);
        const size_t pix = ((size_t)v * g.nv + iv) * g.nu + iu;
        if (!transpose) {
          double sum = 0.0;
          for (const Seg& sg : segs) sum += sg.len * V.at(sg.ix, sg.iy, sg.iz);
          proj[pix] = sum;
        } else {
          for (const Seg& sg : segs) vol_out[((size_t)sg.iz * g.ny + sg.iy) * g.nx + sg.ix] += sg.len * y_in[pix];
        }
      }
    }
  }
}

// Pose gradient with Siddon weights, the paper's discretisation taken literally (Eq.19-20 :179-191, :189
// "Compute matrix G_f^j for each voxel"): per voxel j of the grid, g_j = central differences of the zero-extended
// voxel values (:183), lever arm at the voxel centre r'_j;
//   A_i = sum_j a^ij g_j,  B_i = sum_j a^ij r'_j x g_j;  S_A = sum_i w_i A_i, S_B likewise;
//   route 0: dL/dt = -R S_A, dL/dgamma_k = -w_k.S_B;  route 1: the 12-element G_f^j = [ (R r'_j) g_j^T | -R g_j ].
template <typename T>
void forward_grad_siddon_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                              const float* upstream, double* grad, int route) {
  Vol<T> V{vol, g.nx, g.ny, g.nz};
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    const V3 so = mulT(pose.R, view.s - pose.t);
    std::vector<double> rowacc((size_t)g.nv * 12, 0.0);
#pragma omp parallel for schedule(dynamic, 4)
    for (int iv = 0; iv < g.nv; ++iv) {
      std::vector<double> ts; std::vector<Seg> segs;
      double acc[12] = {0};
      for (int iu = 0; iu < g.nu; ++iu) {
        const double w = (double)upstream[((size_t)v * g.nv + iv) * g.nu + iu];
        V3 d = view.pixel(g, iu, iv) - view.s;
        V3 eo = mulT(pose.R, (1.0 / sqrt(dot(d, d))) * d);
        siddon_segments(g, so, eo, ts, segs);
        V3 A = {0, 0, 0}, B = {0, 0, 0};
        double GM[3][4] = {{0}};
        for (const Seg& sg : segs) {
          const long X = sg.ix, Y = sg.iy, Z = sg.iz;
          V3 gj = {(V.at(X + 1, Y, Z) - V.at(X - 1, Y, Z)) / (2 * g.vx),
                   (V.at(X, Y + 1, Z) - V.at(X, Y - 1, Z)) / (2 * g.vy),
                   (V.at(X, Y, Z + 1) - V.at(X, Y, Z - 1)) / (2 * g.vz)};
          V3 rj = voxel_centre(g, (int)X, (int)Y, (int)Z);
          if (route == 0) {
            A = A + sg.len * gj;
            B = B + sg.len * cross(rj, gj);
          } else {
            V3 lever = mul(pose.R, rj), Rg = mul(pose.R, gj);
            for (int a = 0; a < 3; ++a) {
              GM[a][0] += sg.len * comp(lever, a) * gj.x;
              GM[a][1] += sg.len * comp(lever, a) * gj.y;
              GM[a][2] += sg.len * comp(lever, a) * gj.z;
              GM[a][3] += -sg.len * comp(Rg, a);
            }
          }
        }
        if (route == 0) {
          acc[0] += w * A.x; acc[1] += w * A.y; acc[2] += w * A.z;
          acc[3] += w * B.x; acc[4] += w * B.y; acc[5] += w * B.z;
        } else {
          for (int a = 0; a < 3; ++a) for (int b = 0; b < 4; ++b) acc[a * 4 + b] += w * GM[a][b];
        }
      }
      for (int q = 0; q < 12; ++q) rowacc[(size_t)iv * 12 + q] = acc[q];
    }
    double tot[12] = {0};
    for (int iv = 0; iv < g.nv; ++iv) for (int q = 0; q < 12; ++q) tot[q] += rowacc[(size_t)iv * 12 + q];
    double* out = grad + 6 * v;
    if (route == 0) {
      V3 SA = {tot[0], tot[1], tot[2]}, SB = {tot[3], tot[4], tot[5]};
      V3 dt = mul(pose.R, SA);
      out[0] = -dt.x; out[1] = -dt.y; out[2] = -dt.z;
      const double* th = poses + 6 * v;
      V3 wx = {1, 0, 0};
      V3 wy = mulT(Rx(th[3]), V3{0, 1, 0});
      V3 wz = mulT(mul(Ry(th[4]), Rx(th[3])), V3{0, 0, 1});
      out[3] = -dot(wx, SB); out[4] = -dot(wy, SB); out[5] = -dot(wz, SB);
    } else {
      double GM[3][4];
      for (int a = 0; a < 3; ++a) for (int b = 0; b < 4; ++b) GM[a][b] = tot[a * 4 + b];
      contract_M(pose, GM, out);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// O13: Joseph's projector (BASELINE.json north_star: "trilinear or Joseph interpolation").
// The ray is stepped from voxel-centre plane to voxel-centre plane along its DRIVING axis a* = argmax_a |e'_a|
// (object frame); in each plane the volume is interpolated bilinearly (zero-extended) at the intersection point, and
// every plane carries the path length between consecutive planes, v_a* / |e'_a*|:
//   l_i = (v_a* / |e'_a*|) sum_k bilin_k,   a^ij = (v_a* / |e'_a*|) x (bilinear weight of voxel j in its plane).
// Only intersections on the half-line t > 0 from the source count (as O6).  `visit` receives (weight, ix, iy, iz) for
// every voxel of the GRID with a non-zero weight.
template <typename F>
inline void joseph_weights(const ora_geom& g, V3 so, V3 eo, F visit) {
  const int n[3] = {g.nx, g.ny, g.nz};
  const double v[3] = {g.vx, g.vy, g.vz}, c[3] = {g.cx, g.cy, g.cz};
  int a = 0;
  for (int k = 1; k < 3; ++k) if (fabs(comp(eo, k)) > fabs(comp(eo, a))) a = k;
  const int b = (a + 1) % 3, d = (a + 2) % 3;
  const double ea = comp(eo, a);
  if (fabs(ea) < 1e-300) return;
  const double wlen = v[a] / fabs(ea);
  for (int k = 0; k < n[a]; ++k) {
    const double xa = c[a] + (k - (n[a] - 1) / 2.0) * v[a];            // plane of voxel centres (O1)
    const double t = (xa - comp(so, a)) / ea;
    if (!(t > 0)) continue;
    const double pb = (comp(so, b) + t * comp(eo, b) - c[b]) / v[b] + (n[b] - 1) / 2.0;   // continuous indices
    const double pd = (comp(so, d) + t * comp(eo, d) - c[d]) / v[d] + (n[d] - 1) / 2.0;
    const double fb = floor(pb), fd = floor(pd), ab = pb - fb, ad = pd - fd;
    for (int jd = 0; jd < 2; ++jd) for (int jb = 0; jb < 2; ++jb) {
      const long ib = (long)fb + jb, id = (long)fd + jd;
      if (ib < 0 || id < 0 || ib >= n[b] || id >= n[d]) continue;
      const double w = wlen * (jb ? ab : 1 - ab) * (jd ? ad : 1 - ad);
      if (w == 0.0) continue;
      long idx[3];
      idx[a] = k; idx[b] = ib; idx[d] = id;
      visit(w, idx[0], idx[1], idx[2]);
    }
  }
}

// forward (vol_out == nullptr) or explicit transpose (adjointness pin only)
template <typename T>
void forward_joseph_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                         double* proj, const double* y_in, double* vol_out) {
  Vol<T> V{vol, g.nx, g.ny, g.nz};
  const bool transpose = vol_out != nullptr;
  if (transpose) for (size_t i = 0; i < (size_t)g.nx * g.ny * g.nz; ++i) vol_out[i] = 0.0;
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    const V3 so = mulT(pose.R, view.s - pose.t);
#pragma omp parallel for schedule(dynamic, 4) if (!transpose)
    for (int iv = 0; iv < g.nv; ++iv) {
      for (int iu = 0; iu < g.nu; ++iu) {
        V3 d = view.pixel(g, iu, iv) - view.s;
        V3 eo = mulT(pose.R, (1.0 / sqrt(dot(d, d))) * d);
        const size_t pix = ((size_t)v * g.nv + iv) * g.nu + iu;
        if (!transpose) {
          double sum = 0.0;
          joseph_weights(g, so, eo, [&](double w, long ix, long iy, long iz) { sum += w * V.at(ix, iy, iz); });
          proj[pix] = sum;
        } else {
          const double yi = y_in[pix];
          joseph_weights(g, so, eo, [&](double w, long ix, long iy, long iz) {
            vol_out[((size_t)iz * g.ny + iy) * g.nx + ix] += w * yi;
          });
        }
      }
    }
  }
}

// Pose gradient with Joseph weights and per-voxel G_f^j (as O12): A_i = sum_j a^ij g_j, B_i = sum_j a^ij r'_j x g_j.
template <typename T>
void forward_grad_joseph_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                              const float* upstream, double* grad) {
  Vol<T> V{vol, g.nx, g.ny, g.nz};
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    const V3 so = mulT(pose.R, view.s - pose.t);
    std::vector<double> rowacc((size_t)g.nv * 6, 0.0);
#pragma omp parallel for schedule(dynamic, 4)
    for (int iv = 0; iv < g.nv; ++iv) {
      double acc[6] = {0};
      for (int iu = 0; iu < g.nu; ++iu) {
        const double w = (double)upstream[((size_t)v * g.nv + iv) * g.nu + iu];
        V3 d = view.pixel(g, iu, iv) - view.s;
        V3 eo = mulT(pose.R, (1.0 / sqrt(dot(d, d))) * d);
        V3 A = {0, 0, 0}, B = {0, 0, 0};
        joseph_weights(g, so, eo, [&](double a, long X, long Y, long Z) {
          V3 gj = {(V.at(X + 1, Y, Z) - V.at(X - 1, Y, Z)) / (2 * g.vx),
                   (V.at(X, Y + 1, Z) - V.at(X, Y - 1, Z)) / (2 * g.vy),
                   (V.at(X, Y, Z + 1) - V.at(X, Y, Z - 1)) / (2 * g.vz)};
          V3 rj = voxel_centre(g, (int)X, (int)Y, (int)Z);
          A = A + a * gj;
          B = B + a * cross(rj, gj);
        });
        acc[0] += w * A.x; acc[1] += w * A.y; acc[2] += w * A.z;
        acc[3] += w * B.x; acc[4] += w * B.y; acc[5] += w * B.z;
      }
      for (int q = 0; q < 6; ++q) rowacc[(size_t)iv * 6 + q] = acc[q];
    }
    double tot[6] = {0};
    for (int iv = 0; iv < g.nv; ++iv) for (int q = 0; q < 6; ++q) tot[q] += rowacc[(size_t)iv * 6 + q];
    V3 SA = {tot[0], tot[1], tot[2]}, SB = {tot[3], tot[4], tot[5]};
    V3 dt = mul(pose.R, SA);
    double* out = grad + 6 * v;
    out[0] = -dt.x; out[1] = -dt.y; out[2] = -dt.z;
    const double* th = poses + 6 * v;
    V3 wx = {1, 0, 0};
    V3 wy = mulT(Rx(th[3]), V3{0, 1, 0});
    V3 wz = mulT(mul(Ry(th[4]), Rx(th[3])), V3{0, 0, 1});
    out[3] = -dot(wx, SB); out[4] = -dot(wy, SB); out[5] = -dot(wz, SB);
  }
}

// ------------------------------------------------------------------------------------------------
// O15: distance-driven projector pair [44] (PAPER.md :213, Tables III / IV rows DD) under a rigid
// pose and a general flat detector.  The paper cites the method and gives no formula; reading taken (U14):
//   * everything in the OBJECT frame: source s' = R^T (s - t), detector points X(u, v) = R^T (c + (u - c_u) U +
//     (v - c_v) V - t) for real (u, v) - pixel (iu, iv) covers [iu - 1/2, iu + 1/2] x [iv - 1/2, iv + 1/2];
//   * per VIEW the driving axis a* = argmax_a |n'_a|, n' = direction from s' to the detector's central point
//     ((nu-1)/2, (nv-1)/2); the other two axes (b, d) = ((a*+1)%3, (a*+2)%3); the detector's u pairs with the in-plane
//     axis along which the pixel step U' = R^T U is longer (|U'_b| >= |U'_d|: u<->b, v<->d; else u<->d, v<->b);
//   * per plane k of voxel centres along a* (x_a = c_a + (k - (n_a - 1)/2) v_a): the pixel's boundary mid-points
//     (iu -+ 1/2, iv) and (iu, iv -+ 1/2) are projected from the source onto the plane; in continuous voxel indices
//     they bound the pixel's footprint [B0, B1] along u's axis and [D0, D1] along v's axis (the distance-driven
//     separable footprint, taken per pixel so that in-plane rotations of the pose are followed);
//   * a^ij = L (|[B0,B1] n cell_B(j)| / (B1 - B0)) (|[D0,D1] n cell_D(j)| / (D1 - D0)),  cell(j) = [j - 1/2, j + 1/2],
//     L = v_a* / |e'_a*| with e' the unit direction of the pixel-centre ray: normalised overlap x slab path length
//     (a uniform volume gives the chord); planes behind the source (any of the five rays with t <= 0) are skipped.
// Forward l_i = sum_j a^ij mu_j; the back-projector is its EXACT transpose mu_j = sum_i a^ij l_i (Eq.21 :193-196: DD
// is a matched pair), unit weight only.  `visit(w, ix, iy, iz)` for every grid voxel with a non-zero weight.
struct DDView {
  V3 so, X00, Uo, Vo;          // object frame: source, detector point of index (0, 0), steps per pixel along u and v
  int a, b, d;                 // driving axis and the two in-plane axes
  bool u_is_b;
  DDView(const ora_geom& g, const View& view, const Pose& pose) {
    so = mulT(pose.R, view.s - pose.t);
    Uo = mulT(pose.R, view.U); Vo = mulT(pose.R, view.Vs);
    X00 = mulT(pose.R, view.dc - pose.t) - view.cu * Uo - view.cv * Vo;
    V3 n = X00 + ((g.nu - 1) / 2.0) * Uo + ((g.nv - 1) / 2.0) * Vo - so;
    a = 0;
    for (int k = 1; k < 3; ++k) if (fabs(comp(n, k)) > fabs(comp(n, a))) a = k;
    b = (a + 1) % 3; d = (a + 2) % 3;
    u_is_b = fabs(comp(Uo, b)) >= fabs(comp(Uo, d));
  }
  V3 det(double u, double v) const { return X00 + u * Uo + v * Vo; }
};
template <typename F>
inline void dd_weights(const ora_geom& g, const DDView& W, int iu, int iv, F visit) {
  const int n[3] = {g.nx, g.ny, g.nz};
  const double v[3] = {g.vx, g.vy, g.vz}, c[3] = {g.cx, g.cy, g.cz};
  const int a = W.a, ub = W.u_is_b ? W.b : W.d, vb = W.u_is_b ? W.d : W.b;   // axis paired with u, with v
  const V3 pts[5] = {W.det(iu, iv), W.det(iu - 0.5, iv), W.det(iu + 0.5, iv), W.det(iu, iv - 0.5), W.det(iu, iv + 0.5)};
  V3 dir[5];
  for (int q = 0; q < 5; ++q) dir[q] = pts[q] - W.so;
  const double elen = sqrt(dot(dir[0], dir[0]));
  const double ea = comp(dir[0], a) / elen;
  if (fabs(ea) < 1e-300) return;
  const double L = v[a] / fabs(ea);
  for (int k = 0; k < n[a]; ++k) {
    const double xa = c[a] + (k - (n[a] - 1) / 2.0) * v[a];
    double t[5];
    bool front = true;
    for (int q = 0; q < 5; ++q) {
      const double da = comp(dir[q], a);
      if (fabs(da) < 1e-300) { front = false; break; }
      t[q] = (xa - comp(W.so, a)) / da;
      if (!(t[q] > 0)) { front = false; break; }
    }
    if (!front) continue;
    auto idx = [&](int q, int ax) { return (comp(W.so, ax) + t[q] * comp(dir[q], ax) - c[ax]) / v[ax] + (n[ax] - 1) / 2.0; };
    double B0 = idx(1, ub), B1 = idx(2, ub), D0 = idx(3, vb), D1 = idx(4, vb);
    if (B0 > B1) std::swap(B0, B1);
    if (D0 > D1) std::swap(D0, D1);
    if (!(B1 > B0) || !(D1 > D0)) continue;
    const long jb0 = (long)floor(B0 + 0.5), jb1 = (long)floor(B1 + 0.5);
    const long jd0 = (long)floor(D0 + 0.5), jd1 = (long)floor(D1 + 0.5);
    for (long jd = jd0; jd <= jd1; ++jd) {
      if (jd < 0 || jd >= n[vb]) continue;
      const double od = std::min(D1, jd + 0.5) - std::max(D0, jd - 0.5);
      if (!(od > 0)) continue;
      for (long jb = jb0; jb <= jb1; ++jb) {
        if (jb < 0 || jb >= n[ub]) continue;
        const double ob = std::min(B1, jb + 0.5) - std::max(B0, jb - 0.5);
        if (!(ob > 0)) continue;
        long id[3];
        id[a] = k; id[ub] = jb; id[vb] = jd;
        visit(L * (ob / (B1 - B0)) * (od / (D1 - D0)), id[0], id[1], id[2]);
      }
    }
  }
}

// forward (vol_out == nullptr) or explicit transpose = the DD back-projector, slab [iz0, iz1) of the volume
template <typename T>
void forward_dd_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                     double* proj, const float* y_in, double* vol_out, int iz0, int iz1) {
  Vol<T> V{vol, g.nx, g.ny, g.nz};
  const bool transpose = vol_out != nullptr;
  const size_t nslab = transpose ? (size_t)(iz1 - iz0) * g.ny * g.nx : 0;
  for (size_t i = 0; i < nslab; ++i) vol_out[i] = 0.0;
  int nthr = 1;
#ifdef _OPENMP
  nthr = omp_get_max_threads();
#endif
  std::vector<std::vector<double>> priv(transpose ? nthr : 0);
  for (auto& p : priv) p.assign(nslab, 0.0);
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    const DDView W(g, view, pose);
#pragma omp parallel for schedule(static)      // fixed row -> thread map: the transpose's sums have one order
    for (int iv = 0; iv < g.nv; ++iv) {
      int me = 0;
#ifdef _OPENMP
      me = omp_get_thread_num();
#endif
      for (int iu = 0; iu < g.nu; ++iu) {
        const size_t pix = ((size_t)v * g.nv + iv) * g.nu + iu;
        if (!transpose) {
          double sum = 0.0;
          dd_weights(g, W, iu, iv, [&](double w, long ix, long iy, long iz) { sum += w * V.at(ix, iy, iz); });
          proj[pix] = sum;
        } else {
          const double yi = (double)y_in[pix];
          double* out = priv[me].data();
          dd_weights(g, W, iu, iv, [&](double w, long ix, long iy, long iz) {
            if (iz >= iz0 && iz < iz1) out[((size_t)(iz - iz0) * g.ny + iy) * g.nx + ix] += w * yi;
          });
        }
      }
    }
  }
  for (auto& p : priv) for (size_t i = 0; i < nslab; ++i) vol_out[i] += p[i];      // thread order: fixed
}

// Pose gradient through the DD forward projector: per-voxel G_f^j with the weights a^ij (Eq.19-20 :179-191), as O12.
template <typename T>
void forward_grad_dd_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                          const float* upstream, double* grad) {
  Vol<T> V{vol, g.nx, g.ny, g.nz};
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    const DDView W(g, view, pose);
    std::vector<double> rowacc((size_t)g.nv * 6, 0.0);
#pragma omp parallel for schedule(dynamic, 4)
    for (int iv = 0; iv < g.nv; ++iv) {
      double acc[6] = {0};
      for (int iu = 0; iu < g.nu; ++iu) {
        const double w = (double)upstream[((size_t)v * g.nv + iv) * g.nu + iu];
        V3 A = {0, 0, 0}, B = {0, 0, 0};
        dd_weights(g, W, iu, iv, [&](double a, long X, long Y, long Z) {
          V3 gj = {(V.at(X + 1, Y, Z) - V.at(X - 1, Y, Z)) / (2 * g.vx),
                   (V.at(X, Y + 1, Z) - V.at(X, Y - 1, Z)) / (2 * g.vy),
                   (V.at(X, Y, Z + 1) - V.at(X, Y, Z - 1)) / (2 * g.vz)};
          V3 rj = voxel_centre(g, (int)X, (int)Y, (int)Z);
          A = A + a * gj;
          B = B + a * cross(rj, gj);
        });
        acc[0] += w * A.x; acc[1] += w * A.y; acc[2] += w * A.z;
        acc[3] += w * B.x; acc[4] += w * B.y; acc[5] += w * B.z;
      }
      for (int q = 0; q < 6; ++q) rowacc[(size_t)iv * 6 + q] = acc[q];
    }
    double tot[6] = {0};
    for (int iv = 0; iv < g.nv; ++iv) for (int q = 0; q < 6; ++q) tot[q] += rowacc[(size_t)iv * 6 + q];
    V3 SA = {tot[0], tot[1], tot[2]}, SB = {tot[3], tot[4], tot[5]};
    V3 dt = mul(pose.R, SA);
    double* out = grad + 6 * v;
    out[0] = -dt.x; out[1] = -dt.y; out[2] = -dt.z;
    const double* th = poses + 6 * v;
    V3 wx = {1, 0, 0};
    V3 wy = mulT(Rx(th[3]), V3{0, 1, 0});
    V3 wz = mulT(mul(Ry(th[4]), Rx(th[3])), V3{0, 0, 1});
    out[3] = -dot(wx, SB); out[4] = -dot(wy, SB); out[5] = -dot(wz, SB);
  }
}

// Pose gradient through the DD back-projector, Eq.22 (:198-206) with the DD weights: per detector PIXEL i the
// central differences of the zero-extended projection, D_u^i = (l[iv][iu+1] - l[iv][iu-1]) / 2, D_v^i likewise ("the
// projection gradient is approximated by a central finite difference", "compute G_b^i for each detector pixel"; i runs
// over the detector's pixels); per pair (i, j): a^ij w_j (D_u^i J_u(r_j) + D_v^i J_v(r_j)), J from Eq.13 at the voxel
// centre r_j = R r'_j + t; S_q, S_c and the contraction as O9.
void backproject_grad_dd_impl(const ora_geom& g, int n_views, const double* angles, const double* poses,
                              const float* proj, const float* upstream, double* grad) {
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    const DDView W(g, view, pose);
    Img I{proj + (size_t)v * g.nu * g.nv, g.nu, g.nv};
    const double(*P)[4] = view.P;
    std::vector<double> rowacc((size_t)g.nv * 6, 0.0);
#pragma omp parallel for schedule(dynamic, 4)
    for (int iv = 0; iv < g.nv; ++iv) {
      double acc[6] = {0};
      for (int iu = 0; iu < g.nu; ++iu) {
        const double Du = 0.5 * (I.at(iu + 1, iv) - I.at(iu - 1, iv)), Dv = 0.5 * (I.at(iu, iv + 1) - I.at(iu, iv - 1));
        if (Du == 0.0 && Dv == 0.0) continue;
        dd_weights(g, W, iu, iv, [&](double a, long X, long Y, long Z) {
          const double wj = (double)upstream[((size_t)Z * g.ny + Y) * g.nx + X];
          V3 r = mul(pose.R, voxel_centre(g, (int)X, (int)Y, (int)Z)) + pose.t;
          double up = P[0][0] * r.x + P[0][1] * r.y + P[0][2] * r.z + P[0][3];
          double vp = P[1][0] * r.x + P[1][1] * r.y + P[1][2] * r.z + P[1][3];
          double wp = P[2][0] * r.x + P[2][1] * r.y + P[2][2] * r.z + P[2][3];
          V3 Ju = {(P[0][0] * wp - P[2][0] * up) / (wp * wp), (P[0][1] * wp - P[2][1] * up) / (wp * wp),
                   (P[0][2] * wp - P[2][2] * up) / (wp * wp)};
          V3 Jv = {(P[1][0] * wp - P[2][0] * vp) / (wp * wp), (P[1][1] * wp - P[2][1] * vp) / (wp * wp),
                   (P[1][2] * wp - P[2][2] * vp) / (wp * wp)};
          V3 q = (a * wj) * ((Du * Ju) + (Dv * Jv));
          V3 cq = cross(r - pose.t, q);
          acc[0] += q.x; acc[1] += q.y; acc[2] += q.z;
          acc[3] += cq.x; acc[4] += cq.y; acc[5] += cq.z;
        });
      }
      for (int k = 0; k < 6; ++k) rowacc[(size_t)iv * 6 + k] = acc[k];
    }
    double tot[6] = {0};
    for (int iv = 0; iv < g.nv; ++iv) for (int k = 0; k < 6; ++k) tot[k] += rowacc[(size_t)iv * 6 + k];
    const double* th = poses + 6 * v;
    V3 Sq = {tot[0], tot[1], tot[2]}, Sc = {tot[3], tot[4], tot[5]};
    V3 ax = mul(pose.R, V3{1, 0, 0});
    V3 ay = mul(Rz(th[5]), V3{0, 1, 0});
    V3 az = {0, 0, 1};
    double* out = grad + 6 * v;
    out[0] = Sq.x; out[1] = Sq.y; out[2] = Sq.z;
    out[3] = dot(ax, Sc); out[4] = dot(ay, Sc); out[5] = dot(az, Sc);
  }
}

// ------------------------------------------------------------------------------------------------
// O16 (last item): separable-footprint projector pair [29] (PAPER.md :213, Tables III / IV rows SF)
// under a rigid pose.  The paper cites the method and gives no formula; [29] builds its trapezoids from the corners of
// a voxel whose axes are aligned with the detector's, which a 6-DOF pose breaks (taken literally under an in-plane
// rotation psi the footprint loses a factor cos^2 psi of its mass and the projector no longer converges - tried).
// Reading taken (U16), voxel-driven, everything from Eq.13's Jacobian at the voxel centre:
//   * (u_j, v_j) = p(r_j) and J = d(u, v)/d r' (2 x 3, pixel-index units per mm; Eq.13 :143-146 with P_eff = P [R | t]);
//   * widths of the voxel along the detector axes: wu_k = |J_uk| v_k, wv_k = |J_vk| v_k, k = x', y', z';
//   * T(u) = the unit-area TRAPEZOID that is the convolution of the two widest rects among wu (base w1 + w2, top
//     w1 - w2), centred at u_j; R(v) likewise from wv, centred at v_j  (SF's separable footprint with trapezoids
//     along both axes, "SF-TT", linearised about the voxel centre; the third, narrowest rect of each axis is dropped);
//   * mass M_j = v_x v_y v_z sqrt(det(J J^T)): the integral of the voxel's chord-length image over the detector in
//     pixel units (J annihilates the ray direction, so sqrt(det J J^T) is the area magnification of the plane
//     perpendicular to the ray);
//   * a^ij = M_j * int_{iu-1/2}^{iu+1/2} T(u) du * int_{iv-1/2}^{iv+1/2} R(v) dv   (detector blur = the pixel's rect).
// Voxels behind the source (w' <= 0) contribute nothing.  `visit(w, iu, iv)` for the view's pixels.
struct SFView {
  double E[3][4];               // P_eff: (u', v', w') = E (r'; 1), pixel-index units, object-frame mm
  SFView(const ora_geom& g, const View& view, const Pose& pose) {
    (void)g;
    for (int r = 0; r < 3; ++r) {
      for (int c = 0; c < 3; ++c)
        E[r][c] = view.P[r][0] * pose.R.m[0][c] + view.P[r][1] * pose.R.m[1][c] + view.P[r][2] * pose.R.m[2][c];
      E[r][3] = view.P[r][0] * pose.t.x + view.P[r][1] * pose.t.y + view.P[r][2] * pose.t.z + view.P[r][3];
    }
  }
};
// int_{-inf}^{x} of the unit-area trapezoid centred at c with base b >= top t >= 0
inline double trap_cdf(double c, double b, double t, double x) {
  const double h = 2.0 / (b + t);                   // height: area = h (b + t) / 2 = 1
  const double x0 = c - 0.5 * b, x1 = c - 0.5 * t, x2 = c + 0.5 * t, x3 = c + 0.5 * b;
  double s = 0.0;
  if (x1 > x0) { const double r = std::min(std::max(x, x0), x1) - x0; s += h * r * r / (2.0 * (x1 - x0)); }
  s += h * (std::min(std::max(x, x1), x2) - x1);
  if (x3 > x2) { const double r = std::min(std::max(x, x2), x3) - x2; s += h * (r - r * r / (2.0 * (x3 - x2))); }
  return s;
}
inline void two_widest(const double* w, double* base, double* top) {
  double a = w[0], b = w[1], c = w[2];
  if (a < b) std::swap(a, b);
  if (b < c) std::swap(b, c);
  if (a < b) std::swap(a, b);
  *base = a + b; *top = a - b;
}
template <typename F>
inline void sf_weights(const ora_geom& g, const SFView& S, int ix, int iy, int iz, F visit) {
  const double v[3] = {g.vx, g.vy, g.vz};
  const V3 rc = voxel_centre(g, ix, iy, iz);
  const double up = S.E[0][0] * rc.x + S.E[0][1] * rc.y + S.E[0][2] * rc.z + S.E[0][3];
  const double vp = S.E[1][0] * rc.x + S.E[1][1] * rc.y + S.E[1][2] * rc.z + S.E[1][3];
  const double wp = S.E[2][0] * rc.x + S.E[2][1] * rc.y + S.E[2][2] * rc.z + S.E[2][3];
  if (!(wp > 0)) return;
  const double uj = up / wp, vj = vp / wp;
  double Ju[3], Jv[3], wu[3], wv[3];
  for (int k = 0; k < 3; ++k) {
    Ju[k] = (S.E[0][k] * wp - S.E[2][k] * up) / (wp * wp);      // Eq.13
    Jv[k] = (S.E[1][k] * wp - S.E[2][k] * vp) / (wp * wp);
    wu[k] = fabs(Ju[k]) * v[k]; wv[k] = fabs(Jv[k]) * v[k];
  }
  const double guu = Ju[0] * Ju[0] + Ju[1] * Ju[1] + Ju[2] * Ju[2], gvv = Jv[0] * Jv[0] + Jv[1] * Jv[1] + Jv[2] * Jv[2],
               guv = Ju[0] * Jv[0] + Ju[1] * Jv[1] + Ju[2] * Jv[2];
  const double M = v[0] * v[1] * v[2] * sqrt(std::max(guu * gvv - guv * guv, 0.0));
  double bu, tu, bv, tv;
  two_widest(wu, &bu, &tu);
  two_widest(wv, &bv, &tv);
  if (!(bu > 0) || !(bv > 0) || !(M > 0)) return;
  const long iu0 = std::max((long)floor(uj - 0.5 * bu + 0.5), 0L), iu1 = std::min((long)floor(uj + 0.5 * bu + 0.5), (long)g.nu - 1);
  const long iv0 = std::max((long)floor(vj - 0.5 * bv + 0.5), 0L), iv1 = std::min((long)floor(vj + 0.5 * bv + 0.5), (long)g.nv - 1);
  for (long iv = iv0; iv <= iv1; ++iv) {
    const double fv = trap_cdf(vj, bv, tv, iv + 0.5) - trap_cdf(vj, bv, tv, iv - 0.5);
    if (!(fv > 0)) continue;
    for (long iu = iu0; iu <= iu1; ++iu) {
      const double fu = trap_cdf(uj, bu, tu, iu + 0.5) - trap_cdf(uj, bu, tu, iu - 0.5);
      if (!(fu > 0)) continue;
      visit(M * fu * fv, iu, iv);
    }
  }
}

// mode 0: forward l_i = sum_j a^ij mu_j;  mode 1: back-projection mu_j = sum_i a^ij l_i (exact transpose), slab [iz0, iz1)
template <typename T>
void sf_project_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                     double* proj, const float* y_in, double* vol_out, int iz0, int iz1) {
  const bool back = vol_out != nullptr;
  const size_t npix = (size_t)g.nu * g.nv;
  if (back) for (size_t i = 0; i < (size_t)(iz1 - iz0) * g.ny * g.nx; ++i) vol_out[i] = 0.0;
  int nthr = 1;
#ifdef _OPENMP
  nthr = omp_get_max_threads();
#endif
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    const SFView S(g, view, pose);
    if (back) {
#pragma omp parallel for schedule(dynamic, 1) collapse(2)
      for (int iz = iz0; iz < iz1; ++iz) for (int iy = 0; iy < g.ny; ++iy) for (int ix = 0; ix < g.nx; ++ix) {
        double s = 0.0;
        sf_weights(g, S, ix, iy, iz, [&](double w, long iu, long iv) { s += w * (double)y_in[(size_t)v * npix + (size_t)iv * g.nu + iu]; });
        vol_out[((size_t)(iz - iz0) * g.ny + iy) * g.nx + ix] += s;
      }
    } else {
      std::vector<std::vector<double>> priv(nthr, std::vector<double>(npix, 0.0));
#pragma omp parallel for schedule(static)
      for (int iz = 0; iz < g.nz; ++iz) {
        int me = 0;
#ifdef _OPENMP
        me = omp_get_thread_num();
#endif
        double* out = priv[me].data();
        for (int iy = 0; iy < g.ny; ++iy) for (int ix = 0; ix < g.nx; ++ix) {
          const double mu = (double)vol[((size_t)iz * g.ny + iy) * g.nx + ix];
          if (mu == 0.0) continue;
          sf_weights(g, S, ix, iy, iz, [&](double w, long iu, long iv) { out[(size_t)iv * g.nu + iu] += w * mu; });
        }
      }
      double* dst = proj + (size_t)v * npix;
      for (size_t i = 0; i < npix; ++i) { double s = 0.0; for (int t = 0; t < nthr; ++t) s += priv[t][i]; dst[i] = s; }
    }
  }
}

// mode 0: forward pose gradient  sum_ij w_i a^ij G_f^j = sum_j (A^T w)_j G_f^j  (per-voxel G_f^j, Eq.19-20);
// mode 1: back-projection pose gradient  sum_ij a^ij w_j (D_u^i J_u(r_j) + D_v^i J_v(r_j))  (per-pixel G_b^i, Eq.22; as O15).
template <typename T>
void sf_grad_impl(const ora_geom& g, int n_views, const double* angles, const double* poses, const T* vol,
                  const float* img, const float* upvol, double* grad, int mode) {
  Vol<T> V{vol, g.nx, g.ny, g.nz};
  const size_t npix = (size_t)g.nu * g.nv;
  for (int v = 0; v < n_views; ++v) {
    View view(g, angles, v);
    Pose pose(poses + 6 * v);
    const SFView S(g, view, pose);
    Img I{img + (size_t)v * npix, g.nu, g.nv};
    const double(*P)[4] = view.P;
    std::vector<double> slab((size_t)g.nz * 6, 0.0);
#pragma omp parallel for schedule(dynamic, 1)
    for (int iz = 0; iz < g.nz; ++iz) {
      double acc[6] = {0};
      for (int iy = 0; iy < g.ny; ++iy) for (int ix = 0; ix < g.nx; ++ix) {
        if (mode == 0) {
          double s = 0.0;
          sf_weights(g, S, ix, iy, iz, [&](double w, long iu, long iv) { s += w * I.at(iu, iv); });
          if (s == 0.0) continue;
          V3 gj = {(V.at(ix + 1, iy, iz) - V.at(ix - 1, iy, iz)) / (2 * g.vx),
                   (V.at(ix, iy + 1, iz) - V.at(ix, iy - 1, iz)) / (2 * g.vy),
                   (V.at(ix, iy, iz + 1) - V.at(ix, iy, iz - 1)) / (2 * g.vz)};
          V3 rj = voxel_centre(g, ix, iy, iz), c = cross(rj, gj);
          acc[0] += s * gj.x; acc[1] += s * gj.y; acc[2] += s * gj.z;
          acc[3] += s * c.x; acc[4] += s * c.y; acc[5] += s * c.z;
        } else {
          const double wj = (double)upvol[((size_t)iz * g.ny + iy) * g.nx + ix];
          double su = 0.0, sv = 0.0;
          sf_weights(g, S, ix, iy, iz, [&](double w, long iu, long iv) {
            su += w * 0.5 * (I.at(iu + 1, iv) - I.at(iu - 1, iv));
            sv += w * 0.5 * (I.at(iu, iv + 1) - I.at(iu, iv - 1));
          });
          if (su == 0.0 && sv == 0.0) continue;
          V3 r = mul(pose.R, voxel_centre(g, ix, iy, iz)) + pose.t;
          double up = P[0][0] * r.x + P[0][1] * r.y + P[0][2] * r.z + P[0][3];
          double vp = P[1][0] * r.x + P[1][1] * r.y + P[1][2] * r.z + P[1][3];
          double wp = P[2][0] * r.x + P[2][1] * r.y + P[2][2] * r.z + P[2][3];
          V3 Ju = {(P[0][0] * wp - P[2][0] * up) / (wp * wp), (P[0][1] * wp - P[2][1] * up) / (wp * wp),
                   (P[0][2] * wp - P[2][2] * up) / (wp * wp)};
          V3 Jv = {(P[1][0] * wp - P[2][0] * vp) / (wp * wp), (P[1][1] * wp - P[2][1] * vp) / (wp * wp),
                   (P[1][2] * wp - P[2][2] * vp) / (wp * wp)};
          V3 q = wj * ((su * Ju) + (sv * Jv));
          V3 cq = cross(r - pose.t, q);
          acc[0] += q.x; acc[1] += q.y; acc[2] += q.z; acc[3] += cq.x; acc[4] += cq.y; acc[5] += cq.z;
        }
      }
      for (int k = 0; k < 6; ++k) slab[(size_t)iz * 6 + k] = acc[k];
    }
    double tot[6] = {0};
    for (int iz = 0; iz < g.nz; ++iz) for (int k = 0; k < 6; ++k) tot[k] += slab[(size_t)iz * 6 + k];
    const double* th = poses + 6 * v;
    double* out = grad + 6 * v;
    if (mode == 0) {
      V3 SA = {tot[0], tot[1], tot[2]}, SB = {tot[3], tot[4], tot[5]};
      V3 dt = mul(pose.R, SA);
      out[0] = -dt.x; out[1] = -dt.y; out[2] = -dt.z;
      V3 wx = {1, 0, 0};
      V3 wy = mulT(Rx(th[3]), V3{0, 1, 0});
      V3 wz = mulT(mul(Ry(th[4]), Rx(th[3])), V3{0, 0, 1});
      out[3] = -dot(wx, SB); out[4] = -dot(wy, SB); out[5] = -dot(wz, SB);
    } else {
      V3 Sq = {tot[0], tot[1], tot[2]}, Sc = {tot[3], tot[4], tot[5]};
      V3 ax = mul(pose.R, V3{1, 0, 0});
      V3 ay = mul(Rz(th[5]), V3{0, 1, 0});
      V3 az = {0, 0, 1};
      out[0] = Sq.x; out[1] = Sq.y; out[2] = Sq.z;
      out[3] = dot(ax, Sc); out[4] = dot(ay, Sc); out[5] = dot(az, Sc);
    }
  }
}

extern "C" {

int ora_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void ora_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

void ora_forward_f32(const ora_geom* g, int n_views, const double* angles, const double* poses, const float* vol,
                     double* proj, int64_t* ray_steps) {
  forward_impl<float>(*g, n_views, angles, poses, vol, proj, ray_steps);
}
void ora_forward_f64(const ora_geom* g, int n_views, const double* angles, const double* poses, const double* vol,
                     double* proj, int64_t* ray_steps) {
  forward_impl<double>(*g, n_views, angles, poses, vol, proj, ray_steps);
}
void ora_forward_T(const ora_geom* g, int n_views, const double* angles, const double* poses, const double* y,
                   double* vol_out) {
  forward_T_impl<double>(*g, n_views, angles, poses, y, vol_out);
}
void ora_forward_pose_grad_f32(const ora_geom* g, int n_views, const double* angles, const double* poses,
                               const float* vol, const float* upstream, double* grad, int lever_arm,
                               int grad_mode, int route) {
  forward_grad_impl<float>(*g, n_views, angles, poses, vol, upstream, grad, lever_arm, grad_mode, route);
}
void ora_forward_pose_grad_f64(const ora_geom* g, int n_views, const double* angles, const double* poses,
                               const double* vol, const float* upstream, double* grad, int lever_arm,
                               int grad_mode, int route) {
  forward_grad_impl<double>(*g, n_views, angles, poses, vol, upstream, grad, lever_arm, grad_mode, route);
}
void ora_backproject(const ora_geom* g, int n_views, const double* angles, const double* poses, const float* proj,
                     double* vol_out, int iz0, int iz1) {
  backproject_impl(*g, n_views, angles, poses, proj, vol_out, iz0, iz1);
}
void ora_backproject_T(const ora_geom* g, int n_views, const double* angles, const double* poses, const double* x,
                       double* proj_out) {
  backproject_T_impl(*g, n_views, angles, poses, x, proj_out);
}
void ora_backproject_pose_grad(const ora_geom* g, int n_views, const double* angles, const double* poses,
                               const float* proj, const float* upstream, double* grad, int grad_mode, int route) {
  backproject_grad_impl(*g, n_views, angles, poses, proj, upstream, grad, grad_mode, route);
}
// R(gamma) and dR/dgamma_k, exposed so the tests can pin them (finite differences, orthogonality).
void ora_rotation(const double* pose6, double* R9, double* dR27) {
  Pose p(pose6);
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    R9[i * 3 + j] = p.R.m[i][j];
    for (int k = 0; k < 3; ++k) dR27[k * 9 + i * 3 + j] = p.dR[k].m[i][j];
  }
}
// Projection matrix P (pixel-index units) of a view, exposed so the tests can pin Eq.1.
// `view`: one gantry angle, or (flags & 64) one 12-number view frame.
void ora_projection_matrix(const ora_geom* g, const double* view, double* P12) {
  View v(*g, view, 0);
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 4; ++j) P12[i * 4 + j] = v.P[i][j];
}

// O12: Siddon weights (forward, explicit transpose, pose gradient)
void ora_forward_siddon_f32(const ora_geom* g, int n_views, const double* angles, const double* poses,
                            const float* vol, double* proj) {
  forward_siddon_impl<float>(*g, n_views, angles, poses, vol, proj, nullptr, nullptr);
}
void ora_forward_siddon_f64(const ora_geom* g, int n_views, const double* angles, const double* poses,
                            const double* vol, double* proj) {
  forward_siddon_impl<double>(*g, n_views, angles, poses, vol, proj, nullptr, nullptr);
}
void ora_forward_siddon_T(const ora_geom* g, int n_views, const double* angles, const double* poses, const double* y,
                          double* vol_out) {
  forward_siddon_impl<double>(*g, n_views, angles, poses, (const double*)nullptr, nullptr, y, vol_out);
}
void ora_forward_pose_grad_siddon_f32(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                      const float* vol, const float* upstream, double* grad, int route) {
  forward_grad_siddon_impl<float>(*g, n_views, angles, poses, vol, upstream, grad, route);
}
void ora_forward_pose_grad_siddon_f64(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                      const double* vol, const float* upstream, double* grad, int route) {
  forward_grad_siddon_impl<double>(*g, n_views, angles, poses, vol, upstream, grad, route);
}

// O13: Joseph weights (forward, explicit transpose, pose gradient)
void ora_forward_joseph_f32(const ora_geom* g, int n_views, const double* angles, const double* poses,
                            const float* vol, double* proj) {
  forward_joseph_impl<float>(*g, n_views, angles, poses, vol, proj, nullptr, nullptr);
}
void ora_forward_joseph_f64(const ora_geom* g, int n_views, const double* angles, const double* poses,
                            const double* vol, double* proj) {
  forward_joseph_impl<double>(*g, n_views, angles, poses, vol, proj, nullptr, nullptr);
}
void ora_forward_joseph_T(const ora_geom* g, int n_views, const double* angles, const double* poses, const double* y,
                          double* vol_out) {
  forward_joseph_impl<double>(*g, n_views, angles, poses, (const double*)nullptr, nullptr, y, vol_out);
}
void ora_forward_pose_grad_joseph_f32(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                      const float* vol, const float* upstream, double* grad) {
  forward_grad_joseph_impl<float>(*g, n_views, angles, poses, vol, upstream, grad);
}
void ora_forward_pose_grad_joseph_f64(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                      const double* vol, const float* upstream, double* grad) {
  forward_grad_joseph_impl<double>(*g, n_views, angles, poses, vol, upstream, grad);
}

// O15: distance-driven pair (forward, back-projector = exact transpose, both pose gradients)
void ora_forward_dd_f32(const ora_geom* g, int n_views, const double* angles, const double* poses, const float* vol,
                        double* proj) {
  forward_dd_impl<float>(*g, n_views, angles, poses, vol, proj, nullptr, nullptr, 0, 0);
}
void ora_forward_dd_f64(const ora_geom* g, int n_views, const double* angles, const double* poses, const double* vol,
                        double* proj) {
  forward_dd_impl<double>(*g, n_views, angles, poses, vol, proj, nullptr, nullptr, 0, 0);
}
void ora_backproject_dd(const ora_geom* g, int n_views, const double* angles, const double* poses, const float* proj,
                        double* vol_out, int iz0, int iz1) {
  forward_dd_impl<float>(*g, n_views, angles, poses, (const float*)nullptr, nullptr, proj, vol_out, iz0, iz1);
}
void ora_forward_pose_grad_dd_f32(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                  const float* vol, const float* upstream, double* grad) {
  forward_grad_dd_impl<float>(*g, n_views, angles, poses, vol, upstream, grad);
}
void ora_forward_pose_grad_dd_f64(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                  const double* vol, const float* upstream, double* grad) {
  forward_grad_dd_impl<double>(*g, n_views, angles, poses, vol, upstream, grad);
}
void ora_backproject_pose_grad_dd(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                  const float* proj, const float* upstream, double* grad) {
  backproject_grad_dd_impl(*g, n_views, angles, poses, proj, upstream, grad);
}

// O16: separable-footprint pair (forward, back-projector = exact transpose, both pose gradients)
void ora_forward_sf_f32(const ora_geom* g, int n_views, const double* angles, const double* poses, const float* vol,
                        double* proj) {
  sf_project_impl<float>(*g, n_views, angles, poses, vol, proj, nullptr, nullptr, 0, 0);
}
void ora_forward_sf_f64(const ora_geom* g, int n_views, const double* angles, const double* poses, const double* vol,
                        double* proj) {
  sf_project_impl<double>(*g, n_views, angles, poses, vol, proj, nullptr, nullptr, 0, 0);
}
void ora_backproject_sf(const ora_geom* g, int n_views, const double* angles, const double* poses, const float* proj,
                        double* vol_out, int iz0, int iz1) {
  sf_project_impl<float>(*g, n_views, angles, poses, (const float*)nullptr, nullptr, proj, vol_out, iz0, iz1);
}
void ora_forward_pose_grad_sf_f32(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                  const float* vol, const float* upstream, double* grad) {
  sf_grad_impl<float>(*g, n_views, angles, poses, vol, upstream, nullptr, grad, 0);
}
void ora_forward_pose_grad_sf_f64(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                  const double* vol, const float* upstream, double* grad) {
  sf_grad_impl<double>(*g, n_views, angles, poses, vol, upstream, nullptr, grad, 0);
}
void ora_backproject_pose_grad_sf(const ora_geom* g, int n_views, const double* angles, const double* poses,
                                  const float* proj, const float* upstream, double* grad) {
  sf_grad_impl<float>(*g, n_views, angles, poses, (const float*)nullptr, proj, upstream, grad, 1);
}

}  // extern "C"
