// dfp_fwd_tma.cuh - a3 / a4 with the volume staged in shared memory by TMA (sm_100a).
//
// Same arithmetic per sample as fwd_project_kernel / fwd_grad_kernel (dfp_kernels.cuh), but the 8 (forward) or 32
// (gradient) voxel reads of a sample are LDS from a box of the volume that the block's pixel tile crosses during one
// CHUNK of consecutive samples:
//
//   * the block's rays share one kappa axis (sample k = kref + kappa, tau_k = (k + 1/2) D, fixed in the world:
//     DESIGN.md O6), so a chunk [kappa0, kappa0 + Kc) is a slab of the frustum; its bounding box in voxel
//     indices is found from the tile's four corner rays (positions are convex in the pixel index up to the
//     sagitta of the sphere |r - s| = tau, < 0.01 voxel for a 16-pixel tile; kBoxMargin covers it);
//   * one elected thread issues `cp.async.bulk.tensor.3d` (TMA, SASS UTMALDG) for the chunk's box (BoxShape)
//     straight from the caller's volume: out-of-range elements are ZERO-FILLED by the TMA unit, which is the
//     zero extension of f~ (U7) - no padded / packed copy of the volume is made on this path;
//   * one or two stages (BoxShape), mbarrier (complete_tx) as the "full" signal, __syncthreads as the "empty" one;
//   * the box origin is rounded down to a multiple of 4 floats along x (TMA: 16-byte inner alignment);
//   * Kc is chosen per block so that the box always fits (oblique tiles get shorter chunks);
//   * positions are BOX-LOCAL: every thread keeps its ray in fp64 (Ray) and, once per chunk, re-bases it onto the
//     box origin, so the fp32 position of a sample is a number in [0, 28) with ~1e-6 voxel of error whatever the
//     size of the volume; the shared-memory word index is X + BX*Y + BX*BY*Z of the magic-rounded local position;
//   * gradient: several lanes per ray (interleaved samples) and packed fp32x2 arithmetic (FFMA2 / FADD2);
//   * exact-interpolant mode: a sample within fp32 rounding of a cell face takes cell and fractions from fp64.
// PAPER.md Eq.18 :172-177 (forward), Eq.7-8 :101-113, Eq.19-20 :179-191 (gradient), :207 (on the fly, weights once).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "dfp_kernels.cuh"

namespace dfp {

// Staging boxes (floats).  The x extent times 4 bytes must be a multiple of 16 (TMA inner box).  Bank of a voxel =
// (x + X*y + X*Y*z) mod 32: only x reaches the two low bank bits (rows are 16-byte aligned), so a warp-wide load is
// conflict-free only if the warp's voxels spread along x as well as across (y, z) - DESIGN.md "Kernels", and the
// simulation / measurements quoted there.
// The host picks, per call, the first shape of the op's list that every view's tiles fit with chunks of >= kMinChunk
// samples:
//   shape 0  20 x 20 x 16, two stages : forward, clinical magnification and small pose angles (C2)
//   shape 1  28 x 20 x 20, two stages : forward, wider tiles / larger tilts
//   shape 2  28 x 28 x 20, one stage  : forward fallback before the gather path; gradient fallback
//   shape 3  28 x 28 x 16, one stage  : gradient kernels, 16 x 8-pixel tiles (the stencil needs 2 more cells per axis and
//            a chunk lasts 4x longer than the forward's, so one stage and four blocks per SM hide the TMA latency;
//            long enough along x and y that views at 45 degrees in the xy plane still get ~10-sample chunks) - taken
//            where a view's tiles do not fit shape 7
//   shape 4  20 x 19 x 16, two stages / shape 5  28 x 19 x 20, one stage : forward at >= 0.45 voxel per pixel (C4 / C5)
//   shape 6  28 x 27 x 14, one stage  : gradient, views along one in-plane axis (MODE 5 / 6), five blocks per SM
//   shape 7  28 x 28 x 14, one stage  : gradient kernels (all modes), five blocks per SM - the first choice
template <int SHAPE> struct BoxShape;
template <> struct BoxShape<0> { static constexpr int X = 20, Y = 20, Z = 16, STAGES = 2; };
template <> struct BoxShape<1> { static constexpr int X = 28, Y = 20, Z = 20, STAGES = 2; };
template <> struct BoxShape<2> { static constexpr int X = 28, Y = 28, Z = 20, STAGES = 1; };
#ifndef DFP_GRAD_STAGES
#define DFP_GRAD_STAGES 1
#endif
#ifndef DFP_GRAD_SLOTS
#define DFP_GRAD_SLOTS 2
#endif
#ifndef DFP_GRAD_TV
#define DFP_GRAD_TV 8
#endif
template <> struct BoxShape<3> { static constexpr int X = 28, Y = 28, Z = 16, STAGES = DFP_GRAD_STAGES; };   // gradient, 16 x 8 tiles
// Forward boxes with an ODD y extent (slab pitch = 12 / 20 mod 32 instead of 16): where a warp's 8 x 4-pixel patch spans
// three z slices (>= 0.45 voxel per pixel: the 512^3 configs), slab pitch 16 puts slices z and z + 2 on the same banks;
// 1.76 -> 1.38 wavefronts per load on C5, 1.62 -> 1.36 on C4 (simulated, _and measured_ in DESIGN.md); at C2's 0.39
// voxel per pixel the even extents are the better ones (1.37 against 1.64).
template <> struct BoxShape<4> { static constexpr int X = 20, Y = 19, Z = 16, STAGES = 2; };
#ifndef DFP_S5_STAGES
#define DFP_S5_STAGES 1          // one stage, four blocks per SM: 305 ms against 322 with two stages / two blocks (C5)
#endif
#ifndef DFP_S5_Z
#define DFP_S5_Z 20
#endif
template <> struct BoxShape<5> { static constexpr int X = 28, Y = 19, Z = DFP_S5_Z, STAGES = DFP_S5_STAGES; };
// The gradient kernels of the >= 0.45-voxel-per-pixel configs run FIVE blocks per SM: 14 slices instead of 16 keep a
// box under 44 KB (an 8-pixel-high tile spans ~5 voxels along z there: chunks stay ~20 samples long) and the kernels
// are compiled for 48 registers (13 values of the per-chunk set-up spill; the sample loop does not): 826 -> 810 ms on C5.
#ifndef DFP_S6_Z
#define DFP_S6_Z 14
#endif
#ifndef DFP_CLS_MINB
#define DFP_CLS_MINB 5
#endif
template <> struct BoxShape<6> { static constexpr int X = 28, Y = 27, Z = DFP_S6_Z, STAGES = 1; };   // MODE 5 / 6 (above)
template <> struct BoxShape<7> { static constexpr int X = 28, Y = 28, Z = DFP_S6_Z, STAGES = 1; };   // MODE 1, views near the diagonals
constexpr int kNumShapes = 8;
// words between the stages of a box: the box rounded up to 128 bytes (alignment of a TMA destination)
template <int SHAPE> __host__ __device__ constexpr int tma_stage_words() {
  return (BoxShape<SHAPE>::X * BoxShape<SHAPE>::Y * BoxShape<SHAPE>::Z + 31) / 32 * 32;
}
template <int SHAPE> constexpr int tma_smem_bytes() { return tma_stage_words<SHAPE>() * 4 * BoxShape<SHAPE>::STAGES; }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
// lerp on two lanes of data at once: v0 + a (v1 - v0), rounded exactly like lerp()
__device__ __forceinline__ float2 lerp2(float2 a, float2 v0, float2 v1) { return __ffma2_rn(a, sub2(v1, v0), v0); }

// Lane mapping.  A ray is marched by SLOTS lanes (lane `slot` takes the samples kappa = slot mod SLOTS); a warp covers
// PU x PV pixels x SLOTS consecutive samples, so that the 32 lanes of a warp-wide LDS touch voxels spread over SLOTS
// depth steps as well as the pixel patch.  Block = TU x TV pixels x SLOTS.
// GRAD: 0 forward projection (one lane per ray, 8 x 4-pixel warps, 16 x 16-pixel tile: the kernel is issue-bound and
// a second lane per ray doubles the per-ray set-up), 1 gradient with central differences of f~ (the paper's,
// DESIGN.md O3), 2 gradient with the exact derivative of the trilinear interpolant (DFP_FLAG_GRAD_INTERP: the same 8
// voxels as the forward), 3 FUSED projection + central-difference gradient moments in one traversal
// (dfp_forward_fused_moments).  Gradient kernels: two lanes per ray, 8 x 2-pixel warps, 16 x 8-pixel tile.
// MODE 4 = GRAD 0 on a 16 x 8-pixel tile (128 threads): the forward projector's last resort before the gather kernels,
// for coarse pixels on fine voxels (C1's forward call, 1.2 voxels per pixel: a 16 x 16 tile's frustum holds no box).
// MODE 5 / 6 = GRAD 1 for views whose rays run along ONE in-plane axis, at >= 0.45 voxel per pixel (the 512^3 configs).
// There a warp of 8 x 2 pixels x 2 samples holds ~5 voxels across the rays, 2 along z and only 2 along the rays: when
// the rays run along x, only two x values reach the low bank bits and 15-20 distinct words share 16 banks (1.38
// wavefronts per load whatever the pitches); a warp of 4 x 4 pixels x 2 samples on a box with an ODD y extent (slab pitch
// = 20 mod 32) measures 1.10 when the rays run along y.  MODE 5 is that kernel for the views along y; MODE 6 is the same
// kernel on the TRANSPOSED volume ([z][x][y], x and y of the ray swapped on entry, of the sums on exit) for the views along
// x; views near the diagonals keep MODE 1 (1.10 as it is).  C5: 188 -> 218 Gray-steps/s on the axis-aligned views.
__host__ __device__ constexpr int tma_grad_of(int MODE) { return MODE == 4 ? 0 : (MODE >= 5 ? 1 : MODE); }
template <int MODE> struct TmaLanes {
  static constexpr int GRAD = tma_grad_of(MODE);
  static constexpr int SLOTS = GRAD ? DFP_GRAD_SLOTS : 1, TU = kFwdTU,
                       TV = MODE == 0 ? kFwdTV : (MODE == 4 ? 8 : DFP_GRAD_TV), THREADS = TU * TV * SLOTS;
  static constexpr int PU = SLOTS == 4 ? 4 : (MODE >= 5 ? 4 : 8), PV = 32 / (PU * SLOTS);
#ifndef DFP_FWD_MINB
#define DFP_FWD_MINB 4
#endif
  static constexpr int MINB = THREADS > 256 ? 2 : (MODE == 0 ? DFP_FWD_MINB : 4);
};
template <int MODE, int SHAPE> __host__ __device__ constexpr int tma_min_blocks() {
  return (SHAPE == 6 || SHAPE == 7) ? DFP_CLS_MINB : TmaLanes<MODE>::MINB;
}
template <int MODE>
__device__ __forceinline__ void tma_pixel(int bx, int by, int& iu, int& iv, int& slot) {
  using T = TmaLanes<MODE>;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int WU = T::TU / T::PU;                     // warps across u
  const int pix = lane % (T::PU * T::PV);
  slot = lane / (T::PU * T::PV);
  iu = bx * T::TU + (warp % WU) * T::PU + (pix % T::PU);
  iv = by * T::TV + (warp / WU) * T::PV + (pix / T::PU);
}
#ifndef DFP_FWD_UNROLL
#define DFP_FWD_UNROLL 0         // unroll factor of the forward kernels' sample loop (0: per box shape, see tma_march)
#endif
#ifndef DFP_ORIGIN_PRE
#define DFP_ORIGIN_PRE 2         // bit 0: forward, bit 1: gradient kernels take the next box origin before the barrier
#endif
constexpr int kMaxStages = 2;
constexpr float kBoxMargin = 0.05f;                    // voxels: sagitta of the tile + fp32 rounding
constexpr int kBoxAlignLoss = 3;                       // x cells lost to the 16-byte alignment of the box origin
// Blocks are ordered so that the views of a GROUP of kViewGroup consecutive views run tile by tile, view fastest:
// the blocks resident at one time then cover a few dozen neighbouring tiles of a few neighbouring views, whose frusta
// overlap in the volume - a 512^3 volume (4x the L2) is then pulled from HBM about once per group instead of once
// per view.
#ifndef DFP_VIEW_GROUP
#define DFP_VIEW_GROUP 8
#endif
constexpr int kViewGroup = DFP_VIEW_GROUP;

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap* map, int x, int y, int z, unsigned bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"(reinterpret_cast<unsigned long long>(map)), "r"(x), "r"(y), "r"(z), "r"(bar)
      : "memory");
}

struct TmaBlock {              // block-wide state in shared memory
  float pm[4][3], dp[4][3];    // the tile's corner rays (centred-index coordinates, as in struct Ray, rounded to fp32)
  int kA, kB;                  // union of the live rays' kappa ranges [kA, kB)
  int Kc;                      // samples per chunk (0: nothing to do, -1: the box cannot hold the tile)
  int org[kMaxStages][3];      // per stage: centred index of the box's first cell (the origin of the local positions)
  double orgd[kMaxStages][3];  // the same minus 1/2, as doubles: Ray::pm (position - 1/2) minus it = local position
};

// One chunk's box: centred index of its first cell along each axis, from the tile's four corner rays at the chunk's
// first and last sample.  Called by ALL 32 LANES of a warp (lane -> axis, corner ray, end of the chunk; shuffles for the
// minimum): the origin of the next chunk is then ready in lane 0's registers BEFORE the block's "empty" barrier, and
// the serial section between the barrier and the TMA issue shrinks to the six stores and the issue itself.
template <int MODE, int SHAPE>
__device__ __forceinline__ void chunk_origin(const VolLayout& L, const TmaBlock& B, int chunk, int* oc) {
  constexpr int GRAD = tma_grad_of(MODE);
  const int lane = threadIdx.x & 31;
  const int a = min(lane >> 3, 2), r = (lane >> 1) & 3;
  const int k0 = B.kA + chunk * B.Kc;
  const int k1 = min(k0 + B.Kc, B.kB) - 1;
  float lo = fmaf((float)((lane & 1) ? k1 : k0), B.dp[r][a], B.pm[r][a]);
#pragma unroll
  for (int o = 1; o < 8; o <<= 1) lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o));
  const int o_ = (int)floorf(lo - 0.5f - kBoxMargin) - (GRAD ? 1 : 0);      // centred index of the box's first cell
  oc[0] = __shfl_sync(0xffffffffu, o_, 0);
  oc[1] = __shfl_sync(0xffffffffu, o_, 8);
  oc[2] = __shfl_sync(0xffffffffu, o_, 16);
  // the TMA unit wants the innermost coordinate on a 16-byte boundary (measured on B200: an x origin that is
  // not a multiple of 4 floats raises an illegal-instruction fault): round the x origin down, kBoxAlignLoss
  oc[0] = (((oc[0] + L.hx) >> 2) << 2) - L.hx;
}
// The same by ONE thread (forward kernels: after the barrier, measured faster there than the warp-wide version).
template <int MODE, int SHAPE>
__device__ __forceinline__ void chunk_origin_serial(const VolLayout& L, const TmaBlock& B, int chunk, int* oc) {
  constexpr int GRAD = tma_grad_of(MODE);
  const int k0 = B.kA + chunk * B.Kc;
  const int k1 = min(k0 + B.Kc, B.kB) - 1;
  const float f0 = (float)k0, f1 = (float)k1;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    float lo = 3.0e38f;
#pragma unroll
    for (int r = 0; r < 4; ++r) lo = fminf(lo, fminf(fmaf(f0, B.dp[r][a], B.pm[r][a]), fmaf(f1, B.dp[r][a], B.pm[r][a])));
    oc[a] = (int)floorf(lo - 0.5f - kBoxMargin) - (GRAD ? 1 : 0);
  }
  oc[0] = (((oc[0] + L.hx) >> 2) << 2) - L.hx;
}
// One thread: publish the origin of the stage the chunk lands in and issue its TMA load.
template <int SHAPE>
__device__ __forceinline__ void issue_chunk(const VolLayout& L, TmaBlock& B, const CUtensorMap* map, int chunk,
                                            const int* oc, unsigned tiles_addr, unsigned bar_addr) {
  using S = BoxShape<SHAPE>;
  constexpr int kWords = S::X * S::Y * S::Z;
  const int s = chunk % S::STAGES;
  B.org[s][0] = oc[0]; B.org[s][1] = oc[1]; B.org[s][2] = oc[2];
  B.orgd[s][0] = (double)oc[0] - 0.5; B.orgd[s][1] = (double)oc[1] - 0.5; B.orgd[s][2] = (double)oc[2] - 0.5;
  const unsigned bar = bar_addr + 8u * s;
  mbar_expect_tx(bar, kWords * 4);
  tma_load_3d(tiles_addr + (unsigned)(s * tma_stage_words<SHAPE>() * 4), map, oc[0] + L.hx, oc[1] + L.hy, oc[2] + L.hz, bar);
}

// The chunk loop of one block for one box shape.  acc = {sum} (forward) or {gx,gy,gz,hx,hy,hz[,sum]} (gradient).
template <int MODE, int SHAPE>
__device__ __forceinline__ void tma_march(const VolLayout& L, const CUtensorMap* map, const Ray& r, int slot,
                                          TmaBlock& B, const float* tiles, unsigned tiles_addr, unsigned bar_addr,
                                          float* acc) {
  using S = BoxShape<SHAPE>;
  constexpr int GRAD = tma_grad_of(MODE);
  constexpr int BX = S::X, BXY = S::X * S::Y, kBox = S::X * S::Y * S::Z, kWords = tma_stage_words<SHAPE>();
  constexpr int SLOTS = TmaLanes<MODE>::SLOTS;
  if (threadIdx.x == 0) {
    int Kc = 0;
    if (B.kA < B.kB) {
      // chunk length: extent_a <= span_a + (Kc - 1) slope_a must leave room for the floor / stencil cells
      const float fa = (float)B.kA, fb = (float)(B.kB - 1);
      const int box[3] = {S::X, S::Y, S::Z};
      Kc = 4096;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        float lo0 = 3e38f, hi0 = -3e38f, lo1 = 3e38f, hi1 = -3e38f, slope = 0.f;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const float q0 = fmaf(fa, B.dp[c][a], B.pm[c][a]), q1 = fmaf(fb, B.dp[c][a], B.pm[c][a]);
          lo0 = fminf(lo0, q0); hi0 = fmaxf(hi0, q0);
          lo1 = fminf(lo1, q1); hi1 = fmaxf(hi1, q1);
          slope = fmaxf(slope, fabsf(B.dp[c][a]));
        }
        const float span = fmaxf(hi0 - lo0, hi1 - lo1);
        const float avail =
            (float)(box[a] - 4 - (GRAD ? 2 : 0) - (a == 0 ? kBoxAlignLoss : 0)) - 2.f * kBoxMargin - span;
        if (avail < 0.f) Kc = -1;
        else if (Kc > 0 && slope > 1e-7f) Kc = min(Kc, (int)floorf(avail / slope) + 1);
      }
    }
    B.Kc = Kc;
    if (Kc > 0) {
      const int n_chunks = (B.kB - B.kA + Kc - 1) / Kc;
#pragma unroll
      for (int c = 0; c < S::STAGES; ++c)
        if (c < n_chunks) {
          int oc[3];
          chunk_origin_serial<MODE, SHAPE>(L, B, c, oc);
          issue_chunk<SHAPE>(L, B, map, c, oc, tiles_addr, bar_addr);
        }
    }
  }
  __syncthreads();
  const int Kc = B.Kc, kA = B.kA, kB = B.kB;
  const int n_chunks = Kc > 0 ? (kB - kA + Kc - 1) / Kc : 0;
  const bool warp0 = threadIdx.x < 32;
  const int kend = r.k0 + r.n;
  const float dpx = (float)r.dp[0], dpy = (float)r.dp[1], dpz = (float)r.dp[2];
  const float2 dpxy = make_float2(dpx, dpy);
  // The fp64 ray is touched once per chunk (and in the rare exact-cell path): it is parked in LOCAL memory - an array
  // read through an index the compiler cannot see through - so that its 12 registers stay free for the sample loop
  // (with them live the loop lost 10-20 %: fewer loads in flight at the 64-register budget of four blocks per SM).
  double rd[6];
#pragma unroll
  for (int a = 0; a < 3; ++a) { rd[a] = r.pm[a]; rd[3 + a] = r.dp[a]; }
  int zi;
  asm volatile("mov.u32 %0, 0;" : "=r"(zi));

  float sum = 0.f;
  float gx = 0.f, gy = 0.f, gz = 0.f, hx = 0.f, hy = 0.f, hz = 0.f;
  for (int chunk = 0; chunk < n_chunks; ++chunk) {
    const int s = chunk % S::STAGES;
    const int c_lo = kA + chunk * Kc;
    const int ka = max(c_lo, r.k0), kb = min(min(c_lo + Kc, kB), kend);
    // this lane takes the samples of its ray whose kappa is congruent to its slot (the other slots take the rest)
    const int kfirst = SLOTS == 1 ? ka : ka + ((slot - ka) & (SLOTS - 1));
    // re-base the ray onto the box origin (fp64, once per chunk): position of this lane's first sample - fetched from
    // local memory and advanced BEFORE the wait for the box, so that the loads' latency overlaps it
    const double kd = (double)kfirst;
    const double p0 = fma(kd, rd[zi + 3], rd[zi + 0]), p1 = fma(kd, rd[zi + 4], rd[zi + 1]),
                 p2 = fma(kd, rd[zi + 5], rd[zi + 2]);
    mbar_wait(bar_addr + 8u * s, (unsigned)(chunk / S::STAGES) & 1u);
    // (B.orgd holds the origin minus 1/2: Ray::pm is the position minus 1/2, the local position below is the position)
    const float2 bxy = make_float2((float)(p0 - B.orgd[s][0]), (float)(p1 - B.orgd[s][1]));
    const float bz = (float)(p2 - B.orgd[s][2]);
    // BYTE offset of local cell (X, Y, Z) in stage s from the magic-rounded floats' bits
    unsigned c0 = 4u * ((unsigned)(s * kWords) - (unsigned)kMagicBits * (unsigned)(1 + BX + BXY));
    // keep the constant out of the optimiser's sight: folded into every load's offset it no longer fits the LDS
    // immediate field and each of the 8 / 32 loads of a sample gets its own address add (measured: +20 % time)
    asm volatile("" : "+r"(c0));
    float kf = (float)kfirst, jf = 0.f;
    // forward kernels: the sample loop unrolled by 2 (loop overhead, two samples' loads in flight: C2 7.15 -> 6.70 ms,
    // C4 370 -> 349 ms), by 4 on C5's single-stage box (288 -> 283 ms; by 2 it gains nothing there); the gradient
    // kernels are bound by the shared-memory pipe and keep the plain loop
    constexpr int kUnroll = GRAD != 0 ? 1 : (DFP_FWD_UNROLL ? DFP_FWD_UNROLL : (SHAPE == 5 ? 4 : 2));
#pragma unroll kUnroll
    for (int k = kfirst; k < kb; k += SLOTS) {
      // position, floor and fractions: x and y as one fp32x2 lane pair
      const float2 q2 = __ffma2_rn(make_float2(jf, jf), dpxy, bxy);
      const float qz = fmaf(jf, dpz, bz);
      // floor by the magic add ROUNDED DOWN (t = kMagic + floor(q) exactly), fraction = q - floor(q)
      const float2 t2 = __fadd2_rd(q2, make_float2(kMagic, kMagic));
      const float tz = __fadd_rd(qz, kMagic);
      const float2 a2 = sub2(q2, __fadd2_rn(t2, make_float2(-kMagic, -kMagic)));
      float ax = a2.x, ay = a2.y, az = qz - (tz - kMagic);
      unsigned off = 4u * (unsigned)__float_as_int(t2.x) + (unsigned)(4 * BX) * (unsigned)__float_as_int(t2.y) +
                     (unsigned)(4 * BXY) * (unsigned)__float_as_int(tz) + c0;
      if (GRAD == 2) {
        // the derivative of the interpolant jumps at cell faces: a sample within fp32 rounding of one takes its
        // cell (and fractions) from the fp64 position, as the oracle does
        const float mn = fminf(fminf(fminf(ax, 1.f - ax), fminf(ay, 1.f - ay)), fminf(az, 1.f - az));
        if (mn < kFaceEps) {
          int cell[3];
          float fr[3];
          Ray rr;
#pragma unroll
          for (int a = 0; a < 3; ++a) { rr.pm[a] = rd[zi + a]; rr.dp[a] = rd[zi + 3 + a]; }
          exact_cell(rr, k, cell, fr);
          off = 4u * (unsigned)(s * kWords + (cell[0] - B.org[s][0]) + BX * (cell[1] - B.org[s][1]) + BXY * (cell[2] - B.org[s][2]));
          ax = fr[0]; ay = fr[1]; az = fr[2];
        }
      }
      const float* c = reinterpret_cast<const float*>(reinterpret_cast<const char*>(tiles) + off);
#ifdef DFP_CHECK_BOUNDS   // debug build: every LDS of the sample must fall inside the stage's box (else NaN out)
      {
        const int local = (int)(off / 4u - (unsigned)(s * kWords)), halo = (GRAD == 1 || GRAD == 3) ? 1 : 0;
        const int lo = local - halo * (1 + BX + BXY), hi = local + (1 + halo) * (1 + BX + BXY);
        if (lo < 0 || hi >= kBox) sum = gx = __int_as_float(0x7fc00000);
      }
#endif
      if (!GRAD) {
        // pairs over the two z slices: (r00, r01), (r10, r11), then the y lerp on the pair, the z lerp scalar
        const float2 ax2 = make_float2(ax, ax);
        const float2 rA = lerp2(ax2, make_float2(c[0], c[BXY]), make_float2(c[1], c[BXY + 1]));
        const float2 rB = lerp2(ax2, make_float2(c[BX], c[BXY + BX]), make_float2(c[BX + 1], c[BXY + BX + 1]));
        const float2 ry = lerp2(make_float2(ay, ay), rA, rB);
        sum += lerp(az, ry.x, ry.y);
      } else {
        float ddx, ddy, ddz;
        if (GRAD == 2) {
          // exact gradient of the trilinear interpolant in the sample's cell (per voxel index; G.sg* = 1 / pitch):
          // pairs over the two z slices, as in the forward kernel
          const float2 ax2 = make_float2(ax, ax), ay2 = make_float2(ay, ay);
          const float2 v00 = make_float2(c[0], c[BXY]), v10 = make_float2(c[1], c[BXY + 1]);                      // row y
          const float2 v01 = make_float2(c[BX], c[BXY + BX]), v11 = make_float2(c[BX + 1], c[BXY + BX + 1]);      // row y+1
          const float2 d0 = sub2(v10, v00), d1 = sub2(v11, v01);          // x differences of rows y, y+1
          const float2 rA = __ffma2_rn(ax2, d0, v00), rB = __ffma2_rn(ax2, d1, v01);   // (r00, r01), (r10, r11)
          const float2 dx2 = lerp2(ay2, d0, d1);
          ddx = lerp(az, dx2.x, dx2.y);
          const float2 dy2 = sub2(rB, rA);
          ddy = lerp(az, dy2.x, dy2.y);
          const float2 ry = lerp2(ay2, rA, rB);
          ddz = ry.y - ry.x;
        } else {
        // Packed fp32x2 arithmetic (sm_100 FADD2 / FFMA2: two IEEE-rounded fp32 results per issue slot, the same
        // bits as the scalar code of fwd_grad_kernel).  Pairs run over the two z slices kk = 0, 1 of a row (y + j).
        const float2 ax2 = make_float2(ax, ax), ay2 = make_float2(ay, ay);
        float2 rv2[2], rdx2[2];          // rv2[j] = (rv[j][0], rv[j][1]), likewise rdx2
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const float* r0 = c + j * BX;
          const float* r1 = c + BXY + j * BX;
          const float2 m1 = make_float2(r0[-1], r1[-1]), v0 = make_float2(r0[0], r1[0]);
          const float2 v1 = make_float2(r0[1], r1[1]), v2 = make_float2(r0[2], r1[2]);
          rv2[j] = lerp2(ax2, v0, v1);
          rdx2[j] = lerp2(ax2, sub2(v1, m1), sub2(v2, v0));
        }
        float2 rym2, ryp2;               // ring rows in y: (y-1, z+kk), (y+2, z+kk), paired over kk
        {
          const float* m0 = c - BX;
          const float* m1 = c + BXY - BX;
          const float* p0 = c + 2 * BX;
          const float* p1 = c + BXY + 2 * BX;
          rym2 = lerp2(ax2, make_float2(m0[0], m1[0]), make_float2(m0[1], m1[1]));
          ryp2 = lerp2(ax2, make_float2(p0[0], p1[0]), make_float2(p0[1], p1[1]));
        }
        float2 rzm2, rzp2;               // ring rows in z: (y+j, z-1), (y+j, z+2), paired over j
        {
          const float* m0 = c - BXY;
          const float* m1 = c + BX - BXY;
          const float* p0 = c + 2 * BXY;
          const float* p1 = c + BX + 2 * BXY;
          rzm2 = lerp2(ax2, make_float2(m0[0], m1[0]), make_float2(m0[1], m1[1]));
          rzp2 = lerp2(ax2, make_float2(p0[0], p1[0]), make_float2(p0[1], p1[1]));
        }
        const float2 dx2 = lerp2(ay2, rdx2[0], rdx2[1]);                           // pair over kk
        ddx = lerp(az, dx2.x, dx2.y);
        const float2 dy2 = lerp2(ay2, sub2(rv2[1], rym2), sub2(ryp2, rv2[0]));     // (dy0, dy1)
        ddy = lerp(az, dy2.x, dy2.y);
        // d/dz pairs over j: (rv[0][1], rv[1][1]) - rzm2, rzp2 - (rv[0][0], rv[1][0])
        const float2 az2 = make_float2(az, az);
        const float2 dz2 = lerp2(az2, sub2(make_float2(rv2[0].y, rv2[1].y), rzm2),
                                 sub2(rzp2, make_float2(rv2[0].x, rv2[1].x)));     // (dz0, dz1)
        ddz = lerp(ay, dz2.x, dz2.y);
        if (GRAD == 3) {                 // fused: the projection itself, from the core rows already interpolated in x
          const float2 ry = lerp2(ay2, rv2[0], rv2[1]);
          sum += lerp(az, ry.x, ry.y);
        }
        }
        gx += ddx; gy += ddy; gz += ddz;
        hx = fmaf(kf, ddx, hx); hy = fmaf(kf, ddy, hy); hz = fmaf(kf, ddz, hz);
      }
      kf += (float)SLOTS;
      jf += (float)SLOTS;
    }
    // The origin of the chunk that will reuse this stage.  Gradient kernels: warp 0 works it out BEFORE it joins the
    // barrier (the serial section after the barrier is then the six stores and the issue: C5 903 -> 893 ms); forward
    // kernels: thread 0, after the barrier (a chunk is 4x shorter there, and 20 more instructions in one warp ahead of
    // the barrier hold up the other seven: 305 against 295 ms).
    constexpr bool kPre = (DFP_ORIGIN_PRE >> (GRAD ? 1 : 0)) & 1;
    int oc[3] = {0, 0, 0};
    const bool more = chunk + S::STAGES < n_chunks;
    if (kPre && warp0 && more) chunk_origin<MODE, SHAPE>(L, B, chunk + S::STAGES, oc);
    __syncthreads();                                   // every thread is done with stage s ("empty")
    if (threadIdx.x == 0 && more) {
      if (!kPre) chunk_origin_serial<MODE, SHAPE>(L, B, chunk + S::STAGES, oc);
      issue_chunk<SHAPE>(L, B, map, chunk + S::STAGES, oc, tiles_addr, bar_addr);
    }
  }
  if (!GRAD) {
    acc[0] = sum;
  } else {
    acc[0] = gx; acc[1] = gy; acc[2] = gz; acc[3] = hx; acc[4] = hy; acc[5] = hz;
    if (GRAD == 3) acc[6] = sum;
  }
}

// Grid: one block per (view, pixel tile), 1-D, ordered group of views -> tile -> view within the group (kViewGroup).
struct FwdGrid {
  int n_views, gx, gy;         // views of this launch; tiles per view along u and v
  int n_total;                 // views of the call (layout of the partials)
  const int* ids;              // view index of each of the launch's views, or nullptr: the views 0 .. n_views - 1
};
__device__ __forceinline__ void fwd_block(const FwdGrid& Q, int& view, int& bx, int& by) {
  const unsigned nb = (unsigned)Q.gx * (unsigned)Q.gy, per = (unsigned)kViewGroup * nb;
  const unsigned b = blockIdx.x, grp = b / per, r = b - grp * per;
  const unsigned gsz = min((unsigned)kViewGroup, (unsigned)Q.n_views - grp * kViewGroup);
  const unsigned tile = r / gsz, vg = r - tile * gsz;
  view = (int)(grp * kViewGroup + vg);
  if (Q.ids) view = __ldg(Q.ids + view);
  by = (int)(tile / (unsigned)Q.gx);
  bx = (int)(tile - (unsigned)by * (unsigned)Q.gx);
}

template <int MODE, int SHAPE>
__global__ void __launch_bounds__(TmaLanes<MODE>::THREADS, tma_min_blocks<MODE, SHAPE>()) fwd_tma_kernel(FwdGeom G, FwdGrid Q,
                                                              const FwdView* __restrict__ views,
                                                              const __grid_constant__ CUtensorMap vol_map,
                                                              const float* __restrict__ upstream,
                                                              float* __restrict__ out,
                                                              float* __restrict__ proj_out) {
  constexpr int GRAD = tma_grad_of(MODE);
  constexpr int NSET = GRAD == 3 ? 3 : 1;              // weight sets of the per-view reduction (fused: 1, l, b)
  constexpr int SLOTS = TmaLanes<MODE>::SLOTS;
  extern __shared__ __align__(128) float tiles[];      // STAGES boxes
  __shared__ __align__(8) unsigned long long full_bar[kMaxStages];
  __shared__ TmaBlock B;
  __shared__ float red[TmaLanes<MODE>::THREADS / 32][6 * NSET];

  int view, bx, by, iu, iv, slot;
  fwd_block(Q, view, bx, by);
  tma_pixel<MODE>(bx, by, iu, iv, slot);
  const bool live = iu < G.nu && iv < G.nv;
  const unsigned tiles_addr = smem_u32(tiles), bar_addr = smem_u32(full_bar);

  float ex = 0.f, ey = 0.f, ez = 0.f, px = 0.f, py = 0.f, pz = 0.f;    // ray direction, reference sample (mm)
  Ray r;
  {
    double e_mm[3], ref_mm[3];
    r = setup_ray(G, views[view], iu, iv, GRAD ? e_mm : nullptr, GRAD ? ref_mm : nullptr);
    if (GRAD) {
      ex = (float)e_mm[0]; ey = (float)e_mm[1]; ez = (float)e_mm[2];
      px = (float)ref_mm[0]; py = (float)ref_mm[1]; pz = (float)ref_mm[2];
    }
  }
  if (!live) r.n = 0;
  VolLayout L = G.L;
  if (MODE == 6) {             // the transposed volume: the ray in (y, x, z)
    double sw = r.pm[0]; r.pm[0] = r.pm[1]; r.pm[1] = sw;
    sw = r.dp[0]; r.dp[0] = r.dp[1]; r.dp[1] = sw;
    const int h = L.hx; L.hx = L.hy; L.hy = h;
  }

  if (threadIdx.x == 0) {
    B.kA = 0x7fffffff;
    B.kB = -0x7fffffff;
#pragma unroll
    for (int s = 0; s < kMaxStages; ++s) mbar_init(bar_addr + 8u * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  {  // corner rays of the tile: pixels (0,0), (TU-1,0), (0,TV-1), (TU-1,TV-1) of the block
    constexpr int TU = TmaLanes<MODE>::TU, TV = TmaLanes<MODE>::TV;
    const int cu = iu - bx * TU, cv = iv - by * TV;
    if (slot == 0 && (cu == 0 || cu == TU - 1) && (cv == 0 || cv == TV - 1)) {
      const int c = (cu ? 1 : 0) + (cv ? 2 : 0);
#pragma unroll
      for (int a = 0; a < 3; ++a) { B.pm[c][a] = (float)r.pm[a]; B.dp[c][a] = (float)r.dp[a]; }
    }
  }
  __syncthreads();
  {  // union of the live kappa ranges
    int lo = r.n > 0 ? r.k0 : 0x7fffffff, hi = r.n > 0 ? r.k0 + r.n : -0x7fffffff;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
      hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if ((threadIdx.x & 31) == 0 && lo < hi) {
      atomicMin(&B.kA, lo);
      atomicMax(&B.kB, hi);
    }
  }
  __syncthreads();
  float acc[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  tma_march<MODE, SHAPE>(L, &vol_map, r, slot, B, tiles, tiles_addr, bar_addr, acc);
  if (MODE == 6) {             // back to (x, y, z): the sums of d/dx and d/dy
    float sw = acc[0]; acc[0] = acc[1]; acc[1] = sw;
    sw = acc[3]; acc[3] = acc[4]; acc[4] = sw;
  }
  // the slots of a ray: partial sums over the samples each lane took (slot = lane / (PU * PV): the high lane bits)
  if (SLOTS > 1) {
#pragma unroll
    for (int q = 0; q < (GRAD == 3 ? 7 : GRAD ? 6 : 1); ++q) {
#pragma unroll
      for (int o = 16; o >= 32 / SLOTS; o >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
    }
  }

  const float bad = B.Kc < 0 ? __int_as_float(0x7fc00000) : 0.f;   // NaN: the box cannot hold the tile (host bound wrong)
  if constexpr (!GRAD) {
    if (live && slot == 0) out[((size_t)view * G.nv + iv) * G.nu + iu] = G.step * acc[0] + bad;
    return;
  } else {
  float o6[6 * NSET];
#pragma unroll
  for (int q = 0; q < 6 * NSET; ++q) o6[q] = 0.f;
  if (live && slot == 0) {
    const float gx = acc[0], gy = acc[1], gz = acc[2], hx = acc[3], hy = acc[4], hz = acc[5];
    const size_t pix = ((size_t)view * G.nv + iv) * G.nu + iu;
    const float D = G.step;
    const float sx = gx * G.sgx, sy = gy * G.sgy, sz = gz * G.sgz;
    const float mx = hx * G.sgx * D, my = hy * G.sgy * D, mz = hz * G.sgz * D;
    const float c3 = (py * sz - pz * sy) + (ey * mz - ez * my);
    const float c4 = (pz * sx - px * sz) + (ez * mx - ex * mz);
    const float c5 = (px * sy - py * sx) + (ex * my - ey * mx);
    float wset[NSET];
    if (GRAD == 3) {
      const float l = D * acc[6] + bad;
      proj_out[pix] = l;
      wset[0] = 1.f; wset[NSET > 1 ? 1 : 0] = l; wset[NSET > 2 ? 2 : 0] = __ldg(upstream + pix);   // upstream = target b
    } else {
      wset[0] = __ldg(upstream + pix);
    }
#pragma unroll
    for (int j = 0; j < NSET; ++j) {
      const float wd = wset[j] * D;
      o6[6 * j + 0] = wd * sx + bad; o6[6 * j + 1] = wd * sy; o6[6 * j + 2] = wd * sz;
      o6[6 * j + 3] = wd * c3; o6[6 * j + 4] = wd * c4; o6[6 * j + 5] = wd * c5;
    }
  }
#pragma unroll
  for (int q = 0; q < 6 * NSET; ++q) {
    float v = o6[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    o6[q] = v;
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) {
#pragma unroll
    for (int q = 0; q < 6 * NSET; ++q) red[warp][q] = o6[q];
  }
  __syncthreads();
  if (threadIdx.x < 6 * NSET) {
    float t = 0.f;
#pragma unroll
    for (int wI = 0; wI < TmaLanes<MODE>::THREADS / 32; ++wI) t += red[wI][threadIdx.x];
    const size_t blk = (size_t)by * Q.gx + bx;
    const size_t nblk = (size_t)Q.gx * Q.gy;
    // partials[set][view][block][6]: each weight set is a plain gradient partial array for fwd_contract_kernel
    const int set = threadIdx.x / 6, k = threadIdx.x % 6;
    out[(((size_t)set * Q.n_total + view) * nblk + blk) * 6 + k] = t;
  }
  }  // GRAD
}

}  // namespace dfp
