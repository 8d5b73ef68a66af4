// dfp_bp_tma.cuh - a6 / a7 with the detector patch of each (voxel tile, view) staged in shared memory by TMA.
//
// Same arithmetic, voxel for voxel, as bp_kernel / bp_grad_kernel (dfp_kernels.cuh), but the 4 (back-projection)
// or 12 (gradient) pixel reads of a (voxel, view) pair are LDS from a box of that view's projection:
//
//   * a block owns a tile of 16 x 16 x TZ voxels and loops over ALL views (the volume is written once, a6; the
//     per-view 6-vectors of the tile are reduced in the block, a7/a8);
//   * the image of a convex box under the projective map of Eq.1 is the convex hull of its 8 projected corners
//     (all w' > 0 - the host takes this path only then), so the tile's footprint on the detector is the min/max
//     of 8 corner projections: a PRODUCER warp computes it per view (lanes 0-7 one corner each, shuffle min/max),
//     copies the view's P_eff rows next to the stage and issues ONE `cp.async.bulk.tensor.3d` (SASS UTMALDG) for
//     the box [1][BV][BU] of the caller's projections - out-of-detector pixels are ZERO-FILLED by the TMA unit,
//     which is the zero extension of b~ (U7): no packed copy, no clamps in the inner loop;
//   * STAGES boxes in flight; "full" = mbarrier with complete_tx, "empty" = mbarrier the 8 consumer warps arrive on.
// PAPER.md Eq.1 :60-63, Eq.21 :193-196 (back-projection); Eq.12-17 :139-168, Eq.22 :198-206 (its pose gradient).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "dfp_fwd_tma.cuh"
#include "dfp_kernels.cuh"

namespace dfp {

constexpr int kBpT = 16;                         // voxel tile in x and in y (one consumer thread per column)
constexpr int kBpConsumers = kBpT * kBpT;        // 256 consumer threads = 8 warps
constexpr int kBpTmaThreads = kBpConsumers + 32; // + 1 producer warp
constexpr float kPatchMargin = 0.05f;            // pixels: fp32 rounding of the per-voxel projection

// Detector patch menu (floats): U x V, every U a multiple of 4 (TMA inner box) and = 12 or 20 mod 32.  A warp is an
// 8 x 4 patch of voxel columns at one z: its 32 pixels lie in a thin parallelogram - up to ~16 pixels along u and, by
// the perspective (v scales with the depth, which varies across the tile), 2-5 detector rows.  Bank = (u + U v) mod 32:
// with U = 12 / 20 mod 32 the rows land 12 banks apart and the parallelogram spreads over distinct banks (simulated
// wavefronts per warp load, C5 / C2 / C3: 1.39 / 1.48 / 1.02; the first layout - 16 x 2 columns per warp, U = 4 mod 32 -
// 1.90 / 1.56 / 1.36, measured 2.2 on C5; U = 32, 64, 96 put all rows on the same banks: 2.1-3.5).  The host bounds the largest
// patch any (tile, view) of the call can need and sizes the stages for it; the producer then picks, per (tile,
// view), the SMALLEST patch that holds the actual footprint, so the bytes the TMA unit moves follow the local
// magnification instead of the worst case (near-source tiles and rotated views need 2-4x the median patch).
constexpr int kNumPatches = 6;
__device__ __constant__ int kPatchU[kNumPatches] = {44, 52, 76, 76, 108, 108};
__device__ __constant__ int kPatchV[kNumPatches] = {16, 24, 32, 48, 64, 80};
static const int kPatchUHost[kNumPatches] = {44, 52, 76, 76, 108, 108};
static const int kPatchVHost[kNumPatches] = {16, 24, 32, 48, 64, 80};
struct alignas(64) PatchMaps { CUtensorMap m[kNumPatches]; };
constexpr int kPatchHeader = 64;                 // floats per stage in front of the patch: local P_eff rows, c0, pitch, status, fp64 rows
constexpr int kBpMaxStages = 4;
constexpr int kBpSmemBudget = 72 * 1024;         // dynamic shared memory per block: 3 blocks per SM
inline int bp_stage_words(int kmax) { return kPatchUHost[kmax] * kPatchVHost[kmax] + kPatchHeader; }
inline int bp_num_stages(int kmax) {
  const int n = kBpSmemBudget / (bp_stage_words(kmax) * 4);
  return n > kBpMaxStages ? kBpMaxStages : n;
}

__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Consumer thread -> voxel column of the 16 x 16 tile: a warp is an 8 (x) by 4 (y) patch, two warps across x.
__device__ __forceinline__ int bp_lane_x() { return ((threadIdx.x >> 5) & 1) * 8 + (threadIdx.x & 7); }
__device__ __forceinline__ int bp_lane_y() { return (threadIdx.x >> 6) * 4 + ((threadIdx.x >> 3) & 3); }
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kBpConsumers) : "memory"); }

// Stage header layout (floats).  All rows are LOCAL to the (tile, view): they act on (lx, ly, lz) = voxel index minus
// the tile's first voxel and yield (u, v) relative to the staged patch's first pixel (minus 1/2, for the magic floor):
// [0..11] A rows, [12..20] J rows re-based likewise (gradient only; Eq.13 is invariant under a common shift of u),
// [24] c0b (as bits; see below), [25] status (as bits: 0 ok, 1 no patch of the menu fits), [26] row pitch of the patch
// in BYTES (as bits), [32..55] the A rows again in DOUBLE (12 values; the exact-interpolant mode's slow path).
// The producer derives them in fp64 from BpViewD and rounds once.
struct BpTile {
  int x0, y0, z0, tz;          // first voxel of the tile and its z extent (<= TZ)
};

// Producer: footprint of the tile in view `view`, header, TMA.  Called by the whole producer warp.
template <int HALO>
__device__ __forceinline__ void bp_issue_view(const BpGeom& G, const BpTile& T, const BpViewD* __restrict__ viewsd,
                                              const PatchMaps* maps, int kmax, int stage_words, int view, int stage,
                                              float* smem, unsigned smem_addr, unsigned full_addr) {
  const int lane = threadIdx.x & 31;
  float* hdr = smem + stage * stage_words;
  const double* src = reinterpret_cast<const double*>(viewsd + view);       // A[3][4] then J[3][3]
  // tile origin in centred voxel indices (exact in double); rows with the origin folded into the constant term
  const double X0 = (double)T.x0 - (double)G.hx, Y0 = (double)T.y0 - (double)G.hy, Z0 = (double)T.z0 - (double)G.hz;
  double A[3][4];
#pragma unroll
  for (int r = 0; r < 3; ++r) {
#pragma unroll
    for (int c = 0; c < 4; ++c) A[r][c] = __ldg(src + 4 * r + c);
    A[r][3] = fma(A[r][0], X0, fma(A[r][1], Y0, fma(A[r][2], Z0, A[r][3])));
  }
  // corner (lane & 7) of the tile, local voxel indices
  const double cx = (lane & 1) ? (double)(min(T.x0 + kBpT - 1, G.nx - 1) - T.x0) : 0.0,
               cy = (lane & 2) ? (double)(min(T.y0 + kBpT - 1, G.ny - 1) - T.y0) : 0.0,
               cz = (lane & 4) ? (double)(T.tz - 1) : 0.0;
  const double wp = fma(A[2][0], cx, fma(A[2][1], cy, fma(A[2][2], cz, A[2][3])));
  const double rw = 1.0 / wp;
  float ulo = (float)(fma(A[0][0], cx, fma(A[0][1], cy, fma(A[0][2], cz, A[0][3]))) * rw);
  float vlo = (float)(fma(A[1][0], cx, fma(A[1][1], cy, fma(A[1][2], cz, A[1][3]))) * rw);
  float uhi = ulo, vhi = vlo;
#pragma unroll
  for (int o = 4; o > 0; o >>= 1) {
    ulo = fminf(ulo, __shfl_xor_sync(0xffffffffu, ulo, o));
    uhi = fmaxf(uhi, __shfl_xor_sync(0xffffffffu, uhi, o));
    vlo = fminf(vlo, __shfl_xor_sync(0xffffffffu, vlo, o));
    vhi = fmaxf(vhi, __shfl_xor_sync(0xffffffffu, vhi, o));
  }
  // cells floor(u - CU) = rint(uq) in [rint(lo), rint(hi)], stencil [-HALO, 1 + HALO]  (the same on every lane)
  int ou = (int)floorf(ulo - 0.5f - kPatchMargin) - HALO, ov = (int)floorf(vlo - 0.5f - kPatchMargin) - HALO;
  ou = (((ou + G.CU) >> 2) << 2) - G.CU;                       // 16-byte alignment of the TMA inner coordinate
  const int eu = (int)floorf(uhi + 0.5f + kPatchMargin) + 1 + HALO - ou + 1;
  const int ev = (int)floorf(vhi + 0.5f + kPatchMargin) + 1 + HALO - ov + 1;
  int k = 0;
  while (k <= kmax && (eu > kPatchU[k] || ev > kPatchV[k])) ++k;
  const bool ok = k <= kmax && ulo == ulo && vlo == vlo;
  if (!ok) k = 0;
  // local rows: (u - ou) w' = (A0 - ou A2).(l;1), likewise v; J rows likewise
  if (lane < 12) {
    const int r = lane >> 2, c = lane & 3;
    const double o = r == 0 ? (double)ou : (r == 1 ? (double)ov : 0.0);
    const double a = A[r][c] - o * A[2][c];
    hdr[lane] = (float)a;
    reinterpret_cast<double*>(hdr + 32)[lane] = a;
  } else if (lane < 21) {
    const int r = (lane - 12) / 3, c = (lane - 12) - 3 * r;
    const double o = r == 0 ? (double)ou : (r == 1 ? (double)ov : 0.0);
    hdr[lane] = (float)(__ldg(src + 12 + 3 * r + c) - o * __ldg(src + 12 + 6 + c));
  }
  __syncwarp();                                                  // header words written by lanes 0..20
  if (lane == 0) {
    const int U = kPatchU[k], V = kPatchV[k];
    // SHARED-space byte address of local pixel cell (X, Y) from the magic-rounded floats' bits: 4 X + 4 U Y + c0b
    const unsigned c0b = smem_addr + 4u * (unsigned)(stage * stage_words + kPatchHeader) -
                         (unsigned)kMagicBits * (4u + 4u * (unsigned)U);
    hdr[24] = __uint_as_float(c0b);
    hdr[25] = __uint_as_float(ok ? 0u : 1u);
    hdr[26] = __uint_as_float(4u * (unsigned)U);
    const unsigned bar = full_addr + 8u * stage;
    mbar_expect_tx(bar, U * V * 4);
    // a footprint no patch holds (host bound wrong; never in the tested configs) still loads a patch - from a
    // far corner, all zeros - so that the barrier protocol stays uniform; the consumers write NaN for it
    tma_load_3d(smem_addr + (unsigned)((stage * stage_words + kPatchHeader) * 4), &maps->m[k],
                ok ? ou + G.CU : -4096, ok ? ov + G.CV : -4096, view, bar);
  }
}

// Pixel cell of one (voxel, view) pair inside the staged patch (no clamps: the patch holds the tile's whole
// footprint plus the stencil halo, and out-of-detector pixels were zero-filled): the SHARED-space byte address of
// local pixel (floor u, floor v) is 4*Tu + pitch_bytes*Tv + c0b, two IMADs on the magic-rounded float bits (c0b folds
// the stage base and the magic bias).
template <int OFF>
__device__ __forceinline__ float lds_f32(unsigned addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(addr), "n"(OFF));
  return v;
}

// ------------------------------------------------------------------------------------------------ a6 back
// TZ = voxels along z per thread (register accumulators): 16, or 8 where the magnification is so large that a
// 16-deep tile's footprint exceeds the patch menu (C2: 2.5-3 pixels per voxel).
template <int WEIGHT, int TZ>
__global__ void __launch_bounds__(kBpTmaThreads) bp_tma_kernel(BpGeom G, int n_views, const BpViewD* __restrict__ views,
                                                               const __grid_constant__ PatchMaps maps, int kmax,
                                                               int stage_words, int n_stages, float* __restrict__ vol) {
  extern __shared__ __align__(128) float smem[];
  __shared__ __align__(8) unsigned long long bars[2 * kBpMaxStages];  // full[], empty[]
  const unsigned smem_addr = smem_u32(smem), full_addr = smem_u32(bars), empty_addr = full_addr + 8u * kBpMaxStages;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  BpTile T;
  T.x0 = blockIdx.x * kBpT; T.y0 = blockIdx.y * kBpT; T.z0 = blockIdx.z * TZ;
  T.tz = min(TZ, G.nz - T.z0);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < kBpMaxStages; ++s) {
      mbar_init(full_addr + 8u * s, 1);
      mbar_init(empty_addr + 8u * s, kBpConsumers / 32);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  if (warp == kBpConsumers / 32) {                      // ---- producer warp
    for (int view = 0; view < n_views; ++view) {
      const int s = view % n_stages;
      mbar_wait(empty_addr + 8u * s, ((unsigned)(view / n_stages) & 1u) ^ 1u);
      bp_issue_view<0>(G, T, views, &maps, kmax, stage_words, view, s, smem, smem_addr, full_addr);
    }
    return;
  }
  // ---- consumers: thread = one (x, y) column of the tile, TZ voxels along z in registers
  const int lx = bp_lane_x(), ly = bp_lane_y();
  const int ix = T.x0 + lx, iy = T.y0 + ly;
  const bool live = ix < G.nx && iy < G.ny;
  const float xf = (float)lx, yf = (float)ly;                      // tile-local voxel index
  float acc[TZ];
#pragma unroll
  for (int m = 0; m < TZ; ++m)     // DFP_FLAG_ACCUMULATE: start from the caller's volume (a slice of the views)
    acc[m] = ((G.flags & DFP_FLAG_ACCUMULATE) && live && m < T.tz) ? vol[((size_t)(T.z0 + m) * G.ny + iy) * G.nx + ix] : 0.f;
  bool bad = false;
  for (int view = 0; view < n_views; ++view) {
    const int s = view % n_stages;
    mbar_wait(full_addr + 8u * s, (unsigned)(view / n_stages) & 1u);
    const float* hdr = smem + s * stage_words;
    const unsigned c0 = __float_as_uint(hdr[24]), BU = __float_as_uint(hdr[26]);
#ifdef DFP_CHECK_BOUNDS
    const unsigned chk_lo = smem_addr + 4u * (unsigned)(s * stage_words + kPatchHeader) + BU + 4u,
                   chk_hi = smem_addr + 4u * (unsigned)((s + 1) * stage_words) - 2u * BU - 12u;
#endif
    bad |= __float_as_uint(hdr[25]) != 0u;
    if (live) {
      const float a02 = hdr[2], a12 = hdr[6], a22 = hdr[10];
      const float ub = fmaf(hdr[0], xf, fmaf(hdr[1], yf, hdr[3]));
      const float vb = fmaf(hdr[4], xf, fmaf(hdr[5], yf, hdr[7]));
      const float wb = fmaf(hdr[8], xf, fmaf(hdr[9], yf, hdr[11]));
      const float2 ab2 = make_float2(a02, a12), uvb = make_float2(ub, vb);
#pragma unroll
      for (int m = 0; m < TZ; ++m) {
        if (m < T.tz) {
          // (u, v) as one fp32x2 lane pair: advance along z, perspective divide, floor and fractions
          const float mf = (float)m;
          const float wz = fmaf(mf, a22, wb);
          const float rw = fast_rcp(wz);
          const float2 uvp = __ffma2_rn(make_float2(mf, mf), ab2, uvb);                 // (u', v')
          const float2 uvq = __fmul2_rn(uvp, make_float2(rw, rw));
          const float2 t2 = __fadd2_rn(uvq, make_float2(kMagic, kMagic));
          // fractions from the residual (u' - rint(u) w') / w': the residual is a small number, so neither the rounding of
          // the quotient u = u'/w' (|u| up to 100 pixels) nor that of 1/w' reaches the interpolation weights
          const float2 tr = __fadd2_rn(t2, make_float2(-kMagic, -kMagic));
          const float2 fr = __ffma2_rn(__ffma2_rn(make_float2(-tr.x, -tr.y), make_float2(wz, wz), uvp), make_float2(rw, rw),
                                       make_float2(0.5f, 0.5f));
          const unsigned a0 = 4u * (unsigned)__float_as_int(t2.x) + BU * (unsigned)__float_as_int(t2.y) + c0;
          const unsigned a1 = a0 + BU;
          // the two rows as a pair: lerp along u on both, then along v
          const float2 r2 = lerp2(make_float2(fr.x, fr.x), make_float2(lds_f32<0>(a0), lds_f32<0>(a1)),
                                  make_float2(lds_f32<4>(a0), lds_f32<4>(a1)));
          float val = lerp(fr.y, r2.x, r2.y);
#ifdef DFP_CHECK_BOUNDS
          if (a0 < chk_lo || a0 > chk_hi) val = __int_as_float(0x7fc00000);
#endif
          const float wgt = WEIGHT ? G.sad2 * rw * rw : 1.f;
          acc[m] = fmaf(wgt, val, acc[m]);
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(empty_addr + 8u * s);
  }
  if (live) {
    const float nanv = bad ? __int_as_float(0x7fc00000) : 0.f;
#pragma unroll
    for (int m = 0; m < TZ; ++m)
      if (m < T.tz) vol[((size_t)(T.z0 + m) * G.ny + iy) * G.nx + ix] = acc[m] + nanv;
  }
}

// ------------------------------------------------------------------------------------------------ a7 back gradient
// Per (voxel j, view), as bp_grad_kernel: q' = W [ d~_u l (J1 - u J3) + d~_v l (J2 - v J3) ] / w' (+ b~ dW/dr'),
// six running sums per (thread, view) along the thread's z column with the lever arm factored out.  Per view the
// warp's sums are shuffled together; the 8 warps' results wait in shared memory (two buffers of kBpGradGroup views)
// and are added in fixed order once per group -> partials[tile][view][6]: one consumer barrier per group, not per view.
constexpr int kBpGradGroup = 8;                  // views per cross-warp reduction
constexpr float kFaceEpsBp = 2e-5f;              // |fraction - {0,1}| below this: the fp32 pixel-cell decision is not trusted

// MODE 1 (DFP_FLAG_GRAD_INTERP): exact derivatives of the bilinear interpolant, 4 LDS instead of 12.
template <int WEIGHT, int DW, int TZ, int MODE>
__global__ void __launch_bounds__(kBpTmaThreads) bp_grad_tma_kernel(BpGeom G, int n_views,
                                                                    const BpViewD* __restrict__ views,
                                                                    const __grid_constant__ PatchMaps maps, int kmax,
                                                                    int stage_words, int n_stages,
                                                                    const float* __restrict__ upstream,
                                                                    float* __restrict__ partials) {
  constexpr int NW = kBpConsumers / 32;
  extern __shared__ __align__(128) float smem[];
  __shared__ __align__(8) unsigned long long bars[2 * kBpMaxStages];
  __shared__ float wpart[2][kBpGradGroup][NW][6];
  const unsigned smem_addr = smem_u32(smem), full_addr = smem_u32(bars), empty_addr = full_addr + 8u * kBpMaxStages;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  BpTile T;
  T.x0 = blockIdx.x * kBpT; T.y0 = blockIdx.y * kBpT; T.z0 = blockIdx.z * TZ;
  T.tz = min(TZ, G.nz - T.z0);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < kBpMaxStages; ++s) {
      mbar_init(full_addr + 8u * s, 1);
      mbar_init(empty_addr + 8u * s, NW);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  if (warp == NW) {                                     // ---- producer warp
    for (int view = 0; view < n_views; ++view) {
      const int s = view % n_stages;
      mbar_wait(empty_addr + 8u * s, ((unsigned)(view / n_stages) & 1u) ^ 1u);
      bp_issue_view<1>(G, T, views, &maps, kmax, stage_words, view, s, smem, smem_addr, full_addr);
    }
    return;
  }
  // ---- consumers
  const int lx = bp_lane_x(), ly = bp_lane_y();
  const int ix = T.x0 + lx, iy = T.y0 + ly;
  const bool live = ix < G.nx && iy < G.ny;
  const float xf = (float)lx, yf = (float)ly;                      // tile-local voxel index
  // object-frame mm of the column's first voxel
  const float rx = G.cx + ((float)ix - G.hx) * G.vx, ry = G.cy + ((float)iy - G.hy) * G.vy,
              rz = G.cz + ((float)T.z0 - G.hz) * G.vz;
  const float* wcol = upstream + ((size_t)T.z0 * G.ny + (live ? iy : 0)) * G.nx + (live ? ix : 0);
  const size_t wstride = (size_t)G.ny * G.nx;
  const size_t tile = ((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
  float wreg[TZ];            // the thread's column of the upstream gradient: the same for every view
#pragma unroll
  for (int m = 0; m < TZ; ++m) wreg[m] = (live && m < T.tz) ? __ldg(wcol + (size_t)m * wstride) : 0.f;
  bool bad = false;
  const int n_groups = (n_views + kBpGradGroup - 1) / kBpGradGroup;
  for (int grp = 0; grp < n_groups; ++grp) {
    const int v_lo = grp * kBpGradGroup, v_hi = min(v_lo + kBpGradGroup, n_views);
    for (int view = v_lo; view < v_hi; ++view) {
      const int s = view % n_stages;
      mbar_wait(full_addr + 8u * s, (unsigned)(view / n_stages) & 1u);
      const float* hdr = smem + s * stage_words;
      const unsigned c0 = __float_as_uint(hdr[24]), BU = __float_as_uint(hdr[26]);
#ifdef DFP_CHECK_BOUNDS
      const unsigned chk_lo = smem_addr + 4u * (unsigned)(s * stage_words + kPatchHeader) + BU + 4u,
                     chk_hi = smem_addr + 4u * (unsigned)((s + 1) * stage_words) - 2u * BU - 12u;
#endif
      bad |= __float_as_uint(hdr[25]) != 0u;
      float sm[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      if (live) {
        const float a02 = hdr[2], a12 = hdr[6], a22 = hdr[10];
        const float ub = fmaf(hdr[0], xf, fmaf(hdr[1], yf, hdr[3]));
        const float vb = fmaf(hdr[4], xf, fmaf(hdr[5], yf, hdr[7]));
        const float wb = fmaf(hdr[8], xf, fmaf(hdr[9], yf, hdr[11]));
        const float j00 = hdr[12], j01 = hdr[13], j02 = hdr[14], j10 = hdr[15], j11 = hdr[16], j12 = hdr[17],
                    j20 = hdr[18], j21 = hdr[19], j22 = hdr[20];
        // packed fp32x2 arithmetic on (u, v) / row / column pairs (FFMA2, FADD2, FMUL2: the scalar code's roundings)
        const float2 ab2 = make_float2(a02, a12), uvb = make_float2(ub, vb);
        const float2 j0 = make_float2(j00, j01), j1 = make_float2(j10, j11), j2 = make_float2(j20, j21);
        float2 s01 = make_float2(0.f, 0.f), s34 = make_float2(0.f, 0.f);
        float s2 = 0.f, s5 = 0.f;
#pragma unroll
        for (int m = 0; m < TZ; ++m) {
          if (m < T.tz) {
            const float mf = (float)m;
            const float wz = fmaf(mf, a22, wb);
            const float rw = fast_rcp(wz);
            const float2 uvp = __ffma2_rn(make_float2(mf, mf), ab2, uvb);                 // (u', v')
            const float2 uvq = __fmul2_rn(uvp, make_float2(rw, rw));
            const float2 t2 = __fadd2_rn(uvq, make_float2(kMagic, kMagic));
            // fractions from the residual (u' - rint(u) w') / w': the residual is a small number, so neither the rounding of
            // the quotient u = u'/w' (|u| up to 100 pixels) nor that of 1/w' reaches the interpolation weights
            const float2 tr = __fadd2_rn(t2, make_float2(-kMagic, -kMagic));
            const float2 fr = __ffma2_rn(__ffma2_rn(make_float2(-tr.x, -tr.y), make_float2(wz, wz), uvp), make_float2(rw, rw),
                                         make_float2(0.5f, 0.5f));
            unsigned a0 = 4u * (unsigned)__float_as_int(t2.x) + BU * (unsigned)__float_as_int(t2.y) + c0;
#ifdef DFP_CHECK_BOUNDS
            if (a0 < chk_lo || a0 > chk_hi) s2 = __int_as_float(0x7fc00000);
#endif
            float pa = fr.x, pb = fr.y;
            float dlu, dlv, l00, l01, l10, l11;
            if (MODE == 1) {
              // the derivative of the bilinear interpolant jumps at pixel boundaries: a voxel that projects within
              // fp32 rounding of one takes its cell and fractions from the fp64 rows, as the oracle does
              if (fminf(fminf(pa, 1.f - pa), fminf(pb, 1.f - pb)) < kFaceEpsBp) {
                const double* Ad = reinterpret_cast<const double*>(hdr + 32);
                const double lx = (double)xf, ly = (double)yf, lz = (double)m;
                const double wd = fma(Ad[8], lx, fma(Ad[9], ly, fma(Ad[10], lz, Ad[11])));
                const double ud = fma(Ad[0], lx, fma(Ad[1], ly, fma(Ad[2], lz, Ad[3]))) / wd + 0.5;
                const double vd = fma(Ad[4], lx, fma(Ad[5], ly, fma(Ad[6], lz, Ad[7]))) / wd + 0.5;
                const double fu = floor(ud), fv = floor(vd);
                pa = (float)(ud - fu); pb = (float)(vd - fv);
                a0 = smem_addr + 4u * (unsigned)(s * stage_words + kPatchHeader) + 4u * (unsigned)(int)fu + BU * (unsigned)(int)fv;
              }
              const unsigned a1 = a0 + BU;
              l00 = lds_f32<0>(a0); l01 = lds_f32<4>(a0); l10 = lds_f32<0>(a1); l11 = lds_f32<4>(a1);
              dlu = lerp(pb, l01 - l00, l11 - l10);
              dlv = lerp(pa, l10 - l00, l11 - l01);
            } else {
              // rows v, v+1: columns u-1 .. u+2; rows v-1, v+2: columns u, u+1
              const unsigned a1 = a0 + BU, am = a0 - BU, a2 = a1 + BU;
              const float l0m = lds_f32<-4>(a0), l02 = lds_f32<8>(a0);
              const float l1m = lds_f32<-4>(a1), l12 = lds_f32<8>(a1);
              l00 = lds_f32<0>(a0); l01 = lds_f32<4>(a0); l10 = lds_f32<0>(a1); l11 = lds_f32<4>(a1);
              const float lm0 = lds_f32<0>(am), lm1 = lds_f32<4>(am), l20 = lds_f32<0>(a2), l21 = lds_f32<4>(a2);
              // (du0, du1): rows v, v+1;  (dv0, dv1): columns u, u+1
              const float2 du = lerp2(make_float2(pa, pa), sub2(make_float2(l01, l11), make_float2(l0m, l1m)),
                                      sub2(make_float2(l02, l12), make_float2(l00, l10)));
              dlu = lerp(pb, du.x, du.y);
              const float2 dv = lerp2(make_float2(pb, pb), sub2(make_float2(l10, l11), make_float2(lm0, lm1)),
                                      sub2(make_float2(l20, l21), make_float2(l00, l01)));
              dlv = lerp(pa, dv.x, dv.y);
            }
            const float W = WEIGHT ? G.sad2 * rw * rw : 1.f;
            const float cc = fmaf(dlu, uvq.x, dlv * uvq.y);
            const float2 dlu2 = make_float2(dlu, dlu), dlv2 = make_float2(dlv, dlv);
            float2 q2 = __ffma2_rn(dlu2, j0, __ffma2_rn(dlv2, j1, __fmul2_rn(make_float2(-cc, -cc), j2)));
            float qz = fmaf(dlu, j02, fmaf(dlv, j12, -cc * j22));
            const float sc = (MODE == 1 ? 1.0f : 0.5f) * W * rw * wreg[m];
            if (DW) {
              const float b0 = lerp(pa, l00, l01), b1 = lerp(pa, l10, l11);
              const float bv = lerp(pb, b0, b1);
              const float k = (MODE == 1 ? -2.f : -4.f) * bv;
              q2 = __ffma2_rn(make_float2(k, k), j2, q2);
              qz = fmaf(k, j22, qz);
            }
            const float scm = sc * mf;
            s01 = __ffma2_rn(make_float2(sc, sc), q2, s01);
            s34 = __ffma2_rn(make_float2(scm, scm), q2, s34);
            s2 = fmaf(sc, qz, s2);
            s5 = fmaf(scm, qz, s5);
          }
        }
        sm[0] = s01.x; sm[1] = s01.y; sm[2] = s2; sm[3] = s34.x; sm[4] = s34.y; sm[5] = s5;
        const float mx = sm[3] * G.vz, my = sm[4] * G.vz;
        const float cx = ry * sm[2] - rz * sm[1] - my;
        const float cy = rz * sm[0] - rx * sm[2] + mx;
        const float cz = rx * sm[1] - ry * sm[0];
        sm[3] = cx; sm[4] = cy; sm[5] = cz;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty_addr + 8u * s);     // the patch is free; the sums are in registers
#pragma unroll
      for (int k = 0; k < 6; ++k) {
        float v = sm[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        sm[k] = v;
      }
      if (lane == 0) {
#pragma unroll
        for (int k = 0; k < 6; ++k) wpart[grp & 1][view - v_lo][warp][k] = sm[k];
      }
    }
    consumer_sync();        // group grp complete in wpart[grp & 1]; also: the reducers of group grp-1 are done
    if (threadIdx.x < (v_hi - v_lo) * 6) {
      const int vv = threadIdx.x / 6, k = threadIdx.x % 6;
      float t = 0.f;
#pragma unroll
      for (int w = 0; w < NW; ++w) t += wpart[grp & 1][vv][w][k];
      if (bad) t = __int_as_float(0x7fc00000);
      partials[(tile * n_views + (v_lo + vv)) * 6 + k] = t;
    }
  }
}

}  // namespace dfp
