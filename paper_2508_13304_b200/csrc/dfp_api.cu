// dfp_api.cu - the C ABI of libdfp (include/dfp.h): argument validation, per-view set-up (fp64 on the host,
// dfp_params.h), workspace carving and kernel launches (dfp_kernels.cuh).  No torch types, no exceptions, no
// printing, no host synchronisation in the device-pointer calls.
#include <atomic>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/dfp.h"
#include "dfp_bp_tma.cuh"
#include "dfp_fwd_tma.cuh"
#include "dfp_kernels.cuh"
#include "dfp_params.h"
#include "dfp_dd.cuh"
#include "dfp_sf.cuh"
#include "dfp_joseph.cuh"
#include "dfp_loss.cuh"
#include "dfp_siddon.cuh"

namespace {

using namespace dfp;

thread_local char g_cuda_msg[256] = "no CUDA error recorded";
thread_local int g_launches = 0;
thread_local int g_path = DFP_PATH_GATHER;

thread_local bool g_timing = false;
thread_local cudaEvent_t g_ev[2] = {nullptr, nullptr};
thread_local int g_ev_dev = -1;              // the device the two events belong to
thread_local bool g_ev_valid = false;

void time_begin(cudaStream_t s) {
  g_ev_valid = false;
  if (!g_timing) return;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return;
  if (g_ev[0] && dev != g_ev_dev) {          // events are per device: the caller switched devices
    cudaEventDestroy(g_ev[0]); cudaEventDestroy(g_ev[1]);
    g_ev[0] = g_ev[1] = nullptr;
  }
  if (!g_ev[0]) {
    if (cudaEventCreate(&g_ev[0]) != cudaSuccess || cudaEventCreate(&g_ev[1]) != cudaSuccess) {
      g_ev[0] = g_ev[1] = nullptr;
      cudaGetLastError();
      return;
    }
    g_ev_dev = dev;
  }
  if (cudaEventRecord(g_ev[0], s) != cudaSuccess) cudaGetLastError();   // timing is best effort: never fails the call
}
void time_end(cudaStream_t s) {
  if (!g_timing || !g_ev[1]) return;
  g_ev_valid = cudaEventRecord(g_ev[1], s) == cudaSuccess;
  if (!g_ev_valid) cudaGetLastError();
}

// Per-view constants go to the device through a small ring of PINNED host buffers owned by the calling thread, so
// that the upload is a true asynchronous copy (a cudaMemcpyAsync from pageable memory is staged by the runtime and
// may block the host).  A slot is reused only after the copy that last read it has completed (its event); with
// kStageSlots calls in flight that wait never triggers in practice.  Slots grow on demand and live until the thread
// ends (host memory only: the library still allocates no device memory in the device-pointer calls).
constexpr int kStageSlots = 8;
struct StageRing {
  void* buf[kStageSlots] = {};
  size_t cap[kStageSlots] = {};
  cudaEvent_t ev[kStageSlots] = {};
  int dev[kStageSlots] = {};
  int next = 0;
  ~StageRing() {
    for (int i = 0; i < kStageSlots; ++i) {
      if (ev[i]) cudaEventDestroy(ev[i]);
      if (buf[i]) cudaFreeHost(buf[i]);
    }
  }
};
thread_local StageRing g_stage;

// Copies `bytes` from pageable host memory `src` to device memory `dst` on stream `s` without blocking on the GPU.
cudaError_t upload_async(void* dst, const void* src, size_t bytes, cudaStream_t s) {
  StageRing& R = g_stage;
  const int i = R.next;
  R.next = (R.next + 1) % kStageSlots;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (R.ev[i] && R.dev[i] != dev) { cudaEventDestroy(R.ev[i]); R.ev[i] = nullptr; }
  if (R.ev[i]) {
    e = cudaEventSynchronize(R.ev[i]);       // the copy that last used this slot (kStageSlots uploads ago)
    if (e != cudaSuccess) return e;
  } else {
    e = cudaEventCreateWithFlags(&R.ev[i], cudaEventDisableTiming);
    if (e != cudaSuccess) { R.ev[i] = nullptr; return e; }
    R.dev[i] = dev;
  }
  if (R.cap[i] < bytes) {
    if (R.buf[i]) cudaFreeHost(R.buf[i]);
    R.buf[i] = nullptr; R.cap[i] = 0;
    const size_t want = bytes < 65536 ? 65536 : bytes + bytes / 2;
    e = cudaHostAlloc(&R.buf[i], want, cudaHostAllocDefault);
    if (e != cudaSuccess) { R.buf[i] = nullptr; return e; }
    R.cap[i] = want;
  }
  std::memcpy(R.buf[i], src, bytes);
  e = cudaMemcpyAsync(dst, R.buf[i], bytes, cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return e;
  return cudaEventRecord(R.ev[i], s);
}

int cuda_fail(cudaError_t e, const char* where) {
  std::snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error in %s: %s", where, cudaGetErrorString(e));
  return DFP_ERR_CUDA;
}
#define DFP_CUDA(call, where)                                   \
  do {                                                          \
    cudaError_t e_ = (call);                                    \
    if (e_ != cudaSuccess) return cuda_fail(e_, where);         \
  } while (0)

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

int validate_geometry(const dfp_geometry* g) {
  if (!g) return DFP_ERR_NULL;
  const float f[] = {g->vx, g->vy, g->vz, g->cx, g->cy, g->cz, g->du, g->dv, g->u0, g->v0, g->sad, g->sdd, g->step_mm};
  for (float x : f)
    if (!std::isfinite(x)) return DFP_ERR_NONFINITE;
  if (g->nx <= 0 || g->ny <= 0 || g->nz <= 0 || g->nu <= 0 || g->nv <= 0) return DFP_ERR_DIMS;
  if (!(g->vx > 0) || !(g->vy > 0) || !(g->vz > 0) || !(g->du > 0) || !(g->dv > 0)) return DFP_ERR_DIMS;
  if (!(g->sad > 0) || !(g->sdd > g->sad)) return DFP_ERR_DIMS;
  if (g->bp_weight != 0 && g->bp_weight != 1) return DFP_ERR_DIMS;
  // 32-bit cell indices inside the packed copies; magic-number floor needs |index| < 2^22
  const VolLayout L = make_layout(*g);
  if ((double)L.px * L.py * L.pz >= 2147483648.0) return DFP_ERR_DIMS;
  if ((double)(g->nu + 2 * kPadDet) * (g->nv + 2 * kPadDet) >= 2147483648.0) return DFP_ERR_DIMS;
  if (g->nx > (1 << 21) || g->ny > (1 << 21) || g->nz > (1 << 21) || g->nu > (1 << 21) || g->nv > (1 << 21))
    return DFP_ERR_DIMS;
  return DFP_OK;
}

// Views ride on blockIdx.z (<= 65535): larger batches are run as consecutive slices of kMaxViewsPerLaunch views
// (a multiple of 4, so that every slice's projection / gradient pointers keep their 16-byte alignment).
constexpr int kMaxViewsPerLaunch = 65532;
constexpr int kMaxViews = 1 << 24;

int validate_views(const dfp_geometry& g, int n_views, const float* angles, const float* poses) {
  if (n_views <= 0 || n_views > kMaxViews) return DFP_ERR_DIMS;
  if (!angles || !poses) return DFP_ERR_NULL;
  const int stride = view_stride(g);
  for (int v = 0; v < n_views; ++v) {
    for (int k = 0; k < stride; ++k)
      if (!std::isfinite(angles[(size_t)stride * v + k])) return DFP_ERR_NONFINITE;
    if (stride > 1 && !make_frame(g, angles, v).ok) return DFP_ERR_DIMS;
    for (int k = 0; k < 6; ++k)
      if (!std::isfinite(poses[6 * v + k])) return DFP_ERR_NONFINITE;
  }
  return DFP_OK;
}

// ---- TMA path of the forward kernels (dfp_fwd_tma.cuh) -------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = []() -> EncodeTiledFn {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      return nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// Tensor map over the caller's volume [nz][ny][nx] fp32 with the staging box of dfp_fwd_tma.cuh; elements
// outside the volume read as zero (the zero extension of f~, U7).
// `pitch`: floats between rows of the array the map is made over - the caller's volume when nx % 4 == 0, else a copy
// with its rows padded to a multiple of 4 floats (global strides must be multiples of 16 bytes); the map's extent stays
// nx, so the padding is out of range like everything else beyond the volume.
inline int pitch4(int n) { return (n + 3) / 4 * 4; }
bool make_volume_map(const dfp_geometry& g, const float* d_vol, int pitch, int bx, int by, int bz, CUtensorMap* map) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc || (pitch % 4) != 0 || pitch < g.nx) return false;
  const cuuint64_t dims[3] = {(cuuint64_t)g.nx, (cuuint64_t)g.ny, (cuuint64_t)g.nz};
  const cuuint64_t strides[2] = {(cuuint64_t)pitch * 4, (cuuint64_t)pitch * g.ny * 4};
  const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bz};
  const cuuint32_t es[3] = {1, 1, 1};
  return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(d_vol), dims, strides, box, es,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Conservative host-side bound: can every 16x16-pixel tile of this view march in chunks of >= kMinChunk samples
// inside the staging box?  (The kernel computes the exact chunk length per block; this only picks the path.)
// Positions at path length tau: p = s' + tau e, so a tile's extent along axis a is tau |De_a| with
// |De_a| <= (|Dd_a| + |e_a| (rho_max/|d|) |Dd|) / SDD  for pixel offsets Dd on a detector at distance >= SDD.
constexpr int kMinChunk = 4;
#ifndef DFP_CLASS_TAN
#define DFP_CLASS_TAN 0.5774      // tan(30 deg): a view is "along y" when |e_x| < tan(30 deg) |e_y| (voxel-index units)
#endif
constexpr double kClassTan = DFP_CLASS_TAN;
// volt[z][x][y] = vol[z][y][x]: the volume with y fastest, for the gradient kernel of the views along x (MODE 6)
__global__ void __launch_bounds__(256) transpose_xy_kernel(int nx, int ny, int tpitch, const float* __restrict__ vol,
                                                           float* __restrict__ volt) {
  __shared__ float tile[32][33];
  const size_t slab = (size_t)blockIdx.z * nx * ny, tslab = (size_t)blockIdx.z * nx * tpitch;
  const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
  for (int j = threadIdx.y; j < 32; j += 8) {
    const int x = x0 + threadIdx.x, y = y0 + j;
    if (x < nx && y < ny) tile[j][threadIdx.x] = vol[slab + (size_t)y * nx + x];
  }
  __syncthreads();
  for (int j = threadIdx.y; j < 32; j += 8) {
    const int y = y0 + threadIdx.x, x = x0 + j;
    if (x < nx && y < ny) volt[tslab + (size_t)x * tpitch + y] = tile[threadIdx.x][j];
  }
}
bool tma_view_fits(const dfp_geometry& g, const FwdGeom& G, const FwdView& V, const ViewFrame& F, bool grad,
                   const int* box, int TU, int TV, int min_chunk = kMinChunk, int align_axis = 0) {
  const double v3[3] = {g.vx, g.vy, g.vz}, c3[3] = {g.cx, g.cy, g.cz};
  const double half[3] = {0.5 * g.nx * g.vx + 3 * g.vx, 0.5 * g.ny * g.vy + 3 * g.vy, 0.5 * g.nz * g.vz + 3 * g.vz};
  double tau_max = 0;
  for (int c = 0; c < 8; ++c) {
    double d2 = 0;
    for (int a = 0; a < 3; ++a) {
      const double x = c3[a] + ((c >> a) & 1 ? half[a] : -half[a]) - V.src[a];
      d2 += x * x;
    }
    tau_max = std::fmax(tau_max, std::sqrt(d2));
  }
  double emax[3] = {0, 0, 0}, dmax = 0;
  for (int c = 0; c < 4; ++c) {
    const double iu = (c & 1) ? g.nu - 1 : 0, iv = (c & 2) ? g.nv - 1 : 0;
    double d[3], n2 = 0;
    for (int a = 0; a < 3; ++a) { d[a] = V.d0[a] + iu * V.du[a] + iv * V.dv[a]; n2 += d[a] * d[a]; }
    const double n = std::sqrt(n2);
    dmax = std::fmax(dmax, n);
    for (int a = 0; a < 3; ++a) emax[a] = std::fmax(emax[a], std::fabs(d[a]) / n);
  }
  const double sdd = F.sdd;                  // perpendicular source-detector distance of this view
  const double rho = std::sqrt(std::fmax(dmax * dmax - sdd * sdd, 0.0)) / sdd;
  const double tu = TU - 1, tv = TV - 1;
  // the tile's longer diagonal on the detector (mm): max |tu U +- tv V|
  const double dnorm = std::sqrt(tu * tu * F.ulen * F.ulen + tv * tv * F.vlen * F.vlen + 2.0 * tu * tv * std::fabs(F.udotv));
  for (int a = 0; a < 3; ++a) {
    const double dd = tu * std::fabs(V.du[a]) + tv * std::fabs(V.dv[a]);
    const double span = tau_max * (dd + emax[a] * rho * dnorm) / sdd / v3[a];
    const double slope = (double)G.step * emax[a] / v3[a];
    const double avail = box[a] - 4 - (grad ? 2 : 0) - (a == align_axis ? kBoxAlignLoss : 0) - 2.0 * kBoxMargin - 1.05 * span - 0.05;
    if (avail < (min_chunk - 1) * slope) return false;
  }
  return true;
}

// ---- TMA path of the back-projection kernels (dfp_bp_tma.cuh) -----------------------------------
// Tensor maps over the caller's projections [V][nv][nu] fp32, one per patch of the menu up to kmax.
bool make_proj_maps(const dfp_geometry& g, int V, const float* d_proj, int pitch, int kmax, PatchMaps* maps) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc || (pitch % 4) != 0 || pitch < g.nu) return false;
  const cuuint64_t dims[3] = {(cuuint64_t)g.nu, (cuuint64_t)g.nv, (cuuint64_t)V};
  const cuuint64_t strides[2] = {(cuuint64_t)pitch * 4, (cuuint64_t)pitch * g.nv * 4};
  const cuuint32_t es[3] = {1, 1, 1};
  for (int k = 0; k < kNumPatches; ++k) {
    const int kk = k <= kmax ? k : kmax;                 // unused slots repeat the largest map
    const cuuint32_t box[3] = {(cuuint32_t)kPatchUHost[kk], (cuuint32_t)kPatchVHost[kk], 1};
    if (enc(&maps->m[k], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(d_proj), dims, strides, box, es,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  return true;
}

// Smallest patch of the menu that is guaranteed to hold the footprint of every 16 x 16 x tz voxel tile in this
// view (-1: none, or a voxel is not in front of the source - then the gather path, which handles w' <= 0, runs).
// For two voxels r, r+D of a tile: |Du| <= (|A0.D| + |u| |A2.D|) / w'(r+D)  with u = A0.r / A2.r  (exact).
int bp_view_patch(const BpGeom& G, const BpView& Vw, int tz, int halo) {
  const double lo[3] = {-(double)G.hx, -(double)G.hy, -(double)G.hz};
  const double hi[3] = {G.nx - 1 - (double)G.hx, G.ny - 1 - (double)G.hy, G.nz - 1 - (double)G.hz};
  double wmin = 1e300, umax = 0, vmax = 0, wmax = 0;
  for (int c = 0; c < 8; ++c) {
    const double x = (c & 1) ? hi[0] : lo[0], y = (c & 2) ? hi[1] : lo[1], z = (c & 4) ? hi[2] : lo[2];
    const double u = Vw.A[0][0] * x + Vw.A[0][1] * y + Vw.A[0][2] * z + Vw.A[0][3];
    const double v = Vw.A[1][0] * x + Vw.A[1][1] * y + Vw.A[1][2] * z + Vw.A[1][3];
    const double w = Vw.A[2][0] * x + Vw.A[2][1] * y + Vw.A[2][2] * z + Vw.A[2][3];
    if (!(w > 0)) return -1;
    wmin = std::fmin(wmin, w); wmax = std::fmax(wmax, w);
    umax = std::fmax(umax, std::fabs(u / w)); vmax = std::fmax(vmax, std::fabs(v / w));
  }
  if (!(wmin > 0.02 * wmax)) return -1;
  const double T[3] = {(double)(kBpT - 1), (double)(kBpT - 1), (double)(tz - 1)};
  double eu = 0, ev = 0;
  for (int a = 0; a < 3; ++a) {
    eu += (std::fabs(Vw.A[0][a]) + umax * std::fabs(Vw.A[2][a])) * T[a] / wmin;
    ev += (std::fabs(Vw.A[1][a]) + vmax * std::fabs(Vw.A[2][a])) * T[a] / wmin;
  }
  const int need_u = (int)std::ceil(eu + 2 * kPatchMargin) + 3 + 2 * halo + 3;   // floor cells, stencil, alignment
  const int need_v = (int)std::ceil(ev + 2 * kPatchMargin) + 3 + 2 * halo;
  for (int k = 0; k < kNumPatches; ++k)
    if (need_u <= kPatchUHost[k] && need_v <= kPatchVHost[k]) return k;
  return -1;
}

// Kernels that use more than 48 KiB of dynamic shared memory need the opt-in attribute, per device: set once per
// (thread's current) device and remembered.
cudaError_t ensure_smem_attributes() {
  static bool done[64] = {false};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev >= 0 && dev < 64 && done[dev]) return cudaSuccess;
#define DFP_ATTR(k, bytes)                                                                  \
  if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes)) != cudaSuccess) return e
  DFP_ATTR((fwd_tma_kernel<0, 0>), tma_smem_bytes<0>());
  DFP_ATTR((fwd_tma_kernel<0, 1>), tma_smem_bytes<1>());
  DFP_ATTR((fwd_tma_kernel<0, 2>), tma_smem_bytes<2>());
  DFP_ATTR((fwd_tma_kernel<4, 2>), tma_smem_bytes<2>());
  DFP_ATTR((fwd_tma_kernel<0, 4>), tma_smem_bytes<4>());
  DFP_ATTR((fwd_tma_kernel<0, 5>), tma_smem_bytes<5>());
  DFP_ATTR((fwd_tma_kernel<1, 2>), tma_smem_bytes<2>());
  DFP_ATTR((fwd_tma_kernel<1, 3>), tma_smem_bytes<3>());
  DFP_ATTR((fwd_tma_kernel<1, 7>), tma_smem_bytes<7>());
  DFP_ATTR((fwd_tma_kernel<2, 7>), tma_smem_bytes<7>());
  DFP_ATTR((fwd_tma_kernel<3, 7>), tma_smem_bytes<7>());
  DFP_ATTR((fwd_tma_kernel<5, 6>), tma_smem_bytes<6>());
  DFP_ATTR((fwd_tma_kernel<6, 6>), tma_smem_bytes<6>());
  DFP_ATTR((fwd_tma_kernel<2, 2>), tma_smem_bytes<2>());
  DFP_ATTR((fwd_tma_kernel<2, 3>), tma_smem_bytes<3>());
  DFP_ATTR((fwd_tma_kernel<3, 2>), tma_smem_bytes<2>());
  DFP_ATTR((fwd_tma_kernel<3, 3>), tma_smem_bytes<3>());
  DFP_ATTR((bp_tma_kernel<0, 16>), kBpSmemBudget);
  DFP_ATTR((bp_tma_kernel<1, 16>), kBpSmemBudget);
  DFP_ATTR((bp_tma_kernel<0, 8>), kBpSmemBudget);
  DFP_ATTR((bp_tma_kernel<1, 8>), kBpSmemBudget);
#define DFP_ATTR_G(W, D)                                      \
  DFP_ATTR((bp_grad_tma_kernel<W, D, 16, 0>), kBpSmemBudget); \
  DFP_ATTR((bp_grad_tma_kernel<W, D, 8, 0>), kBpSmemBudget);  \
  DFP_ATTR((bp_grad_tma_kernel<W, D, 16, 1>), kBpSmemBudget); \
  DFP_ATTR((bp_grad_tma_kernel<W, D, 8, 1>), kBpSmemBudget)
  DFP_ATTR_G(0, 0);
  DFP_ATTR_G(1, 0);
  DFP_ATTR_G(1, 1);
#undef DFP_ATTR_G
#undef DFP_ATTR
  if (dev >= 0 && dev < 64) done[dev] = true;
  return cudaSuccess;
}

// ---- workspace carving ---------------------------------------------------------------------------
struct FwdWs {
  size_t off_views, off_dd, off_con, off_pvol, off_part, off_fixed, off_volt, off_ids, total;
  int gx, gy;     // blocks per view (16 x 16-pixel tiles)
  int gy8;        // rows of 16 x 8-pixel tiles (TMA gradient kernel)
};
// `packed`: reserve the gather path's 4x packed copy of the volume (and, for the weight models that use it, the per-voxel
// gradient volume).  packed = false is the layout of a trilinear call that takes the TMA path: only the row-padded
// copy for nx % 4 != 0 lives there.
FwdWs fwd_ws(const dfp_geometry& g, int V, bool grad, int nset = 1, bool packed = true) {
  FwdWs w;
  const VolLayout L = make_layout(g);
  w.gx = (g.nu + kFwdTU - 1) / kFwdTU;
  w.gy = (g.nv + kFwdTV - 1) / kFwdTV;
  w.gy8 = (g.nv + TmaLanes<1>::TV - 1) / TmaLanes<1>::TV;
  size_t o = 0;
  w.off_views = o; o += align_up(sizeof(FwdView) * (size_t)V);
  w.off_dd = o;    o += (g.flags & (DFP_FLAG_DD | DFP_FLAG_SF)) ? align_up(sizeof(DdView) * (size_t)V) : 0;
  w.off_con = o;   o += grad ? align_up(sizeof(FwdContract) * (size_t)V) : 0;
  if (g.flags & (DFP_FLAG_SIDDON | DFP_FLAG_JOSEPH | DFP_FLAG_DD | DFP_FLAG_SF)) packed = true;
  w.off_pvol = o;
  o += packed ? align_up(sizeof(float4) * (size_t)L.px * L.py * L.pz)
              : ((g.nx % 4) ? align_up(sizeof(float) * (size_t)((g.nx + 3) / 4 * 4) * g.ny * g.nz) : 0);
  {
    size_t nblk = (size_t)w.gx * w.gy8;
    if (g.flags & DFP_FLAG_SF) nblk = ((size_t)g.nx * g.ny * g.nz + kSfThreads - 1) / kSfThreads;   // sf_kernel blocks
    w.off_part = o;  o += grad ? align_up(sizeof(float) * 6 * (size_t)nset * V * nblk) : 0;
  }
  // the paper's gradient mode on the TMA path, >= 0.45 voxel per pixel: view lists of the three ray-direction classes and
  // the transposed volume of the views along x (dfp_fwd_tma.cuh, MODE 5 / 6)
  // (taken where a pixel spans >= 0.45 voxel along z; reserved from 0.40 on, and always with explicit view frames, whose
  // pixel pitch is per view)
  const bool classes = grad && nset == 1 && !(g.flags & (DFP_FLAG_GRAD_INTERP | DFP_FLAG_SIDDON | DFP_FLAG_JOSEPH | DFP_FLAG_DD |
                                                         DFP_FLAG_SF | DFP_FLAG_NO_TMA)) &&
                       ((g.flags & DFP_FLAG_VIEW_FRAMES) || (double)g.dv * ((double)g.sad / (double)g.sdd) / (double)g.vz >= 0.40);
  w.off_ids = o;  o += classes ? align_up(sizeof(int) * 3 * (size_t)V) : 0;
  w.off_volt = o; o += classes ? align_up(sizeof(float) * (size_t)g.nx * ((g.ny + 3) / 4 * 4) * g.nz) : 0;
  // sf_kernel<0>: SfFixed (256 bytes) + the 64-bit fixed-point accumulator image
  w.off_fixed = o; o += ((g.flags & DFP_FLAG_SF) && !grad) ? align_up(256 + sizeof(long long) * (size_t)V * g.nu * g.nv) : 0;
  w.total = o;
  return w;
}

constexpr int kBpGradZChunk = 16;
struct BpWs {
  size_t off_views, off_viewsd, off_dd, off_con, off_q, off_part, off_fixed, total;
  int gx, gy, gz;  // voxel tiles (gather path)
  int tx, ty, tz;  // voxel tiles (TMA path)
};
// `packed`: reserve the gather path's 4x packed copy of the projections (false: the layout of a call on the TMA path - only
// the row-padded copy for nu % 4 != 0 lives there; the DD / SF models use neither).
BpWs bp_ws(const dfp_geometry& g, int V, bool grad, bool packed = true) {
  BpWs w;
  w.gx = (g.nx + kBpTX - 1) / kBpTX;
  w.gy = (g.ny + kBpTY - 1) / kBpTY;
  w.gz = grad ? (g.nz + kBpGradZChunk - 1) / kBpGradZChunk : (g.nz + kBpZ - 1) / kBpZ;
  // tiles of the TMA path: 16 x 16 x (16 or 8) voxels; sized for the finer tiling
  w.tx = (g.nx + kBpT - 1) / kBpT;
  w.ty = (g.ny + kBpT - 1) / kBpT;
  w.tz = (g.nz + 7) / 8;
  size_t o = 0;
  w.off_views = o; o += align_up(sizeof(BpView) * (size_t)V);
  w.off_viewsd = o; o += align_up(sizeof(BpViewD) * (size_t)V);
  w.off_dd = o;    o += (g.flags & (DFP_FLAG_DD | DFP_FLAG_SF)) ? align_up(sizeof(DdView) * (size_t)V) : 0;
  w.off_con = o;   o += grad ? align_up(sizeof(BpContract) * (size_t)V) : 0;
  w.off_q = o;
  if (g.flags & (DFP_FLAG_DD | DFP_FLAG_SF)) o += 0;
  else if (packed) o += align_up(sizeof(float4) * (size_t)V * (g.nu + 2 * kPadDet) * (g.nv + 2 * kPadDet));
  else o += (g.nu % 4) ? align_up(sizeof(float) * (size_t)V * ((g.nu + 3) / 4 * 4) * g.nv) : 0;
  w.off_part = o;
  {
    const size_t t_gather = (size_t)w.gx * w.gy * w.gz, t_tma = (size_t)w.tx * w.ty * w.tz;
    size_t tiles = t_gather > t_tma ? t_gather : t_tma;
    if (g.flags & DFP_FLAG_SF) tiles = ((size_t)g.nx * g.ny * g.nz + kSfThreads - 1) / kSfThreads;          // sf_kernel blocks
    if (g.flags & DFP_FLAG_DD) tiles = (size_t)((g.nu + kFwdTU - 1) / kFwdTU) * ((g.nv + kFwdTV - 1) / kFwdTV);   // dd_kernel<3>: pixel tiles
    o += grad ? align_up(sizeof(float) * 6 * (size_t)V * tiles) : 0;
  }
  // dd_kernel<2>: DdFixed (256 bytes) + the 64-bit fixed-point accumulator volume
  w.off_fixed = o; o += ((g.flags & DFP_FLAG_DD) && !grad) ? align_up(256 + sizeof(long long) * (size_t)g.nx * g.ny * g.nz) : 0;
  w.total = o;
  return w;
}

int grid_1d(size_t n, int threads) {
  size_t b = (n + threads - 1) / threads;
  const size_t cap = 148 * 16;           // grid-stride loops: a few waves of the 148 SMs
  return (int)(b < cap ? (b ? b : 1) : cap);
}

int check_common(const dfp_geometry* g, int n_views, const float* angles, const float* poses, const void* a,
                 const void* b, const void* c, void* ws, size_t ws_bytes, size_t need) {
  int st = validate_geometry(g);
  if (st) return st;
  st = validate_views(*g, n_views, angles, poses);
  if (st) return st;
  if (!a || !b || (!c) || !ws) return DFP_ERR_NULL;
  if (!aligned(a, 16) || !aligned(b, 16) || !aligned(c, 16) || !aligned(ws, 256)) return DFP_ERR_ALIGN;
  if (ws_bytes < need) return DFP_ERR_WORKSPACE;
  return DFP_OK;
}

// Which staging box (dfp_fwd_tma.cuh) a trilinear forward call takes for these views: -1 = none, the gather kernels.
// Purely geometric (host): dfp_workspace_bytes_for_views and the call itself must agree on it.
struct FwdChoice { int shape; bool half_tile, wide; };
const int kBoxes[kNumShapes][3] = {{BoxShape<0>::X, BoxShape<0>::Y, BoxShape<0>::Z}, {BoxShape<1>::X, BoxShape<1>::Y, BoxShape<1>::Z},
                                   {BoxShape<2>::X, BoxShape<2>::Y, BoxShape<2>::Z}, {BoxShape<3>::X, BoxShape<3>::Y, BoxShape<3>::Z},
                                   {BoxShape<4>::X, BoxShape<4>::Y, BoxShape<4>::Z}, {BoxShape<5>::X, BoxShape<5>::Y, BoxShape<5>::Z},
                                   {BoxShape<6>::X, BoxShape<6>::Y, BoxShape<6>::Z}, {BoxShape<7>::X, BoxShape<7>::Y, BoxShape<7>::Z}};
FwdChoice fwd_choice(const dfp_geometry& g, const FwdGeom& G, const std::vector<FwdView>& hv, const std::vector<ViewFrame>& hf,
                     int V, bool grad, bool plain_grad = false) {
  // forward: shapes 0, 1, 2 (16 x 16-pixel tiles) - with the odd-extent boxes 4, 5 first where a pixel spans >= 0.45
  // voxel along z (bank conflicts, dfp_fwd_tma.cuh); gradient: shapes 3, 2 (16 x 8-pixel tiles)
#ifndef DFP_WIDE_A
#define DFP_WIDE_A 4
#define DFP_WIDE_B 5
#endif
  // (the paper's gradient mode: the 14-slice box 7, five blocks per SM, before the 16-slice box 3)
  static const int kOrderFwd[3] = {0, 1, 2}, kOrderFwdWide[5] = {DFP_WIDE_A, DFP_WIDE_B, 0, 1, 2}, kOrderGrad[2] = {3, 2},
                   kOrderGradPlain[3] = {7, 3, 2};
  FwdChoice c{-1, false, false};
  c.wide = hf[0].vlen * ((double)g.sad / hf[0].sdd) / (double)g.vz >= 0.45;
  if (g.flags & DFP_FLAG_NO_TMA) return c;
  const int* order = grad ? (plain_grad ? kOrderGradPlain : kOrderGrad) : (c.wide ? kOrderFwdWide : kOrderFwd);
  const int n_order = grad ? (plain_grad ? 3 : 2) : (c.wide ? 5 : 3);
  const int TU = grad ? TmaLanes<1>::TU : TmaLanes<0>::TU, TV = grad ? TmaLanes<1>::TV : TmaLanes<0>::TV;
  for (int i = 0; i < n_order && c.shape < 0; ++i) {
    bool fits = true;
    for (int v = 0; fits && v < V; ++v) fits = tma_view_fits(g, G, hv[v], hf[v], grad, kBoxes[order[i]], TU, TV);
    if (fits) c.shape = order[i];
  }
  // last resort before the gather kernels (coarse pixels on fine voxels, e.g. C1's forward call: 1.2 voxels per
  // pixel): the largest box with chunks of two samples - short chunks, but no packed copy of the volume
  if (c.shape < 0) {
    bool fits = true;
    for (int v = 0; fits && v < V; ++v) fits = tma_view_fits(g, G, hv[v], hf[v], grad, kBoxes[2], TU, TV, 2);
    if (fits) c.shape = 2;
  }
  if (c.shape < 0 && !grad) {          // forward only: the same box under a 16 x 8-pixel tile (MODE 4)
    bool fits = true;
    for (int v = 0; fits && v < V; ++v)
      fits = tma_view_fits(g, G, hv[v], hf[v], false, kBoxes[2], TmaLanes<4>::TU, TmaLanes<4>::TV, 2);
    if (fits) { c.shape = 2; c.half_tile = true; }
  }
  return c;
}

// op = DFP_OP_FORWARD (d_out = projections), DFP_OP_FORWARD_POSE_GRAD (d_up = upstream, d_out = gradients) or
// DFP_OP_FORWARD_FUSED (d_up = target b, d_out = moments [V][3][6], d_proj = projections)
int run_forward_slice(const dfp_geometry* g, int V, const float* angles, const float* poses, const float* d_vol,
                      const float* d_up, float* d_out, void* d_ws, size_t ws_bytes, cudaStream_t s, int op,
                      float* d_proj) {
  if (!g) return DFP_ERR_NULL;
  int st = validate_geometry(g);
  if (st) return st;
  const bool grad = op != DFP_OP_FORWARD, fused = op == DFP_OP_FORWARD_FUSED;
  if (fused && (!d_proj || !aligned(d_proj, 16))) return d_proj ? DFP_ERR_ALIGN : DFP_ERR_NULL;
  if (fused && (g->flags & DFP_FLAG_GRAD_INTERP)) return DFP_ERR_DIMS;      // fused moments: central differences only
  const bool siddon = (g->flags & DFP_FLAG_SIDDON) != 0, joseph = (g->flags & DFP_FLAG_JOSEPH) != 0,
             dd = (g->flags & DFP_FLAG_DD) != 0, sf = (g->flags & DFP_FLAG_SF) != 0;
  // Siddon / Joseph / distance-driven / separable-footprint weights: the two plain calls only, one model at a time
  if ((siddon || joseph || dd || sf) &&
      (fused || (g->flags & DFP_FLAG_GRAD_INTERP) || (int)siddon + (int)joseph + (int)dd + (int)sf > 1))
    return DFP_ERR_DIMS;
  const int nset = fused ? 3 : 1;
  st = check_common(g, V, angles, poses, d_vol, d_out, grad ? (const void*)d_up : (const void*)d_vol, d_ws,
                        ws_bytes, 0);          // everything but the workspace size, which depends on the path
  if (st) return st;
  const bool interp = grad && (g->flags & DFP_FLAG_GRAD_INTERP);
  const FwdGeom G = make_fwd_geom(*g, grad, interp);
  std::vector<FwdView> hv((size_t)V);
  std::vector<FwdContract> hc(grad ? (size_t)V : 0);
  std::vector<ViewFrame> hf((size_t)V);
  for (int v = 0; v < V; ++v) {
    hf[v] = make_frame(*g, angles, v);
    make_fwd_view(hf[v], poses + 6 * v, &hv[v], grad ? &hc[v] : nullptr);
  }
  char* base = static_cast<char*>(d_ws);
  // The kernel path first (host geometry only): a trilinear call whose views fit a staging box needs no packed copy of
  // the volume, and its workspace is laid out without one (dfp_workspace_bytes_for_views returns that size).
  const bool plain = !(siddon || joseph || dd || sf);
  const FwdChoice choice = plain ? fwd_choice(*g, G, hv, hf, V, grad, grad) : FwdChoice{-1, false, false};
  const FwdWs w_tma = fwd_ws(*g, V, grad, nset, false);
  CUtensorMap vol_map;
  // nx % 4 != 0: the TMA kernels read a copy of the volume with 16-byte-aligned rows (1x the volume, at off_pvol - the
  // same offset in both layouts)
  const int vpitch = pitch4(g->nx);
  const float* tma_vol = vpitch == g->nx ? d_vol : reinterpret_cast<const float*>(base + w_tma.off_pvol);
  const bool tma = choice.shape >= 0 && make_volume_map(*g, tma_vol, vpitch, kBoxes[choice.shape][0], kBoxes[choice.shape][1],
                                                        kBoxes[choice.shape][2], &vol_map);
  const FwdWs w = tma ? w_tma : fwd_ws(*g, V, grad, nset, true);
  if (ws_bytes < w.total) return DFP_ERR_WORKSPACE;
  FwdView* dv = reinterpret_cast<FwdView*>(base + w.off_views);
  FwdContract* dc = reinterpret_cast<FwdContract*>(base + w.off_con);
  float4* pvol = reinterpret_cast<float4*>(base + w.off_pvol);
  float* part = reinterpret_cast<float*>(base + w.off_part);
  g_launches = 0;
  DFP_CUDA(upload_async(dv, hv.data(), sizeof(FwdView) * V, s), "view upload");
  if (grad) DFP_CUDA(upload_async(dc, hc.data(), sizeof(FwdContract) * V, s), "view upload");
  const dim3 grid(w.gx, w.gy, V);
  if (sf) {                 // separable-footprint weights (dfp_sf.cuh): voxel-driven
    std::vector<DdView> hd((size_t)V);
    for (int v = 0; v < V; ++v) make_dd_view(*g, hf[v], poses + 6 * v, &hd[v]);
    DdView* ddv = reinterpret_cast<DdView*>(base + w.off_dd);
    DFP_CUDA(upload_async(ddv, hd.data(), sizeof(DdView) * V, s), "view upload");
    const DdGeom DG = make_dd_geom(*g);
    const unsigned nblk = (unsigned)(((size_t)g->nx * g->ny * g->nz + kSfThreads - 1) / kSfThreads);
    g_path = DFP_PATH_GATHER;
    if (!grad) {
      const size_t npix = (size_t)V * g->nu * g->nv, nvox = (size_t)g->nx * g->ny * g->nz;
      SfFixed* fx = reinterpret_cast<SfFixed*>(base + w.off_fixed);
      long long* acc = reinterpret_cast<long long*>(base + w.off_fixed + 256);
      DFP_CUDA(cudaMemsetAsync(fx, 0, 256 + sizeof(long long) * npix, s), "cudaMemsetAsync");
      sf_maxabs_kernel<<<grid_1d(nvox, 256), 256, 0, s>>>(d_vol, nvox, fx);
      time_begin(s);
      sf_kernel<0><<<nblk, kSfThreads, 0, s>>>(DG, V, 0, ddv, d_vol, nullptr, nullptr, fx, reinterpret_cast<float*>(acc));
      time_end(s);
      sf_fixed_to_float_kernel<<<grid_1d(npix, 256), 256, 0, s>>>(DG, acc, fx, npix, d_out);
      g_launches = 3;
    } else {
      time_begin(s);
      sf_kernel<2><<<nblk, kSfThreads, 0, s>>>(DG, V, 0, ddv, d_vol, d_up, nullptr, nullptr, part);
      time_end(s);
      fwd_contract_kernel<<<V, 256, 0, s>>>((int)nblk, part, dc, d_out);
      g_launches = 2;
    }
    DFP_CUDA(cudaGetLastError(), "forward launch (separable-footprint weights)");
    return DFP_OK;
  }
  if (dd) {                 // distance-driven weights (dfp_dd.cuh)
    std::vector<DdView> hd((size_t)V);
    for (int v = 0; v < V; ++v) make_dd_view(*g, hf[v], poses + 6 * v, &hd[v]);
    DdView* ddv = reinterpret_cast<DdView*>(base + w.off_dd);
    DFP_CUDA(upload_async(ddv, hd.data(), sizeof(DdView) * V, s), "view upload");
    const DdGeom DG = make_dd_geom(*g);
    const GradBricks GB = GradBricks::make(g->nx, g->ny, g->nz);
    g_path = DFP_PATH_GATHER;
    time_begin(s);
    if (!grad) {
      dd_kernel<0><<<grid, kFwdThreads, 0, s>>>(DG, ddv, d_vol, nullptr, GB, nullptr, nullptr, 0, d_out);
      time_end(s);
      g_launches = 1;
    } else {
      const int gb = (int)std::min<size_t>((GB.cells() + 255) / 256, (size_t)148 * 64);
      grad_volume_kernel<<<gb, 256, 0, s>>>(GB, G.sgx, G.sgy, G.sgz, d_vol, pvol);
      dd_kernel<1><<<grid, kFwdThreads, 0, s>>>(DG, ddv, d_vol, pvol, GB, d_up, nullptr, 0, part);
      time_end(s);
      fwd_contract_kernel<<<V, 256, 0, s>>>(w.gx * w.gy, part, dc, d_out);
      g_launches = 3;
    }
    DFP_CUDA(cudaGetLastError(), "forward launch (distance-driven weights)");
    return DFP_OK;
  }
  if (siddon || joseph) {   // other weight models (dfp_siddon.cuh, dfp_joseph.cuh): straight over the caller's volume
    g_path = DFP_PATH_GATHER;
    time_begin(s);
    if (!grad) {
      if (siddon) siddon_fwd_kernel<<<grid, kFwdThreads, 0, s>>>(G, dv, d_vol, d_out);
      else {
        pack_volume_kernel<<<grid_1d((size_t)G.L.px * G.L.py * G.L.pz, 256), 256, 0, s>>>(G.L, d_vol, pvol);
        joseph_fwd_kernel<<<grid, kFwdThreads, 0, s>>>(G, dv, pvol, d_out);
        ++g_launches;
      }
      time_end(s);
      ++g_launches;
    } else {
      // per-voxel g_j once per call, into the workspace region the packed volume of the trilinear path would take
      const GradBricks B = GradBricks::make(g->nx, g->ny, g->nz);
      const int gb = (int)std::min<size_t>((B.cells() + 255) / 256, (size_t)148 * 64);
      grad_volume_kernel<<<gb, 256, 0, s>>>(B, G.sgx, G.sgy, G.sgz, d_vol, pvol);
      if (siddon) siddon_grad_kernel<<<grid, kFwdThreads, 0, s>>>(G, dv, pvol, d_up, part);
      else joseph_grad_kernel<<<grid, kFwdThreads, 0, s>>>(G, dv, pvol, d_up, part);
      time_end(s);
      fwd_contract_kernel<<<V, 256, 0, s>>>(w.gx * w.gy, part, dc, d_out);
      g_launches += 3;
    }
    DFP_CUDA(cudaGetLastError(), "forward launch (Siddon / Joseph weights)");
    return DFP_OK;
  }
  // TMA-staged path when every view's tiles fit a staging box: the first box of the op's list that holds them (fwd_choice)
  const int shape = choice.shape;
  const bool half_tile = choice.half_tile, wide = choice.wide;
  const int TU = grad ? TmaLanes<1>::TU : TmaLanes<0>::TU, TV = grad ? TmaLanes<1>::TV : TmaLanes<0>::TV;
  g_path = tma ? DFP_PATH_TMA : DFP_PATH_GATHER;
  if (tma) {
    DFP_CUDA(ensure_smem_attributes(), "cudaFuncSetAttribute");
    if (tma_vol != d_vol) {
      DFP_CUDA(cudaMemcpy2DAsync(pvol, (size_t)vpitch * 4, d_vol, (size_t)g->nx * 4, (size_t)g->nx * 4, (size_t)g->ny * g->nz,
                                 cudaMemcpyDeviceToDevice, s), "cudaMemcpy2DAsync (row-aligned volume)");
    }
    time_begin(s);
    // 1-D grid, one block per (view, tile), ordered view group -> tile -> view (dfp_fwd_tma.cuh: fwd_block)
    const FwdGrid Qf{V, w.gx, w.gy, V, nullptr}, Qg{V, w.gx, w.gy8, V, nullptr};
    const unsigned nbf = (unsigned)V * w.gx * w.gy, nbg = (unsigned)V * w.gx * w.gy8;
    if (fused && shape == 7)
      fwd_tma_kernel<3, 7><<<nbg, TmaLanes<3>::THREADS, tma_smem_bytes<7>(), s>>>(G, Qg, dv, vol_map, d_up, part, d_proj);
    else if (fused && shape == 3)
      fwd_tma_kernel<3, 3><<<nbg, TmaLanes<3>::THREADS, tma_smem_bytes<3>(), s>>>(G, Qg, dv, vol_map, d_up, part, d_proj);
    else if (fused)
      fwd_tma_kernel<3, 2><<<nbg, TmaLanes<3>::THREADS, tma_smem_bytes<2>(), s>>>(G, Qg, dv, vol_map, d_up, part, d_proj);
    else if (grad && interp && shape == 7)
      fwd_tma_kernel<2, 7><<<nbg, TmaLanes<2>::THREADS, tma_smem_bytes<7>(), s>>>(G, Qg, dv, vol_map, d_up, part, nullptr);
    else if (grad && interp && shape == 3)
      fwd_tma_kernel<2, 3><<<nbg, TmaLanes<2>::THREADS, tma_smem_bytes<3>(), s>>>(G, Qg, dv, vol_map, d_up, part, nullptr);
    else if (grad && interp)
      fwd_tma_kernel<2, 2><<<nbg, TmaLanes<2>::THREADS, tma_smem_bytes<2>(), s>>>(G, Qg, dv, vol_map, d_up, part, nullptr);
    else if (grad && (shape == 3 || shape == 7) && wide) {
      // Views by the in-plane direction of their central ray (voxel-index units): along y -> MODE 5, along x -> MODE 6 on
      // the transposed volume, near the diagonals (or where the MODE 5 / 6 box does not hold the view's tiles) -> MODE 1.
      std::vector<int> ids[4];
      CUtensorMap map_y, map_x, map_d;
      const bool ok_y = make_volume_map(*g, tma_vol, vpitch, kBoxes[6][0], kBoxes[6][1], kBoxes[6][2], &map_y);
      const bool ok_d = make_volume_map(*g, tma_vol, vpitch, kBoxes[7][0], kBoxes[7][1], kBoxes[7][2], &map_d);
      float* volt = reinterpret_cast<float*>(base + w.off_volt);
      const int tpitch = pitch4(g->ny);               // rows of the transposed volume [z][x][y], 16-byte aligned
      bool ok_x;
      {
        dfp_geometry gt = *g;
        gt.nx = g->ny; gt.ny = g->nx;
        ok_x = make_volume_map(gt, volt, tpitch, kBoxes[6][0], kBoxes[6][1], kBoxes[6][2], &map_x);
      }
      const int box_y[3] = {kBoxes[6][0], kBoxes[6][1], kBoxes[6][2]}, box_x[3] = {kBoxes[6][1], kBoxes[6][0], kBoxes[6][2]};
      for (int v = 0; v < V; ++v) {
        const double cu = 0.5 * (g->nu - 1), cv = 0.5 * (g->nv - 1);
        const double ex = std::fabs(hv[v].d0[0] + cu * hv[v].du[0] + cv * hv[v].dv[0]) / g->vx;
        const double ey = std::fabs(hv[v].d0[1] + cu * hv[v].du[1] + cv * hv[v].dv[1]) / g->vy;
        int c = 0;
        if (ok_y && ey * kClassTan > ex && tma_view_fits(*g, G, hv[v], hf[v], true, box_y, TU, TV)) c = 1;
        if (ok_x && ex * kClassTan > ey && tma_view_fits(*g, G, hv[v], hf[v], true, box_x, TU, TV, kMinChunk, 1)) c = 2;
        // the rest: the 8 x 2 x 2 kernel, on the 14-slice box (five blocks per SM) where the view's tiles fit it
        if (c == 0 && ok_d && tma_view_fits(*g, G, hv[v], hf[v], true, kBoxes[7], TU, TV)) c = 3;
        ids[c].push_back(v);
      }
      int* dids = reinterpret_cast<int*>(base + w.off_ids);
      std::vector<int> all;
      for (int c = 0; c < 4; ++c) all.insert(all.end(), ids[c].begin(), ids[c].end());
      DFP_CUDA(upload_async(dids, all.data(), sizeof(int) * all.size(), s), "view upload");
      const int* d0 = dids, *d1 = dids + ids[0].size(), *d2 = d1 + ids[1].size(), *d3 = d2 + ids[2].size();
      const unsigned tiles = (unsigned)w.gx * w.gy8;
      if (!ids[0].empty())
        fwd_tma_kernel<1, 3><<<(unsigned)ids[0].size() * tiles, TmaLanes<1>::THREADS, tma_smem_bytes<3>(), s>>>(
            G, FwdGrid{(int)ids[0].size(), w.gx, w.gy8, V, d0}, dv, vol_map, d_up, part, nullptr);
      if (!ids[3].empty()) {
        fwd_tma_kernel<1, 7><<<(unsigned)ids[3].size() * tiles, TmaLanes<1>::THREADS, tma_smem_bytes<7>(), s>>>(
            G, FwdGrid{(int)ids[3].size(), w.gx, w.gy8, V, d3}, dv, map_d, d_up, part, nullptr);
        ++g_launches;
      }
      if (!ids[1].empty()) {
        fwd_tma_kernel<5, 6><<<(unsigned)ids[1].size() * tiles, TmaLanes<5>::THREADS, tma_smem_bytes<6>(), s>>>(
            G, FwdGrid{(int)ids[1].size(), w.gx, w.gy8, V, d1}, dv, map_y, d_up, part, nullptr);
        ++g_launches;
      }
      if (!ids[2].empty()) {
        transpose_xy_kernel<<<dim3((g->nx + 31) / 32, (g->ny + 31) / 32, g->nz), dim3(32, 8), 0, s>>>(g->nx, g->ny, tpitch, d_vol, volt);
        fwd_tma_kernel<6, 6><<<(unsigned)ids[2].size() * tiles, TmaLanes<6>::THREADS, tma_smem_bytes<6>(), s>>>(
            G, FwdGrid{(int)ids[2].size(), w.gx, w.gy8, V, d2}, dv, map_x, d_up, part, nullptr);
        g_launches += 2;
      }
      if (ids[0].empty()) --g_launches;        // (the common count below adds one launch)
    } else if (grad && shape == 7)
      fwd_tma_kernel<1, 7><<<nbg, TmaLanes<1>::THREADS, tma_smem_bytes<7>(), s>>>(G, Qg, dv, vol_map, d_up, part, nullptr);
    else if (grad && shape == 3)
      fwd_tma_kernel<1, 3><<<nbg, TmaLanes<1>::THREADS, tma_smem_bytes<3>(), s>>>(G, Qg, dv, vol_map, d_up, part, nullptr);
    else if (grad)
      fwd_tma_kernel<1, 2><<<nbg, TmaLanes<1>::THREADS, tma_smem_bytes<2>(), s>>>(G, Qg, dv, vol_map, d_up, part, nullptr);
    else if (half_tile)
      fwd_tma_kernel<4, 2><<<(unsigned)V * w.gx * ((g->nv + 7) / 8), TmaLanes<4>::THREADS, tma_smem_bytes<2>(), s>>>(
          G, FwdGrid{V, w.gx, (g->nv + 7) / 8, V, nullptr}, dv, vol_map, nullptr, d_out, nullptr);
    else if (shape == 0)
      fwd_tma_kernel<0, 0><<<nbf, TmaLanes<0>::THREADS, tma_smem_bytes<0>(), s>>>(G, Qf, dv, vol_map, nullptr, d_out, nullptr);
    else if (shape == 1)
      fwd_tma_kernel<0, 1><<<nbf, TmaLanes<0>::THREADS, tma_smem_bytes<1>(), s>>>(G, Qf, dv, vol_map, nullptr, d_out, nullptr);
    else if (shape == 4)
      fwd_tma_kernel<0, 4><<<nbf, TmaLanes<0>::THREADS, tma_smem_bytes<4>(), s>>>(G, Qf, dv, vol_map, nullptr, d_out, nullptr);
    else if (shape == 5)
      fwd_tma_kernel<0, 5><<<nbf, TmaLanes<0>::THREADS, tma_smem_bytes<5>(), s>>>(G, Qf, dv, vol_map, nullptr, d_out, nullptr);
    else
      fwd_tma_kernel<0, 2><<<nbf, TmaLanes<0>::THREADS, tma_smem_bytes<2>(), s>>>(G, Qf, dv, vol_map, nullptr, d_out, nullptr);
    time_end(s);
    ++g_launches;
    const int nblk8 = w.gx * w.gy8;
    for (int set = 0; grad && set < nset; ++set) {       // fused: one contraction per weight set -> moments[v][set][6]
      fwd_contract_kernel<<<V, 256, 0, s>>>(nblk8, part + (size_t)set * V * nblk8 * 6, dc, d_out, 6 * nset, 6 * set);
      ++g_launches;
    }
    DFP_CUDA(cudaGetLastError(), "forward launch (TMA path)");
    return DFP_OK;
  }
  const size_t ncell = (size_t)G.L.px * G.L.py * G.L.pz;
  pack_volume_kernel<<<grid_1d(ncell, 256), 256, 0, s>>>(G.L, d_vol, pvol);
  ++g_launches;
  if (fused) {
    // gather fallback of the fused call, composed from the two gather kernels: projections, then the three
    // weight sets (unit, l, b) one gradient pass each (this path trades the fusion for generality)
    const int nblk = w.gx * w.gy;
    fwd_project_kernel<<<grid, kFwdThreads, 0, s>>>(G, dv, pvol, d_proj);
    ++g_launches;
    const float* ups[3] = {nullptr, d_proj, d_up};
    time_begin(s);
    for (int set = 0; set < 3; ++set) {
      fwd_grad_kernel<0><<<grid, kFwdThreads, 0, s>>>(G, dv, pvol, ups[set], part + (size_t)set * V * nblk * 6);
      fwd_contract_kernel<<<V, 256, 0, s>>>(nblk, part + (size_t)set * V * nblk * 6, dc, d_out, 18, 6 * set);
      g_launches += 2;
    }
    time_end(s);
  } else if (!grad) {
    time_begin(s);
    fwd_project_kernel<<<grid, kFwdThreads, 0, s>>>(G, dv, pvol, d_out);
    time_end(s);
    ++g_launches;
  } else {
    time_begin(s);
    if (interp) fwd_grad_kernel<1><<<grid, kFwdThreads, 0, s>>>(G, dv, pvol, d_up, part);
    else fwd_grad_kernel<0><<<grid, kFwdThreads, 0, s>>>(G, dv, pvol, d_up, part);
    time_end(s);
    fwd_contract_kernel<<<V, 256, 0, s>>>(w.gx * w.gy, part, dc, d_out);
    g_launches += 2;
  }
  DFP_CUDA(cudaGetLastError(), "forward launch");
  return DFP_OK;
}

// Which patch menu entry (dfp_bp_tma.cuh) and tile depth a voxel-driven back-projection call takes for these views:
// kmax < 0 = the gather kernels.  Host geometry only (dfp_workspace_bytes_for_views and the call must agree).
struct BpChoice { int kmax, TZ; };
BpChoice bp_choice(const dfp_geometry& g, const BpGeom& G, const std::vector<BpView>& hv, int V, bool grad) {
  BpChoice c{-1, 16};
  if (g.flags & DFP_FLAG_NO_TMA) return c;
  for (c.TZ = 16; c.TZ >= 8 && c.kmax < 0; c.TZ >>= 1) {
    c.kmax = 0;
    for (int v = 0; v < V && c.kmax >= 0; ++v) {
      const int k = bp_view_patch(G, hv[v], c.TZ, grad ? 1 : 0);
      c.kmax = k < 0 ? -1 : (k > c.kmax ? k : c.kmax);
    }
    if (c.kmax >= 0 && bp_num_stages(c.kmax) < 2) c.kmax = -1;      // a single stage would serialise TMA and compute
    if (c.kmax >= 0) break;
  }
  return c;
}

int run_backproject_slice(const dfp_geometry* g, int V, const float* angles, const float* poses, const float* d_proj,
                          const float* d_up, float* d_out, void* d_ws, size_t ws_bytes, cudaStream_t s, bool grad) {
  if (!g) return DFP_ERR_NULL;
  int st = validate_geometry(g);
  if (st) return st;
  if ((g->flags & (DFP_FLAG_DD | DFP_FLAG_SF)) &&
      (g->bp_weight != 0 || (g->flags & (DFP_FLAG_GRAD_INTERP | DFP_FLAG_SIDDON | DFP_FLAG_JOSEPH)) ||
       (g->flags & (DFP_FLAG_DD | DFP_FLAG_SF)) == (DFP_FLAG_DD | DFP_FLAG_SF)))
    return DFP_ERR_DIMS;     // the DD / SF back-projectors are plain transposes: unit weight, central differences only
  st = check_common(g, V, angles, poses, d_proj, d_out, grad ? (const void*)d_up : (const void*)d_proj, d_ws,
                        ws_bytes, 0);          // everything but the workspace size, which depends on the path
  if (st) return st;
  const BpGeom G = make_bp_geom(*g);
  std::vector<BpView> hv((size_t)V);
  std::vector<BpViewD> hvd((size_t)V);
  std::vector<BpContract> hc(grad ? (size_t)V : 0);
  for (int v = 0; v < V; ++v)
    make_bp_view(*g, G, make_frame(*g, angles, v), poses + 6 * v, &hv[v], grad ? &hc[v] : nullptr, &hvd[v]);
  char* base = static_cast<char*>(d_ws);
  // The kernel path first (host geometry only): on the TMA path the workspace holds no packed copy of the projections
  const bool vd = !(g->flags & (DFP_FLAG_DD | DFP_FLAG_SF));
  const BpChoice choice = vd ? bp_choice(*g, G, hv, V, grad) : BpChoice{-1, 16};
  const BpWs w_tma = bp_ws(*g, V, grad, false);
  PatchMaps maps;
  // nu % 4 != 0: the TMA kernels read a copy of the projections with 16-byte-aligned rows (at off_q, the same offset in
  // both layouts)
  const int ppitch = pitch4(g->nu);
  const float* tma_proj = ppitch == g->nu ? d_proj : reinterpret_cast<const float*>(base + w_tma.off_q);
  const bool tma = choice.kmax >= 0 && make_proj_maps(*g, V, tma_proj, ppitch, choice.kmax, &maps);
  const BpWs w = tma ? w_tma : bp_ws(*g, V, grad, true);
  if (ws_bytes < w.total) return DFP_ERR_WORKSPACE;
  BpView* dv = reinterpret_cast<BpView*>(base + w.off_views);
  BpViewD* dvd = reinterpret_cast<BpViewD*>(base + w.off_viewsd);
  BpContract* dc = reinterpret_cast<BpContract*>(base + w.off_con);
  float4* q = reinterpret_cast<float4*>(base + w.off_q);
  float* part = reinterpret_cast<float*>(base + w.off_part);
  g_launches = 0;
  g_path = DFP_PATH_GATHER;
  DFP_CUDA(upload_async(dv, hv.data(), sizeof(BpView) * V, s), "view upload");
  DFP_CUDA(upload_async(dvd, hvd.data(), sizeof(BpViewD) * V, s), "view upload");
  if (grad) DFP_CUDA(upload_async(dc, hc.data(), sizeof(BpContract) * V, s), "view upload");
  if (g->flags & DFP_FLAG_SF) {   // separable-footprint weights (dfp_sf.cuh): the exact transpose of the SF forward projector
    std::vector<DdView> hd((size_t)V);
    for (int v = 0; v < V; ++v) make_dd_view(*g, make_frame(*g, angles, v), poses + 6 * v, &hd[v]);
    DdView* ddv = reinterpret_cast<DdView*>(base + w.off_dd);
    DFP_CUDA(upload_async(ddv, hd.data(), sizeof(DdView) * V, s), "view upload");
    const DdGeom DG = make_dd_geom(*g);
    const unsigned nblk = (unsigned)(((size_t)g->nx * g->ny * g->nz + kSfThreads - 1) / kSfThreads);
    time_begin(s);
    if (!grad) {
      sf_kernel<1><<<nblk, kSfThreads, 0, s>>>(DG, V, (g->flags & DFP_FLAG_ACCUMULATE) ? 1 : 0, ddv, nullptr, d_proj, nullptr, nullptr, d_out);
      time_end(s);
      g_launches = 1;
    } else {
      sf_kernel<3><<<nblk, kSfThreads, 0, s>>>(DG, V, 0, ddv, nullptr, d_proj, d_up, nullptr, part);
      time_end(s);
      bp_contract_kernel<<<V, 256, 0, s>>>((int)nblk, V, part, dc, d_out);
      g_launches = 2;
    }
    DFP_CUDA(cudaGetLastError(), "back-projection launch (separable-footprint weights)");
    return DFP_OK;
  }
  if (g->flags & DFP_FLAG_DD) {   // distance-driven weights (dfp_dd.cuh): the exact transpose of the DD forward projector
    std::vector<DdView> hd((size_t)V);
    for (int v = 0; v < V; ++v) make_dd_view(*g, make_frame(*g, angles, v), poses + 6 * v, &hd[v]);
    DdView* ddv = reinterpret_cast<DdView*>(base + w.off_dd);
    DFP_CUDA(upload_async(ddv, hd.data(), sizeof(DdView) * V, s), "view upload");
    const DdGeom DG = make_dd_geom(*g);
    const dim3 grid((g->nu + kFwdTU - 1) / kFwdTU, (g->nv + kFwdTV - 1) / kFwdTV, V);
    const GradBricks GB{};
    if (!grad) {
      // fixed-point head-room: sum_i a^ij <= (pixels of the call) x the longest slab length v_a / |e_a| (a normalised
      // overlap is <= 1); |e_a| is smallest at a detector corner
      double Lmax = 0.0;
      for (int v = 0; v < V; ++v) {
        const DdView& D = hd[v];
        double cmin = 1.0;
        for (int c = 0; c < 4; ++c) {
          const double u = (c & 1) ? g->nu - 0.5 : -0.5, vv = (c & 2) ? g->nv - 0.5 : -0.5;
          double d[3], n2 = 0.0;
          for (int x = 0; x < 3; ++x) { d[x] = D.X00[x] + u * D.Uo[x] + vv * D.Vo[x] - D.so[x]; n2 += d[x] * d[x]; }
          cmin = std::min(cmin, std::fabs(d[D.a]) / std::sqrt(n2 > 0 ? n2 : 1.0));
        }
        const double va = D.a == 0 ? g->vx : (D.a == 1 ? g->vy : g->vz);
        Lmax = std::max(Lmax, va / std::max(cmin, 1e-6));
      }
      const int hb = (int)std::ceil(std::log2(Lmax * (double)g->nu * g->nv * V)) + 1;
      const size_t npix = (size_t)V * g->nu * g->nv, nvox = (size_t)g->nx * g->ny * g->nz;
      DdFixed* fx = reinterpret_cast<DdFixed*>(base + w.off_fixed);
      long long* acc = reinterpret_cast<long long*>(base + w.off_fixed + 256);
      DFP_CUDA(cudaMemsetAsync(fx, 0, 256 + sizeof(long long) * nvox, s), "cudaMemsetAsync");
      dd_maxabs_kernel<<<grid_1d(npix, 256), 256, 0, s>>>(d_proj, npix, fx);
      time_begin(s);
      dd_kernel<2><<<grid, kFwdThreads, 0, s>>>(DG, ddv, nullptr, nullptr, GB, d_proj, fx, hb, reinterpret_cast<float*>(acc));
      time_end(s);
      dd_fixed_to_float_kernel<<<grid_1d(nvox, 256), 256, 0, s>>>(acc, fx, hb, nvox, (g->flags & DFP_FLAG_ACCUMULATE) ? 1 : 0, d_out);
      g_launches = 3;
    } else {
      time_begin(s);
      dd_kernel<3><<<grid, kFwdThreads, 0, s>>>(DG, ddv, d_up, nullptr, GB, d_proj, nullptr, 0, part);
      time_end(s);
      bp_contract_kernel<<<V, 256, 0, s>>>((int)(grid.x * grid.y), V, part, dc, d_out);
      g_launches = 2;
    }
    DFP_CUDA(cudaGetLastError(), "back-projection launch (distance-driven weights)");
    return DFP_OK;
  }
  // TMA-staged path: every voxel in front of the source, patches fit the menu (bp_choice)
  const int kmax = choice.kmax, TZ = choice.TZ;
  if (tma) {
    const int stage_words = bp_stage_words(kmax), n_stages = bp_num_stages(kmax);
    const int smem = stage_words * 4 * n_stages;
    DFP_CUDA(ensure_smem_attributes(), "cudaFuncSetAttribute");
    if (tma_proj != d_proj) {
      DFP_CUDA(cudaMemcpy2DAsync(base + w.off_q, (size_t)ppitch * 4, d_proj, (size_t)g->nu * 4, (size_t)g->nu * 4,
                                 (size_t)g->nv * V, cudaMemcpyDeviceToDevice, s), "cudaMemcpy2DAsync (row-aligned projections)");
    }
    const dim3 tgrid(w.tx, w.ty, (g->nz + TZ - 1) / TZ);
    g_path = DFP_PATH_TMA;
#define DFP_BP_ARGS <<<tgrid, kBpTmaThreads, smem, s>>>(G, V, dvd, maps, kmax, stage_words, n_stages
    time_begin(s);
    if (!grad) {
      if (G.bp_weight) { if (TZ == 16) bp_tma_kernel<1, 16> DFP_BP_ARGS, d_out); else bp_tma_kernel<1, 8> DFP_BP_ARGS, d_out); }
      else { if (TZ == 16) bp_tma_kernel<0, 16> DFP_BP_ARGS, d_out); else bp_tma_kernel<0, 8> DFP_BP_ARGS, d_out); }
      time_end(s);
      ++g_launches;
    } else {
      const bool dw = G.bp_weight && (G.flags & DFP_FLAG_DW);
      const bool interp = (G.flags & DFP_FLAG_GRAD_INTERP) != 0;
#define DFP_BP_GRAD(W, D)                                                                            \
  do {                                                                                               \
    if (TZ == 16 && !interp) bp_grad_tma_kernel<W, D, 16, 0> DFP_BP_ARGS, d_up, part);               \
    else if (TZ == 16) bp_grad_tma_kernel<W, D, 16, 1> DFP_BP_ARGS, d_up, part);                     \
    else if (!interp) bp_grad_tma_kernel<W, D, 8, 0> DFP_BP_ARGS, d_up, part);                       \
    else bp_grad_tma_kernel<W, D, 8, 1> DFP_BP_ARGS, d_up, part);                                    \
  } while (0)
      if (!G.bp_weight) DFP_BP_GRAD(0, 0);
      else if (!dw) DFP_BP_GRAD(1, 0);
      else DFP_BP_GRAD(1, 1);
#undef DFP_BP_GRAD
      time_end(s);
      bp_contract_kernel<<<V, 256, 0, s>>>(tgrid.x * tgrid.y * tgrid.z, V, part, dc, d_out);
      g_launches += 2;
    }
#undef DFP_BP_ARGS
    DFP_CUDA(cudaGetLastError(), "back-projection launch (TMA path)");
    return DFP_OK;
  }
  const size_t ncell = (size_t)V * G.pu * G.pv;
  pack_proj_kernel<<<grid_1d(ncell, 256), 256, 0, s>>>(G.nu, G.nv, G.pu, G.pv, (size_t)V, d_proj, q);
  ++g_launches;
  const dim3 grid(w.gx, w.gy, w.gz);
  if (!grad) {
    time_begin(s);
    if (G.bp_weight) bp_kernel<1><<<grid, kBpThreads, 0, s>>>(G, V, dv, q, d_out);
    else bp_kernel<0><<<grid, kBpThreads, 0, s>>>(G, V, dv, q, d_out);
    time_end(s);
    ++g_launches;
  } else {
    const bool dw = G.bp_weight && (G.flags & DFP_FLAG_DW);
    time_begin(s);
    const bool interp = (G.flags & DFP_FLAG_GRAD_INTERP) != 0;
#define DFP_BP_GRAD(W, D)                                                                                       \
  do {                                                                                                          \
    if (interp) bp_grad_kernel<W, D, 1><<<grid, kBpThreads, 0, s>>>(G, V, kBpGradZChunk, dv, dvd, q, d_up, part);    \
    else bp_grad_kernel<W, D, 0><<<grid, kBpThreads, 0, s>>>(G, V, kBpGradZChunk, dv, dvd, q, d_up, part);           \
  } while (0)
    if (!G.bp_weight) DFP_BP_GRAD(0, 0);
    else if (!dw) DFP_BP_GRAD(1, 0);
    else DFP_BP_GRAD(1, 1);
#undef DFP_BP_GRAD
    time_end(s);
    bp_contract_kernel<<<V, 256, 0, s>>>(w.gx * w.gy * w.gz, V, part, dc, d_out);
    g_launches += 2;
  }
  DFP_CUDA(cudaGetLastError(), "back-projection launch");
  return DFP_OK;
}

// More views than one grid holds: consecutive slices on the same stream (the workspace is reused in stream order).
// Everything is validated for the WHOLE call first, so that an error is returned before any kernel is launched.
int run_forward(const dfp_geometry* g, int V, const float* angles, const float* poses, const float* d_vol,
                const float* d_up, float* d_out, void* d_ws, size_t ws_bytes, cudaStream_t s, int op,
                float* d_proj = nullptr) {
  if (V <= kMaxViewsPerLaunch || !g) return run_forward_slice(g, V, angles, poses, d_vol, d_up, d_out, d_ws, ws_bytes, s, op, d_proj);
  int st = validate_geometry(g);
  if (st) return st;
  const bool grad = op != DFP_OP_FORWARD, fused = op == DFP_OP_FORWARD_FUSED;
  st = check_common(g, V, angles, poses, d_vol, d_out, grad ? (const void*)d_up : (const void*)d_vol, d_ws, ws_bytes,
                    fwd_ws(*g, V, grad, fused ? 3 : 1).total);
  if (st) return st;
  const size_t per_view = (size_t)g->nu * g->nv, stride = (size_t)view_stride(*g);
  const int per_out = fused ? 18 : 6;
  int launches = 0;
  for (int v0 = 0; v0 < V; v0 += kMaxViewsPerLaunch) {
    const int n = V - v0 < kMaxViewsPerLaunch ? V - v0 : kMaxViewsPerLaunch;
    st = run_forward_slice(g, n, angles + stride * v0, poses + 6 * (size_t)v0, d_vol, d_up ? d_up + per_view * v0 : nullptr,
                           grad ? d_out + (size_t)per_out * v0 : d_out + per_view * v0, d_ws, ws_bytes, s, op,
                           d_proj ? d_proj + per_view * v0 : nullptr);
    if (st) return st;
    launches += g_launches;
  }
  g_launches = launches;
  return DFP_OK;
}

int run_backproject(const dfp_geometry* g, int V, const float* angles, const float* poses, const float* d_proj,
                    const float* d_up, float* d_out, void* d_ws, size_t ws_bytes, cudaStream_t s, bool grad) {
  if (V <= kMaxViewsPerLaunch || !g) return run_backproject_slice(g, V, angles, poses, d_proj, d_up, d_out, d_ws, ws_bytes, s, grad);
  int st = validate_geometry(g);
  if (st) return st;
  st = check_common(g, V, angles, poses, d_proj, d_out, grad ? (const void*)d_up : (const void*)d_proj, d_ws, ws_bytes,
                    bp_ws(*g, V, grad).total);
  if (st) return st;
  const size_t per_view = (size_t)g->nu * g->nv, stride = (size_t)view_stride(*g);
  int launches = 0;
  for (int v0 = 0; v0 < V; v0 += kMaxViewsPerLaunch) {
    const int n = V - v0 < kMaxViewsPerLaunch ? V - v0 : kMaxViewsPerLaunch;
    dfp_geometry gc = *g;                 // dfp_backproject: the first slice overwrites the volume, the others add to it
    if (!grad && v0) gc.flags |= DFP_FLAG_ACCUMULATE;
    st = run_backproject_slice(&gc, n, angles + stride * v0, poses + 6 * (size_t)v0, d_proj + per_view * v0, d_up,
                               grad ? d_out + 6 * (size_t)v0 : d_out, d_ws, ws_bytes, s, grad);
    if (st) return st;
    launches += g_launches;
  }
  g_launches = launches;
  return DFP_OK;
}

// ---- host-buffer wrappers ------------------------------------------------------------------------
struct DevBuf {
  void* p = nullptr;
  cudaStream_t s;
  explicit DevBuf(cudaStream_t st) : s(st) {}
  cudaError_t alloc(size_t bytes) { return cudaMallocAsync(&p, bytes ? bytes : 256, s); }
  ~DevBuf() { if (p) cudaFreeAsync(p, s); }
};

int run_host(int op, const dfp_geometry* g, int V, const float* angles, const float* poses, const float* h_in,
             const float* h_up, float* h_out, void* stream) {
  int st = validate_geometry(g);
  if (st) return st;
  st = validate_views(*g, V, angles, poses);
  if (st) return st;
  const bool grad = op == DFP_OP_FORWARD_POSE_GRAD || op == DFP_OP_BACKPROJECT_POSE_GRAD;
  if (!h_in || !h_out || (grad && !h_up)) return DFP_ERR_NULL;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  {  // keep the stream-ordered pool's memory across calls (the default trims it at every synchronisation)
    static bool pool_set[64] = {false};
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64 && !pool_set[dev]) {
      cudaMemPool_t pool;
      unsigned long long keep = ~0ull;
      if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess)
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
      pool_set[dev] = true;
    }
  }
  const size_t nvol = (size_t)g->nx * g->ny * g->nz * sizeof(float);
  const size_t nproj = (size_t)V * g->nu * g->nv * sizeof(float);
  const size_t ngrad = (size_t)V * 6 * sizeof(float);
  const bool fwd = op == DFP_OP_FORWARD || op == DFP_OP_FORWARD_POSE_GRAD;
  const size_t n_in = fwd ? nvol : nproj;
  const size_t n_up = grad ? (fwd ? nproj : nvol) : 0;
  const size_t n_out = grad ? ngrad : (fwd ? nproj : nvol);
  // what these views need (a subset of views that take the TMA path takes it too, with a smaller layout): no 4x packed
  // copy on the TMA path
  size_t n_ws = dfp_workspace_bytes_for_views(g, V, angles, poses, op);
  if (n_ws == 0) n_ws = dfp_workspace_bytes(g, V, op);
  DevBuf d_in(s), d_up(s), d_out(s), d_ws(s);
  DFP_CUDA(d_in.alloc(n_in), "cudaMallocAsync");
  DFP_CUDA(d_up.alloc(n_up), "cudaMallocAsync");
  DFP_CUDA(d_out.alloc(n_out), "cudaMallocAsync");
  DFP_CUDA(d_ws.alloc(n_ws), "cudaMallocAsync");
  // a9, view chunking: the per-view arrays move in chunks on a second stream while the kernels of the neighbouring
  // chunk run (the input shared by all views - the volume, or the upstream volume of the back-projection gradient -
  // goes first, on the caller's stream); dfp_backproject sums its chunks with DFP_FLAG_ACCUMULATE.
  const int n_chunks = V < 8 ? 1 : 4;
  if (n_chunks == 1) {
    DFP_CUDA(cudaMemcpyAsync(d_in.p, h_in, n_in, cudaMemcpyHostToDevice, s), "H2D");
    if (grad) DFP_CUDA(cudaMemcpyAsync(d_up.p, h_up, n_up, cudaMemcpyHostToDevice, s), "H2D");
    if (fwd)
      st = run_forward(g, V, angles, poses, (const float*)d_in.p, (const float*)d_up.p, (float*)d_out.p, d_ws.p, n_ws,
                       s, grad ? DFP_OP_FORWARD_POSE_GRAD : DFP_OP_FORWARD);
    else
      st = run_backproject(g, V, angles, poses, (const float*)d_in.p, (const float*)d_up.p, (float*)d_out.p, d_ws.p,
                           n_ws, s, grad);
    if (st) { cudaStreamSynchronize(s); return st; }
    DFP_CUDA(cudaMemcpyAsync(h_out, d_out.p, n_out, cudaMemcpyDeviceToHost, s), "D2H");
    DFP_CUDA(cudaStreamSynchronize(s), "stream synchronize");
    return DFP_OK;
  }
  struct Side {                      // the copy stream and its events, released on every exit path
    cudaStream_t s = nullptr, s2 = nullptr;
    bool ok = false;                 // set on the normal exit (which has synchronised both streams itself)
    cudaEvent_t ev[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    ~Side() {
      // error exit in mid-loop: copies of earlier chunks may still be in flight - wait for them before the device
      // buffers are freed and before the caller regains h_out
      if (!ok) { if (s2) cudaStreamSynchronize(s2); cudaStreamSynchronize(s); }
      for (cudaEvent_t e : ev) if (e) cudaEventDestroy(e);
      if (s2) cudaStreamDestroy(s2);
    }
  } side;
  side.s = s;
  DFP_CUDA(cudaStreamCreateWithFlags(&side.s2, cudaStreamNonBlocking), "cudaStreamCreate");
  for (cudaEvent_t& e : side.ev) DFP_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming), "cudaEventCreate");
  const size_t per_view = (size_t)g->nu * g->nv;            // floats of one view's projection / upstream image
  // shared input on the caller's stream; the copy stream starts after the buffers exist (allocation is stream-ordered)
  const float* h_shared = fwd ? h_in : h_up;                 // volume | upstream volume
  float* d_shared = static_cast<float*>(fwd ? d_in.p : d_up.p);
  const float* h_views = fwd ? h_up : h_in;                  // upstream images | projections (null for dfp_forward)
  float* d_views = static_cast<float*>(fwd ? d_up.p : d_in.p);
  DFP_CUDA(cudaEventRecord(side.ev[0], s), "cudaEventRecord");
  DFP_CUDA(cudaStreamWaitEvent(side.s2, side.ev[0], 0), "cudaStreamWaitEvent");
  if (h_shared) DFP_CUDA(cudaMemcpyAsync(d_shared, h_shared, nvol, cudaMemcpyHostToDevice, s), "H2D");
  int launches = 0;
  for (int c = 0; c < n_chunks; ++c) {
    // chunk boundaries on multiples of 4 views: a chunk reads / writes d_views + v0 nu nv floats and d_grad + 6 v0
    // floats, which must stay 16-byte aligned whatever the parity of nu nv; a chunk that comes out empty is skipped
    const int v0 = (int)((long long)V * c / n_chunks) & ~3;
    const int v1 = c + 1 == n_chunks ? V : (int)((long long)V * (c + 1) / n_chunks) & ~3, nv_c = v1 - v0;
    if (nv_c <= 0) continue;
    const size_t off = (size_t)v0 * per_view;
    if (h_views) {                   // this chunk's per-view input on the copy stream, then the kernels wait for it
      DFP_CUDA(cudaMemcpyAsync(d_views + off, h_views + off, (size_t)nv_c * per_view * 4, cudaMemcpyHostToDevice,
                               side.s2), "H2D");
      DFP_CUDA(cudaEventRecord(side.ev[c], side.s2), "cudaEventRecord");
      DFP_CUDA(cudaStreamWaitEvent(s, side.ev[c], 0), "cudaStreamWaitEvent");
    }
    float* out_c = static_cast<float*>(d_out.p) + (grad ? (size_t)v0 * 6 : off);
    if (fwd)
      st = run_forward(g, nv_c, angles + (size_t)view_stride(*g) * v0, poses + 6 * v0, d_shared, grad ? d_views + off : nullptr, out_c, d_ws.p,
                       n_ws, s, grad ? DFP_OP_FORWARD_POSE_GRAD : DFP_OP_FORWARD);
    else if (grad)
      st = run_backproject(g, nv_c, angles + (size_t)view_stride(*g) * v0, poses + 6 * v0, d_views + off, d_shared, out_c, d_ws.p, n_ws, s, true);
    else {                           // dfp_backproject: the first chunk overwrites the volume, the others add to it
      dfp_geometry gc = *g;
      gc.flags = v0 ? (g->flags | DFP_FLAG_ACCUMULATE) : g->flags;
      st = run_backproject(&gc, nv_c, angles + (size_t)view_stride(*g) * v0, poses + 6 * v0, d_views + off, nullptr, static_cast<float*>(d_out.p),
                           d_ws.p, n_ws, s, false);
    }
    if (st) return st;
    launches += g_launches;
    if (fwd && !grad) {              // dfp_forward: this chunk's projections go home while the next chunk is computed
      DFP_CUDA(cudaEventRecord(side.ev[4 + c], s), "cudaEventRecord");
      DFP_CUDA(cudaStreamWaitEvent(side.s2, side.ev[4 + c], 0), "cudaStreamWaitEvent");
      DFP_CUDA(cudaMemcpyAsync(h_out + off, out_c, (size_t)nv_c * per_view * 4, cudaMemcpyDeviceToHost, side.s2),
               "D2H");
    }
  }
  g_launches = launches;
  if (grad || !fwd) DFP_CUDA(cudaMemcpyAsync(h_out, d_out.p, n_out, cudaMemcpyDeviceToHost, s), "D2H");
  DFP_CUDA(cudaStreamSynchronize(side.s2), "stream synchronize");
  DFP_CUDA(cudaStreamSynchronize(s), "stream synchronize");
  side.ok = true;
  return DFP_OK;
}

}  // namespace

extern "C" {

int dfp_forward(const dfp_geometry* g, int n_views, const float* angles, const float* poses, const float* d_vol,
                float* d_proj, void* d_ws, size_t ws_bytes, void* stream) {
  return run_forward(g, n_views, angles, poses, d_vol, nullptr, d_proj, d_ws, ws_bytes,
                     static_cast<cudaStream_t>(stream), DFP_OP_FORWARD);
}

int dfp_forward_pose_grad(const dfp_geometry* g, int n_views, const float* angles, const float* poses,
                          const float* d_vol, const float* d_dLdproj, float* d_grad, void* d_ws, size_t ws_bytes,
                          void* stream) {
  return run_forward(g, n_views, angles, poses, d_vol, d_dLdproj, d_grad, d_ws, ws_bytes,
                     static_cast<cudaStream_t>(stream), DFP_OP_FORWARD_POSE_GRAD);
}

int dfp_forward_fused_moments(const dfp_geometry* g, int n_views, const float* angles, const float* poses,
                              const float* d_vol, const float* d_target, float* d_proj, float* d_moments, void* d_ws,
                              size_t ws_bytes, void* stream) {
  return run_forward(g, n_views, angles, poses, d_vol, d_target, d_moments, d_ws, ws_bytes,
                     static_cast<cudaStream_t>(stream), DFP_OP_FORWARD_FUSED, d_proj);
}

int dfp_backproject(const dfp_geometry* g, int n_views, const float* angles, const float* poses, const float* d_proj,
                    float* d_vol, void* d_ws, size_t ws_bytes, void* stream) {
  return run_backproject(g, n_views, angles, poses, d_proj, nullptr, d_vol, d_ws, ws_bytes,
                         static_cast<cudaStream_t>(stream), false);
}

int dfp_backproject_pose_grad(const dfp_geometry* g, int n_views, const float* angles, const float* poses,
                              const float* d_proj, const float* d_dLdvol, float* d_grad, void* d_ws, size_t ws_bytes,
                              void* stream) {
  return run_backproject(g, n_views, angles, poses, d_proj, d_dLdvol, d_grad, d_ws, ws_bytes,
                         static_cast<cudaStream_t>(stream), true);
}

int dfp_ncc_pose_grad(const dfp_geometry* g, int n_views, const float* d_proj, const float* d_target,
                      const float* d_moments, float* d_ncc, float* d_grad, void* d_ws, size_t ws_bytes, void* stream) {
  int st = validate_geometry(g);
  if (st) return st;
  if (n_views <= 0 || n_views > kMaxViewsPerLaunch) return DFP_ERR_DIMS;
  if (!d_proj || !d_target || !d_moments || !d_ncc || !d_grad || !d_ws) return DFP_ERR_NULL;
  if (!aligned(d_proj, 16) || !aligned(d_target, 16) || !aligned(d_moments, 8) || !aligned(d_ncc, 4) || !aligned(d_grad, 8) ||
      !aligned(d_ws, 256))
    return DFP_ERR_ALIGN;
  if (ws_bytes < dfp_workspace_bytes(g, n_views, DFP_OP_NCC)) return DFP_ERR_WORKSPACE;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const size_t npix = (size_t)g->nu * g->nv;
  const int nblk = (int)std::min<size_t>(kNccBlocks, (npix + 4 * kNccThreads - 1) / (4 * kNccThreads));
  double* partial = static_cast<double*>(d_ws);
  ncc_partial_kernel<<<dim3(nblk, n_views), kNccThreads, 0, s>>>(npix, d_proj, d_target, partial);
  ncc_finish_kernel<<<n_views, 32, 0, s>>>(npix, nblk, partial, d_moments, d_ncc, d_grad);
  g_launches = 2;
  DFP_CUDA(cudaGetLastError(), "NCC launch");
  return DFP_OK;
}

// The allocation-free variant (include/dfp.h): the partial sums of ncc_partial_kernel in a file-scope device array.
// In HOST code `g_ncc_static` is only the symbol's host-side stand-in, not a device address: its address on the
// current device is looked up once per device, below, and THAT pointer goes to the kernels.
}  // extern "C"
static __device__ __align__(256) double g_ncc_static[5 * (size_t)dfp::kNccBlocks * DFP_NCC_STATIC_MAX_VIEWS];
namespace {
constexpr int kMaxDevices = 64;
std::atomic<double*> g_ncc_static_ptr[kMaxDevices];      // per device; nullptr until the first call on it
// Device address of g_ncc_static on the CURRENT device (no allocation: the array is part of the loaded module).
cudaError_t ncc_static_scratch(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  double* p = g_ncc_static_ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    void* sym = nullptr;
    e = cudaGetSymbolAddress(&sym, g_ncc_static);      // with device `dev` current: that device's copy of the array
    if (e != cudaSuccess) return e;
    p = static_cast<double*>(sym);
    g_ncc_static_ptr[dev].store(p, std::memory_order_release);      // two racing first calls store the same address
  }
  *out = p;
  return cudaSuccess;
}
}  // namespace
extern "C" {

int dfp_ncc_pose_grad_static(const dfp_geometry* g, int n_views, const float* d_proj, const float* d_target,
                             const float* d_moments, float* d_ncc, float* d_grad, void* stream) {
  int st = validate_geometry(g);
  if (st) return st;
  if (n_views <= 0) return DFP_ERR_DIMS;
  if (n_views > DFP_NCC_STATIC_MAX_VIEWS) return DFP_ERR_STATIC_LIMIT;
  if (!d_proj || !d_target || !d_moments || !d_ncc || !d_grad) return DFP_ERR_NULL;
  if (!aligned(d_proj, 16) || !aligned(d_target, 16) || !aligned(d_moments, 8) || !aligned(d_ncc, 4) || !aligned(d_grad, 8))
    return DFP_ERR_ALIGN;
  double* partial = nullptr;
  DFP_CUDA(ncc_static_scratch(&partial), "cudaGetSymbolAddress (static NCC scratch)");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const size_t npix = (size_t)g->nu * g->nv;
  const int nblk = (int)std::min<size_t>(kNccBlocks, (npix + 4 * kNccThreads - 1) / (4 * kNccThreads));
  // every element ncc_finish_kernel reads ([view < n_views][block < nblk][5]) is written by ncc_partial_kernel first:
  // nothing of the previous call's contents is used, nothing has to be cleared
  ncc_partial_kernel<<<dim3(nblk, n_views), kNccThreads, 0, s>>>(npix, d_proj, d_target, partial);
  ncc_finish_kernel<<<n_views, 32, 0, s>>>(npix, nblk, partial, d_moments, d_ncc, d_grad);
  g_launches = 2;
  DFP_CUDA(cudaGetLastError(), "NCC launch (static scratch)");
  return DFP_OK;
}

size_t dfp_workspace_bytes(const dfp_geometry* g, int n_views, int op) {
  if (validate_geometry(g) != DFP_OK || n_views <= 0 || n_views > kMaxViews) return 0;
  switch (op) {
    case DFP_OP_FORWARD: return fwd_ws(*g, n_views, false).total;
    case DFP_OP_FORWARD_POSE_GRAD: return fwd_ws(*g, n_views, true).total;
    case DFP_OP_BACKPROJECT: return bp_ws(*g, n_views, false).total;
    case DFP_OP_BACKPROJECT_POSE_GRAD: return bp_ws(*g, n_views, true).total;
    case DFP_OP_FORWARD_FUSED: return fwd_ws(*g, n_views, true, 3).total;
    case DFP_OP_NCC: return align_up(sizeof(double) * 5 * (size_t)kNccBlocks * (size_t)n_views);
    default: return 0;
  }
}

size_t dfp_workspace_bytes_for_views(const dfp_geometry* g, int n_views, const float* angles, const float* poses, int op) {
  const size_t full = dfp_workspace_bytes(g, n_views, op);
  if (full == 0 || op == DFP_OP_NCC || n_views > kMaxViewsPerLaunch) return full;
  if (validate_views(*g, n_views, angles, poses) != DFP_OK) return 0;
  const int V = n_views;
  if (op == DFP_OP_FORWARD || op == DFP_OP_FORWARD_POSE_GRAD || op == DFP_OP_FORWARD_FUSED) {
    if (g->flags & (DFP_FLAG_SIDDON | DFP_FLAG_JOSEPH | DFP_FLAG_DD | DFP_FLAG_SF)) return full;
    const bool grad = op != DFP_OP_FORWARD, interp = grad && (g->flags & DFP_FLAG_GRAD_INTERP);
    const FwdGeom G = make_fwd_geom(*g, grad, interp);
    std::vector<FwdView> hv((size_t)V);
    std::vector<ViewFrame> hf((size_t)V);
    for (int v = 0; v < V; ++v) {
      hf[v] = make_frame(*g, angles, v);
      make_fwd_view(hf[v], poses + 6 * v, &hv[v], nullptr);
    }
    return fwd_choice(*g, G, hv, hf, V, grad, grad).shape >= 0 ? fwd_ws(*g, V, grad, op == DFP_OP_FORWARD_FUSED ? 3 : 1, false).total : full;
  }
  if (g->flags & (DFP_FLAG_DD | DFP_FLAG_SF)) return full;
  const bool grad = op == DFP_OP_BACKPROJECT_POSE_GRAD;
  const BpGeom G = make_bp_geom(*g);
  std::vector<BpView> hv((size_t)V);
  BpViewD scratch;
  for (int v = 0; v < V; ++v) make_bp_view(*g, G, make_frame(*g, angles, v), poses + 6 * v, &hv[v], nullptr, &scratch);
  return bp_choice(*g, G, hv, V, grad).kmax >= 0 ? bp_ws(*g, V, grad, false).total : full;
}

int dfp_forward_host(const dfp_geometry* g, int n_views, const float* angles, const float* poses, const float* h_vol,
                     float* h_proj, void* stream) {
  return run_host(DFP_OP_FORWARD, g, n_views, angles, poses, h_vol, nullptr, h_proj, stream);
}
int dfp_forward_pose_grad_host(const dfp_geometry* g, int n_views, const float* angles, const float* poses,
                               const float* h_vol, const float* h_dLdproj, float* h_grad, void* stream) {
  return run_host(DFP_OP_FORWARD_POSE_GRAD, g, n_views, angles, poses, h_vol, h_dLdproj, h_grad, stream);
}
int dfp_backproject_host(const dfp_geometry* g, int n_views, const float* angles, const float* poses,
                         const float* h_proj, float* h_vol, void* stream) {
  return run_host(DFP_OP_BACKPROJECT, g, n_views, angles, poses, h_proj, nullptr, h_vol, stream);
}
int dfp_backproject_pose_grad_host(const dfp_geometry* g, int n_views, const float* angles, const float* poses,
                                   const float* h_proj, const float* h_dLdvol, float* h_grad, void* stream) {
  return run_host(DFP_OP_BACKPROJECT_POSE_GRAD, g, n_views, angles, poses, h_proj, h_dLdvol, h_grad, stream);
}

int64_t dfp_count_ray_steps(const dfp_geometry* g, int n_views, const float* angles, const float* poses) {
  if (validate_geometry(g) != DFP_OK || validate_views(*g, n_views, angles, poses) != DFP_OK) return -1;
  // the metric's unit: samples tau_k = (k + 1/2) D whose position lies in the volume box padded by
  // EXACTLY 2 voxels (closed box, continuous voxel index in [-2, n + 1] per axis) - the oracle's clip; one count for
  // both the forward and the gradient pass, whatever (slightly larger or smaller) box the kernels march
  FwdGeom G = make_fwd_geom(*g, true);
  {
    const int n[3] = {g->nx, g->ny, g->nz}, H[3] = {G.L.hx, G.L.hy, G.L.hz};
    for (int a = 0; a < 3; ++a) { G.lo[a] = (float)(-2 - H[a]); G.hi[a] = (float)(n[a] + 1 - H[a]); }
  }
  std::vector<FwdView> hv((size_t)n_views);
  for (int v = 0; v < n_views; ++v) make_fwd_view(make_frame(*g, angles, v), poses + 6 * v, &hv[v], nullptr);
  FwdView* dv = nullptr;
  unsigned long long* dn = nullptr;
  unsigned long long n = 0;
  if (cudaMalloc(&dv, sizeof(FwdView) * n_views) != cudaSuccess) return -1;
  if (cudaMalloc(&dn, sizeof(unsigned long long)) != cudaSuccess) { cudaFree(dv); return -1; }
  cudaMemcpy(dv, hv.data(), sizeof(FwdView) * n_views, cudaMemcpyHostToDevice);
  cudaMemset(dn, 0, sizeof(unsigned long long));
  for (int v0 = 0; v0 < n_views; v0 += kMaxViewsPerLaunch) {
    const int nv = n_views - v0 < kMaxViewsPerLaunch ? n_views - v0 : kMaxViewsPerLaunch;
    const dim3 grid((g->nu + kFwdTU - 1) / kFwdTU, (g->nv + kFwdTV - 1) / kFwdTV, nv);
    count_steps_kernel<<<grid, kFwdThreads>>>(G, dv + v0, dn);
  }
  const cudaError_t e = cudaMemcpy(&n, dn, sizeof(n), cudaMemcpyDeviceToHost);
  cudaFree(dv);
  cudaFree(dn);
  if (e != cudaSuccess) { cuda_fail(e, "count_ray_steps"); return -1; }
  return (int64_t)n;
}

int dfp_set_kernel_timing(int enable) {
  g_timing = enable != 0;
  g_ev_valid = false;
  return DFP_OK;
}

float dfp_last_kernel_ms(void) {
  if (!g_timing || !g_ev_valid) return -1.f;
  float ms = -1.f;
  if (cudaEventSynchronize(g_ev[1]) != cudaSuccess) return -1.f;
  if (cudaEventElapsedTime(&ms, g_ev[0], g_ev[1]) != cudaSuccess) return -1.f;
  return ms;
}

int dfp_last_launch_count(void) { return g_launches; }

int dfp_last_path(void) { return g_path; }

const char* dfp_status_string(int status) {
  switch (status) {
    case DFP_OK: return "ok";
    case DFP_ERR_NULL: return "a required pointer is NULL";
    case DFP_ERR_DIMS: return "invalid dimensions, pitches, distances or view count";
    case DFP_ERR_NONFINITE: return "non-finite value in geometry, angles or poses";
    case DFP_ERR_ALIGN: return "device pointer not 16-byte aligned (workspace: 256-byte)";
    case DFP_ERR_WORKSPACE: return "workspace too small (see dfp_workspace_bytes)";
    case DFP_ERR_CUDA: return g_cuda_msg;
    case DFP_ERR_STATIC_LIMIT:
      return "n_views exceeds DFP_NCC_STATIC_MAX_VIEWS (256), the fixed scratch of dfp_ncc_pose_grad_static: slice the "
             "views or use dfp_ncc_pose_grad with a workspace";
    default: return "unknown status";
  }
}

int dfp_version(void) { return 100; }

}  // extern "C"
