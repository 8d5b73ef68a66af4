/* dfp.h - C ABI of libdfp: differentiable cone-beam forward / back-projector with a 6-DOF rigid pose per view.
 *
 * Implements the hot path of "Differentiable Forward and Back-Projector for Rigid Motion Estimation in X-ray
 * Imaging" (arXiv 2508.13304; citations are lines of /root/reference/PAPER.md) as hand-written CUDA for
 * sm_100a (NVIDIA B200).  There is no CPU fallback: without a CUDA device every compute call returns
 * DFP_ERR_CUDA.  See DESIGN.md for the discretisation (readings U1-U13) and the data layout.
 *
 * Conventions:
 *   vol [nz][ny][nx] fp32, x fastest.  proj [n_views][nv][nu] fp32, u fastest.
 *   pose [n_views][6] = (tx,ty,tz,gx,gy,gz) in mm and RADIANS;  r = R r' + t,  R = Rz(gz) Ry(gy) Rx(gx),
 *   r' = R^T (r - t)                                                      (Table I :27-42, :58-60).
 *   View of gantry angle b: source s = SAD (cos b, sin b, 0); detector centre -(SDD-SAD)(cos b, sin b, 0);
 *   e_u = (-sin b, cos b, 0), e_v = (0,0,1); pixel (iu,iv) centre = centre + (iu-c_u) du e_u + (iv-c_v) dv e_v,
 *   c_u = (nu-1)/2 + u0, c_v = (nv-1)/2 + v0;  d = p(r) of Eq.1 (:60-63) is in pixel-index units.
 *   Gradients [n_views][6] are dL/d(tx,ty,tz) per mm and dL/d(gx,gy,gz) per radian.
 *
 *   With DFP_FLAG_VIEW_FRAMES the `angles` array holds one explicit frame (s, c, U, V: 12 floats) per view instead.
 *
 * Pointer kinds.  `angles`, `poses`, `geometry`: HOST memory, read before the call returns.
 *   d_* : DEVICE memory owned by the caller (e.g. torch tensors), fp32, contiguous, 16-byte aligned; read /
 *   written asynchronously on `stream` (a cudaStream_t passed as void*, NULL = default stream) and must stay
 *   alive until the stream reaches that point.  The library allocates no device memory in these calls and
 *   does not wait for the GPU: all device scratch lives in the caller-provided workspace `d_ws`
 *   (>= dfp_workspace_bytes(...) bytes, 256-byte aligned), and the per-view constants (<= 240 bytes per view, computed
 *   on the host in fp64) reach it through a ring of 8 pinned host staging buffers owned by the calling thread (grown on
 *   demand, freed when the thread ends), i.e. by true asynchronous copies; a call waits on the host only if the 8
 *   previous uploads of this thread are all still pending.  Not meant for CUDA-graph capture.
 *   n_views: 1 .. 2^24; batches of more than 65532 views are run as consecutive grid launches on `stream`.
 *   The dfp_*_host convenience calls take HOST arrays for the big buffers too, allocate and free their own
 *   device scratch on `stream` and return after the result has landed in host memory.
 *
 * Errors.  Every call returns an int status: DFP_OK (0) or a negative code; nothing is thrown, printed or
 *   exited.  Arguments are validated for the whole call before any kernel is launched; only DFP_ERR_CUDA can be
 *   returned after work was queued.  Rays / voxels that miss contribute exact zeros (never NaN).
 */
#ifndef DFP_H_
#define DFP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dfp_geometry {
  int32_t nx, ny, nz;   /* volume dims; vol[iz][iy][ix], x fastest                                          */
  float vx, vy, vz;     /* voxel pitch, mm (> 0)                                                            */
  float cx, cy, cz;     /* volume centre in the OBJECT frame, mm (normally 0)                               */
  int32_t nu, nv;       /* detector columns (u, fastest) and rows (v)                                       */
  float du, dv;         /* pixel pitch, mm (> 0)                                                            */
  float u0, v0;         /* principal-point shift, pixels (0 = centred)                                      */
  float sad, sdd;       /* source-axis and source-detector distance, mm (0 < sad < sdd)                     */
  float step_mm;        /* ray-march step; <= 0 means min(vx,vy,vz)                                         */
  int32_t bp_weight;    /* back-projection weight W: 0 = 1 (pure Eq.2b), 1 = FDK (sad/w')^2                 */
  int32_t flags;        /* bit0 (DFP_FLAG_DW): add the dW/dtheta term in dfp_backproject_pose_grad;
                           bit1 (DFP_FLAG_NO_TMA): forward paths use the global-memory gather kernels even where
                           the TMA-staged kernels apply (same results up to summation order; a testing / profiling
                           switch);
                           bit2 (DFP_FLAG_GRAD_INTERP): the two *_pose_grad calls differentiate the trilinear / bilinear
                           INTERPOLANT exactly (8 voxels / 4 pixels per sample, what automatic differentiation of the
                           discrete projector gives - PAPER.md :211, :346) instead of taking the paper's central finite
                           differences of it (32 voxels / 12 pixels; Eq.19-22, :183, :202);
                           bit3 (DFP_FLAG_SIDDON): dfp_forward and dfp_forward_pose_grad use SIDDON weights - a^ij =
                           length of ray i inside voxel j, voxels as boxes of constant value: the exact radiological
                           path of the paper's own ray-driven projector (:213, ref [28]) - with the gradient's G_f^j
                           taken per voxel (central differences of voxel values, lever arm at the voxel centre,
                           Eq.19 :181, :189) instead of the default fixed-step trilinear ray-march; step_mm is then
                           unused.  Not combinable with DFP_FLAG_GRAD_INTERP or dfp_forward_fused_moments
                           (DFP_ERR_DIMS).  The back-projection calls ignore it;
                           bit5 (DFP_FLAG_JOSEPH): as bit3 with JOSEPH weights - the ray is stepped from voxel-centre
                           plane to voxel-centre plane along its driving axis (largest direction component), bilinear
                           interpolation in each plane, path length v_a/|e_a| per plane; same restrictions; not
                           together with DFP_FLAG_SIDDON;
                           bit4 (DFP_FLAG_ACCUMULATE): dfp_backproject ADDS the views' contribution to d_vol instead of
                           overwriting it, so that the sum over views (Eq.21) can be taken slice by slice of the view
                           arrays (view chunking; a view-sharded multi-GPU reconstruction).  Other calls ignore it;
                           bit6 (DFP_FLAG_VIEW_FRAMES): every call reads its `angles` argument as [n_views][12] explicit
                           VIEW FRAMES instead of [n_views] gantry angles - per view, in the world frame and mm: the
                           source s, the detector reference point c (where the pixel index is (c_u, c_v)), and the
                           displacements U, V of one pixel step along u and v (a flat detector anywhere: tilted, shifted,
                           |U| != |V|, U not orthogonal to V) - for non-circular orbits and per-view calibrated
                           geometries (PAPER.md :244).  Pixel (iu,iv) centre = c + (iu-c_u) U + (iv-c_v) V; Eq.1's w' is
                           the depth from the source along the detector normal in mm; du, dv and sdd are then unused and
                           sad only scales the FDK weight (sad/w')^2.  A frame with U parallel to V or with the source
                           in the detector plane is rejected (DFP_ERR_DIMS).  All kernels and both paths serve it
                           (the per-view set-up is the only code that differs);
                           bit7 (DFP_FLAG_DD): all four calls use the DISTANCE-DRIVEN weights (PAPER.md :213, ref [44]) - per
                           view a driving axis, per plane of voxel centres the pixel's boundaries projected from the source,
                           a^ij = slab path length x normalised overlap of the pixel's footprint with the voxel's cell along
                           the two in-plane axes (U14).  dfp_backproject is then the EXACT transpose of dfp_forward
                           (a matched pair, Eq.21), dfp_forward_pose_grad takes G_f^j per voxel and dfp_backproject_pose_grad
                           G_b^i per detector pixel (Eq.19-22).  bp_weight must be 0; not combinable with bits 2, 3, 5 or
                           dfp_forward_fused_moments (DFP_ERR_DIMS); step_mm is unused;
                           bit8 (DFP_FLAG_SF): as bit7 with SEPARABLE-FOOTPRINT weights (PAPER.md :213, ref [29]) - per
                           (voxel, view) a separable footprint on the detector, trapezoids along u and v built from the
                           Jacobian of Eq.13 at the voxel centre, mass = voxel volume x area magnification (U16).
                           Same restrictions as bit7; not together with it.
                           The two scattering calls (dfp_backproject with bit7, dfp_forward with bit8) add 64-bit
                           fixed-point integers, whose sum does not depend on the order: like every other call of the
                           library they are bit-reproducible.  A NaN / Inf in their input makes every element of
                           their output NaN.                                                                     */
} dfp_geometry;

enum {
  DFP_OK = 0,
  DFP_ERR_NULL = -1,       /* a required pointer is NULL                                                    */
  DFP_ERR_DIMS = -2,       /* non-positive size / pitch, sad <= 0, sdd <= sad, n_views <= 0 or > 2^24, index overflow */
  DFP_ERR_NONFINITE = -3,  /* NaN / Inf in geometry, angles or poses                                        */
  DFP_ERR_ALIGN = -4,      /* a device pointer is not 16-byte (workspace: 256-byte) aligned                 */
  DFP_ERR_WORKSPACE = -5,  /* ws_bytes < dfp_workspace_bytes_for_views(...) (<= dfp_workspace_bytes(...))           */
  DFP_ERR_CUDA = -6,       /* CUDA runtime error (no device, launch failure, out of memory in *_host)       */
  DFP_ERR_STATIC_LIMIT = -7 /* n_views > DFP_NCC_STATIC_MAX_VIEWS in dfp_ncc_pose_grad_static               */
};
enum { DFP_OP_FORWARD = 0, DFP_OP_FORWARD_POSE_GRAD = 1, DFP_OP_BACKPROJECT = 2, DFP_OP_BACKPROJECT_POSE_GRAD = 3,
       DFP_OP_FORWARD_FUSED = 4, DFP_OP_NCC = 5 };
enum { DFP_FLAG_DW = 1, DFP_FLAG_NO_TMA = 2, DFP_FLAG_GRAD_INTERP = 4, DFP_FLAG_SIDDON = 8,
       DFP_FLAG_ACCUMULATE = 16, DFP_FLAG_JOSEPH = 32, DFP_FLAG_VIEW_FRAMES = 64, DFP_FLAG_DD = 128, DFP_FLAG_SF = 256 };

/* Forward projection, Eq.2a :67-69 discretised as Eq.18 :172-177 with a fixed-step, zero-extended
 * trilinear ray-march (U1): proj[v][iv][iu] = D * sum_k f~(R_v^T (s_v + (k+1/2) D e_i - t_v)).
 * d_vol is read, d_proj ([n_views][nv][nu]) is overwritten. */
int dfp_forward(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses,
                const float* d_vol, float* d_proj, void* d_ws, size_t ws_bytes, void* stream);

/* Pose gradient of a loss through the forward projector, Eq.3-8 :81-113, Eq.19-20 :179-191:
 * d_grad[v][0:6] = dL/dtheta_v = sum_i d_dLdproj[v][i] * dl_i/dtheta_v, with the volume gradient taken on
 * the fly by central differences of f~ (:183) and G_f never materialised (:207).  d_grad is overwritten. */
int dfp_forward_pose_grad(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses,
                          const float* d_vol, const float* d_dLdproj, float* d_grad, void* d_ws, size_t ws_bytes,
                          void* stream);

/* Voxel-driven back-projection, Eq.2b :71-75 / Eq.21 :193-196:
 * vol[j] = sum_v W * b~_v(p(R_v r'_j + t_v)), b~ = zero-extended bilinear interpolant, W per bp_weight.
 * d_proj is read, d_vol ([nz][ny][nx]) is overwritten. */
int dfp_backproject(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses,
                    const float* d_proj, float* d_vol, void* d_ws, size_t ws_bytes, void* stream);

/* Pose gradient of a loss through the back-projector, Eq.9-17 :115-168, Eq.22 :198-206:
 * d_grad[v][0:6] = sum_j d_dLdvol[j] * dmu_j/dtheta_v, projection gradient by central differences of b~ (:202),
 * G_b never materialised.  d_grad is overwritten. */
int dfp_backproject_pose_grad(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses,
                              const float* d_proj, const float* d_dLdvol, float* d_grad, void* d_ws,
                              size_t ws_bytes, void* stream);

/* Fused forward projection + pose-gradient MOMENTS in one traversal of the volume (an extension beyond the paper's
 * four operations).  For a loss whose upstream gradient is affine in the projection,
 *     dL/dl_i = alpha_v + beta_v * l_i + gamma_v * b_i        (b = a target image: SSD, NCC - PAPER.md Eq.23, 25)
 * with per-view scalars known only AFTER l is (means, norms), the gradient of Eq.20 (:185) is
 *     dL/dtheta_v = alpha_v m[v][0] + beta_v m[v][1] + gamma_v m[v][2],
 *     m[v][0] = sum_i dl_i/dtheta_v,   m[v][1] = sum_i l_i dl_i/dtheta_v,   m[v][2] = sum_i b_i dl_i/dtheta_v,
 * so one pass that writes l AND the three 6-vectors replaces dfp_forward followed by dfp_forward_pose_grad.
 * d_target: device [n_views][nv][nu] (b); d_proj: device, out, [n_views][nv][nu] (l, as dfp_forward up to fp32
 * summation order); d_moments: device, out, [n_views][3][6], each 6-vector laid out and scaled exactly like the
 * output of dfp_forward_pose_grad with upstream 1, l, b.  Central-difference gradient mode only (DFP_ERR_DIMS with
 * DFP_FLAG_GRAD_INTERP).  Workspace: dfp_workspace_bytes(geometry, n_views, DFP_OP_FORWARD_FUSED).  Same ownership,
 * asynchrony and error behaviour as the four calls above. */
int dfp_forward_fused_moments(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses,
                              const float* d_vol, const float* d_target, float* d_proj, float* d_moments, void* d_ws,
                              size_t ws_bytes, void* stream);

/* The loss of the paper's 2D/3D registration task on the device (Eq.25 :230-235; an extension beyond the four
 * operations): for every view the normalised cross-correlation NCC(l_v, b_v) of its projection
 * with its measured image, and dNCC/dtheta_v = alpha m[v][0] + beta m[v][1] + gamma m[v][2] from the moments of
 * dfp_forward_fused_moments (alpha, beta, gamma: the coefficients of dNCC/dl_i = alpha + beta l_i + gamma b_i) - so that
 * an iteration of the registration loop is two asynchronous calls on one stream and one 28-byte read-back.
 * d_proj, d_target: device [n_views][nv][nu]; d_moments: device [n_views][3][6]; d_ncc: device, out, [n_views];
 * d_grad: device, out, [n_views][6], laid out like the output of dfp_forward_pose_grad.  Sums in fp64, fixed order.
 * A view whose projection or target is constant gets NCC 0 and a zero gradient.  Workspace:
 * dfp_workspace_bytes(geometry, n_views, DFP_OP_NCC).  Same ownership, asynchrony and error behaviour as above. */
int dfp_ncc_pose_grad(const dfp_geometry* geometry, int n_views, const float* d_proj, const float* d_target,
                      const float* d_moments, float* d_ncc, float* d_grad, void* d_ws, size_t ws_bytes, void* stream);

/* dfp_ncc_pose_grad for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same two kernels, the same arguments without the workspace, the same results bit for bit -
 * the per-view partial sums live in a fixed array in the library's own device image instead
 * (static __device__, 5 x 64 x DFP_NCC_STATIC_MAX_VIEWS doubles = 640 KiB, held by every GPU that loads the library
 * until the process exits).  The call allocates and frees nothing, on the host or the device, and synchronises
 * nothing; the first call on a device looks the array's address up (cudaGetSymbolAddress, with that device current).
 * n_views > DFP_NCC_STATIC_MAX_VIEWS is rejected with DFP_ERR_STATIC_LIMIT before any launch (slice the views, or use
 * dfp_ncc_pose_grad with a caller-owned workspace); every other argument is checked as in dfp_ncc_pose_grad.
 * ALL calls on a device share the one array: calls queued on the same stream are ordered and safe; two calls that can
 * overlap on the GPU (different streams, or different host threads on different streams) RACE on it - order them with an
 * event, or give all but one a workspace through dfp_ncc_pose_grad.  The array keeps the last call's partial sums;
 * nothing in it has to start at zero (every element a call reads, it has written first). */
#define DFP_NCC_STATIC_MAX_VIEWS 256
int dfp_ncc_pose_grad_static(const dfp_geometry* geometry, int n_views, const float* d_proj, const float* d_target,
                             const float* d_moments, float* d_ncc, float* d_grad, void* stream);

/* Bytes of device workspace the op needs for this geometry and view count (0 on invalid arguments).
 * View chunking: any n_views may be passed to the calls above; to bound the workspace (and the size of
 * d_proj) call them on consecutive slices of the view arrays - views are independent in forward /
 * forward_pose_grad / *_pose_grad, and dfp_backproject of a slice can be summed by the caller. */
size_t dfp_workspace_bytes(const dfp_geometry* geometry, int n_views, int op);

/* The bytes of workspace the op needs for THESE views (host arrays, as passed to the call; 0 on invalid arguments):
 * dfp_workspace_bytes is the size that serves any views - it reserves the gather kernels' 4x packed copy of the volume
 * (forward calls) or of the projections (back-projection calls), which only views whose tiles fit no staging box take
 * (DFP_PATH_GATHER; none of BASELINE.json's configs).  When these views take the TMA-staged kernels the size returned
 * here leaves that copy out (512^3 volume: 2.1 GiB -> 0.1 GiB for dfp_forward; 360 views of 1024^2: 5.7 -> 0.01 GiB for
 * dfp_backproject); otherwise, and for the other weight models, n_views > 65532 and DFP_OP_NCC, it equals
 * dfp_workspace_bytes.  A call checks ws_bytes against exactly this size for its own views (always <=
 * dfp_workspace_bytes) and returns DFP_ERR_WORKSPACE, before any launch, if it is smaller.  The size depends on the
 * views only through the kernel path they take: a workspace sized for one set of poses serves every other set that
 * takes the same path, and dfp_workspace_bytes serves all. */
size_t dfp_workspace_bytes_for_views(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses,
                                     int op);

/* Same four operations with HOST buffers (h_*: host memory, pinned or pageable).  Each allocates device
 * scratch with cudaMallocAsync on `stream`, copies inputs in, runs the device call above, copies the result
 * out, frees, and synchronises `stream` before returning (also on an error that occurs after work was queued: the
 * caller's buffers are never touched after the call has returned).  With 8 or more views the per-view arrays move in
 * up to 4 chunks (boundaries on multiples of 4 views, so every chunk pointer keeps its 16-byte alignment for any nu, nv)
 * on an internal second stream, overlapped with the kernels of the neighbouring chunk (per-view results do
 * not depend on the chunking; dfp_backproject_host sums its chunks with DFP_FLAG_ACCUMULATE, which changes the
 * fp32 summation order only).  The
 * first host call on a device raises the release threshold of its default stream-ordered memory pool so that
 * later calls reuse the scratch memory. */
int dfp_forward_host(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses,
                     const float* h_vol, float* h_proj, void* stream);
int dfp_forward_pose_grad_host(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses,
                               const float* h_vol, const float* h_dLdproj, float* h_grad, void* stream);
int dfp_backproject_host(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses,
                         const float* h_proj, float* h_vol, void* stream);
int dfp_backproject_pose_grad_host(const dfp_geometry* geometry, int n_views, const float* angles,
                                   const float* poses, const float* h_proj, const float* h_dLdvol, float* h_grad,
                                   void* stream);

/* The unit of the "Gray-steps/s" metric: the number of (ray, sample) pairs, summed over rays and
 * views, whose sample tau_k = (k + 1/2) D lies in the volume box padded by exactly 2 voxels (continuous voxel index in
 * [-2, n + 1] on every axis) - the set the oracle's forward projector counts; one number for both dfp_forward and
 * dfp_forward_pose_grad in the default (trilinear) mode, whatever slightly different box each kernel marches.  Counted
 * by a small kernel that runs the projectors' per-ray clip (fp64) against that box, on the default stream,
 * synchronously; allocates and frees its own scratch.  Returns -1 on invalid arguments or CUDA failure. */
int64_t dfp_count_ray_steps(const dfp_geometry* geometry, int n_views, const float* angles, const float* poses);

/* Kernel timing for roofline accounting.  dfp_set_kernel_timing(1) makes every later device-pointer call on
 * this thread bracket its DOMINANT kernel (fwd_project / fwd_grad / bp / bp_grad; not the packing or the
 * contraction kernels) with two CUDA events recorded on `stream`; dfp_last_kernel_ms() waits for the second
 * event and returns the elapsed milliseconds of that one launch (-1 if timing is off or nothing ran).
 * Off by default; costs two event records per call when on. */
int dfp_set_kernel_timing(int enable);
float dfp_last_kernel_ms(void);

/* Number of kernels the last successful call on this thread launched (for bench accounting). */
int dfp_last_launch_count(void);

/* Kernel path the last successful device-pointer call on this thread took: DFP_PATH_GATHER (global-memory
 * gathers from a packed copy of the input) or DFP_PATH_TMA (input staged tile by tile in shared memory by TMA;
 * taken when every view's tiles fit the staging boxes; with nx % 4 != 0 (forward calls) / nu % 4 != 0 (back-projection
 * calls) it reads a copy of the input with its rows padded to 16 bytes, made per call in the workspace).  The two paths
 * do the same arithmetic per sample / voxel and agree to fp32 summation order.  Both the
 * forward and the back-projection calls have the two paths. */
enum { DFP_PATH_GATHER = 0, DFP_PATH_TMA = 1 };
int dfp_last_path(void);

/* Static description of a status code; for DFP_ERR_CUDA the text of the last CUDA error seen on this thread. */
const char* dfp_status_string(int status);

/* Library version (major*10000 + minor*100 + patch). */
int dfp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DFP_H_ */
