/* include/ts.h -- C ABI of libts: the B200 (sm_100a) differentiable triangle-soup rasteriser,
 * i.e. the hot path of Triangle Splatting SLAM (arxiv/paper_2605_31419).
 *
 * Conventions (all exports):
 *  - Return value: int32 status (TS_OK = 0, negative = error).  No exceptions, no aborts, no stdout.
 *    Argument errors are detected on the host before any launch.  Data-dependent overflow of the
 *    caller-sized buffers is reported asynchronously through ts_frame_status (flags & TS_FLAG_OVERFLOW);
 *    outputs of an overflowed frame are unspecified (never out-of-bounds) and the caller re-binds a larger
 *    workspace and repeats.
 *  - Ownership: every DEVICE buffer is owned by the caller (e.g. torch tensors' data_ptr()), including the
 *    frame workspace.  The library allocates no device memory after ts_create, never frees caller memory and
 *    keeps no caller pointer beyond the call, with one exception: a ts_frame remembers the pose pointer given to
 *    ts_project until the next ts_project on it (the full-gradient ts_render_bwd reads the pose again), so it must
 *    stay valid and unchanged until the frame's backward pass has been enqueued.
 *  - Devices: a ts_ctx belongs to the device given to ts_create; every export that launches work returns
 *    TS_ERR_INVALID_ARG unless that device is the calling thread's current device (cudaSetDevice is the caller's).
 *    Several contexts, one per device, may live in one process.
 *  - Streams: `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All work is enqueued
 *    on it.  No export synchronises except ts_frame_status and ts_frame_view.  All exports may be captured
 *    into a CUDA graph (launch geometry never depends on device-side counts).
 *  - Layout: float32, row-major, contiguous.  pos[V][3], color[V][3], opacity[V] (already activated, in
 *    [0,1]); faces[M][3] int32 vertex indices, or NULL = soup (V == 3M, face m = (3m,3m+1,3m+2), the map
 *    layout the paper uses during SLAM).  Pose T_cw[12] = row-major 3x4 [R|t] IN DEVICE MEMORY
 *    (a tracking loop updates it without the host).  Images are planar: color[3][H][W], depth[H][W],
 *    alpha[H][W].  Pixel (x,y) is sampled at exactly (x,y).
 *  - Gradient outputs ACCUMULATE (+=); the caller zeroes them.  dL_dtau[6] is overwritten, order
 *    (rho_x,rho_y,rho_z,theta_x,theta_y,theta_z), left perturbation T <- Exp(tau) o T (Eq. 6-7).
 */
#ifndef TS_H
#define TS_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ts_ctx ts_ctx;      /* opaque: device properties, one per device */
typedef struct ts_frame ts_frame;  /* opaque: one view's intermediate state inside caller memory */

typedef struct { int32_t width, height; float fx, fy, cx, cy, znear; } ts_camera;
/* sigma: window smoothness (Eq. 3, global constant; 0.5 in the paper).
 * alpha_min: pairs with alpha < alpha_min contribute nothing (0 = literal Eq. 4).  t_min: stop a pixel's walk
 * once its transmittance is <= t_min (the face that crossed IS included; 0 = literal Eq. 4).
 * eps_area: faces with |doubled screen area| <= eps_area are culled. */
typedef struct { float sigma, alpha_min, t_min, eps_area; uint32_t flags; } ts_params;
typedef struct { const float *pos, *color, *opacity; const int32_t *faces; int32_t V, M; } ts_scene; /* device ptrs */

enum { TS_OK = 0, TS_ERR_INVALID_ARG = -1, TS_ERR_WORKSPACE = -2, TS_ERR_CAPACITY = -3, TS_ERR_CUDA = -4,
       TS_ERR_STATE = -5, TS_ERR_STATIC_LIMIT = -6 /* ts_render_fwd_static: scene or image beyond TS_STATIC_MAX_* */ };
enum { TS_GRAD_POS = 1, TS_GRAD_COLOR = 2, TS_GRAD_OPACITY = 4, TS_GRAD_POSE = 8 };
enum { TS_FLAG_OVERFLOW_PAIRS = 1, TS_FLAG_OVERFLOW_VISIBLE = 2 };
/* ts_params.flags */
enum { TS_PARAM_COUNTERS = 0x100,     /* count visits / rect tests / hits into the frame's debug counters */
       TS_PARAM_MIN_OPACITY = 0x200,  /* face opacity = MIN of its vertex opacities instead of their mean (
                                          "+ min opacity" ablation, Table S3); its gradient goes to that
                                          vertex alone (lowest index among equal minima) */
       TS_PARAM_TIGHT_BINNING = 0x400 }; /* a face is binned only into the tiles its TRIANGLE meets, not into every tile
                                          its pixel rect touches (SURVEY.md NEXT-4 "tighter triangle-tile binning";
                                          DESIGN.md reading S31): shorter lists, identical images and gradients; the
                                          tile counts, sorted lists and ranges are then those of the oracle's
                                          tight_binning mode, bit for bit */

const char* ts_strerror(int32_t status);

/* ---- lifecycle ------------------------------------------------------------------------------------------ */
int32_t ts_create(int32_t device, ts_ctx** out);
int32_t ts_destroy(ts_ctx* ctx);
/* Tracing: with on != 0 every export of this context that enqueues work brackets itself with an NVTX
 * range named after the call ("ts_project", "ts_bin_sort", ...), so a timeline / `ncu --nvtx` groups the kernels by API
 * call.  Off by default; without a profiler attached an NVTX call is a no-op stub.  Host-side only, no launch. */
int32_t ts_set_tracing(ts_ctx* ctx, int32_t on);

/* Bytes of device workspace a frame needs for M faces, a WxH image, at most `pair_capacity` (tile, face)
 * pairs (< 2^28) and at most `visible_capacity` faces surviving the cull (0 = M; < 2^28).  About 208 B per pair
 * (the sorted tile lists plus room for every pair in the lists of all eight 8x4 blocks of its tile), 290 B per
 * visible face and 16 B per pixel.  Returns 0 on invalid arguments. */
size_t ts_frame_bytes(const ts_ctx* ctx, int32_t M, int32_t W, int32_t H, uint64_t pair_capacity,
                      uint64_t visible_capacity);
/* Carves `dev_ws` (device memory, >= ts_frame_bytes, 256-byte aligned) into the frame's arrays; allocates
 * only the small host-side handle.  Enqueues a one-time clear of the workspace control block on `stream`. */
int32_t ts_frame_bind(ts_ctx* ctx, void* dev_ws, size_t bytes, int32_t M, int32_t W, int32_t H,
                      uint64_t pair_capacity, uint64_t visible_capacity, void* stream, ts_frame** out);
int32_t ts_frame_release(ts_frame* frame);   /* frees the host handle only */
/* Per-face window smoothness (reading S32): Triangle Splatting [8] learns one sigma per
 * triangle, this paper fixes one global constant.  sigma_dev[M] (device, > 0; NULL = back to the
 * global ts_params.sigma) replaces it for every later ts_project / ts_bin_sort / render call on this frame (the
 * exponent travels in the per-face record: calls before the next ts_bin_sort return TS_ERR_STATE); the renders then run
 * the generic-exponent instantiation.  grad_sigma_dev[M] (device, may be NULL; accumulates, caller zeroes): the
 * full-gradient ts_render_bwd / ts_render_map_l1 / ts_render_bwd_normal add dL/dsigma_m = sum_hits dL/dI I ln x.  Both
 * pointers must stay valid until replaced.  Host call, no launch. */
int32_t ts_frame_set_face_sigma(ts_ctx* ctx, ts_frame* frame, const float* sigma_dev, float* grad_sigma_dev);
/* Synchronises `stream`, then reports the counters of the last ts_project/ts_bin_sort on this frame. */
int32_t ts_frame_status(ts_ctx* ctx, ts_frame* frame, uint32_t* flags, uint32_t* n_visible, uint64_t* n_pairs,
                        void* stream);

/* ---- the five hot-path calls ----------------------------------------------------------------------------- */

/* a1: Eq. 1.  Per face: Q_k = R P_k + t; cull unless all Z_k > znear; u = fx X/Z + cx,
 * v = fy Y/Z + cy; cull degenerate screen area; pixel rect = integer pixel centres inside the vertex AABB,
 * clipped to the image, cull if empty; depth key = float32 bits of the mean camera depth.  Surviving faces get a
 * slot (allocation order, not face order), their screen record (u,v,1/Z)x3 + mean opacity + rect +
 * depth key, and are counted into every 16x16 tile they touch; the per-tile counts are scanned into
 * tile_ranges[NT] = (begin,end).  float32 with a fixed operation order: cull set, rects, depth keys and tile
 * counts are bit-identical to the oracle (N1-N5).  One kernel, one pass over the map.
 * scene->color may be NULL here; scene->opacity must be valid (the mean vertex opacity of PAPER.md:82 is taken here). */
int32_t ts_project(ts_ctx* ctx, const ts_scene* scene, const ts_camera* cam, const ts_params* prm,
                   const float* T_cw_dev, ts_frame* frame, void* stream);

/* a2: "faces are sorted in depth order".  MSD-first radix sort of the (tile, depth) key: the
 * tile digit is a counting sort (scatter of every (tile, face) pair into its tile's segment, fused with the
 * per-face set-up of Eq. 2-3: unit normals, inradius, incentre), then every segment is sorted by
 * (depth_key, face index) in shared memory.  The result equals the stable sort of (tile << 32 | depth_key) with
 * pairs emitted in face order: ties keep ascending face index.  Requires ts_project on the same frame and stream
 * order. */
int32_t ts_bin_sort(ts_ctx* ctx, ts_frame* frame, void* stream);

/* a3: Eq. 2-4.  Per pixel walk its tile's list front to back: phi = max_k L_k,
 * I = ReLU(phi(p)/phi(s))^sigma, alpha = mean-opacity * I, perspective-correct barycentric colour and depth,
 * C += T alpha c, D += T alpha z, T *= (1-alpha); A = 1 - T.  Any output pointer may be NULL. */
int32_t ts_render_fwd(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, float* out_color, float* out_depth,
                      float* out_alpha, void* stream);

/* a5+a6: reverse walk of the same lists (B1-B8), gradients of L given dL/dC, dL/dD, dL/dA
 * (same layouts as the outputs; any may be NULL = 0).  grad_mask selects TS_GRAD_*.  With TS_GRAD_POSE alone
 * ("pose-only", the tracking mode) no per-vertex buffer is touched: per-thread se(3) terms are tree-reduced
 * in-kernel to one 6-vector per 8x4-pixel block.  Otherwise per-face screen-space gradients are warp-reduced, added with
 * global float atomics and pushed through the projection (B7-B8) into grad_pos; colour / opacity gradients are
 * added to grad_color / grad_opacity.  Requires ts_render_fwd on the same frame. */
int32_t ts_render_bwd(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, const float* dL_dcolor,
                      const float* dL_ddepth, const float* dL_dalpha, float* grad_pos, float* grad_color,
                      float* grad_opacity, uint32_t grad_mask, void* stream);

/* a7: Eq. 5-7: dL/dtau = sum_{face vertices} [g_C ; Q x g_C] from the partial sums the
 * last ts_render_bwd (with TS_GRAD_POSE) left in the frame; fixed-order tree reduction (deterministic). */
int32_t ts_pose_jacobian_reduce(ts_ctx* ctx, ts_frame* frame, float* dL_dtau_dev, void* stream);

/* ---- harness helpers (not part of the five; rows a4 / a8 of DESIGN.md) ------------------------------------ */

/* a4: L = 1/(3HW) sum|C-Chat| + lambda_dep/(HW) sum_{Dhat>0}|D-Dhat| (Eq. 8-10 without D-SSIM); writes the
 * cotangent images gC[3][H][W], gD[H][W] and, if loss_dev != NULL, adds L to *loss_dev (caller zeroes). */
int32_t ts_l1_loss_grad(ts_ctx* ctx, int32_t W, int32_t H, const float* C, const float* D, const float* Chat,
                        const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss_dev, void* stream);
/* E_equi of E_map (Eq. 14-15): mean over the faces and their three internal
 * angles of (cos theta - 0.5)^2, in world space.  grad_pos[V][3] += weight * dE_equi/dpos (may be NULL);
 * *loss_dev += weight * E_equi (may be NULL).  Only scene->pos, faces, V, M are read. */
int32_t ts_equi_loss_grad(ts_ctx* ctx, const ts_scene* scene, float weight, float* grad_pos, float* loss_dev, void* stream);
/* D-SSIM term of E_pho (Eq. 8; lambda = 0.2):
 * L_DSSIM = 1 - mean SSIM(C, Chat) over 3 x H x W, 11x11 Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2,
 * C2 = 0.03^2.  On entry gC[3][H][W] holds the cotangent of the L1 term (ts_l1_loss_grad); on exit
 * gC = (1 - lambda) gC + lambda dL_DSSIM/dC, i.e. the cotangent of E_pho.  If loss_dev != NULL, lambda * L_DSSIM is
 * added to *loss_dev.  One launch; both separable passes run in shared memory on a tile + apron (no scratch image).  In a
 * tracking iteration it sits between ts_render_fwd_l1 (which writes C and the L1 cotangents) and ts_render_bwd. */
int32_t ts_dssim_loss_grad(ts_ctx* ctx, int32_t W, int32_t H, const float* C, const float* Chat, float lambda, float* gC,
                           float* loss_dev, void* stream);
/* a3 + a4 in one launch: ts_render_fwd, with the L1 colour + depth loss of ts_l1_loss_grad evaluated on every pixel
 * while its value is still in registers: writes gC, gD (and adds L to *loss_dev if not NULL) exactly as
 * ts_l1_loss_grad would.  out_color / out_depth / out_alpha may be NULL (a tracking loop never reads them). */
int32_t ts_render_fwd_l1(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, float* out_color, float* out_depth,
                         float* out_alpha, const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD,
                         float* loss_dev, void* stream);
/* a3 + a4 + a5 (pose-only) in one launch, the tracking fast path: every 8x4-pixel block is rendered, its L1
 * cotangents are formed in registers and its reverse walk runs at once; leaves the se(3) partial sums for
 * ts_pose_jacobian_reduce / ts_pose_reduce_step exactly as ts_render_fwd_l1 + ts_render_bwd(TS_GRAD_POSE) would
 * (same arithmetic, bit-identical result).  out_*, gC, gD and loss_dev may be NULL.  ts_render_bwd cannot follow
 * this call (the per-pixel walk state is not written out). */
int32_t ts_render_track_l1(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, float* out_color, float* out_depth,
                           float* out_alpha, const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD,
                           float* loss_dev, void* stream);
/* The mapping counterpart of ts_render_track_l1: a3 + a4 + a5 (FULL-gradient) per 8x4-pixel block in one launch, then a6:
 * every block is rendered, its L1 cotangents are formed in registers and its reverse walk runs at once, with the
 * colour / opacity gradients and the per-face screen terms accumulated as by ts_render_bwd (grad_* are added to;
 * TS_GRAD_POSE leaves partial sums for ts_pose_jacobian_reduce).  grad_mask must select at least one of TS_GRAD_POS /
 * TS_GRAD_COLOR / TS_GRAD_OPACITY.  Same arithmetic as ts_render_fwd_l1 + ts_render_bwd; the sums differ from theirs
 * only in the order of the float atomics.  out_*, gC, gD and loss_dev may be NULL.  ts_render_bwd cannot follow. */
int32_t ts_render_map_l1(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, float* out_color, float* out_depth,
                         float* out_alpha, const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD,
                         float* loss_dev, float* grad_pos, float* grad_color, float* grad_opacity, uint32_t grad_mask,
                         void* stream);
/* Per-face statistics for the map-management layer (PAPER.md:137 covisibility of rendered faces,
 * :169 prune by projected area, :175 blur-split by pixel coverage).
 * ts_render_fwd_stats: as ts_render_fwd, and face_pixels[m] += number of pixels face m contributed to (caller zeroes;
 * a face is "rendered" iff its count is non-zero).  out_* may be NULL.
 * ts_face_area: proj_area[m] = |S|/2 in px^2 for every face that survived the last ts_project (other entries are
 * left untouched: zero the array first).  Requires ts_bin_sort on the frame (which publishes the visible count);
 * TS_ERR_STATE otherwise. */
int32_t ts_render_fwd_stats(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, float* out_color, float* out_depth,
                            float* out_alpha, uint32_t* face_pixels, void* stream);
int32_t ts_face_area(ts_ctx* ctx, ts_frame* frame, float* proj_area, void* stream);
/* ts_render_bwd plus the screen-space gradient statistic of the densification test (Table S4 "gradient threshold /
 * percentile"; reading S28): for every face that received a gradient,
 * face_grad2d[m] += || sum_k (dL/du_k, dL/dv_k) ||_2 (the gradient of L under a rigid translation of the face in the
 * image plane, in 1/px) and face_views[m] += 1 (may be NULL); both [M], device, accumulated over calls (caller zeroes).
 * grad_mask must contain TS_GRAD_POS or TS_GRAD_POSE (the statistic is a by-product of the per-face screen gradients;
 * with TS_GRAD_POSE alone the full-gradient path runs, not the pose-only one). */
int32_t ts_render_bwd_stats(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, const float* dL_dcolor,
                            const float* dL_ddepth, const float* dL_dalpha, float* grad_pos, float* grad_color,
                            float* grad_opacity, uint32_t grad_mask, float* face_grad2d, uint32_t* face_views,
                            void* stream);

/* Rendered normal map and its gradient (Eq. 12: the map "returned by the rasteriser" that E_norm
 * compares with the sensor normals; reading S26):
 *   N(p) = sum_n n_n alpha_n T_n,  n_n = unit normal of face n in CAMERA space, oriented towards the camera
 * (n . Q < 0 for the points Q of the face), composited by the same walk as colour / depth / alpha, not renormalised.
 * ts_render_fwd_normal: as ts_render_fwd (out_color / out_depth / out_alpha may be NULL) plus out_normal[3][H][W]
 *   (device, required).  Reads scene->pos and the T_cw given to ts_project (still valid, unchanged).
 * ts_render_bwd_normal: as ts_render_bwd with one more cotangent dL_dnormal[3][H][W] (device, required; the other
 *   three may be NULL = 0): ONE reverse walk for all four outputs.  Full-gradient mode for every grad_mask (the
 *   normal's own dependence on the vertices needs the per-face sums): grad_pos receives both the window path
 *   (B4-B8) and d n / d vertices; TS_GRAD_POSE leaves partial sums for ts_pose_jacobian_reduce that include the
 *   rotation of the normals (a translation of the camera does not turn them).  Requires ts_render_fwd_normal on the
 *   same frame since the last ts_project. */
int32_t ts_render_fwd_normal(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, float* out_color, float* out_depth,
                             float* out_alpha, float* out_normal, void* stream);
int32_t ts_render_bwd_normal(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, const float* dL_dcolor,
                             const float* dL_ddepth, const float* dL_dalpha, const float* dL_dnormal, float* grad_pos,
                             float* grad_color, float* grad_opacity, uint32_t grad_mask, void* stream);

/* The "normal direction of the triangle with highest opacity along each ray" of Fig. 3 (
 * DESIGN.md reading S29): as ts_render_fwd_normal, plus out_normal_top[3][H][W] (device, required) = the camera-space
 * unit normal of the FIRST hit with the largest alpha (face opacity x window) among the hits the walk composites; zero
 * where nothing is hit.  Forward only (a visualisation: piecewise constant, no gradient).  out_normal may be NULL. */
int32_t ts_render_fwd_normal_top(ts_ctx* ctx, const ts_scene* scene, ts_frame* frame, float* out_color, float* out_depth,
                                 float* out_alpha, float* out_normal, float* out_normal_top, void* stream);

/* Normalised depth (E_dep compares a rendered depth with the sensor
 * depth, and D = sum z alpha T under-reads wherever A < 1).  ts_depth_normalise: Dn = D / A where A > eps, else 0.
 * ts_depth_normalise_bwd: given the cotangent gDn of Dn, gD += gDn / A and gA += -gDn D / A^2 (where A > eps); gD, gA are
 * then the dL_ddepth / dL_dalpha of ts_render_bwd (they accumulate: the caller initialises them).  [H][W] device arrays. */
int32_t ts_depth_normalise(ts_ctx* ctx, int32_t W, int32_t H, const float* D, const float* A, float eps, float* Dn, void* stream);
int32_t ts_depth_normalise_bwd(ts_ctx* ctx, int32_t W, int32_t H, const float* D, const float* A, float eps, const float* gDn,
                               float* gD, float* gA, void* stream);

/* E_norm of E_map (Eq. 12 and 15; lambda_norm = 0.05): weight / (H W) * sum over the
 * valid pixels (those with a sensor normal, Nbar_p != 0) of 1 - N_p . Nbar_p (reading S27).  N = the map of
 * ts_render_fwd_normal, Nbar = sensor normals, both [3][H][W] device.  Writes gN[3][H][W] = the cotangent of N (input of
 * ts_render_bwd_normal); adds the weighted loss to *loss_dev if not NULL. */
int32_t ts_normal_loss_grad(ts_ctx* ctx, int32_t W, int32_t H, const float* N, const float* Nbar, float weight, float* gN,
                            float* loss_dev, void* stream);

/* a8: one Adam step on tau, then T_cw <- Exp(-delta) o T_cw, all on the device.
 * state_dev[13] = m[6], v[6], step; lr[6] passed by value (rho then theta). */
int32_t ts_pose_step(ts_ctx* ctx, float* T_cw_dev, const float* dL_dtau_dev, float* state_dev, const float* lr6,
                     float beta1, float beta2, float eps, void* stream);

/* a7 + a8 in one launch: as ts_pose_jacobian_reduce, then the thread that wrote dL/dtau takes the ts_pose_step on
 * T_cw_dev / state_dev (same arguments).  dL_dtau_dev still receives the gradient. */
int32_t ts_pose_reduce_step(ts_ctx* ctx, ts_frame* frame, float* dL_dtau_dev, float* T_cw_dev, float* state_dev,
                            const float* lr6, float beta1, float beta2, float eps, void* stream);

/* Sensor frame -> the targets of a4 ("RGB-D frames are processed", Eq. 8-9 :125-131; DESIGN.md reading
 * S33): rgb_dev u8[H][W][3] interleaved colour and depth_dev u16[H][W] in 1/depth_scale metres (0 = no measurement),
 * both DEVICE memory (the caller uploads the 5 bytes per pixel of a camera frame instead of 16).
 * Chat[c][y][x] = rgb[y][x][c] / 255 (f32[3][H][W]), Dhat[y][x] = depth[y][x] / depth_scale (f32[H][W]); one correctly
 * rounded division each, bit-exact against the oracle's unpack_rgbd.  Either pair (rgb_dev, Chat) or (depth_dev, Dhat)
 * may be NULL; depth_scale > 0.  Pointers of any alignment (4 / 8-byte aligned ones take the vector path). */
int32_t ts_unpack_rgbd(ts_ctx* ctx, int32_t W, int32_t H, const uint8_t* rgb_dev, const uint16_t* depth_dev,
                       float depth_scale, float* Chat, float* Dhat, void* stream);

/* NOT part of the rasteriser's API: a measurement helper for bench.py; it enqueues a dependent-free FP32 FMA loop (`iters` rounds of eight
 * independent chains per thread, 2 x 1024 threads per SM) and returns in *flops_out (HOST) the flops it performs; the
 * caller times it with events on `stream` to get the measured FP32 peak.  scratch_dev: one float of device memory. */
int32_t ts_fp32_probe(ts_ctx* ctx, int32_t iters, float* scratch_dev, uint64_t* flops_out, void* stream);

/* ---- forward render without a caller workspace ------------------------------------------------------------ */

/* Everything above needs a frame workspace that the caller allocates (ts_frame_bytes / ts_frame_bind).  A caller that
 * may not allocate device memory while it runs -- a tracking thread that bans cudaMalloc / cudaFree after start-up because
 * they can stall the whole device for an unbounded time, a plug-in inside a process whose device memory all belongs to the
 * host application's arena, a preview path that must still work when HBM is full -- cannot make one.  This call is for
 * them: ts_project + ts_bin_sort + ts_render_fwd (Eq. 1-4) on a workspace that is part of the library
 * image, a static device array of TS_STATIC_WS_BYTES that every GPU which loads libts.so holds until the process exits.
 *
 * Limits (TS_ERR_STATIC_LIMIT beyond them, decided on the host before any launch): scene->M <= TS_STATIC_MAX_FACES and
 * width * height <= TS_STATIC_MAX_PIXELS.  The (tile, face) pair capacity is whatever fits the rest of the array: at
 * least 13 000 pairs at both maxima, more for smaller inputs.  A view with more pairs overflows like any frame: the
 * images come out empty (zero, never out of bounds) and status_dev says so.
 *
 * Arguments as for ts_project (scene, cam, prm, T_cw_dev) and ts_render_fwd (out_color[3][H][W], out_depth[H][W],
 * out_alpha[H][W]; device, any may be NULL).  status_dev: u32[3] DEVICE memory or NULL, receives (n_visible, n_pairs,
 * flags) in stream order; flags != 0 (TS_FLAG_OVERFLOW_*) means the outputs are not a render.  All work is enqueued on
 * `stream`; no synchronisation.  Calls no cudaMalloc / cudaFree / allocating routine (the frame handle is a few hundred
 * bytes of host heap, freed before returning).  Forward only: the frame is gone when the call returns, ts_render_bwd has
 * nothing to follow.
 *
 * Sharing: there is ONE array per GPU and every call uses all of it.  Contents left by an earlier call are harmless (each
 * call clears what the kernels need at zero, in stream order), but two calls whose work overlaps on the GPU -- different
 * streams without an event between them, or two threads -- race on it and both results are garbage.  Serialise them.
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, once per device, cached); make that
 * first call outside of any stream capture. */
#define TS_STATIC_WS_BYTES (4u << 20)
#define TS_STATIC_MAX_FACES 4096
#define TS_STATIC_MAX_PIXELS 16384
int32_t ts_render_fwd_static(ts_ctx* ctx, const ts_scene* scene, const ts_camera* cam, const ts_params* prm,
                             const float* T_cw_dev, float* out_color, float* out_depth, float* out_alpha,
                             uint32_t* status_dev, void* stream);

/* ---- read-only debug accessors (bit-exact tests) ---------------------------------------------------------- */
enum { TS_VIEW_VIS = 0,          /* u32[n_visible][16]: per visible face, in slot order (slots are NOT in face order):
                                    f32 (u,v,w)x3, f32 mean opacity, i16 x0,y0,x1,y1, u32 face, u32 depth_key,
                                    u32 tiles_touched, u32 0                                                  */
       TS_VIEW_KEYS = 1,         /* u64[n_pairs] sorted keys (tile << 32 | depth_key)                        */
       TS_VIEW_VALS = 2,         /* u32[n_pairs][4] sorted (slot, face, rect_lo, rect_hi) entries            */
       TS_VIEW_TILE_RANGES = 3,  /* u32[NT][2]                                                               */
       TS_VIEW_N_CONTRIB = 4,    /* u32[H][W]: 1 + position in the TILE's sorted list of the pixel's last contributing
                                    entry (0 = none); converted on demand from the renderers' per-block counts by a
                                    small launch on `stream`; needs a forward render (ts_render_fwd[_l1/_stats/_normal...])
                                    since the last ts_bin_sort, TS_ERR_STATE otherwise: the fused ts_render_track_l1 /
                                    ts_render_map_l1 do not write the counts                                           */
       TS_VIEW_COUNTERS = 5,     /* u64[8]: n_visit(warp-level), n_rect, n_hit, ... (TS_PARAM_COUNTERS only)  */
       TS_VIEW_JOBS = 6,         /* u32[8 NT][4] job headers of the render kernels, in ticket order: (tile | block << 28,
                                    begin, end, x0 | y0 << 16); block b = 2 row + column of the tile's 2 x 4 blocks of
                                    8x4 pixels; [begin, end) indexes TS_VIEW_BLOCK_LISTS in entries of four u32        */
       TS_VIEW_BLOCK_LISTS = 7,  /* u32[8 n_pairs][4]: the per-block lists: for every job the entries (slot, face,
                                    rect_lo, rect_hi) of its tile's sorted list whose pixel rect overlaps the block, in
                                    list order (only the ranges named by the job headers are defined)                  */
       TS_VIEW_TIMELINE = 8 };   /* u32[8 NT][4], profiling builds only (compiled with -DTS_JOB_TIMELINE by
                                    paper_2605_31419_b200/timeline.py; TS_ERR_STATE in the normal library): per job of
                                    the last ts_render_track_l1, in ticket order like TS_VIEW_JOBS: (%globaltimer at
                                    start, at end [low 32 bits, ns], list length, persistent warp that ran it)         */
/* Synchronises `stream`; returns the device pointer and element count of an internal array. */
int32_t ts_frame_view(ts_ctx* ctx, ts_frame* frame, int32_t which, const void** dev_ptr, size_t* count,
                      void* stream);

#ifdef __cplusplus
}
#endif
#endif
