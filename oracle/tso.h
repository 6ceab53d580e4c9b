/* oracle/tso.h -- C ABI of the CPU ORACLE for the Triangle Splatting SLAM rasteriser hot path.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this library.  It shares no
 * source, header, table or helper with paper_2605_31419_b200/csrc/ (the CUDA path) and
 * neither side includes the other.
 *
 * What it computes: Eq. 1-4 of the paper for every pixel, and the analytic
 * reverse-mode gradient of that computation including the se(3) pose Jacobian of Eq. 5-7
 * (PAPER.md:107-119), written step by step in the order F1..F8 / B1..B9 of DESIGN.md
 * section 3.  Plain single-threaded C++17, templated on the scalar: `_f32` (the precision
 * the paper's CUDA rasteriser is assumed to use, and the one integer decisions are taken in)
 * and `_f64` (finite differences, accuracy reference).  No blocking, fusion or reordering:
 * "tiled" mode only restricts the per-pixel loop to the pixel's tile list, "brute" mode loops
 * over every visible face; both use the same per-(pixel, face) function.
 *
 * Pins (tests/test_oracle_*.py): closed forms for one triangle, hand-computed worked example,
 * ray-plane depth, two-layer compositing, invariants, brute == tiled, std::stable_sort,
 * central finite differences for every gradient incl. SE(3) perturbations, rigid-motion
 * identity; normal map: plane coefficients, Eq. 11 on the rendered depth, flat-colour equivalence,
 * finite differences.  Parity unpinned: none.
 *
 * All pointers are HOST pointers owned by the caller.  T = float (_f32) or double (_f64).
 */
#ifndef TSO_H
#define TSO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int32_t width, height;
    double fx, fy, cx, cy, znear;      /* cast to T inside; pass float32-representable values for _f32 */
} tso_camera;

typedef struct {
    double sigma, alpha_min, t_min, eps_area;
    double amb_tol;                    /* relative margin for the "ambiguous decision" flag (0 = off) */
    int32_t min_opacity;               /* 0: face opacity = mean of the vertex opacities (the paper's choice);
                                          1: minimum ("+ min opacity" ablation, Table S3; Mesh Splatting) */
    int32_t tight_binning;             /* 0: a face is binned into every tile its pixel rect touches;
                                          1: only into the tiles its TRIANGLE meets (reading S31, NEXT-4) */
    const void* face_sigma;            /* NULL: the global sigma above (the paper); else [M] per-face window
                                          smoothness in the scalar type of the call (Triangle Splatting's learnable
                                          sigma; reading S32) */
    void* grad_face_sigma;             /* NULL or [M] (+=): dL/dsigma_m, accumulated by tso_render_bwd */
} tso_params;

/* F1-F6: project, cull, bounds, depth key.  faces may be NULL (soup: face m = (3m,3m+1,3m+2)).
 * Outputs (all sized M; entries of culled faces are zero):
 *   visible[M] u8, rect[M][4] i16 (x0,y0,x1,y1 inclusive), depth_key[M] u32 (bits of float(zbar)),
 *   tiles_touched[M] u32, scr[M][9] = (u,v,w=1/Z) x 3, Q[M][9] = camera-space (X,Y,Z) x 3,
 *   zbar[M] (mean camera depth, scalar type T).  Returns number of visible faces. */
int64_t tso_project_f32(const float* pos, const int32_t* faces, int32_t V, int32_t M, const float* T_cw,
                        const tso_camera* cam, const tso_params* prm, uint8_t* visible, int16_t* rect,
                        uint32_t* depth_key, uint32_t* tiles_touched, float* scr, float* Q, float* zbar);
int64_t tso_project_f64(const double* pos, const int32_t* faces, int32_t V, int32_t M, const double* T_cw,
                        const tso_camera* cam, const tso_params* prm, uint8_t* visible, int16_t* rect,
                        uint32_t* depth_key, uint32_t* tiles_touched, double* scr, double* Q, double* zbar);

/* F6 tiled mode: emit (tile<<32 | depth_key, face) pairs for m ascending, ty-major then tx, and
 * std::stable_sort by key.  keys/vals sized P = sum(tiles_touched); ranges[NT][2] = (begin,end).
 * Returns P. */
int64_t tso_bin_sort(int32_t M, int32_t W, int32_t H, const uint8_t* visible, const int16_t* rect,
                     const uint32_t* depth_key, const uint32_t* tiles_touched, uint64_t* keys, uint32_t* vals,
                     uint32_t* ranges);

/* tight binning (tso_params.tight_binning = 1): as tso_bin_sort, with the tiles chosen by the overlap rule S31 from the
 * projected vertices scr[M][9] of tso_project (same precision as the project call that counted tiles_touched). */
int64_t tso_bin_sort_tight_f32(int32_t M, int32_t W, int32_t H, const uint8_t* visible, const int16_t* rect,
                               const uint32_t* depth_key, const float* scr, uint64_t* keys, uint32_t* vals, uint32_t* ranges);
int64_t tso_bin_sort_tight_f64(int32_t M, int32_t W, int32_t H, const uint8_t* visible, const int16_t* rect,
                               const uint32_t* depth_key, const double* scr, uint64_t* keys, uint32_t* vals, uint32_t* ranges);

/* F7-F8 forward.  If tile_ranges == NULL: brute mode, `list` holds n_list visible face ids in global depth
 * order and every pixel walks all of it.  Else tiled mode: `list` = sorted vals, tile_ranges[NT][2].
 * Outputs: out_color[3][H][W], out_depth[H][W], out_alpha[H][W]; optional (may be NULL):
 *   n_contrib[H][W] (1 + list position, relative to the walk start, of the last contributing face; 0 = none),
 *   ambig[H][W] u8 (a decision was within amb_tol of flipping), sig[H][W] u64 (hash of the hit sequence),
 *   counters[4] = {N_visit, N_rect, N_hit, 0} (u64). */
void tso_render_fwd_f32(const float* color, const float* opacity, const int32_t* faces, int32_t M,
                        const tso_camera* cam, const tso_params* prm, const uint8_t* visible, const int16_t* rect,
                        const float* scr, const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges,
                        float* out_color, float* out_depth, float* out_alpha, uint32_t* n_contrib, uint8_t* ambig,
                        uint64_t* sig, uint64_t* counters);
void tso_render_fwd_f64(const double* color, const double* opacity, const int32_t* faces, int32_t M,
                        const tso_camera* cam, const tso_params* prm, const uint8_t* visible, const int16_t* rect,
                        const double* scr, const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges,
                        double* out_color, double* out_depth, double* out_alpha, uint32_t* n_contrib,
                        uint8_t* ambig, uint64_t* sig, uint64_t* counters);

/* B1-B6 backward of the compositing.  Same list arguments as forward.  dL_dcolor[3][H][W], dL_ddepth[H][W],
 * dL_dalpha[H][W] (any may be NULL = 0).  Accumulates (+=) into grad_color[V][3], grad_opacity[V] (may be NULL) and
 * g_scr[M][9] = dL/d(u,v,w) per face vertex (caller zeroes). */
void tso_render_bwd_f32(const float* color, const float* opacity, const int32_t* faces, int32_t M,
                        const tso_camera* cam, const tso_params* prm, const uint8_t* visible, const int16_t* rect,
                        const float* scr, const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges,
                        const float* dL_dcolor, const float* dL_ddepth, const float* dL_dalpha, float* grad_color,
                        float* grad_opacity, float* g_scr);
void tso_render_bwd_f64(const double* color, const double* opacity, const int32_t* faces, int32_t M,
                        const tso_camera* cam, const tso_params* prm, const uint8_t* visible, const int16_t* rect,
                        const double* scr, const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges,
                        const double* dL_dcolor, const double* dL_ddepth, const double* dL_dalpha,
                        double* grad_color, double* grad_opacity, double* g_scr);

/* B7-B9: screen -> camera -> world / pose.  grad_pos[V][3] += R^T g_C (may be NULL); dL_dtau[6] = sum over
 * visible face vertices of [g_C ; Q x g_C] (overwritten; may be NULL), tau = (rho, theta), left perturbation. */
void tso_project_bwd_f32(const int32_t* faces, int32_t M, const float* T_cw, const tso_camera* cam,
                         const uint8_t* visible, const float* Q, const float* g_scr, float* grad_pos,
                         float* dL_dtau);
void tso_project_bwd_f64(const int32_t* faces, int32_t M, const double* T_cw, const tso_camera* cam,
                         const uint8_t* visible, const double* Q, const double* g_scr, double* grad_pos,
                         double* dL_dtau);

/* Harness helper a4: L = 1/(3HW) sum|C-Chat| + lambda_dep/(HW) sum_{Dhat>0}|D-Dhat|; sign(0)=0.
 * Writes gC[3][H][W], gD[H][W]; returns L (as double). */
double tso_l1_loss_f32(int32_t W, int32_t H, const float* C, const float* D, const float* Chat, const float* Dhat,
                       double lambda_dep, float* gC, float* gD);
double tso_l1_loss_f64(int32_t W, int32_t H, const double* C, const double* D, const double* Chat,
                       const double* Dhat, double lambda_dep, double* gC, double* gD);

/* Harness helper a8: one Adam step on tau followed by T <- Exp(-delta) o T.
 * state[13] = m[6], v[6], step count.  lr[6] per component. */
void tso_pose_step_f32(float* T_cw, const float* dL_dtau, float* state, const float* lr, float beta1, float beta2,
                       float eps);

/* E_equi of Eq. 14: mean over faces and their three internal angles of (cos theta - 0.5)^2, world
 * space.  faces may be NULL (soup).  Returns E; grad_pos[V][3] (may be NULL) += weight * dE/dpos. */
double tso_equi_f32(const float* pos, const int32_t* faces, int32_t M, double weight, float* grad_pos);
double tso_equi_f64(const double* pos, const int32_t* faces, int32_t M, double weight, double* grad_pos);

/* D-SSIM term of Eq. 8: L = 1 - mean SSIM over 3 channels x H x W, 11x11 Gaussian window
 * (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2 (reading S25).  x = rendered [3][H][W], y = reference.
 * Returns L; g (may be NULL) receives dL/dx. */
double tso_dssim_f32(int32_t W, int32_t H, const float* x, const float* y, float* g);
double tso_dssim_f64(int32_t W, int32_t H, const double* x, const double* y, double* g);

/* Per-face statistics of a render (map management): face_pixels[M] = number of pixels the
 * face contributed to (same walk, hit rule and termination as tso_render_fwd); proj_area[M] = |S|/2 in px^2 (F4),
 * 0 for culled faces.  Either output may be NULL. */
void tso_face_stats_f32(const float* color, const float* opacity, const int32_t* faces, int32_t M, const tso_camera* cam,
                        const tso_params* prm, const uint8_t* visible, const int16_t* rect, const float* scr,
                        const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges, uint32_t* face_pixels,
                        float* proj_area);
void tso_face_stats_f64(const double* color, const double* opacity, const int32_t* faces, int32_t M, const tso_camera* cam,
                        const tso_params* prm, const uint8_t* visible, const int16_t* rect, const double* scr,
                        const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges, uint32_t* face_pixels,
                        double* proj_area);

/* Rendered normal map of Eq. 12, reading S26: N(p) = sum_n n_n alpha_n T_n with n_n the
 * unit normal of the face plane in CAMERA space, oriented towards the camera (n . Q_0 < 0), not renormalised.
 *   tso_face_normal      nrm[M][3] from the world edges rotated by R (zero for culled faces)
 *   tso_render_normal_fwd  out_normal[3][H][W]; same walk, hit rule and termination as tso_render_fwd
 *   tso_render_normal_bwd  dL_dnormal[3][H][W] -> grad_opacity[V] (+=, may be NULL), g_scr[M][9] (+=, the window path
 *                          only: a flat attribute has no interpolation term) and g_nrm[M][3] (+=)
 *   tso_face_normal_bwd  g_nrm -> grad_pos[V][3] (+=, may be NULL) and dL_dtau[6] (+=, may be NULL; rotation part only) */
#define TSO_NRM_DECL(T, sfx)                                                                                           \
    void tso_face_normal_##sfx(const T* pos, const int32_t* faces, int32_t M, const T* T_cw, const uint8_t* visible,  \
                               const T* Q, T* nrm);                                                                    \
    void tso_face_normal_bwd_##sfx(const T* pos, const int32_t* faces, int32_t M, const T* T_cw,                       \
                                   const uint8_t* visible, const T* Q, const T* g_nrm, T* grad_pos, T* dL_dtau);       \
    void tso_render_normal_fwd_##sfx(const T* color, const T* opacity, const int32_t* faces, int32_t M,                \
                                     const tso_camera* cam, const tso_params* prm, const uint8_t* visible,             \
                                     const int16_t* rect, const T* scr, const uint32_t* list, int64_t n_list,          \
                                     const uint32_t* tile_ranges, const T* nrm, T* out_normal);                        \
    void tso_render_normal_top_##sfx(const T* color, const T* opacity, const int32_t* faces, int32_t M,                \
                                     const tso_camera* cam, const tso_params* prm, const uint8_t* visible,             \
                                     const int16_t* rect, const T* scr, const uint32_t* list, int64_t n_list,          \
                                     const uint32_t* tile_ranges, const T* nrm, T* out_normal_top);                    \
    void tso_render_normal_bwd_##sfx(const T* color, const T* opacity, const int32_t* faces, int32_t M,                \
                                     const tso_camera* cam, const tso_params* prm, const uint8_t* visible,             \
                                     const int16_t* rect, const T* scr, const uint32_t* list, int64_t n_list,          \
                                     const uint32_t* tile_ranges, const T* nrm, const T* dL_dnormal, T* grad_opacity,  \
                                     T* g_scr, T* g_nrm);
TSO_NRM_DECL(float, f32)
TSO_NRM_DECL(double, f64)

/* tso_render_normal_top (above): the "normal direction of the triangle with highest opacity along each ray" of Fig. 3
 * (PAPER.md:145), reading S29: among the hits the walk composites (same hit rule and termination), the face
 * normal of the FIRST hit with the largest alpha = face opacity x window; zero where nothing is hit.  Forward only.
 *
 * Normalised depth D / A: Dn = D / A where A > eps, else 0; backward of a cotangent gDn:
 * gD += gDn / A, gA += -gDn D / A^2.  n = H W elements. */
void tso_depth_normalise_f32(int64_t n, const float* D, const float* A, float eps, float* Dn);
void tso_depth_normalise_f64(int64_t n, const double* D, const double* A, double eps, double* Dn);
void tso_depth_normalise_bwd_f32(int64_t n, const float* D, const float* A, float eps, const float* gDn, float* gD, float* gA);
void tso_depth_normalise_bwd_f64(int64_t n, const double* D, const double* A, double eps, const double* gDn, double* gD, double* gA);

/* E_norm of Eq. 12: weight / (H W) * sum over valid pixels (Nbar_p != 0) of 1 - N_p . Nbar_p
 * (reading S27).  N, Nbar, gN are [3][H][W]; gN receives the cotangent of N; returns the weighted loss. */
double tso_normal_loss_f32(int32_t W, int32_t H, const float* N, const float* Nbar, double weight, float* gN);
double tso_normal_loss_f64(int32_t W, int32_t H, const double* N, const double* Nbar, double weight, double* gN);

/* Screen-space gradient statistic of the densification test (reading S28): per face,
 * ||sum_k (dL/du_k, dL/dv_k)||_2 from g_scr[M][9] of tso_render_bwd.  face_grad2d[M] += it, face_views[M] += 1 (may be
 * NULL) for every visible face that received a gradient. */
void tso_screen_grad_stat_f32(int32_t M, const uint8_t* visible, const float* g_scr, float* face_grad2d, uint32_t* face_views);
void tso_screen_grad_stat_f64(int32_t M, const uint8_t* visible, const double* g_scr, double* face_grad2d, uint32_t* face_views);

/* SE(3) exponential, tau = (rho, theta): out[12] = Exp(tau) o T (3x4 row-major). */
void tso_left_perturb_f64(const double* T_cw, const double* tau, double* out);

#ifdef __cplusplus
}
#endif
#endif
