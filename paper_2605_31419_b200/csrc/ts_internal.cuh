// ts_internal.cuh -- shared declarations of the CUDA path (sm_100a only).  Not part of the public ABI.
// Shares nothing with oracle/ (the CPU oracle): no header, helper, table or constant generator.
#pragma once
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>
#include <stdint.h>

#include "../../include/ts.h"

#define TS_TILE 16
#define TS_PROJ_THREADS 256          // faces per project CTA
#define TS_BIN_THREADS 1024          // visible slots per bin/setup CTA iteration (one CTA per SM: one tile scan per SM)
#define TS_SCAN_LOCAL_MAX 4096       // up to this many tiles every binning CTA scans the tile counts itself (smem)
#define TS_SORT_THREADS 128
#define TS_SORT_SMEM 2048            // tile lists up to this length are sorted in shared memory
#define TS_BATCH 128                 // list entries staged per batch in the forward kernel
#define TS_BATCH_BWD 64              // ... in the backward kernel (records are twice as large)
#define TS_REC_F4 10                 // float4 per face record (160 B)
#define TS_SCR_F4 4                  // float4 per raw projected record (64 B)

// Device control block (one per frame, lives at the start of the workspace).  Every field that a kernel
// accumulates into is back at zero when that kernel's grid has finished ("zero at rest"), so a frame can be
// re-used by graph replays without host-side clears.
struct TsCtrl {
    uint32_t n_visible;      // faces surviving the cull (may exceed vis_cap on overflow)
    uint32_t n_pairs;        // (tile, face) pairs (may exceed pair_cap on overflow)
    uint32_t flags;          // TS_FLAG_*
    uint32_t max_list;       // longest tile list of the last ts_project
    uint32_t vis_counter;    // slot allocator of the project kernel (zeroed by the sort kernel)
    uint32_t job_ticket[2];  // work queues of the forward / backward render kernels (zero at rest)
    uint32_t job_done[2];    // warps finished, per render kernel (zero at rest)
    uint32_t reduce_done;    // pose-reduction CTAs finished (zero at rest)
    uint32_t pad[2];
    unsigned long long counters[8];   // debug counters (TS_PARAM_COUNTERS)
    uint32_t bucket_cursor[32];       // per list-length bucket: job headers published so far (zeroed by the sort kernel)
};

// Everything a kernel needs to know about a frame; passed by value.
struct TsFrameDev {
    int32_t M, W, H, tiles_x, tiles_y, NT;
    uint32_t pair_cap, vis_cap;
    uint32_t prm_flags;               // ts_params.flags of the last ts_project (host-side copy, travels with the launches)
    TsCtrl* ctrl;
    uint32_t* tile_count;             // [NT] pairs per tile, counted by the project kernel (zeroed by the sort kernel)
    uint32_t* tile_cursor;            // [NT] write cursor of the binning pass, relative to the tile's begin (zero at rest)
    uint32_t* tile_offset;            // [NT] exclusive scan of tile_count (only used when NT > TS_SCAN_LOCAL_MAX)
    uint4* tile_order;                // [NT] tile headers (tile, begin, end, x0 | y0 << 16), tiles by descending list length
    uint2* tile_ranges;               // [NT] (begin, end) into the pair arrays
    float4* scr;                      // [vis_cap][4]: (u0,v0,w0,u1) (v1,w1,u2,v2) (w2,obar,rect_lo,rect_hi) (face,key,tiles,0)
    float4* rec;                      // [vis_cap][10]: per-face render record, see ts_raster.cuh
    float* gscr;                      // [vis_cap][9]: dL/d(u,v,w) per face vertex (full-gradient mode), zero at rest
    float4* nrm;                      // [vis_cap]: camera-space unit face normal towards the camera (normal-map calls only)
    float* gnrm;                      // [vis_cap][3]: dL/dn per face (normal-map backward), zero at rest
    uint4* pair_a;                    // [pair_cap] binned, unsorted: (depth_key, face, slot, rect_lo)
    uint32_t* pair_b;                 // [pair_cap] binned, unsorted: rect_hi
    unsigned long long* big_key;      // [pair_cap] scratch of the oversize-segment sort
    uint32_t* big_idx;                // [pair_cap] scratch of the oversize-segment sort
    unsigned long long* skey;         // [pair_cap] sorted: tile << 32 | depth_key
    uint4* sorted;                    // [pair_cap] sorted: (slot, face, rect_lo, rect_hi)
    uint4* blist;                     // [8 * pair_cap] per-BLOCK lists, what the renderers walk: the entries (slot, face,
                                      // rect_lo, rect_hi) of a tile's sorted list whose pixel rect overlaps the 8x4-pixel
                                      // block, in list order; block k of a tile whose list is [b, e) owns
                                      // [8 b + k (e - b), 8 b + (k + 1)(e - b))
    uint4* job_order;                 // [8 * NT] job headers (tile | block << 28, begin, end into blist, x0 | y0 << 16);
                                      // job 8 p + k = block k of the tile at position p of tile_order
    uint32_t* n_contrib;              // [H*W] per pixel: 1 + the position IN ITS BLOCK'S LIST of the last contributing entry
    uint32_t* n_contrib_view;         // [H*W] scratch of TS_VIEW_N_CONTRIB (positions in the tile's list)
    float* t_last;                    // [H*W] transmittance in front of the last contributing face
    float* pose_partials;             // [n_partials_cap][6], then [32][6] block partials of the final reduction
    uint32_t n_partials_cap;
};

struct TsCamDev { int32_t W, H; float fx, fy, cx, cy, znear; };
struct TsPrmDev { float sigma, alpha_min, t_min, eps_area; uint32_t flags; };

// Host-side handle.
struct ts_ctx {
    int device;
    int num_sms;
    int max_smem_optin;
    int tracing;             // ts_set_tracing: every launching export brackets itself with an NVTX range named after it
};
struct ts_frame {
    TsFrameDev d;
    TsCamDev cam;
    TsPrmDev prm;
    const float* T_cw;       // device pointer given to the last ts_project (read again by the projection backward)
    const float* face_sigma; // ts_frame_set_face_sigma: per-face window smoothness [M] (NULL = the global sigma of ts_params)
    float* grad_sigma;       // ... and where the full-gradient backward adds dL/dsigma_m [M] (may be NULL)
    int have_project, have_sort, have_fwd;
    int have_normals;        // f.nrm holds the face normals of the current projection (ts_render_fwd_normal ran)
    int counters_dirty;      // ts_project ran but ts_bin_sort has not consumed (and re-zeroed) its counters yet
    uint32_t pose_src;       // 0 = none, 1 = per-tile partials (pose-only), 2 = per-block partials (projection backward)
    uint32_t n_pose_partials;
    size_t bytes;
    void* base;
};

// every launching export runs on the device of its context (ts_create): a mismatch with the current device is an
// argument error, not a launch on the wrong GPU
inline bool on_ctx_device(const ts_ctx* ctx) {
    int cur = -1;
    return ctx && cudaGetDevice(&cur) == cudaSuccess && cur == ctx->device;
}

// NVTX range around one export (tracing): pushed on entry and popped on every return path when the
// context has tracing on; nothing but a load and a branch otherwise.  The range covers the HOST side of the call (argument
// checks and the enqueue); a profiler attributes the kernels launched inside it to the range.
struct TsTraceRange {
    bool on;
    TsTraceRange(const ts_ctx* ctx, const char* name) : on(ctx && ctx->tracing) {
        if (on) nvtxRangePushA(name);
    }
    ~TsTraceRange() {
        if (on) nvtxRangePop();
    }
    TsTraceRange(const TsTraceRange&) = delete;
    TsTraceRange& operator=(const TsTraceRange&) = delete;
};
#define TS_TRACE(ctx) TsTraceRange ts_trace_range__((ctx), __func__)

#define TS_CUDA_CHECK_LAUNCH()                              \
    do {                                                    \
        cudaError_t e__ = cudaGetLastError();               \
        if (e__ != cudaSuccess) return TS_ERR_CUDA;         \
    } while (0)

// effective counts: an overflowed frame renders nothing (outputs stay in bounds)
__device__ __forceinline__ uint32_t ts_eff_pairs(const TsFrameDev& f) {
    const volatile TsCtrl* c = f.ctrl;
    return (c->flags != 0) ? 0u : c->n_pairs;
}
__device__ __forceinline__ uint32_t ts_eff_visible(const TsFrameDev& f) {
    const volatile TsCtrl* c = f.ctrl;
    return (c->flags != 0) ? 0u : c->n_visible;
}

// Tight binning (ts_params.flags & TS_PARAM_TIGHT_BINNING; reading S31): does the triangle with screen
// vertices (u_k, v_k) meet the box of pixel centres [bx0,bx1] x [by0,by1]?  For each edge k (from q_{k+1} to q_{k+2})
// the un-normalised outward edge function E_k(p) = s (ey (px - ua) - ex (py - va)) is taken at the corner of the box
// where it is smallest; the box is left out iff some E_k there exceeds 2^-10 (|ex| + |ey|): every pixel of the box is
// then at least ~1e-3 px outside edge k and cannot pass the hit rule.  Explicit round-to-nearest operations in a fixed
// order: the decision is bit-identical to the float32 oracle's, and to itself in the projection and binning kernels.
__device__ __forceinline__ bool ts_tile_overlaps(const float u[3], const float v[3], int bx0, int by0, int bx1, int by1) {
    const float a = __fsub_rn(u[1], u[0]), b = __fsub_rn(v[2], v[0]), c = __fsub_rn(v[1], v[0]), d = __fsub_rn(u[2], u[0]);
    const float S = __fmaf_rn(a, b, -__fmul_rn(c, d));
    const float s = S > 0.0f ? 1.0f : -1.0f;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const int ia = (k + 1) % 3, ib = (k + 2) % 3;
        const float ex = __fsub_rn(u[ib], u[ia]), ey = __fsub_rn(v[ib], v[ia]);
        const float sx = __fmul_rn(s, ey), sy = -__fmul_rn(s, ex);
        const float px = sx > 0.0f ? (float)bx0 : (float)bx1, py = sy > 0.0f ? (float)by0 : (float)by1;
        const float dx = __fsub_rn(px, u[ia]), dy = __fsub_rn(py, v[ia]);
        const float E = __fmaf_rn(sx, dx, __fmul_rn(sy, dy));
        const float margin = __fmul_rn(0.0009765625f, __fadd_rn(fabsf(ex), fabsf(ey)));
        if (E > margin) return false;
    }
    return true;
}
// is tile (tx, ty) of the face's rect [x0,x1] x [y0,y1] one the face is binned into?
__device__ __forceinline__ bool ts_tile_included(bool tight, const float u[3], const float v[3], int x0, int y0, int x1, int y1,
                                                 int tx, int ty) {
    if (!tight) return true;
    return ts_tile_overlaps(u, v, max(x0, tx * TS_TILE), max(y0, ty * TS_TILE), min(x1, tx * TS_TILE + TS_TILE - 1),
                            min(y1, ty * TS_TILE + TS_TILE - 1));
}

// launchers (one per .cu)
int32_t ts_launch_project(const ts_ctx*, ts_frame*, const ts_scene*, cudaStream_t);
int32_t ts_launch_sort(const ts_ctx*, ts_frame*, cudaStream_t);
int32_t ts_launch_render_fwd(const ts_ctx*, ts_frame*, const ts_scene*, float* oc, float* od, float* oa, const float* Chat,
                             const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss, uint32_t* face_pixels,
                             cudaStream_t);
int32_t ts_launch_face_area(const ts_ctx*, ts_frame*, float* area, cudaStream_t);
int32_t ts_launch_ncontrib_view(const ts_ctx*, ts_frame*, cudaStream_t);
int32_t ts_launch_render_fwd_normal(const ts_ctx*, ts_frame*, const ts_scene*, float* oc, float* od, float* oa, float* on,
                                    cudaStream_t, float* on_top = nullptr);
int32_t ts_launch_render_bwd_normal(const ts_ctx*, ts_frame*, const ts_scene*, const float* gC, const float* gD,
                                    const float* gA, const float* gN, float* grad_pos, float* grad_color,
                                    float* grad_opacity, uint32_t mask, cudaStream_t);
int32_t ts_launch_render_bwd(const ts_ctx*, ts_frame*, const ts_scene*, const float*, const float*, const float*,
                             float*, float*, float*, uint32_t, cudaStream_t, float* face_grad2d = nullptr,
                             uint32_t* face_views = nullptr);
int32_t ts_launch_render_track(const ts_ctx*, ts_frame*, const ts_scene*, float* oc, float* od, float* oa, const float* Chat,
                               const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss, cudaStream_t);
int32_t ts_launch_render_map(const ts_ctx*, ts_frame*, const ts_scene*, float* oc, float* od, float* oa, const float* Chat,
                             const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss, float* grad_pos,
                             float* grad_color, float* grad_opacity, uint32_t mask, cudaStream_t);
int32_t ts_launch_pose_reduce(const ts_ctx*, ts_frame*, float* out, float* T_cw, float* state, const float* lr6, float beta1,
                              float beta2, float eps, cudaStream_t);
