// ts_internal.cuh -- shared declarations of the CUDA path (sm_100a only).  Not part of the public ABI.
// Shares nothing with oracle/ (the CPU oracle): no header, helper, table or constant generator.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ts.h"

#define TS_TILE 16
#define TS_PROJ_THREADS 256          // faces per project tile
#define TS_SORT_THREADS 256
#define TS_SORT_ITEMS 8              // keys per thread per onesweep tile
#define TS_SORT_TILE (TS_SORT_THREADS * TS_SORT_ITEMS)
#define TS_RADIX_BITS 8
#define TS_RADIX 256
#define TS_MAX_PASSES 8
#define TS_BATCH 128                 // list entries staged per batch in the render kernels

// Device control block (one per frame, lives at the start of the workspace).
struct TsCtrl {
    uint32_t n_visible;      // faces surviving the cull (may exceed vis_cap on overflow)
    uint32_t n_pairs;        // (tile, face) pairs emitted (may exceed pair_cap on overflow)
    uint32_t flags;          // TS_FLAG_*
    uint32_t epoch;          // chained-scan epoch (1..15), advanced by the last project block
    uint32_t proj_ticket;    // dynamic tile id of the project kernel
    uint32_t proj_done;      // blocks finished
    uint32_t sort_ticket[TS_MAX_PASSES];
    uint32_t max_list;       // longest tile list (hybrid path)
    uint32_t pad[1];
    unsigned long long counters[8];   // debug counters
};

// Everything a kernel needs to know about a frame; passed by value.
struct TsFrameDev {
    int32_t M, W, H, tiles_x, tiles_y, NT;
    uint32_t pair_cap, vis_cap;
    int32_t key_bits, n_passes;
    uint32_t n_proj_tiles, n_sort_tiles_cap;
    TsCtrl* ctrl;
    unsigned long long* scan_state;   // [n_proj_tiles]
    uint32_t* vis_face;               // [vis_cap]
    int2* rect;                       // [vis_cap]  (x0 | y0<<16, x1 | y1<<16) as int16 pairs
    uint32_t* depth_key;              // [vis_cap]
    uint32_t* tiles_touched;          // [vis_cap]
    float4* scr;                      // [vis_cap][3]: (u0,v0,w0,u1) (v1,w1,u2,v2) (w2, obar, rect_lo, rect_hi)
    float* gscr;                      // [vis_cap][9]: dL/d(u,v,w) per face vertex (full-gradient mode), kept zero
    unsigned long long* keys[2];      // [pair_cap] ping-pong
    uint32_t* vals[2];                // [pair_cap]
    uint32_t* hist;                   // [TS_MAX_PASSES][256]
    uint32_t* sort_state;             // [n_passes][n_sort_tiles_cap][256]
    uint2* tile_ranges;               // [NT]
    uint32_t* n_contrib;              // [H*W]
    float* t_last;                    // [H*W] transmittance in front of the last contributing face
    float* pose_partials;             // [n_partials_cap][6]
    uint32_t n_partials_cap;
};

struct TsCamDev { int32_t W, H; float fx, fy, cx, cy, znear; };
struct TsPrmDev { float sigma, alpha_min, t_min, eps_area; uint32_t flags; };

// Host-side handle.
struct ts_ctx {
    int device;
    int num_sms;
    int max_smem_optin;
};
struct ts_frame {
    TsFrameDev d;
    TsCamDev cam;
    TsPrmDev prm;
    const float* T_cw;       // device pointer given to the last ts_project
    int sorted_buf;          // which ping-pong buffer holds the sorted pairs
    int have_project, have_sort, have_fwd;
    uint32_t pose_src;       // 0 = none, 1 = per-tile partials (pose-only), 2 = per-block partials (epilogue)
    uint32_t n_pose_partials;
    size_t bytes;
    void* base;
};

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

// launchers (one per .cu)
int32_t ts_launch_project(const ts_ctx*, ts_frame*, const ts_scene*, cudaStream_t);
int32_t ts_launch_sort(const ts_ctx*, ts_frame*, cudaStream_t);
int32_t ts_launch_render_fwd(const ts_ctx*, ts_frame*, const ts_scene*, float*, float*, float*, cudaStream_t);
int32_t ts_launch_render_bwd(const ts_ctx*, ts_frame*, const ts_scene*, const float*, const float*, const float*,
                             float*, float*, float*, uint32_t, cudaStream_t);
int32_t ts_launch_pose_reduce(const ts_ctx*, ts_frame*, float*, cudaStream_t);
