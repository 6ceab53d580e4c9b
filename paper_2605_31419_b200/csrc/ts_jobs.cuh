// ts_jobs.cuh -- work distribution of the compositing kernels.
//
// A JOB is one 8x4-pixel block of one 16x16 tile, owned by ONE WARP from start to finish: the warp reads the
// tile's sorted list 32 entries at a time, keeps the entries whose pixel rect overlaps its block (one lane mask per
// entry, one ballot per chunk), copies their records into its private slice of shared memory and walks them.
// There is no CTA-wide barrier anywhere: warps never wait for each other, so a crowded block does not stall the
// seven other blocks of its tile, and nobody idles while records are being fetched.
//
// Jobs are pulled from a global ticket counter by persistent warps (grid = a few CTAs per SM), in the order
// tile_order[] fixes: tiles with the longest lists first, so the tail of the launch is made of the cheapest jobs.
// The last warp to finish re-zeroes the ticket and the finish counter ("zero at rest": graph replays need no memset).
#pragma once
#include "ts_raster.cuh"

#define TS_JOB_WARPS 8               // warps per CTA of the render kernels
#define TS_BLOCKS_PER_TILE 8         // 8x4 blocks in a 16x16 tile

struct TsJob {
    int tile, blk, px, py;           // px, py: this lane's pixel
    int tx0, ty0;                    // tile origin
    uint2 range;
    bool inside;
};

// which = 0 forward, 1 backward
__device__ __forceinline__ uint32_t ts_job_take(const TsFrameDev& f, int which, int lane) {
    uint32_t j = 0;
    if (lane == 0) j = atomicAdd(&f.ctrl->job_ticket[which], 1u);
    return __shfl_sync(0xffffffffu, j, 0);
}

__device__ __forceinline__ void ts_job_finish(const TsFrameDev& f, int which, int lane) {
    if (lane == 0) {
        const uint32_t total = gridDim.x * TS_JOB_WARPS;
        if (atomicAdd(&f.ctrl->job_done[which], 1u) == total - 1u) {
            // every warp has taken its last ticket: re-arm for the next launch
            f.ctrl->job_ticket[which] = 0u;
            f.ctrl->job_done[which] = 0u;
        }
    }
}

__device__ __forceinline__ void ts_job_decode(const TsFrameDev& f, uint32_t j, int lane, TsJob& job) {
    job.tile = (int)__ldg(f.tile_order + (j >> 3));
    job.blk = (int)(j & 7u);
    job.tx0 = (job.tile % f.tiles_x) * TS_TILE, job.ty0 = (job.tile / f.tiles_x) * TS_TILE;
    job.px = job.tx0 + ((job.blk & 1) << 3) + (lane & 7);
    job.py = job.ty0 + ((job.blk >> 1) << 2) + (lane >> 3);
    job.inside = job.px < f.W && job.py < f.H;
    job.range = f.tile_ranges[job.tile];
}

// lane mask of a sorted-list entry (slot, face, rect_lo, rect_hi) for this job's block
__device__ __forceinline__ uint32_t ts_entry_mask(const TsJob& job, const uint4 ent) {
    const int rlo = (int)ent.z, rhi = (int)ent.w;
    const int rx0 = max((int)(short)(rlo & 0xffff) - job.tx0, 0), ry0 = max((rlo >> 16) - job.ty0, 0);
    const int rx1 = min((int)(short)(rhi & 0xffff) - job.tx0, 15), ry1 = min((rhi >> 16) - job.ty0, 15);
    return ts_lane_mask(job.blk, rx0, ry0, rx1, ry1);
}

// the nine vertex-colour floats of a face
__device__ __forceinline__ void ts_load_colors(const ts_scene& sc, uint32_t face, float col[9]) {
    if (sc.faces == nullptr) {
        const float* cp = sc.color + 9 * (size_t)face;
#pragma unroll
        for (int j = 0; j < 9; ++j) col[j] = __ldg(cp + j);
    } else {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const float* cp = sc.color + 3 * (size_t)__ldg(sc.faces + 3 * (size_t)face + k);
            col[3 * k] = __ldg(cp), col[3 * k + 1] = __ldg(cp + 1), col[3 * k + 2] = __ldg(cp + 2);
        }
    }
}
