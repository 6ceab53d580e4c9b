// ts_jobs.cuh -- work distribution of the compositing kernels.
//
// A JOB is one 8x4-pixel block of one 16x16 tile, owned by ONE WARP from start to finish: the warp reads the
// BLOCK's list (the entries of the tile's sorted list whose pixel rect overlaps the block, in list order; built once
// per frame by the sort kernel) 32 entries at a time, drops those whose triangle misses the block (exact cull, one
// entry per lane), copies the records of the others into its private slice of shared memory and walks them.
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

// which = 0 forward, 1 backward.  The ticket is REQUESTED by lane 0 (ts_job_request) and READ later (ts_job_ticket, a
// shuffle), so that its round trip to L2 overlaps whatever lies in between.  Inline PTX on purpose: nvcc turns
// `if (lane == 0) atomicAdd(p, 1)` into a warp-aggregated atomic whose broadcast shuffle waits for the result on the
// spot (5 % of the fused kernel's stall samples sat on that shuffle).
__device__ __forceinline__ uint32_t ts_job_request(const TsFrameDev& f, int which, int lane) {
    uint32_t j = 0;
    if (lane == 0) asm volatile("atom.global.add.u32 %0, [%1], 1;" : "=r"(j) : "l"(&f.ctrl->job_ticket[which]) : "memory");
    return j;
}
__device__ __forceinline__ uint32_t ts_job_ticket(uint32_t requested) { return __shfl_sync(0xffffffffu, requested, 0); }
__device__ __forceinline__ uint32_t ts_job_take(const TsFrameDev& f, int which, int lane) {
    return ts_job_ticket(ts_job_request(f, which, lane));
}

// When is the NEXT ticket taken?  Requesting it at the start of the current job hides the atomic's round trip, but it also
// reserves a job for as long as the current one lasts: a warp on a 60 us job sits on a mid-list ticket all that time and
// runs it afterwards, and at the end of the launch every warp still owes "this job + one reserved job" (measured at config
// 2, profiles/r03_timeline_config2.md: first warp out of work at 71 us, last job finished at 85 us).  So the request is made
// early only where the reservation is short and harmless -- the current job's list has at most TS_PREFETCH_MAX_LEN entries
// and the ticket is not among the last TS_TAIL_ROUNDS x (persistent warps) -- and at the END of the job otherwise (a long
// job does not notice one exposed round trip; in the tail, finishing order matters more than latency).  Warp-uniform.
#ifndef TS_PREFETCH_MAX_LEN
#define TS_PREFETCH_MAX_LEN 8u
#endif
#ifndef TS_TAIL_ROUNDS
#define TS_TAIL_ROUNDS 4u
#endif
__device__ __forceinline__ bool ts_job_prefetch_next(uint32_t j, uint32_t n_jobs, uint32_t list_len, uint32_t total_warps) {
    return list_len <= TS_PREFETCH_MAX_LEN && j + TS_TAIL_ROUNDS * total_warps < n_jobs;
}

// total = persistent warps of the launch
__device__ __forceinline__ void ts_job_finish_n(const TsFrameDev& f, int which, int lane, uint32_t total) {
    if (lane == 0) {
        if (atomicAdd(&f.ctrl->job_done[which], 1u) == total - 1u) {
            // every warp has taken its last ticket: re-arm for the next launch
            f.ctrl->job_ticket[which] = 0u;
            f.ctrl->job_done[which] = 0u;
        }
    }
}
__device__ __forceinline__ void ts_job_finish(const TsFrameDev& f, int which, int lane) {
    ts_job_finish_n(f, which, lane, gridDim.x * TS_JOB_WARPS);
}

__device__ __forceinline__ void ts_job_decode(const TsFrameDev& f, uint32_t j, int lane, TsJob& job) {
    const uint4 h = __ldg(f.job_order + j);     // (tile | block << 28, begin, end, x0 | y0 << 16): one load per job
    job.tile = (int)(h.x & 0x0fffffffu);
    job.blk = (int)(h.x >> 28);
    job.tx0 = (int)(h.w & 0xffffu), job.ty0 = (int)(h.w >> 16);
    job.px = job.tx0 + ((job.blk & 1) << 3) + (lane & 7);
    job.py = job.ty0 + ((job.blk >> 1) << 2) + (lane >> 3);
    job.inside = job.px < f.W && job.py < f.H;
    job.range = make_uint2(h.y, h.z);           // the block's list in f.blist
}

// lane mask of a list entry (slot, face, rect_lo, rect_hi) for this job's block
__device__ __forceinline__ uint32_t ts_entry_mask(const TsJob& job, const uint4 ent) {
    const int rlo = (int)ent.z, rhi = (int)ent.w;
    const int rx0 = max((int)(short)(rlo & 0xffff) - job.tx0, 0), ry0 = max((rlo >> 16) - job.ty0, 0);
    const int rx1 = min((int)(short)(rhi & 0xffff) - job.tx0, 15), ry1 = min((rhi >> 16) - job.ty0, 15);
    return ts_lane_mask(job.blk, rx0, ry0, rx1, ry1);
}
// the exact cull of ts_raster.cuh for this job's block
__device__ __forceinline__ bool ts_job_block_misses(const TsJob& job, const uint4 ent, const float4 r0, const float4 r1,
                                                    const float4 r2) {
    return ts_block_misses(job.tx0 + ((job.blk & 1) << 3), job.ty0 + ((job.blk >> 1) << 2), (int)ent.z, (int)ent.w, r0, r1, r2);
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
