// ts_render_bwd.cu -- a5/a6/a7: reverse-order backward of the compositing (B1-B9).
//   render_bwd_kernel : persistent warps, one 8x4-pixel block per job (ts_jobs.cuh), one pixel per lane; walks the
//       tile list BACK from the block's last contributing entry, 32 entries at a time; recomputes alpha
//       bit-identically to the forward kernel (ts_raster.cuh), recovers the transmittance in front of each face by
//       T_n = T_{n+1}/(1-alpha_n), keeps ONE scalar "behind" accumulator R = R^c.gC + R^d gD + R^a gA (no division
//       by T), and forms the per-hit gradients wrt the face's screen vertices (u,v,w) x 3, its vertex colours and
//       its opacity.
//       POSE-ONLY mode (tracking): the per-pixel walk only does the sequential part of a hit (alpha, T_n, dL/dalpha)
//       and queues it; whenever 32 hits are queued every lane finishes one of them (B4-B6, then the nine screen
//       terms straight through d(u,v,w)/dtau, Eq. 5-7) into six per-thread accumulators --
//       all 32 lanes busy instead of the ~8 that hit a given face, no shuffle, no atomic, no per-face buffer.
//       The accumulators are tree-reduced once per job into a per-job partial (fixed order: deterministic).
//       FULL mode (mapping): per face the terms are reduced across the warp with shuffles BEFORE any global
//       atomic (one lane issues the RED.ADD.F32s).
//   proj_bwd_kernel   : full mode only; per visible face, screen -> camera -> world (B7-B8) and the se(3) terms
//       [g_C ; Q x g_C], tree-reduced per CTA into fixed-order partials.
//   pose_reduce_kernel: fixed-order final reduction of the partials to dL/dtau[6].
#include "ts_bwd_job.cuh"
#include "ts_fwd_job.cuh"
#include "ts_normal.cuh"
#include "ts_pose.cuh"

#include <cooperative_groups.h>
namespace cg = cooperative_groups;

namespace {

// ATTR: colour / opacity gradients (B1, B4).  GEOM: screen-space vertex gradients into gscr (B5-B6).
// POSE: pose-only; hits are queued by the per-pixel walk and finished 32 at a time (ts_bwd_pose_hit).
// NRM: also the cotangent of the rendered normal map (Eq. 12); full-gradient mode only.
template <int SM, bool ATTR, bool GEOM, bool POSE, bool NRM = false>
__global__ void __launch_bounds__(TS_JOB_WARPS * 32, NRM ? 2 : 3)
render_bwd_kernel(TsFrameDev f, ts_scene sc, float sigma, float alpha_min, float fx, float fy,
                  const float* __restrict__ gCi, const float* __restrict__ gDi, const float* __restrict__ gAi,
                  float* __restrict__ grad_color, float* __restrict__ grad_opacity, const float* __restrict__ gNi = nullptr,
                  float* __restrict__ grad_sigma = nullptr) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    BwdWarpSmem& sm = reinterpret_cast<BwdWarpSmem*>(smem_raw)[threadIdx.x >> 5];
    const uint32_t n_jobs = (uint32_t)f.NT * TS_BLOCKS_PER_TILE;
    const size_t hw = (size_t)f.W * f.H;

    uint32_t j = ts_job_take(f, 1, lane);
    while (j < n_jobs) {
        TsJob job;
        ts_job_decode(f, j, lane, job);
        const size_t p = (size_t)job.py * f.W + job.px;
        uint32_t ncon = 0;
        float Tcur = 1.0f, gC0 = 0.f, gC1 = 0.f, gC2 = 0.f, gD = 0.f, gA = 0.f, gN0 = 0.f, gN1 = 0.f, gN2 = 0.f;
        if (job.inside && job.range.y > job.range.x) {
            ncon = f.n_contrib[p];
            Tcur = f.t_last[p];
            if (gCi) gC0 = gCi[p], gC1 = gCi[hw + p], gC2 = gCi[2 * hw + p];
            if (gDi) gD = gDi[p];
            if (gAi) gA = gAi[p];
            if (NRM) gN0 = gNi[p], gN1 = gNi[hw + p], gN2 = gNi[2 * hw + p];
        }
        const bool pre = ts_job_prefetch_next(j, n_jobs, job.range.y - job.range.x, gridDim.x * TS_JOB_WARPS);
        const uint32_t j_next = pre ? ts_job_request(f, 1, lane) : 0u;   // next ticket: early (read at the end of this job) or late
        float tau[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        ts_bwd_walk<SM, ATTR, GEOM, POSE, NRM>(f, sc, job, lane, sm, sigma, alpha_min, fx, fy, ncon, Tcur, gC0, gC1, gC2, gD, gA,
                                               grad_color, grad_opacity, tau, gN0, gN1, gN2, 0xffffffffu, grad_sigma);
        if (POSE) {
            // per-thread -> per-job partial (fixed shuffle tree; the final reduction runs over jobs in index order)
#pragma unroll
            for (int jj = 0; jj < 6; ++jj) tau[jj] = warp_sum(tau[jj]);
            if (lane < 6) {
                float v = tau[0];
#pragma unroll
                for (int jj = 1; jj < 6; ++jj) v = (lane == jj) ? tau[jj] : v;
                // partials are indexed by (tile, block), not by ticket: the sum order does not depend on scheduling
                f.pose_partials[6 * ((size_t)job.tile * TS_BLOCKS_PER_TILE + job.blk) + lane] = v;
            }
        }
        j = pre ? ts_job_ticket(j_next) : ts_job_take(f, 1, lane);
    }
    ts_job_finish(f, 1, lane);
}

// ---------------------------------------------------------------------------------------------------------------
// Fused tracking job: a3 + a4 + a5 (pose-only) for one 8x4-pixel block without leaving the warp.  The forward
// walk leaves C, D, T, n_contrib and T_last of the lane's pixel in registers; the L1 cotangents (sign images) are
// formed from them and the target pixel; the backward walk starts at once, while the tile's records are still warm
// in L1.  Compared with ts_render_fwd_l1 + ts_render_bwd this saves a launch boundary and its tail, one job
// prologue / epilogue per block and the n_contrib / T_last / gC / gD round trip.  Arithmetic is the same code
// (ts_fwd_walk, ts_bwd_walk), so results are bit-identical to the two-launch sequence.
union TrackWarpSmem {
    FwdWarpSmem fwd;
    BwdWarpSmem bwd;
};

// POSE = true: the tracking job above.  POSE = false: the MAPPING job, the same forward walk and loss followed by the
// full-gradient backward walk (ATTR: colours / opacities, GEOM: screen-space vertex terms into gscr, which
// proj_bwd_kernel consumes afterwards).
template <int SM, bool ATTR = false, bool GEOM = false, bool POSE = true>
__global__ void __launch_bounds__(TS_JOB_WARPS * 32, 3)
render_track_kernel(TsFrameDev f, ts_scene sc, float sigma, float alpha_min, float t_min, float fx, float fy,
                    float* __restrict__ out_color, float* __restrict__ out_depth, float* __restrict__ out_alpha,
                    const float* __restrict__ Chat, const float* __restrict__ Dhat, float wc, float wd,
                    float* __restrict__ gCo, float* __restrict__ gDo, float* __restrict__ loss,
                    float* __restrict__ grad_color = nullptr, float* __restrict__ grad_opacity = nullptr,
                    float* __restrict__ grad_sigma = nullptr) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    TrackWarpSmem& sm = reinterpret_cast<TrackWarpSmem*>(smem_raw)[threadIdx.x >> 5];
    const uint32_t n_jobs = (uint32_t)f.NT * TS_BLOCKS_PER_TILE;
    const size_t hw = (size_t)f.W * f.H;
    unsigned long long dummy0 = 0, dummy1 = 0, dummy2 = 0;
    float loss_acc = 0.0f;

    uint32_t j = ts_job_take(f, 0, lane);
    while (j < n_jobs) {
#ifdef TS_JOB_TIMELINE
        // instrumented build only (paper_2605_31419_b200/timeline.py): when did this warp start and finish job j
        unsigned long long tl_t0;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tl_t0));
#endif
        TsJob job;
        ts_job_decode(f, j, lane, job);
        uint4 ent = make_uint4(0u, 0u, 0u, 0u);
        if (job.range.x + lane < job.range.y) ent = f.blist[job.range.x + lane];
        const bool pre = ts_job_prefetch_next(j, n_jobs, job.range.y - job.range.x, gridDim.x * TS_JOB_WARPS);
        const uint32_t j_next = pre ? ts_job_request(f, 0, lane) : 0u;   // next ticket: early (read at the end of this job) or late
        FwdPix o;
        // the chunk the forward walk staged last (with the whole record) is where the backward walk begins
        uint32_t staged_lo = 0xffffffffu;
        ts_fwd_walk<SM, false, false, false, true, BwdWarpSmem>(f, sc, job, lane, sm.bwd, sigma, alpha_min, t_min, ent, o, dummy0,
                                                                dummy1, dummy2, nullptr, nullptr, &staged_lo);
        float gC0 = 0.f, gC1 = 0.f, gC2 = 0.f, gD = 0.f;
        if (job.inside) {
            const size_t p = (size_t)job.py * f.W + job.px;
            if (out_color) out_color[p] = o.C0, out_color[hw + p] = o.C1, out_color[2 * hw + p] = o.C2;
            if (out_depth) out_depth[p] = o.D;
            if (out_alpha) out_alpha[p] = 1.0f - o.T;
            // a4: L = wc sum|C - Chat| + wd sum_{Dhat > 0} |D - Dhat|  (same arithmetic as l1_loss_grad_kernel)
            const float d0 = o.C0 - __ldg(Chat + p), d1 = o.C1 - __ldg(Chat + hw + p), d2 = o.C2 - __ldg(Chat + 2 * hw + p);
            gC0 = d0 > 0.f ? wc : (d0 < 0.f ? -wc : 0.f);
            gC1 = d1 > 0.f ? wc : (d1 < 0.f ? -wc : 0.f);
            gC2 = d2 > 0.f ? wc : (d2 < 0.f ? -wc : 0.f);
            loss_acc += wc * fabsf(d0) + wc * fabsf(d1) + wc * fabsf(d2);
            const float dh = __ldg(Dhat + p);
            if (dh > 0.f) {
                const float d = o.D - dh;
                gD = d > 0.f ? wd : (d < 0.f ? -wd : 0.f);
                loss_acc += wd * fabsf(d);
            }
            if (gCo) gCo[p] = gC0, gCo[hw + p] = gC1, gCo[2 * hw + p] = gC2;
            if (gDo) gDo[p] = gD;
        }
        __syncwarp();                                      // the forward walk's shared-memory slice is re-used
        float tau[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        ts_bwd_walk<SM, ATTR, GEOM, POSE>(f, sc, job, lane, sm.bwd, sigma, alpha_min, fx, fy, o.last, o.Tlast, gC0, gC1,
                                          gC2, gD, 0.0f, grad_color, grad_opacity, tau, 0.f, 0.f, 0.f, staged_lo, grad_sigma);
        if (POSE) {
#pragma unroll
            for (int jj = 0; jj < 6; ++jj) tau[jj] = warp_sum(tau[jj]);
            if (lane < 6) {
                float v = tau[0];
#pragma unroll
                for (int jj = 1; jj < 6; ++jj) v = (lane == jj) ? tau[jj] : v;
                f.pose_partials[6 * ((size_t)job.tile * TS_BLOCKS_PER_TILE + job.blk) + lane] = v;
            }
        }
        __syncwarp();
#ifdef TS_JOB_TIMELINE
        {
            unsigned long long tl_t1;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tl_t1));
            // (start ns, end ns, list length, persistent warp) per ticket; TS_VIEW_TIMELINE; the array is the scratch of
            // TS_VIEW_N_CONTRIB, which the fused kernels never touch
            if (lane == 0)
                reinterpret_cast<uint4*>(f.n_contrib_view)[j] = make_uint4((uint32_t)tl_t0, (uint32_t)tl_t1, job.range.y - job.range.x,
                                                                           blockIdx.x * TS_JOB_WARPS + (threadIdx.x >> 5));
        }
#endif
        j = pre ? ts_job_ticket(j_next) : ts_job_take(f, 0, lane);
    }
    ts_job_finish(f, 0, lane);
    if (loss) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) loss_acc += __shfl_xor_sync(0xffffffffu, loss_acc, d);
        if (lane == 0) atomicAdd(loss, loss_acc);
    }
}

template <int SM>
void launch_track(const ts_ctx* ctx, const ts_frame* fr, const ts_scene& sc, float* oc, float* od, float* oa, const float* Chat,
                  const float* Dhat, float wc, float wd, float* gC, float* gD, float* loss, cudaStream_t st) {
    const TsFrameDev& f = fr->d;
    const size_t smem = sizeof(TrackWarpSmem) * TS_JOB_WARPS;
    cudaFuncSetAttribute(render_track_kernel<SM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);   // per device
    const uint32_t grid = (uint32_t)min((int64_t)ctx->num_sms * 3, ((int64_t)f.NT * TS_BLOCKS_PER_TILE + TS_JOB_WARPS - 1) / TS_JOB_WARPS);
    render_track_kernel<SM><<<grid, TS_JOB_WARPS * 32, smem, st>>>(f, sc, fr->prm.sigma, fr->prm.alpha_min, fr->prm.t_min,
                                                                  fr->cam.fx, fr->cam.fy, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss);
}

template <int SM, bool ATTR, bool GEOM>
void launch_map(const ts_ctx* ctx, const ts_frame* fr, const ts_scene& sc, float* oc, float* od, float* oa, const float* Chat,
                const float* Dhat, float wc, float wd, float* gC, float* gD, float* loss, float* gcol, float* gopa,
                cudaStream_t st) {
    const TsFrameDev& f = fr->d;
    const size_t smem = sizeof(TrackWarpSmem) * TS_JOB_WARPS;
    cudaFuncSetAttribute(render_track_kernel<SM, ATTR, GEOM, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const uint32_t grid = (uint32_t)min((int64_t)ctx->num_sms * 3, ((int64_t)f.NT * TS_BLOCKS_PER_TILE + TS_JOB_WARPS - 1) / TS_JOB_WARPS);
    render_track_kernel<SM, ATTR, GEOM, false><<<grid, TS_JOB_WARPS * 32, smem, st>>>(
        f, sc, fr->prm.sigma, fr->prm.alpha_min, fr->prm.t_min, fr->cam.fx, fr->cam.fy, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss,
        gcol, gopa, fr->grad_sigma);
}

template <int SM>
void launch_map_sm(const ts_ctx* ctx, const ts_frame* fr, const ts_scene& sc, float* oc, float* od, float* oa, const float* Chat,
                   const float* Dhat, float wc, float wd, float* gC, float* gD, float* loss, float* gcol, float* gopa, bool attr,
                   bool geom, cudaStream_t st) {
    if (attr && geom) launch_map<SM, true, true>(ctx, fr, sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, gcol, gopa, st);
    else if (geom) launch_map<SM, false, true>(ctx, fr, sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, gcol, gopa, st);
    else launch_map<SM, true, false>(ctx, fr, sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, gcol, gopa, st);
}

}  // namespace

namespace {

constexpr int PB_THREADS = 256;

// a6 + the per-vertex terms of a7 (full-gradient mode).  Persistent grid-stride over visible slots; consumes and
// re-zeroes gscr.
// NRM: also consumes gnrm (dL/dn per face) and pushes it through n = s (a x b)/|a x b| (ts_normal.cuh) to the vertices
// (P1 += R^T g_a, P2 += R^T g_b, P0 -= both) and to the rotation part of the pose (a x g_a + b x g_b; a translation of
// the camera does not turn the normals).
// face_grad2d / face_views (may be NULL): the screen-space gradient statistic of the densification test (reading S28):
// ||sum_k (dL/du_k, dL/dv_k)|| added per face, and a count of the views in which the face received a gradient.
template <bool SOUP, bool NRM = false>
__global__ void __launch_bounds__(PB_THREADS)
proj_bwd_kernel(TsFrameDev f, const float* __restrict__ pos, const int32_t* __restrict__ faces,
                const float* __restrict__ Tcw, TsCamDev cam, float* __restrict__ grad_pos, int want_pose,
                float* __restrict__ face_grad2d = nullptr, uint32_t* __restrict__ face_views = nullptr) {
    __shared__ float sT[12];
    __shared__ float red[PB_THREADS / 32][6];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < 12) sT[tid] = __ldg(Tcw + tid);
    __syncthreads();
    const uint32_t nvis = min(ts_eff_visible(f), f.vis_cap);
    float tau[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    for (uint32_t slot = blockIdx.x * PB_THREADS + tid; slot < nvis; slot += gridDim.x * PB_THREADS) {
        float* gs = f.gscr + 9 * (size_t)slot;
        float g9[9];
        bool any = false;
#pragma unroll
        for (int j = 0; j < 9; ++j) {
            g9[j] = gs[j];
            any |= (g9[j] != 0.0f);
        }
        float gn[3] = {0.f, 0.f, 0.f};
        if (NRM) {
            float* gp = f.gnrm + 3 * (size_t)slot;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                gn[j] = gp[j];
                any |= (gn[j] != 0.0f);
            }
            if (any) gp[0] = gp[1] = gp[2] = 0.0f;
        }
        if (!any) continue;
#pragma unroll
        for (int j = 0; j < 9; ++j) gs[j] = 0.0f;
        const uint32_t m = __float_as_uint(f.scr[TS_SCR_F4 * (size_t)slot + 3].x);
        if (face_grad2d) {
            bool any_scr = false;
#pragma unroll
            for (int j = 0; j < 9; ++j) any_scr |= (g9[j] != 0.0f);
            if (any_scr) {
                const float sx = (g9[0] + g9[3]) + g9[6], sy = (g9[1] + g9[4]) + g9[7];
                face_grad2d[m] += sqrtf(sx * sx + sy * sy);          // one slot per face: no other writer
                if (face_views) face_views[m] += 1u;
            }
        }
        size_t vid[3];
        float P[3][3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            vid[k] = SOUP ? (size_t)3 * m + k : (size_t)__ldg(faces + 3 * (size_t)m + k);
            P[k][0] = __ldg(pos + 3 * vid[k]), P[k][1] = __ldg(pos + 3 * vid[k] + 1), P[k][2] = __ldg(pos + 3 * vid[k] + 2);
        }
        if (NRM) {
            TsFaceNormal fn;
            ts_face_normal_geom(sT, P, fn);
            float ga[3], gb[3];
            ts_face_normal_bwd(fn, gn, ga, gb);
            if (grad_pos) {
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    const float wa = sT[j] * ga[0] + sT[4 + j] * ga[1] + sT[8 + j] * ga[2];
                    const float wb = sT[j] * gb[0] + sT[4 + j] * gb[1] + sT[8 + j] * gb[2];
                    atomicAdd(grad_pos + 3 * vid[1] + j, wa);
                    atomicAdd(grad_pos + 3 * vid[2] + j, wb);
                    atomicAdd(grad_pos + 3 * vid[0] + j, -(wa + wb));
                }
            }
            tau[3] += (fn.a[1] * ga[2] - fn.a[2] * ga[1]) + (fn.b[1] * gb[2] - fn.b[2] * gb[1]);
            tau[4] += (fn.a[2] * ga[0] - fn.a[0] * ga[2]) + (fn.b[2] * gb[0] - fn.b[0] * gb[2]);
            tau[5] += (fn.a[0] * ga[1] - fn.a[1] * ga[0]) + (fn.b[0] * gb[1] - fn.b[1] * gb[0]);
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const size_t v = vid[k];
            const float px = P[k][0], py = P[k][1], pz = P[k][2];
            const float X = __fmaf_rn(sT[0], px, __fmaf_rn(sT[1], py, __fmaf_rn(sT[2], pz, sT[3])));
            const float Y = __fmaf_rn(sT[4], px, __fmaf_rn(sT[5], py, __fmaf_rn(sT[6], pz, sT[7])));
            const float Z = __fmaf_rn(sT[8], px, __fmaf_rn(sT[9], py, __fmaf_rn(sT[10], pz, sT[11])));
            const float iz = 1.0f / Z, iz2 = iz * iz;
            const float gu = g9[3 * k], gv = g9[3 * k + 1], gw = g9[3 * k + 2];
            // B7: d(u,v,w)/d(X,Y,Z)
            const float gX = cam.fx * iz * gu, gY = cam.fy * iz * gv;
            const float gZ = -(cam.fx * X * gu + cam.fy * Y * gv + gw) * iz2;
            if (grad_pos) {   // B8: R^T g_C
                atomicAdd(grad_pos + 3 * v + 0, sT[0] * gX + sT[4] * gY + sT[8] * gZ);
                atomicAdd(grad_pos + 3 * v + 1, sT[1] * gX + sT[5] * gY + sT[9] * gZ);
                atomicAdd(grad_pos + 3 * v + 2, sT[2] * gX + sT[6] * gY + sT[10] * gZ);
            }
            // B9: [g ; Q x g]  (Eq. 7)
            tau[0] += gX, tau[1] += gY, tau[2] += gZ;
            tau[3] += Y * gZ - Z * gY, tau[4] += Z * gX - X * gZ, tau[5] += X * gY - Y * gX;
        }
    }
    if (!want_pose) return;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) tau[j] += __shfl_xor_sync(0xffffffffu, tau[j], d);
        if (lane == 0) red[warp][j] = tau[j];
    }
    __syncthreads();
    if (tid < 6) {
        float s = 0.f;
#pragma unroll
        for (int w = 0; w < PB_THREADS / 32; ++w) s += red[w][tid];
        f.pose_partials[6 * (size_t)blockIdx.x + tid] = s;
    }
}

// a7: fixed-order tree reduction of the partials, in ONE round trip: a thread-block cluster of PR_BLOCKS CTAs, CTA g
// sums a fixed contiguous slice of the partials (fixed per-thread order, fixed shuffle / shared-memory tree) and puts
// its six sums into the shared memory of CTA 0 through distributed shared memory; after the cluster barrier the first
// six threads of CTA 0 add the block sums in index order and write dL/dtau -- the result does not depend on
// scheduling, and there is no global atomic, fence or second trip to L2.  Optionally one warp of CTA 0 then takes the
// Adam / Exp step on the pose (a8), which saves a launch in the tracking loop.
constexpr int PR_THREADS = 1024, PR_BLOCKS = 8;

__global__ void __cluster_dims__(PR_BLOCKS, 1, 1) __launch_bounds__(PR_THREADS)
pose_reduce_kernel(TsFrameDev f, uint32_t n, float* __restrict__ out, float* __restrict__ T_cw, float* __restrict__ state,
                   TsLr6 lr, float beta1, float beta2, float eps) {
    __shared__ float sm[PR_THREADS / 32][6];
    __shared__ float sb[PR_BLOCKS][6];                                   // CTA 0's copy receives the block sums
    __shared__ float tot[6];
    cg::cluster_group cluster = cg::this_cluster();
    // a CTA's shared memory may only be written from another CTA of the cluster once that CTA is known to have started:
    // every thread arrives here and waits just before the remote store, after the load phase, where the barrier has long
    // completed (it stays off the critical path)
    cluster.barrier_arrive();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t rank = cluster.block_rank();
    const uint32_t per = (n + PR_BLOCKS - 1) / PR_BLOCKS;
    const uint32_t i0 = min(n, rank * per), i1 = min(n, i0 + per);
    float a[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    const float2* p2 = reinterpret_cast<const float2*>(f.pose_partials);
    for (uint32_t ib = i0; ib < i1; ib += 4 * PR_THREADS) {              // 12 independent loads in flight per thread
        float2 v[4][3];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t i = ib + k * PR_THREADS + tid;
#pragma unroll
            for (int q = 0; q < 3; ++q) v[k][q] = i < i1 ? __ldcg(p2 + 3 * (size_t)i + q) : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k)
            a[0] += v[k][0].x, a[1] += v[k][0].y, a[2] += v[k][1].x, a[3] += v[k][1].y, a[4] += v[k][2].x, a[5] += v[k][2].y;
    }
#pragma unroll
    for (int j = 0; j < 6; ++j) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) a[j] += __shfl_xor_sync(0xffffffffu, a[j], d);
        if (lane == 0) sm[warp][j] = a[j];
    }
    __syncthreads();
    cluster.barrier_wait();                                               // all CTAs of the cluster are running
    if (tid < 6) {
        float s = 0.f;
#pragma unroll
        for (int w = 0; w < PR_THREADS / 32; ++w) s += sm[w][tid];
        float* dst = cluster.map_shared_rank(&sb[0][0], 0);               // CTA 0's sb
        dst[6 * rank + tid] = s;
    }
    cluster.sync();
    if (rank != 0) return;
    if (tid < 6) {
        float s = 0.f;
#pragma unroll
        for (int g = 0; g < PR_BLOCKS; ++g) s += sb[g][tid];
        out[tid] = s;
        tot[tid] = s;
    }
    __syncthreads();
    if (T_cw && tid < 32) ts_pose_step_warp(T_cw, tot, state, lr, beta1, beta2, eps);
}

template <int SM, bool ATTR, bool GEOM, bool POSE>
void launch_one(const ts_ctx* ctx, const ts_frame* fr, const ts_scene& sc, const float* gC, const float* gD, const float* gA,
                float* gcol, float* gopa, cudaStream_t st) {
    const TsFrameDev& f = fr->d;
    const size_t smem = sizeof(BwdWarpSmem) * TS_JOB_WARPS;
    // opt-in above 48 KB of dynamic shared memory; the attribute is per device, so it is set at every launch
    cudaFuncSetAttribute(render_bwd_kernel<SM, ATTR, GEOM, POSE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const uint32_t grid = (uint32_t)min((int64_t)ctx->num_sms * 3, ((int64_t)f.NT * TS_BLOCKS_PER_TILE + TS_JOB_WARPS - 1) / TS_JOB_WARPS);
    render_bwd_kernel<SM, ATTR, GEOM, POSE><<<grid, TS_JOB_WARPS * 32, smem, st>>>(f, sc, fr->prm.sigma, fr->prm.alpha_min,
                                                                                   fr->cam.fx, fr->cam.fy, gC, gD, gA, gcol, gopa,
                                                                                   nullptr, fr->grad_sigma);
}

template <int SM>
void launch_bwd_sm(const ts_ctx* ctx, const ts_frame* fr, const ts_scene& sc, const float* gC, const float* gD, const float* gA,
                   float* gcol, float* gopa, bool attr, bool geom, bool pose_only, cudaStream_t st) {
    if (pose_only) launch_one<SM, false, false, true>(ctx, fr, sc, gC, gD, gA, gcol, gopa, st);
    else if (attr && geom) launch_one<SM, true, true, false>(ctx, fr, sc, gC, gD, gA, gcol, gopa, st);
    else if (geom) launch_one<SM, false, true, false>(ctx, fr, sc, gC, gD, gA, gcol, gopa, st);
    else launch_one<SM, true, false, false>(ctx, fr, sc, gC, gD, gA, gcol, gopa, st);
}

}  // namespace

int32_t ts_launch_render_bwd(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, const float* gC, const float* gD,
                             const float* gA, float* grad_pos, float* grad_color, float* grad_opacity, uint32_t mask,
                             cudaStream_t st, float* face_grad2d, uint32_t* face_views) {
    const bool attr = (mask & (TS_GRAD_COLOR | TS_GRAD_OPACITY)) != 0;
    const bool geom = (mask & (TS_GRAD_POS | TS_GRAD_POSE)) != 0;
    const bool pose_only = (mask == TS_GRAD_POSE) && !face_grad2d;   // the statistic needs the per-face sums
    if (!attr && !geom) return TS_OK;
    float* gcol = (mask & TS_GRAD_COLOR) ? grad_color : nullptr;
    float* gopa = (mask & TS_GRAD_OPACITY) ? grad_opacity : nullptr;
    switch (ts_frame_sigma_mode(fr)) {
        case 1: launch_bwd_sm<1>(ctx, fr, *sc, gC, gD, gA, gcol, gopa, attr, geom, pose_only, st); break;
        case 2: launch_bwd_sm<2>(ctx, fr, *sc, gC, gD, gA, gcol, gopa, attr, geom, pose_only, st); break;
        case 3: launch_bwd_sm<3>(ctx, fr, *sc, gC, gD, gA, gcol, gopa, attr, geom, pose_only, st); break;
        default: launch_bwd_sm<0>(ctx, fr, *sc, gC, gD, gA, gcol, gopa, attr, geom, pose_only, st); break;
    }
    fr->pose_src = 0;
    if (pose_only) {
        fr->pose_src = 1, fr->n_pose_partials = (uint32_t)fr->d.NT * TS_BLOCKS_PER_TILE;
    } else if (geom) {
        const int grid = (int)min((uint32_t)(ctx->num_sms * 4), fr->d.n_partials_cap);
        const int want_pose = (mask & TS_GRAD_POSE) ? 1 : 0;
        float* gp = (mask & TS_GRAD_POS) ? grad_pos : nullptr;
        if (sc->faces == nullptr)
            proj_bwd_kernel<true><<<grid, PB_THREADS, 0, st>>>(fr->d, sc->pos, nullptr, fr->T_cw, fr->cam, gp, want_pose,
                                                               face_grad2d, face_views);
        else
            proj_bwd_kernel<false><<<grid, PB_THREADS, 0, st>>>(fr->d, sc->pos, sc->faces, fr->T_cw, fr->cam, gp, want_pose,
                                                                face_grad2d, face_views);
        if (want_pose) fr->pose_src = 2, fr->n_pose_partials = (uint32_t)grid;
    }
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

namespace {

template <int SM>
void launch_bwd_normal_sm(const ts_ctx* ctx, const ts_frame* fr, const ts_scene& sc, const float* gC, const float* gD,
                          const float* gA, const float* gN, float* gcol, float* gopa, bool attr, bool geom, cudaStream_t st) {
    const TsFrameDev& f = fr->d;
    const size_t smem = sizeof(BwdWarpSmem) * TS_JOB_WARPS;
    const uint32_t grid = (uint32_t)min((int64_t)ctx->num_sms * 2, ((int64_t)f.NT * TS_BLOCKS_PER_TILE + TS_JOB_WARPS - 1) / TS_JOB_WARPS);
    const float sg = fr->prm.sigma, am = fr->prm.alpha_min, fx = fr->cam.fx, fy = fr->cam.fy;
#define TS_LAUNCH_BN(A, G)                                                                                                  \
    do {                                                                                                                    \
        cudaFuncSetAttribute(render_bwd_kernel<SM, A, G, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
        render_bwd_kernel<SM, A, G, false, true><<<grid, TS_JOB_WARPS * 32, smem, st>>>(f, sc, sg, am, fx, fy, gC, gD, gA, gcol, gopa, gN, \
                                                                                        fr->grad_sigma);                       \
    } while (0)
    if (attr && geom) TS_LAUNCH_BN(true, true);
    else if (geom) TS_LAUNCH_BN(false, true);
    else TS_LAUNCH_BN(true, false);
#undef TS_LAUNCH_BN
}

}  // namespace

// Normal-map variant of ts_launch_render_bwd: the cotangents of all four raster outputs in one backward pass.
int32_t ts_launch_render_bwd_normal(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, const float* gC, const float* gD,
                                    const float* gA, const float* gN, float* grad_pos, float* grad_color,
                                    float* grad_opacity, uint32_t mask, cudaStream_t st) {
    const bool attr = (mask & (TS_GRAD_COLOR | TS_GRAD_OPACITY)) != 0;
    const bool geom = (mask & (TS_GRAD_POS | TS_GRAD_POSE)) != 0;
    if (!attr && !geom) return TS_OK;
    float* gcol = (mask & TS_GRAD_COLOR) ? grad_color : nullptr;
    float* gopa = (mask & TS_GRAD_OPACITY) ? grad_opacity : nullptr;
    switch (ts_frame_sigma_mode(fr)) {
        case 1: launch_bwd_normal_sm<1>(ctx, fr, *sc, gC, gD, gA, gN, gcol, gopa, attr, geom, st); break;
        case 2: launch_bwd_normal_sm<2>(ctx, fr, *sc, gC, gD, gA, gN, gcol, gopa, attr, geom, st); break;
        case 3: launch_bwd_normal_sm<3>(ctx, fr, *sc, gC, gD, gA, gN, gcol, gopa, attr, geom, st); break;
        default: launch_bwd_normal_sm<0>(ctx, fr, *sc, gC, gD, gA, gN, gcol, gopa, attr, geom, st); break;
    }
    fr->pose_src = 0;
    if (geom) {
        const int grid = (int)min((uint32_t)(ctx->num_sms * 4), fr->d.n_partials_cap);
        const int want_pose = (mask & TS_GRAD_POSE) ? 1 : 0;
        float* gp = (mask & TS_GRAD_POS) ? grad_pos : nullptr;
        if (sc->faces == nullptr)
            proj_bwd_kernel<true, true><<<grid, PB_THREADS, 0, st>>>(fr->d, sc->pos, nullptr, fr->T_cw, fr->cam, gp, want_pose);
        else
            proj_bwd_kernel<false, true><<<grid, PB_THREADS, 0, st>>>(fr->d, sc->pos, sc->faces, fr->T_cw, fr->cam, gp, want_pose);
        if (want_pose) fr->pose_src = 2, fr->n_pose_partials = (uint32_t)grid;
    }
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

int32_t ts_launch_render_track(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, float* oc, float* od, float* oa,
                               const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss,
                               cudaStream_t st) {
    const double n = (double)fr->d.W * (double)fr->d.H;
    const float wc = (float)(1.0 / (3.0 * n)), wd = (float)((double)lambda_dep / n);
    switch (ts_frame_sigma_mode(fr)) {
        case 1: launch_track<1>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, st); break;
        case 2: launch_track<2>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, st); break;
        case 3: launch_track<3>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, st); break;
        default: launch_track<0>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, st); break;
    }
    fr->pose_src = 1, fr->n_pose_partials = (uint32_t)fr->d.NT * TS_BLOCKS_PER_TILE;
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

// a3 + a4 + a5 (full-gradient) + a6 in two launches: the mapping counterpart of ts_launch_render_track.
int32_t ts_launch_render_map(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, float* oc, float* od, float* oa,
                             const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss,
                             float* grad_pos, float* grad_color, float* grad_opacity, uint32_t mask, cudaStream_t st) {
    const bool attr = (mask & (TS_GRAD_COLOR | TS_GRAD_OPACITY)) != 0;
    const bool geom = (mask & (TS_GRAD_POS | TS_GRAD_POSE)) != 0;
    const double n = (double)fr->d.W * (double)fr->d.H;
    const float wc = (float)(1.0 / (3.0 * n)), wd = (float)((double)lambda_dep / n);
    float* gcol = (mask & TS_GRAD_COLOR) ? grad_color : nullptr;
    float* gopa = (mask & TS_GRAD_OPACITY) ? grad_opacity : nullptr;
    switch (ts_frame_sigma_mode(fr)) {
        case 1: launch_map_sm<1>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, gcol, gopa, attr, geom, st); break;
        case 2: launch_map_sm<2>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, gcol, gopa, attr, geom, st); break;
        case 3: launch_map_sm<3>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, gcol, gopa, attr, geom, st); break;
        default: launch_map_sm<0>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, gcol, gopa, attr, geom, st); break;
    }
    fr->pose_src = 0;
    if (geom) {
        const int grid = (int)min((uint32_t)(ctx->num_sms * 4), fr->d.n_partials_cap);
        const int want_pose = (mask & TS_GRAD_POSE) ? 1 : 0;
        float* gp = (mask & TS_GRAD_POS) ? grad_pos : nullptr;
        if (sc->faces == nullptr)
            proj_bwd_kernel<true><<<grid, PB_THREADS, 0, st>>>(fr->d, sc->pos, nullptr, fr->T_cw, fr->cam, gp, want_pose);
        else
            proj_bwd_kernel<false><<<grid, PB_THREADS, 0, st>>>(fr->d, sc->pos, sc->faces, fr->T_cw, fr->cam, gp, want_pose);
        if (want_pose) fr->pose_src = 2, fr->n_pose_partials = (uint32_t)grid;
    }
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

int32_t ts_launch_pose_reduce(const ts_ctx*, ts_frame* fr, float* out, float* T_cw, float* state, const float* lr6,
                              float beta1, float beta2, float eps, cudaStream_t st) {
    if (fr->pose_src == 0) return TS_ERR_STATE;
    TsLr6 lr;
    for (int i = 0; i < 6; ++i) lr.v[i] = lr6 ? lr6[i] : 0.0f;
    pose_reduce_kernel<<<PR_BLOCKS, PR_THREADS, 0, st>>>(fr->d, fr->n_pose_partials, out, T_cw, state, lr, beta1, beta2, eps);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
