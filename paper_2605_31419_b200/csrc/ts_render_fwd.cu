// ts_render_fwd.cu -- a3: front-to-back compositing (Eq. 2-4).
// Persistent warps, one 8x4-pixel block of a 16x16 tile per job (ts_jobs.cuh), one pixel per lane.  The block's
// list (built by the sort kernel) is read 32 entries at a time (one coalesced LDG.128 per lane: slot, face, rect);
// lanes whose entry's triangle meets the block copy the pre-built face record (ts_raster.cuh; four LDG.128 + nine
// colour floats) into the warp's private shared-memory slice, in list order; the warp then walks the staged entries,
// reading each record with broadcast LDS.128 and testing "my pixel is in the rect" with one shift of the entry's
// lane mask.  Pixels stop at T <= t_min, the warp when all its pixels stopped.  No CTA barrier, no atomics.
#include "ts_fwd_job.cuh"
#include "ts_normal.cuh"

namespace {

// optional fused a4: L1 colour + depth loss against a target frame, evaluated on the pixel values while they are
// still in registers (Eq. 8-10 without D-SSIM; same arithmetic as l1_loss_grad_kernel in ts_helpers.cu)
struct FwdLoss {
    const float* Chat;
    const float* Dhat;
    float* gC;
    float* gD;
    float* loss;
    float wc, wd;
};

template <int SM, bool COUNT, bool LOSS, bool STATS, bool NRM = false>
__global__ void __launch_bounds__(TS_JOB_WARPS * 32)
render_fwd_kernel(TsFrameDev f, ts_scene sc, float sigma, float alpha_min, float t_min, float* __restrict__ out_color,
                  float* __restrict__ out_depth, float* __restrict__ out_alpha, FwdLoss L, uint32_t* __restrict__ face_pixels,
                  float* __restrict__ out_normal = nullptr, float* __restrict__ out_normal_top = nullptr) {
    __shared__ FwdWarpSmem smem[TS_JOB_WARPS];
    __shared__ float4 smem_n[NRM ? TS_JOB_WARPS * 32 : 1];
    const int lane = threadIdx.x & 31;
    FwdWarpSmem& sm = smem[threadIdx.x >> 5];
    const uint32_t n_jobs = (uint32_t)f.NT * TS_BLOCKS_PER_TILE;
    const size_t hw = (size_t)f.W * f.H;
    unsigned long long n_rect = 0, n_hit = 0, n_visit = 0;
    float loss_acc = 0.0f;

    uint32_t j = ts_job_take(f, 0, lane);
    while (j < n_jobs) {
        TsJob job;
        ts_job_decode(f, j, lane, job);
        uint4 ent = make_uint4(0u, 0u, 0u, 0u);
        if (job.range.x + lane < job.range.y) ent = f.blist[job.range.x + lane];
        const bool pre = ts_job_prefetch_next(j, n_jobs, job.range.y - job.range.x, gridDim.x * TS_JOB_WARPS);
        const uint32_t j_next = pre ? ts_job_request(f, 0, lane) : 0u;   // next ticket: early (read at the end of this job) or late
        FwdPix o;
        ts_fwd_walk<SM, COUNT, STATS, NRM>(f, sc, job, lane, sm, sigma, alpha_min, t_min, ent, o, n_visit, n_rect, n_hit, face_pixels,
                                           smem_n + (NRM ? (threadIdx.x & ~31) : 0));
        const float T = o.T, C0 = o.C0, C1 = o.C1, C2 = o.C2, D = o.D, Tlast = o.Tlast;
        const uint32_t last = o.last;
        if (job.inside) {
            const size_t p = (size_t)job.py * f.W + job.px;
            if (out_color) out_color[p] = C0, out_color[hw + p] = C1, out_color[2 * hw + p] = C2;
            if (out_depth) out_depth[p] = D;
            if (out_alpha) out_alpha[p] = 1.0f - T;
            if (NRM && out_normal) out_normal[p] = o.N0, out_normal[hw + p] = o.N1, out_normal[2 * hw + p] = o.N2;
            if (NRM && out_normal_top) out_normal_top[p] = o.Nt0, out_normal_top[hw + p] = o.Nt1, out_normal_top[2 * hw + p] = o.Nt2;
            f.n_contrib[p] = last;
            f.t_last[p] = Tlast;
            if (LOSS) {
                const float c[3] = {C0, C1, C2};
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    const float d = c[ch] - __ldg(L.Chat + ch * hw + p);
                    L.gC[ch * hw + p] = d > 0.f ? L.wc : (d < 0.f ? -L.wc : 0.f);
                    loss_acc += L.wc * fabsf(d);
                }
                const float dh = __ldg(L.Dhat + p);
                float g = 0.f;
                if (dh > 0.f) {
                    const float d = D - dh;
                    g = d > 0.f ? L.wd : (d < 0.f ? -L.wd : 0.f);
                    loss_acc += L.wd * fabsf(d);
                }
                L.gD[p] = g;
            }
        }
        j = pre ? ts_job_ticket(j_next) : ts_job_take(f, 0, lane);
    }
    ts_job_finish(f, 0, lane);
    if (LOSS && L.loss) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) loss_acc += __shfl_xor_sync(0xffffffffu, loss_acc, d);
        if (lane == 0) atomicAdd(L.loss, loss_acc);       // one atomic per persistent warp
    }
    if (COUNT) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            n_rect += __shfl_xor_sync(0xffffffffu, n_rect, d);
            n_hit += __shfl_xor_sync(0xffffffffu, n_hit, d);
        }
        if (lane == 0) {
            atomicAdd(&f.ctrl->counters[0], n_visit);     // warp-level visits (lane 0's count)
            atomicAdd(&f.ctrl->counters[1], n_rect);
            atomicAdd(&f.ctrl->counters[2], n_hit);
        }
    }
}

template <int SM>
void launch_sm(const ts_ctx* ctx, const ts_frame* fr, const ts_scene& sc, float* oc, float* od, float* oa, const FwdLoss* L,
               uint32_t* face_pixels, cudaStream_t st) {
    const TsFrameDev& f = fr->d;
    const bool count = (fr->prm.flags & TS_PARAM_COUNTERS) != 0;
    const uint32_t grid = (uint32_t)min((int64_t)ctx->num_sms * 4, ((int64_t)f.NT * TS_BLOCKS_PER_TILE + TS_JOB_WARPS - 1) / TS_JOB_WARPS);
    const float sg = fr->prm.sigma, am = fr->prm.alpha_min, tm = fr->prm.t_min;
    const FwdLoss none = {nullptr, nullptr, nullptr, nullptr, nullptr, 0.f, 0.f};
    if (face_pixels) render_fwd_kernel<SM, false, false, true><<<grid, TS_JOB_WARPS * 32, 0, st>>>(f, sc, sg, am, tm, oc, od, oa, none, face_pixels);
    else if (L) render_fwd_kernel<SM, false, true, false><<<grid, TS_JOB_WARPS * 32, 0, st>>>(f, sc, sg, am, tm, oc, od, oa, *L, nullptr);
    else if (count) render_fwd_kernel<SM, true, false, false><<<grid, TS_JOB_WARPS * 32, 0, st>>>(f, sc, sg, am, tm, oc, od, oa, none, nullptr);
    else render_fwd_kernel<SM, false, false, false><<<grid, TS_JOB_WARPS * 32, 0, st>>>(f, sc, sg, am, tm, oc, od, oa, none, nullptr);
}

// projected area of every visible face, |S| / 2 with S of F4 (same operation order as the projection: bit-exact)
__global__ void __launch_bounds__(256) face_area_kernel(TsFrameDev f, float* __restrict__ area) {
    const uint32_t nvis = min(ts_eff_visible(f), f.vis_cap);
    for (uint32_t slot = blockIdx.x * blockDim.x + threadIdx.x; slot < nvis; slot += gridDim.x * blockDim.x) {
        const float4* s4 = f.scr + TS_SCR_F4 * (size_t)slot;
        const float4 s0 = s4[0], s1 = s4[1], s3 = s4[3];
        const float a = __fsub_rn(s0.w, s0.x), b = __fsub_rn(s1.w, s0.y), c = __fsub_rn(s1.x, s0.y), d = __fsub_rn(s1.z, s0.x);
        const float S = __fmaf_rn(a, b, -__fmul_rn(c, d));
        area[__float_as_uint(s3.x)] = 0.5f * fabsf(S);
    }
}

// Eq. 12 / reading S26: unit normal of every visible face in camera space, towards the camera.  The edge vectors are
// taken in world space (exact differences of nearby floats) and rotated; the orientation is the sign of the plane
// offset m . Q_0.
template <bool SOUP>
__global__ void __launch_bounds__(256)
face_normal_kernel(TsFrameDev f, const float* __restrict__ pos, const int32_t* __restrict__ faces, const float* __restrict__ Tcw) {
    __shared__ float sT[12];
    if (threadIdx.x < 12) sT[threadIdx.x] = __ldg(Tcw + threadIdx.x);
    __syncthreads();
    const uint32_t nvis = min(ts_eff_visible(f), f.vis_cap);
    for (uint32_t slot = blockIdx.x * blockDim.x + threadIdx.x; slot < nvis; slot += gridDim.x * blockDim.x) {
        const uint32_t m = __float_as_uint(f.scr[TS_SCR_F4 * (size_t)slot + 3].x);
        float P[3][3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const size_t v = SOUP ? (size_t)3 * m + k : (size_t)__ldg(faces + 3 * (size_t)m + k);
            P[k][0] = __ldg(pos + 3 * v), P[k][1] = __ldg(pos + 3 * v + 1), P[k][2] = __ldg(pos + 3 * v + 2);
        }
        float4 n;
        ts_face_normal(sT, P, n);
        f.nrm[slot] = n;
    }
}

}  // namespace

int32_t ts_launch_render_fwd_normal(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, float* oc, float* od, float* oa,
                                    float* on, cudaStream_t st, float* on_top) {
    const TsFrameDev& f = fr->d;
    if (sc->faces == nullptr) face_normal_kernel<true><<<ctx->num_sms * 4, 256, 0, st>>>(f, sc->pos, nullptr, fr->T_cw);
    else face_normal_kernel<false><<<ctx->num_sms * 4, 256, 0, st>>>(f, sc->pos, sc->faces, fr->T_cw);
    const uint32_t grid = (uint32_t)min((int64_t)ctx->num_sms * 4, ((int64_t)f.NT * TS_BLOCKS_PER_TILE + TS_JOB_WARPS - 1) / TS_JOB_WARPS);
    const float sg = fr->prm.sigma, am = fr->prm.alpha_min, tm = fr->prm.t_min;
    const FwdLoss none = {nullptr, nullptr, nullptr, nullptr, nullptr, 0.f, 0.f};
    switch (ts_frame_sigma_mode(fr)) {
        case 1: render_fwd_kernel<1, false, false, false, true><<<grid, TS_JOB_WARPS * 32, 0, st>>>(f, *sc, sg, am, tm, oc, od, oa, none, nullptr, on, on_top); break;
        case 2: render_fwd_kernel<2, false, false, false, true><<<grid, TS_JOB_WARPS * 32, 0, st>>>(f, *sc, sg, am, tm, oc, od, oa, none, nullptr, on, on_top); break;
        case 3: render_fwd_kernel<3, false, false, false, true><<<grid, TS_JOB_WARPS * 32, 0, st>>>(f, *sc, sg, am, tm, oc, od, oa, none, nullptr, on, on_top); break;
        default: render_fwd_kernel<0, false, false, false, true><<<grid, TS_JOB_WARPS * 32, 0, st>>>(f, *sc, sg, am, tm, oc, od, oa, none, nullptr, on, on_top); break;
    }
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

int32_t ts_launch_face_area(const ts_ctx* ctx, ts_frame* fr, float* area, cudaStream_t st) {
    face_area_kernel<<<ctx->num_sms * 4, 256, 0, st>>>(fr->d, area);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

int32_t ts_launch_render_fwd(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, float* oc, float* od, float* oa,
                             const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss,
                             uint32_t* face_pixels, cudaStream_t st) {
    FwdLoss L;
    const FwdLoss* Lp = nullptr;
    if (gC) {
        const double n = (double)fr->d.W * (double)fr->d.H;
        L = FwdLoss{Chat, Dhat, gC, gD, loss, (float)(1.0 / (3.0 * n)), (float)((double)lambda_dep / n)};
        Lp = &L;
    }
    switch (ts_frame_sigma_mode(fr)) {
        case 1: launch_sm<1>(ctx, fr, *sc, oc, od, oa, Lp, face_pixels, st); break;
        case 2: launch_sm<2>(ctx, fr, *sc, oc, od, oa, Lp, face_pixels, st); break;
        case 3: launch_sm<3>(ctx, fr, *sc, oc, od, oa, Lp, face_pixels, st); break;
        default: launch_sm<0>(ctx, fr, *sc, oc, od, oa, Lp, face_pixels, st); break;
    }
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
