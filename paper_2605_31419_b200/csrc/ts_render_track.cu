// ts_render_track.cu -- the tracking fast path ts_render_track_l1: a3 + a4 + a5 (pose-only) of one 8x4-pixel block
// without leaving the warp (100 of these per frame), with a HIT LOG.
//
// The forward walk is ts_fwd_walk's (same staging, same visits, same arithmetic: images bit-identical to
// ts_render_fwd).  Every hit is also appended to a compact per-warp log in shared memory: (alpha, sum_k omega_k c_k,
// z, lhat_k, face slot, face, pixel lane, link to the pixel's previous hit).  After the L1 cotangents of the block
// are known (a4), the backward pass never evaluates a window again and never stages a record again:
//   chain     every lane walks ITS pixel's hits back to front through the links: T_n = T_{n+1}/(1 - alpha_n),
//             S_n = c_n.gC + z_n gD,  dL/dalpha_n = T_n (S_n - R),  R <- alpha_n S_n + (1 - alpha_n) R  (DESIGN.md
//             B2-B3); (dL/dalpha, T alpha) overwrite the log entry;
//   geometry  the log is dealt 32 entries at a time to the lanes, every lane finishes one hit: B4-B6 and straight
//             through d(u,v,w)/dtau (Eq. 5-7) into six per-thread accumulators; the face record (ten rows, most of
//             them only needed here) and the vertex colours are read from global memory / L1 by the lanes that
//             hold a hit of that face, not staged for every entry of the list.
// The accumulators are tree-reduced once per job into pose_partials[tile * 8 + block] (fixed order: deterministic).
// A block whose hits do not fit the log (deep pixels, long lists) falls back to the reverse walk of ts_bwd_job.cuh,
// which re-evaluates the windows (the visit form of round 1).
#include "ts_bwd_job.cuh"
#include "ts_fwd_job.cuh"

namespace {

constexpr uint32_t TL_FULL = 0xffffffffu;
constexpr uint32_t TL_NIL = 0xffu;

template <int CAP>
struct LogWarpSmem {
    FwdWarpSmem fwd;                  // staging of the forward walk (rows R0-R2, kappa, colours; masks, slots, faces)
    float4 fa[CAP];                   // (alpha, sum_k omega_k c_k [3])  ->  (dL/dalpha, T alpha, -, -) after the chain
    float2 fz[CAP];                   // (z, bits of: previous hit of the same pixel (TL_NIL = none) | pixel lane << 8 |
                                      //  position of the entry in the tile list << 13)
    float4 pix[32];                   // (gC0, gC1, gC2, gD) of the block's pixels
};
constexpr uint32_t TL_POS_MAX = 1u << 19;      // list positions the log can name; a longer list takes the fallback
template <int CAP>
union TrackLogSmem {
    LogWarpSmem<CAP> log;
    BwdWarpSmem bwd;                  // fallback: the reverse walk that re-evaluates
};

// Forward walk of one job with the hit log.  Same visits and arithmetic as ts_fwd_walk (ts_fwd_job.cuh).
// used = hits of the job (the log holds them all iff used <= CAP), mylast = the lane's last logged hit.
template <int SM, int CAP>
__device__ __forceinline__ void tl_fwd_walk(const TsFrameDev& f, const ts_scene& sc, const TsJob& job, int lane, LogWarpSmem<CAP>& sm,
                                            float sigma, float alpha_min, float t_min, uint4 ent, FwdPix& o, uint32_t& used,
                                            uint32_t& mylast) {
    FwdWarpSmem& st = sm.fwd;
    const float fpx = (float)job.px, fpy = (float)job.py;
    float T = 1.0f, C0 = 0.0f, C1 = 0.0f, C2 = 0.0f, D = 0.0f, Tlast = 1.0f;
    uint32_t last = 0;
    const uint32_t lt = (1u << lane) - 1u;
    bool done = !job.inside;
    bool warp_done = __all_sync(TL_FULL, done);
    used = 0, mylast = TL_NIL;
    for (uint32_t c0 = job.range.x; c0 < job.range.y && !warp_done; c0 += 32) {
        const uint32_t n = min(32u, job.range.y - c0);
        const uint4 cur = ent;
        if (c0 + 32 + lane < job.range.y) ent = f.blist[c0 + 32 + lane];     // prefetch the next chunk
        uint32_t lmask = (uint32_t)lane < n ? ts_entry_mask(job, cur) : 0u;
        if (!__any_sync(TL_FULL, lmask != 0u)) continue;
        __syncwarp();                                   // previous chunk's reads are done
        if (lmask) {
            const float4* rp = f.rec + TS_REC_F4 * (size_t)cur.x;
            const float4 r0 = __ldg(rp), r1 = __ldg(rp + 1), r2 = __ldg(rp + 2), r3 = __ldg(rp + 3);
            float col[9];
            ts_load_colors(sc, cur.y, col);
            if (ts_job_block_misses(job, cur, r0, r1, r2)) lmask = 0u;
            st.r[lane][0] = r0, st.r[lane][1] = r1, st.r[lane][2] = r2;
            st.r[lane][3] = make_float4(r3.x, r3.y, r3.z, col[0]);
            st.r[lane][4] = make_float4(col[1], col[2], col[3], col[4]);
            st.r[lane][5] = make_float4(col[5], col[6], col[7], col[8]);
            st.lm[lane] = lmask, st.slot[lane] = cur.x, st.face[lane] = cur.y;
        }
        __syncwarp();
        uint32_t ov = __ballot_sync(TL_FULL, lmask != 0u);
        const uint32_t pos0 = (c0 - job.range.x) + 1u;
        while (ov) {
            const int e = __ffs(ov) - 1;
            ov &= ov - 1;
            const bool in_rect = !done && ((st.lm[e] >> lane) & 1u);
            float l[3], x, I, alpha;
            bool hit = false;
            if (in_rect) {
                const float4 r0 = st.r[e][0], r1 = st.r[e][1], r2 = st.r[e][2];
                hit = ts_eval_alpha<SM>(r0, r1, r2, fpx, fpy, sigma, alpha_min, f.scr, st.slot[e], l, x, I, alpha);
            }
            const uint32_t hm = __ballot_sync(TL_FULL, hit);
            if (hit) {
                const float4 r3 = st.r[e][3], r4 = st.r[e][4], r5 = st.r[e][5];
                const float o0 = l[0] * r3.x, o1 = l[1] * r3.y, o2 = l[2] * r3.z;   // omega_k = lhat_k kappa_k
                const float Om = (o0 + o1) + o2;
                const float z = ts_rcp_approx(Om);
                const float wgt = T * alpha, wz = wgt * z;
                const float c0v = fmaf(o0, r3.w, fmaf(o1, r4.z, o2 * r5.y));
                const float c1v = fmaf(o0, r4.x, fmaf(o1, r4.w, o2 * r5.z));
                const float c2v = fmaf(o0, r4.y, fmaf(o1, r5.x, o2 * r5.w));
                C0 = fmaf(wz, c0v, C0), C1 = fmaf(wz, c1v, C1), C2 = fmaf(wz, c2v, C2);
                D += wz;
                Tlast = T;
                T = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                last = pos0 + (uint32_t)e;
                if (T <= t_min) done = true;
                const uint32_t fi = used + (uint32_t)__popc(hm & lt);
                if (fi < (uint32_t)CAP) {
                    sm.fa[fi] = make_float4(alpha, c0v, c1v, c2v);
                    sm.fz[fi] = make_float2(z, __uint_as_float(mylast | ((uint32_t)lane << 8) | ((pos0 + (uint32_t)e - 1u) << 13)));
                    mylast = fi;
                }
            }
            used += (uint32_t)__popc(hm);
        }
        warp_done = __all_sync(TL_FULL, done);
    }
    o.T = T, o.C0 = C0, o.C1 = C1, o.C2 = C2, o.D = D, o.Tlast = Tlast, o.last = last;
}

// B4 (window) + B5 (interpolation) + B6 (screen-space vertex terms) of ONE hit, as ts_bwd_geom, on explicit rows.
template <int SM>
__device__ __forceinline__ void tl_geom(const float4 r0, const float4 r1, const float4 r2, const float4 q4, const float4 q5,
                                        const float4 q6, const float4 q7, const float l[3], float x, float I, float ga, float wgt,
                                        float z, float d0, float d1, float d2, float cg, float zgd, float sigma, float g[9]) {
    const float gI = r2.w * ga;
    float gx;
    if (SM == 1) gx = gI;
    else if (SM == 2) gx = 0.5f * gI * ts_rcp_approx(I);
    else if (SM == 3) gx = 2.0f * gI * x;
    else gx = gI * sigma * I * ts_rcp_approx(x);
    const float wz = wgt * z, base = cg + zgd;
    const float go0 = wz * (d0 - base), go1 = wz * (d1 - base), go2 = wz * (d2 - base);
    const float b0 = -l[0] * q4.x, b1 = -l[1] * q4.y, b2 = -l[2] * q4.z;      // b_k = -lhat_k rho_k
    g[2] = b0 * go0, g[5] = b1 * go1, g[8] = b2 * go2;                        // dL/dw_k
    const float t0 = q5.x * go0 * q4.x, t1 = q5.y * go1 * q4.y, t2 = q5.z * go2 * q4.z;
    const float Gx = -(t0 * r0.z + t1 * r1.x + t2 * r1.z), Gy = -(t0 * r0.w + t1 * r1.y + t2 * r1.w);
    float q0x = -b0 * Gx, q0y = -b0 * Gy, q1x = -b1 * Gx, q1y = -b1 * Gy, q2x = -b2 * Gx, q2y = -b2 * Gy;
    if (l[0] >= l[1] && l[0] >= l[2]) {
        const float t = b2 + b0 * q5.w, mgx = r0.z * gx, mgy = r0.w * gx;
        q1x += (1.0f - t) * mgx, q1y += (1.0f - t) * mgy, q2x += t * mgx, q2y += t * mgy;
    } else if (l[1] >= l[2]) {
        const float t = b0 + b1 * q6.x, mgx = r1.x * gx, mgy = r1.y * gx;
        q2x += (1.0f - t) * mgx, q2y += (1.0f - t) * mgy, q0x += t * mgx, q0y += t * mgy;
    } else {
        const float t = b1 + b2 * q6.y, mgx = r1.z * gx, mgy = r1.w * gx;
        q0x += (1.0f - t) * mgx, q0y += (1.0f - t) * mgy, q1x += t * mgx, q1y += t * mgy;
    }
    const float xg = x * gx;
    g[0] = q0x + xg * q6.z, g[1] = q0y + xg * q6.w, g[3] = q1x + xg * q7.x, g[4] = q1y + xg * q7.y;
    g[6] = q2x + xg * q7.z, g[7] = q2y + xg * q7.w;
}

// chain phase (B2-B3): this lane's pixel walks its logged hits back to front
template <int CAP>
__device__ __forceinline__ void tl_chain(LogWarpSmem<CAP>& sm, uint32_t fi, float Tlast, float gC0, float gC1, float gC2, float gD) {
    float Tcur = Tlast, Rs = 0.0f;
    bool first = true;
    while (fi != TL_NIL) {
        const float4 a = sm.fa[fi];
        const float2 zc = sm.fz[fi];
        const float z = zc.x;
        const uint32_t nx = __float_as_uint(zc.y) & 0xffu;
        const float one_m = __fsub_rn(1.0f, a.x);
        const float Tn = first ? Tcur : Tcur * ts_rcp_approx(one_m);
        Tcur = Tn, first = false;
        const float S = (a.y * gC0 + a.z * gC1 + a.w * gC2 + gD) * z;     // c . gC + z gD
        const float ga = Tn * (S - Rs);                                   // B2
        Rs = a.x * S + one_m * Rs;                                        // B3
        *reinterpret_cast<float2*>(&sm.fa[fi]) = make_float2(ga, Tn * a.x);
        fi = nx;
    }
}

// geometry phase: one logged hit per lane, through B4-B7 + B9 (Eq. 5-7) into the lane's six accumulators.  The entry
// (slot, face) is read again from the block's list, the record and the colours from global memory / L1, and
// lhat_k is formed again exactly as the forward walk formed it (ts_eval_alpha: same operations, same refinement rule).
template <int SM, int CAP>
__device__ __forceinline__ void tl_geometry(const LogWarpSmem<CAP>& sm, const TsFrameDev& f, const ts_scene& sc, const TsJob& job,
                                            int lane, uint32_t used, float fx, float fy, float sigma, float alpha_min, float tau[6]) {
    for (uint32_t g0 = 0; g0 < used; g0 += 32u) {
        const uint32_t fi = g0 + (uint32_t)lane;
        if (fi >= used) continue;
        const float2 zc = sm.fz[fi];
        const uint32_t code = __float_as_uint(zc.y), pl = (code >> 8) & 31u;
        const uint4 ent = __ldg(f.blist + job.range.x + (code >> 13));           // (slot, face, rect_lo, rect_hi)
        const float4* rp = f.rec + TS_REC_F4 * (size_t)ent.x;
        const float4 r0 = __ldg(rp), r1 = __ldg(rp + 1), r2 = __ldg(rp + 2), r3 = __ldg(rp + 3);
        const float4 q4 = __ldg(rp + 4), q5 = __ldg(rp + 5), q6 = __ldg(rp + 6), q7 = __ldg(rp + 7), n0 = __ldg(rp + 8), n1 = __ldg(rp + 9);
        float col[9];
        ts_load_colors(sc, ent.y, col);
        const float4 a = sm.fa[fi];
        const float ga = a.x, wgt = a.y;
        const float4 pg = sm.pix[pl];
        // the hit's pixel: lane pl of the block
        const float fpx = (float)(job.tx0 + ((job.blk & 1) << 3) + (int)(pl & 7u)), fpy = (float)(job.ty0 + ((job.blk >> 1) << 2) + (int)(pl >> 3));
        float l[3], x, I, alpha;
        ts_eval_alpha<SM>(r0, r1, r2, fpx, fpy, sigma, alpha_min, f.scr, ent.x, l, x, I, alpha);
        const float z = zc.x;
        const float o0 = l[0] * r3.x, o1 = l[1] * r3.y, o2 = l[2] * r3.z;
        const float d0 = col[0] * pg.x + col[1] * pg.y + col[2] * pg.z;
        const float d1 = col[3] * pg.x + col[4] * pg.y + col[5] * pg.z;
        const float d2 = col[6] * pg.x + col[7] * pg.y + col[8] * pg.z;
        const float cg = (o0 * d0 + o1 * d1 + o2 * d2) * z;
        float g[9];
        tl_geom<SM>(r0, r1, r2, q4, q5, q6, q7, l, x, I, ga, wgt, z, d0, d1, d2, cg, z * pg.w, sigma, g);
        // B7 + B9: with Q = (xn, yn, 1)/w,  Z g_C = (a, b, c),  a = fx gu, b = fy gv, c = -(xn a + yn b) - w gw
        {
            const float aa = fx * g[0], bb = fy * g[1], cc = -(n0.x * aa + n0.y * bb) - q5.x * g[2];
            tau[0] += q5.x * aa, tau[1] += q5.x * bb, tau[2] += q5.x * cc;
            tau[3] += n0.y * cc - bb, tau[4] += aa - n0.x * cc, tau[5] += n0.x * bb - n0.y * aa;
        }
        {
            const float aa = fx * g[3], bb = fy * g[4], cc = -(n0.z * aa + n0.w * bb) - q5.y * g[5];
            tau[0] += q5.y * aa, tau[1] += q5.y * bb, tau[2] += q5.y * cc;
            tau[3] += n0.w * cc - bb, tau[4] += aa - n0.z * cc, tau[5] += n0.z * bb - n0.w * aa;
        }
        {
            const float aa = fx * g[6], bb = fy * g[7], cc = -(n1.x * aa + n1.y * bb) - q5.z * g[8];
            tau[0] += q5.z * aa, tau[1] += q5.z * bb, tau[2] += q5.z * cc;
            tau[3] += n1.y * cc - bb, tau[4] += aa - n1.x * cc, tau[5] += n1.x * bb - n1.y * aa;
        }
    }
}

template <int SM, int CAP>
__global__ void __launch_bounds__(TS_JOB_WARPS * 32, 3)
render_track_log_kernel(TsFrameDev f, ts_scene sc, float sigma, float alpha_min, float t_min, float fx, float fy,
                        float* __restrict__ out_color, float* __restrict__ out_depth, float* __restrict__ out_alpha,
                        const float* __restrict__ Chat, const float* __restrict__ Dhat, float wc, float wd,
                        float* __restrict__ gCo, float* __restrict__ gDo, float* __restrict__ loss) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    TrackLogSmem<CAP>& sm = reinterpret_cast<TrackLogSmem<CAP>*>(smem_raw)[threadIdx.x >> 5];
    const uint32_t n_jobs = (uint32_t)f.NT * TS_BLOCKS_PER_TILE;
    const size_t hw = (size_t)f.W * f.H;
    float loss_acc = 0.0f;

    uint32_t j = ts_job_take(f, 0, lane);
    while (j < n_jobs) {
        TsJob job;
        ts_job_decode(f, j, lane, job);
        uint4 ent = make_uint4(0u, 0u, 0u, 0u);
        if (job.range.x + lane < job.range.y) ent = f.blist[job.range.x + lane];
        const uint32_t j_next = ts_job_request(f, 0, lane);   // next ticket: read at the end of this job
        FwdPix o;
        uint32_t used, mylast;
        tl_fwd_walk<SM, CAP>(f, sc, job, lane, sm.log, sigma, alpha_min, t_min, ent, o, used, mylast);
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
        float tau[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (used <= (uint32_t)CAP && job.range.y - job.range.x <= TL_POS_MAX) {
            // the log holds every hit of the block: chain, then geometry
            sm.log.pix[lane] = make_float4(gC0, gC1, gC2, gD);
            tl_chain<CAP>(sm.log, mylast, o.Tlast, gC0, gC1, gC2, gD);
            __syncwarp();
            tl_geometry<SM, CAP>(sm.log, f, sc, job, lane, used, fx, fy, sigma, alpha_min, tau);
        } else {
            __syncwarp();                                  // the shared-memory slice is re-used by the reverse walk
            ts_bwd_walk<SM, false, false, true>(f, sc, job, lane, sm.bwd, sigma, alpha_min, fx, fy, o.last, o.Tlast, gC0, gC1, gC2,
                                                gD, 0.0f, nullptr, nullptr, tau);
        }
#pragma unroll
        for (int jj = 0; jj < 6; ++jj) tau[jj] = warp_sum(tau[jj]);
        if (lane < 6) {
            float v = tau[0];
#pragma unroll
            for (int jj = 1; jj < 6; ++jj) v = (lane == jj) ? tau[jj] : v;
            f.pose_partials[6 * ((size_t)job.tile * TS_BLOCKS_PER_TILE + job.blk) + lane] = v;
        }
        __syncwarp();
        j = ts_job_ticket(j_next);
    }
    ts_job_finish(f, 0, lane);
    if (loss) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) loss_acc += __shfl_xor_sync(TL_FULL, loss_acc, d);
        if (lane == 0) atomicAdd(loss, loss_acc);
    }
}

constexpr int TL_CAP = 192;

template <int SM>
void launch_track_log(const ts_ctx* ctx, const ts_frame* fr, const ts_scene& sc, float* oc, float* od, float* oa, const float* Chat,
                      const float* Dhat, float wc, float wd, float* gC, float* gD, float* loss, cudaStream_t st) {
    const TsFrameDev& f = fr->d;
    const size_t smem = sizeof(TrackLogSmem<TL_CAP>) * TS_JOB_WARPS;
    // opt-in above 48 KB of dynamic shared memory; the attribute is per device, so it is set at every launch
    cudaFuncSetAttribute(render_track_log_kernel<SM, TL_CAP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const uint32_t grid = (uint32_t)min((int64_t)ctx->num_sms * 3, ((int64_t)f.NT * TS_BLOCKS_PER_TILE + TS_JOB_WARPS - 1) / TS_JOB_WARPS);
    render_track_log_kernel<SM, TL_CAP><<<grid, TS_JOB_WARPS * 32, smem, st>>>(f, sc, fr->prm.sigma, fr->prm.alpha_min, fr->prm.t_min,
                                                                               fr->cam.fx, fr->cam.fy, oc, od, oa, Chat, Dhat, wc, wd, gC,
                                                                               gD, loss);
}

}  // namespace

int32_t ts_launch_render_track(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, float* oc, float* od, float* oa,
                               const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss,
                               cudaStream_t st) {
    if (!ctx->track_log) return ts_launch_render_track_v1(ctx, fr, sc, oc, od, oa, Chat, Dhat, lambda_dep, gC, gD, loss, st);
    const double n = (double)fr->d.W * (double)fr->d.H;
    const float wc = (float)(1.0 / (3.0 * n)), wd = (float)((double)lambda_dep / n);
    switch (ts_frame_sigma_mode(fr)) {
        case 1: launch_track_log<1>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, st); break;
        case 2: launch_track_log<2>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, st); break;
        case 3: launch_track_log<3>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, st); break;
        default: launch_track_log<0>(ctx, fr, *sc, oc, od, oa, Chat, Dhat, wc, wd, gC, gD, loss, st); break;
    }
    fr->pose_src = 1, fr->n_pose_partials = (uint32_t)fr->d.NT * TS_BLOCKS_PER_TILE;
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
