// ts_bwd_job.cuh -- the backward walk of ONE job (one 8x4-pixel block, one warp): DESIGN.md B1-B9.
// Shared by render_bwd_kernel and the fused tracking kernel (ts_render_bwd.cu).
#pragma once
#include "ts_jobs.cuh"

struct BwdWarpSmem {
    float4 r[32][13];                 // R0 R1 R2 | kap,c00 | colours | colours | R4 R5 R6 R7 | R8 R9 | pad: a 208 B
                                      // stride spreads the lanes' rows over all banks (192 B put them on two bank quads)
    uint32_t lm[32];
    uint32_t slot[32];
    uint32_t face[32];
    // ring of hits waiting for the packed second phase, and the block's cotangents
    float4 q_a[64];                   // (dL/dalpha, T alpha, lhat_0, lhat_1)
    float2 q_b[64];                   // (lhat_2, bits of: entry index | pixel lane << 8)
    float4 pix[32];                   // (gC0, gC1, gC2, gD) of the lane's pixel
};

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// B4 (window) + B5 (interpolation) + B6 (screen-space vertex terms) of ONE hit.  R = the staged record
// (rows as in BwdWarpSmem::r), l = lhat_k, x = -max l, I = x^sigma, ga = dL/dalpha, wgt = T alpha,
// z, d_k = c_k.gC, cg = c.gC, zgd = z gD.  Outputs g[9] = dL/d(u0,v0,w0,u1,v1,w1,u2,v2,w2).
template <int SM>
__device__ __forceinline__ void ts_bwd_geom(const BwdWarpSmem& sm, uint32_t e, const float l[3], float x, float I, float ga, float wgt,
                                            float z, float d0, float d1, float d2, float cg, float zgd, float sigma,
                                            float g[9]) {
    const float4 r0 = sm.r[e][0], r1 = sm.r[e][1], r2 = sm.r[e][2];
    const float4 q4 = sm.r[e][6], q5 = sm.r[e][7], q6 = sm.r[e][8], q7 = sm.r[e][9];   // record rows R4..R7
    // B4 window: gx = dL/dx
    const float gI = r2.w * ga;
    float gx;
    if (SM == 1) gx = gI;
    else if (SM == 2) gx = 0.5f * gI * ts_rcp_approx(I);
    else if (SM == 3) gx = 2.0f * gI * x;
    else gx = gI * sigma * I * ts_rcp_approx(x);
    // B5 interpolation
    const float wz = wgt * z, base = cg + zgd;
    const float go0 = wz * (d0 - base), go1 = wz * (d1 - base), go2 = wz * (d2 - base);
    const float b0 = -l[0] * q4.x, b1 = -l[1] * q4.y, b2 = -l[2] * q4.z;      // b_k = -lhat_k rho_k
    g[2] = b0 * go0, g[5] = b1 * go1, g[8] = b2 * go2;                        // dL/dw_k
    // B6 (i): G = sum_k (w_k go_k) grad_p b_k,  grad_p b_k = -rho_k m_k
    const float t0 = q5.x * go0 * q4.x, t1 = q5.y * go1 * q4.y, t2 = q5.z * go2 * q4.z;
    const float Gx = -(t0 * r0.z + t1 * r1.x + t2 * r1.z), Gy = -(t0 * r0.w + t1 * r1.y + t2 * r1.w);
    float q0x = -b0 * Gx, q0y = -b0 * Gy, q1x = -b1 * Gx, q1y = -b1 * Gy, q2x = -b2 * Gx, q2y = -b2 * Gy;
    // B6 (ii): x = -lhat_{k*}; edge k* runs from a = q_{k*+1} to b = q_{k*+2};  t = b_{k*+2} + b_{k*} tau_{k*}
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
    // B6 (iii): through the inradius
    const float xg = x * gx;
    g[0] = q0x + xg * q6.z, g[1] = q0y + xg * q6.w, g[3] = q1x + xg * q7.x, g[4] = q1y + xg * q7.y;
    g[6] = q2x + xg * q7.z, g[7] = q2y + xg * q7.w;
}

// Pose-only second phase, one QUEUED hit per lane (lanes hold hits of different pixels and faces): recompute the
// interpolation terms from the queued lhat_k, run B4-B6 and push the nine screen terms through B7 + B9
// (Eq. 5-7): with Q = (xn, yn, 1)/w,  Z g_C = (a, b, c),  a = fx gu, b = fy gv, c = -(xn a + yn b) - w gw;
// rho += w (a,b,c);  theta += Q x g_C.
template <int SM>
__device__ __forceinline__ void ts_bwd_pose_hit(const BwdWarpSmem& sm, uint32_t e, const float4 pg, float l0, float l1, float l2, float ga,
                                                float wgt, float fx, float fy, float sigma, float tau[6]) {
    const float4 r3 = sm.r[e][3], r4 = sm.r[e][4], r5 = sm.r[e][5];
    const float l[3] = {l0, l1, l2};
    const float x = -fmaxf(l0, fmaxf(l1, l2));
    const float sg = SM == 0 ? sm.r[e][12].x : sigma;             // per-entry exponent in the generic instantiation (S32)
    const float I = ts_window_pow<SM>(x, sg);
    const float o0 = l0 * r3.x, o1 = l1 * r3.y, o2 = l2 * r3.z;
    const float Om = (o0 + o1) + o2, z = ts_rcp_approx(Om);
    const float d0 = r3.w * pg.x + r4.x * pg.y + r4.y * pg.z;
    const float d1 = r4.z * pg.x + r4.w * pg.y + r5.x * pg.z;
    const float d2 = r5.y * pg.x + r5.z * pg.y + r5.w * pg.z;
    const float cg = (o0 * d0 + o1 * d1 + o2 * d2) * z;
    float g[9];
    ts_bwd_geom<SM>(sm, e, l, x, I, ga, wgt, z, d0, d1, d2, cg, z * pg.w, sg, g);
    const float4 q5 = sm.r[e][7], n0 = sm.r[e][10], n1 = sm.r[e][11];
    {
        const float a = fx * g[0], b = fy * g[1], c = -(n0.x * a + n0.y * b) - q5.x * g[2];
        tau[0] += q5.x * a, tau[1] += q5.x * b, tau[2] += q5.x * c;
        tau[3] += n0.y * c - b, tau[4] += a - n0.x * c, tau[5] += n0.x * b - n0.y * a;
    }
    {
        const float a = fx * g[3], b = fy * g[4], c = -(n0.z * a + n0.w * b) - q5.y * g[5];
        tau[0] += q5.y * a, tau[1] += q5.y * b, tau[2] += q5.y * c;
        tau[3] += n0.w * c - b, tau[4] += a - n0.z * c, tau[5] += n0.z * b - n0.w * a;
    }
    {
        const float a = fx * g[6], b = fy * g[7], c = -(n1.x * a + n1.y * b) - q5.z * g[8];
        tau[0] += q5.z * a, tau[1] += q5.z * b, tau[2] += q5.z * c;
        tau[3] += n1.y * c - b, tau[4] += a - n1.x * c, tau[5] += n1.x * b - n1.y * a;
    }
}

// Full-gradient second phase, one QUEUED hit per lane: the 9 screen terms (GEOM) and / or the 9 colour terms + the
// opacity term (ATTR) of the lane's hit; hits of the same face sit in consecutive lanes (they were queued by one
// visit), so a segmented shuffle reduction adds them up per face BEFORE any global atomic, and the first lane of every
// run issues the RED.ADD.F32s.  `active` = this lane holds a hit.
// NRM (normal-map backward, Eq. 12): the staged record carries the face normal in row 10 and row 11 of staged index
// `pixel lane` carries that pixel's dL/dN (neither row is used outside pose-only mode); with GEOM the per-face dL/dn =
// sum wgt dL/dN goes to f.gnrm.
template <int SM, bool ATTR, bool GEOM, bool NRM = false>
__device__ __forceinline__ void ts_bwd_full_group(const TsFrameDev& f, const ts_scene& sc, BwdWarpSmem& sm, int lane,
                                                  bool active, uint32_t code, float l0, float l1, float l2, float ga,
                                                  float wgt, float sigma, float* __restrict__ grad_color,
                                                  float* __restrict__ grad_opacity, float* __restrict__ grad_sigma = nullptr) {
    const uint32_t e = code & 0xffu;
    float acc[19];
    float accn[3] = {0.f, 0.f, 0.f};
    float accs = 0.f;                                              // dL/dsigma of the hit's face (generic instantiation, S32)
    const bool want_sigma = SM == 0 && grad_sigma != nullptr;
#pragma unroll
    for (int j = 0; j < 19; ++j) acc[j] = 0.f;
    if (active) {
        const float4 pg = sm.pix[code >> 8];
        if (NRM && GEOM) {
            const float4 pn = sm.r[code >> 8][11];
            accn[0] = wgt * pn.x, accn[1] = wgt * pn.y, accn[2] = wgt * pn.z;
        }
        const float4 r3 = sm.r[e][3], r4 = sm.r[e][4], r5 = sm.r[e][5];
        const float l[3] = {l0, l1, l2};
        const float x = -fmaxf(l0, fmaxf(l1, l2));
        const float sg = SM == 0 ? sm.r[e][12].x : sigma;
        const float I = ts_window_pow<SM>(x, sg);
        if (want_sigma) accs = ga * sm.r[e][2].w * I * __logf(x);     // I = x^sigma: dL/dsigma += dL/dI I ln x
        const float o0 = l0 * r3.x, o1 = l1 * r3.y, o2 = l2 * r3.z;
        const float Om = (o0 + o1) + o2, z = ts_rcp_approx(Om);
        if (ATTR) {
            // B1 colours, B4 opacity (one value per face; /3 applied when written)
            const float w0 = o0 * z * wgt, w1 = o1 * z * wgt, w2 = o2 * z * wgt;
            acc[9] = w0 * pg.x, acc[10] = w0 * pg.y, acc[11] = w0 * pg.z;
            acc[12] = w1 * pg.x, acc[13] = w1 * pg.y, acc[14] = w1 * pg.z;
            acc[15] = w2 * pg.x, acc[16] = w2 * pg.y, acc[17] = w2 * pg.z;
            acc[18] = I * ga;
        }
        if (GEOM) {
            const float d0 = r3.w * pg.x + r4.x * pg.y + r4.y * pg.z;
            const float d1 = r4.z * pg.x + r4.w * pg.y + r5.x * pg.z;
            const float d2 = r5.y * pg.x + r5.z * pg.y + r5.w * pg.z;
            const float cg = (o0 * d0 + o1 * d1 + o2 * d2) * z;
            ts_bwd_geom<SM>(sm, e, l, x, I, ga, wgt, z, d0, d1, d2, cg, z * pg.w, sg, acc);
        }
    }
    // segmented reduction over runs of equal staged index (inactive lanes never match anybody)
    const uint32_t key = active ? e : 0x100u + (uint32_t)lane;
    // only as many doubling steps as the longest run needs (runs average ~8 hits; a chunk-end group is short)
    const uint32_t kp = __shfl_up_sync(0xffffffffu, key, 1);
    const bool run_start = lane == 0 || kp != key;
    const uint32_t starts = __ballot_sync(0xffffffffu, run_start);
    const int my_start = 31 - __clz((int)(starts & (0xffffffffu >> (31 - lane))));
    const uint32_t max_off = __reduce_max_sync(0xffffffffu, active ? (uint32_t)(lane - my_start) : 0u);
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        if ((uint32_t)d > max_off) break;
        const uint32_t kd = __shfl_down_sync(0xffffffffu, key, d);
        const bool same = (lane + d < 32) && kd == key;
        if (GEOM) {
#pragma unroll
            for (int j = 0; j < 9; ++j) {
                const float t = __shfl_down_sync(0xffffffffu, acc[j], d);
                if (same) acc[j] += t;
            }
        }
        if (ATTR) {
#pragma unroll
            for (int j = 9; j < 19; ++j) {
                const float t = __shfl_down_sync(0xffffffffu, acc[j], d);
                if (same) acc[j] += t;
            }
        }
        if (NRM && GEOM) {
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const float t = __shfl_down_sync(0xffffffffu, accn[j], d);
                if (same) accn[j] += t;
            }
        }
        if (want_sigma) {
            const float t = __shfl_down_sync(0xffffffffu, accs, d);
            if (same) accs += t;
        }
    }
    if (active && run_start) {                                 // first lane of a run
        if (want_sigma) atomicAdd(grad_sigma + sm.face[e], accs);
        if (GEOM) {
            float* gs = f.gscr + 9 * (size_t)sm.slot[e];
#pragma unroll
            for (int j = 0; j < 9; ++j) atomicAdd(gs + j, acc[j]);
            if (NRM) {
                float* gn = f.gnrm + 3 * (size_t)sm.slot[e];
#pragma unroll
                for (int j = 0; j < 3; ++j) atomicAdd(gn + j, accn[j]);
            }
        }
        if (ATTR) {
            const uint32_t m = sm.face[e];
            uint32_t v[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) v[k] = sc.faces ? (uint32_t)__ldg(sc.faces + 3 * (size_t)m + k) : 3u * m + k;
            if (grad_color) {
#pragma unroll
                for (int k = 0; k < 3; ++k)
#pragma unroll
                    for (int ch = 0; ch < 3; ++ch) atomicAdd(grad_color + 3 * (size_t)v[k] + ch, acc[9 + 3 * k + ch]);
            }
            if (grad_opacity) {
                if (f.prm_flags & TS_PARAM_MIN_OPACITY) {
                    // min mode: the gradient goes to the vertex with the lowest opacity (lowest index among equals)
                    const float p0 = __ldg(sc.opacity + v[0]), p1 = __ldg(sc.opacity + v[1]), p2 = __ldg(sc.opacity + v[2]);
                    int km = 0;
                    float pm = p0;
                    if (p1 < pm) km = 1, pm = p1;
                    if (p2 < pm) km = 2;
                    atomicAdd(grad_opacity + (km == 0 ? v[0] : (km == 1 ? v[1] : v[2])), acc[18]);
                } else {
                    const float go = acc[18] * (1.0f / 3.0f);
#pragma unroll
                    for (int k = 0; k < 3; ++k) atomicAdd(grad_opacity + v[k], go);
                }
            }
        }
    }
}

// ncon / Tcur = the forward walk's n_contrib and T in front of the last contributing face for this lane's pixel;
// gC*, gD, gA = the pixel's cotangents.  The per-pixel walk does the sequential part of every hit and queues it;
// 32 queued hits at a time are finished with all lanes busy: POSE: tau[6] += the lane's se(3) terms
// (ts_bwd_pose_hit); otherwise segmented per-face reduction + atomics into f.gscr / grad_color / grad_opacity
// (ts_bwd_full_group).
template <int SM, bool ATTR, bool GEOM, bool POSE, bool NRM = false>
__device__ __forceinline__ void ts_bwd_walk(const TsFrameDev& f, const ts_scene& sc, const TsJob& job, int lane,
                                            BwdWarpSmem& sm, float sigma, float alpha_min, float fx, float fy,
                                            uint32_t ncon, float Tcur, float gC0, float gC1, float gC2, float gD,
                                            float gA, float* __restrict__ grad_color, float* __restrict__ grad_opacity,
                                            float tau[6], float gN0 = 0.f, float gN1 = 0.f, float gN2 = 0.f,
                                            uint32_t prestaged_lo = 0xffffffffu, float* __restrict__ grad_sigma = nullptr) {
    static_assert(!(NRM && POSE), "the normal-map backward runs in full-gradient mode");
    const float fpx = (float)job.px, fpy = (float)job.py;
    const uint32_t lt = (1u << lane) - 1u;
    const uint32_t n_walk = min(__reduce_max_sync(0xffffffffu, ncon), job.range.y - job.range.x);
    sm.pix[lane] = make_float4(gC0, gC1, gC2, gD);
    if (NRM) sm.r[lane][11] = make_float4(gN0, gN1, gN2, 0.f);       // row 11 is free outside pose-only mode
    float Rs = 0.f;                    // R^c.gC + R^d gD + R^a gA behind the current face
    bool first = true;
    uint32_t qn = 0, qh = 0;           // queued hits and the ring's head (warp-uniform)

    for (uint32_t hi = n_walk; hi > 0;) {
        const uint32_t lo = (hi - 1u) & ~31u;           // chunks are aligned like the forward walk's
        const uint32_t n = hi - lo;
        uint4 cur = make_uint4(0u, 0u, 0u, 0u);
        uint32_t lmask;
        const bool prestaged = lo == prestaged_lo;
        if (prestaged) {
            // the forward walk of this job left exactly this chunk staged, rows 0-11, masks after the block cull
            lmask = (uint32_t)lane < n ? sm.lm[lane] : 0u;
        } else {
            if ((uint32_t)lane < n) cur = f.blist[job.range.x + lo + lane];
            lmask = (uint32_t)lane < n ? ts_entry_mask(job, cur) : 0u;
        }
        hi = lo;
        __syncwarp();
        if (lmask && !prestaged) {
            // staged at the lane's own index (no compaction); the walk follows the set bits of `ov` backwards
            const float4* rp = f.rec + TS_REC_F4 * (size_t)cur.x;
            float4 r[TS_REC_F4];
#pragma unroll
            for (int i = 0; i < (POSE ? 10 : 8); ++i) r[i] = __ldg(rp + i);
            float col[9];
            ts_load_colors(sc, cur.y, col);
            if (ts_job_block_misses(job, cur, r[0], r[1], r[2])) lmask = 0u;
            float4* d = sm.r[lane];
            d[0] = r[0], d[1] = r[1], d[2] = r[2];
            d[3] = make_float4(r[3].x, r[3].y, r[3].z, col[0]);
            d[4] = make_float4(col[1], col[2], col[3], col[4]);
            d[5] = make_float4(col[5], col[6], col[7], col[8]);
            d[6] = r[4], d[7] = r[5], d[8] = r[6], d[9] = r[7];
            if (POSE) d[10] = r[8], d[11] = r[9];
            if (NRM) d[10] = f.nrm[cur.x];
            if (SM == 0) d[12] = make_float4(r[3].w, 0.f, 0.f, 0.f);  // the entry's window exponent (S32)
            sm.lm[lane] = lmask, sm.slot[lane] = cur.x, sm.face[lane] = cur.y;
        }
        __syncwarp();
        uint32_t ov = __ballot_sync(0xffffffffu, lmask != 0u);
        while (ov) {
            const int e = 31 - __clz(ov);
            ov &= ~(1u << e);
            const bool in_rect = lo + (uint32_t)e < ncon && ((sm.lm[e] >> lane) & 1u);
            if (!__any_sync(0xffffffffu, in_rect)) continue;
            float l[3], x, I, alpha;
            bool hit = false;
            {
                const float4 r0 = sm.r[e][0], r1 = sm.r[e][1], r2 = sm.r[e][2];
                const float sg = SM == 0 ? sm.r[e][12].x : sigma;
                hit = in_rect && ts_eval_alpha<SM>(r0, r1, r2, fpx, fpy, sg, alpha_min, f.scr, sm.slot[e], l, x, I, alpha);
            }
            const uint32_t hm = __ballot_sync(0xffffffffu, hit);
            if (!hm) continue;
            if (hit) {
                const float4 r3 = sm.r[e][3], r4 = sm.r[e][4], r5 = sm.r[e][5];
                // transmittance in front of this face
                const float one_m = __fsub_rn(1.0f, alpha);
                const float Tn = first ? Tcur : Tcur * ts_rcp_approx(one_m);
                Tcur = Tn, first = false;
                const float o0 = l[0] * r3.x, o1 = l[1] * r3.y, o2 = l[2] * r3.z;
                const float Om = (o0 + o1) + o2, z = ts_rcp_approx(Om);
                // d_k = c_k . gC
                const float d0 = r3.w * gC0 + r4.x * gC1 + r4.y * gC2;
                const float d1 = r4.z * gC0 + r4.w * gC1 + r5.x * gC2;
                const float d2 = r5.y * gC0 + r5.z * gC1 + r5.w * gC2;
                const float cg = (o0 * d0 + o1 * d1 + o2 * d2) * z;       // c . gC
                const float zgd = z * gD;
                float S = cg + zgd + gA;
                if (NRM) {
                    const float4 nf = sm.r[e][10];
                    S += nf.x * gN0 + nf.y * gN1 + nf.z * gN2;            // flat attribute: n . dL/dN
                }
                const float wgt = Tn * alpha;
                const float ga = Tn * (S - Rs);                           // B2
                Rs = alpha * S + one_m * Rs;                              // B3
                {
                    // the sequential part of this hit is done; the rest (B4-B9) waits in the queue
                    const uint32_t qi = (qh + qn + (uint32_t)__popc(hm & lt)) & 63u;
                    sm.q_a[qi] = make_float4(ga, wgt, l[0], l[1]);
                    sm.q_b[qi] = make_float2(l[2], __uint_as_float((uint32_t)e | ((uint32_t)lane << 8)));
                }
                (void)x, (void)I;
            }
            qn += (uint32_t)__popc(hm);
            if (qn >= 32u) {
                // a full group: every lane finishes one queued hit
                __syncwarp();
                const float4 qa = sm.q_a[(qh + lane) & 63u];
                const float2 qb = sm.q_b[(qh + lane) & 63u];
                const uint32_t code = __float_as_uint(qb.y);
                const float qga = qa.x, qw = qa.y, ql0 = qa.z, ql1 = qa.w, ql2 = qb.x;
                qh = (qh + 32u) & 63u, qn -= 32u;       // the remainder (< 32 entries) stays where it is
                if (POSE)
                    ts_bwd_pose_hit<SM>(sm, code & 0xffu, sm.pix[code >> 8], ql0, ql1, ql2, qga, qw, fx, fy, sigma, tau);
                else
                    ts_bwd_full_group<SM, ATTR, GEOM, NRM>(f, sc, sm, lane, true, code, ql0, ql1, ql2, qga, qw, sigma, grad_color, grad_opacity, grad_sigma);
                __syncwarp();
            }
        }
        if (qn) {
            // the staged records are about to be replaced: finish what is still queued (partial group)
            __syncwarp();
            const bool act = (uint32_t)lane < qn;
            float4 qa = make_float4(0.f, 0.f, 0.f, 0.f);
            float2 qb = make_float2(0.f, 0.f);
            if (act) qa = sm.q_a[(qh + lane) & 63u], qb = sm.q_b[(qh + lane) & 63u];
            const uint32_t code = __float_as_uint(qb.y);
            const float qga = qa.x, qw = qa.y, ql0 = qa.z, ql1 = qa.w, ql2 = qb.x;
            if (POSE) {
                if (act) ts_bwd_pose_hit<SM>(sm, code & 0xffu, sm.pix[code >> 8], ql0, ql1, ql2, qga, qw, fx, fy, sigma, tau);
            } else {
                ts_bwd_full_group<SM, ATTR, GEOM, NRM>(f, sc, sm, lane, act, code, ql0, ql1, ql2, qga, qw, sigma, grad_color, grad_opacity, grad_sigma);
            }
            qn = 0, qh = 0;
            __syncwarp();
        }
    }
}
