// ts_fwd_job.cuh -- the forward walk of ONE job (one 8x4-pixel block, one warp): Eq. 2-4.
// Shared by render_fwd_kernel (ts_render_fwd.cu) and the fused tracking kernel (ts_render_bwd.cu).
#pragma once
#include "ts_jobs.cuh"

struct FwdWarpSmem {
    float4 r[32][7];                  // R0 R1 R2 | kap0 kap1 kap2 c00 | c01 c02 c10 c11 | c12 c20 c21 c22 | pad (bank spread)
    uint32_t lm[32];                  // lane mask of the entry for this block
    uint32_t slot[32];
    uint32_t face[32];                // only written / read by the statistics instantiation
};

struct FwdPix {                       // what the walk leaves for this lane's pixel
    float T, C0, C1, C2, D, Tlast;
    uint32_t last;
    float N0, N1, N2;                 // composited face normals (NRM instantiation only)
    float Nt0, Nt1, Nt2;              // normal of the first hit with the largest alpha (NRM instantiation only; reading S29)
};

// `ent` = the lane's entry of the first 32-entry chunk of the tile list (already requested by the caller, so that
// its round trip overlaps the caller's ticket atomic).  NRM: also composite the flat per-face normal f.nrm[slot]
// (Eq. 12, reading S26), staged in the warp's `nsm[32]`.
// FULLREC (fused tracking job): SMEM is the backward's BwdWarpSmem (rows 0-5 mean the same in both layouts); for the
// LAST chunk of the tile list the lanes also stage record rows R4-R9 into rows 6-11 and every lane publishes its lane
// mask, so that the pose-only backward walk of the same job -- which begins in that chunk unless every pixel
// terminated earlier -- can start without loading anything again (ts_bwd_walk, `prestaged_lo`; *staged_lo = list
// position of that chunk relative to the tile's begin, 0xffffffff if it was not staged).
template <int SM, bool COUNT, bool STATS = false, bool NRM = false, bool FULLREC = false, class SMEM = FwdWarpSmem>
__device__ __forceinline__ void ts_fwd_walk(const TsFrameDev& f, const ts_scene& sc, const TsJob& job, int lane,
                                            SMEM& sm, float sigma, float alpha_min, float t_min, uint4 ent,
                                            FwdPix& o, unsigned long long& n_visit, unsigned long long& n_rect,
                                            unsigned long long& n_hit, uint32_t* __restrict__ face_pixels = nullptr,
                                            float4* nsm = nullptr, uint32_t* staged_lo = nullptr) {
    // generic-sigma instantiation (SM == 0): the exponent of entry e is staged in the slice's pad row (reading S32)
    constexpr int SIGROW = FULLREC ? 12 : 6;
    const float fpx = (float)job.px, fpy = (float)job.py;
    float T = 1.0f, C0 = 0.0f, C1 = 0.0f, C2 = 0.0f, D = 0.0f, Tlast = 1.0f;
    float N0 = 0.0f, N1 = 0.0f, N2 = 0.0f, Nt0 = 0.0f, Nt1 = 0.0f, Nt2 = 0.0f, a_top = 0.0f;
    uint32_t last = 0;
    const uint32_t lt = (1u << lane) - 1u;
    (void)lt;
    bool done = !job.inside;
    bool warp_done = __all_sync(0xffffffffu, done);
    for (uint32_t c0 = job.range.x; c0 < job.range.y && !warp_done; c0 += 32) {
        const uint32_t n = min(32u, job.range.y - c0);
        const uint4 cur = ent;
        if (c0 + 32 + lane < job.range.y) ent = f.blist[c0 + 32 + lane];     // prefetch the next chunk
        uint32_t lmask = (uint32_t)lane < n ? ts_entry_mask(job, cur) : 0u;   // (never 0 for an entry of the block's list)
        __syncwarp();                                   // previous chunk's reads are done
        if (lmask) {
            // records are staged at the lane's own index (no compaction: nothing has to stay in registers
            // across the ballot); the walk below follows the set bits of `ov` in list order
            const float4* rp = f.rec + TS_REC_F4 * (size_t)cur.x;
            const float4 r0 = __ldg(rp), r1 = __ldg(rp + 1), r2 = __ldg(rp + 2), r3 = __ldg(rp + 3);
            float col[9];
            ts_load_colors(sc, cur.y, col);
            if (ts_job_block_misses(job, cur, r0, r1, r2)) lmask = 0u;
            sm.r[lane][0] = r0, sm.r[lane][1] = r1, sm.r[lane][2] = r2;
            sm.r[lane][3] = make_float4(r3.x, r3.y, r3.z, col[0]);
            sm.r[lane][4] = make_float4(col[1], col[2], col[3], col[4]);
            sm.r[lane][5] = make_float4(col[5], col[6], col[7], col[8]);
            if (SM == 0) sm.r[lane][SIGROW] = make_float4(r3.w, 0.f, 0.f, 0.f);
            sm.lm[lane] = lmask, sm.slot[lane] = cur.x;
            if (STATS) sm.face[lane] = cur.y;
            if (NRM) nsm[lane] = f.nrm[cur.x];
            if (FULLREC && lmask && c0 + 32u >= job.range.y) {   // (only the list's last chunk: that is where the backward begins)
                // the rest of the record, in two batches to keep the live range short
                const float4 a0 = __ldg(rp + 4), a1 = __ldg(rp + 5), a2 = __ldg(rp + 6);
                sm.r[lane][6] = a0, sm.r[lane][7] = a1, sm.r[lane][8] = a2;
                const float4 b0 = __ldg(rp + 7), b1 = __ldg(rp + 8), b2 = __ldg(rp + 9);
                sm.r[lane][9] = b0, sm.r[lane][10] = b1, sm.r[lane][11] = b2;
                sm.face[lane] = cur.y;                  // (read by the full-gradient backward only)
            }
        }
        if (FULLREC && c0 + 32u >= job.range.y) {
            if (!lmask) sm.lm[lane] = 0u;               // lanes without an entry for this block
            *staged_lo = c0 - job.range.x;
        }
        __syncwarp();
        uint32_t ov = __ballot_sync(0xffffffffu, lmask != 0u);
        const uint32_t pos0 = (c0 - job.range.x) + 1u;
        while (ov) {
            const int e = __ffs(ov) - 1;
            ov &= ov - 1;
            const bool in_rect = !done && ((sm.lm[e] >> lane) & 1u);
            if (COUNT) n_visit += 1, n_rect += in_rect ? 1 : 0;
            // (no warp votes here: after the exact block cull nearly every visit has a lane inside the rect and a
            // hit, so "skip if nobody ..." tests cost more than they save)
            float l[3], x, I, alpha;
            bool hit = false;
            if (in_rect) {
                const float4 r0 = sm.r[e][0], r1 = sm.r[e][1], r2 = sm.r[e][2];
                const float sg = SM == 0 ? sm.r[e][SIGROW].x : sigma;
                hit = ts_eval_alpha<SM>(r0, r1, r2, fpx, fpy, sg, alpha_min, f.scr, sm.slot[e], l, x, I, alpha);
            }
            if (STATS) {
                // statistics: the face contributed to popc(hm) pixels of this block (one RED per visit)
                const uint32_t hm = __ballot_sync(0xffffffffu, hit);
                if (hm && lane == __ffs(hm) - 1) atomicAdd(face_pixels + sm.face[e], (uint32_t)__popc(hm));
            }
            if (hit) {
                const float4 r3 = sm.r[e][3], r4 = sm.r[e][4], r5 = sm.r[e][5];
                if (COUNT) n_hit += 1;
                const float o0 = l[0] * r3.x, o1 = l[1] * r3.y, o2 = l[2] * r3.z;   // omega_k = lhat_k kappa_k
                const float Om = (o0 + o1) + o2;
                const float z = ts_rcp_approx(Om);
                const float wgt = T * alpha, wz = wgt * z;
                C0 = fmaf(wz, fmaf(o0, r3.w, fmaf(o1, r4.z, o2 * r5.y)), C0);
                C1 = fmaf(wz, fmaf(o0, r4.x, fmaf(o1, r4.w, o2 * r5.z)), C1);
                C2 = fmaf(wz, fmaf(o0, r4.y, fmaf(o1, r5.x, o2 * r5.w)), C2);
                D += wz;
                if (NRM) {
                    const float4 nf = nsm[e];
                    N0 = fmaf(wgt, nf.x, N0), N1 = fmaf(wgt, nf.y, N1), N2 = fmaf(wgt, nf.z, N2);
                    if (alpha > a_top) a_top = alpha, Nt0 = nf.x, Nt1 = nf.y, Nt2 = nf.z;     // Fig. 3 (right), reading S29
                }
                Tlast = T;
                T = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                last = pos0 + (uint32_t)e;
                if (T <= t_min) done = true;
            }
        }
        warp_done = __all_sync(0xffffffffu, done);      // once per chunk: pixels rarely all terminate inside one
    }
    o.T = T, o.C0 = C0, o.C1 = C1, o.C2 = C2, o.D = D, o.Tlast = Tlast, o.last = last;
    if (NRM) o.N0 = N0, o.N1 = N1, o.N2 = N2, o.Nt0 = Nt0, o.Nt1 = Nt1, o.Nt2 = Nt2;
}
