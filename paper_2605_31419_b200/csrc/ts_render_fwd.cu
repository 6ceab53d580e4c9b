// ts_render_fwd.cu -- a3: per-tile front-to-back compositing (Eq. 2-4).
// One CTA per 16x16 tile, one thread per pixel.  The tile's sorted list is consumed in batches of TS_BATCH
// entries: 128 threads each copy ONE pre-built face record (ts_raster.cuh; four LDG.128 + the vertex colours)
// into shared memory and derive, for each of the CTA's eight 8x4-pixel warp blocks, the 32-bit mask of lanes whose
// pixel lies inside the face's rect.  A warp then visits only the entries whose mask is non-zero for its block,
// reads each record with broadcast LDS.128 and tests "my pixel is in the rect" with one shift.  Pixels stop at
// T <= t_min, warps when all their pixels stopped, the CTA when all warps stopped.
#include "ts_raster.cuh"

namespace {

struct FwdSmem {
    float4 r[TS_BATCH][6];            // R0 R1 R2 | kap0 kap1 kap2 c00 | c01 c02 c10 c11 | c12 c20 c21 c22
    uint32_t lm[8][TS_BATCH];         // lane masks per warp block
    uint32_t slot[TS_BATCH];
    uint32_t masks[8][TS_BATCH / 32]; // entries with a non-zero lane mask, per warp block
};

template <int SM, bool COUNT>
__global__ void __launch_bounds__(256)
render_fwd_kernel(TsFrameDev f, ts_scene sc, float sigma, float alpha_min, float t_min, float* __restrict__ out_color,
                  float* __restrict__ out_depth, float* __restrict__ out_alpha) {
    __shared__ FwdSmem sm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x, tx0 = (tile % f.tiles_x) * TS_TILE, ty0 = (tile / f.tiles_x) * TS_TILE;
    int lx, ly;
    ts_thread_pixel(tid, lx, ly);
    const int px = tx0 + lx, py = ty0 + ly;
    const bool inside = px < f.W && py < f.H;
    const float fpx = (float)px, fpy = (float)py;
    const uint2 range = f.tile_ranges[tile];
    float T = 1.0f, C0 = 0.0f, C1 = 0.0f, C2 = 0.0f, D = 0.0f, Tlast = 1.0f;
    uint32_t last = 0;
    bool done = !inside;
    unsigned long long n_rect = 0, n_hit = 0, n_visit = 0;

    for (uint32_t b0 = range.x; b0 < range.y; b0 += TS_BATCH) {
        const int nb = (int)min((uint32_t)TS_BATCH, range.y - b0);
        if (__syncthreads_and(done)) break;            // also fences the previous batch's reads
        if (tid < TS_BATCH) {
            uint32_t lmask[8];
#pragma unroll
            for (int w = 0; w < 8; ++w) lmask[w] = 0u;
            if (tid < nb) {
                const uint2 sf = f.sorted[b0 + tid];   // (slot, face)
                const float4* rp = f.rec + TS_REC_F4 * (size_t)sf.x;
                const float4 r0 = __ldg(rp), r1 = __ldg(rp + 1), r2 = __ldg(rp + 2), r3 = __ldg(rp + 3), r4 = __ldg(rp + 4);
                float col[9];
                if (sc.faces == nullptr) {
                    const float* cp = sc.color + 9 * (size_t)sf.y;
#pragma unroll
                    for (int j = 0; j < 9; ++j) col[j] = __ldg(cp + j);
                } else {
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        const float* cp = sc.color + 3 * (size_t)__ldg(sc.faces + 3 * (size_t)sf.y + k);
                        col[3 * k] = __ldg(cp), col[3 * k + 1] = __ldg(cp + 1), col[3 * k + 2] = __ldg(cp + 2);
                    }
                }
                sm.r[tid][0] = r0, sm.r[tid][1] = r1, sm.r[tid][2] = r2;
                sm.r[tid][3] = make_float4(r3.x, r3.y, r3.z, col[0]);
                sm.r[tid][4] = make_float4(col[1], col[2], col[3], col[4]);
                sm.r[tid][5] = make_float4(col[5], col[6], col[7], col[8]);
                sm.slot[tid] = sf.x;
                const int rlo = __float_as_int(r3.w), rhi = __float_as_int(r4.w);
                const int rx0 = max((int)(short)(rlo & 0xffff) - tx0, 0), ry0 = max((rlo >> 16) - ty0, 0);
                const int rx1 = min((int)(short)(rhi & 0xffff) - tx0, 15), ry1 = min((rhi >> 16) - ty0, 15);
#pragma unroll
                for (int w = 0; w < 8; ++w) lmask[w] = ts_lane_mask(w, rx0, ry0, rx1, ry1);
            }
#pragma unroll
            for (int w = 0; w < 8; ++w) {
                sm.lm[w][tid] = lmask[w];
                const uint32_t bal = __ballot_sync(0xffffffffu, lmask[w] != 0u);
                if (lane == 0) sm.masks[w][warp] = bal;
            }
        }
        __syncthreads();
        bool warp_done = __all_sync(0xffffffffu, done);
        for (int g = 0; g < (nb + 31) / 32 && !warp_done; ++g) {
            uint32_t m = sm.masks[warp][g];
            while (m) {
                const int e = (g << 5) + __ffs(m) - 1;
                m &= m - 1;
                const bool in_rect = !done && ((sm.lm[warp][e] >> lane) & 1u);
                if (COUNT) n_visit += 1, n_rect += in_rect ? 1 : 0;
                if (!__any_sync(0xffffffffu, in_rect)) continue;
                const float4 r0 = sm.r[e][0], r1 = sm.r[e][1], r2 = sm.r[e][2];
                const float4* s4 = f.scr + TS_SCR_F4 * (size_t)sm.slot[e];
                float l[3], x, I, alpha;
                const bool hit = in_rect && ts_eval_alpha<SM>(r0, r1, r2, fpx, fpy, sigma, alpha_min, s4, l, x, I, alpha);
                if (!__any_sync(0xffffffffu, hit)) continue;
                const float4 r3 = sm.r[e][3], r4 = sm.r[e][4], r5 = sm.r[e][5];
                if (hit) {
                    if (COUNT) n_hit += 1;
                    const float o0 = l[0] * r3.x, o1 = l[1] * r3.y, o2 = l[2] * r3.z;   // omega_k = lhat_k kappa_k
                    const float Om = (o0 + o1) + o2;
                    const float z = __fdividef(1.0f, Om);
                    const float wgt = T * alpha, wz = wgt * z;
                    C0 = fmaf(wz, fmaf(o0, r3.w, fmaf(o1, r4.z, o2 * r5.y)), C0);
                    C1 = fmaf(wz, fmaf(o0, r4.x, fmaf(o1, r4.w, o2 * r5.z)), C1);
                    C2 = fmaf(wz, fmaf(o0, r4.y, fmaf(o1, r5.x, o2 * r5.w)), C2);
                    D += wz;
                    Tlast = T;
                    T = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                    last = (b0 - range.x) + (uint32_t)e + 1u;
                    if (T <= t_min) done = true;
                }
                if (__all_sync(0xffffffffu, done)) { warp_done = true; break; }
            }
        }
    }
    if (inside) {
        const size_t p = (size_t)py * f.W + px, hw = (size_t)f.W * f.H;
        if (out_color) out_color[p] = C0, out_color[hw + p] = C1, out_color[2 * hw + p] = C2;
        if (out_depth) out_depth[p] = D;
        if (out_alpha) out_alpha[p] = 1.0f - T;
        f.n_contrib[p] = last;
        f.t_last[p] = Tlast;
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
void launch_sm(const ts_frame* fr, const ts_scene& sc, float* oc, float* od, float* oa, cudaStream_t st) {
    const TsFrameDev& f = fr->d;
    const bool count = (fr->prm.flags & 0x100u) != 0;
    if (count)
        render_fwd_kernel<SM, true><<<f.NT, 256, 0, st>>>(f, sc, fr->prm.sigma, fr->prm.alpha_min, fr->prm.t_min, oc, od, oa);
    else
        render_fwd_kernel<SM, false><<<f.NT, 256, 0, st>>>(f, sc, fr->prm.sigma, fr->prm.alpha_min, fr->prm.t_min, oc, od, oa);
}

}  // namespace

int32_t ts_launch_render_fwd(const ts_ctx*, ts_frame* fr, const ts_scene* sc, float* oc, float* od, float* oa,
                             cudaStream_t st) {
    switch (ts_sigma_mode(fr->prm.sigma)) {
        case 1: launch_sm<1>(fr, *sc, oc, od, oa, st); break;
        case 2: launch_sm<2>(fr, *sc, oc, od, oa, st); break;
        case 3: launch_sm<3>(fr, *sc, oc, od, oa, st); break;
        default: launch_sm<0>(fr, *sc, oc, od, oa, st); break;
    }
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
