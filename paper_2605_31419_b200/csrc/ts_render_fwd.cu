// ts_render_fwd.cu -- a3: per-tile front-to-back compositing (Eq. 2-4).
// One CTA per 16x16 tile, one thread per pixel.  The tile's sorted list is consumed in batches of TS_BATCH
// entries: 128 threads each set up ONE face (edge functions normalised by the inradius, perspective weights,
// colours) and park it in shared memory as 7 float4; a ballot per 8x4-pixel warp block records which entries can
// touch that block at all, so a warp visits only faces whose pixel rect overlaps its own 32 pixels and reads each
// record with broadcast LDS.128.  Pixels stop at T <= t_min, warps when all their pixels stopped, the CTA when
// all warps stopped.
#include "ts_raster.cuh"

namespace {

struct FwdRec { float4 r[7]; };   // 112 B, see stage_face()

__device__ __forceinline__ void stage_face(const TsFrameDev& f, const ts_scene& sc, uint32_t slot, FwdRec& out,
                                           int& x0, int& y0, int& x1, int& y1) {
    const float4* s4 = f.scr + 3 * (size_t)slot;
    const float4 s0 = __ldg(s4), s1 = __ldg(s4 + 1), s2 = __ldg(s4 + 2);
    TsGeom g;
    ts_face_geom(s0, s1, s2, g);
    const uint32_t m = __ldg(f.vis_face + slot);
    float col[9];
    if (sc.faces == nullptr) {
        const float* cp = sc.color + 9 * (size_t)m;
#pragma unroll
        for (int j = 0; j < 9; ++j) col[j] = __ldg(cp + j);
    } else {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const float* cp = sc.color + 3 * (size_t)__ldg(sc.faces + 3 * (size_t)m + k);
            col[3 * k] = __ldg(cp), col[3 * k + 1] = __ldg(cp + 1), col[3 * k + 2] = __ldg(cp + 2);
        }
    }
    out.r[0] = make_float4(g.refx, g.refy, s2.z, s2.w);
    out.r[1] = make_float4(g.mx[0], g.my[0], g.mx[1], g.my[1]);
    out.r[2] = make_float4(g.mx[2], g.my[2], g.c[0], g.c[1]);
    out.r[3] = make_float4(g.c[2], g.obar, g.kap[0], g.kap[1]);
    out.r[4] = make_float4(g.kap[2], col[0], col[1], col[2]);
    out.r[5] = make_float4(col[3], col[4], col[5], col[6]);
    out.r[6] = make_float4(col[7], col[8], __uint_as_float(slot), 0.0f);
    x0 = g.x0, y0 = g.y0, x1 = g.x1, y1 = g.y1;
}

template <int SM, bool COUNT>
__global__ void __launch_bounds__(256)
render_fwd_kernel(TsFrameDev f, ts_scene sc, const uint32_t* __restrict__ vals, float sigma, float alpha_min,
                  float t_min, float* __restrict__ out_color, float* __restrict__ out_depth,
                  float* __restrict__ out_alpha) {
    __shared__ FwdRec recs[TS_BATCH];
    __shared__ uint32_t masks[8][TS_BATCH / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x, tx0 = (tile % f.tiles_x) * TS_TILE, ty0 = (tile / f.tiles_x) * TS_TILE;
    int lx, ly;
    ts_thread_pixel(tid, lx, ly);
    const int px = tx0 + lx, py = ty0 + ly;
    const bool inside = px < f.W && py < f.H;
    const float fpx = (float)px, fpy = (float)py;
    uint2 range = f.tile_ranges[tile];
    if (ts_eff_pairs(f) == 0) range = make_uint2(0u, 0u);
    float T = 1.0f, C0 = 0.0f, C1 = 0.0f, C2 = 0.0f, D = 0.0f, Tlast = 1.0f;
    uint32_t last = 0;
    bool done = !inside;
    unsigned long long n_rect = 0, n_hit = 0, n_visit = 0;

    for (uint32_t b0 = range.x; b0 < range.y; b0 += TS_BATCH) {
        const int nb = (int)min((uint32_t)TS_BATCH, range.y - b0);
        if (__syncthreads_and(done)) break;            // also fences the previous batch's reads
        if (tid < TS_BATCH) {
            uint32_t sub = 0;
            if (tid < nb) {
                int x0, y0, x1, y1;
                stage_face(f, sc, __ldg(vals + b0 + tid), recs[tid], x0, y0, x1, y1);
                sub = ts_subtile_mask(max(x0 - tx0, 0), max(y0 - ty0, 0), min(x1 - tx0, 15), min(y1 - ty0, 15));
            }
#pragma unroll
            for (int w = 0; w < 8; ++w) {
                const uint32_t bal = __ballot_sync(0xffffffffu, (sub >> w) & 1u);
                if (lane == 0) masks[w][warp] = bal;
            }
        }
        __syncthreads();
        bool warp_done = __all_sync(0xffffffffu, done);
        for (int g = 0; g < (nb + 31) / 32 && !warp_done; ++g) {
            uint32_t m = masks[warp][g];
            while (m) {
                const int e = (g << 5) + __ffs(m) - 1;
                m &= m - 1;
                const FwdRec& R = recs[e];
                const float4 r0 = R.r[0];
                const int rlo = __float_as_int(r0.z), rhi = __float_as_int(r0.w);
                const bool in_rect = !done && px >= (int)(short)(rlo & 0xffff) && px <= (int)(short)(rhi & 0xffff) &&
                                     py >= (rlo >> 16) && py <= (rhi >> 16);
                if (COUNT) n_visit += 1, n_rect += in_rect ? 1 : 0;
                if (!__any_sync(0xffffffffu, in_rect)) continue;
                const float4 r1 = R.r[1], r2 = R.r[2], r3 = R.r[3];
                const float4* s4 = f.scr + 3 * (size_t)__float_as_uint(R.r[6].z);
                float l[3], x, I, alpha;
                const bool hit = in_rect && ts_eval_alpha<SM>(r0.x, r0.y, r1.x, r1.y, r1.z, r1.w, r2.x, r2.y, r2.z, r2.w,
                                                              r3.x, r3.y, fpx, fpy, sigma, alpha_min, s4, l, x, I, alpha);
                if (!__any_sync(0xffffffffu, hit)) continue;
                const float4 r4 = R.r[4], r5 = R.r[5], r6 = R.r[6];
                if (hit) {
                    if (COUNT) n_hit += 1;
                    const float o0 = l[0] * r3.z, o1 = l[1] * r3.w, o2 = l[2] * r4.x;   // omega_k = lhat_k kappa_k
                    const float Om = (o0 + o1) + o2;
                    const float z = __fdividef(1.0f, Om);
                    const float wgt = T * alpha, wz = wgt * z;
                    C0 = fmaf(wz, fmaf(o0, r4.y, fmaf(o1, r5.x, o2 * r5.w)), C0);
                    C1 = fmaf(wz, fmaf(o0, r4.z, fmaf(o1, r5.y, o2 * r6.x)), C1);
                    C2 = fmaf(wz, fmaf(o0, r4.w, fmaf(o1, r5.z, o2 * r6.y)), C2);
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
void launch_sm(const ts_frame* fr, const ts_scene& sc, const uint32_t* vals, float* oc, float* od, float* oa,
               cudaStream_t st) {
    const TsFrameDev& f = fr->d;
    const bool count = (fr->prm.flags & 0x100u) != 0;
    if (count)
        render_fwd_kernel<SM, true><<<f.NT, 256, 0, st>>>(f, sc, vals, fr->prm.sigma, fr->prm.alpha_min, fr->prm.t_min, oc, od, oa);
    else
        render_fwd_kernel<SM, false><<<f.NT, 256, 0, st>>>(f, sc, vals, fr->prm.sigma, fr->prm.alpha_min, fr->prm.t_min, oc, od, oa);
}

}  // namespace

int32_t ts_launch_render_fwd(const ts_ctx*, ts_frame* fr, const ts_scene* sc, float* oc, float* od, float* oa,
                             cudaStream_t st) {
    const uint32_t* vals = fr->d.vals[fr->sorted_buf];
    switch (ts_sigma_mode(fr->prm.sigma)) {
        case 1: launch_sm<1>(fr, *sc, vals, oc, od, oa, st); break;
        case 2: launch_sm<2>(fr, *sc, vals, oc, od, oa, st); break;
        case 3: launch_sm<3>(fr, *sc, vals, oc, od, oa, st); break;
        default: launch_sm<0>(fr, *sc, vals, oc, od, oa, st); break;
    }
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
