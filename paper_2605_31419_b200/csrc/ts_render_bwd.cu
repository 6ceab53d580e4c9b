// ts_render_bwd.cu -- a5/a6/a7: reverse-order backward of the compositing (B1-B9).
//   render_bwd_kernel : one CTA per tile, one thread per pixel, walks the tile list BACK from the last
//       contributing entry; recomputes alpha bit-identically to the forward kernel (ts_raster.cuh), recovers the
//       transmittance in front of each face by T_n = T_{n+1}/(1-alpha_n), keeps the "behind" accumulators
//       R^c, R^d, R^a (no division by T), and forms the per-hit gradients wrt the face's screen vertices
//       (u,v,w) x 3, its vertex colours and its opacity.  Per face these are reduced across the warp with
//       shuffles BEFORE any global atomic (one lane issues the RED.ADD.F32s).
//   proj_bwd_kernel   : per visible face, screen -> camera -> world (B7-B8) and the se(3) terms
//       [g_C ; Q x g_C] of Eq. 5-7, tree-reduced per CTA into fixed-order partials.
//   pose_reduce_kernel: fixed-order final reduction of the partials to dL/dtau[6].
#include "ts_raster.cuh"

namespace {

struct BwdRec { float4 r[12]; };   // 192 B, see stage_face_bwd()

__device__ __forceinline__ void stage_face_bwd(const TsFrameDev& f, const ts_scene& sc, uint32_t slot, BwdRec& out,
                                               uint32_t& face, int& x0, int& y0, int& x1, int& y1) {
    const float4* s4 = f.scr + 3 * (size_t)slot;
    const float4 s0 = __ldg(s4), s1 = __ldg(s4 + 1), s2 = __ldg(s4 + 2);
    TsGeom g;
    ts_face_geom(s0, s1, s2, g);
    const uint32_t m = __ldg(f.vis_face + slot);
    face = m;
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
    // d r / d q_j = -rho_j n_j - (r / sum ell) (u_{j,j+1} + u_{j,j+2}),  u_{j,i} = (q_j - q_i)/|q_j - q_i|;
    // stored as drr_j = -(1/r) dr/dq_j so that gq_j += (x * gx) * drr_j  (B6 iii)
    float drrx[3], drry[3];
    const float rs = g.r * g.inv_sumell;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int i1 = (j + 1) % 3, i2 = (j + 2) % 3;
        const float u1x = (g.qx[j] - g.qx[i1]) * g.inv_ell[i2], u1y = (g.qy[j] - g.qy[i1]) * g.inv_ell[i2];
        const float u2x = (g.qx[j] - g.qx[i2]) * g.inv_ell[i1], u2y = (g.qy[j] - g.qy[i2]) * g.inv_ell[i1];
        const float drx = -g.rho[j] * g.nx[j] - rs * (u1x + u2x), dry = -g.rho[j] * g.ny[j] - rs * (u1y + u2y);
        drrx[j] = -drx * g.inv_r, drry[j] = -dry * g.inv_r;
    }
    out.r[0] = make_float4(g.refx, g.refy, s2.z, s2.w);
    out.r[1] = make_float4(g.mx[0], g.my[0], g.mx[1], g.my[1]);
    out.r[2] = make_float4(g.mx[2], g.my[2], g.c[0], g.c[1]);
    out.r[3] = make_float4(g.c[2], g.obar, g.kap[0], g.kap[1]);
    out.r[4] = make_float4(g.kap[2], col[0], col[1], col[2]);
    out.r[5] = make_float4(col[3], col[4], col[5], col[6]);
    out.r[6] = make_float4(col[7], col[8], g.rho[0], g.rho[1]);
    out.r[7] = make_float4(g.rho[2], g.w[0], g.w[1], g.w[2]);
    out.r[8] = make_float4(g.qx[0] - g.refx, g.qy[0] - g.refy, g.qx[1] - g.refx, g.qy[1] - g.refy);
    out.r[9] = make_float4(g.qx[2] - g.refx, g.qy[2] - g.refy, g.inv_ell[0] * g.inv_ell[0], g.inv_ell[1] * g.inv_ell[1]);
    out.r[10] = make_float4(g.inv_ell[2] * g.inv_ell[2], drrx[0], drry[0], drrx[1]);
    out.r[11] = make_float4(drry[1], drrx[2], drry[2], __uint_as_float(slot));
    x0 = g.x0, y0 = g.y0, x1 = g.x1, y1 = g.y1;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// ATTR: also colour / opacity gradients (B1, B4).  GEOM: screen-space vertex gradients (B5-B6).
template <int SM, bool ATTR, bool GEOM>
__global__ void __launch_bounds__(256)
render_bwd_kernel(TsFrameDev f, ts_scene sc, const uint32_t* __restrict__ vals, float sigma, float alpha_min,
                  const float* __restrict__ gCi, const float* __restrict__ gDi, const float* __restrict__ gAi,
                  float* __restrict__ grad_color, float* __restrict__ grad_opacity) {
    __shared__ BwdRec recs[TS_BATCH];
    __shared__ uint32_t faces_s[TS_BATCH];
    __shared__ uint32_t masks[8][TS_BATCH / 32];
    __shared__ uint32_t s_max;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x, tx0 = (tile % f.tiles_x) * TS_TILE, ty0 = (tile / f.tiles_x) * TS_TILE;
    int lx, ly;
    ts_thread_pixel(tid, lx, ly);
    const int px = tx0 + lx, py = ty0 + ly;
    const bool inside = px < f.W && py < f.H;
    const float fpx = (float)px, fpy = (float)py;
    uint2 range = f.tile_ranges[tile];
    if (ts_eff_pairs(f) == 0) range = make_uint2(0u, 0u);
    const size_t p = (size_t)py * f.W + px, hw = (size_t)f.W * f.H;
    uint32_t ncon = 0;
    float Tcur = 1.0f, gC0 = 0.f, gC1 = 0.f, gC2 = 0.f, gD = 0.f, gA = 0.f;
    if (inside && range.y > range.x) {
        ncon = f.n_contrib[p];
        Tcur = f.t_last[p];
        if (gCi) gC0 = gCi[p], gC1 = gCi[hw + p], gC2 = gCi[2 * hw + p];
        if (gDi) gD = gDi[p];
        if (gAi) gA = gAi[p];
    }
    if (tid == 0) s_max = 0;
    __syncthreads();
    const uint32_t wmax = __reduce_max_sync(0xffffffffu, ncon);
    if (lane == 0 && wmax) atomicMax(&s_max, wmax);
    __syncthreads();
    const uint32_t n_walk = min(s_max, range.y - range.x);
    float Rc0 = 0.f, Rc1 = 0.f, Rc2 = 0.f, Rd = 0.f, Ra = 0.f;
    bool first = true;

    for (uint32_t hi = n_walk; hi > 0;) {
        const uint32_t lo = hi > TS_BATCH ? hi - TS_BATCH : 0u;
        const int nb = (int)(hi - lo);
        __syncthreads();
        if (tid < TS_BATCH) {
            uint32_t sub = 0;
            if (tid < nb) {
                int x0, y0, x1, y1;
                uint32_t face;
                stage_face_bwd(f, sc, __ldg(vals + range.x + lo + tid), recs[tid], face, x0, y0, x1, y1);
                faces_s[tid] = face;
                sub = ts_subtile_mask(max(x0 - tx0, 0), max(y0 - ty0, 0), min(x1 - tx0, 15), min(y1 - ty0, 15));
            }
#pragma unroll
            for (int w = 0; w < 8; ++w) {
                const uint32_t bal = __ballot_sync(0xffffffffu, (sub >> w) & 1u);
                if (lane == 0) masks[w][warp] = bal;
            }
        }
        __syncthreads();
        if (wmax > lo) {
            for (int g = (nb - 1) >> 5; g >= 0; --g) {
                uint32_t mk = masks[warp][g];
                while (mk) {
                    const int bit = 31 - __clz(mk);
                    mk &= ~(1u << bit);
                    const int e = (g << 5) + bit;
                    const uint32_t idx = lo + (uint32_t)e;          // list position relative to range.x
                    const BwdRec& R = recs[e];
                    const float4 r0 = R.r[0];
                    const int rlo = __float_as_int(r0.z), rhi = __float_as_int(r0.w);
                    const bool in_rect = idx < ncon && px >= (int)(short)(rlo & 0xffff) && px <= (int)(short)(rhi & 0xffff) &&
                                         py >= (rlo >> 16) && py <= (rhi >> 16);
                    if (!__any_sync(0xffffffffu, in_rect)) continue;
                    const float4 r1 = R.r[1], r2 = R.r[2], r3 = R.r[3];
                    const float4* s4 = f.scr + 3 * (size_t)__float_as_uint(R.r[11].w);
                    float l[3], x, I, alpha;
                    const bool hit = in_rect && ts_eval_alpha<SM>(r0.x, r0.y, r1.x, r1.y, r1.z, r1.w, r2.x, r2.y, r2.z,
                                                                  r2.w, r3.x, r3.y, fpx, fpy, sigma, alpha_min, s4, l, x, I, alpha);
                    const uint32_t hm = __ballot_sync(0xffffffffu, hit);
                    if (!hm) continue;
                    const float4 r4 = R.r[4], r5 = R.r[5], r6 = R.r[6];
                    float acc[19];
#pragma unroll
                    for (int j = 0; j < 19; ++j) acc[j] = 0.f;
                    if (hit) {
                        // transmittance in front of this face
                        const float one_m = __fsub_rn(1.0f, alpha);
                        const float Tn = first ? Tcur : __fdiv_rn(Tcur, one_m);
                        Tcur = Tn, first = false;
                        const float o0 = l[0] * r3.z, o1 = l[1] * r3.w, o2 = l[2] * r4.x;
                        const float Om = (o0 + o1) + o2, z = __fdividef(1.0f, Om);
                        const float lam0 = o0 * z, lam1 = o1 * z, lam2 = o2 * z;
                        const float c0 = lam0 * r4.y + lam1 * r5.x + lam2 * r5.w;
                        const float c1 = lam0 * r4.z + lam1 * r5.y + lam2 * r6.x;
                        const float c2 = lam0 * r4.w + lam1 * r5.z + lam2 * r6.y;
                        const float wgt = Tn * alpha;
                        // B2
                        const float ga = Tn * ((c0 - Rc0) * gC0 + (c1 - Rc1) * gC1 + (c2 - Rc2) * gC2 + (z - Rd) * gD +
                                               (1.0f - Ra) * gA);
                        // B3
                        Rc0 = alpha * c0 + one_m * Rc0, Rc1 = alpha * c1 + one_m * Rc1, Rc2 = alpha * c2 + one_m * Rc2;
                        Rd = alpha * z + one_m * Rd, Ra = alpha + one_m * Ra;
                        if (ATTR) {
                            // B1 colours, B4 opacity (one value per face; /3 applied when written)
                            const float w0 = lam0 * wgt, w1 = lam1 * wgt, w2 = lam2 * wgt;
                            acc[9] = w0 * gC0, acc[10] = w0 * gC1, acc[11] = w0 * gC2;
                            acc[12] = w1 * gC0, acc[13] = w1 * gC1, acc[14] = w1 * gC2;
                            acc[15] = w2 * gC0, acc[16] = w2 * gC1, acc[17] = w2 * gC2;
                            acc[18] = I * ga;
                        }
                        if (GEOM) {
                            const float4 r7 = R.r[7], r8 = R.r[8], r9 = R.r[9], r10 = R.r[10], r11 = R.r[11];
                            // B4 window: gx = dL/dx
                            const float gI = r3.y * ga;
                            float gx;
                            if (SM == 1) gx = gI;
                            else if (SM == 2) gx = 0.5f * gI * __fdividef(1.0f, I);
                            else if (SM == 3) gx = 2.0f * gI * x;
                            else gx = gI * sigma * I * __fdividef(1.0f, x);
                            // B5 interpolation
                            const float cg = c0 * gC0 + c1 * gC1 + c2 * gC2;
                            const float wz = wgt * z, zgd = z * gD;
                            const float go0 = wz * ((r4.y * gC0 + r4.z * gC1 + r4.w * gC2) - cg - zgd);
                            const float go1 = wz * ((r5.x * gC0 + r5.y * gC1 + r5.z * gC2) - cg - zgd);
                            const float go2 = wz * ((r5.w * gC0 + r6.x * gC1 + r6.y * gC2) - cg - zgd);
                            const float b0 = -l[0] * r6.z, b1 = -l[1] * r6.w, b2 = -l[2] * r7.x;      // b_k = -lhat_k rho_k
                            const float gb0 = r7.y * go0, gb1 = r7.z * go1, gb2 = r7.w * go2;         // w_k * gomega_k
                            acc[2] = b0 * go0, acc[5] = b1 * go1, acc[8] = b2 * go2;                 // dL/dw_k
                            // B6 (i): G = sum_k gb_k grad_p b_k,  grad_p b_k = -rho_k m_k
                            const float t0 = gb0 * r6.z, t1 = gb1 * r6.w, t2 = gb2 * r7.x;
                            const float Gx = -(t0 * r1.x + t1 * r1.z + t2 * r2.x), Gy = -(t0 * r1.y + t1 * r1.w + t2 * r2.y);
                            float q0x = -b0 * Gx, q0y = -b0 * Gy, q1x = -b1 * Gx, q1y = -b1 * Gy, q2x = -b2 * Gx, q2y = -b2 * Gy;
                            // B6 (ii): x = -lhat_{k*}; edge k* runs from a = q_{k*+1} to b = q_{k*+2}
                            const int ks = (l[0] >= l[1] && l[0] >= l[2]) ? 0 : (l[1] >= l[2] ? 1 : 2);
                            const float dx = fpx - r0.x, dy = fpy - r0.y;
                            float ax, ay, bx, by, mkx, mky, il2;
                            if (ks == 0) ax = r8.z, ay = r8.w, bx = r9.x, by = r9.y, mkx = r1.x, mky = r1.y, il2 = r9.z;
                            else if (ks == 1) ax = r9.x, ay = r9.y, bx = r8.x, by = r8.y, mkx = r1.z, mky = r1.w, il2 = r9.w;
                            else ax = r8.x, ay = r8.y, bx = r8.z, by = r8.w, mkx = r2.x, mky = r2.y, il2 = r10.x;
                            const float ex = bx - ax, ey = by - ay;
                            const float t = ((dx - ax) * ex + (dy - ay) * ey) * il2;
                            const float vax = (1.0f - t) * mkx * gx, vay = (1.0f - t) * mky * gx;
                            const float vbx = t * mkx * gx, vby = t * mky * gx;
                            if (ks == 0) q1x += vax, q1y += vay, q2x += vbx, q2y += vby;
                            else if (ks == 1) q2x += vax, q2y += vay, q0x += vbx, q0y += vby;
                            else q0x += vax, q0y += vay, q1x += vbx, q1y += vby;
                            // B6 (iii): through the inradius
                            const float xg = x * gx;
                            q0x += xg * r10.y, q0y += xg * r10.z, q1x += xg * r10.w, q1y += xg * r11.x;
                            q2x += xg * r11.y, q2y += xg * r11.z;
                            acc[0] = q0x, acc[1] = q0y, acc[3] = q1x, acc[4] = q1y, acc[6] = q2x, acc[7] = q2y;
                        }
                    }
                    // reduce across the warp, then one lane issues the atomics
                    const bool single = (hm & (hm - 1)) == 0;
                    const int src = __ffs(hm) - 1;
                    if (!single) {
                        if (GEOM) {
#pragma unroll
                            for (int j = 0; j < 9; ++j) acc[j] = warp_sum(acc[j]);
                        }
                        if (ATTR) {
#pragma unroll
                            for (int j = 9; j < 19; ++j) acc[j] = warp_sum(acc[j]);
                        }
                    }
                    if (lane == src) {
                        if (GEOM) {
                            float* gs = f.gscr + 9 * (size_t)__float_as_uint(R.r[11].w);
#pragma unroll
                            for (int j = 0; j < 9; ++j) atomicAdd(gs + j, acc[j]);
                        }
                        if (ATTR) {
                            const uint32_t m = faces_s[e];
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
                                const float go = acc[18] * (1.0f / 3.0f);
#pragma unroll
                                for (int k = 0; k < 3; ++k) atomicAdd(grad_opacity + v[k], go);
                            }
                        }
                    }
                }
            }
        }
        hi = lo;
    }
}

}  // namespace

namespace {

constexpr int PB_THREADS = 256;

// a6 + the per-vertex terms of a7.  Persistent grid-stride over visible slots; consumes and re-zeroes gscr.
template <bool SOUP>
__global__ void __launch_bounds__(PB_THREADS)
proj_bwd_kernel(TsFrameDev f, const float* __restrict__ pos, const int32_t* __restrict__ faces,
                const float* __restrict__ Tcw, TsCamDev cam, float* __restrict__ grad_pos, int want_pose) {
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
        if (!any) continue;
#pragma unroll
        for (int j = 0; j < 9; ++j) gs[j] = 0.0f;
        const uint32_t m = f.vis_face[slot];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const size_t v = SOUP ? (size_t)3 * m + k : (size_t)__ldg(faces + 3 * (size_t)m + k);
            const float px = __ldg(pos + 3 * v), py = __ldg(pos + 3 * v + 1), pz = __ldg(pos + 3 * v + 2);
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

// a7: fixed-order tree reduction of the partials
__global__ void __launch_bounds__(256) pose_reduce_kernel(const float* __restrict__ partials, uint32_t n, float* __restrict__ out) {
    __shared__ float sm[256][6];
    const int tid = threadIdx.x;
    float a[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    for (uint32_t i = tid; i < n; i += 256)
#pragma unroll
        for (int j = 0; j < 6; ++j) a[j] += partials[6 * (size_t)i + j];
#pragma unroll
    for (int j = 0; j < 6; ++j) sm[tid][j] = a[j];
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (tid < s)
#pragma unroll
            for (int j = 0; j < 6; ++j) sm[tid][j] += sm[tid + s][j];
        __syncthreads();
    }
    if (tid < 6) out[tid] = sm[0][tid];
}

template <int SM>
void launch_bwd_sm(const ts_frame* fr, const ts_scene& sc, const uint32_t* vals, const float* gC, const float* gD,
                   const float* gA, float* gcol, float* gopa, bool attr, bool geom, cudaStream_t st) {
    const TsFrameDev& f = fr->d;
    const float sg = fr->prm.sigma, am = fr->prm.alpha_min;
    if (attr && geom) render_bwd_kernel<SM, true, true><<<f.NT, 256, 0, st>>>(f, sc, vals, sg, am, gC, gD, gA, gcol, gopa);
    else if (geom) render_bwd_kernel<SM, false, true><<<f.NT, 256, 0, st>>>(f, sc, vals, sg, am, gC, gD, gA, gcol, gopa);
    else render_bwd_kernel<SM, true, false><<<f.NT, 256, 0, st>>>(f, sc, vals, sg, am, gC, gD, gA, gcol, gopa);
}

}  // namespace

int32_t ts_launch_render_bwd(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, const float* gC, const float* gD,
                             const float* gA, float* grad_pos, float* grad_color, float* grad_opacity, uint32_t mask,
                             cudaStream_t st) {
    const bool attr = (mask & (TS_GRAD_COLOR | TS_GRAD_OPACITY)) != 0;
    const bool geom = (mask & (TS_GRAD_POS | TS_GRAD_POSE)) != 0;
    if (!attr && !geom) return TS_OK;
    float* gcol = (mask & TS_GRAD_COLOR) ? grad_color : nullptr;
    float* gopa = (mask & TS_GRAD_OPACITY) ? grad_opacity : nullptr;
    const uint32_t* vals = fr->d.vals[fr->sorted_buf];
    switch (ts_sigma_mode(fr->prm.sigma)) {
        case 1: launch_bwd_sm<1>(fr, *sc, vals, gC, gD, gA, gcol, gopa, attr, geom, st); break;
        case 2: launch_bwd_sm<2>(fr, *sc, vals, gC, gD, gA, gcol, gopa, attr, geom, st); break;
        case 3: launch_bwd_sm<3>(fr, *sc, vals, gC, gD, gA, gcol, gopa, attr, geom, st); break;
        default: launch_bwd_sm<0>(fr, *sc, vals, gC, gD, gA, gcol, gopa, attr, geom, st); break;
    }
    fr->pose_src = 0;
    if (geom) {
        const int grid = (int)fr->d.n_partials_cap;
        const int want_pose = (mask & TS_GRAD_POSE) ? 1 : 0;
        float* gp = (mask & TS_GRAD_POS) ? grad_pos : nullptr;
        if (sc->faces == nullptr)
            proj_bwd_kernel<true><<<grid, PB_THREADS, 0, st>>>(fr->d, sc->pos, nullptr, fr->T_cw, fr->cam, gp, want_pose);
        else
            proj_bwd_kernel<false><<<grid, PB_THREADS, 0, st>>>(fr->d, sc->pos, sc->faces, fr->T_cw, fr->cam, gp, want_pose);
        if (want_pose) fr->pose_src = 2, fr->n_pose_partials = (uint32_t)grid;
    }
    (void)ctx;
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

int32_t ts_launch_pose_reduce(const ts_ctx*, ts_frame* fr, float* out, cudaStream_t st) {
    if (fr->pose_src == 0) return TS_ERR_STATE;
    pose_reduce_kernel<<<1, 256, 0, st>>>(fr->d.pose_partials, fr->n_pose_partials, out);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
