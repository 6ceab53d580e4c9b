// ts_raster.cuh -- the per-face render record (F7), written once per visible face by the binning kernel, and the
// per-(pixel, face) window evaluation (F8.1-3) shared by the forward and backward compositing kernels.  Every
// operation that decides alpha is written with explicit round-to-nearest intrinsics so that the backward kernel
// recomputes bit-identical alpha / transmittance values (no freedom for the compiler to contract differently in
// the two kernels).
//
// Formulation: with the incentre-normalised edge functions
//     lhat_k(p) = L_k(p) / r = m_k . (p - ref) + c_k,   m_k = n_k / r,   c_k = n_k . (ref - q_{k+1}) / r
// (ref = the float-rounded incentre, so |lhat_k| <= ~1 inside the face and c_k ~ -1), Eq. 2-3 become
//     phi(p)/phi(s) = -max_k lhat_k(p) =: x,     I = x^sigma  (x > 0).
// Screen barycentrics are b_k = -lhat_k * rho_k with rho_k = r/h_k = ell_k / sum(ell), and the perspective
// weights are omega_k = lhat_k * kappa_k with kappa_k = -rho_k w_k.
//
// Record layout, 10 float4 = 160 B per visible face (global memory, f.rec + 10 * slot):
//   R0  refx  refy  m0x   m0y        R5  w0     w1     w2     tau0
//   R1  m1x   m1y   m2x   m2y        R6  tau1   tau2   drr0x  drr0y
//   R2  c0    c1    c2    obar       R7  drr1x  drr1y  drr2x  drr2y
//   R3  kap0  kap1  kap2  sigma_f    R8  xn0    yn0    xn1    yn1
//   R4  rho0  rho1  rho2  rect_hi    R9  xn2    yn2    -      -
// R0-R2 decide alpha (forward and backward), R3 interpolates, R4-R7 are the backward-only geometry terms
// (tau_k = foot of vertex k on its opposite edge, drr_j = -(1/r) dr/dq_j), R8-R9 the normalised camera
// coordinates (X/Z, Y/Z) of the vertices for the in-kernel se(3) terms.
#pragma once
#include "ts_internal.cuh"

struct TsGeom {
    float qx[3], qy[3], w[3];
    float nx[3], ny[3], ell[3], inv_ell[3];
    float absS, sgn, sumell, inv_sumell, r, inv_r;
    float refx, refy, mx[3], my[3], c[3], rho[3], kap[3];
    float obar;
};

__device__ __forceinline__ float ts_sqrt_approx(float x) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float ts_rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float ts_rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ void ts_face_geom(const float4 s0, const float4 s1, const float4 s2, float obar, TsGeom& g) {
    g.qx[0] = s0.x, g.qy[0] = s0.y, g.w[0] = s0.z;
    g.qx[1] = s0.w, g.qy[1] = s1.x, g.w[1] = s1.y;
    g.qx[2] = s1.z, g.qy[2] = s1.w, g.w[2] = s2.x;
    g.obar = obar;
    // signed doubled area with the same operation order as the projection (N3): same sign on both sides
    const float a = __fsub_rn(g.qx[1], g.qx[0]), b = __fsub_rn(g.qy[2], g.qy[0]);
    const float c = __fsub_rn(g.qy[1], g.qy[0]), d = __fsub_rn(g.qx[2], g.qx[0]);
    const float S = __fmaf_rn(a, b, -__fmul_rn(c, d));
    g.sgn = S > 0.0f ? 1.0f : -1.0f;
    g.absS = fabsf(S);
    // The record only has to be the same for the forward and the backward kernel (it is: both read it), not
    // correctly rounded: lengths and reciprocals use the MUFU approximations (<= 2 ulp), which keeps this
    // latency-bound set-up chain short.  Decisions next to an edge never depend on it (ts_refine_lhat).
    float sum = 0.0f;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const int ia = (k + 1) % 3, ib = (k + 2) % 3;
        const float ex = __fsub_rn(g.qx[ib], g.qx[ia]), ey = __fsub_rn(g.qy[ib], g.qy[ia]);
        const float l2 = __fmaf_rn(ex, ex, __fmul_rn(ey, ey));
        g.inv_ell[k] = ts_rsqrt_approx(l2);
        g.ell[k] = __fmul_rn(l2, g.inv_ell[k]);
        g.nx[k] = __fmul_rn(__fmul_rn(g.sgn, ey), g.inv_ell[k]);
        g.ny[k] = -__fmul_rn(__fmul_rn(g.sgn, ex), g.inv_ell[k]);
        sum = __fadd_rn(sum, g.ell[k]);
    }
    g.sumell = sum;
    g.inv_sumell = ts_rcp_approx(sum);
    g.r = __fmul_rn(g.absS, g.inv_sumell);
    g.inv_r = __fmul_rn(sum, ts_rcp_approx(g.absS));
    // reference point: incentre = sum(ell_k q_k) / sum(ell) (ell_k is the edge opposite vertex k), float-rounded
    g.refx = __fmul_rn(__fmaf_rn(g.ell[0], g.qx[0], __fmaf_rn(g.ell[1], g.qx[1], __fmul_rn(g.ell[2], g.qx[2]))), g.inv_sumell);
    g.refy = __fmul_rn(__fmaf_rn(g.ell[0], g.qy[0], __fmaf_rn(g.ell[1], g.qy[1], __fmul_rn(g.ell[2], g.qy[2]))), g.inv_sumell);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const int ia = (k + 1) % 3;
        g.mx[k] = __fmul_rn(g.nx[k], g.inv_r);
        g.my[k] = __fmul_rn(g.ny[k], g.inv_r);
        const float dx = __fsub_rn(g.refx, g.qx[ia]), dy = __fsub_rn(g.refy, g.qy[ia]);
        g.c[k] = __fmul_rn(__fmaf_rn(g.nx[k], dx, __fmul_rn(g.ny[k], dy)), g.inv_r);
        g.rho[k] = __fmul_rn(g.ell[k], g.inv_sumell);
        g.kap[k] = -__fmul_rn(g.rho[k], g.w[k]);
    }
}

#define TS_NEEDLE_RATIO 400.0f        // perimeter / inradius above which a face is always evaluated on the compensated path

// F7 + the backward-only per-face terms -> the 10-float4 record.  s0..s2 = raw screen record, obar = mean vertex
// opacity, cam for (xn, yn).
__device__ __forceinline__ void ts_build_record(const float4 s0, const float4 s1, const float4 s2, float obar,
                                                const TsCamDev& cam, float4* __restrict__ out) {
    TsGeom g;
    ts_face_geom(s0, s1, s2, obar, g);
    // d r / d q_j = -rho_j n_j - (r / sum ell) (u_{j,j+1} + u_{j,j+2}),  u_{j,i} = (q_j - q_i)/|q_j - q_i|;
    // stored as drr_j = -(1/r) dr/dq_j so that gq_j += (x * gx) * drr_j  (B6 iii)
    float drrx[3], drry[3], tau[3], xn[3], yn[3];
    const float rs = g.r * g.inv_sumell;
    const float ifx = ts_rcp_approx(cam.fx), ify = ts_rcp_approx(cam.fy);
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int i1 = (j + 1) % 3, i2 = (j + 2) % 3;
        const float u1x = (g.qx[j] - g.qx[i1]) * g.inv_ell[i2], u1y = (g.qy[j] - g.qy[i1]) * g.inv_ell[i2];
        const float u2x = (g.qx[j] - g.qx[i2]) * g.inv_ell[i1], u2y = (g.qy[j] - g.qy[i2]) * g.inv_ell[i1];
        const float drx = -g.rho[j] * g.nx[j] - rs * (u1x + u2x), dry = -g.rho[j] * g.ny[j] - rs * (u1y + u2y);
        drrx[j] = -drx * g.inv_r, drry[j] = -dry * g.inv_r;
        // edge j runs from a = q_{j+1} to b = q_{j+2}; tau_j = ((q_j - a) . e) / |e|^2  (B6 ii)
        const float ex = g.qx[i2] - g.qx[i1], ey = g.qy[i2] - g.qy[i1];
        tau[j] = ((g.qx[j] - g.qx[i1]) * ex + (g.qy[j] - g.qy[i1]) * ey) * (g.inv_ell[j] * g.inv_ell[j]);
        xn[j] = (g.qx[j] - cam.cx) * ifx, yn[j] = (g.qy[j] - cam.cy) * ify;
    }
    // Needle faces (perimeter / inradius above TS_NEEDLE_RATIO; an equilateral triangle has 10.4): the affine form's
    // absolute error ~3e-7 * |p - ref| / r is no longer small next to the image tolerance anywhere inside the face, not
    // only next to an edge.  Their offsets c_k are stored as NaN: every evaluation then yields x = NaN, which
    // ts_eval_alpha sends down the compensated path (ts_refine_lhat) and ts_block_misses never culls.  m_k stay
    // exact (the backward reads them).  No cost for the other faces (N11).
    if (g.sumell * g.inv_r > TS_NEEDLE_RATIO) g.c[0] = g.c[1] = g.c[2] = __int_as_float(0x7fc00000);
    out[0] = make_float4(g.refx, g.refy, g.mx[0], g.my[0]);
    out[1] = make_float4(g.mx[1], g.my[1], g.mx[2], g.my[2]);
    out[2] = make_float4(g.c[0], g.c[1], g.c[2], g.obar);
    out[3] = make_float4(g.kap[0], g.kap[1], g.kap[2], s2.z);
    out[4] = make_float4(g.rho[0], g.rho[1], g.rho[2], s2.w);
    out[5] = make_float4(g.w[0], g.w[1], g.w[2], tau[0]);
    out[6] = make_float4(tau[1], tau[2], drrx[0], drry[0]);
    out[7] = make_float4(drrx[1], drry[1], drrx[2], drry[2]);
    out[8] = make_float4(xn[0], yn[0], xn[1], yn[1]);
    out[9] = make_float4(xn[2], yn[2], 0.0f, 0.0f);
}

// sigma dispatch: 0 = generic exp2(sigma log2 x), 1 = sigma 1, 2 = sigma 0.5, 3 = sigma 2
template <int SM>
__device__ __forceinline__ float ts_window_pow(float x, float sigma) {
    if (SM == 1) return x;
    if (SM == 2) return ts_sqrt_approx(x);
    if (SM == 3) return __fmul_rn(x, x);
    return __powf(x, sigma);
}
__host__ __device__ inline int ts_sigma_mode(float sigma) {
    return sigma == 1.0f ? 1 : (sigma == 0.5f ? 2 : (sigma == 2.0f ? 3 : 0));
}
// Per-face sigma (reading S32) runs through the generic instantiation (SM = 0), which takes the exponent of entry e from
// the staged copy of record row R3's last float instead of the launch parameter.
inline int ts_frame_sigma_mode(const ts_frame* fr) { return fr->face_sigma ? 0 : ts_sigma_mode(fr->prm.sigma); }

// Near an edge (|x| below this band) the fast affine form above loses RELATIVE accuracy in x (its absolute error is
// ~2e-7), and for sigma < 1 dI/dx = sigma x^(sigma-1) amplifies that beyond the gradient tolerance.  There -- for
// well under 1 % of the visited lanes -- x and lhat_k are recomputed from the raw screen vertices with the
// compensated 2x2 determinant (N6), which is accurate to a few ulp relative, like the oracle's.
#define TS_REFINE_BAND 1e-3f

// scr = the frame's raw screen records, slot = the face's slot: the record address is formed here, on the rare path
static __device__ __noinline__ float3 ts_refine_lhat(const float4* __restrict__ scr, uint32_t slot, float px, float py) {
    const float4* s4 = scr + TS_SCR_F4 * (size_t)slot;
    const float4 s0 = __ldg(s4), s1 = __ldg(s4 + 1);
    const float qx[3] = {s0.x, s0.w, s1.z}, qy[3] = {s0.y, s1.x, s1.w};
    const float a = __fsub_rn(qx[1], qx[0]), b = __fsub_rn(qy[2], qy[0]);
    const float c = __fsub_rn(qy[1], qy[0]), d = __fsub_rn(qx[2], qx[0]);
    const float S = __fmaf_rn(a, b, -__fmul_rn(c, d));
    const float sgn = S > 0.0f ? 1.0f : -1.0f;
    float ell[3], cr[3], sum = 0.0f;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const int ia = (k + 1) % 3, ib = (k + 2) % 3;
        const float ex = __fsub_rn(qx[ib], qx[ia]), ey = __fsub_rn(qy[ib], qy[ia]);
        const float dx = __fsub_rn(px, qx[ia]), dy = __fsub_rn(py, qy[ia]);
        ell[k] = __fsqrt_rn(__fmaf_rn(ex, ex, __fmul_rn(ey, ey)));
        sum = __fadd_rn(sum, ell[k]);
        const float w = __fmul_rn(ey, dx), e = __fmaf_rn(ey, dx, -w), g = __fmaf_rn(ex, dy, -w);
        cr[k] = __fsub_rn(g, e);                       // cross(e_k, p - q_{k+1}), compensated
    }
    const float inv_r = __fdiv_rn(sum, fabsf(S));
    float l[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) l[k] = __fmul_rn(__fdiv_rn(-__fmul_rn(sgn, cr[k]), ell[k]), inv_r);   // L_k / r
    return make_float3(l[0], l[1], l[2]);
}

// F8.1-3.  Returns true if the face contributes at (px,py); l[] = lhat_k, x, I, alpha are outputs.
// r0..r2 = record rows R0-R2; scr / slot locate the face's raw screen record (only read inside the refinement band).
template <int SM>
__device__ __forceinline__ bool ts_eval_alpha(const float4 r0, const float4 r1, const float4 r2, float px, float py,
                                              float sigma, float alpha_min, const float4* __restrict__ scr,
                                              uint32_t slot, float l[3],
                                              float& x, float& I, float& alpha) {
    const float dx = __fsub_rn(px, r0.x), dy = __fsub_rn(py, r0.y);
    l[0] = __fmaf_rn(r0.z, dx, __fmaf_rn(r0.w, dy, r2.x));
    l[1] = __fmaf_rn(r1.x, dx, __fmaf_rn(r1.y, dy, r2.y));
    l[2] = __fmaf_rn(r1.z, dx, __fmaf_rn(r1.w, dy, r2.z));
    x = -fmaxf(l[0], fmaxf(l[1], l[2]));
    if (!(fabsf(x) >= TS_REFINE_BAND)) {              // also taken when x is NaN (needle faces, see ts_build_record)
        const float3 lr = ts_refine_lhat(scr, slot, px, py);
        l[0] = lr.x, l[1] = lr.y, l[2] = lr.z;
        x = -fmaxf(l[0], fmaxf(l[1], l[2]));
    }
    if (!(x > 0.0f)) return false;
    I = ts_window_pow<SM>(x, sigma);
    alpha = __fmul_rn(r2.w, I);
    return alpha >= alpha_min;
}

// thread -> pixel mapping inside a 16x16 tile: warp w owns the 8x4 block at (8*(w&1), 4*(w>>1)), lane l the pixel
// (l & 7, l >> 3) of it; keeping a warp's pixels compact lets whole warps skip faces whose rect misses their block.
__device__ __forceinline__ void ts_thread_pixel(int tid, int& lx, int& ly) {
    const int w = tid >> 5, l = tid & 31;
    lx = ((w & 1) << 3) + (l & 7);
    ly = ((w >> 1) << 2) + (l >> 3);
}

// 32-bit lane mask of warp block `w`: bit l set iff lane l's pixel lies inside the tile-relative rect
// [rx0,rx1] x [ry0,ry1] (already clamped to 0..15).
__device__ __forceinline__ uint32_t ts_lane_mask(int w, int rx0, int ry0, int rx1, int ry1) {
    const int bx = (w & 1) << 3, by = (w >> 1) << 2;
    const int cx0 = max(rx0 - bx, 0), cx1 = min(rx1 - bx, 7);
    const int cy0 = max(ry0 - by, 0), cy1 = min(ry1 - by, 3);
    if (cx0 > cx1 || cy0 > cy1) return 0u;
    const uint32_t col = ((2u << cx1) - (1u << cx0)) & 0xffu;
    const uint32_t rows = (0xffffffffu >> (8 * (3 - cy1))) & (0xffffffffu << (8 * cy0));
    return (col * 0x01010101u) & rows;
}

// Exact block cull (run by the render kernels when they stage an entry of a block's list): the entry's rect
// overlaps the block with origin (bx, by), but does the TRIANGLE?  For each edge the normalised edge function is
// evaluated at the corner of (rect n block) where it is smallest; if that minimum is already above the refinement
// band, every pixel of the block has x < -band for this face: no hit, and no refinement either, so dropping the
// entry cannot change any result.  r0..r2 = record rows R0-R2; (rlo, rhi) = the entry's pixel rect.
__device__ __forceinline__ bool ts_block_misses(int bx, int by, int rlo, int rhi, const float4 r0, const float4 r1,
                                                const float4 r2) {
    const float x0 = (float)max((int)(short)(rlo & 0xffff), bx) - r0.x, x1 = (float)min((int)(short)(rhi & 0xffff), bx + 7) - r0.x;
    const float y0 = (float)max(rlo >> 16, by) - r0.y, y1 = (float)min(rhi >> 16, by + 3) - r0.y;
    const float l0 = fmaf(r0.z, r0.z > 0.f ? x0 : x1, fmaf(r0.w, r0.w > 0.f ? y0 : y1, r2.x));
    const float l1 = fmaf(r1.x, r1.x > 0.f ? x0 : x1, fmaf(r1.y, r1.y > 0.f ? y0 : y1, r2.y));
    const float l2 = fmaf(r1.z, r1.z > 0.f ? x0 : x1, fmaf(r1.w, r1.w > 0.f ? y0 : y1, r2.z));
    return fmaxf(l0, fmaxf(l1, l2)) > 4.0f * TS_REFINE_BAND;
}
