// ts_dssim.cu -- D-SSIM term of E_pho (Eq. 8; lambda = 0.2): harness helper next to
// ts_l1_loss_grad.  L_DSSIM = 1 - mean SSIM over 3 channels x H x W with the 11x11 Gaussian
// window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2 (reading S25).
//
// ONE launch, no scratch image: a CTA owns a 32x32 tile of one channel and does BOTH separable 11-tap convolutions in
// shared memory.  The gradient at a pixel needs the maps M0..M2 on its 11x11 neighbourhood, and every M needs the
// window sums of x, y, x^2, y^2, xy on ITS neighbourhood, so the CTA reads the images on the tile + a 10-pixel apron
// (52 x 52), forms the window sums and
//     M0 = w (d_mu1 - 2 mu1 d_s11 - mu2 d_s12),  M1 = w d_s11,  M2 = w d_s12        (w = -lambda / 3HW)
// on the tile + a 5-pixel apron (42 x 42; zero outside the image, like the zero padding of the forward window), then
//     gC <- (1 - lambda) gC + conv(M0) + 2 x conv(M1) + y conv(M2)
// on the tile (the window is symmetric, so the adjoint of the zero-padded convolution is the same convolution).  The
// apron costs 2.6x the reads of the tile (all L2 hits: the forward pass has just written C) and 1.7x the window sums;
// it saves the 9 HW floats of the two-pass form and a launch.  SSIM itself is summed into the loss on the tile only.
#include <cmath>

#include "ts_internal.cuh"

namespace {

constexpr int DT = 32, DR = 5;
constexpr int DN = 384;              // threads per CTA: every pass but the last fits one round of tasks (364, 294, 336, 256)
constexpr int DB = DT + 2 * DR;      // 42: tile + apron of the M maps
constexpr int DA = DT + 4 * DR;      // 52: tile + apron of the images

struct Gauss11 { float g[11]; };

struct DssimSmem {
    union {
        struct { float sx[DA][DA + 1], sy[DA][DA + 1]; } in;    // images (steps 1-2)
        float m[3][DB][DB + 1];                                  // M maps (steps 3-4)
    } a;
    union {
        float hs[5][DA][DB + 1];                                 // row sums of x, y, x^2, y^2, xy (steps 2-3); odd row pitch:
        float hm[3][DB][DT + 1];                                 // row sums of the M maps (steps 4-5)    lanes that differ in the row hit different banks
    } b;
    float red[DN / 32];
};

__global__ void __launch_bounds__(DN, 3)
dssim_fused_kernel(int W, int H, const float* __restrict__ X, const float* __restrict__ Y, Gauss11 G, float wgt,
                   float lambda, float keep, float* __restrict__ gC, float* __restrict__ loss, int vec2) {
    extern __shared__ __align__(16) unsigned char dssim_raw[];
    DssimSmem& S = *reinterpret_cast<DssimSmem*>(dssim_raw);
    const int tid = threadIdx.x, x0 = blockIdx.x * DT, y0 = blockIdx.y * DT;
    const size_t hw = (size_t)W * H;
    const float* Xc = X + blockIdx.z * hw;
    const float* Yc = Y + blockIdx.z * hw;
    // 1. images on the tile + 10-pixel apron, zero padded; two pixels per load where the row pitch allows it (the
    //    apron starts at an even column: x0 - 10)
    if (vec2) {                                              // (W even, images 8-byte aligned)
        // all of a thread's loads are issued before its first store (one round trip, not one per iteration)
        constexpr int N1 = (DA * (DA / 2) + DN - 1) / DN;
        float2 vx[N1], vy[N1];
#pragma unroll
        for (int it = 0; it < N1; ++it) {
            const int i = tid + it * DN;
            const int r = i / (DA / 2), c = 2 * (i - r * (DA / 2)), gx = x0 + c - 2 * DR, gy = y0 + r - 2 * DR;
            vx[it] = make_float2(0.f, 0.f), vy[it] = make_float2(0.f, 0.f);
            if (i < DA * (DA / 2) && gx >= 0 && gx + 1 < W && gy >= 0 && gy < H) {   // (gx and W are even: both pixels in or both out)
                vx[it] = __ldg(reinterpret_cast<const float2*>(Xc + (size_t)gy * W + gx));
                vy[it] = __ldg(reinterpret_cast<const float2*>(Yc + (size_t)gy * W + gx));
            }
        }
#pragma unroll
        for (int it = 0; it < N1; ++it) {
            const int i = tid + it * DN;
            if (i >= DA * (DA / 2)) break;
            const int r = i / (DA / 2), c = 2 * (i - r * (DA / 2));
            S.a.in.sx[r][c] = vx[it].x, S.a.in.sx[r][c + 1] = vx[it].y;
            S.a.in.sy[r][c] = vy[it].x, S.a.in.sy[r][c + 1] = vy[it].y;
        }
    } else {
        for (int i = tid; i < DA * DA; i += DN) {
            const int r = i / DA, c = i - r * DA, gx = x0 + c - 2 * DR, gy = y0 + r - 2 * DR;
            const bool in = gx >= 0 && gx < W && gy >= 0 && gy < H;
            S.a.in.sx[r][c] = in ? __ldg(Xc + (size_t)gy * W + gx) : 0.0f;
            S.a.in.sy[r][c] = in ? __ldg(Yc + (size_t)gy * W + gx) : 0.0f;
        }
    }
    __syncthreads();
    // Every pass is register-blocked: a thread produces a run of 6 (or 4) consecutive outputs ALONG the convolution,
    // so the 16 (14) inputs it needs are read from shared memory once instead of 11 times per output; tasks are dealt
    // so that the lanes of a warp differ in the OTHER coordinate (rows: stride 53 / 43 words, columns: stride 1), which
    // keeps the reads free of bank conflicts.
    // 2. horizontal pass: 52 rows x 42 columns (7 runs of 6)
    for (int i = tid; i < DA * (DB / 6); i += DN) {
        const int r = i % DA, c0 = (i / DA) * 6;
        float vx[16], vy[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) vx[k] = S.a.in.sx[r][c0 + k], vy[k] = S.a.in.sy[r][c0 + k];
        float vxx[16], vyy[16], vxy[16];                        // the products once per input, not once per tap
#pragma unroll
        for (int k = 0; k < 16; ++k) vxx[k] = vx[k] * vx[k], vyy[k] = vy[k] * vy[k], vxy[k] = vx[k] * vy[k];
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f;
#pragma unroll
            for (int k = 0; k < 11; ++k) {
                const float g = G.g[k];
                a0 = fmaf(g, vx[j + k], a0), a1 = fmaf(g, vy[j + k], a1), a2 = fmaf(g, vxx[j + k], a2), a3 = fmaf(g, vyy[j + k], a3),
                a4 = fmaf(g, vxy[j + k], a4);
            }
            S.b.hs[0][r][c0 + j] = a0, S.b.hs[1][r][c0 + j] = a1, S.b.hs[2][r][c0 + j] = a2, S.b.hs[3][r][c0 + j] = a3,
            S.b.hs[4][r][c0 + j] = a4;
        }
    }
    __syncthreads();
    // 3. vertical pass + SSIM + the three maps on 42 x 42 (7 runs of 6 rows; the images in S.a are dead from here on)
    const float C1 = 0.01f * 0.01f, C2 = 0.03f * 0.03f;
    float acc = 0.0f;
    for (int i = tid; i < DB * (DB / 6); i += DN) {
        const int c = i % DB, r0 = (i / DB) * 6, gx = x0 + c - DR;
        float st[5][6];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
            float v[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) v[k] = S.b.hs[q][r0 + k][c];
#pragma unroll
            for (int j = 0; j < 6; ++j) {
                float a = 0.f;
#pragma unroll
                for (int k = 0; k < 11; ++k) a = fmaf(G.g[k], v[j + k], a);
                st[q][j] = a;
            }
        }
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            const int r = r0 + j, gy = y0 + r - DR;
            float m0 = 0.f, m1 = 0.f, m2 = 0.f;
            if (gx >= 0 && gx < W && gy >= 0 && gy < H) {
                const float mu1 = st[0][j], mu2 = st[1][j], e11 = st[2][j], e22 = st[3][j], e12 = st[4][j];
                const float s11 = e11 - mu1 * mu1, s22 = e22 - mu2 * mu2, s12 = e12 - mu1 * mu2;
                const float A1 = 2.f * mu1 * mu2 + C1, A2 = 2.f * s12 + C2, B1 = mu1 * mu1 + mu2 * mu2 + C1, B2 = s11 + s22 + C2;
                const float iB1 = __fdividef(1.0f, B1), iB2 = __fdividef(1.0f, B2);     // (B1 >= C1, B2 >= C2: MUFU.RCP is enough)
                if (r >= DR && r < DR + DT && c >= DR && c < DR + DT) acc += A1 * A2 * iB1 * iB2;   // the tile's own pixels
                const float d_mu1_direct = 2.f * mu2 * A2 * iB1 * iB2 - A1 * A2 * 2.f * mu1 * iB1 * iB1 * iB2;
                const float d_s11 = -A1 * A2 * iB1 * iB2 * iB2;
                const float d_s12 = 2.f * A1 * iB1 * iB2;
                m0 = wgt * (d_mu1_direct - 2.f * mu1 * d_s11 - mu2 * d_s12), m1 = wgt * d_s11, m2 = wgt * d_s12;
            }
            // (S.a.m aliases the images, which step 2 has finished reading: the barrier after step 2 covers it)
            S.a.m[0][r][c] = m0, S.a.m[1][r][c] = m1, S.a.m[2][r][c] = m2;
        }
    }
    __syncthreads();
    // 4. horizontal pass of the maps: 42 rows x 32 columns, 8 runs of 4 (S.b.hs is dead: every thread passed the barrier)
    for (int i = tid; i < DB * (DT / 4); i += DN) {
        const int r = i % DB, c0 = (i / DB) * 4;
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            float v[14];
#pragma unroll
            for (int k = 0; k < 14; ++k) v[k] = S.a.m[q][r][c0 + k];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float a = 0.f;
#pragma unroll
                for (int k = 0; k < 11; ++k) a = fmaf(G.g[k], v[j + k], a);
                S.b.hm[q][r][c0 + j] = a;
            }
        }
    }
    __syncthreads();
    // 5. vertical pass + the cotangent of E_pho on the tile (8 runs of 4 rows)
    for (int i = tid; i < DT * (DT / 4); i += DN) {
        const int c = i % DT, r0 = (i / DT) * 4, gx = x0 + c;
        // the pixel's cotangent and images are requested first: they arrive under the convolution
        float g0[4], xv[4], yv[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int gy = y0 + r0 + j;
            g0[j] = xv[j] = yv[j] = 0.f;
            if (gx < W && gy < H) {
                const size_t p = blockIdx.z * hw + (size_t)gy * W + gx;
                g0[j] = gC[p], xv[j] = __ldg(X + p), yv[j] = __ldg(Y + p);
            }
        }
        float cc[3][4];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            float v[14];
#pragma unroll
            for (int k = 0; k < 14; ++k) v[k] = S.b.hm[q][r0 + k][c];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float a = 0.f;
#pragma unroll
                for (int k = 0; k < 11; ++k) a = fmaf(G.g[k], v[j + k], a);
                cc[q][j] = a;
            }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int gy = y0 + r0 + j;
            if (gx >= W || gy >= H) continue;
            const size_t p = blockIdx.z * hw + (size_t)gy * W + gx;
            gC[p] = keep * g0[j] + cc[0][j] + 2.0f * xv[j] * cc[1][j] + yv[j] * cc[2][j];
        }
    }
    if (loss) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
        if ((tid & 31) == 0) S.red[tid >> 5] = acc;
        __syncthreads();
        if (tid == 0) {
            float t = 0.f;
            for (int w = 0; w < DN / 32; ++w) t += S.red[w];
            // lambda * L = lambda * (1 - sum / 3HW): the constant is added once, by block (0,0,0)
            float v = wgt * t;                                        // wgt = -lambda / 3HW
            if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) v += lambda;
            atomicAdd(loss, v);
        }
    }
}

}  // namespace

extern "C" int32_t ts_dssim_loss_grad(ts_ctx* ctx, int32_t W, int32_t H, const float* C, const float* Chat, float lambda,
                                      float* gC, float* loss_dev, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || W <= 0 || H <= 0 || !C || !Chat || !gC || !(lambda >= 0.0f) || !(lambda <= 1.0f))
        return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    Gauss11 G;
    double g[11], sum = 0.0;
    for (int i = 0; i < 11; ++i) sum += (g[i] = exp(-(double)((i - 5) * (i - 5)) / (2.0 * 1.5 * 1.5)));
    for (int i = 0; i < 11; ++i) G.g[i] = (float)(g[i] / sum);
    const float wgt = (float)(-(double)lambda / (3.0 * (double)W * (double)H));
    const dim3 grid((W + DT - 1) / DT, (H + DT - 1) / DT, 3);
    cudaFuncSetAttribute(dssim_fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(DssimSmem));   // per device
    const int vec2 = (W & 1) == 0 && ((reinterpret_cast<uintptr_t>(C) | reinterpret_cast<uintptr_t>(Chat)) & 7u) == 0;
    dssim_fused_kernel<<<grid, DN, sizeof(DssimSmem), (cudaStream_t)stream>>>(W, H, C, Chat, G, wgt, lambda, 1.0f - lambda, gC,
                                                                               loss_dev, vec2);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
