// ts_dssim.cu -- D-SSIM term of E_pho (Eq. 8; lambda = 0.2): harness helper next to
// ts_l1_loss_grad.  L_DSSIM = 1 - mean SSIM over 3 channels x H x W with the 11x11 Gaussian
// window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2 (reading S25).
//
// Two HBM-bound passes over the image, each a separable 11-tap convolution through shared memory on 32x32 tiles
// with a 5-pixel halo:
//   dssim_fwd_kernel : window sums of x, y, x^2, y^2, xy -> SSIM map (summed into the loss) and the three maps
//                      M0 = w (d_mu1 - 2 mu1 d_s11 - mu2 d_s12), M1 = w d_s11, M2 = w d_s12   (w = -lambda / 3HW)
//   dssim_bwd_kernel : gC <- (1 - lambda) gC + conv(M0) + 2 x conv(M1) + y conv(M2)
// (the window is symmetric, so the adjoint of the zero-padded convolution is the same convolution).
#include <cmath>

#include "ts_internal.cuh"

namespace {

constexpr int DT = 32, DR = 5, DIN = DT + 2 * DR;   // tile, window radius, tile + halo

struct Gauss11 { float g[11]; };

__global__ void __launch_bounds__(256)
dssim_fwd_kernel(int W, int H, const float* __restrict__ X, const float* __restrict__ Y, Gauss11 G, float wgt,
                 float lambda, float* __restrict__ M, float* __restrict__ loss) {
    __shared__ float sx[DIN][DIN + 1], sy[DIN][DIN + 1];
    __shared__ float hs[5][DIN][DT];
    __shared__ float s_red[8];
    const int tid = threadIdx.x, x0 = blockIdx.x * DT, y0 = blockIdx.y * DT;
    const size_t hw = (size_t)W * H;
    const float* Xc = X + blockIdx.z * hw;
    const float* Yc = Y + blockIdx.z * hw;
    for (int i = tid; i < DIN * DIN; i += 256) {
        const int r = i / DIN, c = i - r * DIN, gx = x0 + c - DR, gy = y0 + r - DR;
        const bool in = gx >= 0 && gx < W && gy >= 0 && gy < H;
        sx[r][c] = in ? __ldg(Xc + (size_t)gy * W + gx) : 0.0f;       // zero padding
        sy[r][c] = in ? __ldg(Yc + (size_t)gy * W + gx) : 0.0f;
    }
    __syncthreads();
    for (int i = tid; i < DIN * DT; i += 256) {                       // horizontal pass
        const int r = i / DT, c = i - r * DT;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f;
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            const float a = sx[r][c + k], b = sy[r][c + k], g = G.g[k];
            a0 = fmaf(g, a, a0), a1 = fmaf(g, b, a1), a2 = fmaf(g, a * a, a2), a3 = fmaf(g, b * b, a3), a4 = fmaf(g, a * b, a4);
        }
        hs[0][r][c] = a0, hs[1][r][c] = a1, hs[2][r][c] = a2, hs[3][r][c] = a3, hs[4][r][c] = a4;
    }
    __syncthreads();
    const float C1 = 0.01f * 0.01f, C2 = 0.03f * 0.03f;
    float acc = 0.0f;
    for (int i = tid; i < DT * DT; i += 256) {                        // vertical pass + SSIM
        const int r = i / DT, c = i - r * DT, gx = x0 + c, gy = y0 + r;
        if (gx >= W || gy >= H) continue;
        float mu1 = 0.f, mu2 = 0.f, e11 = 0.f, e22 = 0.f, e12 = 0.f;
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            const float g = G.g[k];
            mu1 = fmaf(g, hs[0][r + k][c], mu1), mu2 = fmaf(g, hs[1][r + k][c], mu2);
            e11 = fmaf(g, hs[2][r + k][c], e11), e22 = fmaf(g, hs[3][r + k][c], e22), e12 = fmaf(g, hs[4][r + k][c], e12);
        }
        const float s11 = e11 - mu1 * mu1, s22 = e22 - mu2 * mu2, s12 = e12 - mu1 * mu2;
        const float A1 = 2.f * mu1 * mu2 + C1, A2 = 2.f * s12 + C2, B1 = mu1 * mu1 + mu2 * mu2 + C1, B2 = s11 + s22 + C2;
        const float iB1 = 1.0f / B1, iB2 = 1.0f / B2;
        acc += A1 * A2 * iB1 * iB2;
        const float d_mu1_direct = 2.f * mu2 * A2 * iB1 * iB2 - A1 * A2 * 2.f * mu1 * iB1 * iB1 * iB2;
        const float d_s11 = -A1 * A2 * iB1 * iB2 * iB2;
        const float d_s12 = 2.f * A1 * iB1 * iB2;
        const size_t p = (size_t)gy * W + gx;
        float* Mc = M + 3 * blockIdx.z * hw;
        Mc[p] = wgt * (d_mu1_direct - 2.f * mu1 * d_s11 - mu2 * d_s12);
        Mc[hw + p] = wgt * d_s11;
        Mc[2 * hw + p] = wgt * d_s12;
    }
    if (loss) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
        if ((tid & 31) == 0) s_red[tid >> 5] = acc;
        __syncthreads();
        if (tid == 0) {
            float t = 0.f;
            for (int w = 0; w < 8; ++w) t += s_red[w];
            // lambda * L = lambda * (1 - sum / 3HW): the constant is added once, by block (0,0,0)
            float v = wgt * t;                                        // wgt = -lambda / 3HW
            if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) v += lambda;
            atomicAdd(loss, v);
        }
    }
}

__global__ void __launch_bounds__(256)
dssim_bwd_kernel(int W, int H, const float* __restrict__ X, const float* __restrict__ Y, Gauss11 G, float keep,
                 const float* __restrict__ M, float* __restrict__ gC) {
    __shared__ float sm[3][DIN][DIN + 1];
    __shared__ float hs[3][DIN][DT];
    const int tid = threadIdx.x, x0 = blockIdx.x * DT, y0 = blockIdx.y * DT;
    const size_t hw = (size_t)W * H;
    const float* Mc = M + 3 * blockIdx.z * hw;
    for (int i = tid; i < DIN * DIN; i += 256) {
        const int r = i / DIN, c = i - r * DIN, gx = x0 + c - DR, gy = y0 + r - DR;
        const bool in = gx >= 0 && gx < W && gy >= 0 && gy < H;
        const size_t p = (size_t)gy * W + gx;
#pragma unroll
        for (int q = 0; q < 3; ++q) sm[q][r][c] = in ? __ldg(Mc + q * hw + p) : 0.0f;
    }
    __syncthreads();
    for (int i = tid; i < DIN * DT; i += 256) {
        const int r = i / DT, c = i - r * DT;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            const float g = G.g[k];
            a0 = fmaf(g, sm[0][r][c + k], a0), a1 = fmaf(g, sm[1][r][c + k], a1), a2 = fmaf(g, sm[2][r][c + k], a2);
        }
        hs[0][r][c] = a0, hs[1][r][c] = a1, hs[2][r][c] = a2;
    }
    __syncthreads();
    for (int i = tid; i < DT * DT; i += 256) {
        const int r = i / DT, c = i - r * DT, gx = x0 + c, gy = y0 + r;
        if (gx >= W || gy >= H) continue;
        float c0 = 0.f, c1 = 0.f, c2 = 0.f;
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            const float g = G.g[k];
            c0 = fmaf(g, hs[0][r + k][c], c0), c1 = fmaf(g, hs[1][r + k][c], c1), c2 = fmaf(g, hs[2][r + k][c], c2);
        }
        const size_t p = blockIdx.z * hw + (size_t)gy * W + gx;
        gC[p] = keep * gC[p] + c0 + 2.0f * __ldg(X + p) * c1 + __ldg(Y + p) * c2;
    }
}

}  // namespace

extern "C" int32_t ts_dssim_loss_grad(ts_ctx* ctx, int32_t W, int32_t H, const float* C, const float* Chat, float lambda,
                                      float* gC, float* loss_dev, float* scratch, void* stream) {
    if (!ctx || W <= 0 || H <= 0 || !C || !Chat || !gC || !scratch || !(lambda >= 0.0f) || !(lambda <= 1.0f))
        return TS_ERR_INVALID_ARG;
    Gauss11 G;
    double g[11], sum = 0.0;
    for (int i = 0; i < 11; ++i) sum += (g[i] = exp(-(double)((i - 5) * (i - 5)) / (2.0 * 1.5 * 1.5)));
    for (int i = 0; i < 11; ++i) G.g[i] = (float)(g[i] / sum);
    const float wgt = (float)(-(double)lambda / (3.0 * (double)W * (double)H));
    const dim3 grid((W + DT - 1) / DT, (H + DT - 1) / DT, 3);
    dssim_fwd_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(W, H, C, Chat, G, wgt, lambda, scratch, loss_dev);
    dssim_bwd_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(W, H, C, Chat, G, 1.0f - lambda, scratch, gC);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
