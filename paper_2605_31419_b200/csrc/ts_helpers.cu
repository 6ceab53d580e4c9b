// ts_helpers.cu -- harness helpers a4 (L1 colour+depth loss gradient, Eq. 8-10 without D-SSIM) and a8 (on-device
// Adam step on tau followed by T <- Exp(-delta) o T).  Elementwise / tiny; they exist so that a whole tracking
// iteration stays on the device and can be captured into one CUDA graph.
#include "ts_pose.cuh"

namespace {

__global__ void __launch_bounds__(256)
l1_loss_grad_kernel(size_t n, const float* __restrict__ C, const float* __restrict__ D, const float* __restrict__ Ch,
                    const float* __restrict__ Dh, float wc, float wd, float* __restrict__ gC, float* __restrict__ gD,
                    float* __restrict__ loss) {
    float acc = 0.f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float d = C[c * n + i] - Ch[c * n + i];
            gC[c * n + i] = d > 0.f ? wc : (d < 0.f ? -wc : 0.f);
            acc += wc * fabsf(d);
        }
        const float dh = Dh[i];
        float g = 0.f;
        if (dh > 0.f) {
            const float d = D[i] - dh;
            g = d > 0.f ? wd : (d < 0.f ? -wd : 0.f);
            acc += wd * fabsf(d);
        }
        gD[i] = g;
    }
    if (loss) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
        __shared__ float s[8];
        if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            float t = 0.f;
            for (int w = 0; w < 8; ++w) t += s[w];
            atomicAdd(loss, t);
        }
    }
}

__global__ void pose_step_kernel(float* __restrict__ T, const float* __restrict__ g, float* __restrict__ state, TsLr6 lr,
                                 float beta1, float beta2, float eps) {
    ts_pose_step_warp(T, g, state, lr, beta1, beta2, eps);   // launched with exactly one warp
}

// E_equi (Eq. 14): per face, world space.  One thread per face; the loss is block-reduced into one
// atomic per CTA, the gradient goes to grad_pos with RED.ADD (a soup face owns its three vertices: no contention).
template <bool SOUP>
__global__ void __launch_bounds__(256)
equi_loss_grad_kernel(int M, const float* __restrict__ pos, const int32_t* __restrict__ faces, float gscale, float lscale,
                      float* __restrict__ grad_pos, float* __restrict__ loss) {
    float acc = 0.f;
    for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < M; m += gridDim.x * blockDim.x) {
        size_t id[3];
        float P[3][3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            id[k] = SOUP ? (size_t)3 * m + k : (size_t)__ldg(faces + 3 * (size_t)m + k);
#pragma unroll
            for (int a = 0; a < 3; ++a) P[k][a] = __ldg(pos + 3 * id[k] + a);
        }
        bool ok = true;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            float l2 = 0.f;
#pragma unroll
            for (int a = 0; a < 3; ++a) l2 += (P[(k + 1) % 3][a] - P[k][a]) * (P[(k + 1) % 3][a] - P[k][a]);
            ok = ok && l2 > 1e-24f;
        }
        if (!ok) continue;                                       // an edge of zero length: no angle
        float G[3][3] = {{0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}};
#pragma unroll
        for (int n = 0; n < 3; ++n) {
            const int b = (n + 1) % 3, c = (n + 2) % 3;
            float u[3], v[3], uu = 0.f, vv = 0.f, uv = 0.f;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                u[a] = P[b][a] - P[n][a], v[a] = P[c][a] - P[n][a];
                uu += u[a] * u[a], vv += v[a] * v[a], uv += u[a] * v[a];
            }
            const float ilu = rsqrtf(uu), ilv = rsqrtf(vv), iluv = ilu * ilv, cs = uv * iluv;
            acc += (cs - 0.5f) * (cs - 0.5f);
            const float gcs = gscale * 2.0f * (cs - 0.5f);        // dE/dcos
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float du = v[a] * iluv - cs * u[a] * ilu * ilu, dv = u[a] * iluv - cs * v[a] * ilv * ilv;
                G[b][a] += gcs * du, G[c][a] += gcs * dv, G[n][a] -= gcs * (du + dv);
            }
        }
        if (grad_pos) {
#pragma unroll
            for (int k = 0; k < 3; ++k)
#pragma unroll
                for (int a = 0; a < 3; ++a) atomicAdd(grad_pos + 3 * id[k] + a, G[k][a]);
        }
    }
    if (loss) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
        __shared__ float s[8];
        if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            float t = 0.f;
            for (int w = 0; w < 8; ++w) t += s[w];
            atomicAdd(loss, lscale * t);
        }
    }
}

// E_norm (Eq. 12): w sum over valid pixels (Nbar != 0) of 1 - N . Nbar; gN = -w Nbar there, 0 elsewhere.
__global__ void __launch_bounds__(256)
normal_loss_grad_kernel(size_t n, const float* __restrict__ N, const float* __restrict__ Nb, float w, float* __restrict__ gN,
                        float* __restrict__ loss) {
    float acc = 0.f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float b0 = Nb[i], b1 = Nb[n + i], b2 = Nb[2 * n + i];
        const bool valid = b0 != 0.f || b1 != 0.f || b2 != 0.f;
        if (valid) acc += w * (1.0f - (N[i] * b0 + N[n + i] * b1 + N[2 * n + i] * b2));
        gN[i] = valid ? -w * b0 : 0.f, gN[n + i] = valid ? -w * b1 : 0.f, gN[2 * n + i] = valid ? -w * b2 : 0.f;
    }
    if (loss) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
        __shared__ float s[8];
        if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            float t = 0.f;
            for (int k = 0; k < 8; ++k) t += s[k];
            atomicAdd(loss, t);
        }
    }
}

}  // namespace

extern "C" int32_t ts_normal_loss_grad(ts_ctx* ctx, int32_t W, int32_t H, const float* N, const float* Nbar, float weight,
                                       float* gN, float* loss_dev, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || W <= 0 || H <= 0 || !N || !Nbar || !gN) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    const size_t n = (size_t)W * H;
    const int grid = (int)((n + 255) / 256 < (size_t)ctx->num_sms * 8 ? (n + 255) / 256 : (size_t)ctx->num_sms * 8);
    normal_loss_grad_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(n, N, Nbar, (float)((double)weight / (double)n), gN, loss_dev);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

extern "C" int32_t ts_equi_loss_grad(ts_ctx* ctx, const ts_scene* sc, float weight, float* grad_pos, float* loss_dev,
                                     void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !sc->pos || sc->M <= 0 || (!grad_pos && !loss_dev)) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->faces == nullptr && sc->V != 3 * sc->M) return TS_ERR_INVALID_ARG;
    const float scale = (float)((double)weight / (3.0 * (double)sc->M));
    const int grid = (int)(((size_t)sc->M + 255) / 256 < (size_t)ctx->num_sms * 8 ? ((size_t)sc->M + 255) / 256 : (size_t)ctx->num_sms * 8);
    if (sc->faces == nullptr)
        equi_loss_grad_kernel<true><<<grid, 256, 0, (cudaStream_t)stream>>>(sc->M, sc->pos, nullptr, scale, scale, grad_pos, loss_dev);
    else
        equi_loss_grad_kernel<false><<<grid, 256, 0, (cudaStream_t)stream>>>(sc->M, sc->pos, sc->faces, scale, scale, grad_pos, loss_dev);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

extern "C" int32_t ts_l1_loss_grad(ts_ctx* ctx, int32_t W, int32_t H, const float* C, const float* D, const float* Chat,
                                   const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss_dev,
                                   void* stream) {
    TS_TRACE(ctx);
    if (!ctx || W <= 0 || H <= 0 || !C || !D || !Chat || !Dhat || !gC || !gD) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    const size_t n = (size_t)W * H;
    const float wc = (float)(1.0 / (3.0 * (double)n)), wd = (float)((double)lambda_dep / (double)n);
    const int grid = (int)((n + 255) / 256 < (size_t)ctx->num_sms * 8 ? (n + 255) / 256 : (size_t)ctx->num_sms * 8);
    l1_loss_grad_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(n, C, D, Chat, Dhat, wc, wd, gC, gD, loss_dev);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

extern "C" int32_t ts_pose_step(ts_ctx* ctx, float* T_cw_dev, const float* dL_dtau_dev, float* state_dev,
                                const float* lr6, float beta1, float beta2, float eps, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !T_cw_dev || !dL_dtau_dev || !state_dev || !lr6) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    TsLr6 lr;
    for (int i = 0; i < 6; ++i) lr.v[i] = lr6[i];
    pose_step_kernel<<<1, 32, 0, (cudaStream_t)stream>>>(T_cw_dev, dL_dtau_dev, state_dev, lr, beta1, beta2, eps);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

// Normalised depth D / A (E_dep of Eq. 9 / 13 compares a rendered depth with the sensor depth, and
// D = sum z alpha T under-reads wherever A < 1): elementwise, HBM-bound.
namespace {
__global__ void __launch_bounds__(256) depth_normalise_kernel(size_t n, const float* __restrict__ D, const float* __restrict__ A,
                                                              float eps, float* __restrict__ Dn) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = A[i];
        Dn[i] = a > eps ? __fdiv_rn(D[i], a) : 0.0f;
    }
}
__global__ void __launch_bounds__(256) depth_normalise_bwd_kernel(size_t n, const float* __restrict__ D, const float* __restrict__ A,
                                                                  float eps, const float* __restrict__ gDn, float* __restrict__ gD,
                                                                  float* __restrict__ gA) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = A[i];
        if (!(a > eps)) continue;
        const float g = gDn[i], ia = __fdiv_rn(1.0f, a);
        gD[i] += g * ia;
        gA[i] += -g * D[i] * ia * ia;
    }
}
}  // namespace

extern "C" int32_t ts_depth_normalise(ts_ctx* ctx, int32_t W, int32_t H, const float* D, const float* A, float eps, float* Dn,
                                      void* stream) {
    TS_TRACE(ctx);
    if (!ctx || W <= 0 || H <= 0 || !D || !A || !Dn || !(eps >= 0.0f)) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    const size_t n = (size_t)W * H;
    const int grid = (int)((n + 255) / 256 < (size_t)ctx->num_sms * 8 ? (n + 255) / 256 : (size_t)ctx->num_sms * 8);
    depth_normalise_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(n, D, A, eps, Dn);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

extern "C" int32_t ts_depth_normalise_bwd(ts_ctx* ctx, int32_t W, int32_t H, const float* D, const float* A, float eps,
                                          const float* gDn, float* gD, float* gA, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || W <= 0 || H <= 0 || !D || !A || !gDn || !gD || !gA || !(eps >= 0.0f)) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    const size_t n = (size_t)W * H;
    const int grid = (int)((n + 255) / 256 < (size_t)ctx->num_sms * 8 ? (n + 255) / 256 : (size_t)ctx->num_sms * 8);
    depth_normalise_bwd_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(n, D, A, eps, gDn, gD, gA);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

// Measurement helper ("measure a dependent-free FMA loop and print both nominal and measured
// peaks"): every thread runs `iters` rounds of eight independent FMA chains; 16 flops per thread and round.
namespace {
__global__ void __launch_bounds__(1024) fp32_probe_kernel(int iters, float a, float b, float* __restrict__ out) {
    float x0 = threadIdx.x * 1e-3f, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
#pragma unroll 4
    for (int i = 0; i < iters; ++i) {
        x0 = fmaf(x0, a, b), x1 = fmaf(x1, a, b), x2 = fmaf(x2, a, b), x3 = fmaf(x3, a, b);
        x4 = fmaf(x4, a, b), x5 = fmaf(x5, a, b), x6 = fmaf(x6, a, b), x7 = fmaf(x7, a, b);
    }
    const float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456f) out[0] = s;                       // never true: keeps the chains alive
}
}  // namespace

extern "C" int32_t ts_fp32_probe(ts_ctx* ctx, int32_t iters, float* scratch_dev, uint64_t* flops_out, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || iters <= 0 || !scratch_dev || !flops_out) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    const int grid = ctx->num_sms * 2;
    fp32_probe_kernel<<<grid, 1024, 0, (cudaStream_t)stream>>>(iters, 0.999f, 1e-3f, scratch_dev);
    *flops_out = (uint64_t)grid * 1024ull * 16ull * (uint64_t)iters;
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

// TS_VIEW_N_CONTRIB: the renderers count a pixel's last contributing entry in its BLOCK's list (ts_jobs.cuh); the
// view gives it as 1 + the entry's position in the TILE's sorted list, the oracle's n_contrib.
namespace {
__global__ void __launch_bounds__(256) ncontrib_view_kernel(TsFrameDev f) {
    const uint32_t j = (blockIdx.x * 256u + threadIdx.x) >> 5, lane = threadIdx.x & 31u;
    if (j >= (uint32_t)f.NT * 8u) return;
    const uint4 h = f.job_order[j];
    const int blk = (int)(h.x >> 28);
    const int px = (int)(h.w & 0xffffu) + ((blk & 1) << 3) + (int)(lane & 7u), py = (int)(h.w >> 16) + ((blk >> 1) << 2) + (int)(lane >> 3);
    if (px >= f.W || py >= f.H) return;
    const size_t p = (size_t)py * f.W + px;
    const uint32_t nb = h.z > h.y ? f.n_contrib[p] : 0u;
    uint32_t pos = 0;
    if (nb && nb <= h.z - h.y) {                     // (a count beyond the job's list cannot come from this sort: reads as "none")
        // (a debug accessor: a linear search of the tile's list for the entry's slot, which is unique in it)
        const uint32_t slot = f.blist[h.y + nb - 1u].x;
        const uint2 tr = f.tile_ranges[h.x & 0x0fffffffu];
        for (uint32_t i = tr.x; i < tr.y; ++i)
            if (f.sorted[i].x == slot) { pos = i - tr.x + 1u; break; }
    }
    f.n_contrib_view[p] = pos;
}
}  // namespace

int32_t ts_launch_ncontrib_view(const ts_ctx*, ts_frame* fr, cudaStream_t st) {
    const uint32_t threads = (uint32_t)fr->d.NT * 8u * 32u;
    ncontrib_view_kernel<<<(threads + 255u) / 256u, 256, 0, st>>>(fr->d);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}

// Sensor frame -> targets of Eq. 8-9 (reading S33): 5 bytes read, 16 written per pixel; HBM-bound.  One thread
// per four consecutive pixels (three 32-bit loads of colour and one 64-bit load of depth when the pointers allow it,
// byte loads otherwise); the four results of a plane go out as one float4 store when the planes are 16-byte aligned
// and the pixel count is a multiple of four (ST4), as scalar stores otherwise.
namespace {
template <bool VEC>
__global__ void __launch_bounds__(256) unpack_rgbd_kernel(size_t n, const uint8_t* __restrict__ rgb, const uint16_t* __restrict__ dep,
                                                          float depth_scale, float* __restrict__ Chat, float* __restrict__ Dhat, bool ST4) {
    const size_t n4 = (n + 3) / 4;
    for (size_t q = blockIdx.x * (size_t)blockDim.x + threadIdx.x; q < n4; q += (size_t)gridDim.x * blockDim.x) {
        const size_t p0 = 4 * q;
        uint32_t c[12], d[4];
        if (VEC && p0 + 4 <= n) {
            if (rgb) {
                const uint32_t* r32 = reinterpret_cast<const uint32_t*>(rgb + 3 * p0);
                const uint32_t w0 = __ldg(r32), w1 = __ldg(r32 + 1), w2 = __ldg(r32 + 2);
#pragma unroll
                for (int i = 0; i < 4; ++i) c[i] = (w0 >> (8 * i)) & 0xffu, c[4 + i] = (w1 >> (8 * i)) & 0xffu, c[8 + i] = (w2 >> (8 * i)) & 0xffu;
            }
            if (dep) {
                const uint2 w = __ldg(reinterpret_cast<const uint2*>(dep + p0));
                d[0] = w.x & 0xffffu, d[1] = w.x >> 16, d[2] = w.y & 0xffffu, d[3] = w.y >> 16;
            }
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const bool in = p0 + i < n;
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) c[3 * i + ch] = (rgb && in) ? rgb[3 * (p0 + i) + ch] : 0u;
                d[i] = (dep && in) ? dep[p0 + i] : 0u;
            }
        }
        if (ST4) {                                           // (n % 4 == 0: every thread owns four whole pixels)
            if (rgb) {
#pragma unroll
                for (int ch = 0; ch < 3; ++ch)
                    *reinterpret_cast<float4*>(Chat + ch * n + p0) =
                        make_float4(__fdiv_rn((float)c[ch], 255.0f), __fdiv_rn((float)c[3 + ch], 255.0f),
                                    __fdiv_rn((float)c[6 + ch], 255.0f), __fdiv_rn((float)c[9 + ch], 255.0f));
            }
            if (dep)
                *reinterpret_cast<float4*>(Dhat + p0) = make_float4(__fdiv_rn((float)d[0], depth_scale), __fdiv_rn((float)d[1], depth_scale),
                                                                    __fdiv_rn((float)d[2], depth_scale), __fdiv_rn((float)d[3], depth_scale));
            continue;
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if (p0 + i >= n) break;
            if (rgb) {
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) Chat[ch * n + p0 + i] = __fdiv_rn((float)c[3 * i + ch], 255.0f);
            }
            if (dep) Dhat[p0 + i] = __fdiv_rn((float)d[i], depth_scale);
        }
    }
}
}  // namespace

extern "C" int32_t ts_unpack_rgbd(ts_ctx* ctx, int32_t W, int32_t H, const uint8_t* rgb_dev, const uint16_t* depth_dev,
                                  float depth_scale, float* Chat, float* Dhat, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || W <= 0 || H <= 0 || (!rgb_dev && !depth_dev) || (rgb_dev && !Chat) || (depth_dev && (!Dhat || !(depth_scale > 0.0f))))
        return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    const size_t n = (size_t)W * H, n4 = (n + 3) / 4;
    const int grid = (int)((n4 + 255) / 256 < (size_t)ctx->num_sms * 8 ? (n4 + 255) / 256 : (size_t)ctx->num_sms * 8);
    const bool vec = (reinterpret_cast<uintptr_t>(rgb_dev) & 3u) == 0 && (reinterpret_cast<uintptr_t>(depth_dev) & 7u) == 0;
    const bool st4 = (n & 3u) == 0 && (reinterpret_cast<uintptr_t>(Chat) & 15u) == 0 && (reinterpret_cast<uintptr_t>(Dhat) & 15u) == 0;
    if (vec) unpack_rgbd_kernel<true><<<grid, 256, 0, (cudaStream_t)stream>>>(n, rgb_dev, depth_dev, depth_scale, Chat, Dhat, st4);
    else unpack_rgbd_kernel<false><<<grid, 256, 0, (cudaStream_t)stream>>>(n, rgb_dev, depth_dev, depth_scale, Chat, Dhat, st4);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
