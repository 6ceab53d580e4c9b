// ts_pose.cuh -- a8: one Adam step on tau followed by T <- Exp(-delta) o T (left perturbation, Eq. 6-7,
// PAPER.md:111-117; learning rates PAPER.md:440-441).  Single-thread device routine shared by ts_pose_step and by
// the fused tail of the pose reduction.
#pragma once
#include "ts_internal.cuh"

struct TsLr6 { float v[6]; };

// state[13] = m[6], v[6], step count.  Called by ONE FULL WARP (all 32 lanes converged): lanes 0-5 take the Adam
// update of one component each, every lane then forms Exp(delta) redundantly and lanes 0-11 write one entry of the
// new pose each -- a single thread would spend ~5 us on this chain of dependent powf / sinf / divisions.
__device__ __forceinline__ void ts_pose_step_warp(float* __restrict__ T, const float* __restrict__ g, float* __restrict__ state,
                                                  const TsLr6& lr, float beta1, float beta2, float eps) {
    const int lane = threadIdx.x & 31;
    const float t = state[12] + 1.0f;
    float di = 0.0f;
    if (lane < 6) {
        const float c1 = 1.0f - powf(beta1, t), c2 = 1.0f - powf(beta2, t);
        const float gi = g[lane];
        const float m = beta1 * state[lane] + (1.0f - beta1) * gi;
        const float v = beta2 * state[6 + lane] + (1.0f - beta2) * gi * gi;
        float lri = lr.v[0];
#pragma unroll
        for (int i = 1; i < 6; ++i) lri = (lane == i) ? lr.v[i] : lri;
        di = -lri * (m / c1) / (sqrtf(v / c2) + eps);
        state[lane] = m, state[6 + lane] = v;
    }
    // every lane also reads the pose entries it will need before anybody overwrites them
    const int oi = (lane < 12 ? lane : 0) >> 2, oj = (lane < 12 ? lane : 0) & 3;
    const float T0 = T[oj], T1 = T[4 + oj], T2 = T[8 + oj];
    __syncwarp();
    if (lane == 0) state[12] = t;
    float d[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) d[i] = __shfl_sync(0xffffffffu, di, i);
    // Exp(d): rotation by Rodrigues, translation V(theta) rho
    const float wx = d[3], wy = d[4], wz = d[5];
    const float th2 = wx * wx + wy * wy + wz * wz, th = sqrtf(th2);
    float A, B, Cc;
    if (th < 1e-4f) {
        A = 1.0f - th2 / 6.0f, B = 0.5f - th2 / 24.0f, Cc = 1.0f / 6.0f - th2 / 120.0f;
    } else {
        A = sinf(th) / th, B = (1.0f - cosf(th)) / th2, Cc = (th - sinf(th)) / (th2 * th);
    }
    const float K[9] = {0.f, -wz, wy, wz, 0.f, -wx, -wy, wx, 0.f};
    float K2[9], R[9], V[9];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) K2[3 * i + j] = K[3 * i] * K[j] + K[3 * i + 1] * K[3 + j] + K[3 * i + 2] * K[6 + j];
#pragma unroll
    for (int i = 0; i < 9; ++i) {
        const float I = (i % 4 == 0) ? 1.0f : 0.0f;
        R[i] = I + A * K[i] + B * K2[i];
        V[i] = I + B * K[i] + Cc * K2[i];
    }
    const float tt[3] = {V[0] * d[0] + V[1] * d[1] + V[2] * d[2], V[3] * d[0] + V[4] * d[1] + V[5] * d[2],
                         V[6] * d[0] + V[7] * d[1] + V[8] * d[2]};
    const float r0 = oi == 0 ? R[0] : (oi == 1 ? R[3] : R[6]), r1 = oi == 0 ? R[1] : (oi == 1 ? R[4] : R[7]);
    const float r2 = oi == 0 ? R[2] : (oi == 1 ? R[5] : R[8]), tv = oi == 0 ? tt[0] : (oi == 1 ? tt[1] : tt[2]);
    const float o = r0 * T0 + r1 * T1 + r2 * T2 + (oj == 3 ? tv : 0.0f);
    if (lane < 12) T[lane] = o;
}
