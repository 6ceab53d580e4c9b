// ts_pose.cuh -- a8: one Adam step on tau followed by T <- Exp(-delta) o T (left perturbation, Eq. 6-7,
// PAPER.md:111-117; learning rates PAPER.md:440-441).  Single-thread device routine shared by ts_pose_step and by
// the fused tail of the pose reduction.
#pragma once
#include "ts_internal.cuh"

struct TsLr6 { float v[6]; };

// state[13] = m[6], v[6], step count
__device__ __forceinline__ void ts_pose_step_dev(float* __restrict__ T, const float* __restrict__ g, float* __restrict__ state,
                                                 const TsLr6& lr, float beta1, float beta2, float eps) {
    float* m = state;
    float* v = state + 6;
    const float t = state[12] + 1.0f;
    state[12] = t;
    const float c1 = 1.0f - powf(beta1, t), c2 = 1.0f - powf(beta2, t);
    float d[6];
    for (int i = 0; i < 6; ++i) {
        const float gi = g[i];
        m[i] = beta1 * m[i] + (1.0f - beta1) * gi;
        v[i] = beta2 * v[i] + (1.0f - beta2) * gi * gi;
        d[i] = -lr.v[i] * (m[i] / c1) / (sqrtf(v[i] / c2) + eps);
    }
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
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) K2[3 * i + j] = K[3 * i] * K[j] + K[3 * i + 1] * K[3 + j] + K[3 * i + 2] * K[6 + j];
    for (int i = 0; i < 9; ++i) {
        const float I = (i % 4 == 0) ? 1.0f : 0.0f;
        R[i] = I + A * K[i] + B * K2[i];
        V[i] = I + B * K[i] + Cc * K2[i];
    }
    const float tt[3] = {V[0] * d[0] + V[1] * d[1] + V[2] * d[2], V[3] * d[0] + V[4] * d[1] + V[5] * d[2],
                         V[6] * d[0] + V[7] * d[1] + V[8] * d[2]};
    float o[12];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 4; ++j)
            o[4 * i + j] = R[3 * i] * T[j] + R[3 * i + 1] * T[4 + j] + R[3 * i + 2] * T[8 + j] + (j == 3 ? tt[i] : 0.0f);
    for (int i = 0; i < 12; ++i) T[i] = o[i];
}
