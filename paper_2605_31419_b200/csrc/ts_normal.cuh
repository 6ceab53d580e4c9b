// ts_normal.cuh -- face normals of the rendered normal map (Eq. 12; reading S26) and the
// reverse mode of their dependence on the vertices / the pose.
//   n = s m / |m|,  m = a x b,  a = R (P1 - P0),  b = R (P2 - P0),  s = -sign(m . Q0)  (towards the camera)
// The edges are differenced in WORLD space (nearby floats subtract exactly) and then rotated.
#pragma once
#include "ts_internal.cuh"

struct TsFaceNormal {
    float a[3], b[3], n[3];
    float s_over_len;                 // s / |m|
};

// T = row-major 3x4 pose, P = the three world vertices.
__device__ __forceinline__ void ts_face_normal_geom(const float* T, const float P[3][3], TsFaceNormal& g) {
    const float e1[3] = {P[1][0] - P[0][0], P[1][1] - P[0][1], P[1][2] - P[0][2]};
    const float e2[3] = {P[2][0] - P[0][0], P[2][1] - P[0][1], P[2][2] - P[0][2]};
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        g.a[i] = T[4 * i] * e1[0] + T[4 * i + 1] * e1[1] + T[4 * i + 2] * e1[2];
        g.b[i] = T[4 * i] * e2[0] + T[4 * i + 1] * e2[1] + T[4 * i + 2] * e2[2];
    }
    const float m0 = g.a[1] * g.b[2] - g.a[2] * g.b[1], m1 = g.a[2] * g.b[0] - g.a[0] * g.b[2],
                m2 = g.a[0] * g.b[1] - g.a[1] * g.b[0];
    float Q0[3];
#pragma unroll
    for (int i = 0; i < 3; ++i)
        Q0[i] = __fmaf_rn(T[4 * i], P[0][0], __fmaf_rn(T[4 * i + 1], P[0][1], __fmaf_rn(T[4 * i + 2], P[0][2], T[4 * i + 3])));
    const float off = m0 * Q0[0] + m1 * Q0[1] + m2 * Q0[2];
    const float il = rsqrtf(m0 * m0 + m1 * m1 + m2 * m2);
    g.s_over_len = off < 0.0f ? il : -il;
    g.n[0] = g.s_over_len * m0, g.n[1] = g.s_over_len * m1, g.n[2] = g.s_over_len * m2;
}

__device__ __forceinline__ void ts_face_normal(const float* T, const float P[3][3], float4& n) {
    TsFaceNormal g;
    ts_face_normal_geom(T, P, g);
    n = make_float4(g.n[0], g.n[1], g.n[2], 0.0f);
}

// gn = dL/dn  ->  ga = dL/da, gb = dL/db (camera space).  g_m = s (gn - n (n . gn)) / |m|,  ga = b x g_m,  gb = g_m x a.
__device__ __forceinline__ void ts_face_normal_bwd(const TsFaceNormal& g, const float gn[3], float ga[3], float gb[3]) {
    const float ngn = g.n[0] * gn[0] + g.n[1] * gn[1] + g.n[2] * gn[2];
    float gm[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) gm[i] = g.s_over_len * (gn[i] - g.n[i] * ngn);
    ga[0] = g.b[1] * gm[2] - g.b[2] * gm[1], ga[1] = g.b[2] * gm[0] - g.b[0] * gm[2], ga[2] = g.b[0] * gm[1] - g.b[1] * gm[0];
    gb[0] = gm[1] * g.a[2] - gm[2] * g.a[1], gb[1] = gm[2] * g.a[0] - gm[0] * g.a[2], gb[2] = gm[0] * g.a[1] - gm[1] * g.a[0];
}
