// ts_project.cu -- a1: project + cull + bounds (Eq. 1) in ONE streaming pass over the map:
// 36 B read per face (soup), float4 loads staged through shared memory, no inter-CTA dependency and no tail.
// Surviving faces get a slot from a per-CTA-aggregated atomic counter (slots are NOT in face order: every later
// stage orders by face index explicitly), write their 64 B raw screen record and count themselves into the tiles
// they touch (RED.ADD on tile_count).  The scan of the tile counts is done by the binning kernel (ts_sort.cu).
//
// Arithmetic follows the fixed operation order N1-N5 of DESIGN.md with explicit round-to-nearest intrinsics,
// so cull decisions, pixel rects, tile counts and depth keys are bit-identical to the float32 oracle.
#include "ts_internal.cuh"

namespace {

struct FaceOut {
    float u[3], v[3], w[3];
    int x0, y0, x1, y1;
    uint32_t key, tiles;
    bool vis;
};

// N1-N5.  p = 9 floats (three world vertices), T = row-major 3x4 pose.
__device__ __forceinline__ void project_face(const float* p, const float* T, const TsCamDev& cam, float eps_area, bool tight,
                                             FaceOut& o) {
    float X[3], Y[3], Z[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float px = p[3 * k], py = p[3 * k + 1], pz = p[3 * k + 2];
        X[k] = __fmaf_rn(T[0], px, __fmaf_rn(T[1], py, __fmaf_rn(T[2], pz, T[3])));
        Y[k] = __fmaf_rn(T[4], px, __fmaf_rn(T[5], py, __fmaf_rn(T[6], pz, T[7])));
        Z[k] = __fmaf_rn(T[8], px, __fmaf_rn(T[9], py, __fmaf_rn(T[10], pz, T[11])));
    }
    o.vis = false;
    o.tiles = 0;
    if (!(Z[0] > cam.znear) || !(Z[1] > cam.znear) || !(Z[2] > cam.znear)) return;   // F2 (NaN culls)
    // Conservative frustum pre-cull (most of the map is outside the view): if all three vertices are more than two
    // pixels beyond the same image border -- decided without a division, with a margin ~1000x the rounding error of
    // these expressions -- the exact path below would find an empty pixel rect (F5) and cull the face as well, so
    // skipping it cannot change any result.
    {
        const float ax = cam.cx + 2.0f, bx = cam.cx - (float)(cam.W + 1), ay = cam.cy + 2.0f, by = cam.cy - (float)(cam.H + 1);
        bool l = true, r = true, t = true, b = true;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            l = l && (cam.fx * X[k] + ax * Z[k] < 0.0f);      // u_k < -2
            r = r && (cam.fx * X[k] + bx * Z[k] > 0.0f);      // u_k > W + 1
            t = t && (cam.fy * Y[k] + ay * Z[k] < 0.0f);      // v_k < -2
            b = b && (cam.fy * Y[k] + by * Z[k] > 0.0f);      // v_k > H + 1
        }
        if (l || r || t || b) return;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        o.w[k] = __fdiv_rn(1.0f, Z[k]);                                               // N2
        o.u[k] = __fmaf_rn(cam.fx, __fmul_rn(X[k], o.w[k]), cam.cx);
        o.v[k] = __fmaf_rn(cam.fy, __fmul_rn(Y[k], o.w[k]), cam.cy);
    }
    const float a = __fsub_rn(o.u[1], o.u[0]), b = __fsub_rn(o.v[2], o.v[0]);         // N3
    const float c = __fsub_rn(o.v[1], o.v[0]), d = __fsub_rn(o.u[2], o.u[0]);
    const float S = __fmaf_rn(a, b, -__fmul_rn(c, d));
    const float aS = fabsf(S);
    if (!(aS > eps_area) || !(aS < 1e10f)) return;
    const float umin = fminf(o.u[0], fminf(o.u[1], o.u[2])), umax = fmaxf(o.u[0], fmaxf(o.u[1], o.u[2]));
    const float vmin = fminf(o.v[0], fminf(o.v[1], o.v[2])), vmax = fmaxf(o.v[0], fmaxf(o.v[1], o.v[2]));
    o.x0 = (int)fminf(fmaxf(ceilf(umin), 0.0f), (float)cam.W);                        // N4
    o.x1 = (int)fminf(fmaxf(floorf(umax), -1.0f), (float)(cam.W - 1));
    o.y0 = (int)fminf(fmaxf(ceilf(vmin), 0.0f), (float)cam.H);
    o.y1 = (int)fminf(fmaxf(floorf(vmax), -1.0f), (float)(cam.H - 1));
    if (o.x0 > o.x1 || o.y0 > o.y1) return;
    const float zb = __fmul_rn(__fadd_rn(__fadd_rn(Z[0], Z[1]), Z[2]), 1.0f / 3.0f);  // N5
    o.key = __float_as_uint(zb);
    o.tiles = (uint32_t)(((o.x1 >> 4) - (o.x0 >> 4) + 1) * ((o.y1 >> 4) - (o.y0 >> 4) + 1));
    if (tight) {
        // tiles_touched = the tiles the triangle meets (reading S31)
        uint32_t nt = 0;
        for (int ty = o.y0 >> 4; ty <= (o.y1 >> 4); ++ty)
            for (int tx = o.x0 >> 4; tx <= (o.x1 >> 4); ++tx)
                nt += ts_tile_overlaps(o.u, o.v, max(o.x0, tx * TS_TILE), max(o.y0, ty * TS_TILE), min(o.x1, tx * TS_TILE + TS_TILE - 1),
                                       min(o.y1, ty * TS_TILE + TS_TILE - 1)) ? 1u : 0u;
        o.tiles = nt;
    }
    o.vis = true;
}

template <bool SOUP>
__global__ void __launch_bounds__(TS_PROJ_THREADS)
project_kernel(TsFrameDev f, const float* __restrict__ pos, const int32_t* __restrict__ faces,
               const float* __restrict__ opacity, const float* __restrict__ Tcw, TsCamDev cam, float eps_area,
               int pos_aligned) {
    __shared__ __align__(16) float sp[TS_PROJ_THREADS * 9];
    __shared__ float sT[12];
    __shared__ uint32_t s_w[TS_PROJ_THREADS / 32];
    __shared__ uint32_t s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < 12) sT[tid] = __ldg(Tcw + tid);
    const int64_t face0 = (int64_t)blockIdx.x * TS_PROJ_THREADS;
    const int n_here = (int)min((int64_t)TS_PROJ_THREADS, (int64_t)f.M - face0);
    float p[9];
    if (SOUP) {
        // coalesced, vectorised staging of 36 B/face through shared memory (stride-9 reads are conflict-free)
        const float* src = pos + face0 * 9;
        const int nfl = n_here * 9;
        if (pos_aligned) {
            const float4* src4 = reinterpret_cast<const float4*>(src);
            const int n4 = nfl >> 2;
            for (int i = tid; i < n4; i += TS_PROJ_THREADS) reinterpret_cast<float4*>(sp)[i] = __ldg(src4 + i);
            for (int i = (n4 << 2) + tid; i < nfl; i += TS_PROJ_THREADS) sp[i] = __ldg(src + i);
        } else {
            for (int i = tid; i < nfl; i += TS_PROJ_THREADS) sp[i] = __ldg(src + i);
        }
        __syncthreads();
        if (tid < n_here) {
#pragma unroll
            for (int j = 0; j < 9; ++j) p[j] = sp[tid * 9 + j];
        }
    } else {
        if (tid < n_here) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const int v = __ldg(faces + (face0 + tid) * 3 + k);
                p[3 * k] = __ldg(pos + 3 * (int64_t)v), p[3 * k + 1] = __ldg(pos + 3 * (int64_t)v + 1),
                p[3 * k + 2] = __ldg(pos + 3 * (int64_t)v + 2);
            }
        }
        __syncthreads();   // sT
    }
    FaceOut o;
    o.vis = false, o.tiles = 0;
    const bool tight = (f.prm_flags & TS_PARAM_TIGHT_BINNING) != 0;
    if (tid < n_here) project_face(p, sT, cam, eps_area, tight, o);
    // mean vertex opacity of the survivors: requested now, so that its round trip overlaps the slot atomic
    float ob = 0.0f;
    if (o.vis) {
        const int64_t m = face0 + tid;
        float o0, o1, o2;
        if (SOUP) {
            o0 = __ldg(opacity + 3 * m), o1 = __ldg(opacity + 3 * m + 1), o2 = __ldg(opacity + 3 * m + 2);
        } else {
            o0 = __ldg(opacity + __ldg(faces + 3 * m)), o1 = __ldg(opacity + __ldg(faces + 3 * m + 1)),
            o2 = __ldg(opacity + __ldg(faces + 3 * m + 2));
        }
        ob = (f.prm_flags & TS_PARAM_MIN_OPACITY) ? fminf(o0, fminf(o1, o2)) : (o0 + o1 + o2) * (1.0f / 3.0f);
    }

    // slot allocation: warp ballot -> CTA total -> one global atomic per CTA
    const uint32_t bal = __ballot_sync(0xffffffffu, o.vis);
    if (lane == 0) s_w[warp] = __popc(bal);
    __syncthreads();
    if (tid == 0) {
        uint32_t tot = 0;
#pragma unroll
        for (int w = 0; w < TS_PROJ_THREADS / 32; ++w) {
            const uint32_t c = s_w[w];
            s_w[w] = tot;
            tot += c;
        }
        s_base = tot ? atomicAdd(&f.ctrl->vis_counter, tot) : 0u;
    }
    __syncthreads();
    if (o.vis) {
        const uint32_t slot = s_base + s_w[warp] + __popc(bal & ((1u << lane) - 1u));
        if (slot < f.vis_cap) {
            const uint32_t m = (uint32_t)(face0 + tid);
            const int rlo = (o.x0 & 0xffff) | (o.y0 << 16), rhi = (o.x1 & 0xffff) | (o.y1 << 16);
            float4* s4 = f.scr + TS_SCR_F4 * (size_t)slot;
            s4[0] = make_float4(o.u[0], o.v[0], o.w[0], o.u[1]);
            s4[1] = make_float4(o.v[1], o.w[1], o.u[2], o.v[2]);
            s4[2] = make_float4(o.w[2], ob, __int_as_float(rlo), __int_as_float(rhi));
            s4[3] = make_float4(__uint_as_float(m), __uint_as_float(o.key), __uint_as_float(o.tiles), 0.0f);
            for (int ty = o.y0 >> 4; ty <= (o.y1 >> 4); ++ty)
                for (int tx = o.x0 >> 4; tx <= (o.x1 >> 4); ++tx)
                    if (ts_tile_included(tight, o.u, o.v, o.x0, o.y0, o.x1, o.y1, tx, ty)) atomicAdd(f.tile_count + ty * f.tiles_x + tx, 1u);
        }
    }

}

}  // namespace

int32_t ts_launch_project(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, cudaStream_t stream) {
    (void)ctx;
    const TsFrameDev& f = fr->d;
    const int aligned = ((reinterpret_cast<uintptr_t>(sc->pos) & 15u) == 0) ? 1 : 0;
    const uint32_t grid = (uint32_t)((f.M + TS_PROJ_THREADS - 1) / TS_PROJ_THREADS);
    if (sc->faces == nullptr)
        project_kernel<true><<<grid, TS_PROJ_THREADS, 0, stream>>>(f, sc->pos, nullptr, sc->opacity, fr->T_cw, fr->cam,
                                                                   fr->prm.eps_area, aligned);
    else
        project_kernel<false><<<grid, TS_PROJ_THREADS, 0, stream>>>(f, sc->pos, sc->faces, sc->opacity, fr->T_cw,
                                                                    fr->cam, fr->prm.eps_area, aligned);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
