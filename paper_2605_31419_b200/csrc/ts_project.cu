// ts_project.cu -- a1: project + cull + bounds (Eq. 1), fused with the single-pass chained
// scan that gives every surviving face its slot and pair offset, and with the emission of the unsorted
// (tile<<32 | depth, slot) pairs.  One kernel, one pass over the map: 36 B read per face (soup), float4 loads.
//
// Arithmetic follows the fixed operation order N1-N5 of DESIGN.md with explicit round-to-nearest intrinsics,
// so cull decisions, pixel rects, tile counts and depth keys are bit-identical to the float32 oracle.
#include "ts_internal.cuh"

namespace {

// chained-scan state: flag(2) | pairs(30) | epoch(4) | visible(28)
constexpr unsigned long long ST_AGG = 1ull << 62, ST_PREFIX = 2ull << 62, ST_FLAGS = 3ull << 62;
__device__ __forceinline__ unsigned long long st_pack(unsigned long long flag, uint32_t vis, uint32_t pairs,
                                                      uint32_t epoch) {
    return flag | ((unsigned long long)(pairs & 0x3FFFFFFFu) << 32) | ((unsigned long long)(epoch & 0xFu) << 28) |
           (unsigned long long)(vis & 0x0FFFFFFFu);
}
__device__ __forceinline__ uint32_t st_vis(unsigned long long s) { return (uint32_t)(s & 0x0FFFFFFFull); }
__device__ __forceinline__ uint32_t st_pairs(unsigned long long s) { return (uint32_t)((s >> 32) & 0x3FFFFFFFull); }
__device__ __forceinline__ uint32_t st_epoch(unsigned long long s) { return (uint32_t)((s >> 28) & 0xFull); }

struct FaceOut {
    float u[3], v[3], w[3];
    int x0, y0, x1, y1;
    uint32_t key, tiles;
    bool vis;
};

// N1-N5.  p = 9 floats (three world vertices), T = row-major 3x4 pose.
__device__ __forceinline__ void project_face(const float* p, const float* T, const TsCamDev& cam, float eps_area,
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
    o.vis = true;
}

template <bool SOUP>
__global__ void __launch_bounds__(TS_PROJ_THREADS)
project_kernel(TsFrameDev f, const float* __restrict__ pos, const int32_t* __restrict__ faces,
               const float* __restrict__ opacity, const float* __restrict__ Tcw, TsCamDev cam, float eps_area,
               int pos_aligned) {
    __shared__ __align__(16) float sp[TS_PROJ_THREADS * 9];
    __shared__ float sT[12];
    __shared__ uint32_t s_tile, s_epoch;
    __shared__ uint32_t s_wv[8], s_wp[8];
    __shared__ uint32_t s_excl_vis, s_excl_pairs;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    volatile TsCtrl* ctrl = f.ctrl;
    if (tid == 0) {
        s_tile = atomicAdd((uint32_t*)&f.ctrl->proj_ticket, 1u);   // ticket order => look-back always progresses
        s_epoch = ctrl->epoch;
    }
    if (tid < 12) sT[tid] = __ldg(Tcw + tid);
    __syncthreads();
    const uint32_t tile = s_tile, epoch = s_epoch;
    const int64_t face0 = (int64_t)tile * TS_PROJ_THREADS;
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
    } else if (tid < n_here) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int v = __ldg(faces + (face0 + tid) * 3 + k);
            p[3 * k] = __ldg(pos + 3 * (int64_t)v), p[3 * k + 1] = __ldg(pos + 3 * (int64_t)v + 1),
            p[3 * k + 2] = __ldg(pos + 3 * (int64_t)v + 2);
        }
    }
    FaceOut o;
    o.vis = false, o.tiles = 0;
    if (tid < n_here) project_face(p, sT, cam, eps_area, o);

    // block-wide exclusive scan of (visible, tiles)
    uint32_t iv = o.vis ? 1u : 0u, ip = o.tiles;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t tv = __shfl_up_sync(0xffffffffu, iv, d), tp = __shfl_up_sync(0xffffffffu, ip, d);
        if (lane >= d) iv += tv, ip += tp;
    }
    if (lane == 31) s_wv[warp] = iv, s_wp[warp] = ip;
    __syncthreads();
    if (warp == 0) {
        uint32_t wv = lane < 8 ? s_wv[lane] : 0u, wp = lane < 8 ? s_wp[lane] : 0u;
        uint32_t cv = wv, cp = wp;
#pragma unroll
        for (int d = 1; d < 8; d <<= 1) {
            const uint32_t tv = __shfl_up_sync(0xffffffffu, cv, d), tp = __shfl_up_sync(0xffffffffu, cp, d);
            if (lane >= d) cv += tv, cp += tp;
        }
        const uint32_t tot_v = __shfl_sync(0xffffffffu, cv, 7), tot_p = __shfl_sync(0xffffffffu, cp, 7);
        if (lane < 8) s_wv[lane] = cv - wv, s_wp[lane] = cp - wp;
        // decoupled look-back (warp-parallel window of 32 predecessors)
        volatile unsigned long long* st = f.scan_state;
        if (lane == 0) st[tile] = st_pack(tile == 0 ? ST_PREFIX : ST_AGG, tot_v, tot_p, epoch);
        uint32_t ex_v = 0, ex_p = 0;
        int64_t look = (int64_t)tile - 1;
        while (look >= 0) {
            const int64_t t = look - lane;
            unsigned long long s = 0;
            bool ready = (t < 0);
            while (!__all_sync(0xffffffffu, ready)) {
                if (!ready) {
                    s = st[t];
                    ready = ((s & ST_FLAGS) != 0) && st_epoch(s) == epoch;
                }
            }
            const bool is_prefix = (t >= 0) && ((s & ST_FLAGS) == ST_PREFIX);
            const uint32_t pm = __ballot_sync(0xffffffffu, is_prefix);
            const int stop = pm ? (__ffs(pm) - 1) : 31;         // nearest predecessor holding an inclusive prefix
            uint32_t cv2 = (t >= 0 && lane <= stop) ? st_vis(s) : 0u, cp2 = (t >= 0 && lane <= stop) ? st_pairs(s) : 0u;
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                cv2 += __shfl_xor_sync(0xffffffffu, cv2, d);
                cp2 += __shfl_xor_sync(0xffffffffu, cp2, d);
            }
            ex_v += cv2, ex_p += cp2;
            if (pm) break;
            look -= 32;
        }
        if (lane == 0) {
            if (tile != 0) st[tile] = st_pack(ST_PREFIX, ex_v + tot_v, ex_p + tot_p, epoch);
            s_excl_vis = ex_v, s_excl_pairs = ex_p;
            if (tile == f.n_proj_tiles - 1) {
                const uint32_t nv = ex_v + tot_v, np = ex_p + tot_p;
                ctrl->n_visible = nv, ctrl->n_pairs = np;
                uint32_t fl = 0;
                if (np > f.pair_cap) fl |= TS_FLAG_OVERFLOW_PAIRS;
                if (nv > f.vis_cap) fl |= TS_FLAG_OVERFLOW_VISIBLE;
                ctrl->flags = fl;
            }
        }
    }
    __syncthreads();
    if (o.vis) {
        const uint32_t slot = s_excl_vis + s_wv[warp] + iv - 1u;
        uint32_t poff = s_excl_pairs + s_wp[warp] + ip - o.tiles;
        if (slot < f.vis_cap) {
            const uint32_t m = (uint32_t)(face0 + tid);
            float ob;
            if (SOUP) {
                ob = (__ldg(opacity + 3 * (int64_t)m) + __ldg(opacity + 3 * (int64_t)m + 1) +
                      __ldg(opacity + 3 * (int64_t)m + 2)) * (1.0f / 3.0f);
            } else {
                ob = (__ldg(opacity + __ldg(faces + 3 * (int64_t)m)) + __ldg(opacity + __ldg(faces + 3 * (int64_t)m + 1)) +
                      __ldg(opacity + __ldg(faces + 3 * (int64_t)m + 2))) * (1.0f / 3.0f);
            }
            const int rlo = (o.x0 & 0xffff) | (o.y0 << 16), rhi = (o.x1 & 0xffff) | (o.y1 << 16);
            f.vis_face[slot] = m;
            f.rect[slot] = make_int2(rlo, rhi);
            f.depth_key[slot] = o.key;
            f.tiles_touched[slot] = o.tiles;
            float4* s4 = f.scr + 3 * (int64_t)slot;
            s4[0] = make_float4(o.u[0], o.v[0], o.w[0], o.u[1]);
            s4[1] = make_float4(o.v[1], o.w[1], o.u[2], o.v[2]);
            s4[2] = make_float4(o.w[2], ob, __int_as_float(rlo), __int_as_float(rhi));
            // F6 emission: ty-major then tx, face order is the scan order
            for (int ty = o.y0 >> 4; ty <= (o.y1 >> 4); ++ty)
                for (int tx = o.x0 >> 4; tx <= (o.x1 >> 4); ++tx) {
                    if (poff < f.pair_cap) {
                        f.keys[0][poff] = ((unsigned long long)(uint32_t)(ty * f.tiles_x + tx) << 32) | o.key;
                        f.vals[0][poff] = slot;
                    }
                    ++poff;
                }
        }
    }
    // the last block to finish re-arms the tickets and advances the epoch for the next call
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        const uint32_t done = atomicAdd((uint32_t*)&f.ctrl->proj_done, 1u);
        if (done == gridDim.x - 1) {
            ctrl->proj_done = 0;
            ctrl->proj_ticket = 0;
            ctrl->epoch = (epoch % 15u) + 1u;
            __threadfence();
        }
    }
}

}  // namespace

int32_t ts_launch_project(const ts_ctx* ctx, ts_frame* fr, const ts_scene* sc, cudaStream_t stream) {
    (void)ctx;
    const TsFrameDev& f = fr->d;
    const int aligned = ((reinterpret_cast<uintptr_t>(sc->pos) & 15u) == 0) ? 1 : 0;
    if (sc->faces == nullptr)
        project_kernel<true><<<f.n_proj_tiles, TS_PROJ_THREADS, 0, stream>>>(f, sc->pos, nullptr, sc->opacity, fr->T_cw,
                                                                             fr->cam, fr->prm.eps_area, aligned);
    else
        project_kernel<false><<<f.n_proj_tiles, TS_PROJ_THREADS, 0, stream>>>(f, sc->pos, sc->faces, sc->opacity,
                                                                              fr->T_cw, fr->cam, fr->prm.eps_area, aligned);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
