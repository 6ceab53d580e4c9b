// ts_sort.cu -- a2: bin + sort ("faces are sorted in depth order") as an MSD-first radix sort of
// the (tile, depth) key, shaped for P ~ 1e5..1e6 pairs where a global LSD sort is pure launch latency:
//   bin_setup_kernel : the most-significant digit IS the tile id, and its histogram and exclusive scan already
//       exist (tile_count -> tile_ranges / tile_cursor, made by the project kernel), so the MSD pass is one
//       scatter: every visible face writes (depth_key << 32 | face, slot) into the segment of each tile it
//       touches (cursor atomics; faces that touch many tiles are spread over the warp).  The same pass builds
//       the face's 160 B render record once (F7), instead of once per (tile, face) pair inside the renderers.
//   tile_sort_kernel : one CTA per tile sorts its segment by the remaining 60 key bits (depth, then face index:
//       the result is exactly the stable sort of (tile << 32 | depth) with faces emitted in index order, F6) in
//       shared memory -- rank sort for short lists, bitonic network above -- and writes the sorted (slot, face)
//       list the renderers walk plus the sorted 64-bit keys.  Segments longer than TS_SORT_SMEM run the same
//       network in global memory (slow, correct, rare).
// Integer only; bit-exact against the oracle's std::stable_sort.
#include "ts_raster.cuh"

namespace {

__global__ void __launch_bounds__(TS_BIN_THREADS)
bin_setup_kernel(TsFrameDev f, TsCamDev cam) {
    const int lane = threadIdx.x & 31;
    const uint32_t nvis = min(ts_eff_visible(f), f.vis_cap);
    const uint32_t n_round = (nvis + TS_BIN_THREADS - 1) / TS_BIN_THREADS * TS_BIN_THREADS;
    for (uint32_t slot = blockIdx.x * TS_BIN_THREADS + threadIdx.x; slot < n_round; slot += gridDim.x * TS_BIN_THREADS) {
        const bool live = slot < nvis;
        int tx0 = 0, ty0 = 0, ntx = 0, nty = 0;
        unsigned long long key = 0;
        if (live) {
            const float4* s4 = f.scr + TS_SCR_F4 * (size_t)slot;
            const float4 s0 = s4[0], s1 = s4[1], s2 = s4[2], s3 = s4[3];
            float4 rec[TS_REC_F4];
            ts_build_record(s0, s1, s2, cam, rec);
            float4* out = f.rec + TS_REC_F4 * (size_t)slot;
#pragma unroll
            for (int i = 0; i < TS_REC_F4; ++i) out[i] = rec[i];
            const int rlo = __float_as_int(s2.z), rhi = __float_as_int(s2.w);
            const int x0 = (int)(short)(rlo & 0xffff), y0 = rlo >> 16, x1 = (int)(short)(rhi & 0xffff), y1 = rhi >> 16;
            tx0 = x0 >> 4, ty0 = y0 >> 4, ntx = (x1 >> 4) - tx0 + 1, nty = (y1 >> 4) - ty0 + 1;
            key = ((unsigned long long)__float_as_uint(s3.y) << 32) | __float_as_uint(s3.x);
        }
        const int nt = ntx * nty;
        // narrow faces (the common case): the owning lane scatters its <= 4 pairs itself
        if (nt <= 4) {
            for (int i = 0; i < nt; ++i) {
                const int ty = ty0 + i / ntx, tx = tx0 + i % ntx;
                const uint32_t pos = atomicAdd(f.tile_cursor + ty * f.tiles_x + tx, 1u);
                if (pos < f.pair_cap) f.pkey[pos] = key, f.pslot[pos] = slot;
            }
        }
        // wide faces: the whole warp scatters one face's tiles together
        uint32_t wide = __ballot_sync(0xffffffffu, nt > 4);
        while (wide) {
            const int src = __ffs(wide) - 1;
            wide &= wide - 1;
            const int btx0 = __shfl_sync(0xffffffffu, tx0, src), bty0 = __shfl_sync(0xffffffffu, ty0, src);
            const int bntx = __shfl_sync(0xffffffffu, ntx, src), bnt = __shfl_sync(0xffffffffu, nt, src);
            const unsigned long long bkey = __shfl_sync(0xffffffffu, key, src);
            const uint32_t bslot = __shfl_sync(0xffffffffu, slot, src);
            for (int i = lane; i < bnt; i += 32) {
                const int ty = bty0 + i / bntx, tx = btx0 + i % bntx;
                const uint32_t pos = atomicAdd(f.tile_cursor + ty * f.tiles_x + tx, 1u);
                if (pos < f.pair_cap) f.pkey[pos] = bkey, f.pslot[pos] = bslot;
            }
        }
    }
}

// ascending compare-exchange network for arbitrary n (indices >= n behave as +inf and never move): bitonic sort in
// the "mirror first step" form, in which every exchange puts the smaller key at the lower index.
template <typename KP, typename VP>
__device__ __forceinline__ void cta_sort_network(KP k, VP v, uint32_t n) {
    uint32_t N = 1;
    while (N < n) N <<= 1;
    const uint32_t half = N >> 1;
    for (uint32_t size = 2; size <= N; size <<= 1) {
        const uint32_t hs = size >> 1;
        for (uint32_t t = threadIdx.x; t < half; t += blockDim.x) {
            const uint32_t blk = t / hs, off = t - blk * hs;
            const uint32_t lo = blk * size + off, hi = blk * size + size - 1 - off;
            if (hi < n) {
                const unsigned long long a = k[lo], b = k[hi];
                if (b < a) {
                    k[lo] = b, k[hi] = a;
                    const uint32_t va = v[lo];
                    v[lo] = v[hi], v[hi] = va;
                }
            }
        }
        __syncthreads();
        for (uint32_t stride = hs >> 1; stride > 0; stride >>= 1) {
            for (uint32_t t = threadIdx.x; t < half; t += blockDim.x) {
                const uint32_t lo = 2 * stride * (t / stride) + (t % stride), hi = lo + stride;
                if (hi < n) {
                    const unsigned long long a = k[lo], b = k[hi];
                    if (b < a) {
                        k[lo] = b, k[hi] = a;
                        const uint32_t va = v[lo];
                        v[lo] = v[hi], v[hi] = va;
                    }
                }
            }
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(TS_SORT_THREADS) tile_sort_kernel(TsFrameDev f) {
    __shared__ unsigned long long sk[TS_SORT_SMEM];
    __shared__ uint32_t sv[TS_SORT_SMEM];
    const uint32_t tile = blockIdx.x;
    const uint2 range = f.tile_ranges[tile];
    const uint32_t n = range.y - range.x;
    if (n == 0) return;
    const unsigned long long thi = (unsigned long long)tile << 32;
    unsigned long long* gk = f.pkey + range.x;
    uint32_t* gv = f.pslot + range.x;
    if (n <= TS_SORT_THREADS) {
        // rank sort: keys are unique (the face index is part of the key), so ranks are a permutation
        unsigned long long mine = 0;
        uint32_t mv = 0;
        if (threadIdx.x < n) mine = gk[threadIdx.x], mv = gv[threadIdx.x], sk[threadIdx.x] = mine;
        __syncthreads();
        if (threadIdx.x < n) {
            uint32_t rank = 0;
            for (uint32_t j = 0; j < n; ++j) rank += (sk[j] < mine) ? 1u : 0u;
            f.sorted[range.x + rank] = make_uint2(mv, (uint32_t)mine);
            f.skey[range.x + rank] = thi | (mine >> 32);
        }
        return;
    }
    if (n <= TS_SORT_SMEM) {
        for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) sk[i] = gk[i], sv[i] = gv[i];
        __syncthreads();
        cta_sort_network(sk, sv, n);
        for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
            const unsigned long long kk = sk[i];
            f.sorted[range.x + i] = make_uint2(sv[i], (uint32_t)kk);
            f.skey[range.x + i] = thi | (kk >> 32);
        }
        return;
    }
    // oversize segment: same network, in place in global memory (volatile: exchanged across threads between barriers)
    cta_sort_network((volatile unsigned long long*)gk, (volatile uint32_t*)gv, n);
    for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
        const unsigned long long kk = gk[i];
        f.sorted[range.x + i] = make_uint2(gv[i], (uint32_t)kk);
        f.skey[range.x + i] = thi | (kk >> 32);
    }
}

}  // namespace

int32_t ts_launch_sort(const ts_ctx* ctx, ts_frame* fr, cudaStream_t stream) {
    const TsFrameDev& f = fr->d;
    const uint32_t grid_bin = (uint32_t)min((uint64_t)(f.vis_cap + TS_BIN_THREADS - 1) / TS_BIN_THREADS,
                                            (uint64_t)ctx->num_sms * 16u);
    bin_setup_kernel<<<grid_bin, TS_BIN_THREADS, 0, stream>>>(f, fr->cam);
    tile_sort_kernel<<<f.NT, TS_SORT_THREADS, 0, stream>>>(f);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
