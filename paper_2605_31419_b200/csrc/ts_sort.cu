// ts_sort.cu -- a2: stable LSD radix sort of the (tile<<32 | depth) keys ("faces are sorted in depth order",
// PAPER.md:103) as a hand-written onesweep: one upfront histogram of every digit, then ONE kernel per 8-bit
// digit that ranks, resolves its global offsets by decoupled look-back and scatters -- each key is read and
// written once per digit.  Launch geometry never depends on the (device-side) pair count: persistent CTAs pull
// tile indices from a ticket counter, which also guarantees look-back progress.  Integer only; bit-exact.
#include "ts_internal.cuh"

namespace {

constexpr uint32_t SS_AGG = 1u << 30, SS_PREFIX = 2u << 30, SS_FLAGS = 3u << 30, SS_VAL = (1u << 30) - 1u;

// zero what this sort will use: digit histograms, look-back states of the tiles in play, tickets, tile ranges
__global__ void sort_prep_kernel(TsFrameDev f) {
    const uint32_t n = ts_eff_pairs(f);
    const uint32_t n_tiles = (n + TS_SORT_TILE - 1) / TS_SORT_TILE;
    const size_t stride = (size_t)gridDim.x * blockDim.x, gid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (size_t i = gid; i < (size_t)TS_MAX_PASSES * TS_RADIX; i += stride) f.hist[i] = 0;
    for (int p = 0; p < f.n_passes; ++p) {
        uint32_t* st = f.sort_state + (size_t)p * f.n_sort_tiles_cap * TS_RADIX;
        for (size_t i = gid; i < (size_t)n_tiles * TS_RADIX; i += stride) st[i] = 0;
    }
    for (size_t i = gid; i < (size_t)f.NT; i += stride) f.tile_ranges[i] = make_uint2(0u, 0u);
    if (gid < TS_MAX_PASSES) f.ctrl->sort_ticket[gid] = 0;
}

// all digit histograms in one read of the keys
__global__ void __launch_bounds__(256) sort_hist_kernel(TsFrameDev f) {
    __shared__ uint32_t sh[TS_MAX_PASSES * TS_RADIX];
    const uint32_t n = ts_eff_pairs(f);
    for (int i = threadIdx.x; i < f.n_passes * TS_RADIX; i += blockDim.x) sh[i] = 0;
    __syncthreads();
    const unsigned long long* keys = f.keys[0];
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const unsigned long long k = keys[i];
        for (int p = 0; p < f.n_passes; ++p) atomicAdd(&sh[p * TS_RADIX + (uint32_t)((k >> (8 * p)) & 0xffu)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < f.n_passes * TS_RADIX; i += blockDim.x)
        if (sh[i]) atomicAdd(&f.hist[i], sh[i]);
}

// one digit: rank (warp match), look back, scatter.  Stable: keys keep their input order within a digit.
__global__ void __launch_bounds__(TS_SORT_THREADS)
onesweep_pass_kernel(TsFrameDev f, int pass, const unsigned long long* __restrict__ kin,
                     const uint32_t* __restrict__ vin, unsigned long long* __restrict__ kout,
                     uint32_t* __restrict__ vout) {
    __shared__ uint32_t wh[TS_SORT_THREADS / 32][TS_RADIX];   // per-warp digit counts -> exclusive warp prefixes
    __shared__ uint32_t base[TS_RADIX];                        // global position of this tile's first key per digit
    __shared__ uint32_t gofs[TS_RADIX];                        // exclusive scan of the global digit histogram
    __shared__ uint32_t s_tile;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n = ts_eff_pairs(f);
    const uint32_t n_tiles = (n + TS_SORT_TILE - 1) / TS_SORT_TILE;
    const int shift = 8 * pass;
    uint32_t* state = f.sort_state + (size_t)pass * f.n_sort_tiles_cap * TS_RADIX;
    // exclusive scan of hist[pass] (256 entries, redone by every CTA: cheaper than a launch)
    {
        const uint32_t h = f.hist[pass * TS_RADIX + tid];
        uint32_t incl = h;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        if (lane == 31) base[warp] = incl;
        __syncthreads();
        uint32_t woff = 0;
        for (int w = 0; w < warp; ++w) woff += base[w];
        __syncthreads();
        gofs[tid] = woff + incl - h;
    }
    for (;;) {
        __syncthreads();
        if (tid == 0) s_tile = atomicAdd(&f.ctrl->sort_ticket[pass], 1u);
        for (int i = tid; i < (TS_SORT_THREADS / 32) * TS_RADIX; i += TS_SORT_THREADS) (&wh[0][0])[i] = 0;
        __syncthreads();
        const uint32_t tile = s_tile;
        if (tile >= n_tiles) break;
        const uint32_t wbase = tile * TS_SORT_TILE + warp * (TS_SORT_ITEMS * 32);
        unsigned long long key[TS_SORT_ITEMS];
        uint32_t val[TS_SORT_ITEMS], ofs[TS_SORT_ITEMS], dig[TS_SORT_ITEMS];
#pragma unroll
        for (int i = 0; i < TS_SORT_ITEMS; ++i) {
            const uint32_t idx = wbase + i * 32 + lane;
            const bool ok = idx < n;
            key[i] = ok ? kin[idx] : 0ull;
            val[i] = ok ? vin[idx] : 0u;
            dig[i] = ok ? (uint32_t)((key[i] >> shift) & 0xffu) : (0x100u | lane);   // invalid lanes match nobody
        }
#pragma unroll
        for (int i = 0; i < TS_SORT_ITEMS; ++i) {
            const uint32_t peers = __match_any_sync(0xffffffffu, dig[i]);
            const int leader = __ffs(peers) - 1;
            uint32_t old = 0;
            if (lane == leader && dig[i] < 0x100u) {
                old = wh[warp][dig[i]];
                wh[warp][dig[i]] = old + __popc(peers);
            }
            old = __shfl_sync(0xffffffffu, old, leader);
            ofs[i] = old + __popc(peers & ((1u << lane) - 1u));
            __syncwarp();
        }
        __syncthreads();
        // per digit: warp counts -> exclusive warp prefixes, tile count
        uint32_t cnt = 0;
#pragma unroll
        for (int w = 0; w < TS_SORT_THREADS / 32; ++w) {
            const uint32_t t = wh[w][tid];
            wh[w][tid] = cnt;
            cnt += t;
        }
        // decoupled look-back for digit `tid`
        volatile uint32_t* st = state;
        st[(size_t)tile * TS_RADIX + tid] = (tile == 0 ? SS_PREFIX : SS_AGG) | cnt;
        uint32_t excl = 0;
        for (int64_t t = (int64_t)tile - 1; t >= 0; --t) {
            uint32_t s;
            do { s = st[(size_t)t * TS_RADIX + tid]; } while ((s & SS_FLAGS) == 0);
            excl += s & SS_VAL;
            if ((s & SS_FLAGS) == SS_PREFIX) break;
        }
        if (tile != 0) st[(size_t)tile * TS_RADIX + tid] = SS_PREFIX | (excl + cnt);
        base[tid] = gofs[tid] + excl;
        __syncthreads();
#pragma unroll
        for (int i = 0; i < TS_SORT_ITEMS; ++i) {
            if (dig[i] < 0x100u) {
                const uint32_t dst = base[dig[i]] + wh[warp][dig[i]] + ofs[i];
                kout[dst] = key[i];
                vout[dst] = val[i];
            }
        }
    }
}

// tile_ranges from the sorted keys
__global__ void tile_ranges_kernel(TsFrameDev f, const unsigned long long* __restrict__ keys) {
    const uint32_t n = ts_eff_pairs(f);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const uint32_t t = (uint32_t)(keys[i] >> 32);
        if (t >= (uint32_t)f.NT) continue;
        if (i == 0 || (uint32_t)(keys[i - 1] >> 32) != t) f.tile_ranges[t].x = (uint32_t)i;
        if (i + 1 == n || (uint32_t)(keys[i + 1] >> 32) != t) f.tile_ranges[t].y = (uint32_t)(i + 1);
    }
}

}  // namespace

int32_t ts_launch_sort(const ts_ctx* ctx, ts_frame* fr, cudaStream_t stream) {
    const TsFrameDev& f = fr->d;
    const int grid_small = ctx->num_sms * 2;
    sort_prep_kernel<<<grid_small, 256, 0, stream>>>(f);
    sort_hist_kernel<<<grid_small, 256, 0, stream>>>(f);
    const uint32_t grid_pass = (uint32_t)min((uint64_t)f.n_sort_tiles_cap, (uint64_t)ctx->num_sms * 4u);
    int cur = 0;
    for (int p = 0; p < f.n_passes; ++p) {
        onesweep_pass_kernel<<<grid_pass, TS_SORT_THREADS, 0, stream>>>(f, p, f.keys[cur], f.vals[cur], f.keys[cur ^ 1],
                                                                        f.vals[cur ^ 1]);
        cur ^= 1;
    }
    fr->sorted_buf = cur;
    tile_ranges_kernel<<<grid_small, 256, 0, stream>>>(f, f.keys[cur]);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
