// ts_sort.cu -- a2: bin + sort ("faces are sorted in depth order") as an MSD-first radix sort of
// the (tile, depth) key, shaped for P ~ 1e5..1e6 pairs where a global LSD sort is pure launch latency:
//   bin_setup_kernel : the most-significant digit IS the tile id and its histogram already exists (tile_count,
//       made by the project kernel).  Every CTA scans the NT counts into shared memory by itself (13 KB of L2
//       reads: cheaper than a scan kernel or a last-CTA tail; every CTA also publishes its slice of tile_ranges and
//       of the heaviest-first tile order, CTA 0 the frame counters), then the MSD pass is one scatter:
//       every visible face writes (depth_key, face, slot, rect) into the segment of each tile it touches (cursor
//       atomics; faces that touch many tiles are spread over the warp).  The same pass builds the face's 160 B
//       render record once (F7: unit normals, inradius, incentre, mean opacity), instead of once per (tile, face)
//       pair inside the renderers.
//   tile_sort_kernel : one CTA per tile sorts its segment by the remaining 60 key bits (depth, then face index:
//       exactly the stable sort of (tile << 32 | depth) with faces emitted in index order, F6) in shared memory --
//       rank sort for short lists, a compare-exchange network above -- and writes the sorted
//       (slot, face, rect) list plus the sorted 64-bit keys.  Segments longer than TS_SORT_SMEM run the same
//       network in global memory (slow, correct, rare).  The group that sorted a tile then copies every entry into
//       the list of each 8x4-pixel block its rect overlaps -- the PER-BLOCK lists the renderers walk -- and writes
//       the tile's eight job headers (build_block_lists).  It also re-zeroes the counters.
// Integer only; bit-exact against the oracle's std::stable_sort (the per-block lists: against their definition,
// tests/test_gpu_parity.py check_block_lists).
#include "ts_raster.cuh"

namespace {

// a CTA or a warp-aligned part of one, with its own barrier (0 = the CTA barrier, else a named barrier)
struct TsGroup {
    int tid, n, bar;
    __device__ __forceinline__ void sync() const {
        if (bar == 0) __syncthreads();
        else asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(n) : "memory");
    }
};

// exclusive scan of tile_count[0..NT) by one CTA, in place in `offs` (shared memory, or global for the fallback).
// Pass 1 copies the counts with coalesced loads (every binning CTA does this at the same time: strided loads would
// multiply the L2 requests on the few slices that hold the 13 KB of counts) unless the caller has done so already
// (PRELOADED); pass 2 gives every thread a contiguous run of tiles (stride `per` words: conflict-free for odd
// `per`) and, with `hist`, counts the tiles per list-length bucket (0 = empty, b = floor(log2 c) + 1; zeroed by the
// caller).  Returns the total and the longest list.
template <bool PRELOADED>
__device__ __forceinline__ void cta_scan_tiles(const TsFrameDev& f, uint32_t* offs, uint32_t* s_tmp /*[2*warps+2]*/,
                                               uint32_t& total, uint32_t& gmax, const TsGroup g, uint32_t* hist = nullptr) {
    const int tid = g.tid, lane = tid & 31, warp = tid >> 5, nwarp = g.n >> 5, nthr = g.n;
    if (!PRELOADED) {
        for (int base = 0; base < f.NT; base += 8 * nthr) {      // 8 independent loads in flight per thread
            uint32_t c[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int t = base + k * nthr + tid;
                c[k] = t < f.NT ? __ldcg(f.tile_count + t) : 0u;
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int t = base + k * nthr + tid;
                if (t < f.NT) offs[t] = c[k];
            }
        }
        g.sync();
    }
    const int per = ((f.NT + nthr - 1) / nthr) | 1;
    const int t0 = min(f.NT, tid * per), t1 = min(f.NT, t0 + per);
    uint32_t sum = 0, mx = 0;
    for (int t = t0; t < t1; ++t) {
        const uint32_t c = offs[t];
        sum += c, mx = max(mx, c);
        if (hist) atomicAdd(&hist[32 - __clz(c)], 1u);
    }
    uint32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
    }
    mx = __reduce_max_sync(0xffffffffu, mx);
    if (lane == 31) s_tmp[warp] = incl;
    if (lane == 0) s_tmp[nwarp + warp] = mx;
    g.sync();
    if (warp == 0) {                                            // warp totals -> exclusive warp offsets, total, max
        const uint32_t c = lane < nwarp ? s_tmp[lane] : 0u;
        uint32_t m2 = lane < nwarp ? s_tmp[nwarp + lane] : 0u, in2 = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, in2, d);
            if (lane >= d) in2 += t;
        }
        m2 = __reduce_max_sync(0xffffffffu, m2);
        if (lane < nwarp) s_tmp[lane] = in2 - c;
        if (lane == 31) s_tmp[2 * nwarp] = in2, s_tmp[2 * nwarp + 1] = m2;
    }
    g.sync();
    const uint32_t woff = s_tmp[warp];
    total = s_tmp[2 * nwarp], gmax = s_tmp[2 * nwarp + 1];
    uint32_t run = woff + incl - sum;
    for (int t = t0; t < t1; ++t) {
        const uint32_t c = offs[t];
        offs[t] = run;
        run += c;
    }
    g.sync();
}

// One CTA (the fallback scan): tile_ranges, frame counters, and the tile order (descending log2 bucket of the list length) that
// the persistent render kernels pull work in.  Counts are recovered from the offsets (no second trip to memory).
__device__ __forceinline__ void publish_tiles(const TsFrameDev& f, const uint32_t* offs, uint32_t nv, uint32_t total,
                                              uint32_t gmax, uint32_t fl, uint32_t* s_hist /*[34]*/, const TsGroup g) {
    const int tid = g.tid;
    if (tid < 34) s_hist[tid] = 0;
    g.sync();
    for (int t = tid; t < f.NT; t += g.n) {
        const uint32_t o = offs[t], c = (t + 1 < f.NT ? offs[t + 1] : total) - o;
        f.tile_ranges[t] = (fl || c == 0u) ? make_uint2(0u, 0u) : make_uint2(o, o + c);   // empty tile = (0,0)
        // bucket 0 = empty, b = floor(log2 c) + 1; only ~10 buckets are in use, so the histogram is aggregated per
        // warp (match) before it touches shared memory: one atomic per (warp, bucket), not 32-way conflicts
        const int b = 32 - __clz(c);
        const uint32_t peers = __match_any_sync(__activemask(), b);
        if ((int)(tid & 31) == __ffs(peers) - 1) atomicAdd(&s_hist[b], (uint32_t)__popc(peers));
    }
    g.sync();
    if (tid == 0) {
        uint32_t run = 0;
        for (int b = 32; b >= 0; --b) {                        // heaviest bucket first
            const uint32_t c = s_hist[b];
            s_hist[b] = run;
            run += c;
        }
        volatile TsCtrl* ctrl = f.ctrl;
        ctrl->n_visible = nv, ctrl->n_pairs = total, ctrl->flags = fl, ctrl->max_list = gmax;
    }
    g.sync();
    for (int t = tid; t < f.NT; t += g.n) {
        const uint32_t c = (t + 1 < f.NT ? offs[t + 1] : total) - offs[t];
        const int b = 32 - __clz(c);
        const uint32_t act = __activemask(), peers = __match_any_sync(act, b);
        const int leader = __ffs(peers) - 1, lane = tid & 31;
        uint32_t base = 0;
        if (lane == leader) base = atomicAdd(&s_hist[b], (uint32_t)__popc(peers));
        base = __shfl_sync(act, base, leader);
        const uint32_t o = offs[t];
        const uint32_t xy = (uint32_t)((t % f.tiles_x) * TS_TILE) | ((uint32_t)((t / f.tiles_x) * TS_TILE) << 16);
        f.tile_order[base + __popc(peers & ((1u << lane) - 1u))] =
            (fl || c == 0u) ? make_uint4((uint32_t)t, 0u, 0u, xy) : make_uint4((uint32_t)t, o, o + c, xy);
    }
}

// One warp of every binning CTA: publishes the tile ranges and job headers of the CTA's slice of the tiles.  The
// headers go into tile_order by descending list-length bucket: the bucket begins come from the CTA's own histogram
// (every CTA has scanned all counts), the place inside a bucket from a cursor in global memory that all CTAs share
// (the order inside a bucket is free).  CTA 0 also writes the frame counters.
__device__ __forceinline__ void publish_slice(const TsFrameDev& f, const uint32_t* offs, uint32_t nv, uint32_t total,
                                              uint32_t gmax, uint32_t fl, const uint32_t* hist) {
    const int lane = threadIdx.x & 31;
    const uint32_t h = hist[31 - lane];                        // lane 0 = the heaviest bucket (lists < 2^31: b <= 31)
    uint32_t incl = h;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
    }
    const uint32_t start = incl - h;                            // begin of bucket 31 - lane
    const int S = (f.NT + (int)gridDim.x - 1) / (int)gridDim.x;
    const int t0 = min(f.NT, (int)blockIdx.x * S), t1 = min(f.NT, t0 + S);
    for (int base = t0; base < t1; base += 32) {                // (warp-uniform)
        const int t = base + lane;
        const bool on = t < t1;
        uint32_t o = 0, c = 0;
        if (on) o = offs[t], c = (t + 1 < f.NT ? offs[t + 1] : total) - o;
        const int b = on ? 32 - __clz(c) : 32;                  // 32 = the lanes past the slice
        const uint32_t peers = __match_any_sync(0xffffffffu, b);
        const int leader = __ffs(peers) - 1;
        uint32_t at = 0;
        if (on && lane == leader) at = atomicAdd(&f.ctrl->bucket_cursor[b], (uint32_t)__popc(peers));
        at = __shfl_sync(0xffffffffu, at, leader);
        const uint32_t bstart = __shfl_sync(0xffffffffu, start, (31 - b) & 31);
        if (on) {
            const bool empty = fl || c == 0u;
            const uint32_t xy = (uint32_t)((t % f.tiles_x) * TS_TILE) | ((uint32_t)((t / f.tiles_x) * TS_TILE) << 16);
            f.tile_ranges[t] = empty ? make_uint2(0u, 0u) : make_uint2(o, o + c);     // empty tile = (0,0)
            f.tile_order[bstart + at + __popc(peers & ((1u << lane) - 1u))] =
                empty ? make_uint4((uint32_t)t, 0u, 0u, xy) : make_uint4((uint32_t)t, o, o + c, xy);
        }
    }
    if (blockIdx.x == 0 && lane == 0) {
        volatile TsCtrl* ctrl = f.ctrl;
        ctrl->n_visible = nv, ctrl->n_pairs = total, ctrl->flags = fl, ctrl->max_list = gmax;
    }
}

// fallback for NT > TS_SCAN_LOCAL_MAX: one CTA scans into global memory
__global__ void __launch_bounds__(1024) tile_scan_kernel(TsFrameDev f) {
    __shared__ uint32_t s_tmp[66];
    __shared__ uint32_t s_hist[34];
    uint32_t total, gmax;
    const TsGroup g{(int)threadIdx.x, (int)blockDim.x, 0};
    cta_scan_tiles<false>(f, f.tile_offset, s_tmp, total, gmax, g);
    const uint32_t nv = *(volatile uint32_t*)&f.ctrl->vis_counter;
    uint32_t fl = 0;
    if (total > f.pair_cap) fl |= TS_FLAG_OVERFLOW_PAIRS;
    if (nv > f.vis_cap) fl |= TS_FLAG_OVERFLOW_VISIBLE;
    publish_tiles(f, f.tile_offset, nv, total, gmax, fl, s_hist, g);
}

#define TS_BIN_SCAN_WARPS 8          // warps of a binning CTA that scan the tile counts while the others set faces up

template <bool LOCAL>
__global__ void __launch_bounds__(TS_BIN_THREADS)
bin_setup_kernel(TsFrameDev f, TsCamDev cam, const float* __restrict__ face_sigma, float sigma_global) {
    __shared__ uint32_t s_offs[LOCAL ? TS_SCAN_LOCAL_MAX : 1];
    __shared__ uint32_t s_tmp[2 * (TS_BIN_THREADS / 32) + 2];
    __shared__ uint32_t s_hist[34];
    __shared__ uint32_t s_tot[2];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // This kernel is one wave of dependent round trips, so they are kept few and overlapped: the last
    // TS_BIN_SCAN_WARPS warps scan the tile counts (the scatter needs the offsets) while the other warps fetch their
    // first raw records (speculatively: n_visible arrives with them) and build the render records, which need no
    // offset.  Slots are dealt to the grid warp by warp, so that the live ones spread over all SMs.
    constexpr int SLOT_WARPS = LOCAL ? TS_BIN_THREADS / 32 - TS_BIN_SCAN_WARPS : TS_BIN_THREADS / 32;
    const bool scanner = LOCAL && warp >= SLOT_WARPS;
    const TsGroup sg{(int)threadIdx.x - SLOT_WARPS * 32, TS_BIN_SCAN_WARPS * 32, 1};
    const uint32_t stride = gridDim.x * SLOT_WARPS * 32u;
    uint32_t slot = ((uint32_t)warp * gridDim.x + blockIdx.x) * 32u + (uint32_t)lane;
    float4 s0, s1, s2, s3;
    s0 = s1 = s2 = s3 = make_float4(0.f, 0.f, 0.f, 0.f);
    uint32_t nv = 0, fl = 0, total = 0, gmax = 0;
    const uint32_t* offs = s_offs;
    if (!scanner && slot < f.vis_cap) {
        const float4* s4 = f.scr + TS_SCR_F4 * (size_t)slot;
        s0 = __ldcg(s4), s1 = __ldcg(s4 + 1), s2 = __ldcg(s4 + 2), s3 = __ldcg(s4 + 3);
    }
    if (LOCAL) {
        // every thread of the CTA brings in its share of the tile counts (one round trip for all of them), then the
        // scan warps take over
        constexpr int PER = TS_SCAN_LOCAL_MAX / TS_BIN_THREADS;
        uint32_t c[PER];
#pragma unroll
        for (int k = 0; k < PER; ++k) {
            const int t = k * TS_BIN_THREADS + (int)threadIdx.x;
            c[k] = t < f.NT ? __ldcg(f.tile_count + t) : 0u;
        }
        nv = __ldcg(&f.ctrl->vis_counter);
        if (threadIdx.x < 34) s_hist[threadIdx.x] = 0u;
#pragma unroll
        for (int k = 0; k < PER; ++k) {
            const int t = k * TS_BIN_THREADS + (int)threadIdx.x;
            if (t < f.NT) s_offs[t] = c[k];
        }
        __syncthreads();
        if (scanner) {
            cta_scan_tiles<true>(f, s_offs, s_tmp, total, gmax, sg, s_hist);
            if (sg.tid == 0) s_tot[0] = total, s_tot[1] = gmax;
        }
    } else {
        const volatile TsCtrl* ctrl = f.ctrl;
        nv = ctrl->n_visible, fl = ctrl->flags;
        offs = f.tile_offset;
    }
    const uint32_t nlive = min(nv, f.vis_cap);
    bool synced = !LOCAL;
    for (;; slot += stride) {
        const bool live = !scanner && slot < nlive;
        int tx0 = 0, ty0 = 0, ntx = 0, nty = 0;
        uint4 pa = make_uint4(0u, 0u, slot, 0u);
        uint32_t pb = 0;
        if (live) {
            float4 rec[TS_REC_F4];
            ts_build_record(s0, s1, s2, s2.y, cam, rec);
            // row R3's last float: the face's window smoothness (reading S32; read by the generic-sigma kernels only)
            rec[3].w = face_sigma ? __ldg(face_sigma + __float_as_uint(s3.x)) : sigma_global;
            float4* out = f.rec + TS_REC_F4 * (size_t)slot;
#pragma unroll
            for (int i = 0; i < TS_REC_F4; ++i) out[i] = rec[i];
            const int rlo = __float_as_int(s2.z), rhi = __float_as_int(s2.w);
            const int x0 = (int)(short)(rlo & 0xffff), y0 = rlo >> 16, x1 = (int)(short)(rhi & 0xffff), y1 = rhi >> 16;
            tx0 = x0 >> 4, ty0 = y0 >> 4, ntx = (x1 >> 4) - tx0 + 1, nty = (y1 >> 4) - ty0 + 1;
            pa = make_uint4(__float_as_uint(s3.y), __float_as_uint(s3.x), slot, (uint32_t)rlo);
            pb = (uint32_t)rhi;
        }
        if (!synced) {
            // the offsets are ready from here on; the first scan warp goes on to publish the CTA's share of the tile
            // ranges and job headers (CTA 0: the frame counters too), the other scan warps are done
            __syncthreads();
            synced = true;
            total = s_tot[0], gmax = s_tot[1];
            if (total > f.pair_cap) fl |= TS_FLAG_OVERFLOW_PAIRS;
            if (nv > f.vis_cap) fl |= TS_FLAG_OVERFLOW_VISIBLE;
            if (scanner) {
                if (warp == SLOT_WARPS) publish_slice(f, s_offs, nv, total, gmax, fl, s_hist);
                return;
            }
        }
        const uint32_t nvis = fl ? 0u : nlive;                 // an overflowed frame bins nothing
        const uint32_t n_round = (nvis + 31u) & ~31u;
        if (slot >= n_round) break;                            // warp-uniform
        const int nt = (fl || !live) ? 0 : ntx * nty;
        const bool tight = (f.prm_flags & TS_PARAM_TIGHT_BINNING) != 0;
        const float fu[3] = {s0.x, s0.w, s1.z}, fv[3] = {s0.y, s1.x, s1.w};           // the face's screen vertices
        const int frx0 = (int)(short)(__float_as_int(s2.z) & 0xffff), fry0 = __float_as_int(s2.z) >> 16;
        const int frx1 = (int)(short)(__float_as_int(s2.w) & 0xffff), fry1 = __float_as_int(s2.w) >> 16;
        // narrow faces (the common case): the owning lane scatters its <= 4 pairs itself; the cursor atomics are
        // issued together so that they cost one round trip, not four
        {
            int tt[4];
            uint32_t pos[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                // i < 4 pairs over ntx columns: row = i / ntx by comparisons (an integer division is a subroutine call)
                const int row = (i >= ntx ? 1 : 0) + (i >= 2 * ntx ? 1 : 0) + (i >= 3 * ntx ? 1 : 0);
                tt[i] = (ty0 + row) * f.tiles_x + tx0 + (i - row * ntx);
                pos[i] = 0xffffffffu;
                // (tight binning: only the tiles the triangle meets, by the rule the projection counted with)
                if (nt <= 4 && i < nt && ts_tile_included(tight, fu, fv, frx0, fry0, frx1, fry1, tx0 + (i - row * ntx), ty0 + row))
                    pos[i] = atomicAdd(f.tile_cursor + tt[i], 1u);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (nt <= 4 && i < nt && pos[i] != 0xffffffffu) {
                    const uint32_t q = offs[tt[i]] + pos[i];
                    if (q < f.pair_cap) f.pair_a[q] = pa, f.pair_b[q] = pb;
                }
            }
        }
        // wide faces: their (face, tile) pairs are flattened over the warp, 32 pairs per round trip
        const uint32_t wnt = nt > 4 ? (uint32_t)nt : 0u;
        if (__any_sync(0xffffffffu, wnt != 0u)) {
            uint32_t incl = wnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            const uint32_t W = __shfl_sync(0xffffffffu, incl, 31);
            for (uint32_t p0 = 0; p0 < W; p0 += 32) {
                const uint32_t p = p0 + lane;
                int lo = 0, hi = 31;                            // owner = first lane whose inclusive prefix exceeds p
#pragma unroll
                for (int it = 0; it < 5; ++it) {
                    const int mid = (lo + hi) >> 1;
                    const uint32_t v = __shfl_sync(0xffffffffu, incl, mid);
                    if (v <= p) lo = mid + 1; else hi = mid;
                }
                const int own = lo & 31;
                const uint32_t o_incl = __shfl_sync(0xffffffffu, incl, own), o_nt = __shfl_sync(0xffffffffu, wnt, own);
                const int btx0 = __shfl_sync(0xffffffffu, tx0, own), bty0 = __shfl_sync(0xffffffffu, ty0, own);
                const int bntx = __shfl_sync(0xffffffffu, ntx, own);
                uint4 ba;
                ba.x = __shfl_sync(0xffffffffu, pa.x, own), ba.y = __shfl_sync(0xffffffffu, pa.y, own);
                ba.z = __shfl_sync(0xffffffffu, pa.z, own), ba.w = __shfl_sync(0xffffffffu, pa.w, own);
                const uint32_t bb = __shfl_sync(0xffffffffu, pb, own);
                float wu[3], wv[3];
                if (tight) {                                    // (warp-uniform)
#pragma unroll
                    for (int k = 0; k < 3; ++k) wu[k] = __shfl_sync(0xffffffffu, fu[k], own), wv[k] = __shfl_sync(0xffffffffu, fv[k], own);
                }
                if (p < W) {
                    const int i = (int)(p - (o_incl - o_nt));
                    const int wty = bty0 + i / bntx, wtx = btx0 + i % bntx;
                    const int t = wty * f.tiles_x + wtx;
                    const int wx0 = (int)(short)(ba.w & 0xffffu), wy0 = (int)ba.w >> 16, wx1 = (int)(short)(bb & 0xffffu), wy1 = (int)bb >> 16;
                    if (ts_tile_included(tight, wu, wv, wx0, wy0, wx1, wy1, wtx, wty)) {
                        const uint32_t q = offs[t] + atomicAdd(f.tile_cursor + t, 1u);
                        if (q < f.pair_cap) f.pair_a[q] = ba, f.pair_b[q] = bb;
                    }
                }
            }
        }
        if (slot + stride < nvis) {
            const float4* s4 = f.scr + TS_SCR_F4 * (size_t)(slot + stride);
            s0 = __ldcg(s4), s1 = __ldcg(s4 + 1), s2 = __ldcg(s4 + 2), s3 = __ldcg(s4 + 3);
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
    // (all sizes and strides are powers of two: shifts and masks, no integer division)
    uint32_t lg_hs = 0;
    for (uint32_t size = 2; size <= N; size <<= 1, ++lg_hs) {
        const uint32_t hs = size >> 1;
        for (uint32_t t = threadIdx.x; t < half; t += blockDim.x) {
            const uint32_t blk = t >> lg_hs, off = t & (hs - 1u);
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
        uint32_t lg_st = lg_hs;
        for (uint32_t stride = hs >> 1; stride > 0; stride >>= 1) {
            --lg_st;
            for (uint32_t t = threadIdx.x; t < half; t += blockDim.x) {
                const uint32_t lo = ((t >> lg_st) << (lg_st + 1u)) + (t & (stride - 1u)), hi = lo + stride;
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

__device__ __forceinline__ void emit_sorted(const TsFrameDev& f, uint32_t base, uint32_t rank, uint32_t src,
                                            unsigned long long thi) {
    const uint4 a = f.pair_a[base + src];
    f.sorted[base + rank] = make_uint4(a.z, a.y, a.w, f.pair_b[base + src]);     // (slot, face, rect_lo, rect_hi)
    f.skey[base + rank] = thi | a.x;
}

// Per-block lists (what the render kernels walk).  Once a tile's list [h.y, h.z) is sorted, the group that sorted it
// (one warp, NW = 1, or the whole CTA) goes through it in order and copies every entry to the end of the list of each
// of the tile's eight 8x4 blocks its pixel rect overlaps (ordered compaction: ballots inside a warp, per-warp counts in
// shared memory across the CTA; integer work only -- the exact triangle-vs-block cull stays with the render kernels,
// which have the face records at hand).  Block k of the tile owns blist[8 h.y + k n ...) (n = the tile's list
// length: no allocation, no overflow).  Then the eight job headers of the tile, at the tile's position `p` of
// tile_order.  SRC_SMEM: the sorted entries are in shared memory (the rank sorts leave them there), otherwise they are
// read back from f.sorted.
template <int NW, bool SRC_SMEM>
__device__ __forceinline__ void build_block_lists(const TsFrameDev& f, uint32_t p, const uint4 h, uint32_t gtid,
                                                  uint32_t (*wcnt)[8][NW] /* shared [2][8][NW], NW > 1 only */,
                                                  const uint4* se = nullptr) {
    const uint32_t lane = gtid & 31u, w = gtid >> 5, lt = (1u << lane) - 1u;
    const uint32_t n = h.z - h.y;
    const int tx0 = (int)(h.w & 0xffffu), ty0 = (int)(h.w >> 16);
    uint4* out = f.blist + 8 * (size_t)h.y;
    uint32_t run[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) run[k] = 0u;
    uint32_t par = 0;
    for (uint32_t c = 0; c < n; c += 32u * NW, par ^= 1u) {          // (uniform over the group)
        const uint32_t i = c + gtid;
        uint4 ent = make_uint4(0u, 0u, 0u, 0u);
        uint32_t bits = 0;
        if (i < n) {
            ent = SRC_SMEM ? se[i] : __ldcg(f.sorted + h.y + i);     // (f.sorted: written by this group a moment ago)
            // columns / rows of blocks the rect reaches: x in [tx0 + 8 c, +7], y in [ty0 + 4 r, +3]
            const int x0 = (int)(short)(ent.z & 0xffffu) - tx0, y0 = ((int)ent.z >> 16) - ty0;
            const int x1 = (int)(short)(ent.w & 0xffffu) - tx0, y1 = ((int)ent.w >> 16) - ty0;
            const uint32_t cols = (x0 <= 7 && x1 >= 0 ? 1u : 0u) | (x0 <= 15 && x1 >= 8 ? 2u : 0u);
#pragma unroll
            for (int r = 0; r < 4; ++r)
                if (y0 <= 4 * r + 3 && y1 >= 4 * r) bits |= cols << (2 * r);
        }
        uint32_t bal[8], before[8], mine = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            bal[k] = __ballot_sync(0xffffffffu, (bits >> k) & 1u);
            before[k] = 0u;
            if ((int)lane == k) mine = (uint32_t)__popc(bal[k]);
        }
        if (NW > 1) {
            if (lane < 8u) wcnt[par][lane][w] = mine;
            __syncthreads();
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                uint32_t tot = 0;
#pragma unroll
                for (int ww = 0; ww < NW; ++ww) {
                    const uint32_t cw = wcnt[par][k][ww];
                    if ((uint32_t)ww < w) before[k] += cw;
                    tot += cw;
                }
                bal[k] &= lt;
                before[k] += run[k], run[k] += tot;
            }
        } else {
#pragma unroll
            for (int k = 0; k < 8; ++k) before[k] = run[k], run[k] += (uint32_t)__popc(bal[k]), bal[k] &= lt;
        }
#pragma unroll
        for (int k = 0; k < 8; ++k)
            if ((bits >> k) & 1u) out[(uint32_t)k * n + before[k] + (uint32_t)__popc(bal[k])] = ent;
    }
    if (gtid < 8u) {
        uint32_t cnt = run[0];
#pragma unroll
        for (int k = 1; k < 8; ++k) cnt = gtid == (uint32_t)k ? run[k] : cnt;
        const uint32_t b0 = 8u * h.y + gtid * n;
        f.job_order[8 * (size_t)p + gtid] = make_uint4(h.x | (gtid << 28), b0, b0 + cnt, h.w);
    }
}

// One CTA per position b of the job-header array tile_order (tiles by descending list length, written by the binning
// kernel; every tile appears once).  A LONG list (more than TS_SORT_WARP_MAX pairs) is sorted by the CTA at its own
// position: rank sort up to 2 x threads, compare-exchange network in shared memory up to TS_SORT_SMEM, the same
// network in global scratch above.  SHORT lists (nine in ten at the paper's tracking workloads) are sorted four to a
// CTA by the CTA at the first position of their group of four, ONE WARP per list -- keys in the warp's slice of
// shared memory, rank sort with the pair data in registers, no CTA barrier; the other three CTAs of a short group
// exit at once.  Two dependent loads (header, pairs) precede every sort, whatever its kind.
#define TS_SORT_TILES (TS_SORT_THREADS / 32)
#define TS_SORT_WARP_MAX 64

__global__ void __launch_bounds__(TS_SORT_THREADS) tile_sort_kernel(TsFrameDev f, unsigned long long* __restrict__ gkeys,
                                                                    uint32_t* __restrict__ gidx) {
    __shared__ unsigned long long sk[TS_SORT_SMEM];
    __shared__ uint32_t sv[TS_SORT_SMEM];
    __shared__ uint32_t wcnt[2][8][TS_SORT_THREADS / 32];
    __shared__ uint4 se[2 * TS_SORT_THREADS];               // the sorted entries (rank-sort paths)
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, b = blockIdx.x;
    const bool leader = (b % TS_SORT_TILES) == 0;
    const uint4 hb = __ldcg(f.tile_order + b);              // (tile, begin, end, xy)
    uint4 hw = make_uint4(0u, 0u, 0u, 0u);
    if (leader && b + warp < (uint32_t)f.NT) hw = __ldcg(f.tile_order + b + warp);
    // this kernel is the last reader of the project / binning counters: leave them at zero for the next frame
    if (tid == 0) {
        f.tile_count[hb.x] = 0u, f.tile_cursor[hb.x] = 0u;
        if (b == 0) f.ctrl->vis_counter = 0u;
    }
    if (b == 0 && tid < 32) f.ctrl->bucket_cursor[tid] = 0u;
    const uint32_t nb = hb.z - hb.y;
    if (nb > TS_SORT_WARP_MAX) {
        // ---- a long list: the whole CTA ------------------------------------------------------------------------
        const uint2 range = make_uint2(hb.y, hb.z);
        const uint32_t n = nb;
        const unsigned long long thi = (unsigned long long)hb.x << 32;
        if (n <= 2 * TS_SORT_THREADS) {
            // rank sort, pair data kept in registers: keys are unique (the face index is part of the key), so the
            // ranks are a permutation
            uint4 a[2];
            uint32_t bb[2];
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const uint32_t i = tid + k * TS_SORT_THREADS;
                if (i < n) {
                    a[k] = f.pair_a[range.x + i], bb[k] = f.pair_b[range.x + i];
                    sk[i] = ((unsigned long long)a[k].x << 32) | a[k].y;
                }
            }
            __syncthreads();
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const uint32_t i = tid + k * TS_SORT_THREADS;
                if (i < n) {
                    const unsigned long long mine = ((unsigned long long)a[k].x << 32) | a[k].y;
                    uint32_t rank = 0;
                    for (uint32_t j = 0; j < n; ++j) rank += (sk[j] < mine) ? 1u : 0u;
                    const uint4 ent = make_uint4(a[k].z, a[k].y, a[k].w, bb[k]);            // (slot, face, rect_lo, rect_hi)
                    f.sorted[range.x + rank] = ent;
                    f.skey[range.x + rank] = thi | a[k].x;
                    se[rank] = ent;
                }
            }
            __syncthreads();
            build_block_lists<TS_SORT_THREADS / 32, true>(f, b, hb, tid, wcnt, se);
            if (!leader) return;
            __syncthreads();
            goto short_lists;
        } else if (n <= TS_SORT_SMEM) {
            for (uint32_t i = tid; i < n; i += TS_SORT_THREADS) {
                const uint4 a = f.pair_a[range.x + i];
                sk[i] = ((unsigned long long)a.x << 32) | a.y;
                sv[i] = i;
            }
            __syncthreads();
            cta_sort_network(sk, sv, n);
            for (uint32_t i = tid; i < n; i += TS_SORT_THREADS) emit_sorted(f, range.x, i, sv[i], thi);
        } else {
            // oversize segment: same network in global scratch (volatile: exchanged across threads between barriers)
            unsigned long long* gk = gkeys + range.x;
            uint32_t* gv = gidx + range.x;
            for (uint32_t i = tid; i < n; i += TS_SORT_THREADS) {
                const uint4 a = f.pair_a[range.x + i];
                gk[i] = ((unsigned long long)a.x << 32) | a.y;
                gv[i] = i;
            }
            __syncthreads();
            cta_sort_network((volatile unsigned long long*)gk, (volatile uint32_t*)gv, n);
            for (uint32_t i = tid; i < n; i += TS_SORT_THREADS) emit_sorted(f, range.x, i, gv[i], thi);
        }
        __syncthreads();                                    // the sorted list is complete (and visible to the CTA)
        build_block_lists<TS_SORT_THREADS / 32, false>(f, b, hb, tid, wcnt);
        if (!leader) return;
        __syncthreads();                                    // the shared arrays are re-used below
    }
short_lists:
    if (!leader || b + warp >= (uint32_t)f.NT) return;
    // ---- the group's short lists: one warp each ------------------------------------------------------------------
    const uint32_t n = hw.z - hw.y;
    if (n > TS_SORT_WARP_MAX) return;                       // (sorted by the CTA at its own position)
    if (n == 0) {                                           // an empty tile still has its eight (empty) jobs
        if (lane < 8u) f.job_order[8 * (size_t)(b + warp) + lane] = make_uint4(hw.x | (lane << 28), 0u, 0u, hw.w);
        return;
    }
    unsigned long long* wk = sk + warp * TS_SORT_WARP_MAX;
    uint4* we = se + warp * TS_SORT_WARP_MAX;
    const unsigned long long thi = (unsigned long long)hw.x << 32;
    uint4 a[2];
    uint32_t bb[2];
    unsigned long long mine[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const uint32_t i = lane + 32u * k;
        mine[k] = ~0ull;
        if (i < n) {
            a[k] = f.pair_a[hw.y + i], bb[k] = f.pair_b[hw.y + i];
            mine[k] = ((unsigned long long)a[k].x << 32) | a[k].y;             // (depth key, face): unique
            wk[i] = mine[k];
        }
    }
    __syncwarp();
    uint32_t r0 = 0, r1 = 0;
    for (uint32_t j = 0; j < n; ++j) {
        const unsigned long long kj = wk[j];
        r0 += (kj < mine[0]) ? 1u : 0u, r1 += (kj < mine[1]) ? 1u : 0u;
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const uint32_t i = lane + 32u * k, rank = k ? r1 : r0;
        if (i < n) {
            const uint4 ent = make_uint4(a[k].z, a[k].y, a[k].w, bb[k]);
            f.sorted[hw.y + rank] = ent;
            f.skey[hw.y + rank] = thi | a[k].x;
            we[rank] = ent;
        }
    }
    __syncwarp();
    build_block_lists<1, true>(f, b + warp, hw, lane, nullptr, we);
}

}  // namespace

int32_t ts_launch_sort(const ts_ctx* ctx, ts_frame* fr, cudaStream_t stream) {
    const TsFrameDev& f = fr->d;
    const uint32_t grid_bin = (uint32_t)min((uint64_t)(f.vis_cap + TS_BIN_THREADS - 1) / TS_BIN_THREADS,
                                            (uint64_t)ctx->num_sms);
    if (f.NT <= TS_SCAN_LOCAL_MAX) {
        bin_setup_kernel<true><<<grid_bin, TS_BIN_THREADS, 0, stream>>>(f, fr->cam, fr->face_sigma, fr->prm.sigma);
    } else {
        tile_scan_kernel<<<1, 1024, 0, stream>>>(f);
        bin_setup_kernel<false><<<grid_bin, TS_BIN_THREADS, 0, stream>>>(f, fr->cam, fr->face_sigma, fr->prm.sigma);
    }
    tile_sort_kernel<<<f.NT, TS_SORT_THREADS, 0, stream>>>(f, f.big_key, f.big_idx);
    TS_CUDA_CHECK_LAUNCH();
    return TS_OK;
}
