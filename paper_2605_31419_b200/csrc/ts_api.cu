// ts_api.cu -- the C-ABI boundary (include/ts.h): context, frame workspace carving, status / debug views and
// host-side argument validation for the five hot-path calls.  No device memory is allocated here: the frame lives
// entirely inside caller-provided memory.
#include <new>

#include "ts_internal.cuh"

namespace {

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

struct Layout {
    size_t ctrl, tile_count, tile_cursor, tile_offset, tile_order, tile_ranges, scr, rec, gscr, nrm, gnrm, pair_a, pair_b, big_key, big_idx, skey, sorted, blist, job_order,
        n_contrib, n_contrib_view, t_last,
        pose_partials, total;
    int32_t tiles_x, tiles_y, NT;
    uint32_t n_partials_cap;
};

bool make_layout(const ts_ctx* ctx, int32_t M, int32_t W, int32_t H, uint64_t pair_cap, uint64_t vis_cap, Layout& L) {
    if (!ctx || M <= 0 || W <= 0 || H <= 0 || W > 32767 || H > 32767 || pair_cap == 0 || pair_cap >= (1ull << 28) ||
        vis_cap == 0 || vis_cap >= (1ull << 28) || (uint64_t)M >= (1ull << 28))
        return false;
    L.tiles_x = (W + TS_TILE - 1) / TS_TILE, L.tiles_y = (H + TS_TILE - 1) / TS_TILE, L.NT = L.tiles_x * L.tiles_y;
    L.n_partials_cap = (uint32_t)L.NT * 8u > (uint32_t)ctx->num_sms * 4u ? (uint32_t)L.NT * 8u : (uint32_t)ctx->num_sms * 4u;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes); return r; };
    L.ctrl = take(sizeof(TsCtrl));
    L.tile_count = take(4ull * L.NT);
    L.tile_cursor = take(4ull * L.NT);
    L.tile_offset = take(4ull * L.NT);
    L.tile_order = take(16ull * L.NT);
    L.tile_ranges = take(8ull * L.NT);
    L.scr = take(16ull * TS_SCR_F4 * vis_cap);
    L.rec = take(16ull * TS_REC_F4 * vis_cap);
    L.gscr = take(36ull * vis_cap);
    L.nrm = take(16ull * vis_cap);
    L.gnrm = take(12ull * vis_cap);
    L.pair_a = take(16ull * pair_cap);
    L.pair_b = take(4ull * pair_cap);
    L.big_key = take(8ull * pair_cap);
    L.big_idx = take(4ull * pair_cap);
    L.skey = take(8ull * pair_cap);
    L.sorted = take(16ull * pair_cap);
    L.blist = take(16ull * 8ull * pair_cap);
    L.job_order = take(16ull * 8ull * L.NT);
    L.n_contrib = take(4ull * W * H);
    L.n_contrib_view = take(4ull * W * H);
    L.t_last = take(4ull * W * H);
    L.pose_partials = take(24ull * (L.n_partials_cap + 32u));
    L.total = o;
    return true;
}

}  // namespace

extern "C" {

const char* ts_strerror(int32_t s) {
    switch (s) {
        case TS_OK: return "ok";
        case TS_ERR_INVALID_ARG: return "invalid argument";
        case TS_ERR_WORKSPACE: return "workspace too small or misaligned";
        case TS_ERR_CAPACITY: return "pair / visible-face capacity exceeded";
        case TS_ERR_CUDA: return "CUDA error";
        case TS_ERR_STATE: return "call out of order for this frame";
        case TS_ERR_STATIC_LIMIT:
            return "too large for the built-in workspace of ts_render_fwd_static (more than TS_STATIC_MAX_FACES faces or "
                   "TS_STATIC_MAX_PIXELS pixels): allocate a frame and use ts_project / ts_bin_sort / ts_render_fwd";
        default: return "unknown status";
    }
}

int32_t ts_create(int32_t device, ts_ctx** out) {
    if (!out) return TS_ERR_INVALID_ARG;
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || device < 0 || device >= n) return TS_ERR_CUDA;
    cudaDeviceProp p;
    if (cudaGetDeviceProperties(&p, device) != cudaSuccess) return TS_ERR_CUDA;
    ts_ctx* c = new (std::nothrow) ts_ctx;
    if (!c) return TS_ERR_CUDA;
    c->device = device, c->num_sms = p.multiProcessorCount, c->max_smem_optin = (int)p.sharedMemPerBlockOptin, c->tracing = 0;
    *out = c;
    return TS_OK;
}

int32_t ts_set_tracing(ts_ctx* ctx, int32_t on) {
    if (!ctx) return TS_ERR_INVALID_ARG;
    ctx->tracing = on ? 1 : 0;
    return TS_OK;
}

int32_t ts_destroy(ts_ctx* ctx) {
    delete ctx;
    return TS_OK;
}

size_t ts_frame_bytes(const ts_ctx* ctx, int32_t M, int32_t W, int32_t H, uint64_t pair_capacity,
                      uint64_t visible_capacity) {
    Layout L;
    if (visible_capacity == 0) visible_capacity = (uint64_t)(M > 0 ? M : 0);
    if (!make_layout(ctx, M, W, H, pair_capacity, visible_capacity, L)) return 0;
    return L.total;
}

int32_t ts_frame_bind(ts_ctx* ctx, void* dev_ws, size_t bytes, int32_t M, int32_t W, int32_t H, uint64_t pair_capacity,
                      uint64_t visible_capacity, void* stream, ts_frame** out) {
    TS_TRACE(ctx);
    if (!out || !dev_ws) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    Layout L;
    if (visible_capacity == 0) visible_capacity = (uint64_t)(M > 0 ? M : 0);
    if (!make_layout(ctx, M, W, H, pair_capacity, visible_capacity, L)) return TS_ERR_INVALID_ARG;
    if (bytes < L.total || (reinterpret_cast<uintptr_t>(dev_ws) & 255u)) return TS_ERR_WORKSPACE;
    ts_frame* fr = new (std::nothrow) ts_frame();
    if (!fr) return TS_ERR_CUDA;
    char* b = static_cast<char*>(dev_ws);
    TsFrameDev& d = fr->d;
    d.M = M, d.W = W, d.H = H, d.tiles_x = L.tiles_x, d.tiles_y = L.tiles_y, d.NT = L.NT;
    d.pair_cap = (uint32_t)pair_capacity, d.vis_cap = (uint32_t)visible_capacity;
    d.n_partials_cap = L.n_partials_cap;
    d.ctrl = reinterpret_cast<TsCtrl*>(b + L.ctrl);
    d.tile_count = reinterpret_cast<uint32_t*>(b + L.tile_count);
    d.tile_cursor = reinterpret_cast<uint32_t*>(b + L.tile_cursor);
    d.tile_offset = reinterpret_cast<uint32_t*>(b + L.tile_offset);
    d.tile_order = reinterpret_cast<uint4*>(b + L.tile_order);
    d.tile_ranges = reinterpret_cast<uint2*>(b + L.tile_ranges);
    d.scr = reinterpret_cast<float4*>(b + L.scr);
    d.rec = reinterpret_cast<float4*>(b + L.rec);
    d.gscr = reinterpret_cast<float*>(b + L.gscr);
    d.nrm = reinterpret_cast<float4*>(b + L.nrm);
    d.gnrm = reinterpret_cast<float*>(b + L.gnrm);
    d.pair_a = reinterpret_cast<uint4*>(b + L.pair_a);
    d.pair_b = reinterpret_cast<uint32_t*>(b + L.pair_b);
    d.big_key = reinterpret_cast<unsigned long long*>(b + L.big_key);
    d.big_idx = reinterpret_cast<uint32_t*>(b + L.big_idx);
    d.skey = reinterpret_cast<unsigned long long*>(b + L.skey);
    d.sorted = reinterpret_cast<uint4*>(b + L.sorted);
    d.blist = reinterpret_cast<uint4*>(b + L.blist);
    d.job_order = reinterpret_cast<uint4*>(b + L.job_order);
    d.n_contrib = reinterpret_cast<uint32_t*>(b + L.n_contrib);
    d.n_contrib_view = reinterpret_cast<uint32_t*>(b + L.n_contrib_view);
    d.t_last = reinterpret_cast<float*>(b + L.t_last);
    d.pose_partials = reinterpret_cast<float*>(b + L.pose_partials);
    fr->bytes = L.total, fr->base = dev_ws;
    cudaStream_t st = (cudaStream_t)stream;
    // one-time clears: control block, tile counters / cursors / ranges (contiguous), the zero-at-rest gradient
    // accumulators
    if (cudaMemsetAsync(b + L.ctrl, 0, L.scr - L.ctrl, st) != cudaSuccess ||
        cudaMemsetAsync(b + L.gscr, 0, 36ull * visible_capacity, st) != cudaSuccess ||
        cudaMemsetAsync(b + L.gnrm, 0, 12ull * visible_capacity, st) != cudaSuccess) {
        delete fr;
        return TS_ERR_CUDA;
    }
    *out = fr;
    return TS_OK;
}

int32_t ts_frame_set_face_sigma(ts_ctx* ctx, ts_frame* fr, const float* sigma_dev, float* grad_sigma_dev) {
    if (!ctx || !fr) return TS_ERR_INVALID_ARG;
    if (!sigma_dev && grad_sigma_dev) return TS_ERR_INVALID_ARG;
    fr->face_sigma = sigma_dev, fr->grad_sigma = grad_sigma_dev;
    // the exponent travels in the per-face record, which ts_bin_sort builds: the frame has to be projected and binned again
    fr->have_sort = fr->have_fwd = fr->have_normals = 0;
    return TS_OK;
}

int32_t ts_frame_release(ts_frame* frame) {
    delete frame;
    return TS_OK;
}

int32_t ts_frame_status(ts_ctx* ctx, ts_frame* fr, uint32_t* flags, uint32_t* n_visible, uint64_t* n_pairs, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !fr) return TS_ERR_INVALID_ARG;
    TsCtrl h;
    if (cudaMemcpyAsync(&h, fr->d.ctrl, sizeof(TsCtrl), cudaMemcpyDeviceToHost, (cudaStream_t)stream) != cudaSuccess ||
        cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess)
        return TS_ERR_CUDA;
    if (flags) *flags = h.flags;
    if (n_visible) *n_visible = h.n_visible;
    if (n_pairs) *n_pairs = h.n_pairs;
    return h.flags ? TS_ERR_CAPACITY : TS_OK;
}

int32_t ts_project(ts_ctx* ctx, const ts_scene* sc, const ts_camera* cam, const ts_params* prm, const float* T_cw_dev,
                   ts_frame* fr, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !cam || !prm || !T_cw_dev || !fr || !sc->pos || !sc->opacity) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M || cam->width != fr->d.W || cam->height != fr->d.H) return TS_ERR_INVALID_ARG;
    if (sc->faces == nullptr && sc->V != 3 * sc->M) return TS_ERR_INVALID_ARG;
    if (!(prm->sigma > 0.0f) || !(prm->alpha_min >= 0.0f) || !(prm->t_min >= 0.0f) || !(prm->eps_area >= 0.0f) ||
        !(cam->znear > 0.0f))
        return TS_ERR_INVALID_ARG;
    fr->cam = TsCamDev{cam->width, cam->height, cam->fx, cam->fy, cam->cx, cam->cy, cam->znear};
    fr->prm = TsPrmDev{prm->sigma, prm->alpha_min, prm->t_min, prm->eps_area, prm->flags};
    fr->d.prm_flags = prm->flags;
    fr->T_cw = T_cw_dev;
    fr->have_sort = fr->have_fwd = fr->have_normals = 0;
    fr->pose_src = 0;
    if (fr->counters_dirty) {
        // the previous ts_project was never followed by ts_bin_sort: its slot / tile counters are still live
        char* b = static_cast<char*>(fr->base);
        if (cudaMemsetAsync(b, 0, reinterpret_cast<char*>(fr->d.tile_offset) - b, (cudaStream_t)stream) != cudaSuccess)
            return TS_ERR_CUDA;
    }
    const int32_t s = ts_launch_project(ctx, fr, sc, (cudaStream_t)stream);
    fr->have_project = (s == TS_OK);
    fr->counters_dirty = 1;
    return s;
}

int32_t ts_bin_sort(ts_ctx* ctx, ts_frame* fr, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !fr) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (!fr->have_project) return TS_ERR_STATE;
    if (!fr->counters_dirty) return TS_ERR_STATE;          // one ts_bin_sort per ts_project
    const int32_t s = ts_launch_sort(ctx, fr, (cudaStream_t)stream);
    fr->have_sort = (s == TS_OK);
    fr->counters_dirty = 0;
    return s;
}

int32_t ts_render_fwd(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, float* out_color, float* out_depth,
                      float* out_alpha, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if (!fr->have_sort) return TS_ERR_STATE;
    const int32_t s = ts_launch_render_fwd(ctx, fr, sc, out_color, out_depth, out_alpha, nullptr, nullptr, 0.f, nullptr, nullptr,
                                           nullptr, nullptr, (cudaStream_t)stream);
    fr->have_fwd = (s == TS_OK);
    return s;
}

int32_t ts_render_fwd_l1(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, float* out_color, float* out_depth, float* out_alpha,
                         const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss_dev,
                         void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color || !Chat || !Dhat || !gC || !gD) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if (!fr->have_sort) return TS_ERR_STATE;
    const int32_t s = ts_launch_render_fwd(ctx, fr, sc, out_color, out_depth, out_alpha, Chat, Dhat, lambda_dep, gC, gD, loss_dev,
                                           nullptr, (cudaStream_t)stream);
    fr->have_fwd = (s == TS_OK);
    return s;
}

int32_t ts_render_fwd_stats(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, float* out_color, float* out_depth,
                            float* out_alpha, uint32_t* face_pixels, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color || !face_pixels) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if (!fr->have_sort) return TS_ERR_STATE;
    const int32_t s = ts_launch_render_fwd(ctx, fr, sc, out_color, out_depth, out_alpha, nullptr, nullptr, 0.f, nullptr, nullptr,
                                           nullptr, face_pixels, (cudaStream_t)stream);
    fr->have_fwd = (s == TS_OK);
    return s;
}

int32_t ts_render_fwd_normal(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, float* out_color, float* out_depth,
                             float* out_alpha, float* out_normal, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color || !sc->pos || !out_normal) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if (!fr->have_sort) return TS_ERR_STATE;
    const int32_t s = ts_launch_render_fwd_normal(ctx, fr, sc, out_color, out_depth, out_alpha, out_normal, (cudaStream_t)stream);
    fr->have_fwd = (s == TS_OK);
    fr->have_normals = (s == TS_OK);
    return s;
}

int32_t ts_render_fwd_normal_top(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, float* out_color, float* out_depth,
                                 float* out_alpha, float* out_normal, float* out_normal_top, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color || !sc->pos || !out_normal_top) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if (!fr->have_sort) return TS_ERR_STATE;
    const int32_t s = ts_launch_render_fwd_normal(ctx, fr, sc, out_color, out_depth, out_alpha, out_normal, (cudaStream_t)stream,
                                                  out_normal_top);
    fr->have_fwd = (s == TS_OK);
    fr->have_normals = (s == TS_OK);
    return s;
}

int32_t ts_render_bwd_normal(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, const float* dL_dcolor, const float* dL_ddepth,
                             const float* dL_dalpha, const float* dL_dnormal, float* grad_pos, float* grad_color,
                             float* grad_opacity, uint32_t grad_mask, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color || !sc->pos || !dL_dnormal) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_POS) && !grad_pos) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_COLOR) && !grad_color) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_OPACITY) && !grad_opacity) return TS_ERR_INVALID_ARG;
    if (grad_mask & ~(uint32_t)(TS_GRAD_POS | TS_GRAD_COLOR | TS_GRAD_OPACITY | TS_GRAD_POSE)) return TS_ERR_INVALID_ARG;
    if (!fr->have_fwd || !fr->have_normals) return TS_ERR_STATE;
    return ts_launch_render_bwd_normal(ctx, fr, sc, dL_dcolor, dL_ddepth, dL_dalpha, dL_dnormal, grad_pos, grad_color,
                                       grad_opacity, grad_mask, (cudaStream_t)stream);
}

int32_t ts_face_area(ts_ctx* ctx, ts_frame* fr, float* proj_area, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !fr || !proj_area) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (!fr->have_sort) return TS_ERR_STATE;              // the visible count is published by ts_bin_sort
    return ts_launch_face_area(ctx, fr, proj_area, (cudaStream_t)stream);
}

int32_t ts_render_track_l1(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, float* out_color, float* out_depth, float* out_alpha,
                           const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss_dev,
                           void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color || !Chat || !Dhat) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if (!fr->have_sort) return TS_ERR_STATE;
    fr->have_fwd = 0;                                       // n_contrib / T_last are not written: no ts_render_bwd after this
    return ts_launch_render_track(ctx, fr, sc, out_color, out_depth, out_alpha, Chat, Dhat, lambda_dep, gC, gD, loss_dev,
                                  (cudaStream_t)stream);
}

int32_t ts_render_map_l1(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, float* out_color, float* out_depth, float* out_alpha,
                         const float* Chat, const float* Dhat, float lambda_dep, float* gC, float* gD, float* loss_dev,
                         float* grad_pos, float* grad_color, float* grad_opacity, uint32_t grad_mask, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color || !sc->pos || !Chat || !Dhat) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_POS) && !grad_pos) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_COLOR) && !grad_color) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_OPACITY) && !grad_opacity) return TS_ERR_INVALID_ARG;
    if (grad_mask & ~(uint32_t)(TS_GRAD_POS | TS_GRAD_COLOR | TS_GRAD_OPACITY | TS_GRAD_POSE)) return TS_ERR_INVALID_ARG;
    if (!(grad_mask & (TS_GRAD_POS | TS_GRAD_COLOR | TS_GRAD_OPACITY))) return TS_ERR_INVALID_ARG;   // pose-only: ts_render_track_l1
    if (!fr->have_sort) return TS_ERR_STATE;
    fr->have_fwd = 0;                                       // n_contrib / T_last are not written
    return ts_launch_render_map(ctx, fr, sc, out_color, out_depth, out_alpha, Chat, Dhat, lambda_dep, gC, gD, loss_dev, grad_pos,
                                grad_color, grad_opacity, grad_mask, (cudaStream_t)stream);
}

int32_t ts_render_bwd(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, const float* dL_dcolor, const float* dL_ddepth,
                      const float* dL_dalpha, float* grad_pos, float* grad_color, float* grad_opacity,
                      uint32_t grad_mask, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color || !sc->pos) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_POS) && !grad_pos) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_COLOR) && !grad_color) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_OPACITY) && !grad_opacity) return TS_ERR_INVALID_ARG;
    if (grad_mask & ~(uint32_t)(TS_GRAD_POS | TS_GRAD_COLOR | TS_GRAD_OPACITY | TS_GRAD_POSE)) return TS_ERR_INVALID_ARG;
    if (!fr->have_fwd) return TS_ERR_STATE;
    return ts_launch_render_bwd(ctx, fr, sc, dL_dcolor, dL_ddepth, dL_dalpha, grad_pos, grad_color, grad_opacity,
                                grad_mask, (cudaStream_t)stream);
}

int32_t ts_render_bwd_stats(ts_ctx* ctx, const ts_scene* sc, ts_frame* fr, const float* dL_dcolor, const float* dL_ddepth,
                            const float* dL_dalpha, float* grad_pos, float* grad_color, float* grad_opacity,
                            uint32_t grad_mask, float* face_grad2d, uint32_t* face_views, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !sc || !fr || !sc->color || !sc->pos || !face_grad2d) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    if (sc->M != fr->d.M) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_POS) && !grad_pos) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_COLOR) && !grad_color) return TS_ERR_INVALID_ARG;
    if ((grad_mask & TS_GRAD_OPACITY) && !grad_opacity) return TS_ERR_INVALID_ARG;
    if (grad_mask & ~(uint32_t)(TS_GRAD_POS | TS_GRAD_COLOR | TS_GRAD_OPACITY | TS_GRAD_POSE)) return TS_ERR_INVALID_ARG;
    if (!(grad_mask & (TS_GRAD_POS | TS_GRAD_POSE))) return TS_ERR_INVALID_ARG;      // the statistic is a by-product of B5-B6
    if (!fr->have_fwd) return TS_ERR_STATE;
    return ts_launch_render_bwd(ctx, fr, sc, dL_dcolor, dL_ddepth, dL_dalpha, grad_pos, grad_color, grad_opacity, grad_mask,
                                (cudaStream_t)stream, face_grad2d, face_views);
}

int32_t ts_pose_jacobian_reduce(ts_ctx* ctx, ts_frame* fr, float* dL_dtau_dev, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !fr || !dL_dtau_dev) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    return ts_launch_pose_reduce(ctx, fr, dL_dtau_dev, nullptr, nullptr, nullptr, 0.f, 0.f, 0.f, (cudaStream_t)stream);
}

int32_t ts_pose_reduce_step(ts_ctx* ctx, ts_frame* fr, float* dL_dtau_dev, float* T_cw_dev, float* state_dev,
                            const float* lr6, float beta1, float beta2, float eps, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !fr || !dL_dtau_dev || !T_cw_dev || !state_dev || !lr6) return TS_ERR_INVALID_ARG;
    if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
    return ts_launch_pose_reduce(ctx, fr, dL_dtau_dev, T_cw_dev, state_dev, lr6, beta1, beta2, eps, (cudaStream_t)stream);
}

int32_t ts_frame_view(ts_ctx* ctx, ts_frame* fr, int32_t which, const void** dev_ptr, size_t* count, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !fr || !dev_ptr || !count) return TS_ERR_INVALID_ARG;
    TsCtrl h;
    if (cudaMemcpyAsync(&h, fr->d.ctrl, sizeof(TsCtrl), cudaMemcpyDeviceToHost, (cudaStream_t)stream) != cudaSuccess ||
        cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess)
        return TS_ERR_CUDA;
    const size_t nv = h.flags ? 0 : h.n_visible, np = h.flags ? 0 : h.n_pairs;
    const TsFrameDev& d = fr->d;
    switch (which) {
        case TS_VIEW_VIS: *dev_ptr = d.scr, *count = 16 * nv; break;
        case TS_VIEW_KEYS: *dev_ptr = d.skey, *count = np; break;
        case TS_VIEW_VALS: *dev_ptr = d.sorted, *count = 4 * np; break;
        case TS_VIEW_TILE_RANGES: *dev_ptr = d.tile_ranges, *count = 2 * (size_t)d.NT; break;
        case TS_VIEW_N_CONTRIB: {
            // (the renderers keep block-list positions: converted to positions in the tile's list on demand)
            // only a forward render on the CURRENT sort leaves counts that index its block lists: after ts_bin_sort alone,
            // or after the fused ts_render_track_l1 / ts_render_map_l1 (which do not write them), the counts are those of
            // an older sort
            if (!fr->have_sort || !fr->have_fwd) return TS_ERR_STATE;
            if (!on_ctx_device(ctx)) return TS_ERR_INVALID_ARG;
            if (ts_launch_ncontrib_view(ctx, fr, (cudaStream_t)stream) != TS_OK ||
                cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess)
                return TS_ERR_CUDA;
            *dev_ptr = d.n_contrib_view, *count = (size_t)d.W * d.H;
            break;
        }
        case TS_VIEW_COUNTERS: *dev_ptr = &d.ctrl->counters[0], *count = 8; break;
        case TS_VIEW_JOBS:
            if (!fr->have_sort) return TS_ERR_STATE;
            *dev_ptr = d.job_order, *count = 4 * 8 * (size_t)d.NT;
            break;
        case TS_VIEW_BLOCK_LISTS:
            if (!fr->have_sort) return TS_ERR_STATE;
            *dev_ptr = d.blist, *count = 4 * 8 * np;
            break;
        case TS_VIEW_TIMELINE:
#ifdef TS_JOB_TIMELINE
            if (!fr->have_sort || (size_t)d.W * d.H < 32u * (size_t)d.NT) return TS_ERR_STATE;
            *dev_ptr = d.n_contrib_view, *count = 4 * 8 * (size_t)d.NT;
            break;
#else
            return TS_ERR_STATE;                             // not an instrumented build
#endif
        default: return TS_ERR_INVALID_ARG;
    }
    return TS_OK;
}

}  // extern "C"
