// ts_static.cu -- ts_render_fwd_static: the forward render (a1 + a2 + a3) for callers that cannot allocate device memory.
//
// Every kernel of the hot path keeps its intermediate state (visible-face records, tile counters, the binned and sorted
// pair lists, the per-block lists, the per-pixel walk state) in a frame workspace that the CALLER allocates and hands to
// ts_frame_bind.  Some users of this library have no way to produce that buffer once they are running:
//   - a tracking thread with a frame deadline: cudaMalloc / cudaFree take a driver lock, may synchronise the whole
//     device and have no bound on their latency, so such a loop bans them after start-up;
//   - a component living inside a host process whose device memory has all been handed to that process's own arena
//     (an inference server, a simulator): the arena is not ours to carve from, and a cudaMalloc beside it either fails
//     or breaks the host's memory accounting;
//   - a monitoring or preview path that must still draw a thumbnail of the map when HBM is exhausted, i.e. exactly when
//     an allocation would fail.
// For them the workspace lives inside the library image: a file-scope __device__ array of TS_STATIC_WS_BYTES (4 MiB),
// present on every GPU that loads libts.so from module load until the process exits, whether or not it is ever used.
// The entry point below binds a frame onto that array, runs the unchanged projection, binning / sort and compositing
// kernels on it, and drops the (host-side) frame handle again.  It calls no cudaMalloc, cudaFree, cudaMallocAsync or any
// library routine that allocates device memory; the only heap traffic is the few hundred bytes of HOST memory behind the
// frame handle of ts_frame_bind, freed before the call returns.
//
// The array's name is only a handle in host code, not a device address (passing it to a kernel would make the kernel
// read host memory or fault): its address on a given device comes from cudaGetSymbolAddress, asked once per device
// with that device current (static_ws_on_device below), and only that pointer is ever handed to a launch.
#include <mutex>

#include "ts_internal.cuh"

static __device__ __align__(256) unsigned char ts_static_ws[TS_STATIC_WS_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_ws_addr[kMaxDevices];          // device address of ts_static_ws on device d; NULL = not asked yet

// The address of this device's copy of the array.  First use on a device asks the runtime (which may load the module on
// that device: do it before any stream capture starts); later uses read the cached pointer.  `device` is current.
int32_t static_ws_on_device(int device, void** out) {
    if (device < 0 || device >= kMaxDevices) return TS_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_ws_addr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, ts_static_ws);
        if (e != cudaSuccess || p == nullptr) return TS_ERR_CUDA;
        if (reinterpret_cast<uintptr_t>(p) & 255u) return TS_ERR_WORKSPACE;
        g_ws_addr[device] = p;
    }
    *out = g_ws_addr[device];
    return TS_OK;
}

// The largest pair capacity whose frame still fits the array (0 = not even one pair fits).  ts_frame_bytes grows
// monotonically with the capacity, so a bisection over the public size query is enough; host arithmetic only.
uint64_t fitting_pair_capacity(const ts_ctx* ctx, int32_t M, int32_t W, int32_t H) {
    auto fits = [&](uint64_t pc) {
        const size_t b = ts_frame_bytes(ctx, M, W, H, pc, (uint64_t)M);
        return b != 0 && b <= (size_t)TS_STATIC_WS_BYTES;
    };
    if (!fits(1)) return 0;
    uint64_t lo = 1, hi = (uint64_t)TS_STATIC_WS_BYTES / 16u;      // a pair costs far more than 16 B: hi never fits
    while (hi - lo > 1) {
        const uint64_t mid = lo + (hi - lo) / 2;
        if (fits(mid)) lo = mid; else hi = mid;
    }
    return lo;
}

}  // namespace

extern "C" int32_t ts_render_fwd_static(ts_ctx* ctx, const ts_scene* scene, const ts_camera* cam, const ts_params* prm,
                                        const float* T_cw_dev, float* out_color, float* out_depth, float* out_alpha,
                                        uint32_t* status_dev, void* stream) {
    TS_TRACE(ctx);
    if (!ctx || !scene || !cam || !prm || !T_cw_dev || !scene->pos || !scene->color || !scene->opacity)
        return TS_ERR_INVALID_ARG;
    if (scene->M <= 0 || cam->width <= 0 || cam->height <= 0) return TS_ERR_INVALID_ARG;
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != ctx->device) return TS_ERR_INVALID_ARG;
    // the stated maximum, checked before anything touches the device
    if (scene->M > TS_STATIC_MAX_FACES || (int64_t)cam->width * cam->height > TS_STATIC_MAX_PIXELS) return TS_ERR_STATIC_LIMIT;
    const uint64_t pair_cap = fitting_pair_capacity(ctx, scene->M, cam->width, cam->height);
    if (pair_cap == 0) return TS_ERR_STATIC_LIMIT;

    void* ws = nullptr;
    int32_t s = static_ws_on_device(ctx->device, &ws);
    if (s != TS_OK) return s;

    // The array still holds whatever the previous call (of any size) left there.  ts_frame_bind treats its workspace as
    // uninitialised memory and enqueues, on `stream`, the clears of everything a kernel expects to find at zero (control
    // block, tile counters / cursors / ranges, the zero-at-rest accumulators), so a stale array is no different from a
    // fresh allocation.
    ts_frame* fr = nullptr;
    s = ts_frame_bind(ctx, ws, (size_t)TS_STATIC_WS_BYTES, scene->M, cam->width, cam->height, pair_cap, (uint64_t)scene->M,
                      stream, &fr);
    if (s != TS_OK) return s;
    s = ts_project(ctx, scene, cam, prm, T_cw_dev, fr, stream);
    if (s == TS_OK) s = ts_bin_sort(ctx, fr, stream);
    if (s == TS_OK) s = ts_render_fwd(ctx, scene, fr, out_color, out_depth, out_alpha, stream);
    if (s == TS_OK && status_dev) {
        // TsCtrl starts with (n_visible, n_pairs, flags): a device-to-device copy in stream order, no allocation
        if (cudaMemcpyAsync(status_dev, fr->d.ctrl, 3 * sizeof(uint32_t), cudaMemcpyDeviceToDevice, (cudaStream_t)stream) !=
            cudaSuccess)
            s = TS_ERR_CUDA;
    }
    // the launches carry the frame description by value: the host handle is not needed once they are enqueued
    ts_frame_release(fr);
    return s;
}
