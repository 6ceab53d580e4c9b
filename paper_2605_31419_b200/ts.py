"""Thin ctypes binding of libts.so (include/ts.h).  Argument marshalling only: every step of the hot path runs in
the CUDA kernels of paper_2605_31419_b200/csrc.  PyTorch is used for device memory and streams, nothing else.

There is NO CPU fallback: importing this module without a built libts.so raises, and every call on a machine
without a CUDA device fails with TsError.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# TS_LIBTS: path of another build of the same sources (the profiling build of timeline.py); unset = the product library
_SO = os.environ.get("TS_LIBTS") or os.path.join(_HERE, "libts.so")

OK, ERR_INVALID_ARG, ERR_WORKSPACE, ERR_CAPACITY, ERR_CUDA, ERR_STATE, ERR_STATIC_LIMIT = 0, -1, -2, -3, -4, -5, -6
STATIC_WS_BYTES, STATIC_MAX_FACES, STATIC_MAX_PIXELS = 4 << 20, 4096, 16384   # ts_render_fwd_static (include/ts.h)
GRAD_POS, GRAD_COLOR, GRAD_OPACITY, GRAD_POSE = 1, 2, 4, 8
GRAD_ALL = 15
FLAG_OVERFLOW_PAIRS, FLAG_OVERFLOW_VISIBLE = 1, 2
PARAM_COUNTERS = 0x100   # ts_params.flags: count visits / rect tests / hits (debug instantiation)
PARAM_MIN_OPACITY = 0x200   # ts_params.flags: face opacity = min instead of mean of the vertex opacities (ablation)
PARAM_TIGHT_BINNING = 0x400  # ts_params.flags: bin a face only into the tiles its triangle meets (reading S31)
VIEW_VIS, VIEW_KEYS, VIEW_VALS, VIEW_TILE_RANGES, VIEW_N_CONTRIB, VIEW_COUNTERS, VIEW_JOBS, VIEW_BLOCK_LISTS, VIEW_TIMELINE = range(9)
_VIEW_DTYPES = {VIEW_VIS: torch.int32, VIEW_KEYS: torch.int64, VIEW_VALS: torch.int32,
                VIEW_TILE_RANGES: torch.int32, VIEW_N_CONTRIB: torch.int32, VIEW_COUNTERS: torch.int64,
                VIEW_JOBS: torch.int32, VIEW_BLOCK_LISTS: torch.int32, VIEW_TIMELINE: torch.int32}

EXPORTS = ["ts_strerror", "ts_create", "ts_destroy", "ts_frame_bytes", "ts_frame_bind", "ts_frame_release",
           "ts_frame_status", "ts_project", "ts_bin_sort", "ts_render_fwd", "ts_render_fwd_l1", "ts_render_track_l1", "ts_render_map_l1", "ts_render_fwd_stats", "ts_face_area", "ts_render_bwd",
           "ts_render_fwd_normal", "ts_render_bwd_normal", "ts_normal_loss_grad", "ts_render_bwd_stats",
           "ts_pose_jacobian_reduce", "ts_l1_loss_grad", "ts_dssim_loss_grad", "ts_equi_loss_grad", "ts_pose_step", "ts_pose_reduce_step", "ts_frame_view",
           "ts_fp32_probe", "ts_frame_set_face_sigma", "ts_render_fwd_normal_top", "ts_depth_normalise", "ts_depth_normalise_bwd", "ts_unpack_rgbd",
           "ts_render_fwd_static", "ts_set_tracing"]


class TsError(RuntimeError):
    pass


class ts_camera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("znear", C.c_float)]


class ts_params(C.Structure):
    _fields_ = [("sigma", C.c_float), ("alpha_min", C.c_float), ("t_min", C.c_float), ("eps_area", C.c_float),
                ("flags", C.c_uint32)]


class ts_scene(C.Structure):
    _fields_ = [("pos", C.c_void_p), ("color", C.c_void_p), ("opacity", C.c_void_p), ("faces", C.c_void_p),
                ("V", C.c_int32), ("M", C.c_int32)]


def _load():
    if not os.path.exists(_SO):
        raise ImportError(f"{_SO} is missing: build it with `python -m paper_2605_31419_b200.build` "
                          "(nvcc, sm_100a).  There is no CPU fallback.")
    lib = C.CDLL(_SO)
    for name in EXPORTS:
        getattr(lib, name)          # fail loudly on a stale library
    lib.ts_strerror.restype = C.c_char_p
    lib.ts_frame_bytes.restype = C.c_size_t
    lib.ts_frame_bytes.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_uint64, C.c_uint64]
    lib.ts_frame_bind.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_int32, C.c_int32, C.c_int32, C.c_uint64,
                                  C.c_uint64, C.c_void_p, C.POINTER(C.c_void_p)]
    lib.ts_project.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.POINTER(ts_camera), C.POINTER(ts_params),
                               C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_bin_sort.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_render_fwd.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                  C.c_void_p]
    lib.ts_render_fwd_l1.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_render_track_l1.argtypes = lib.ts_render_fwd_l1.argtypes
    lib.ts_render_fwd_stats.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_void_p]
    lib.ts_face_area.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_render_bwd.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                  C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
    lib.ts_render_fwd_normal.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_void_p]
    lib.ts_render_bwd_normal.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
    lib.ts_normal_loss_grad.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p,
                                        C.c_void_p, C.c_void_p]
    lib.ts_render_bwd_stats.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_render_map_l1.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
    lib.ts_pose_jacobian_reduce.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_l1_loss_grad.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_void_p, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_dssim_loss_grad.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p,
                                       C.c_void_p, C.c_void_p]
    lib.ts_equi_loss_grad.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_pose_step.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_float), C.c_float,
                                 C.c_float, C.c_float, C.c_void_p]
    lib.ts_pose_reduce_step.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_float),
                                        C.c_float, C.c_float, C.c_float, C.c_void_p]
    lib.ts_frame_status.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_uint32), C.POINTER(C.c_uint32),
                                    C.POINTER(C.c_uint64), C.c_void_p]
    lib.ts_frame_view.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_void_p), C.POINTER(C.c_size_t),
                                  C.c_void_p]
    lib.ts_render_fwd_normal_top.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                             C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_unpack_rgbd.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_void_p,
                                   C.c_void_p]
    lib.ts_depth_normalise.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_void_p]
    lib.ts_depth_normalise_bwd.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p,
                                           C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_frame_set_face_sigma.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_fp32_probe.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.POINTER(C.c_uint64), C.c_void_p]
    lib.ts_render_fwd_static.argtypes = [C.c_void_p, C.POINTER(ts_scene), C.POINTER(ts_camera), C.POINTER(ts_params), C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ts_frame_release.argtypes = [C.c_void_p]
    lib.ts_destroy.argtypes = [C.c_void_p]
    lib.ts_set_tracing.argtypes = [C.c_void_p, C.c_int32]
    lib.ts_create.argtypes = [C.c_int32, C.POINTER(C.c_void_p)]
    return lib


lib = _load()


def _check(status):
    if status != OK:
        raise TsError(f"libts: {lib.ts_strerror(status).decode()} ({status})")


def _ptr(t, dtype=torch.float32):
    if t is None:
        return None
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise TsError(f"expected a contiguous CUDA tensor of {dtype}, got {t.dtype} on {t.device}")
    return t.data_ptr()


def _stream(stream=None):
    return (stream if stream is not None else torch.cuda.current_stream()).cuda_stream


class Context:
    def __init__(self, device=0):
        h = C.c_void_p()
        _check(lib.ts_create(int(device), C.byref(h)))
        self.h, self.device = h, int(device)

    def set_tracing(self, on=True):
        """NVTX range per ts_* call of this context (off by default)."""
        _check(lib.ts_set_tracing(self.h, 1 if on else 0))

    def close(self):
        if self.h:
            lib.ts_destroy(self.h)
            self.h = None


class Scene:
    """Device-resident map (V, F): pos[V,3], color[V,3], opacity[V] float32; faces[M,3] int32 or None (soup)."""

    def __init__(self, pos, color, opacity, faces=None):
        self.pos, self.color, self.opacity, self.faces = pos, color, opacity, faces
        self.V = int(pos.shape[0])
        self.M = self.V // 3 if faces is None else int(faces.shape[0])
        self.c = ts_scene(_ptr(pos), _ptr(color), _ptr(opacity), _ptr(faces, torch.int32), self.V, self.M)


class Frame:
    """One view's intermediate state; the workspace is a torch uint8 tensor owned here (caller memory for libts)."""

    def __init__(self, ctx, M, W, H, pair_capacity, visible_capacity=0, stream=None):
        self.ctx, self.M, self.W, self.H = ctx, int(M), int(W), int(H)
        n = lib.ts_frame_bytes(ctx.h, self.M, self.W, self.H, int(pair_capacity), int(visible_capacity))
        if n == 0:
            raise TsError("ts_frame_bytes: invalid arguments")
        self.ws = torch.empty(n + 256, dtype=torch.uint8, device=f"cuda:{ctx.device}")
        off = (-self.ws.data_ptr()) % 256
        self.ws_ptr = self.ws.data_ptr() + off
        self.ws_off = off
        h = C.c_void_p()
        _check(lib.ts_frame_bind(ctx.h, self.ws_ptr, n, self.M, self.W, self.H, int(pair_capacity),
                                 int(visible_capacity), _stream(stream), C.byref(h)))
        self.h, self.bytes = h, n

    def release(self):
        if self.h:
            lib.ts_frame_release(self.h)
            self.h = None


def make_camera(cam):
    return ts_camera(int(cam.width), int(cam.height), cam.fx, cam.fy, cam.cx, cam.cy, cam.znear)


def make_params(p, flags=0):
    if getattr(p, "min_opacity", False):
        flags |= PARAM_MIN_OPACITY
    if getattr(p, "tight_binning", False):
        flags |= PARAM_TIGHT_BINNING
    return ts_params(p.sigma, p.alpha_min, p.t_min, p.eps_area, flags)


def ts_project(ctx, scene, cam, prm, T_cw, frame, stream=None):
    _check(lib.ts_project(ctx.h, C.byref(scene.c), C.byref(cam), C.byref(prm), _ptr(T_cw), frame.h, _stream(stream)))


def ts_bin_sort(ctx, frame, stream=None):
    _check(lib.ts_bin_sort(ctx.h, frame.h, _stream(stream)))


def ts_render_fwd(ctx, scene, frame, out_color, out_depth, out_alpha, stream=None):
    _check(lib.ts_render_fwd(ctx.h, C.byref(scene.c), frame.h, _ptr(out_color), _ptr(out_depth), _ptr(out_alpha),
                             _stream(stream)))


def ts_render_fwd_l1(ctx, scene, frame, out_color, out_depth, out_alpha, Chat, Dhat, lambda_dep, gC, gD, loss=None,
                     stream=None):
    _check(lib.ts_render_fwd_l1(ctx.h, C.byref(scene.c), frame.h, _ptr(out_color), _ptr(out_depth), _ptr(out_alpha),
                                _ptr(Chat), _ptr(Dhat), float(lambda_dep), _ptr(gC), _ptr(gD), _ptr(loss), _stream(stream)))


def ts_render_track_l1(ctx, scene, frame, out_color, out_depth, out_alpha, Chat, Dhat, lambda_dep, gC=None, gD=None,
                       loss=None, stream=None):
    _check(lib.ts_render_track_l1(ctx.h, C.byref(scene.c), frame.h, _ptr(out_color), _ptr(out_depth), _ptr(out_alpha),
                                  _ptr(Chat), _ptr(Dhat), float(lambda_dep), _ptr(gC), _ptr(gD), _ptr(loss), _stream(stream)))


def ts_render_fwd_stats(ctx, scene, frame, out_color, out_depth, out_alpha, face_pixels, stream=None):
    _check(lib.ts_render_fwd_stats(ctx.h, C.byref(scene.c), frame.h, _ptr(out_color), _ptr(out_depth), _ptr(out_alpha),
                                   _ptr(face_pixels, torch.int32), _stream(stream)))


def ts_face_area(ctx, frame, proj_area, stream=None):
    _check(lib.ts_face_area(ctx.h, frame.h, _ptr(proj_area), _stream(stream)))


def ts_render_bwd(ctx, scene, frame, dL_dcolor, dL_ddepth, dL_dalpha, grad_pos, grad_color, grad_opacity, grad_mask,
                  stream=None):
    _check(lib.ts_render_bwd(ctx.h, C.byref(scene.c), frame.h, _ptr(dL_dcolor), _ptr(dL_ddepth), _ptr(dL_dalpha),
                             _ptr(grad_pos), _ptr(grad_color), _ptr(grad_opacity), int(grad_mask), _stream(stream)))


def ts_render_fwd_normal(ctx, scene, frame, out_color, out_depth, out_alpha, out_normal, stream=None):
    _check(lib.ts_render_fwd_normal(ctx.h, C.byref(scene.c), frame.h, _ptr(out_color), _ptr(out_depth), _ptr(out_alpha),
                                    _ptr(out_normal), _stream(stream)))


def ts_render_bwd_normal(ctx, scene, frame, dL_dcolor, dL_ddepth, dL_dalpha, dL_dnormal, grad_pos, grad_color,
                         grad_opacity, grad_mask, stream=None):
    _check(lib.ts_render_bwd_normal(ctx.h, C.byref(scene.c), frame.h, _ptr(dL_dcolor), _ptr(dL_ddepth), _ptr(dL_dalpha),
                                    _ptr(dL_dnormal), _ptr(grad_pos), _ptr(grad_color), _ptr(grad_opacity),
                                    int(grad_mask), _stream(stream)))


def ts_normal_loss_grad(ctx, W, H, N, Nbar, weight, gN, loss=None, stream=None):
    _check(lib.ts_normal_loss_grad(ctx.h, int(W), int(H), _ptr(N), _ptr(Nbar), float(weight), _ptr(gN), _ptr(loss),
                                   _stream(stream)))


def ts_render_bwd_stats(ctx, scene, frame, dL_dcolor, dL_ddepth, dL_dalpha, grad_pos, grad_color, grad_opacity, grad_mask,
                        face_grad2d, face_views=None, stream=None):
    _check(lib.ts_render_bwd_stats(ctx.h, C.byref(scene.c), frame.h, _ptr(dL_dcolor), _ptr(dL_ddepth), _ptr(dL_dalpha),
                                   _ptr(grad_pos), _ptr(grad_color), _ptr(grad_opacity), int(grad_mask),
                                   _ptr(face_grad2d), _ptr(face_views, torch.int32), _stream(stream)))


def ts_render_map_l1(ctx, scene, frame, out_color, out_depth, out_alpha, Chat, Dhat, lambda_dep, gC, gD, loss, grad_pos,
                     grad_color, grad_opacity, grad_mask, stream=None):
    _check(lib.ts_render_map_l1(ctx.h, C.byref(scene.c), frame.h, _ptr(out_color), _ptr(out_depth), _ptr(out_alpha),
                                _ptr(Chat), _ptr(Dhat), float(lambda_dep), _ptr(gC), _ptr(gD), _ptr(loss), _ptr(grad_pos),
                                _ptr(grad_color), _ptr(grad_opacity), int(grad_mask), _stream(stream)))


def ts_pose_jacobian_reduce(ctx, frame, dL_dtau, stream=None):
    _check(lib.ts_pose_jacobian_reduce(ctx.h, frame.h, _ptr(dL_dtau), _stream(stream)))


def ts_l1_loss_grad(ctx, W, H, Cimg, Dimg, Chat, Dhat, lambda_dep, gC, gD, loss=None, stream=None):
    _check(lib.ts_l1_loss_grad(ctx.h, int(W), int(H), _ptr(Cimg), _ptr(Dimg), _ptr(Chat), _ptr(Dhat),
                               float(lambda_dep), _ptr(gC), _ptr(gD), _ptr(loss), _stream(stream)))


def ts_dssim_loss_grad(ctx, W, H, Cimg, Chat, lam, gC, loss=None, stream=None):
    _check(lib.ts_dssim_loss_grad(ctx.h, int(W), int(H), _ptr(Cimg), _ptr(Chat), float(lam), _ptr(gC), _ptr(loss),
                                  _stream(stream)))


def ts_equi_loss_grad(ctx, scene, weight, grad_pos, loss=None, stream=None):
    _check(lib.ts_equi_loss_grad(ctx.h, C.byref(scene.c), float(weight), _ptr(grad_pos), _ptr(loss), _stream(stream)))


def ts_pose_step(ctx, T_cw, dL_dtau, state, lr6, beta1=0.9, beta2=0.999, eps=1e-8, stream=None):
    lr = (C.c_float * 6)(*[float(x) for x in lr6])
    _check(lib.ts_pose_step(ctx.h, _ptr(T_cw), _ptr(dL_dtau), _ptr(state), lr, beta1, beta2, eps, _stream(stream)))


def ts_pose_reduce_step(ctx, frame, dL_dtau, T_cw, state, lr6, beta1=0.9, beta2=0.999, eps=1e-8, stream=None):
    lr = (C.c_float * 6)(*[float(x) for x in lr6])
    _check(lib.ts_pose_reduce_step(ctx.h, frame.h, _ptr(dL_dtau), _ptr(T_cw), _ptr(state), lr, beta1, beta2, eps,
                                   _stream(stream)))


def ts_render_fwd_normal_top(ctx, scene, frame, out_color, out_depth, out_alpha, out_normal, out_normal_top, stream=None):
    _check(lib.ts_render_fwd_normal_top(ctx.h, C.byref(scene.c), frame.h, _ptr(out_color), _ptr(out_depth), _ptr(out_alpha),
                                        _ptr(out_normal), _ptr(out_normal_top), _stream(stream)))


def ts_unpack_rgbd(ctx, W, H, rgb, depth, depth_scale, Chat, Dhat, stream=None):
    """rgb: uint8 [H, W, 3]; depth: uint16 (or its int16 bit pattern) [H, W]; both CUDA tensors, or None."""
    if depth is not None and depth.dtype not in (torch.uint16, torch.int16):
        raise TsError("depth must be a 16-bit integer tensor")
    _check(lib.ts_unpack_rgbd(ctx.h, int(W), int(H), _ptr(rgb, torch.uint8), _ptr(depth, depth.dtype if depth is not None else None),
                              float(depth_scale), _ptr(Chat), _ptr(Dhat), _stream(stream)))


def ts_depth_normalise(ctx, W, H, D, A, eps, Dn, stream=None):
    _check(lib.ts_depth_normalise(ctx.h, int(W), int(H), _ptr(D), _ptr(A), float(eps), _ptr(Dn), _stream(stream)))


def ts_depth_normalise_bwd(ctx, W, H, D, A, eps, gDn, gD, gA, stream=None):
    _check(lib.ts_depth_normalise_bwd(ctx.h, int(W), int(H), _ptr(D), _ptr(A), float(eps), _ptr(gDn), _ptr(gD), _ptr(gA),
                                      _stream(stream)))


def ts_render_fwd_static(ctx, scene, cam, prm, T_cw, out_color, out_depth, out_alpha, status=None, stream=None):
    """Forward render of a small view with no Frame and no device allocation inside libts: for callers that must not
    allocate while they run (a real-time tracking loop, a plug-in inside a process whose device memory belongs to the
    host's arena, a preview when HBM is full).  The workspace is a 4 MiB static device array inside libts.so, shared by
    every call on the device: calls that overlap on the GPU race, so keep them on one stream (or order them with
    events).  Limits: scene.M <= STATIC_MAX_FACES, W * H <= STATIC_MAX_PIXELS (TsError "too large for the built-in
    workspace" beyond).  status: int32 CUDA tensor of 3 (n_visible, n_pairs, flags; flags != 0 = pair overflow, the images
    are empty) or None.  The output tensors are the caller's, as everywhere in this binding."""
    _check(lib.ts_render_fwd_static(ctx.h, C.byref(scene.c), C.byref(cam), C.byref(prm), _ptr(T_cw), _ptr(out_color),
                                    _ptr(out_depth), _ptr(out_alpha), _ptr(status, torch.int32), _stream(stream)))


def ts_frame_set_face_sigma(ctx, frame, sigma, grad_sigma=None):
    """Per-face window smoothness [M] (None = the global sigma again) and where dL/dsigma accumulates (may be None).
    The frame keeps the tensors alive."""
    frame._sigma_refs = (sigma, grad_sigma)
    _check(lib.ts_frame_set_face_sigma(ctx.h, frame.h, _ptr(sigma), _ptr(grad_sigma)))


def ts_fp32_probe(ctx, iters, scratch, stream=None):
    """Enqueues the dependent-free FMA loop; returns the flops it performs (time it with events)."""
    fl = C.c_uint64()
    _check(lib.ts_fp32_probe(ctx.h, int(iters), _ptr(scratch), C.byref(fl), _stream(stream)))
    return int(fl.value)


def ts_frame_status(ctx, frame, stream=None, check=True):
    fl, nv, npairs = C.c_uint32(), C.c_uint32(), C.c_uint64()
    st = lib.ts_frame_status(ctx.h, frame.h, C.byref(fl), C.byref(nv), C.byref(npairs), _stream(stream))
    if check:
        _check(st)
    return fl.value, nv.value, npairs.value


def ts_frame_view(ctx, frame, which, stream=None):
    """Copy of an internal array as a torch tensor (debug / bit-exact tests)."""
    p, n = C.c_void_p(), C.c_size_t()
    _check(lib.ts_frame_view(ctx.h, frame.h, int(which), C.byref(p), C.byref(n), _stream(stream)))
    dt = _VIEW_DTYPES[which]
    nbytes = n.value * torch.empty((), dtype=dt).element_size()
    off = (p.value or 0) - frame.ws.data_ptr()
    if nbytes == 0:
        return torch.empty(0, dtype=dt, device=frame.ws.device)
    return frame.ws[off:off + nbytes].view(dt).clone()
