"""ctypes binding of the CPU oracle (oracle/tso.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py may import this module.  It shares no code
with the CUDA path (paper_2605_31419_b200/csrc) and does not import it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from types import SimpleNamespace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtso.so")
_SRC = [os.path.join(_HERE, "tso.cpp"), os.path.join(_HERE, "tso.h")]


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off: no implicit FMA contraction, the float32 path uses explicit fma."""
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-o", _SO, _SRC[0]]
    subprocess.check_call(cmd)
    return _SO


class _Cam(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_double), ("fy", C.c_double),
                ("cx", C.c_double), ("cy", C.c_double), ("znear", C.c_double)]


class _Prm(C.Structure):
    _fields_ = [("sigma", C.c_double), ("alpha_min", C.c_double), ("t_min", C.c_double),
                ("eps_area", C.c_double), ("amb_tol", C.c_double), ("min_opacity", C.c_int32),
                ("tight_binning", C.c_int32), ("face_sigma", C.c_void_p), ("grad_face_sigma", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.tso_project_f32.restype = C.c_int64
        _lib.tso_project_f64.restype = C.c_int64
        _lib.tso_bin_sort.restype = C.c_int64
        _lib.tso_bin_sort_tight_f32.restype = C.c_int64
        _lib.tso_bin_sort_tight_f64.restype = C.c_int64
        _lib.tso_l1_loss_f32.restype = C.c_double
        _lib.tso_l1_loss_f64.restype = C.c_double
        _lib.tso_dssim_f32.restype = C.c_double
        _lib.tso_equi_f32.restype = C.c_double
        _lib.tso_equi_f64.restype = C.c_double
        _lib.tso_dssim_f64.restype = C.c_double
        _lib.tso_normal_loss_f32.restype = C.c_double
        _lib.tso_normal_loss_f64.restype = C.c_double
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _q(prec, x):
    """Quantise python scalars to float32-representable doubles for the f32 oracle."""
    return float(np.float32(x)) if prec == "f32" else float(x)


class Oracle:
    """One view of one scene.  prec = 'f32' (parity) or 'f64' (finite differences / accuracy reference)."""

    def __init__(self, pos, color, opacity, faces, T_cw, cam, params, prec="f32", amb_tol=0.0, face_sigma=None):
        self.prec = prec
        self.dt = np.float32 if prec == "f32" else np.float64
        self.sfx = "_" + prec
        self.pos = np.ascontiguousarray(pos, dtype=self.dt).reshape(-1, 3)
        self.color = np.ascontiguousarray(color, dtype=self.dt).reshape(-1, 3)
        self.opacity = np.ascontiguousarray(opacity, dtype=self.dt).reshape(-1)
        self.faces = None if faces is None else np.ascontiguousarray(faces, dtype=np.int32).reshape(-1, 3)
        self.V = self.pos.shape[0]
        self.M = self.V // 3 if self.faces is None else self.faces.shape[0]
        self.T_cw = np.ascontiguousarray(np.asarray(T_cw)[:3, :4], dtype=self.dt)
        self.W, self.H = int(cam.width), int(cam.height)
        self.cam = _Cam(self.W, self.H, _q(prec, cam.fx), _q(prec, cam.fy), _q(prec, cam.cx), _q(prec, cam.cy),
                        _q(prec, cam.znear))
        self.prm = _Prm(_q(prec, params.sigma), _q(prec, params.alpha_min), _q(prec, params.t_min),
                        _q(prec, params.eps_area), float(amb_tol), int(bool(getattr(params, "min_opacity", False))),
                        int(bool(getattr(params, "tight_binning", False))), None, None)
        # per-face window smoothness (reading S32); its gradient is returned by backward() as grad_sigma
        self.face_sigma = None if face_sigma is None else np.ascontiguousarray(face_sigma, self.dt)
        if self.face_sigma is not None:
            self.prm.face_sigma = self.face_sigma.ctypes.data
        self.tiles_x, self.tiles_y = (self.W + 15) // 16, (self.H + 15) // 16
        self.NT = self.tiles_x * self.tiles_y
        self._proj = None
        self._bins = None

    def _fn(self, name):
        return getattr(lib(), name + self.sfx)

    # ------------------------------------------------------------------ F1-F6
    def project(self):
        if self._proj is None:
            M = self.M
            o = SimpleNamespace(
                visible=np.zeros(M, np.uint8), rect=np.zeros((M, 4), np.int16), depth_key=np.zeros(M, np.uint32),
                tiles_touched=np.zeros(M, np.uint32), scr=np.zeros((M, 9), self.dt), Q=np.zeros((M, 9), self.dt),
                zbar=np.zeros(M, self.dt))
            o.n_visible = self._fn("tso_project")(
                _p(self.pos), _p(self.faces), C.c_int32(self.V), C.c_int32(M), _p(self.T_cw), C.byref(self.cam),
                C.byref(self.prm), _p(o.visible), _p(o.rect), _p(o.depth_key), _p(o.tiles_touched), _p(o.scr),
                _p(o.Q), _p(o.zbar))
            self._proj = o
        return self._proj

    def bin_sort(self):
        """Tiled mode lists.  f32: std::stable_sort on (tile<<32 | float bits).  f64: same tiles, order by the
        double mean depth (then face index) so that finite differences see a consistent order."""
        if self._bins is None:
            pr = self.project()
            P = int(pr.tiles_touched.sum(dtype=np.int64))
            keys = np.zeros(max(P, 1), np.uint64)
            vals = np.zeros(max(P, 1), np.uint32)
            ranges = np.zeros((self.NT, 2), np.uint32)
            if self.prm.tight_binning:
                Pn = self._fn("tso_bin_sort_tight")(C.c_int32(self.M), C.c_int32(self.W), C.c_int32(self.H), _p(pr.visible),
                                                    _p(pr.rect), _p(pr.depth_key), _p(pr.scr), _p(keys), _p(vals), _p(ranges))
            else:
                Pn = lib().tso_bin_sort(C.c_int32(self.M), C.c_int32(self.W), C.c_int32(self.H), _p(pr.visible),
                                        _p(pr.rect), _p(pr.depth_key), _p(pr.tiles_touched), _p(keys), _p(vals),
                                        _p(ranges))
            assert Pn == P
            keys, vals = keys[:P], vals[:P]
            if self.prec == "f64" and P > 0:
                tile = (keys >> np.uint64(32)).astype(np.int64)
                order = np.lexsort((vals, pr.zbar[vals], tile))
                keys, vals = keys[order], vals[order]
            self._bins = SimpleNamespace(P=P, keys=keys, vals=np.ascontiguousarray(vals), ranges=ranges)
        return self._bins

    def global_order(self):
        """Brute mode list: all visible faces in ascending (depth, face index)."""
        pr = self.project()
        ids = np.nonzero(pr.visible)[0].astype(np.uint32)
        k = pr.depth_key[ids] if self.prec == "f32" else pr.zbar[ids]
        return np.ascontiguousarray(ids[np.lexsort((ids, k))])

    def _lists(self, mode):
        if mode == "brute":
            lst = self.global_order()
            return lst, None
        b = self.bin_sort()
        return b.vals, b.ranges

    # ------------------------------------------------------------------ F7-F8
    def forward(self, mode="tiled", color=None, opacity=None):
        pr = self.project()
        lst, ranges = self._lists(mode)
        H, W = self.H, self.W
        o = SimpleNamespace(color=np.zeros((3, H, W), self.dt), depth=np.zeros((H, W), self.dt),
                            alpha=np.zeros((H, W), self.dt), n_contrib=np.zeros((H, W), np.uint32),
                            ambig=np.zeros((H, W), np.uint8), sig=np.zeros((H, W), np.uint64),
                            counters=np.zeros(4, np.uint64))
        col = self.color if color is None else np.ascontiguousarray(color, self.dt)
        opa = self.opacity if opacity is None else np.ascontiguousarray(opacity, self.dt)
        self._fn("tso_render_fwd")(
            _p(col), _p(opa), _p(self.faces), C.c_int32(self.M), C.byref(self.cam), C.byref(self.prm),
            _p(pr.visible), _p(pr.rect), _p(pr.scr), _p(lst), C.c_int64(lst.shape[0]), _p(ranges), _p(o.color),
            _p(o.depth), _p(o.alpha), _p(o.n_contrib), _p(o.ambig), _p(o.sig), _p(o.counters))
        return o

    def face_stats(self, mode="tiled"):
        """Per-face pixel counts and projected areas of this view."""
        pr = self.project()
        lst, ranges = self._lists(mode)
        o = SimpleNamespace(face_pixels=np.zeros(self.M, np.uint32), proj_area=np.zeros(self.M, self.dt))
        self._fn("tso_face_stats")(
            _p(self.color), _p(self.opacity), _p(self.faces), C.c_int32(self.M), C.byref(self.cam), C.byref(self.prm),
            _p(pr.visible), _p(pr.rect), _p(pr.scr), _p(lst), C.c_int64(lst.shape[0]), _p(ranges), _p(o.face_pixels),
            _p(o.proj_area))
        return o

    # ------------------------------------------------------------------ B1-B9
    def backward(self, gC=None, gD=None, gA=None, mode="tiled", want=("pos", "color", "opacity", "pose")):
        pr = self.project()
        lst, ranges = self._lists(mode)
        cv = lambda a: None if a is None else np.ascontiguousarray(a, self.dt)
        gC, gD, gA = cv(gC), cv(gD), cv(gA)
        o = SimpleNamespace()
        o.grad_color = np.zeros_like(self.color) if "color" in want else None
        o.grad_opacity = np.zeros_like(self.opacity) if "opacity" in want else None
        o.g_scr = np.zeros((self.M, 9), self.dt)
        o.grad_sigma = np.zeros(self.M, self.dt) if self.face_sigma is not None else None
        self.prm.grad_face_sigma = None if o.grad_sigma is None else o.grad_sigma.ctypes.data
        self._fn("tso_render_bwd")(
            _p(self.color), _p(self.opacity), _p(self.faces), C.c_int32(self.M), C.byref(self.cam),
            C.byref(self.prm), _p(pr.visible), _p(pr.rect), _p(pr.scr), _p(lst), C.c_int64(lst.shape[0]),
            _p(ranges), _p(gC), _p(gD), _p(gA), _p(o.grad_color), _p(o.grad_opacity), _p(o.g_scr))
        self.prm.grad_face_sigma = None
        o.grad_pos = np.zeros_like(self.pos) if "pos" in want else None
        o.dL_dtau = np.zeros(6, self.dt)
        self._fn("tso_project_bwd")(_p(self.faces), C.c_int32(self.M), _p(self.T_cw), C.byref(self.cam),
                                    _p(pr.visible), _p(pr.Q), _p(o.g_scr), _p(o.grad_pos), _p(o.dL_dtau))
        if "stat" in want:
            o.face_grad2d, o.face_views = np.zeros(self.M, self.dt), np.zeros(self.M, np.uint32)
            self._fn("tso_screen_grad_stat")(C.c_int32(self.M), _p(pr.visible), _p(o.g_scr), _p(o.face_grad2d),
                                             _p(o.face_views))
        return o

    # ------------------------------------------------------------------ normal map (Eq. 12, reading S26)
    def face_normals(self):
        """nrm[M,3]: camera-space unit normals towards the camera (zero for culled faces)."""
        pr = self.project()
        nrm = np.zeros((self.M, 3), self.dt)
        self._fn("tso_face_normal")(_p(self.pos), _p(self.faces), C.c_int32(self.M), _p(self.T_cw), _p(pr.visible),
                                    _p(pr.Q), _p(nrm))
        return nrm

    def normal_forward(self, mode="tiled"):
        pr = self.project()
        lst, ranges = self._lists(mode)
        nrm = self.face_normals()
        N = np.zeros((3, self.H, self.W), self.dt)
        self._fn("tso_render_normal_fwd")(
            _p(self.color), _p(self.opacity), _p(self.faces), C.c_int32(self.M), C.byref(self.cam), C.byref(self.prm),
            _p(pr.visible), _p(pr.rect), _p(pr.scr), _p(lst), C.c_int64(lst.shape[0]), _p(ranges), _p(nrm), _p(N))
        return N

    def normal_top(self, mode="tiled"):
        """Normal of the highest-opacity hit along each ray (Fig. 3 right, reading S29)."""
        pr = self.project()
        lst, ranges = self._lists(mode)
        nrm = self.face_normals()
        N = np.zeros((3, self.H, self.W), self.dt)
        self._fn("tso_render_normal_top")(
            _p(self.color), _p(self.opacity), _p(self.faces), C.c_int32(self.M), C.byref(self.cam), C.byref(self.prm),
            _p(pr.visible), _p(pr.rect), _p(pr.scr), _p(lst), C.c_int64(lst.shape[0]), _p(ranges), _p(nrm), _p(N))
        return N

    def normal_backward(self, gN, mode="tiled", want=("pos", "opacity", "pose")):
        """Gradient of sum(gN * N): grad_pos (window path through B7-B8 plus the normal's own dependence on the
        vertices), grad_opacity, dL_dtau."""
        pr = self.project()
        lst, ranges = self._lists(mode)
        nrm = self.face_normals()
        gN = np.ascontiguousarray(gN, self.dt)
        o = SimpleNamespace()
        o.grad_opacity = np.zeros_like(self.opacity) if "opacity" in want else None
        o.g_scr = np.zeros((self.M, 9), self.dt)
        o.g_nrm = np.zeros((self.M, 3), self.dt)
        self._fn("tso_render_normal_bwd")(
            _p(self.color), _p(self.opacity), _p(self.faces), C.c_int32(self.M), C.byref(self.cam), C.byref(self.prm),
            _p(pr.visible), _p(pr.rect), _p(pr.scr), _p(lst), C.c_int64(lst.shape[0]), _p(ranges), _p(nrm), _p(gN),
            _p(o.grad_opacity), _p(o.g_scr), _p(o.g_nrm))
        o.grad_pos = np.zeros_like(self.pos) if "pos" in want else None
        o.dL_dtau = np.zeros(6, self.dt)
        self._fn("tso_project_bwd")(_p(self.faces), C.c_int32(self.M), _p(self.T_cw), C.byref(self.cam),
                                    _p(pr.visible), _p(pr.Q), _p(o.g_scr), _p(o.grad_pos), _p(o.dL_dtau))
        self._fn("tso_face_normal_bwd")(_p(self.pos), _p(self.faces), C.c_int32(self.M), _p(self.T_cw),
                                        _p(pr.visible), _p(pr.Q), _p(o.g_nrm), _p(o.grad_pos), _p(o.dL_dtau))
        return o

    def l1_loss(self, Cimg, Dimg, Chat, Dhat, lambda_dep):
        cv = lambda a: np.ascontiguousarray(a, self.dt)
        Cimg, Dimg, Chat, Dhat = cv(Cimg), cv(Dimg), cv(Chat), cv(Dhat)
        gC, gD = np.zeros_like(Cimg), np.zeros_like(Dimg)
        L = self._fn("tso_l1_loss")(C.c_int32(self.W), C.c_int32(self.H), _p(Cimg), _p(Dimg), _p(Chat), _p(Dhat),
                                    C.c_double(lambda_dep), _p(gC), _p(gD))
        return L, gC, gD


def equi(pos, faces=None, weight=1.0, prec="f64", grad=True):
    """E_equi (Eq. 14) of a face set; returns (E, weight * dE/dpos or None)."""
    dt = np.float32 if prec == "f32" else np.float64
    pos = np.ascontiguousarray(pos, dt).reshape(-1, 3)
    faces = None if faces is None else np.ascontiguousarray(faces, np.int32).reshape(-1, 3)
    M = pos.shape[0] // 3 if faces is None else faces.shape[0]
    g = np.zeros_like(pos) if grad else None
    E = getattr(lib(), "tso_equi_" + prec)(_p(pos), _p(faces), C.c_int32(M), C.c_double(weight), _p(g))
    return E, g


def normal_loss(N, Nbar, weight=1.0, prec="f64"):
    """weight * E_norm (Eq. 12) of a rendered normal map N [3,H,W] against sensor normals Nbar; returns (L, dL/dN)."""
    dt = np.float32 if prec == "f32" else np.float64
    N, Nbar = np.ascontiguousarray(N, dt), np.ascontiguousarray(Nbar, dt)
    assert N.shape == Nbar.shape and N.ndim == 3 and N.shape[0] == 3
    g = np.zeros_like(N)
    L = getattr(lib(), "tso_normal_loss_" + prec)(C.c_int32(N.shape[2]), C.c_int32(N.shape[1]), _p(N), _p(Nbar),
                                                  C.c_double(weight), _p(g))
    return L, g


def dssim(x, y, prec="f64", grad=True):
    """L_DSSIM = 1 - mean SSIM (Eq. 8) of x (rendered, [3,H,W]) against y; returns (L, dL/dx or None)."""
    dt = np.float32 if prec == "f32" else np.float64
    x, y = np.ascontiguousarray(x, dt), np.ascontiguousarray(y, dt)
    assert x.shape == y.shape and x.ndim == 3 and x.shape[0] == 3
    g = np.zeros_like(x) if grad else None
    L = getattr(lib(), "tso_dssim_" + prec)(C.c_int32(x.shape[2]), C.c_int32(x.shape[1]), _p(x), _p(y), _p(g))
    return L, g


def depth_normalise(D, A, eps=1e-6, prec="f64"):
    dt = np.float32 if prec == "f32" else np.float64
    D, A = np.ascontiguousarray(D, dt), np.ascontiguousarray(A, dt)
    out = np.zeros_like(D)
    ce = C.c_float(eps) if prec == "f32" else C.c_double(eps)
    getattr(lib(), "tso_depth_normalise_" + prec)(C.c_int64(D.size), _p(D), _p(A), ce, _p(out))
    return out


def depth_normalise_bwd(D, A, gDn, eps=1e-6, prec="f64"):
    dt = np.float32 if prec == "f32" else np.float64
    D, A, gDn = (np.ascontiguousarray(x, dt) for x in (D, A, gDn))
    gD, gA = np.zeros_like(D), np.zeros_like(D)
    ce = C.c_float(eps) if prec == "f32" else C.c_double(eps)
    getattr(lib(), "tso_depth_normalise_bwd_" + prec)(C.c_int64(D.size), _p(D), _p(A), ce, _p(gDn), _p(gD), _p(gA))
    return gD, gA


def unpack_rgbd(rgb_u8, depth_u16, depth_scale, prec="f64"):
    """Sensor frame -> the targets of Eq. 8-9 (PAPER.md:74 "RGB-D frames are processed", :125-131; DESIGN.md reading
    S33): rgb_u8 [H][W][3] interleaved 8-bit colour, depth_u16 [H][W] in 1/depth_scale metres (0 = no measurement).
    Chat[c][y][x] = rgb[y][x][c] / 255, Dhat[y][x] = depth[y][x] / depth_scale; one correctly rounded division each
    (plain numpy, no blocking)."""
    dt = np.float32 if prec == "f32" else np.float64
    rgb = np.asarray(rgb_u8)
    dep = np.asarray(depth_u16)
    assert rgb.dtype == np.uint8 and rgb.ndim == 3 and rgb.shape[2] == 3 and dep.dtype == np.uint16 and dep.shape == rgb.shape[:2]
    H, W = dep.shape
    Chat = np.empty((3, H, W), dt)
    for c in range(3):
        Chat[c] = rgb[:, :, c].astype(dt) / dt(255)
    Dhat = dep.astype(dt) / dt(depth_scale)
    return Chat, Dhat


def left_perturb(T_cw, tau):
    T = np.ascontiguousarray(np.asarray(T_cw)[:3, :4], np.float64)
    tau = np.ascontiguousarray(tau, np.float64)
    out = np.zeros((3, 4), np.float64)
    lib().tso_left_perturb_f64(_p(T), _p(tau), _p(out))
    return out


def pose_step_f32(T_cw, g, state, lr, beta1=0.9, beta2=0.999, eps=1e-8):
    T = np.ascontiguousarray(T_cw, np.float32).copy()
    st = np.ascontiguousarray(state, np.float32).copy()
    lib().tso_pose_step_f32(_p(T), _p(np.ascontiguousarray(g, np.float32)), _p(st),
                            _p(np.ascontiguousarray(lr, np.float32)), C.c_float(beta1), C.c_float(beta2),
                            C.c_float(eps))
    return T, st
