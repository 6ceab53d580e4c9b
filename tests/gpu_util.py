"""Helpers for the -m gpu parity tests: drive the CUDA path through the C-ABI binding and the oracle on the same
seeded inputs, and compare with the tolerances of DESIGN.md section 6."""
import numpy as np
import torch

from paper_2605_31419_b200 import ts

IMG_TOL = 1e-4     # north_star: float32 images, depth and alpha to a relative error of 1e-4
GRAD_TOL = 1e-3    # north_star: gradients to a relative error of 1e-3 (atomic-order differences only)


def dev(a, dtype=torch.float32):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).cuda().contiguous()


class GpuView:
    """One view rendered by libts.  All arguments are numpy; results come back as numpy."""

    def __init__(self, ctx, pos, color, opacity, faces, T_cw, cam, params, pair_capacity=None, visible_capacity=0,
                 flags=0):
        self.ctx = ctx
        self.scene = ts.Scene(dev(pos), dev(color), dev(opacity), None if faces is None else dev(faces, torch.int32))
        self.cam, self.prm = ts.make_camera(cam), ts.make_params(params, flags)
        self.W, self.H = int(cam.width), int(cam.height)
        self.T = dev(np.asarray(T_cw, np.float32)[:3, :4].reshape(-1))
        M = self.scene.M
        self.frame = ts.Frame(ctx, M, self.W, self.H, pair_capacity or max(4 * M, 1024), visible_capacity)
        self.projected = self.sorted = False

    def project(self):
        ts.ts_project(self.ctx, self.scene, self.cam, self.prm, self.T, self.frame)
        self.projected = True
        return self

    def sort(self):
        if not self.projected:
            self.project()
        ts.ts_bin_sort(self.ctx, self.frame)
        self.sorted = True
        return self

    def status(self, check=True):
        return ts.ts_frame_status(self.ctx, self.frame, check=check)

    def view(self, which):
        return ts.ts_frame_view(self.ctx, self.frame, which).cpu().numpy()

    def forward(self):
        if not self.sorted:
            self.sort()
        C = torch.empty(3, self.H, self.W, device="cuda")
        D = torch.empty(self.H, self.W, device="cuda")
        A = torch.empty(self.H, self.W, device="cuda")
        ts.ts_render_fwd(self.ctx, self.scene, self.frame, C, D, A)
        self.C, self.D, self.A = C, D, A
        return C.cpu().numpy(), D.cpu().numpy(), A.cpu().numpy()

    def backward(self, gC, gD, gA, mask=ts.GRAD_ALL):
        V = self.scene.V
        gp = torch.zeros(V, 3, device="cuda") if mask & ts.GRAD_POS else None
        gc = torch.zeros(V, 3, device="cuda") if mask & ts.GRAD_COLOR else None
        go = torch.zeros(V, device="cuda") if mask & ts.GRAD_OPACITY else None
        cv = lambda a: None if a is None else dev(a)
        ts.ts_render_bwd(self.ctx, self.scene, self.frame, cv(gC), cv(gD), cv(gA), gp, gc, go, mask)
        tau = None
        if mask & ts.GRAD_POSE:
            tau = torch.zeros(6, device="cuda")
            ts.ts_pose_jacobian_reduce(self.ctx, self.frame, tau)
        torch.cuda.synchronize()
        n = lambda t: None if t is None else t.cpu().numpy()
        return n(gp), n(gc), n(go), n(tau)

    def close(self):
        self.frame.release()


def scatter_per_face(M, vis_face, arr, fill=0):
    out = np.full((M,) + arr.shape[1:], fill, dtype=arr.dtype)
    out[vis_face] = arr
    return out


def assert_images_close(name, got, ref, ok_mask, scale=1.0, tol=IMG_TOL):
    """|d| <= tol |ref| + tol * scale on every unambiguous pixel and relative L2 <= tol."""
    got, ref = got.astype(np.float64), ref.astype(np.float64)
    m = np.broadcast_to(ok_mask, ref.shape)
    d = np.abs(got - ref)
    bound = tol * np.abs(ref) + tol * scale
    bad = (d > bound) & m
    assert not bad.any(), f"{name}: {bad.sum()} pixels off, worst {d[bad].max():.3e} (bound {bound[bad].min():.3e})"
    nrm = np.linalg.norm(ref[m])
    if nrm > 0:
        assert np.linalg.norm((got - ref)[m]) / nrm <= tol, f"{name}: relative L2 {np.linalg.norm((got - ref)[m]) / nrm:.3e}"


def assert_grad_close(name, got, ref, tol=GRAD_TOL):
    got, ref = got.astype(np.float64), ref.astype(np.float64)
    mx = np.abs(ref).max()
    assert mx > 0, f"{name}: reference gradient is identically zero"
    d = np.abs(got - ref)
    bad = d > tol * np.abs(ref) + tol * mx
    assert not bad.any(), f"{name}: {bad.sum()} entries off, worst {d.max():.3e} vs max|ref| {mx:.3e}"
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert rel <= tol, f"{name}: relative L2 {rel:.3e}"
