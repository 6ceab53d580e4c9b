"""-m gpu parity tests: the CUDA path (through the C ABI) against the float32 oracle on the same seeded inputs.
Integer work (cull set, rects, depth keys, tile counts, sorted keys/vals, tile ranges) must be bit-exact;
images to 1e-4, gradients to 1e-3."""
import numpy as np
import pytest
import torch

from paper_2605_31419_b200 import scenes

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2605_31419_b200 import ts
    c = ts.Context(0)
    yield c
    c.close()


def small_cfg(i):
    """Sizes the oracle finishes in seconds that still span many tiles, several batches and ragged tails."""
    if i == 0:
        return scenes.config0()
    if i == 1:
        return scenes.config1(n_faces=100_000)
    if i == 2:
        return scenes.config2(n_faces=120_000)
    if i == 3:
        return scenes.config3(n_faces=150_000, n_views=2)
    return scenes.config4(n_faces=200_000)


def both(ctx, oracle_mod, sc, view=0, params=None, faces=None, T=None, **kw):
    from gpu_util import GpuView
    prm = params or sc.params
    T = sc.T_start[view] if T is None else T
    o = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, faces, T, sc.cam, prm, "f32", amb_tol=5e-4)
    g = GpuView(ctx, sc.pos, sc.color, sc.opacity, faces, T, sc.cam, prm, **kw)
    return o, g


def check_project_and_sort(o, g, M):
    from gpu_util import scatter_per_face
    from paper_2605_31419_b200 import ts
    g.sort()
    flags, nvis, npairs = g.status()
    pr, b = o.project(), o.bin_sort()
    assert flags == 0 and nvis == pr.n_visible and npairs == b.P
    vis = g.view(ts.VIEW_VIS).reshape(-1, 16)                                  # one 64 B record per slot
    vf = vis[:, 12].view(np.uint32).astype(np.int64)                           # slot -> face (allocation order)
    assert np.array_equal(np.sort(vf), np.nonzero(pr.visible)[0])              # same cull set
    rect = np.ascontiguousarray(vis[:, 10:12]).view(np.int16).reshape(-1, 4)   # x0,y0,x1,y1
    assert np.array_equal(scatter_per_face(M, vf, rect), pr.rect)
    assert np.array_equal(scatter_per_face(M, vf, vis[:, 13].view(np.uint32)), pr.depth_key)
    assert np.array_equal(scatter_per_face(M, vf, vis[:, 14].view(np.uint32)), pr.tiles_touched)
    assert np.array_equal(vis[:, :9].view(np.uint32), pr.scr[vf].view(np.uint32))   # (u,v,w) bit for bit
    assert np.array_equal(g.view(ts.VIEW_KEYS).view(np.uint64), b.keys)
    sv = g.view(ts.VIEW_VALS).reshape(-1, 4).astype(np.int64)                  # sorted (slot, face, rect_lo, rect_hi)
    assert np.array_equal(sv[:, 1], b.vals.astype(np.int64))
    assert np.array_equal(vf[sv[:, 0]], sv[:, 1])
    assert np.array_equal(g.view(ts.VIEW_TILE_RANGES).reshape(-1, 2).view(np.uint32), b.ranges)
    check_block_lists(g, sv, b.ranges.astype(np.int64))


def check_block_lists(g, sv, ranges):
    """The per-block lists the render kernels walk (integer work: exact).  Every tile has eight jobs, one per 8x4
    block; a job's list is the subsequence, in order, of its tile's sorted list whose pixel rect overlaps the block."""
    from paper_2605_31419_b200 import ts
    jobs = g.view(ts.VIEW_JOBS).reshape(-1, 4).view(np.uint32).astype(np.int64)
    bl = g.view(ts.VIEW_BLOCK_LISTS).reshape(-1, 4).astype(np.int64)
    NT = ranges.shape[0]
    assert jobs.shape[0] == 8 * NT
    tile, blk = jobs[:, 0] & 0x0fffffff, jobs[:, 0] >> 28
    assert np.array_equal(np.sort(tile * 8 + blk), np.arange(8 * NT))             # every (tile, block) exactly once
    assert np.array_equal(tile.reshape(-1, 8), np.repeat(tile[::8], 8).reshape(-1, 8))   # a tile's jobs are consecutive
    n_tile = ranges[tile, 1] - ranges[tile, 0]
    assert np.all(np.diff(np.floor(np.log2(np.maximum(n_tile[::8], 1)))) <= 0)          # longest lists first (by log2 bucket)
    x0 = (sv[:, 2] & 0xffff).astype(np.int16).astype(np.int64)
    y0 = sv[:, 2] >> 16
    x1 = (sv[:, 3] & 0xffff).astype(np.int16).astype(np.int64)
    y1 = sv[:, 3] >> 16
    total = 0
    for j in range(jobs.shape[0]):
        tb, te = ranges[tile[j]]
        bx, by = (jobs[j, 3] & 0xffff) + 8 * (blk[j] & 1), (jobs[j, 3] >> 16) + 4 * (blk[j] >> 1)
        s = slice(tb, te)
        keep = (x0[s] <= bx + 7) & (x1[s] >= bx) & (y0[s] <= by + 3) & (y1[s] >= by)
        want = sv[s][keep]
        got = bl[jobs[j, 1]:jobs[j, 2]]
        assert got.shape == want.shape and np.array_equal(got, want), (j, tile[j], blk[j])
        total += want.shape[0]
    assert total >= sv.shape[0]                                                   # every pair is in at least one block


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_project_and_sort_bit_exact(ctx, oracle_mod, cfg):
    sc = small_cfg(cfg)
    o, g = both(ctx, oracle_mod, sc)
    check_project_and_sort(o, g, sc.M)
    g.close()


def check_forward(o, g):
    from gpu_util import assert_images_close
    from paper_2605_31419_b200 import ts
    f = o.forward("tiled")
    C, D, A = g.forward()
    ok = f.ambig == 0
    # pixels where a hit's alpha is within 0.05 % of alpha_min (or T of t_min): the keep/skip decision may differ
    # in the last float32 bit between the two sides (reading N8); they are excluded, and must stay rare
    # (measured: 0 - 22 pixels of 816 000 on the five configs)
    n_amb = int((~ok).sum())
    print(f"ambiguous pixels: {n_amb} of {ok.size}")
    assert n_amb <= 2 + 5e-4 * ok.size, "too many ambiguous pixels"
    # the walk's integer output: list position of the last contributing entry, equal on every unambiguous pixel
    nc = g.view(ts.VIEW_N_CONTRIB).reshape(ok.shape)
    assert np.array_equal(nc[ok], f.n_contrib[ok]), f"n_contrib differs on {(nc[ok] != f.n_contrib[ok]).sum()} pixels"
    assert_images_close("color", C, f.color, ok[None])
    assert_images_close("alpha", A, f.alpha, ok)
    assert_images_close("depth", D, f.depth, ok, scale=float(np.abs(f.depth).max()))
    return f, ok


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_forward_parity(ctx, oracle_mod, cfg):
    sc = small_cfg(cfg)
    o, g = both(ctx, oracle_mod, sc)
    f, ok = check_forward(o, g)
    assert f.alpha.max() > 0.5
    g.close()


def check_backward(o, g, ok, seed, mask_sets):
    from gpu_util import assert_grad_close
    from paper_2605_31419_b200 import ts
    rng = np.random.default_rng(seed)
    H, W = ok.shape
    gC = (rng.normal(size=(3, H, W)) * ok[None]).astype(np.float32)
    gD = (rng.normal(size=(H, W)) * ok).astype(np.float32)
    gA = (rng.normal(size=(H, W)) * ok).astype(np.float32)
    ref = o.backward(gC, gD, gA)
    for mask in mask_sets:
        gp, gc, go, tau = g.backward(gC, gD, gA, mask)
        if mask & ts.GRAD_POS:
            assert_grad_close("grad_pos", gp, ref.grad_pos)
        if mask & ts.GRAD_COLOR:
            assert_grad_close("grad_color", gc, ref.grad_color)
        if mask & ts.GRAD_OPACITY:
            assert_grad_close("grad_opacity", go, ref.grad_opacity)
        if mask & ts.GRAD_POSE:
            assert np.abs(tau - ref.dL_dtau).max() <= 1e-3 * np.abs(ref.dL_dtau).max(), (tau, ref.dL_dtau)
    return ref


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_backward_parity(ctx, oracle_mod, cfg):
    from paper_2605_31419_b200 import ts
    sc = small_cfg(cfg)
    o, g = both(ctx, oracle_mod, sc)
    f, ok = check_forward(o, g)
    check_backward(o, g, ok, 100 + cfg, [ts.GRAD_ALL, ts.GRAD_POSE, ts.GRAD_COLOR | ts.GRAD_OPACITY, ts.GRAD_POS])
    g.close()


@pytest.mark.parametrize("sigma,amin,tmin", [(1.0, 0.0, 0.0), (0.5, 0.0, 0.0), (2.0, 1 / 255, 1e-4), (0.7, 1 / 255, 1e-4)])
def test_sigma_and_threshold_variants(ctx, oracle_mod, sigma, amin, tmin):
    from paper_2605_31419_b200 import ts
    sc = scenes.config0()
    prm = scenes.Params(sigma=sigma, alpha_min=amin, t_min=tmin)
    o, g = both(ctx, oracle_mod, sc, params=prm)
    f, ok = check_forward(o, g)
    check_backward(o, g, ok, 7, [ts.GRAD_ALL])
    g.close()


def test_l1_loss_and_tracking_gradient(ctx, oracle_mod):
    """Config-0 recipe: L1 colour+depth loss against a render of the jittered copy, gradients wrt everything."""
    from gpu_util import assert_grad_close, dev
    from paper_2605_31419_b200 import ts
    sc = scenes.config0()
    tgt = oracle_mod.Oracle(sc.pos_target, sc.color, sc.opacity, None, sc.T_gt[0], sc.cam, sc.params, "f32").forward()
    o, g = both(ctx, oracle_mod, sc)
    f, ok = check_forward(o, g)
    L, gC, gD = o.l1_loss(f.color, f.depth, tgt.color, tgt.depth, sc.params.lambda_dep)
    gCd, gDd, loss = torch.empty_like(g.C), torch.empty_like(g.D), torch.zeros(1, device="cuda")
    ts.ts_l1_loss_grad(ctx, g.W, g.H, dev(f.color), dev(f.depth), dev(tgt.color), dev(tgt.depth), sc.params.lambda_dep,
                       gCd, gDd, loss)
    assert np.array_equal(gCd.cpu().numpy(), gC) and np.array_equal(gDd.cpu().numpy(), gD)
    assert abs(loss.item() - L) <= 1e-5 * L
    ref = o.backward(gC, gD, None)
    gp, gc, go, tau = g.backward(gC, gD, None, ts.GRAD_ALL)
    assert_grad_close("grad_pos", gp, ref.grad_pos)
    assert_grad_close("grad_color", gc, ref.grad_color)
    assert_grad_close("grad_opacity", go, ref.grad_opacity)
    assert np.abs(tau - ref.dL_dtau).max() <= 1e-3 * np.abs(ref.dL_dtau).max()
    g.close()


def test_pose_step_matches_oracle(ctx, oracle_mod):
    from gpu_util import dev
    from paper_2605_31419_b200 import ts
    rng = np.random.default_rng(3)
    T = scenes.look_level((0.3, -0.2, 0.0), 0.6).astype(np.float32)
    state = np.zeros(13, np.float32)
    lr = [1e-3] * 3 + [3e-3] * 3
    Td, sd = dev(T.reshape(-1)), dev(state)
    for it in range(5):
        gvec = rng.normal(size=6).astype(np.float32)
        T, state = oracle_mod.pose_step_f32(T, gvec, state, lr)
        ts.ts_pose_step(ctx, Td, dev(gvec), sd, lr)
        assert np.allclose(Td.cpu().numpy().reshape(3, 4), T, atol=2e-6)
        assert np.allclose(sd.cpu().numpy(), state, rtol=1e-5, atol=1e-7)


def test_pose_reduce_step_equals_separate_calls(ctx, oracle_mod):
    """ts_pose_reduce_step (a7 + a8 fused) gives the same gradient and the same updated pose as the two calls."""
    from gpu_util import dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(1)
    o, g = both(ctx, oracle_mod, sc)
    C, D, A = g.forward()
    rng = np.random.default_rng(11)
    gC, gD = dev(rng.normal(size=C.shape).astype(np.float32)), dev(rng.normal(size=D.shape).astype(np.float32))
    lr = [1e-3] * 3 + [3e-3] * 3
    res = []
    for fused in (False, True):
        T, st, tau = g.T.clone(), torch.zeros(13, device="cuda"), torch.zeros(6, device="cuda")
        ts.ts_render_bwd(ctx, g.scene, g.frame, gC, gD, None, None, None, None, ts.GRAD_POSE)
        if fused:
            ts.ts_pose_reduce_step(ctx, g.frame, tau, T, st, lr)
        else:
            ts.ts_pose_jacobian_reduce(ctx, g.frame, tau)
            ts.ts_pose_step(ctx, T, tau, st, lr)
        torch.cuda.synchronize()
        res.append((tau.cpu().numpy(), T.cpu().numpy(), st.cpu().numpy()))
    for a, b in zip(*res):
        assert np.array_equal(a, b)
    assert np.abs(res[0][0]).max() > 0
    g.close()


def test_render_fwd_l1_equals_separate_calls(ctx, oracle_mod):
    """ts_render_fwd_l1 (a3 + a4 fused) writes the same images and cotangents as ts_render_fwd + ts_l1_loss_grad."""
    from gpu_util import dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(2)
    o, g = both(ctx, oracle_mod, sc)
    C, D, A = g.forward()
    rng = np.random.default_rng(5)
    Chat = dev(np.clip(C + rng.normal(0, 0.05, C.shape), 0, 1).astype(np.float32))
    Dhat = dev((D * (rng.uniform(size=D.shape) > 0.2) * rng.uniform(0.9, 1.1, D.shape)).astype(np.float32))
    gC1, gD1, L1 = torch.empty_like(g.C), torch.empty_like(g.D), torch.zeros(1, device="cuda")
    ts.ts_l1_loss_grad(ctx, g.W, g.H, g.C, g.D, Chat, Dhat, 0.05, gC1, gD1, L1)
    C2, D2, A2 = torch.empty_like(g.C), torch.empty_like(g.D), torch.empty_like(g.A)
    gC2, gD2, L2 = torch.empty_like(g.C), torch.empty_like(g.D), torch.zeros(1, device="cuda")
    ts.ts_render_fwd_l1(ctx, g.scene, g.frame, C2, D2, A2, Chat, Dhat, 0.05, gC2, gD2, L2)
    torch.cuda.synchronize()
    assert torch.equal(C2, g.C) and torch.equal(D2, g.D) and torch.equal(A2, g.A)
    assert torch.equal(gC1, gC2) and torch.equal(gD1, gD2)
    assert abs(L1.item() - L2.item()) <= 1e-5 * abs(L1.item()) and L1.item() > 0
    # outputs are optional in the fused call
    ts.ts_render_fwd_l1(ctx, g.scene, g.frame, None, None, None, Chat, Dhat, 0.05, gC2, gD2, None)
    torch.cuda.synchronize()
    assert torch.equal(gC1, gC2) and torch.equal(gD1, gD2)
    g.close()


def fused_cotangents_agree(gC, gD, gCo, gDo, ok):
    """The L1 sign images of the CUDA path (from its own render) and of the oracle (from its own) may differ only where
    abs(C - Chat) is within float rounding: they must agree on >= 99.9 % of the unambiguous pixels."""
    same = (gC == gCo).all(axis=0) & (gD == gDo)
    frac = same[ok].mean() if ok.any() else 1.0
    print(f"L1 cotangent images agree on {100 * frac:.4f} % of the unambiguous pixels")
    assert frac >= 0.999
    return same


@pytest.mark.parametrize("cfg", [0, 1, 2, 4])
def test_render_track_l1_equals_separate_calls(ctx, oracle_mod, cfg):
    """ts_render_track_l1 (a3 + a4 + a5 pose-only fused) == ts_render_fwd_l1 + ts_render_bwd(POSE): images, loss
    cotangents and the pose gradient bit for bit (same arithmetic); and its pose gradient matches the oracle's, fed with
    the same cotangent images, to 1e-3."""
    from gpu_util import dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(cfg)
    o, g = both(ctx, oracle_mod, sc)
    f, ok = check_forward(o, g)
    # a target that differs from the render: the ground-truth pose where the config has a start pose, else jittered vertices
    tgt_pos = sc.pos_target if sc.pos_target is not None else sc.pos
    tgt = oracle_mod.Oracle(tgt_pos, sc.color, sc.opacity, None, sc.T_gt[0], sc.cam, sc.params, "f32").forward("tiled")
    Chat, Dhat = dev(tgt.color), dev(tgt.depth)
    lam = sc.params.lambda_dep
    gC, gD, L1 = torch.empty_like(g.C), torch.empty_like(g.D), torch.zeros(1, device="cuda")
    ts.ts_render_fwd_l1(ctx, g.scene, g.frame, None, None, None, Chat, Dhat, lam, gC, gD, L1)
    ts.ts_render_bwd(ctx, g.scene, g.frame, gC, gD, None, None, None, None, ts.GRAD_POSE)
    tau1 = torch.zeros(6, device="cuda")
    ts.ts_pose_jacobian_reduce(ctx, g.frame, tau1)
    cx = ctx
    C2, D2, A2 = torch.empty_like(g.C), torch.empty_like(g.D), torch.empty_like(g.A)
    gC2, gD2, L2 = torch.empty_like(g.C), torch.empty_like(g.D), torch.zeros(1, device="cuda")
    ts.ts_render_track_l1(cx, g.scene, g.frame, C2, D2, A2, Chat, Dhat, lam, gC2, gD2, L2)
    tau2 = torch.zeros(6, device="cuda")
    ts.ts_pose_jacobian_reduce(cx, g.frame, tau2)
    torch.cuda.synchronize()
    assert torch.equal(C2, g.C) and torch.equal(D2, g.D) and torch.equal(A2, g.A)
    assert torch.equal(gC, gC2) and torch.equal(gD, gD2)
    assert tau1.abs().max().item() > 0
    assert torch.equal(tau1, tau2)
    assert abs(L1.item() - L2.item()) <= 1e-5 * abs(L1.item())
    # against the oracle: its own loss cotangents agree with the kernel's on (nearly) every pixel, and its backward pass
    # of the kernel's cotangent images gives the kernel's pose gradient to 1e-3
    Lo, gCo, gDo = o.l1_loss(f.color, f.depth, tgt.color, tgt.depth, lam)
    gCn, gDn = gC2.cpu().numpy(), gD2.cpu().numpy()
    fused_cotangents_agree(gCn, gDn, gCo, gDo, ok)
    assert abs(L2.item() - Lo) <= 1e-4 * abs(Lo)
    ref = o.backward(gCn, gDn, None, want=("pose",))
    t2 = tau2.cpu().numpy()
    assert np.abs(t2 - ref.dL_dtau).max() <= 1e-3 * np.abs(ref.dL_dtau).max(), (t2, ref.dL_dtau)
    with pytest.raises(ts.TsError):
        ts.ts_render_bwd(ctx, g.scene, g.frame, gC, gD, None, None, None, None, ts.GRAD_POSE)   # no walk state after track
    g.close()


def test_mapping_step_accumulates_over_views(ctx, oracle_mod):
    """Config-3 recipe at a small size: one mapping step = fwd+bwd over the keyframes, per-vertex gradients
    ACCUMULATED (+=) over the views into the same buffers; compared with the sum of the oracle's."""
    from gpu_util import GpuView, assert_grad_close, dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(3)
    V = sc.pos.shape[0]
    gp, gc, go = torch.zeros(V, 3, device="cuda"), torch.zeros(V, 3, device="cuda"), torch.zeros(V, device="cuda")
    ref_p, ref_c, ref_o = np.zeros((V, 3)), np.zeros((V, 3)), np.zeros(V)
    rng = np.random.default_rng(33)
    for view in range(len(sc.T_start)):
        T = sc.T_start[view]
        o = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, None, T, sc.cam, sc.params, "f32", amb_tol=5e-4)
        g = GpuView(ctx, sc.pos, sc.color, sc.opacity, None, T, sc.cam, sc.params)
        f, ok = check_forward(o, g)
        H, W = ok.shape
        gC = (rng.normal(size=(3, H, W)) * ok[None]).astype(np.float32)
        gD = (rng.normal(size=(H, W)) * ok).astype(np.float32)
        ref = o.backward(gC, gD, None)
        ref_p += ref.grad_pos
        ref_c += ref.grad_color
        ref_o += ref.grad_opacity
        ts.ts_render_bwd(ctx, g.scene, g.frame, dev(gC), dev(gD), None, gp, gc, go,
                         ts.GRAD_POS | ts.GRAD_COLOR | ts.GRAD_OPACITY)
        torch.cuda.synchronize()
        g.close()
    assert_grad_close("grad_pos", gp.cpu().numpy(), ref_p)
    assert_grad_close("grad_color", gc.cpu().numpy(), ref_c)
    assert_grad_close("grad_opacity", go.cpu().numpy(), ref_o)


@pytest.mark.parametrize("cfg", [0, 2, 4])
def test_face_statistics_match_the_oracle(ctx, oracle_mod, cfg):
    """ts_render_fwd_stats / ts_face_area against the oracle's per-face pixel counts and projected areas: areas bit
    for bit; pixel counts equal wherever no keep / skip decision was within rounding (N8), and never off by more than
    the number of ambiguous pixels."""
    from paper_2605_31419_b200 import ts
    sc = small_cfg(cfg)
    o, g = both(ctx, oracle_mod, sc)
    g.sort()
    M, H, W = sc.M, g.H, g.W
    C, D, A = torch.empty(3, H, W, device="cuda"), torch.empty(H, W, device="cuda"), torch.empty(H, W, device="cuda")
    fp, area = torch.zeros(M, dtype=torch.int32, device="cuda"), torch.zeros(M, device="cuda")
    ts.ts_render_fwd_stats(ctx, g.scene, g.frame, C, D, A, fp)
    ts.ts_face_area(ctx, g.frame, area)
    torch.cuda.synchronize()
    f, st = o.forward("tiled"), o.face_stats("tiled")
    assert np.array_equal(area.cpu().numpy().view(np.uint32), st.proj_area.view(np.uint32))
    got, ref = fp.cpu().numpy().astype(np.int64), st.face_pixels.astype(np.int64)
    n_amb = int((f.ambig != 0).sum())
    assert np.abs(got - ref).sum() <= 4 * n_amb and got.sum() > 0
    if n_amb == 0:
        assert np.array_equal(got, ref)
    # the statistics instantiation renders the same image
    C2 = torch.empty_like(C)
    ts.ts_render_fwd(ctx, g.scene, g.frame, C2, None, None)
    torch.cuda.synchronize()
    assert torch.equal(C, C2)
    g.close()


@pytest.mark.parametrize("W,H", [(64, 48), (50, 37), (131, 70), (1200, 680)])
def test_dssim_loss_and_gradient(ctx, oracle_mod, W, H):
    """ts_dssim_loss_grad against the oracle's D-SSIM (Eq. 8): lambda * L and (1 - lambda) gC + lambda dL/dC."""
    from gpu_util import assert_grad_close, dev
    from paper_2605_31419_b200 import ts
    rng = np.random.default_rng(W)
    yy, xx = np.mgrid[0:H, 0:W]
    base = 0.5 + 0.4 * np.sin(0.3 * xx + 0.2 * yy)[None] * np.array([1.0, 0.7, -0.5])[:, None, None]
    x = np.clip(base + rng.normal(0, 0.05, (3, H, W)), 0, 1).astype(np.float32)
    y = np.clip(base + rng.normal(0, 0.05, (3, H, W)), 0, 1).astype(np.float32)
    lam = 0.2
    g_l1 = rng.normal(size=(3, H, W)).astype(np.float32) / (3 * H * W)
    L64, g64 = oracle_mod.dssim(x, y, "f64")
    L32, g32 = oracle_mod.dssim(x, y, "f32")
    gC, loss = dev(g_l1), torch.zeros(1, device="cuda")
    ts.ts_dssim_loss_grad(ctx, W, H, dev(x), dev(y), lam, gC, loss)
    torch.cuda.synchronize()
    assert abs(loss.item() - lam * L64) <= 2e-5 * lam * L64
    got = gC.cpu().numpy()
    assert_grad_close("dssim grad vs f64 oracle", got, (1 - lam) * g_l1.astype(np.float64) + lam * g64)
    assert_grad_close("dssim grad vs f32 oracle", got, (1 - lam) * g_l1 + lam * g32)
    # lambda = 0 leaves the L1 cotangent untouched
    gC0 = dev(g_l1)
    ts.ts_dssim_loss_grad(ctx, W, H, dev(x), dev(y), 0.0, gC0, None)
    torch.cuda.synchronize()
    assert np.array_equal(gC0.cpu().numpy(), g_l1)


def test_tracking_gradient_with_full_photometric_loss(ctx, oracle_mod):
    """E_track = (1 - lambda) L1 + lambda L_DSSIM + lambda_dep E_dep (Eq. 8-10, lambda = 0.2,
    lambda_dep = 0.05): ts_render_fwd -> ts_l1_loss_grad -> ts_dssim_loss_grad -> ts_render_bwd(pose-only) ->
    ts_pose_jacobian_reduce against the same chain through the oracle."""
    from gpu_util import dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(1)
    lam, lam_dep = 0.2, sc.params.lambda_dep
    tgt = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_gt[0], sc.cam, sc.params, "f32").forward("tiled")
    o, g = both(ctx, oracle_mod, sc)
    f, ok = check_forward(o, g)
    # oracle chain (on the oracle's own forward images)
    L1, gC, gD = o.l1_loss(f.color, f.depth, tgt.color, tgt.depth, lam_dep)
    Ls, gS = oracle_mod.dssim(f.color, tgt.color, "f32")
    gC_o = ((1 - lam) * gC + lam * gS) * ok[None]
    ref = o.backward(gC_o.astype(np.float32), (gD * ok).astype(np.float32), None, want=("pose",))
    # CUDA chain
    H, W = g.H, g.W
    gCd, gDd = torch.empty_like(g.C), torch.empty_like(g.D)
    ts.ts_l1_loss_grad(ctx, W, H, g.C, g.D, dev(tgt.color), dev(tgt.depth), lam_dep, gCd, gDd, None)
    ts.ts_dssim_loss_grad(ctx, W, H, g.C, dev(tgt.color), lam, gCd, None)
    okd = dev(ok.astype(np.float32))
    gCd *= okd[None]
    gDd *= okd
    ts.ts_render_bwd(ctx, g.scene, g.frame, gCd, gDd, None, None, None, None, ts.GRAD_POSE)
    tau = torch.zeros(6, device="cuda")
    ts.ts_pose_jacobian_reduce(ctx, g.frame, tau)
    torch.cuda.synchronize()
    t = tau.cpu().numpy()
    # the two cotangent images: equal L1 sign part on (nearly) every pixel (it can flip where |C - Chat| is within
    # float rounding between the two forwards), D-SSIM part to the gradient tolerance
    gCn, gDn = gCd.cpu().numpy(), gDd.cpu().numpy()
    close = (np.abs(gCn - gC_o) <= 1e-3 * np.abs(gC_o).max()).all(axis=0) & (gDn == (gD * ok))
    assert close[ok].mean() >= 0.999, close[ok].mean()
    # the backward pass proper: both sides get the SAME cotangent images (the CUDA chain's), gradient to 1e-3
    ref_same = o.backward(gCn, gDn, None, want=("pose",))
    assert np.abs(t - ref_same.dL_dtau).max() <= 1e-3 * np.abs(ref_same.dL_dtau).max(), (t, ref_same.dL_dtau)
    # and the whole chain end to end (each side on its own cotangents) stays within the few flipped pixels
    assert np.abs(t - ref.dL_dtau).max() <= 5e-3 * np.abs(ref.dL_dtau).max(), (t, ref.dL_dtau)
    g.close()


@pytest.mark.parametrize("indexed", [False, True])
def test_equi_regulariser(ctx, oracle_mod, indexed):
    """ts_equi_loss_grad against the oracle's E_equi (Eq. 14): value and gradient, soup and shared vertices."""
    from gpu_util import assert_grad_close, dev
    from paper_2605_31419_b200 import ts
    rng = np.random.default_rng(4)
    if indexed:
        pos = rng.normal(size=(500, 3)).astype(np.float32)
        faces = rng.integers(0, 500, size=(3000, 3)).astype(np.int32)
        faces = faces[(faces[:, 0] != faces[:, 1]) & (faces[:, 1] != faces[:, 2]) & (faces[:, 0] != faces[:, 2])]
    else:
        pos, faces = scenes.config0(n_faces=3000).pos, None
    w = 0.37
    E, g = oracle_mod.equi(pos, faces, weight=w, prec="f64")
    scene = ts.Scene(dev(pos), dev(np.zeros_like(pos)), dev(np.zeros(pos.shape[0], np.float32)),
                     None if faces is None else dev(faces, torch.int32))
    gp, loss = torch.zeros(pos.shape[0], 3, device="cuda"), torch.zeros(1, device="cuda")
    ts.ts_equi_loss_grad(ctx, scene, w, gp, loss)
    torch.cuda.synchronize()
    assert abs(loss.item() - w * E) <= 1e-5 * w * E
    assert_grad_close("equi grad", gp.cpu().numpy(), g)


def needle_scene():
    """Config-4 soup re-indexed so that every second face borrows a vertex of the previous face in the array -- which
    lies anywhere in the room: thousands of needle-shaped faces hundreds of pixels long and a fraction of a pixel to a
    few pixels wide (perimeter / inradius up to 1e5), the case note N11 of DESIGN.md is about."""
    sc = small_cfg(4)
    rng = np.random.default_rng(5)
    n_face = 60_000
    faces = np.arange(3 * n_face, dtype=np.int32).reshape(-1, 3)
    share = rng.random(n_face) < 0.5
    faces[1:][share[1:], 0] = faces[:-1][share[1:], 1]
    return sc, sc.pos[: 3 * n_face], sc.color[: 3 * n_face], sc.opacity[: 3 * n_face], faces


def grid_mesh(n=40, seed=21):
    """A shared-vertex height-field mesh (2 (n-1)^2 faces on n^2 vertices): every vertex collects the gradients of up to
    six faces."""
    rng = np.random.default_rng(seed)
    gx, gy = np.meshgrid(np.linspace(-1.3, 1.3, n), np.linspace(-1.0, 1.0, n))
    pos = np.stack([gx, gy, 3.0 + 0.3 * np.sin(3 * gx) * np.cos(2 * gy)], axis=-1).reshape(-1, 3)
    pos += rng.normal(0, 0.006, pos.shape)
    idx = np.arange(n * n).reshape(n, n)
    f1 = np.stack([idx[:-1, :-1], idx[:-1, 1:], idx[1:, :-1]], axis=-1).reshape(-1, 3)
    f2 = np.stack([idx[1:, 1:], idx[1:, :-1], idx[:-1, 1:]], axis=-1).reshape(-1, 3)
    faces = np.concatenate([f1, f2]).astype(np.int32)
    sc = scenes.config0(n_faces=10)
    sc.params = scenes.Params(sigma=0.5)
    return (sc, pos.astype(np.float32), rng.uniform(0, 1, (n * n, 3)).astype(np.float32),
            rng.uniform(0.3, 1.0, n * n).astype(np.float32), faces)


def test_needle_faces(ctx, oracle_mod):
    """Faces far outside the paper's size range (needles hundreds of pixels long): images still to 1e-4 and per-vertex
    gradients to 1e-3 (relative L2), because such faces are evaluated on the compensated path everywhere (N11)."""
    from gpu_util import GpuView, assert_grad_close
    from paper_2605_31419_b200 import ts
    sc, pos, col, opa, faces = needle_scene()
    o = oracle_mod.Oracle(pos, col, opa, faces, sc.T_start[0], sc.cam, sc.params, "f32", amb_tol=5e-4)
    g = GpuView(ctx, pos, col, opa, faces, sc.T_start[0], sc.cam, sc.params, pair_capacity=o.bin_sort().P + 1024)
    f, ok = check_forward(o, g)
    assert (f.alpha > 0.5).mean() > 0.5
    rng = np.random.default_rng(77)
    H, W = ok.shape
    gC = (rng.normal(size=(3, H, W)) * ok[None]).astype(np.float32)
    gD = (rng.normal(size=(H, W)) * ok).astype(np.float32)
    ref = o.backward(gC, gD, None)
    gp, gc, go, tau = g.backward(gC, gD, None, ts.GRAD_ALL)
    assert_grad_close("grad_color", gc, ref.grad_color)
    assert_grad_close("grad_opacity", go, ref.grad_opacity)
    # Vertex positions and pose of needles: d x / d q grows like 1/r, and so does the rounding of ANY float32 evaluation
    # of the geometry terms.  The bound is therefore taken from the arithmetic itself (SURVEY.md pin P14: the float32
    # oracle against the float64 oracle on the same inputs sets the achievable floor): relative L2 to 1e-3 as everywhere,
    # single entries to max(1e-3, 2 x that floor).  (measured floor: ~1.5e-3 for grad_pos, ~2e-3 for the pose, whose
    # components are sums of 1e6-sized terms of both signs)
    o64 = oracle_mod.Oracle(pos, col, opa, faces, sc.T_start[0], sc.cam, sc.params, "f64")
    ref64 = o64.backward(gC.astype(np.float64), gD.astype(np.float64), None)
    floor_pos = np.abs(ref.grad_pos - ref64.grad_pos).max() / np.abs(ref64.grad_pos).max()
    floor_tau = np.abs(ref.dL_dtau - ref64.dL_dtau).max() / np.abs(ref64.dL_dtau).max()
    print(f"needles: float32-vs-float64 oracle floor grad_pos {floor_pos:.2e}, pose {floor_tau:.2e}")
    d = np.abs(gp.astype(np.float64) - ref.grad_pos)
    assert np.linalg.norm(d) <= 1e-3 * np.linalg.norm(ref.grad_pos)
    assert d.max() <= max(1e-3, 2 * floor_pos) * np.abs(ref.grad_pos).max()
    assert np.abs(tau - ref.dL_dtau).max() <= max(1e-3, 2 * floor_tau) * np.abs(ref.dL_dtau).max(), (tau, ref.dL_dtau)
    g.close()


@pytest.mark.parametrize("cfg", [0, 2, 3, "mesh"])
def test_normal_map_forward_and_backward(ctx, oracle_mod, cfg):
    """ts_render_fwd_normal / ts_render_bwd_normal (Eq. 12) against the oracle: the normal map to the
    image tolerance, colour / depth / alpha bit-identical to ts_render_fwd, and ONE backward pass for the cotangents of
    all four outputs against the sum of the oracle's colour/depth/alpha backward and its normal backward."""
    from gpu_util import assert_grad_close, assert_images_close, dev
    from paper_2605_31419_b200 import ts
    if cfg == "mesh":
        sc, pos, col, opa, faces = grid_mesh()
    else:
        sc = small_cfg(cfg)
        pos, col, opa, faces = sc.pos, sc.color, sc.opacity, None
    o = oracle_mod.Oracle(pos, col, opa, faces, sc.T_start[0], sc.cam, sc.params, "f32", amb_tol=5e-4)
    from gpu_util import GpuView
    g = GpuView(ctx, pos, col, opa, faces, sc.T_start[0], sc.cam, sc.params)
    f, ok = check_forward(o, g)
    H, W = ok.shape
    C, D, A = torch.empty(3, H, W, device="cuda"), torch.empty(H, W, device="cuda"), torch.empty(H, W, device="cuda")
    N = torch.empty(3, H, W, device="cuda")
    ts.ts_render_fwd_normal(ctx, g.scene, g.frame, C, D, A, N)
    torch.cuda.synchronize()
    assert torch.equal(C, g.C) and torch.equal(D, g.D) and torch.equal(A, g.A)
    Nref = o.normal_forward("tiled")
    assert np.abs(Nref).max() > 0.5
    assert_images_close("normal", N.cpu().numpy(), Nref, ok[None])
    # outputs other than the normal map are optional
    N2 = torch.empty_like(N)
    ts.ts_render_fwd_normal(ctx, g.scene, g.frame, None, None, None, N2)
    torch.cuda.synchronize()
    assert torch.equal(N, N2)

    rng = np.random.default_rng(700 + (9 if cfg == "mesh" else cfg))
    gC = (rng.normal(size=(3, H, W)) * ok[None]).astype(np.float32)
    gD = (rng.normal(size=(H, W)) * ok).astype(np.float32)
    gA = (rng.normal(size=(H, W)) * ok).astype(np.float32)
    gN = (rng.normal(size=(3, H, W)) * ok[None]).astype(np.float32)
    r1, r2 = o.backward(gC, gD, gA), o.normal_backward(gN)
    V = pos.shape[0]
    for mask in (ts.GRAD_ALL, ts.GRAD_POS, ts.GRAD_POSE, ts.GRAD_OPACITY | ts.GRAD_COLOR):
        gp, gc, go = torch.zeros(V, 3, device="cuda"), torch.zeros(V, 3, device="cuda"), torch.zeros(V, device="cuda")
        ts.ts_render_bwd_normal(ctx, g.scene, g.frame, dev(gC), dev(gD), dev(gA), dev(gN), gp, gc, go, mask)
        if mask & ts.GRAD_POS:
            assert_grad_close("grad_pos", gp.cpu().numpy(), r1.grad_pos + r2.grad_pos)
        if mask & ts.GRAD_COLOR:
            assert_grad_close("grad_color", gc.cpu().numpy(), r1.grad_color)
        if mask & ts.GRAD_OPACITY:
            assert_grad_close("grad_opacity", go.cpu().numpy(), r1.grad_opacity + r2.grad_opacity)
        if mask & ts.GRAD_POSE:
            tau = torch.zeros(6, device="cuda")
            ts.ts_pose_jacobian_reduce(ctx, g.frame, tau)
            ref = r1.dL_dtau + r2.dL_dtau
            assert np.abs(tau.cpu().numpy() - ref).max() <= 1e-3 * np.abs(ref).max(), (tau, ref)
    # the normal cotangent alone (E_norm is the only loss on N): d<gN, N>
    gp, go = torch.zeros(V, 3, device="cuda"), torch.zeros(V, device="cuda")
    ts.ts_render_bwd_normal(ctx, g.scene, g.frame, None, None, None, dev(gN), gp, None, go,
                            ts.GRAD_POS | ts.GRAD_OPACITY | ts.GRAD_POSE)
    tau = torch.zeros(6, device="cuda")
    ts.ts_pose_jacobian_reduce(ctx, g.frame, tau)
    assert_grad_close("grad_pos (normal only)", gp.cpu().numpy(), r2.grad_pos)
    assert_grad_close("grad_opacity (normal only)", go.cpu().numpy(), r2.grad_opacity)
    assert np.abs(tau.cpu().numpy() - r2.dL_dtau).max() <= 1e-3 * np.abs(r2.dL_dtau).max()
    # the frame's accumulators are back at rest: a plain backward afterwards is unaffected
    gp2 = torch.zeros(V, 3, device="cuda")
    ts.ts_render_bwd(ctx, g.scene, g.frame, dev(gC), dev(gD), dev(gA), gp2, None, None, ts.GRAD_POS)
    assert_grad_close("grad_pos (after)", gp2.cpu().numpy(), r1.grad_pos)
    g.close()


def test_normal_calls_need_their_forward(ctx, oracle_mod):
    from gpu_util import GpuView, dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(0)
    g = GpuView(ctx, sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, sc.params)
    g.forward()
    gN = torch.zeros(3, g.H, g.W, device="cuda")
    gp = torch.zeros(sc.pos.shape[0], 3, device="cuda")
    with pytest.raises(ts.TsError):
        ts.ts_render_bwd_normal(ctx, g.scene, g.frame, None, None, None, gN, gp, None, None, ts.GRAD_POS)
    with pytest.raises(ts.TsError):
        ts.ts_render_fwd_normal(ctx, g.scene, g.frame, None, None, None, None)
    g.close()


def test_mapping_objective_gradient(ctx, oracle_mod):
    """One view of E_map = E_pho + lambda_dep E_dep + lambda_norm E_norm + lambda_equi E_equi (Eq. 15, PAPER.md:165-167;
    weights of Table S4) at the config-3 recipe: ts_render_fwd_normal -> ts_l1_loss_grad ->
    ts_dssim_loss_grad -> ts_normal_loss_grad -> ts_render_bwd_normal -> ts_equi_loss_grad, against the same chain
    through the oracle.  The target colour / depth / sensor normals are rendered from the unperturbed scene."""
    from gpu_util import assert_grad_close, dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(3)
    lam, lam_dep, lam_norm, lam_equi = 0.2, 0.05, 0.05, 1.2
    T = sc.T_start[0]
    gt = oracle_mod.Oracle(sc.pos_target, sc.color_target, sc.opacity, None, T, sc.cam, sc.params, "f32")
    tgt, Ngt = gt.forward("tiled"), gt.normal_forward("tiled")
    seen = tgt.alpha > 0.2                                  # (150 k faces cover the small case only sparsely)
    Nbar = np.where(seen[None], Ngt / np.maximum(np.linalg.norm(Ngt, axis=0), 1e-12)[None], 0.0).astype(np.float32)
    assert seen.mean() > 0.15 and (~seen).sum() > 0         # there are pixels without a sensor normal as well
    o, g = both(ctx, oracle_mod, sc)
    f, ok = check_forward(o, g)
    H, W, V = g.H, g.W, sc.pos.shape[0]
    # oracle chain, on the oracle's own images
    No = o.normal_forward("tiled")
    L1, gC, gD = o.l1_loss(f.color, f.depth, tgt.color, tgt.depth, lam_dep)
    Ls, gS = oracle_mod.dssim(f.color, tgt.color, "f32")
    Ln, gN = oracle_mod.normal_loss(No, Nbar, lam_norm, "f32")
    Le, gE = oracle_mod.equi(sc.pos, None, lam_equi, "f32")
    gC_o = (((1 - lam) * gC + lam * gS) * ok[None]).astype(np.float32)
    r1 = o.backward(gC_o, (gD * ok).astype(np.float32), None)
    r2 = o.normal_backward((gN * ok[None]).astype(np.float32))
    ref_pos = r1.grad_pos + r2.grad_pos + gE
    ref_opa = r1.grad_opacity + r2.grad_opacity
    # CUDA chain
    C, D, A = torch.empty(3, H, W, device="cuda"), torch.empty(H, W, device="cuda"), torch.empty(H, W, device="cuda")
    N = torch.empty(3, H, W, device="cuda")
    gCd, gDd, gNd = torch.empty_like(C), torch.empty_like(D), torch.empty_like(N)
    loss = torch.zeros(1, device="cuda")
    gp, gc, go = torch.zeros(V, 3, device="cuda"), torch.zeros(V, 3, device="cuda"), torch.zeros(V, device="cuda")
    ts.ts_render_fwd_normal(ctx, g.scene, g.frame, C, D, A, N)
    ts.ts_l1_loss_grad(ctx, W, H, C, D, dev(tgt.color), dev(tgt.depth), lam_dep, gCd, gDd, None)
    ts.ts_dssim_loss_grad(ctx, W, H, C, dev(tgt.color), lam, gCd, None)
    ts.ts_normal_loss_grad(ctx, W, H, N, dev(Nbar), lam_norm, gNd, loss)
    okd = dev(ok.astype(np.float32))
    gCd *= okd[None]
    gDd *= okd
    gNd *= okd[None]
    ts.ts_render_bwd_normal(ctx, g.scene, g.frame, gCd, gDd, None, gNd, gp, gc, go, ts.GRAD_POS | ts.GRAD_COLOR | ts.GRAD_OPACITY)
    ts.ts_equi_loss_grad(ctx, g.scene, lam_equi, gp, None)
    torch.cuda.synchronize()
    assert abs(float(loss.item()) - Ln) <= 1e-4 * abs(Ln) + 1e-7
    # the backward pass proper: both sides get the SAME cotangent images (the CUDA chain's; its L1 sign image can differ
    # from the oracle's where |C - Chat| is within float rounding between the two forwards), gradients to 1e-3
    s1 = o.backward(gCd.cpu().numpy(), gDd.cpu().numpy(), None)
    s2 = o.normal_backward(gNd.cpu().numpy())
    assert_grad_close("grad_pos", gp.cpu().numpy(), s1.grad_pos + s2.grad_pos + gE)
    assert_grad_close("grad_color", gc.cpu().numpy(), s1.grad_color)
    assert_grad_close("grad_opacity", go.cpu().numpy(), s1.grad_opacity + s2.grad_opacity)
    # and the whole chain end to end (each side on its own cotangents) stays within the few flipped pixels
    assert np.linalg.norm(gp.cpu().numpy() - ref_pos) <= 5e-3 * np.linalg.norm(ref_pos)
    assert np.linalg.norm(go.cpu().numpy() - ref_opa) <= 5e-3 * np.linalg.norm(ref_opa)
    # and the normal term alone, whose cotangent does not depend on a sign image, to the gradient tolerance
    gp2, go2 = torch.zeros(V, 3, device="cuda"), torch.zeros(V, device="cuda")
    ts.ts_render_bwd_normal(ctx, g.scene, g.frame, None, None, None, gNd, gp2, None, go2, ts.GRAD_POS | ts.GRAD_OPACITY)
    torch.cuda.synchronize()
    assert_grad_close("grad_pos (E_norm)", gp2.cpu().numpy(), r2.grad_pos)
    assert_grad_close("grad_opacity (E_norm)", go2.cpu().numpy(), r2.grad_opacity)
    g.close()


@pytest.mark.parametrize("indexed", [False, True])
def test_min_opacity_variant(ctx, oracle_mod, indexed):
    """TS_PARAM_MIN_OPACITY ("+ min opacity" ablation, PAPER.md:82 and Table S3): images and all gradients against the
    oracle in the same mode; the opacity gradient lands on one vertex per face; and the mode does change the image."""
    from gpu_util import GpuView
    from paper_2605_31419_b200 import ts
    if indexed:
        sc, pos, col, opa, faces = grid_mesh(n=30, seed=4)
    else:
        sc = small_cfg(2)
        pos, col, opa, faces = sc.pos, sc.color, sc.opacity, None
    prm = scenes.Params(sigma=sc.params.sigma, alpha_min=sc.params.alpha_min, t_min=sc.params.t_min, min_opacity=True)
    o = oracle_mod.Oracle(pos, col, opa, faces, sc.T_start[0], sc.cam, prm, "f32", amb_tol=5e-4)
    g = GpuView(ctx, pos, col, opa, faces, sc.T_start[0], sc.cam, prm)
    f, ok = check_forward(o, g)
    ref = check_backward(o, g, ok, 91, [ts.GRAD_ALL, ts.GRAD_POSE])
    if not indexed:
        tri = opa.reshape(-1, 3)
        not_min = (tri != tri.min(axis=1, keepdims=True)).reshape(-1)
        assert np.all(ref.grad_opacity[not_min] == 0)
    g2 = GpuView(ctx, pos, col, opa, faces, sc.T_start[0], sc.cam, sc.params)
    A_mean = g2.forward()[2]
    assert np.abs(A_mean - g.A.cpu().numpy()).max() > 0.05
    g.close(), g2.close()


@pytest.mark.parametrize("cfg", [0, 2])
def test_screen_gradient_statistic(ctx, oracle_mod, cfg):
    """ts_render_bwd_stats (densification statistic, reading S28) against the oracle's; gradients are the
    same as ts_render_bwd's; accumulation over two calls; the pose still comes out with TS_GRAD_POSE alone."""
    from gpu_util import assert_grad_close, dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(cfg)
    o, g = both(ctx, oracle_mod, sc)
    f, ok = check_forward(o, g)
    rng = np.random.default_rng(55 + cfg)
    H, W = ok.shape
    gC = (rng.normal(size=(3, H, W)) * ok[None]).astype(np.float32)
    gD = (rng.normal(size=(H, W)) * ok).astype(np.float32)
    ref = o.backward(gC, gD, None, want=("pos", "pose", "stat"))
    V, M = sc.pos.shape[0], sc.M
    gp = torch.zeros(V, 3, device="cuda")
    st, views = torch.zeros(M, device="cuda"), torch.zeros(M, dtype=torch.int32, device="cuda")
    ts.ts_render_bwd_stats(ctx, g.scene, g.frame, dev(gC), dev(gD), None, gp, None, None, ts.GRAD_POS, st, views)
    torch.cuda.synchronize()
    assert_grad_close("grad_pos", gp.cpu().numpy(), ref.grad_pos)
    assert_grad_close("face_grad2d", st.cpu().numpy(), ref.face_grad2d)
    # a face "received a gradient" iff any of its nine screen terms is non-zero: the same set up to faces whose only
    # contributions sit on ambiguous pixels (zeroed cotangents on both sides)
    assert (views.cpu().numpy().astype(np.int64) != ref.face_views).sum() <= 2 + 1e-3 * M
    assert views.sum().item() > 0
    # second call: accumulates; pose-only mask goes through the full-gradient path and still leaves dL/dtau
    ts.ts_render_bwd_stats(ctx, g.scene, g.frame, dev(gC), dev(gD), None, None, None, None, ts.GRAD_POSE, st, None)
    tau = torch.zeros(6, device="cuda")
    ts.ts_pose_jacobian_reduce(ctx, g.frame, tau)
    torch.cuda.synchronize()
    assert_grad_close("face_grad2d x2", st.cpu().numpy(), 2 * ref.face_grad2d)
    assert np.abs(tau.cpu().numpy() - ref.dL_dtau).max() <= 1e-3 * np.abs(ref.dL_dtau).max()
    with pytest.raises(ts.TsError):
        ts.ts_render_bwd_stats(ctx, g.scene, g.frame, dev(gC), None, None, None, None, None, ts.GRAD_COLOR, st, None)
    g.close()


@pytest.mark.parametrize("cfg", [0, 3, 4])
def test_render_map_l1_equals_separate_calls(ctx, oracle_mod, cfg):
    """ts_render_map_l1 (a3 + a4 + a5 full-gradient + a6 fused) against ts_render_fwd_l1 + ts_render_bwd: images, loss
    cotangents bit for bit; per-vertex gradients and the pose to the order of the float atomics; every mask shape."""
    from gpu_util import assert_grad_close, dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(cfg)
    o, g = both(ctx, oracle_mod, sc)
    f, ok = check_forward(o, g)
    tgt_pos = sc.pos_target if sc.pos_target is not None else sc.pos
    tgt_col = sc.color_target if sc.color_target is not None else sc.color
    tgt = oracle_mod.Oracle(tgt_pos, tgt_col, sc.opacity, None, sc.T_gt[0], sc.cam, sc.params, "f32").forward("tiled")
    Chat, Dhat = dev(tgt.color), dev(tgt.depth)
    lam, V = sc.params.lambda_dep, sc.pos.shape[0]
    z3, z1 = (lambda: torch.zeros(V, 3, device="cuda")), (lambda: torch.zeros(V, device="cuda"))
    gC, gD, L1 = torch.empty_like(g.C), torch.empty_like(g.D), torch.zeros(1, device="cuda")
    gp1, gc1, go1 = z3(), z3(), z1()
    ts.ts_render_fwd_l1(ctx, g.scene, g.frame, None, None, None, Chat, Dhat, lam, gC, gD, L1)
    ts.ts_render_bwd(ctx, g.scene, g.frame, gC, gD, None, gp1, gc1, go1, ts.GRAD_ALL)
    tau1 = torch.zeros(6, device="cuda")
    ts.ts_pose_jacobian_reduce(ctx, g.frame, tau1)
    C2, D2, A2 = torch.empty_like(g.C), torch.empty_like(g.D), torch.empty_like(g.A)
    gC2, gD2, L2 = torch.empty_like(g.C), torch.empty_like(g.D), torch.zeros(1, device="cuda")
    gp2, gc2, go2 = z3(), z3(), z1()
    ts.ts_render_map_l1(ctx, g.scene, g.frame, C2, D2, A2, Chat, Dhat, lam, gC2, gD2, L2, gp2, gc2, go2, ts.GRAD_ALL)
    tau2 = torch.zeros(6, device="cuda")
    ts.ts_pose_jacobian_reduce(ctx, g.frame, tau2)
    torch.cuda.synchronize()
    assert torch.equal(C2, g.C) and torch.equal(D2, g.D) and torch.equal(A2, g.A)
    assert torch.equal(gC, gC2) and torch.equal(gD, gD2)
    assert abs(L1.item() - L2.item()) <= 1e-5 * abs(L1.item())
    n = lambda t: t.cpu().numpy()
    assert_grad_close("grad_pos", n(gp2), n(gp1), tol=2e-5)
    assert_grad_close("grad_color", n(gc2), n(gc1), tol=2e-5)
    assert_grad_close("grad_opacity", n(go2), n(go1), tol=2e-5)
    assert np.abs(n(tau2) - n(tau1)).max() <= 1e-4 * np.abs(n(tau1)).max()
    # partial masks; accumulation (+=) into the same buffers
    ts.ts_render_map_l1(ctx, g.scene, g.frame, None, None, None, Chat, Dhat, lam, None, None, None, gp2, None, None, ts.GRAD_POS)
    ts.ts_render_map_l1(ctx, g.scene, g.frame, None, None, None, Chat, Dhat, lam, None, None, None, None, gc2, go2,
                        ts.GRAD_COLOR | ts.GRAD_OPACITY)
    torch.cuda.synchronize()
    assert_grad_close("grad_pos x2", n(gp2), 2 * n(gp1), tol=2e-5)
    assert_grad_close("grad_color x2", n(gc2), 2 * n(gc1), tol=2e-5)
    assert_grad_close("grad_opacity x2", n(go2), 2 * n(go1), tol=2e-5)
    with pytest.raises(ts.TsError):
        ts.ts_render_map_l1(ctx, g.scene, g.frame, None, None, None, Chat, Dhat, lam, None, None, None, None, None, None, ts.GRAD_POSE)
    with pytest.raises(ts.TsError):
        ts.ts_render_bwd(ctx, g.scene, g.frame, gC, gD, None, gp1, None, None, ts.GRAD_POS)      # no walk state after map
    g.close()


@pytest.mark.parametrize("cfg", [0, 2, 3])
def test_normalised_depth_and_top_normal(ctx, oracle_mod, cfg):
    """NEXT-2 remainder: Dn = D / A with its backward pass through ts_render_bwd (gD, gA cotangents), and the normal of
    the highest-opacity hit (Fig. 3, reading S29), against the oracle."""
    from gpu_util import assert_grad_close, assert_images_close, dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(cfg)
    o, g = both(ctx, oracle_mod, sc)
    f, ok = check_forward(o, g)
    H, W, V = g.H, g.W, sc.pos.shape[0]
    eps = 1e-3
    # forward: elementwise on the GPU's own images against the oracle routine on the same images (exact division), and
    # against the oracle's own chain to the image tolerance where A is not tiny
    Dn = torch.empty_like(g.D)
    ts.ts_depth_normalise(ctx, W, H, g.D, g.A, eps, Dn)
    torch.cuda.synchronize()
    Dg, Ag = g.D.cpu().numpy(), g.A.cpu().numpy()
    assert np.array_equal(Dn.cpu().numpy(), oracle_mod.depth_normalise(Dg, Ag, eps, "f32"))
    ref_dn = oracle_mod.depth_normalise(f.depth, f.alpha, eps, "f32")
    solid = ok & (f.alpha > 0.05) & (Ag > 0.05)
    assert solid.mean() > 0.05
    assert_images_close("normalised depth", Dn.cpu().numpy(), ref_dn, solid, scale=float(np.abs(ref_dn).max()), tol=2e-4)
    # backward: cotangent of Dn -> (gD, gA) -> ts_render_bwd, against the oracle chain fed with the same cotangent
    rng = np.random.default_rng(60 + cfg)
    gDn = (rng.normal(size=(H, W)) * solid).astype(np.float32)
    gD, gA = torch.zeros(H, W, device="cuda"), torch.zeros(H, W, device="cuda")
    ts.ts_depth_normalise_bwd(ctx, W, H, g.D, g.A, eps, dev(gDn), gD, gA)
    gDo, gAo = oracle_mod.depth_normalise_bwd(f.depth, f.alpha, gDn, eps, "f32")
    torch.cuda.synchronize()
    assert np.allclose(gD.cpu().numpy(), gDo, rtol=2e-4, atol=2e-4 * np.abs(gDo).max())
    assert np.allclose(gA.cpu().numpy(), gAo, rtol=5e-4, atol=5e-4 * np.abs(gAo).max())
    ref = o.backward(None, gDo, gAo)
    gp, gc, go = torch.zeros(V, 3, device="cuda"), torch.zeros(V, 3, device="cuda"), torch.zeros(V, device="cuda")
    ts.ts_render_bwd(ctx, g.scene, g.frame, None, dev(gDo), dev(gAo), gp, gc, go, ts.GRAD_ALL)
    tau = torch.zeros(6, device="cuda")
    ts.ts_pose_jacobian_reduce(ctx, g.frame, tau)
    torch.cuda.synchronize()
    assert_grad_close("grad_pos (D/A)", gp.cpu().numpy(), ref.grad_pos)
    assert_grad_close("grad_opacity (D/A)", go.cpu().numpy(), ref.grad_opacity)
    assert np.abs(tau.cpu().numpy() - ref.dL_dtau).max() <= 1e-3 * np.abs(ref.dL_dtau).max()
    # top normal: a flat per-face attribute picked by an argmax over alphas: equal wherever the argmax is not a
    # near-tie between the two float32 implementations (pixels whose top alpha leads by less than 1e-4 are skipped)
    N, Nt = torch.empty(3, H, W, device="cuda"), torch.empty(3, H, W, device="cuda")
    ts.ts_render_fwd_normal_top(ctx, g.scene, g.frame, None, None, None, N, Nt)
    torch.cuda.synchronize()
    top_ref, N_ref = o.normal_top("tiled"), o.normal_forward("tiled")
    assert_images_close("normal map", N.cpu().numpy(), N_ref, ok[None])
    d = np.abs(Nt.cpu().numpy() - top_ref).max(axis=0)
    bad = (d > 1e-5) & ok
    print(f"top normal differs on {bad.sum()} of {ok.sum()} pixels (argmax near-ties)")
    assert bad.sum() <= 2 + 2e-4 * ok.size
    assert np.abs(np.linalg.norm(top_ref, axis=0)[f.n_contrib > 0] - 1.0).max() < 1e-5
    g.close()


@pytest.mark.parametrize("cfg", [0, 1, 2, 4])
def test_tight_binning(ctx, oracle_mod, cfg):
    """NEXT-4 remainder: TS_PARAM_TIGHT_BINNING (reading S31).  Tile counts, sorted keys / values and ranges bit-exact
    against the oracle's tight mode; images bit-identical to the loose lists' (no dropped pair could contribute);
    gradients to tolerance; fewer pairs."""
    from gpu_util import GpuView
    from paper_2605_31419_b200 import ts
    sc = small_cfg(cfg)
    prm = scenes.Params(**{**sc.params.__dict__, "tight_binning": True})
    o, g = both(ctx, oracle_mod, sc, params=prm)
    check_project_and_sort(o, g, sc.M)
    f, ok = check_forward(o, g)
    loose = GpuView(ctx, sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, sc.params)
    Cl, Dl, Al = loose.forward()
    assert np.array_equal(Cl, g.C.cpu().numpy()) and np.array_equal(Dl, g.D.cpu().numpy()) and np.array_equal(Al, g.A.cpu().numpy())
    n_tight, n_loose = g.status()[2], loose.status()[2]
    print(f"pairs: {n_loose} -> {n_tight} ({100.0 * (n_loose - n_tight) / max(1, n_loose):.1f} % dropped)")
    assert n_tight < n_loose
    check_backward(o, g, ok, 80 + cfg, [ts.GRAD_ALL, ts.GRAD_POSE])
    loose.close()
    g.close()


def test_tight_binning_wide_faces(ctx, oracle_mod):
    """Faces that span many tiles (the flattened scatter path of the binning kernel) under tight binning."""
    sc = scenes.config0(n_faces=60)
    rng = np.random.default_rng(3)
    pos = sc.pos.reshape(-1, 3, 3).copy()
    pos[:, :, :2] = (pos[:, :1, :2] + rng.normal(0, 0.9, (60, 3, 2)))            # ~50-pixel triangles
    sc.pos = pos.reshape(-1, 3).astype(np.float32)
    prm = scenes.Params(**{**sc.params.__dict__, "tight_binning": True})
    o, g = both(ctx, oracle_mod, sc, params=prm)
    check_project_and_sort(o, g, sc.M)
    assert o.project().tiles_touched.max() > 4
    check_forward(o, g)
    g.close()


@pytest.mark.parametrize("cfg", [0, 2, 3])
def test_per_face_sigma(ctx, oracle_mod, cfg):
    """NEXT-4 remainder: per-face window smoothness (ts_frame_set_face_sigma, reading S32): images, all gradients incl.
    dL/dsigma_m and the pose against the oracle; the fused launches; a constant array equals the global constant."""
    from gpu_util import GpuView, assert_grad_close, assert_images_close, dev
    from paper_2605_31419_b200 import ts
    sc = small_cfg(cfg)
    rng = np.random.default_rng(90 + cfg)
    sig = rng.uniform(0.4, 2.0, sc.M).astype(np.float32)
    o = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, sc.params, "f32", amb_tol=5e-4, face_sigma=sig)
    g = GpuView(ctx, sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, sc.params)
    sig_d, gs_d = dev(sig), torch.zeros(sc.M, device="cuda")
    ts.ts_frame_set_face_sigma(ctx, g.frame, sig_d, gs_d)
    check_project_and_sort(o, g, sc.M)
    f, ok = check_forward(o, g)
    # the window really differs from the global-sigma render
    plain = GpuView(ctx, sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, sc.params)
    assert np.abs(plain.forward()[2] - g.A.cpu().numpy()).max() > 0.05
    plain.close()
    H, W = ok.shape
    gC = (rng.normal(size=(3, H, W)) * ok[None]).astype(np.float32)
    gD = (rng.normal(size=(H, W)) * ok).astype(np.float32)
    gA = (rng.normal(size=(H, W)) * ok).astype(np.float32)
    ref = o.backward(gC, gD, gA)
    gp, gc, go, tau = g.backward(gC, gD, gA, ts.GRAD_ALL)
    torch.cuda.synchronize()
    assert_grad_close("grad_pos", gp, ref.grad_pos)
    assert_grad_close("grad_color", gc, ref.grad_color)
    assert_grad_close("grad_opacity", go, ref.grad_opacity)
    assert_grad_close("grad_sigma", gs_d.cpu().numpy(), ref.grad_sigma)
    assert np.abs(tau - ref.dL_dtau).max() <= 1e-3 * np.abs(ref.dL_dtau).max()
    # pose-only mode and the fused tracking launch (both run the visit form with the generic exponent)
    _, _, _, tau_p = g.backward(gC, gD, gA, ts.GRAD_POSE)
    assert np.abs(tau_p - ref.dL_dtau).max() <= 1e-3 * np.abs(ref.dL_dtau).max()
    tgt_pos = sc.pos_target if sc.pos_target is not None else sc.pos
    tgt = oracle_mod.Oracle(tgt_pos, sc.color, sc.opacity, None, sc.T_gt[0], sc.cam, sc.params, "f32", face_sigma=sig).forward("tiled")
    Chat, Dhat, lam = dev(tgt.color), dev(tgt.depth), sc.params.lambda_dep
    C2, D2, A2 = torch.empty_like(g.C), torch.empty_like(g.D), torch.empty_like(g.A)
    gC2, gD2 = torch.empty_like(g.C), torch.empty_like(g.D)
    ts.ts_render_track_l1(ctx, g.scene, g.frame, C2, D2, A2, Chat, Dhat, lam, gC2, gD2, None)
    tau2 = torch.zeros(6, device="cuda")
    ts.ts_pose_jacobian_reduce(ctx, g.frame, tau2)
    torch.cuda.synchronize()
    assert torch.equal(C2, g.C) and torch.equal(A2, g.A)
    ref2 = o.backward(gC2.cpu().numpy(), gD2.cpu().numpy(), None, want=("pose",))
    assert np.abs(tau2.cpu().numpy() - ref2.dL_dtau).max() <= 1e-3 * np.abs(ref2.dL_dtau).max()
    # the fused mapping launch accumulates dL/dsigma too
    V = sc.pos.shape[0]
    gs_d.zero_()
    gp3, gc3, go3 = torch.zeros(V, 3, device="cuda"), torch.zeros(V, 3, device="cuda"), torch.zeros(V, device="cuda")
    ts.ts_render_map_l1(ctx, g.scene, g.frame, None, None, None, Chat, Dhat, lam, gC2, gD2, None, gp3, gc3, go3, ts.GRAD_ALL)
    torch.cuda.synchronize()
    ref3 = o.backward(gC2.cpu().numpy(), gD2.cpu().numpy(), None)
    assert_grad_close("grad_sigma (map)", gs_d.cpu().numpy(), ref3.grad_sigma)
    assert_grad_close("grad_pos (map)", gp3.cpu().numpy(), ref3.grad_pos)
    # a constant array is the global constant (generic exponent against the sqrt fast path: to rounding)
    ts.ts_frame_set_face_sigma(ctx, g.frame, dev(np.full(sc.M, sc.params.sigma, np.float32)), None)
    with pytest.raises(ts.TsError):
        ts.ts_render_fwd(ctx, g.scene, g.frame, C2, D2, A2)            # the record is stale: project + bin again
    g.projected = g.sorted = False
    Cc, Dc, Ac = g.forward()
    ts.ts_frame_set_face_sigma(ctx, g.frame, None, None)
    g.projected = g.sorted = False
    Cg, Dg, Ag = g.forward()
    assert np.abs(Cc - Cg).max() <= 2e-5 and np.abs(Ac - Ag).max() <= 2e-5
    g.close()
