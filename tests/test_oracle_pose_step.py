"""Pin P25: the oracle's pose step (a8, harness helper; reading S23: Adam on tau with the paper's learning rates,
PAPER.md:440-441) against torch.optim.Adam -- a library routine the oracle shares no code with -- and against the
numpy SE(3) exponential.  A wrong bias-correction exponent, a swapped beta or a missing eps fails it."""
import numpy as np
import torch

from paper_2605_31419_b200 import scenes


def test_p25_pose_step_is_adam_then_left_exp(oracle_mod):
    rng = np.random.default_rng(25)
    T = scenes.look_level((0.3, -0.2, 0.0), 0.6).astype(np.float32)
    lr = [1e-3] * 3 + [3e-3] * 3                       # translation, rotation
    state = np.zeros(13, np.float32)
    # torch's Adam on a 6-vector that starts at zero: its step k moves the parameter by delta_k
    p_rho = torch.zeros(3, dtype=torch.float64, requires_grad=True)
    p_th = torch.zeros(3, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([{"params": [p_rho], "lr": lr[0]}, {"params": [p_th], "lr": lr[3]}], betas=(0.9, 0.999), eps=1e-8)
    T_ref = T.astype(np.float64)
    for k in range(5):
        g = (rng.normal(size=6) * 10.0 ** rng.uniform(-3, 1)).astype(np.float32)
        T, state = oracle_mod.pose_step_f32(T, g, state, lr)
        before = np.concatenate([p_rho.detach().numpy().copy(), p_th.detach().numpy().copy()])
        p_rho.grad, p_th.grad = torch.tensor(g[:3], dtype=torch.float64), torch.tensor(g[3:], dtype=torch.float64)
        opt.step()
        delta = np.concatenate([p_rho.detach().numpy(), p_th.detach().numpy()]) - before
        T_ref = scenes.se3_exp(delta) @ np.vstack([T_ref, [0, 0, 0, 1]])     # T <- Exp(delta) o T, numpy exponential
        T_ref = T_ref[:3]
        assert np.allclose(T, T_ref, atol=3e-6), (k, np.abs(T - T_ref).max())
        m = np.concatenate([opt.state[p_rho]["exp_avg"].numpy(), opt.state[p_th]["exp_avg"].numpy()])
        v = np.concatenate([opt.state[p_rho]["exp_avg_sq"].numpy(), opt.state[p_th]["exp_avg_sq"].numpy()])
        # (float32: 1.0f - 0.999f = 0.00100004673, 4.7e-5 off the exact 0.001 torch uses in float64)
        assert np.allclose(state[:6], m, rtol=1e-5, atol=1e-9) and np.allclose(state[6:12], v, rtol=1e-4, atol=1e-12)
        assert state[12] == k + 1
    # the first step of Adam moves every component by lr * sign(g) (bias correction makes mhat / sqrt(vhat) = +-1)
    T1, s1 = oracle_mod.pose_step_f32(np.concatenate([np.eye(3), np.zeros((3, 1))], 1).astype(np.float32),
                                      np.array([2.0, -3.0, 0.5, 0, 0, 0], np.float32), np.zeros(13, np.float32), lr)
    assert np.allclose(T1[:, 3], [-1e-3, 1e-3, -1e-3], atol=1e-8)
