"""Pins for the oracle's Adam step, mask, projection and fit loop
(SURVEY.md §8(c-6), (c-7)): torch.optim.Adam (float64), the closed-form first
step, the frozen-set identity and the fit fixtures of SPEC.md:253-255, 280."""
import numpy as np
import torch

import oracle
import workloads as wl


def _rand_params(N, seed):
    r = np.random.default_rng(seed)
    return oracle.Params(r.uniform(0, 50, (N, 2)), np.stack([r.uniform(1, 4, N), r.uniform(-2, 2, N),
                                                              r.uniform(1, 4, N)], 1),
                         r.uniform(0, 1, (N, 3)), r.uniform(0.2, 1, N))


def test_adam_matches_torch_optim_adam():
    N, steps = 40, 25
    p = _rand_params(N, 0)
    lr = [1e-2, 3e-3, 5e-3, 2e-3]
    t = [torch.tensor(a.copy(), dtype=torch.float64, requires_grad=True) for a in (p.mu, p.chol, p.rgb, p.opacity)]
    opt = torch.optim.Adam([{"params": [t[i]], "lr": lr[i]} for i in range(4)], betas=(0.9, 0.999), eps=1e-8)
    m = np.zeros((N, 9))
    v = np.zeros((N, 9))
    r = np.random.default_rng(5)
    for k in range(1, steps + 1):
        g = r.standard_normal((N, 9)) * 10.0 ** r.uniform(-6, 0, (N, 9))
        oracle.adam(p, g, m, v, lr, k, l_min=-1e30)  # projection disabled for this pin
        for ten, sl in zip(t, (slice(0, 2), slice(2, 5), slice(5, 8), 8)):
            ten.grad = torch.tensor(g[:, sl].copy(), dtype=torch.float64)
        opt.step()
    assert np.allclose(p.mu, t[0].detach().numpy(), rtol=1e-12, atol=1e-14)
    assert np.allclose(p.chol, t[1].detach().numpy(), rtol=1e-12, atol=1e-14)
    assert np.allclose(p.rgb, t[2].detach().numpy(), rtol=1e-12, atol=1e-14)
    assert np.allclose(p.opacity, t[3].detach().numpy(), rtol=1e-12, atol=1e-14)


def test_adam_first_step_and_constant_gradient():
    N = 8
    p = _rand_params(N, 1)
    p0 = p.copy()
    g = np.random.default_rng(2).standard_normal((N, 9))
    m = np.zeros((N, 9))
    v = np.zeros((N, 9))
    lr = 1e-2
    oracle.adam(p, g, m, v, lr, 1, l_min=-1e30)
    step = -lr * g / (np.abs(g) + 1e-8)          # first step from zero moments
    assert np.allclose(p.flat9() - p0.flat9(), step, rtol=1e-9, atol=1e-15)
    for k in range(2, 11):                        # constant gradient: k steps of the same size
        oracle.adam(p, g, m, v, lr, k, l_min=-1e30)
    assert np.allclose(p.flat9() - p0.flat9(), 10 * step, rtol=1e-7)


def test_adam_mask_and_projection():
    N = 10
    p = _rand_params(N, 3)
    p.chol[0] = [0.1004, 0.0, 0.1004]
    p0 = p.copy()
    g = np.ones((N, 9))
    m = np.random.default_rng(4).standard_normal((N, 9))
    v = np.abs(np.random.default_rng(5).standard_normal((N, 9)))
    m[0] = 0.0                                    # row 0 steps by exactly -lr: 0.1004 - 0.01 < l_min
    v[0] = 0.0
    m0, v0 = m.copy(), v.copy()
    active = np.zeros(N, dtype=np.uint8)
    active[[0, 3]] = 1
    oracle.adam(p, g, m, v, 1e-2, 1, active=active)
    frozen = [n for n in range(N) if not active[n]]
    assert np.array_equal(p.flat9()[frozen], p0.flat9()[frozen])     # bit-identical
    assert np.array_equal(m[frozen], m0[frozen]) and np.array_equal(v[frozen], v0[frozen])
    assert not np.array_equal(p.flat9()[3], p0.flat9()[3])
    assert p.chol[0, 0] == 0.1 and p.chol[0, 2] == 0.1                # projected to l_min
    # empty active set -> output equals input
    q = p.copy()
    oracle.adam(q, g, m, v, 1e-2, 2, active=np.zeros(N, dtype=np.uint8))
    assert np.array_equal(q.flat9(), p.flat9())


def test_fit_fixed_point():
    """Target == initial render -> gradients ~ 0, set unchanged after 10 iterations."""
    W, H, N = 48, 32, 30
    p = oracle.Params.from_f32(wl.random_gaussians(N, W, H, s_min=1.5, s_max=5.0, config_index=90,
                                                   opacity_range=(0.1, 0.3)))
    target = oracle.render(W, H, p).astype(np.float32)  # float32 target: residual ~1e-8
    p0 = p.copy()
    # Adam normalises the step: with |g| ~ 1e-9 >> eps*... use lr tiny steps check via loss instead
    rep = oracle.fit(W, H, p, target, 10, lr=1e-6)
    assert rep.final_loss < 1e-12
    assert np.abs(p.flat9() - p0.flat9()).max() <= 10 * 1e-6 + 1e-12


def test_fit_recovers_displacement():
    """one Gaussian, target = render of a copy shifted by 2 px."""
    W = H = 48
    truth = oracle.Params(np.array([[25.0, 23.0]]), np.array([[4.0, 0.5, 3.0]]), np.array([[0.8, 0.5, 0.3]]),
                          np.ones(1))
    target = oracle.render(W, H, truth, dense=True).astype(np.float32)
    p = truth.copy()
    p.mu[0, 0] -= 2.0
    rep = oracle.fit(W, H, p, target, 500, lr=[2e-2, 0.0, 0.0, 0.0])
    assert np.abs(p.mu - truth.mu).max() < 0.1
    assert rep.first_nonfinite_iter == 0


def test_fit_descends_on_tiny_config():
    """configs[0]: 64x64, 256 Gaussians, lr 1e-2, 100 iterations."""
    frame, _ = wl.talking_head_frame(wl.SPEC_TINY)
    p = oracle.Params.from_f32(wl.tiny_gaussians())
    rep = oracle.fit(64, 64, p, frame, 100, lr=1e-2, trace=True)
    assert rep.loss_trace[-1] < 0.1 * rep.loss_trace[0]
    sm = np.convolve(rep.loss_trace, np.ones(10) / 10, mode="valid")
    assert np.all(np.diff(sm) < 0)  # smoothed trace decreases
    assert 15.0 < rep.psnr < 40.0
    assert np.all(p.chol[:, 0] >= 0.1) and np.all(p.chol[:, 2] >= 0.1)


def test_fit_is_deterministic_and_thread_count_independent():
    frame, _ = wl.talking_head_frame(wl.SPEC_TINY)
    a = oracle.Params.from_f32(wl.tiny_gaussians())
    b = a.copy()
    oracle.set_threads(1)
    ra = oracle.fit(64, 64, a, frame, 5)
    oracle.set_threads(0)
    rb = oracle.fit(64, 64, b, frame, 5)
    assert np.array_equal(a.flat9(), b.flat9()) and ra.final_loss == rb.final_loss


# --------------------------------------------------------------------------- c-12: schedule + early stop

def test_lr_schedule_hand_values():
    """base at iter 0, exactly base x 0.5 at the 60 % boundary, x 0.25 from 85 %,
    non-increasing."""
    base, iters = 4e-3, 1000
    assert oracle.lr_schedule(0, iters, base) == base
    assert oracle.lr_schedule(599, iters, base) == base
    assert oracle.lr_schedule(600, iters, base) == base * 0.5
    assert oracle.lr_schedule(849, iters, base) == base * 0.5
    assert oracle.lr_schedule(850, iters, base) == base * 0.25
    lrs = [oracle.lr_schedule(i, 37, base) for i in range(37)]
    assert all(a >= b for a, b in zip(lrs, lrs[1:])) and lrs[-1] == base * 0.25


def test_fit_sched_reduces_to_fit_and_stops_early():
    frame, _ = wl.talking_head_frame(wl.SPEC_TINY)
    g = wl.tiny_gaussians()
    # no decay, no target: the scheduled loop is the c-7 loop (the C implementation), bit for bit
    pa, pb = oracle.Params.from_f32(g), oracle.Params.from_f32(g)
    ra = oracle.fit(64, 64, pa, frame, 25, lr=1e-2)
    rb = oracle.fit_sched(64, 64, pb, frame, 25, lr=1e-2, decay=1.0, target_psnr=0.0)
    assert np.array_equal(pa.flat9(), pb.flat9()) and ra.psnr == rb.psnr and rb.iters_run == 25
    # early stop: at the first check whose PSNR reaches the target, not before
    pc = oracle.Params.from_f32(g)
    full = oracle.fit_sched(64, 64, pc, frame, 100, lr=1e-2)
    target = full.psnr - 1.5
    pd = oracle.Params.from_f32(g)
    rd = oracle.fit_sched(64, 64, pd, frame, 100, lr=1e-2, target_psnr=target, check_every=10)
    assert rd.iters_run % 10 == 0 and 0 < rd.iters_run < 100 and rd.psnr >= target
    pe = oracle.Params.from_f32(g)
    re_ = oracle.fit_sched(64, 64, pe, frame, 100, lr=1e-2)          # the same trajectory, cut one check earlier
    pf = oracle.Params.from_f32(g)
    # (the schedule depends on the total count, so the shorter run is emulated by a target never reached)
    rf = oracle.fit_sched(64, 64, pf, frame, 100, lr=1e-2, target_psnr=1e9, check_every=10)
    assert rf.iters_run == 100 and np.array_equal(pe.flat9(), pf.flat9()) and re_.psnr == rf.psnr
    # decay makes late steps smaller: with the schedule the last update is a quarter of the base step
    ph, pi = oracle.Params.from_f32(g), oracle.Params.from_f32(g)
    oracle.fit_sched(64, 64, ph, frame, 20, lr=1e-2, decay=1.0)
    oracle.fit_sched(64, 64, pi, frame, 20, lr=1e-2, decay=0.5)
    assert not np.array_equal(ph.flat9(), pi.flat9())
