"""Pins for the oracle's analytic gradients.

Checked against: central finite differences of the oracle's own render + loss
(SPEC.md:143, 148, 530), torch autograd in float64 on a dense restatement of
Eq. 2 (library pin), the closed forms for G == 1, and the zero cases.
"""
import math

import numpy as np
import pytest
import torch

import oracle
import workloads as wl


def _scene(seed, W=16, H=16, N=5):
    r = np.random.default_rng(1000 + seed)
    mu = r.uniform(2, 14, (N, 2))
    chol = np.stack([r.uniform(1.0, 3.0, N), r.uniform(-1.5, 1.5, N), r.uniform(1.0, 3.0, N)], axis=1)
    rgb = r.uniform(0.1, 1.0, (N, 3))
    op = r.uniform(0.3, 1.0, N)
    target = r.uniform(0, 1, (H, W, 3)).astype(np.float32)
    return oracle.Params(mu, chol, rgb, op), target


def _loss_of(W, H, p, target, dense):
    L, _ = oracle.loss(oracle.render(W, H, p, dense=dense), target)
    return L


@pytest.mark.parametrize("dense", [True, False])
def test_gradients_match_central_finite_differences(dense):
    """>= 20 random 16x16 scenes with 5 Gaussians, every one of the 9 partials."""
    W = H = 16
    h = 1e-5
    worst = 0.0
    for seed in range(20):
        p, target = _scene(seed)
        img = oracle.render(W, H, p, dense=dense)
        _, G = oracle.loss(img, target)
        grad = oracle.backward(W, H, p, G, dense=dense)
        scale = np.abs(grad).max(axis=0)
        arrays = [(p.mu, 0, 2), (p.chol, 2, 3), (p.rgb, 5, 3), (p.opacity[:, None], 8, 1)]
        for n in range(p.n):
            for arr, off, k in arrays:
                for j in range(k):
                    tgt_arr = p.opacity if off == 8 else arr
                    idx = n if off == 8 else (n, j)
                    old = tgt_arr[idx]
                    tgt_arr[idx] = old + h
                    lp = _loss_of(W, H, p, target, dense)
                    tgt_arr[idx] = old - h
                    lm = _loss_of(W, H, p, target, dense)
                    tgt_arr[idx] = old
                    fd = (lp - lm) / (2 * h)
                    an = grad[n, off + j]
                    err = abs(fd - an) / max(abs(an), 1e-3 * scale[off + j], 1e-12)
                    worst = max(worst, err)
                    assert err < 1e-3, (seed, n, off + j, fd, an)
    assert worst < 1e-4  # float64 central differences are far inside the 1e-3 bar


def _torch_dense_loss(mu, chol, rgb, op, target):
    """Dense restatement of Eq. 2 + MSE in torch float64 (conic form, not the
    oracle's whitened form)."""
    H, W, _ = target.shape
    ys, xs = torch.meshgrid(torch.arange(H, dtype=torch.float64) + 0.5,
                            torch.arange(W, dtype=torch.float64) + 0.5, indexing="ij")
    l1, l2, l3 = chol[:, 0], chol[:, 1], chol[:, 2]
    L = torch.stack([torch.stack([l1, torch.zeros_like(l1)], -1), torch.stack([l2, l3], -1)], -2)  # [N,2,2]
    Sinv = torch.linalg.inv(L @ L.transpose(-1, -2))
    d = torch.stack([xs[None] - mu[:, 0, None, None], ys[None] - mu[:, 1, None, None]], -1)  # [N,H,W,2]
    sig = 0.5 * torch.einsum("nhwi,nij,nhwj->nhw", d, Sinv, d)
    w = torch.exp(-sig)
    C = torch.einsum("nhw,nc->hwc", w, op[:, None] * rgb)
    return ((C - target) ** 2).mean()


def test_gradients_match_torch_autograd_dense():
    W = H = 16
    for seed in range(5):
        p, target = _scene(seed + 100, N=6)
        _, G = oracle.loss(oracle.render(W, H, p, dense=True), target)
        grad = oracle.backward(W, H, p, G, dense=True)
        t = [torch.tensor(a, dtype=torch.float64, requires_grad=True) for a in (p.mu, p.chol, p.rgb, p.opacity)]
        loss = _torch_dense_loss(*t, torch.tensor(target, dtype=torch.float64))
        loss.backward()
        ref = np.concatenate([t[0].grad.numpy(), t[1].grad.numpy(), t[2].grad.numpy(), t[3].grad.numpy()[:, None]], 1)
        assert np.allclose(grad, ref, rtol=1e-9, atol=1e-15)


def test_closed_form_gradients_for_unit_image_gradient():
    """G == 1, one Gaussian, dense, canvas holds the footprint:
    dL/dc' = 2 pi l1 l3, dL/dl1 = 2 pi l3 c', dL/dl3 = 2 pi l1 c', dL/dl2 = dL/dmu = 0."""
    W = H = 128
    l = np.array([2.0, 1.0, 3.0])
    c = np.array([0.4, 0.7, 0.2])
    o = 0.8
    p = oracle.Params(np.array([[64.2, 63.7]]), l[None].copy(), c[None].copy(), np.array([o]))
    G = np.ones((H, W, 3))
    g = oracle.backward(W, H, p, G, dense=True)[0]
    two_pi = 2 * math.pi
    csum = o * c.sum()  # sum over channels of c'
    assert abs(g[0]) < 1e-9 and abs(g[1]) < 1e-9
    assert math.isclose(g[2], two_pi * l[2] * csum, rel_tol=1e-7)   # 6 pi * sum c'
    assert abs(g[3]) < 1e-9
    assert math.isclose(g[4], two_pi * l[0] * csum, rel_tol=1e-7)   # 4 pi * sum c'
    assert np.allclose(g[5:8], o * two_pi * l[0] * l[2], rtol=1e-7)
    assert math.isclose(g[8], two_pi * l[0] * l[2] * c.sum(), rel_tol=1e-7)


def test_zero_cases():
    W, H, N = 48, 32, 20
    g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=5.0, config_index=80)
    g.mu[3] = [-100.0, -100.0]     # outside all tiles
    g.mu[4] = [W + 60.0, 5.0]
    p = oracle.Params.from_f32(g)
    # zero image gradient -> all-zero gradients
    assert np.all(oracle.backward(W, H, p, np.zeros((H, W, 3))) == 0.0)
    # Gaussians outside all tiles get exactly zero gradient (north_star)
    Gr = np.random.default_rng(0).standard_normal((H, W, 3))
    gr = oracle.backward(W, H, p, Gr)
    assert np.all(gr[3] == 0.0) and np.all(gr[4] == 0.0)
    assert np.abs(gr[0]).max() > 0
    # single-pixel loss at mu: dC/dc' = 1 and dC/dmu = 0
    one = oracle.Params(np.array([[8.5, 8.5]]), np.array([[1.5, 0.3, 2.0]]), np.array([[0.5, 0.5, 0.5]]), np.ones(1))
    G1 = np.zeros((16, 16, 3))
    G1[8, 8, 0] = 1.0
    g1 = oracle.backward(16, 16, one, G1)[0]
    assert g1[0] == 0.0 and g1[1] == 0.0 and g1[5] == 1.0 and g1[6] == 0.0


def test_subset_backward_matches_full():
    W, H, N = 64, 48, 50
    p = oracle.Params.from_f32(wl.random_gaussians(N, W, H, s_min=1.0, s_max=6.0, config_index=81))
    Gr = np.random.default_rng(1).standard_normal((H, W, 3))
    full = oracle.backward(W, H, p, Gr)
    sub = oracle.backward(W, H, p, Gr, subset=[3, 17, 42])
    assert np.array_equal(sub[[3, 17, 42]], full[[3, 17, 42]])
    assert np.all(sub[0] == 0)
