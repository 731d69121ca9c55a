"""Pins for the oracle's render, loss and PSNR.

Checked against: the worked values the reference texts print, the closed form
sum_p c' exp(-sigma) = 2 pi sqrt(det Sigma) c' (BASELINE.json north_star),
scipy.stats.multivariate_normal (a library routine for the same density),
permutation invariance, and the 3-sigma truncation bound.
"""
import math

import numpy as np
import pytest
from scipy.stats import multivariate_normal

import oracle
import workloads as wl


def _one(mu, l, c, o=1.0):
    return oracle.Params(np.array([mu], dtype=np.float64), np.array([l], dtype=np.float64),
                         np.array([c], dtype=np.float64), np.array([o], dtype=np.float64))


def test_render_worked_values():
    c = [0.3, 0.5, 0.7]
    # value c' at mu (pixel (8,8) has centre (8.5,8.5))
    img = oracle.render(32, 32, _one([8.5, 8.5], [1, 0, 1], c))
    assert np.allclose(img[8, 8], c, atol=1e-15)
    # two coincident Gaussians -> 2c', pre-clamp
    p2 = oracle.Params(np.array([[8.5, 8.5]] * 2), np.array([[1.0, 0, 1]] * 2), np.array([c] * 2), np.ones(2))
    img = oracle.render(32, 32, p2)
    assert np.allclose(img[8, 8], [0.6, 1.0, 1.4], atol=1e-15)
    # c'/2 at d = (sqrt(2 ln 2), 0), l = (1,0,1)
    d = math.sqrt(2 * math.log(2))
    img = oracle.render(32, 32, _one([8.5 - d, 8.5], [1, 0, 1], c))
    assert np.allclose(img[8, 8], 0.5 * np.array(c), rtol=1e-14)
    # opacity premultiplies the colour: c' = o c
    img = oracle.render(32, 32, _one([8.5, 8.5], [1, 0, 1], c, o=0.25))
    assert np.allclose(img[8, 8], 0.25 * np.array(c), atol=1e-15)


@pytest.mark.parametrize("l,size", [([2.0, 1.0, 3.0], 128), ([2.0, 0.0, 2.0], 64), ([3.0, -2.0, 1.5], 128)])
def test_dense_footprint_integral_closed_form(l, size):
    """sum over the pixel grid of c' exp(-sigma) = 2 pi |l1 l3| c' (scales >= 1.5 px)."""
    c = np.array([0.2, 0.9, 0.5])
    img = oracle.render(size, size, _one([size / 2 + 0.3, size / 2 - 0.2], l, c, o=0.7), dense=True)
    got = img.sum(axis=(0, 1))
    want = 2 * math.pi * abs(l[0] * l[2]) * 0.7 * c
    assert np.allclose(got, want, rtol=1e-7)


def test_tile_list_integral_within_truncation_bound():
    """Tile-list mode keeps at least the mass inside the 3-sigma ellipse:
    sum in [1 - exp(-4.5), 1] x 2 pi sqrt(det Sigma) c'."""
    for l in ([2.0, 1.0, 3.0], [4.0, 0.0, 1.5], [1.5, 0.5, 5.0]):
        img = oracle.render(160, 160, _one([77.3, 81.9], l, [1.0, 1.0, 1.0]))
        full = 2 * math.pi * abs(l[0] * l[2])
        s = img[..., 0].sum()
        assert (1 - math.exp(-4.5)) * full <= s <= full * (1 + 1e-9)


def test_dense_render_against_scipy_multivariate_normal():
    W, H, N = 40, 28, 12
    g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=6.0, config_index=70)
    p = oracle.Params.from_f32(g)
    img = oracle.render(W, H, p, dense=True)
    ys, xs = np.meshgrid(np.arange(H) + 0.5, np.arange(W) + 0.5, indexing="ij")
    pts = np.stack([xs, ys], axis=-1)
    ref = np.zeros((H, W, 3))
    for n in range(N):
        l1, l2, l3 = p.chol[n]
        L = np.array([[l1, 0.0], [l2, l3]])
        S = L @ L.T
        w = multivariate_normal(mean=p.mu[n], cov=S).pdf(pts) * (2 * math.pi * math.sqrt(np.linalg.det(S)))
        ref += w[..., None] * (p.opacity[n] * p.rgb[n])[None, None, :]
    assert np.allclose(img, ref, rtol=1e-10, atol=1e-13)


def test_tile_mode_equals_brute_force_over_lists():
    """Tile-list mode sums exactly the Gaussians whose rectangle covers the tile."""
    W, H, N = 70, 50, 80
    g = wl.random_gaussians(N, W, H, s_min=0.8, s_max=7.0, config_index=71, margin=8.0)
    p = oracle.Params.from_f32(g)
    rect, rng, lst = oracle.bin(W, H, p)
    img = oracle.render(W, H, p)
    TX = (W + 15) // 16
    r = np.random.default_rng(0)
    for _ in range(200):
        x, y = int(r.integers(W)), int(r.integers(H))
        t = (y // 16) * TX + x // 16
        acc = np.zeros(3)
        for n in lst[rng[t]:rng[t + 1]]:
            l1, l2, l3 = p.chol[n]
            L = np.array([[l1, 0.0], [l2, l3]])
            d = np.array([x + 0.5, y + 0.5]) - p.mu[n]
            acc += p.opacity[n] * p.rgb[n] * math.exp(-0.5 * d @ np.linalg.inv(L @ L.T) @ d)
        assert np.allclose(img[y, x], acc, rtol=1e-10, atol=1e-14)


def test_permutation_invariance():
    W, H, N = 64, 48, 100
    g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=8.0, config_index=72)
    p = oracle.Params.from_f32(g)
    a = oracle.render(W, H, p)
    perm = np.random.default_rng(3).permutation(N)
    q = oracle.Params(p.mu[perm].copy(), p.chol[perm].copy(), p.rgb[perm].copy(), p.opacity[perm].copy())
    b = oracle.render(W, H, q)
    assert np.allclose(a, b, rtol=0, atol=1e-13)


def test_tile_subset_render_matches_full():
    W, H, N = 64, 48, 60
    p = oracle.Params.from_f32(wl.random_gaussians(N, W, H, s_min=1.0, s_max=8.0, config_index=73))
    full = oracle.render(W, H, p)
    part = oracle.render(W, H, p, tiles=[0, 5, 11])
    TX = 4
    for t in (0, 5, 11):
        ty, tx = divmod(t, TX)
        assert np.array_equal(part[ty * 16:ty * 16 + 16, tx * 16:tx * 16 + 16], full[ty * 16:ty * 16 + 16, tx * 16:tx * 16 + 16])
    assert part[16:32, 32:48].sum() == 0.0  # tile 6 untouched


def test_truncation_is_small_cutoff_3_vs_6():
    """cutoff 6 vs 3 changes the PSNR by < 0.05 dB (here on a random
    scene against a target, which bounds the same truncation error)."""
    W, H, N = 96, 64, 300
    p = oracle.Params.from_f32(wl.random_gaussians(N, W, H, s_min=1.0, s_max=6.0, config_index=74))
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 74))
    a = oracle.psnr(oracle.render(W, H, p, cutoff=3.0), frame)
    b = oracle.psnr(oracle.render(W, H, p, cutoff=6.0), frame)
    assert abs(a - b) < 0.05
    dense = oracle.render(W, H, p, dense=True)
    assert np.abs(oracle.render(W, H, p) - dense).max() < 0.011 * N  # each term truncated below exp(-4.5)


def test_loss_and_psnr_hand_values():
    W, H = 20, 12
    tgt = np.full((H, W, 3), 0.5, dtype=np.float32)
    img = np.full((H, W, 3), 0.5 + 16 / 255)
    L, G = oracle.loss(img, tgt)
    assert math.isclose(L, (16 / 255) ** 2, rel_tol=1e-12)
    assert np.allclose(G, 2 * (16 / 255) / (3 * W * H), rtol=1e-12)
    assert abs(oracle.psnr(img, tgt) - 20 * math.log10(255 / 16)) < 1e-9  # 24.0484 dB
    assert oracle.psnr(tgt.astype(np.float64), tgt) == 99.0
    # the loss sees the unclamped sum, PSNR the clamped one
    img2 = np.full((H, W, 3), 1.5)
    L2, _ = oracle.loss(img2, tgt)
    assert math.isclose(L2, 1.0, rel_tol=1e-12)
    assert abs(oracle.psnr(img2, tgt) - 10 * math.log10(1 / 0.25)) < 1e-9
