"""Pins for the oracle's ROI initialiser and P-frame selection
(SURVEY.md §8(c-8), (c-9)): scipy.ndimage's Sobel as the library routine for the
weights, a numpy restatement of the counter generator, a chi-square test of the
sampled distribution, and a brute-force union for the selection."""
import math

import numpy as np
import pytest
from scipy import ndimage

import oracle
import workloads as wl

M64 = (1 << 64) - 1


def _splitmix(seed, i, k):
    z = (seed + (8 * i + k + 1) * 0x9E3779B97F4A7C15) & M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M64
    return z ^ (z >> 31)


def test_counter_generator_matches_python_restatement():
    for seed in (0, 1, 250509324, M64):
        for i in (0, 1, 77, 49999):
            for k in range(6):
                assert oracle.rnd64(seed, i, k) == _splitmix(seed, i, k)
    # SplitMix64's published first output for state 0 advanced once by the golden gamma
    assert oracle.rnd64(0, 0, 0) == 0xE220A8397B1DCDAF


def test_roi_weights_against_scipy_sobel():
    spec = wl.scaled_spec(96, 64, 91)
    frame, mask = wl.talking_head_frame(spec)
    w_in, w_out = oracle.roi_weights(frame, mask)
    q = np.floor(np.float32(255.0) * frame + np.float32(0.5)).astype(np.int64)
    grey = q.sum(axis=2)
    gx = ndimage.sobel(grey, axis=1, mode="nearest")
    gy = ndimage.sobel(grey, axis=0, mode="nearest")
    mag = np.floor(np.sqrt((gx * gx + gy * gy).astype(np.float64))).astype(np.int64)
    # guard the float sqrt against perfect squares
    mag = np.where((mag + 1) ** 2 <= gx * gx + gy * gy, mag + 1, mag)
    want_in = np.where(mask > 0, mag + 1, 0)
    assert np.array_equal(w_in, want_in)
    assert np.array_equal(w_out, (mask == 0).astype(np.int32))


def test_init_roi_structure_and_distribution():
    spec = wl.scaled_spec(96, 64, 92)
    frame, mask = wl.talking_head_frame(spec)
    H, W = mask.shape
    N = 20000
    mu, chol, rgb, op, pix = oracle.init_roi(frame, mask, N, seed=7, s_min=1.0, s_max=4.0)
    N_in = (7 * N) // 10
    ys, xs = pix // W, pix % W
    assert np.all(mask[ys[:N_in], xs[:N_in]] == 1) and np.all(mask[ys[N_in:], xs[N_in:]] == 0)
    # position = pixel centre + jitter in [-0.5, 0.5)
    assert np.all(np.floor(mu[:, 0]) == xs) | np.all(np.abs(mu[:, 0] - xs - 0.5) <= 0.5)
    assert np.all(np.abs(mu[:, 0] - (xs + 0.5)) <= 0.5) and np.all(np.abs(mu[:, 1] - (ys + 0.5)) <= 0.5)
    # colour copied from the frame, opacity 1
    assert np.array_equal(rgb, frame[ys, xs]) and np.all(op == 1.0)
    # sampled indices reproduce the inverse-CDF rule with the python generator
    w_in, w_out = oracle.roi_weights(frame, mask)
    c_in = np.cumsum(w_in.ravel().astype(np.uint64))
    c_out = np.cumsum(w_out.ravel().astype(np.uint64))
    for i in (0, 1, 5, N_in - 1, N_in, N - 1):
        c = c_in if i < N_in else c_out
        tgt = _splitmix(7, i, 0) % int(c[-1])
        assert pix[i] == int(np.searchsorted(c, tgt, side="right"))
    # chi-square of the inside samples against the weights, coarse 8x8-pixel cells
    cells = (ys[:N_in] // 8) * (W // 8) + xs[:N_in] // 8
    obs = np.bincount(cells, minlength=(H // 8) * (W // 8)).astype(np.float64)
    exp = w_in.reshape(H // 8, 8, W // 8, 8).sum(axis=(1, 3)).ravel().astype(np.float64)
    exp = exp / exp.sum() * N_in
    keep = exp > 5
    chi2 = ((obs[keep] - exp[keep]) ** 2 / exp[keep]).sum()
    dof = keep.sum() - 1
    assert chi2 < dof + 6 * math.sqrt(2 * dof)
    assert obs[~keep & (exp == 0)].sum() == 0
    # scales log-uniform in [s_min, s_max]: eigenvalues of L L^T are s1^2, s2^2
    L = np.zeros((N, 2, 2))
    L[:, 0, 0], L[:, 1, 0], L[:, 1, 1] = chol[:, 0], chol[:, 1], chol[:, 2]
    ev = np.linalg.eigvalsh(L @ L.transpose(0, 2, 1))
    s = np.sqrt(ev)
    assert s.min() >= 1.0 * (1 - 1e-5) and s.max() <= 4.0 * (1 + 1e-5)
    logs = np.log(s.ravel())
    assert abs(logs.mean() - 0.5 * math.log(4.0)) < 0.02          # uniform in log
    assert abs(logs.var() - math.log(4.0) ** 2 / 12) < 0.01
    assert np.all(chol[:, 0] > 0) and np.all(chol[:, 2] > 0)
    # determinism and seed sensitivity
    again = oracle.init_roi(frame, mask, N, seed=7, s_min=1.0, s_max=4.0)
    assert all(np.array_equal(a, b) for a, b in zip((mu, chol, rgb, op, pix), again))
    other = oracle.init_roi(frame, mask, N, seed=8, s_min=1.0, s_max=4.0)
    assert not np.array_equal(other[0], mu)


def test_init_roi_edge_cases():
    frame, mask = wl.talking_head_frame(wl.scaled_spec(48, 32, 93))
    with pytest.raises(ValueError):
        oracle.init_roi(frame, np.zeros_like(mask), 10, 1, 1.0, 4.0)       # empty ROI
    mu, chol, rgb, op, pix = oracle.init_roi(frame, np.ones_like(mask), 10, 1, 1.0, 4.0)  # no outside pixels
    assert len(pix) == 10                                                   # all N go inside
    mu, *_ = oracle.init_roi(frame, mask, 1, 1, 2.0, 2.0)                   # N=1 -> N_in=0, one outside sample
    assert mu.shape == (1, 2)


def _pframe_scene():
    W, H, N = 64, 64, 20
    g = wl.random_gaussians(N, W, H, s_min=1.5, s_max=5.0, config_index=94, opacity_range=(0.3, 0.9))
    return W, H, oracle.Params.from_f32(g)


def test_pframe_select_identical_frame_selects_nothing():
    W, H, p = _pframe_scene()
    frame = np.clip(oracle.render(W, H, p), 0, 1).astype(np.float32)
    resid, flag, active, na = oracle.pframe_select(W, H, p, frame, tau=0.02)
    assert na == 0 and not flag.any() and resid.max() < 1e-7
    q = p.copy()
    act, rep = oracle.encode_pframe(W, H, q, frame, 0.02, 50)
    assert rep.iters_run == 0 and rep.n_active == 0 and np.array_equal(q.flat9(), p.flat9())


def test_pframe_select_all_changed_selects_every_listed_gaussian():
    W, H, p = _pframe_scene()
    p.mu[5] = [-500.0, -500.0]                                   # culled: never selected
    frame = np.clip(oracle.render(W, H, p) + 0.5, 0, 1).astype(np.float32)
    frame[frame > 0.99] = 0.0                                    # keep every tile's residual large
    resid, flag, active, na = oracle.pframe_select(W, H, p, frame, tau=0.02)
    _, _, lst = oracle.bin(W, H, p)
    assert flag.all()
    assert set(np.nonzero(active)[0]) == set(lst.tolist()) and active[5] == 0


def test_pframe_select_brute_force_union():
    """<= 64x64, <= 20 Gaussians: changed tiles and the union of their lists by brute force."""
    W, H, p = _pframe_scene()
    base = np.clip(oracle.render(W, H, p), 0, 1)
    frame = base.copy()
    frame[20:30, 36:44] += 0.4          # a moving-square style change touching tiles (2,1)
    frame[50:52, 3:5] += 0.2            # small change: tile mean stays below tau
    frame = np.clip(frame, 0, 1).astype(np.float32)
    tau = 0.02
    resid, flag, active, na = oracle.pframe_select(W, H, p, frame, tau)
    rect, rng, lst = oracle.bin(W, H, p)
    TX = 4
    want_active = np.zeros(p.n, dtype=np.uint8)
    for t in range(16):
        ty, tx = divmod(t, TX)
        blk_f = frame[ty * 16:ty * 16 + 16, tx * 16:tx * 16 + 16].astype(np.float64)
        blk_r = base[ty * 16:ty * 16 + 16, tx * 16:tx * 16 + 16]
        r = np.abs(blk_f - blk_r).mean()
        assert math.isclose(resid[t], r, rel_tol=1e-9, abs_tol=1e-12)
        assert flag[t] == (1 if r > tau else 0)
        if r > tau:
            for n in range(p.n):        # brute force: rectangle overlap, not the list
                if rect[n, 0] <= tx <= rect[n, 2] and rect[n, 1] <= ty <= rect[n, 3]:
                    want_active[n] = 1
    assert np.array_equal(active, want_active) and na == want_active.sum()
    assert 0 < na < p.n and flag.sum() >= 1 and flag[12] == 0


def test_encode_pframe_freezes_unselected_gaussians():
    W, H, p = _pframe_scene()
    base = np.clip(oracle.render(W, H, p), 0, 1)
    frame = base.copy()
    frame[20:30, 36:44] += 0.4
    frame = np.clip(frame, 0, 1).astype(np.float32)
    q = p.copy()
    active, rep = oracle.encode_pframe(W, H, q, frame, 0.02, 40)
    assert rep.iters_run == 40 and 0 < rep.n_active < p.n
    frozen = np.nonzero(active == 0)[0]
    assert np.array_equal(q.flat9()[frozen], p.flat9()[frozen])
    assert not np.array_equal(q.flat9()[active == 1], p.flat9()[active == 1])
    L0, _ = oracle.loss(oracle.render(W, H, p), frame)
    assert rep.final_loss < L0


# --------------------------------------------------------------------------- c-13: pixel-granular selection

def _tiny_scene(seed=0, n=18, W=64, H=48):
    g = wl.random_gaussians(n, W, H, s_min=1.5, s_max=5.0, opacity_range=(0.3, 0.9), config_index=95 + seed)
    return W, H, g, oracle.Params.from_f32(g)


def test_pixel_selection_trivial_cases():
    W, H, g, p = _tiny_scene()
    img = np.clip(oracle.render(W, H, p), 0, 1).astype(np.float32)
    ch, resid, act, na = oracle.pframe_select_pixels(W, H, p, img, 0.01)
    assert ch.sum() == 0 and na == 0                                   # identical frames
    f = img.copy()
    f[20, 30, 1] += 0.5
    ch, resid, act, na = oracle.pframe_select_pixels(W, H, p, np.clip(f, 0, 1.5), 0.1)
    assert ch.sum() == 1 and ch[20, 30] == 1                           # one pixel changed by 0.5
    ch, _, _, na = oracle.pframe_select_pixels(W, H, p, img + np.float32(0.05), 0.1)
    assert ch.sum() == 0 and na == 0                                   # uniform sub-threshold shift
    ch_d, _, _, _ = oracle.pframe_select_pixels(W, H, p, np.clip(f, 0, 1.5), 0.1, dilate=True)
    assert ch_d.sum() == 9 and ch_d[19:22, 29:32].all()                # dilation by one pixel


def _brute_pixel_weights(p, n, xs, ys):
    """exp(-1/2 d^T Sigma^-1 d) of Gaussian n at the given pixel centres: numpy's matrix inverse of Sigma = L L^T,
    no tile lists, no whitened coordinates (an independent formulation of c-1/c-3)."""
    Si = np.linalg.inv(oracle.cov_from_chol(p.chol[n]))
    d = np.stack([xs + 0.5 - p.mu[n, 0], ys + 0.5 - p.mu[n, 1]], 1)
    return np.exp(-0.5 * np.einsum("pi,ij,pj->p", d, Si, d))


def test_pixel_selection_against_brute_force():
    """the selection equals a brute-force evaluation of exp(-sigma) >= eps over all
    pixel x Gaussian pairs (float64, no tile lists) -- for eps above exp(-4.5) = 0.0111, where the
    restriction to a tile's list cannot bind (a pixel outside the 3-sigma box has weight < 0.0111).
    The oracle decides in float64 too, so the two agree exactly unless a weight is within 1e-12 of eps."""
    for seed in range(4):
        W, H, g, p = _tiny_scene(seed)
        r = np.random.default_rng(seed)
        changed = (r.uniform(size=(H, W)) < 0.01).astype(np.uint8)
        eps = 0.02
        _, _, act, na, wmax = oracle.pframe_select_pixels(W, H, p, np.zeros((H, W, 3), np.float32), 0.0, eps=eps,
                                                          changed=changed, want_wmax=True)
        ys, xs = np.nonzero(changed)
        brute = np.zeros(g.n, np.uint8)
        bmax = np.zeros(g.n)
        for n in range(g.n):
            w = _brute_pixel_weights(p, n, xs, ys)
            brute[n] = (w >= eps).any()
            bmax[n] = w.max()
        clear = np.abs(bmax - eps) > 1e-12
        assert np.array_equal(act[clear], brute[clear]) and clear.all()
        # wmax is the brute-force maximum wherever the maximum is reached inside a listed tile (weight >= exp(-4.5))
        inside = bmax >= np.exp(-4.5)
        assert np.allclose(wmax[inside], bmax[inside], rtol=1e-12, atol=0.0)
        assert np.array_equal(act, (wmax >= eps).astype(np.uint8))
        assert 0 < act.sum() < g.n


def test_pixel_selection_at_default_eps_what_the_tile_list_restriction_drops():
    """DESIGN.md §3 c-13 at the DEFAULT eps = 0.01 < exp(-4.5) = 0.0111: "listed in the pixel's tile" is part of
    the definition, so a changed pixel just outside a Gaussian's 3-sigma box can have 0.01 <= weight < 0.0111
    and not count.  Pin: against the brute force without tile lists the oracle never selects MORE; every
    Gaussian it misses is one whose qualifying changed pixels all have weight in [eps, exp(-4.5)) and lie in
    tiles that do not list it; and that happens for at most 2 % of the Gaussians on dense change maps."""
    e45 = float(np.exp(-4.5))
    dropped = total = 0
    for seed in range(6):
        W, H, g, p = _tiny_scene(seed)
        r = np.random.default_rng(100 + seed)
        changed = (r.uniform(size=(H, W)) < 0.3).astype(np.uint8)       # dense: box edges are hit often
        _, _, act, na, wmax = oracle.pframe_select_pixels(W, H, p, np.zeros((H, W, 3), np.float32), 0.0, eps=0.01,
                                                          changed=changed, want_wmax=True)
        rect, rng_o, lst_o = oracle.bin(W, H, p)
        TX = (W + 15) // 16
        ys, xs = np.nonzero(changed)
        tile_of_px = (ys // 16) * TX + xs // 16
        for n in range(g.n):
            w = _brute_pixel_weights(p, n, xs, ys)
            hit = w >= 0.01
            brute = bool(hit.any())
            assert not (act[n] and not brute)                            # never more than the brute force
            if brute and not act[n]:
                listed = set(np.nonzero([n in lst_o[rng_o[t]:rng_o[t + 1]] for t in range(len(rng_o) - 1)])[0].tolist())
                assert all(wi < e45 and int(t) not in listed for wi, t in zip(w[hit], tile_of_px[hit]))
                dropped += 1
            total += 1
    assert dropped <= 0.02 * total, (dropped, total)


def test_pixel_selection_all_changed_and_vs_tile_rule():
    W, H, g, p = _tiny_scene(5, n=30)
    allch = np.ones((H, W), np.uint8)
    _, _, act, na = oracle.pframe_select_pixels(W, H, p, np.zeros((H, W, 3), np.float32), 0.0, changed=allch)
    rect, _, lst = oracle.bin(W, H, p)
    listed = np.zeros(g.n, np.uint8)
    listed[np.unique(lst)] = 1
    assert np.array_equal(act, listed)                                   # union saturates
    # pixel-granular selection is a subset of the tile-granular one for the same changed content
    frame = np.clip(oracle.render(W, H, p), 0, 1).astype(np.float32)
    frame[17:20, 33:36] = 1.0 - frame[17:20, 33:36]                      # a 3x3 patch changes
    ch, resid, act_px, _ = oracle.pframe_select_pixels(W, H, p, frame, 0.2)
    assert 0 < ch.sum() <= 9
    TX = (W + 15) // 16
    tiles = np.unique((np.nonzero(ch)[0] // 16) * TX + np.nonzero(ch)[1] // 16)
    _, rng_o, lst_o = oracle.bin(W, H, p)
    tile_sel = np.zeros(g.n, np.uint8)
    for t in tiles:
        tile_sel[lst_o[rng_o[t]:rng_o[t + 1]]] = 1
    assert np.all(act_px <= tile_sel) and 0 < act_px.sum() < tile_sel.sum()
