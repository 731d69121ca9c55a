"""Pins for the oracle's ROI-restricted loss, PSNR, fit and selections (DESIGN.md §3 c-16; "encoding
only the region of interest").  None of them re-calls the function under test:
hand values, a numpy restatement over the masked pixels, finite differences, and the reductions to c-4 / c-9 / c-13
when the ROI covers the frame."""
import numpy as np
import pytest

import oracle
import workloads as wl


def _scene(W, H, N, seed):
    g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=5.0, opacity_range=(0.1, 0.6), config_index=seed, margin=4.0)
    return g, oracle.Params.from_f32(g)


def test_hand_values_and_reduction_to_the_full_frame():
    # image 0, target 16/255 inside a 2x2 ROI, anything outside: L = (16/255)^2, PSNR = 24.0484 dB
    # (the 16/255 example of SPEC.md:281 restricted to the ROI)
    img = np.zeros((4, 4, 3))
    tgt = np.full((4, 4, 3), 16 / 255, np.float32)
    tgt[0, 0] = 1.0
    tgt[3, 2] = 0.7
    roi = np.zeros((4, 4), np.uint8)
    roi[1:3, 1:3] = 1
    L, G = oracle.loss_roi(img, tgt, roi)
    t = float(np.float32(16 / 255))
    assert abs(L - t * t) < 1e-15
    assert abs(oracle.psnr_roi(img, tgt, roi) - 24.0484) < 2e-4
    assert np.all(G[roi == 0] == 0.0)
    assert np.allclose(G[roi != 0], -2.0 * t / 12.0, rtol=0, atol=1e-15)      # 2 (C - T) / (3 |M|), |M| = 4
    # a full ROI is c-4, bit for bit
    r = np.random.default_rng(0)
    img = r.uniform(-0.2, 1.3, (9, 7, 3))
    tgt = r.uniform(0, 1, (9, 7, 3)).astype(np.float32)
    ones = np.ones((9, 7), np.uint8)
    L0, G0 = oracle.loss(img, tgt)
    L1, G1 = oracle.loss_roi(img, tgt, ones)
    assert L0 == L1 and np.array_equal(G0, G1) and oracle.psnr(img, tgt) == oracle.psnr_roi(img, tgt, ones)
    with pytest.raises(ValueError):
        oracle.loss_roi(img, tgt, np.zeros((9, 7), np.uint8))


def test_numpy_restatement_and_finite_differences():
    r = np.random.default_rng(1)
    H, W = 13, 11
    img = r.uniform(-0.3, 1.4, (H, W, 3))
    tgt = r.uniform(0, 1, (H, W, 3)).astype(np.float32)
    roi = (r.uniform(size=(H, W)) < 0.4).astype(np.uint8)
    L, G = oracle.loss_roi(img, tgt, roi)
    m = roi.astype(bool)
    d = img - tgt.astype(np.float64)
    assert abs(L - (d[m] ** 2).mean()) < 1e-15
    mse = ((np.clip(img, 0, 1) - tgt.astype(np.float64))[m] ** 2).mean()
    assert abs(oracle.psnr_roi(img, tgt, roi) - 10 * np.log10(1 / mse)) < 1e-10
    for (y, x, ch) in [(0, 0, 0), (5, 3, 1), (12, 10, 2), (7, 7, 0)]:
        h = 1e-6
        a, b = img.copy(), img.copy()
        a[y, x, ch] += h
        b[y, x, ch] -= h
        fd = (oracle.loss_roi(a, tgt, roi)[0] - oracle.loss_roi(b, tgt, roi)[0]) / (2 * h)
        assert abs(fd - G[y, x, ch]) < 1e-9


def test_fit_with_roi_full_mask_is_the_plain_fit_and_outside_gaussians_do_not_move():
    W, H, N = 64, 48, 60
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 31))
    g, p = _scene(W, H, N, 32)
    a, b = oracle.Params.from_f32(g), oracle.Params.from_f32(g)
    ra = oracle.fit(W, H, a, frame, 15, lr=1e-2)
    rb = oracle.fit(W, H, b, frame, 15, lr=1e-2, roi=np.ones((H, W), np.uint8))
    assert ra.final_loss == rb.final_loss and np.array_equal(a.mu, b.mu) and np.array_equal(a.rgb, b.rgb)
    # ROI = the left 16 columns: a Gaussian none of whose tiles touches them has zero gradient and stays put
    roi = np.zeros((H, W), np.uint8)
    roi[:, :16] = 1
    c = oracle.Params.from_f32(g)
    rc = oracle.fit(W, H, c, frame, 15, lr=1e-2, roi=roi)
    _, rng, lst = oracle.bin(W, H, p)
    TX = (W + 15) // 16
    touched = np.zeros(N, bool)
    for t in range(len(rng) - 1):
        if t % TX == 0:
            touched[lst[rng[t]:rng[t + 1]]] = True
    far = ~touched
    # (membership is evaluated per iteration; Gaussians that start far and have zero gradient never move)
    assert far.any()
    assert np.array_equal(c.mu[far], p.mu[far]) and np.array_equal(c.chol[far], p.chol[far])
    assert np.array_equal(c.rgb[far], p.rgb[far])
    # the loss it reports is the ROI loss of its final render
    img = oracle.render(W, H, c)
    assert abs(rc.final_loss - oracle.loss_roi(img, frame, roi)[0]) < 1e-15
    assert rc.final_loss < oracle.loss_roi(oracle.render(W, H, p), frame, roi)[0]


def test_selections_with_roi():
    W, H, N = 80, 48, 150
    g, p = _scene(W, H, N, 41)
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 42))
    r = np.random.default_rng(3)
    roi = np.zeros((H, W), np.uint8)
    roi[8:40, 20:70] = 1
    roi[r.uniform(size=(H, W)) < 0.1] = 0
    tau = 0.15
    resid, flag, act, na = oracle.pframe_select(W, H, p, frame, tau, roi=roi)
    img = np.clip(oracle.render(W, H, p), 0, 1)
    TX, TY = (W + 15) // 16, (H + 15) // 16
    _, rng, lst = oracle.bin(W, H, p)
    want = np.zeros(N, np.uint8)
    for t in range(TX * TY):
        ys, xs = slice(16 * (t // TX), min(H, 16 * (t // TX) + 16)), slice(16 * (t % TX), min(W, 16 * (t % TX) + 16))
        m = roi[ys, xs].astype(bool)
        ref = np.abs(frame[ys, xs].astype(np.float64) - img[ys, xs])[m].mean() if m.any() else 0.0
        assert abs(resid[t] - ref) < 1e-12
        assert flag[t] == (ref > tau)
        if ref > tau:
            want[lst[rng[t]:rng[t + 1]]] = 1
    assert np.array_equal(act, want) and na == want.sum()
    # a full ROI is c-9
    r0 = oracle.pframe_select(W, H, p, frame, tau)
    r1 = oracle.pframe_select(W, H, p, frame, tau, roi=np.ones((H, W), np.uint8))
    assert np.array_equal(r0[0], r1[0]) and np.array_equal(r0[2], r1[2])
    # pixel-granular: the raw change map is the unrestricted one intersected with the ROI; dilation follows
    ch0, _, _, _ = oracle.pframe_select_pixels(W, H, p, frame, tau)
    ch, actp, nap = oracle.pframe_select_pixels_roi(W, H, p, frame, tau, roi)
    assert np.array_equal(ch != 0, (ch0 != 0) & (roi != 0))
    chd, _, _ = oracle.pframe_select_pixels_roi(W, H, p, frame, tau, roi, dilate=True)
    assert np.all(chd[ch != 0] == 1) and chd.sum() >= ch.sum()
    full = oracle.pframe_select_pixels_roi(W, H, p, frame, tau, np.ones((H, W), np.uint8))
    assert np.array_equal(full[1], oracle.pframe_select_pixels(W, H, p, frame, tau)[2])
    assert set(np.flatnonzero(actp)) <= set(np.flatnonzero(full[1]))
