"""Pins of the oracle's superpixel initialiser (c-11): the worked
examples SPEC.md gives, closed forms, brute force on tiny inputs, numpy's own mean / covariance on
the final labels, and the properties the paper claims for the initialisation."""
import numpy as np
import pytest

import oracle
import workloads as wl


def _cov(chol):
    l1, l2, l3 = chol
    return np.array([[l1 * l1, l1 * l2], [l1 * l2, l2 * l2 + l3 * l3]])


def test_spec_square_segment_covariance():
    """one 10x10 square of colour 0.5 -> mu at the centre, point covariance
    (10^2-1)/12 = 8.25 per axis; as unit squares +1/12: the continuous square's 100/12."""
    f = np.full((40, 40, 3), 0.5, np.float32)
    m = np.zeros((40, 40), np.uint8)
    m[10:20, 15:25] = 1
    mu, chol, rgb, op, lab, S = oracle.init_superpixel(f, m, 1)
    assert len(mu) == 1 and np.allclose(mu[0], [20.0, 15.0])
    assert np.allclose(_cov(chol[0]), np.diag([8.25 + 1 / 12, 8.25 + 1 / 12]), atol=1e-5)
    assert np.allclose(rgb[0], 0.5, atol=1e-5) and op[0] == 1.0
    assert (lab >= 0).sum() == 100 and np.all(lab[m == 0] == -1) and np.all(lab[m == 1] == 0)


def test_degenerate_segments():
    f = np.random.default_rng(0).uniform(0, 1, (12, 20, 3)).astype(np.float32)
    m = np.zeros((12, 20), np.uint8)
    m[5, 7] = 1                                   # one pixel
    mu, chol, rgb, _, _, _ = oracle.init_superpixel(f, m, 1)
    assert np.allclose(mu[0], [7.5, 5.5]) and np.allclose(_cov(chol[0]), np.eye(2) / 12, atol=1e-6)
    assert np.allclose(rgb[0], f[5, 7], atol=1e-5)
    m[:] = 0
    m[4, 3:12] = 1                                # a horizontal line of 9 pixels
    mu, chol, _, _, _, _ = oracle.init_superpixel(f, m, 1)
    assert np.allclose(_cov(chol[0]), np.diag([(81 - 1) / 12 + 1 / 12, 1 / 12]), atol=1e-5)
    with pytest.raises(ValueError):
        oracle.init_superpixel(f, np.zeros((12, 20), np.uint8), 4)


def test_spec_examples_of_the_segmentation():
    f = np.full((30, 50, 3), 0.3, np.float32)
    m = np.zeros((30, 50), np.uint8)
    m[3:27, 4:40] = 1
    _, _, _, _, lab, _ = oracle.init_superpixel(f, m, 1)          # uniform ROI, N = 1
    assert set(np.unique(lab[m == 1])) == {0}
    # two separated uniform blobs, N = 2, high compactness -> one segment per blob
    f2 = np.zeros((24, 60, 3), np.float32)
    m2 = np.zeros((24, 60), np.uint8)
    f2[6:16, 4:14] = (0.9, 0.1, 0.1)
    m2[6:16, 4:14] = 1
    f2[6:16, 44:54] = (0.1, 0.1, 0.9)
    m2[6:16, 44:54] = 1
    mu, _, rgb, _, lab, _ = oracle.init_superpixel(f2, m2, 2, compactness=40)
    assert len(mu) == 2
    assert len(np.unique(lab[6:16, 4:14])) == 1 and len(np.unique(lab[6:16, 44:54])) == 1
    assert lab[8, 8] != lab[8, 48]
    assert np.allclose(rgb[lab[8, 8]], (0.9, 0.1, 0.1), atol=1e-4)
    # N = ROI pixel count -> every pixel its own segment
    m3 = np.zeros((10, 10), np.uint8)
    m3[2:5, 3:7] = 1
    f3 = np.random.default_rng(1).uniform(0, 1, (10, 10, 3)).astype(np.float32)
    mu, _, rgb, _, lab, grid = oracle.init_superpixel(f3, m3, 12)
    assert grid == (4, 3) and len(mu) == 12 and len(np.unique(lab[m3 == 1])) == 12
    ys, xs = np.nonzero(m3)
    assert np.allclose(mu[lab[ys, xs]], np.stack([xs + 0.5, ys + 0.5], 1))


def _features(frame, ys, xs):
    q = np.floor(255.0 * frame[ys, xs].astype(np.float32) + np.float32(0.5)).astype(np.int64)
    return np.concatenate([np.stack([16 * xs + 8, 16 * ys + 8], 1), 16 * q], 1)


def test_seeds_and_first_assignment_brute_force():
    """iters = 0: labels come from the seeds alone.  Brute force in numpy with an independent
    formulation: seeds = the ROI pixel nearest each occupied cell's centre, assignment = argmin of
    the SLIC distance over ALL seeds (with a high compactness the 3x3 restriction never binds)."""
    frame, mask = wl.talking_head_frame(wl.scaled_spec(96, 64, 90))
    N, m = 40, 60
    mu, chol, rgb, op, lab, (GX, GY) = oracle.init_superpixel(frame, mask, N, compactness=m, iters=0)
    ys, xs = np.nonzero(mask)
    x0, y0 = xs.min(), ys.min()
    bw, bh = xs.max() - x0 + 1, ys.max() - y0 + 1
    assert GY == max(1, int(np.floor(GX * bh / bw + 0.5)))

    def occupied(gx):
        gy = max(1, int(np.floor(gx * bh / bw + 0.5)))
        return len(np.unique(((ys - y0) * gy // bh) * 100_000 + (xs - x0) * gx // bw))

    assert occupied(GX) <= N < occupied(GX + 1)            # the finest grid that fits (K grows with GX here)
    cxs, cys = (xs - x0) * GX // bw, (ys - y0) * GY // bh
    cell = cys * 100_000 + cxs
    seeds = []
    for c in np.unique(cell):                               # ascending cell id = ascending cluster index
        sel = np.nonzero(cell == c)[0]
        # the cell's centre: midpoint of the pixel centres of its first and last column / row
        cx, cy = c % 100_000, c // 100_000
        colx = np.nonzero(np.arange(bw) * GX // bw == cx)[0]
        rowy = np.nonzero(np.arange(bh) * GY // bh == cy)[0]
        mx = x0 + 0.5 * (colx[0] + colx[-1]) + 0.5
        my = y0 + 0.5 * (rowy[0] + rowy[-1]) + 0.5
        d = (xs[sel] + 0.5 - mx) ** 2 + (ys[sel] + 0.5 - my) ** 2
        seeds.append(sel[np.argmin(d)])                     # first minimum = smallest row-major index
    assert len(seeds) == len(mu) <= N
    F = _features(frame, ys, xs).astype(np.float64)
    Cn = F[seeds]
    S2 = max(1, (bw * bh) // (GX * GY))
    D = S2 * ((F[:, None, 2:] - Cn[None, :, 2:]) ** 2).sum(-1) + (m * m) * ((F[:, None, :2] - Cn[None, :, :2]) ** 2).sum(-1)
    brute = np.argmin(D, axis=1)
    got = lab[ys, xs]
    # the oracle drops clusters that ended up empty; with iters = 0 every seed keeps itself
    assert np.array_equal(got, brute)


def test_segment_statistics_against_numpy_and_partition():
    frame, mask = wl.talking_head_frame(wl.scaled_spec(160, 96, 91))
    N = 120
    mu, chol, rgb, op, lab, S = oracle.init_superpixel(frame, mask, N, compactness=10, iters=10)
    K = len(mu)
    assert 0 < K <= N and np.all(op == 1.0)
    assert np.all(lab[mask == 0] == -1) and np.all(lab[mask != 0] >= 0)
    assert np.array_equal(np.unique(lab[mask != 0]), np.arange(K))          # every segment non-empty
    ys, xs = np.nonzero(mask)
    for k in range(0, K, 7):
        s = lab[ys, xs] == k
        P = np.stack([xs[s] + 0.5, ys[s] + 0.5])
        assert np.allclose(mu[k], P.mean(1), atol=1e-4)
        cov = np.atleast_2d(np.cov(P, bias=True)) if s.sum() > 1 else np.zeros((2, 2))
        assert np.allclose(_cov(chol[k]), cov + np.eye(2) / 12, atol=1e-3)
        assert np.allclose(rgb[k], frame[ys[s], xs[s]].mean(0), atol=2e-5)


def test_kmeans_objective_does_not_increase():
    frame, mask = wl.talking_head_frame(wl.scaled_spec(128, 96, 92))
    ys, xs = np.nonzero(mask)
    F = _features(frame, ys, xs).astype(np.float64)
    prev = None
    for it in (0, 1, 2, 4, 8):
        _, _, _, _, lab, (GX, GY) = oracle.init_superpixel(frame, mask, 60, compactness=10, iters=it)
        S2 = max(1, ((xs.max() - xs.min() + 1) * (ys.max() - ys.min() + 1)) // (GX * GY))
        l = lab[ys, xs]
        obj = 0.0
        for k in np.unique(l):
            Fk = F[l == k]
            c = Fk.mean(0)
            obj += S2 * ((Fk[:, 2:] - c[2:]) ** 2).sum() + 100.0 * ((Fk[:, :2] - c[:2]) ** 2).sum()
        if prev is not None:
            assert obj <= prev * 1.001
        prev = obj


def test_superpixel_init_renders_closer_than_sampled_init():
    """The paper's point (Table 1 direction): Gaussians placed from the
    superpixels start nearer the frame than the same number of sampled Gaussians."""
    W, H, N = 160, 96, 150
    frame, mask = wl.talking_head_frame(wl.scaled_spec(W, H, 93), noise_sigma=0.0)
    target = frame * (mask[..., None] != 0)
    mu, chol, rgb, op, _, _ = oracle.init_superpixel(frame, mask, N)
    pa = oracle.Params.from_f32(wl.GaussianSet(mu, chol, rgb, op))
    mu2, chol2, rgb2, op2, _ = oracle.init_roi(frame, np.where(mask != 0, 1, 0).astype(np.uint8), len(mu), 3, 1.0, 4.0)
    pb = oracle.Params.from_f32(wl.GaussianSet(mu2, chol2, rgb2, op2))
    a = oracle.psnr(oracle.render(W, H, pa), target)
    b = oracle.psnr(oracle.render(W, H, pb), target)
    assert a > b + 1.0, (a, b)
    # ... and stay ahead after the same number of fit iterations (Table 1's direction)
    fa = oracle.fit(W, H, pa, target, 40, lr=1e-2).psnr
    fb = oracle.fit(W, H, pb, target, 40, lr=1e-2).psnr
    assert fa > fb, (fa, fb)
