"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(configs[2]: 1920x1080 / 50,000 Gaussians from gs_init_roi; configs[4]: 1920x1080 / 70,000 and
3840x2160 / 200,000 random sets).  Bins are compared in full and bit for bit (the oracle's
binning is cheap); pixels on sampled tiles and gradients on sampled Gaussians, which the oracle
computes one by one; the loss over the whole frame; one fit iteration on sampled Gaussians.
Also: the code paths the small cases do not reach (lists longer than one shared-memory chunk in
team and single-warp mode, frames whose rows cannot be bulk-copied)."""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

GROUPS = {"mu": slice(0, 2), "chol": slice(2, 5), "rgb": slice(5, 8), "opacity": slice(8, 9)}


@pytest.fixture(scope="module")
def gs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2505_09324_b200 as gs
    gs.lib()
    return gs


def _np(t):
    return t.detach().cpu().numpy()


def _gset(p):
    return wl.GaussianSet(_np(p.mu), _np(p.chol), _np(p.rgb), _np(p.opacity))


def _assert_bins(gs, ctx, W, H, g):
    _, rng_o, lst_o = oracle.bin(W, H, oracle.Params.from_f32(g))
    rng_g, lst_g = gs.gs_get_bins(ctx)
    assert np.array_equal(_np(rng_g), rng_o)
    assert np.array_equal(_np(lst_g), lst_o)
    return rng_o, lst_o


def _tile_pixels(img, W, H, t):
    TX = (W + 15) // 16
    tx, ty = t % TX, t // TX
    return img[ty * 16:min(H, ty * 16 + 16), tx * 16:min(W, tx * 16 + 16)]


def _sample_tiles(rng_o, k, seed):
    """k tiles: the longest lists, the frame's last (partial) tiles, and random ones."""
    n = np.diff(rng_o)
    T = len(n)
    r = np.random.default_rng(seed)
    pick = set(np.argsort(-n)[:k // 4].tolist()) | {T - 1, T - 2, 0} | set(r.integers(0, T, k).tolist())
    return np.array(sorted(pick))[: k + 8]


def _assert_grads(a, b, rel=1e-3, floor=1e-4, scale_from=None):
    ref = b if scale_from is None else scale_from
    for name, sl in GROUPS.items():
        scale = np.abs(ref[:, sl]).max()
        tol = rel * np.abs(b[:, sl]) + floor * scale + 1e-30
        bad = np.abs(a[:, sl] - b[:, sl]) > tol
        assert not bad.any(), (name, int(bad.sum()), float(np.abs(a[:, sl] - b[:, sl]).max()), float(scale))


# ------------------------------------------------------------------ configs[2]: 1080p fit

@pytest.fixture(scope="module")
def fit1080(gs):
    W, H, N = 1920, 1080, 50_000
    frame, mask = wl.talking_head_frame(wl.SPEC_1080P, 0)
    ctx = gs.Context(W, H, N, max_pairs=1_000_000)
    fd = torch.as_tensor(frame).cuda()
    p = gs.gs_init_roi(ctx, fd, torch.as_tensor(mask).cuda(), N, 1, 1.0, 8.0)
    yield gs, ctx, W, H, N, frame, fd, p
    ctx.close()


def test_full_size_fit_bins_pixels_loss(fit1080):
    gs, ctx, W, H, N, frame, fd, p = fit1080
    g = _gset(p)
    po = oracle.Params.from_f32(g)
    img = _np(gs.gs_render(ctx, p))
    rng_o, lst_o = _assert_bins(gs, ctx, W, H, g)
    assert len(lst_o) > 200_000 and np.diff(rng_o).max() > 128        # the head tiles are crowded
    tiles = _sample_tiles(rng_o, 48, 0)
    ref = oracle.render(W, H, po, tiles=tiles)
    for t in tiles:
        # the initial image is saturated (colours from the frame add up): values reach ~100, so the
        # 1e-4 absolute bar is taken relative to max(1, |C|) (binary32 sums of ~170 terms)
        a, b = _tile_pixels(img, W, H, t), _tile_pixels(ref, W, H, t)
        assert np.all(np.abs(a - b) <= 1e-4 * np.maximum(1.0, np.abs(b))), int(t)
    # loss and PSNR over the whole frame against the oracle's full render
    full = oracle.render(W, H, po)
    L, _ = oracle.loss(full, frame)
    loss, psnr = gs.gs_loss_psnr(ctx, fd, p)
    assert abs(loss - L) <= 1e-5 * L
    assert abs(psnr - oracle.psnr(full, frame)) < 1e-3


def test_full_size_backward_sampled_gaussians(fit1080):
    gs, ctx, W, H, N, frame, fd, p = fit1080
    g = _gset(p)
    po = oracle.Params.from_f32(g)
    G = wl.random_image_grad(W, H, 62)
    got = _np(gs.gs_render_backward(ctx, p, torch.as_tensor(G).cuda()).flat9())
    r = np.random.default_rng(5)
    # sampled Gaussians, among them the ones listed in the most crowded tile
    _, rng_o, lst_o = oracle.bin(W, H, po)
    tmax = int(np.argmax(np.diff(rng_o)))
    subset = np.unique(np.concatenate([r.integers(0, N, 400), lst_o[rng_o[tmax]:rng_o[tmax] + 64]]))
    ref = oracle.backward(W, H, po, G.astype(np.float64), subset=subset)
    _assert_grads(got[subset], ref[subset])


def test_full_size_fit_iteration_sampled_gaussians(fit1080):
    """One iteration of the timed loop (gs_fit_steps, resume=1: fit-tiles kernel + fused Adam/bin)
    at full size: gradients of the L2 loss on sampled Gaussians through the Adam step, and the bins
    the fused Adam kernel leaves for the next iteration, bit for bit."""
    gs, ctx, W, H, N, frame, fd, p = fit1080
    q = p.clone()
    g = _gset(q)
    po = oracle.Params.from_f32(g)
    _, Go = oracle.loss(oracle.render(W, H, po), frame)
    r = np.random.default_rng(6)
    subset = np.unique(r.integers(0, N, 300))
    gref = oracle.backward(W, H, po, Go, subset=subset)
    st = gs.AdamState.zeros(N)
    gs.gs_fit_steps(ctx, fd, q, st, 1, t0=1, lr=1e-2, resume=True)
    assert gs.gs_status(ctx) == 0
    # first Adam step from zero moments: m = (1 - beta1) g  ->  the kernel's gradient is m / 0.1
    got = _np(st.m)[subset] / (1.0 - np.float32(0.9))
    _assert_grads(got, gref[subset], scale_from=gref[subset])
    # parameters moved by -lr * g / (|g| + eps) (c-6, first step from zero moments); compared where
    # |g| >> eps (elsewhere the step is ill-conditioned in g), up to the binary32 spacing of theta
    before = _np(p.flat9())[subset].astype(np.float64)
    step = _np(q.flat9())[subset].astype(np.float64) - before
    gs_ = gref[subset]
    exp = -1e-2 * gs_ / (np.abs(gs_) + 1e-8)
    big = np.abs(gs_) > 1e-6
    big[:, 2] = big[:, 4] = False                      # l1, l3 may be clipped by the projection
    tol = 3e-5 + 1.3e-7 * np.abs(before)
    assert np.all(np.abs(step - exp)[big] <= tol[big])
    _assert_bins(gs, ctx, W, H, _gset(q))               # bins left by the fused Adam kernel


# ------------------------------------------------------------------ configs[4]: decode stress

@pytest.mark.parametrize("W,H,N", [(1920, 1080, 70_000), (3840, 2160, 200_000)])
def test_full_size_decode_bins_and_sampled_tiles(gs, W, H, N):
    g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=16.0, config_index=4)
    ctx = gs.Context(W, H, N, max_pairs=6_000_000)
    p = gs.Params.from_numpy(g)
    dec = _np(gs.gs_decode(ctx, p))
    rng_o, lst_o = _assert_bins(gs, ctx, W, H, g)
    assert gs.gs_status(ctx) == 0
    tiles = _sample_tiles(rng_o, 40, 1)
    ref = np.clip(oracle.render(W, H, oracle.Params.from_f32(g), tiles=tiles), 0.0, 1.0)
    for t in tiles:
        assert np.abs(_tile_pixels(dec, W, H, t) - _tile_pixels(ref, W, H, t)).max() < 1e-4, int(t)
    assert dec.min() >= 0.0 and dec.max() <= 1.0
    # decode is bit-reproducible (lists are summed in ascending id order)
    assert torch.equal(gs.gs_decode(ctx, p), torch.as_tensor(dec).cuda())
    ctx.close()


# ------------------------------------------------------------------ paths the small cases miss

def test_long_lists_team_and_single_warp_streaming(gs):
    """Tiles listed far beyond one shared-memory chunk (64 entries): the CTA team streams slices of
    more than one chunk, and -- on the first launch of a context, when every tile is still filed as
    short -- a single warp streams the whole list.  Forward + loss + backward against the oracle."""
    W, H, N = 160, 96, 2400
    g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=4.0, opacity_range=(0.002, 0.01), config_index=81)
    g.mu[:1500] = np.array([72.0, 40.0]) + np.random.default_rng(2).uniform(-6, 6, (1500, 2))
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 82))
    po = oracle.Params.from_f32(g)
    _, rng_o, _ = oracle.bin(W, H, po)
    assert np.diff(rng_o).max() > 1024                # slices of > 256 entries per warp
    _, Go = oracle.loss(oracle.render(W, H, po), frame)
    gref = oracle.backward(W, H, po, Go)
    fd = torch.as_tensor(frame).cuda()
    for launches_before in (0, 1):                     # 0: all tiles filed as short; 1: classes known
        ctx = gs.Context(W, H, N, max_pairs=400_000)
        p = gs.Params.from_numpy(g)
        if launches_before:
            gs.gs_render(ctx, p)
        st = gs.AdamState.zeros(N)
        gs.gs_fit_steps(ctx, fd, p, st, 1, t0=1, lr=0.0)
        assert gs.gs_status(ctx) == 0
        got = _np(st.m) / (1.0 - np.float32(0.9))
        _assert_grads(got, gref)
        Gt = torch.as_tensor(Go.astype(np.float32)).cuda()
        _assert_grads(_np(gs.gs_render_backward(ctx, p, Gt).flat9()), gref)
        ctx.close()


@pytest.mark.parametrize("W,H", [(150, 70), (333, 95)])
def test_fit_iteration_on_frames_without_tensor_map(gs, W, H):
    """Row pitch not a multiple of 16 bytes: the fit kernel loads target rows with plain loads."""
    N = 900
    g = wl.random_gaussians(N, W, H, s_min=1.5, s_max=6.0, opacity_range=(0.1, 0.5), config_index=83, margin=8.0)
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 84))
    po = oracle.Params.from_f32(g)
    L, Go = oracle.loss(oracle.render(W, H, po), frame)
    gref = oracle.backward(W, H, po, Go)
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    st = gs.AdamState.zeros(N)
    gs.gs_fit_steps(ctx, torch.as_tensor(frame).cuda(), p, st, 1, t0=1, lr=0.0)
    _assert_grads(_np(st.m) / (1.0 - np.float32(0.9)), gref)
    loss, _ = gs.gs_loss_psnr(ctx, torch.as_tensor(frame).cuda(), p)
    assert abs(loss - L) <= 1e-5 * L
    ctx.close()


@pytest.mark.parametrize("frac", [0.3, 0.02])
def test_masked_fit_iteration_selective_refit(gs, frac):
    """Selective refit (P-frames): with an active mask the fit kernel produces gradients only for
    active Gaussians (frozen list entries are dropped before the backward pass, tiles without an
    active Gaussian are skipped); those gradients equal the oracle's, frozen rows stay untouched."""
    W, H, N = 320, 208, 3000
    g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=6.0, opacity_range=(0.05, 0.3), config_index=85, margin=6.0)
    g.mu[:400] = np.array([150.0, 100.0]) + np.random.default_rng(3).uniform(-10, 10, (400, 2))   # team tiles
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 86))
    po = oracle.Params.from_f32(g)
    _, Go = oracle.loss(oracle.render(W, H, po), frame)
    gref = oracle.backward(W, H, po, Go)
    r = np.random.default_rng(4)
    act = (r.uniform(size=N) < frac).astype(np.uint8)
    if frac < 0.1:
        act[:] = 0
        act[(g.mu[:, 0] < 64) & (g.mu[:, 1] < 64)] = 1          # a corner region: most tiles idle
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    gs.gs_render(ctx, p)                                         # files the tiles under their classes
    st = gs.AdamState.zeros(N)
    before = p.flat9().clone()
    gs.gs_fit_steps(ctx, torch.as_tensor(frame).cuda(), p, st, 1, t0=1, lr=1e-2, active=torch.as_tensor(act).cuda())
    assert gs.gs_status(ctx) == 0
    a = act.astype(bool)
    got = _np(st.m) / (1.0 - np.float32(0.9))
    _assert_grads(got[a], gref[a], scale_from=gref)
    assert np.all(_np(st.m)[~a] == 0.0) and np.all(_np(st.v)[~a] == 0.0)
    fz = torch.as_tensor(~a).cuda()
    assert torch.equal(p.flat9()[fz], before[fz])
    assert not torch.equal(p.flat9()[~fz], before[~fz])
    ctx.close()


# ------------------------------------------------------------------ configs[1], configs[3]: PSNR parity of whole fits

def test_iframe_fit_roi_config_psnr_parity(gs):
    """configs[1] in full: 480x272, 4,096 Gaussians from the ROI initialiser (70 % in the ROI by Sobel
    weight), scales [1,4], lr 1e-2, 1,000 iterations; PSNR within 0.05 dB of the oracle's fit of the
    same initial set."""
    W, H, N = 480, 272, 4096
    frame, mask = wl.talking_head_frame(wl.SPEC_ROI)
    mu, chol, rgb, op, _ = oracle.init_roi(frame, mask, N, 11, 1.0, 4.0)
    g = wl.GaussianSet(mu, chol, rgb, op)
    po = oracle.Params.from_f32(g)
    rep_o = oracle.fit(W, H, po, frame, 1000, lr=1e-2)
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    st = gs.AdamState.zeros(N)
    rep = gs.gs_encode_iframe(ctx, torch.as_tensor(frame).cuda(), p, st, 1000, lr=1e-2)
    assert rep.status == 0 and rep.iters_run == 1000
    assert abs(rep.psnr - rep_o.psnr) < 0.05, (rep.psnr, rep_o.psnr)
    assert rep.psnr > 25.0
    ctx.close()


def test_pframe_sequence_psnr_parity(gs):
    """configs[3] scaled to 480x272 and 4 frames: frame 0 as an I-frame (300 iterations), then P-frames
    that reuse the previous Gaussians and refit the selected subset (100 iterations), head moving
    2 px and 0.5 deg per frame, fresh noise.  tau at the 85th percentile of the oracle's first
    P-frame residuals (configs[3]'s 0.02 is at the noise floor and selects everything).  Per frame:
    PSNR within 0.05 dB, selected counts within 2 %."""
    W, H, N = 480, 272, 4096
    spec = wl.FrameSpec(W, H, (240.0, 119.0), (59.5, 76.5), True, 3)
    frames = [wl.talking_head_frame(spec, k) for k in range(4)]
    mu, chol, rgb, op, _ = oracle.init_roi(frames[0][0], frames[0][1], N, 12, 1.0, 4.0)
    g = wl.GaussianSet(mu, chol, rgb, op)
    po = oracle.Params.from_f32(g)
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    st = gs.AdamState.zeros(N)
    r_o = oracle.fit(W, H, po, frames[0][0], 300, lr=1e-2)
    r_g = gs.gs_encode_iframe(ctx, torch.as_tensor(frames[0][0]).cuda(), p, st, 300, lr=1e-2)
    assert abs(r_g.psnr - r_o.psnr) < 0.05
    tau = float(np.quantile(oracle.pframe_select(W, H, po, frames[1][0], 0.02)[0], 0.85))
    for k in (1, 2, 3):
        act_o, r_o = oracle.encode_pframe(W, H, po, frames[k][0], tau, 100, lr=1e-2)
        act_g, r_g = gs.gs_encode_pframe(ctx, torch.as_tensor(frames[k][0]).cuda(), p, st, tau, 100, lr=1e-2)
        assert r_g.status == 0 and r_g.iters_run == 100
        assert 0 < r_o.n_active < N
        assert abs(r_g.n_active - r_o.n_active) <= 0.02 * N, (k, r_g.n_active, r_o.n_active)
        assert abs(r_g.psnr - r_o.psnr) < 0.05, (k, r_g.psnr, r_o.psnr)
    ctx.close()


def test_iframe_fit_1080p_psnr_parity(fit1080):
    """configs[2] at full size, a bounded number of iterations (the oracle needs ~0.15 s per
    iteration on 16 cores): 60 iterations of the I-frame fit from the same initial set, PSNR within
    0.05 dB and loss within 2 %."""
    gs, ctx, W, H, N, frame, fd, p = fit1080
    q = p.clone()
    po = oracle.Params.from_f32(_gset(q))
    rep_o = oracle.fit(W, H, po, frame, 60, lr=1e-2)
    st = gs.AdamState.zeros(N)
    rep = gs.gs_encode_iframe(ctx, fd, q, st, 60, lr=1e-2)
    assert rep.status == 0 and rep.iters_run == 60
    assert abs(rep.psnr - rep_o.psnr) < 0.05, (rep.psnr, rep_o.psnr)
    assert abs(rep.final_loss - rep_o.final_loss) < 2e-2 * rep_o.final_loss


# ------------------------------------------------------------------ configs[2], configs[3] at their stated sizes and iteration counts

def _fullsize_golden():
    """tests/golden/fullsize_oracle.json, written by tests/golden/make_fullsize_oracle.py (oracle/ only)."""
    import json
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fullsize_oracle.json")
    with open(path) as f:
        return json.load(f)


def _init_sha(mu, chol, rgb, op):
    import hashlib
    h = hashlib.sha256()
    for a in (mu, chol, rgb, op):
        h.update(np.ascontiguousarray(a, dtype=np.float32).tobytes())
    return h.hexdigest()


def test_config2_full_2000_iterations_psnr_parity(gs):
    """configs[2] IN FULL: 1920x1080, 50,000 Gaussians from the ROI initialiser, 2,000
    fwd+bwd+Adam iterations, lr 1e-2.  The oracle's fit of this initial set is stored (make_fullsize_oracle.py:
    ~5 min of float64 on 16 cores); the initial set is regenerated here by the oracle's initialiser and must
    hash to the stored SHA-256, so both sides start from the same arrays.  PSNR within 0.05 dB, loss within 2 %."""
    gold = _fullsize_golden()["config2"]
    W, H, N = 1920, 1080, 50_000
    frame, mask = wl.talking_head_frame(wl.SPEC_1080P, 0)
    mu, chol, rgb, op, _ = oracle.init_roi(frame, mask, N, gold["init_seed"], 1.0, 8.0)
    assert _init_sha(mu, chol, rgb, op) == gold["init_sha256"], "the oracle's initial set differs from the stored run"
    ctx = gs.Context(W, H, N, max_pairs=1_000_000)
    fd = torch.as_tensor(frame).cuda()
    p = gs.Params.from_numpy(wl.GaussianSet(mu, chol, rgb, op))
    st = gs.AdamState.zeros(N)
    rep = gs.gs_encode_iframe(ctx, fd, p, st, gold["iters"], lr=1e-2)
    assert rep.status == 0 and rep.iters_run == gold["iters"]
    assert abs(rep.psnr - gold["psnr"]) < 0.05, (rep.psnr, gold["psnr"])
    assert abs(rep.final_loss - gold["final_loss"]) < 2e-2 * gold["final_loss"], (rep.final_loss, gold["final_loss"])
    ctx.close()


def test_config3_1080p_sequence_psnr_and_selection_parity(gs):
    """configs[3] at 1080p: frame 0 as an I-frame of 2,000 iterations, then three P-frames of
    200 iterations each on the Gaussians the tile-residual rule selects at the config's tau = 0.02.  Against
    the stored oracle run of the same initial set: per-frame PSNR within 0.05 dB, selected count within 2 % of N."""
    gold = _fullsize_golden()["config3"]
    W, H, N = 1920, 1080, 50_000
    frames = [wl.talking_head_frame(wl.SPEC_PSEQ, k) for k in range(4)]
    mu, chol, rgb, op, _ = oracle.init_roi(frames[0][0], frames[0][1], N, gold["init_seed"], 1.0, 8.0)
    assert _init_sha(mu, chol, rgb, op) == gold["init_sha256"], "the oracle's initial set differs from the stored run"
    ctx = gs.Context(W, H, N, max_pairs=1_000_000)
    p = gs.Params.from_numpy(wl.GaussianSet(mu, chol, rgb, op))
    st = gs.AdamState.zeros(N)
    rep = gs.gs_encode_iframe(ctx, torch.as_tensor(frames[0][0]).cuda(), p, st, gold["iframe_iters"], lr=1e-2)
    assert rep.status == 0 and abs(rep.psnr - gold["iframe"]["psnr"]) < 0.05, (rep.psnr, gold["iframe"]["psnr"])
    for g in gold["pframes"]:
        k = g["frame"]
        act, r = gs.gs_encode_pframe(ctx, torch.as_tensor(frames[k][0]).cuda(), p, st, gold["tau"],
                                     gold["pframe_iters"], lr=1e-2)
        assert r.status == 0 and r.iters_run == g["iters_run"]
        assert abs(r.n_active - g["n_active"]) <= 0.02 * N, (k, r.n_active, g["n_active"])
        assert abs(r.psnr - g["psnr"]) < 0.05, (k, r.psnr, g["psnr"])
    ctx.close()


def test_strict_pixel_bar_after_300_iterations_render_and_fit_forward(fit1080):
    """The 1e-4 ABSOLUTE pixel bar of north_star (Eq. 2) at 1080p x 50k on an unsaturated set:
    after 300 fit iterations the image is in [0,1] (the saturated initial image needed a relative bar).
    (1) gs_render on sampled tiles against the oracle's render of the same parameters: |dC| <= 1e-4, strictly;
    (2) the FIT kernel's own forward pass, seen through the per-tile sums of (C - T)^2 it leaves
        (gs_get_tile_loss after one more iteration with lr = 0): within what a per-pixel error of 1e-4 allows,
        sum_tile (2 |C - T| 1e-4 + 1e-8), and within 2e-5 relative (binary32 sums of 768 squares)."""
    gs, ctx, W, H, N, frame, fd, p = fit1080
    q = p.clone()
    st = gs.AdamState.zeros(N)
    gs.gs_fit_steps(ctx, fd, q, st, 300, t0=1, lr=1e-2, resume=True)
    gs.gs_fit_steps(ctx, fd, q, st, 1, t0=301, lr=0.0, resume=True)       # lr = 0: q unchanged, the kernel's forward of q
    sq_fit = _np(gs.gs_get_tile_loss(ctx))
    assert gs.gs_status(ctx) == 0
    po = oracle.Params.from_f32(_gset(q))
    img = _np(gs.gs_render(ctx, q))
    rng_o, lst_o = _assert_bins(gs, ctx, W, H, _gset(q))
    tiles = _sample_tiles(rng_o, 64, 3)
    ref = oracle.render(W, H, po, tiles=tiles)
    assert float(ref.max()) < 1.5                                          # no longer saturated
    for t in tiles:
        a, b = _tile_pixels(img, W, H, t), _tile_pixels(ref, W, H, t)
        assert np.abs(a - b).max() <= 1e-4, (int(t), float(np.abs(a - b).max()))
        d = b - _tile_pixels(frame, W, H, t).astype(np.float64)
        sq_ref = float((d * d).sum())
        allow = float((2e-4 * np.abs(d) + 1e-8).sum())
        assert abs(sq_fit[t] - sq_ref) <= allow, (int(t), sq_fit[t], sq_ref, allow)
        assert abs(sq_fit[t] - sq_ref) <= 2e-5 * sq_ref + 1e-9, (int(t), sq_fit[t], sq_ref)


# ------------------------------------------------------------------ run-to-run reproducibility of a fit (waiver, bounded)

def test_fit_run_to_run_spread_is_bounded(gs):
    """The fit is reproducible to rounding, not bit for bit (DESIGN.md §3 "Determinism"): tile lists are summed in
    arrival order and gradient moments meet in binary32 atomics.  This bounds what that costs: three runs of the
    same 300-iteration fit of configs[1] end within 0.005 dB of each other, within 2e-3 in 99.9 % of the parameters
    and within one learning rate (1e-2: an Adam step never exceeds lr, and where a gradient is at rounding level
    the sign of m / sqrt(v) follows the summation order, so single entries drift by a fraction of a step per
    iteration -- 2.5e-3 was seen on one B200 lease, 1.6e-3 on others) in every one, and the quantised codes a bitstream would carry (16 / 6 / 8 bits) differ in under 1 % of the values, by one
    level.  Renders (gs_render, gs_decode) ARE bit-reproducible: their lists are sorted first."""
    W, H, N = 480, 272, 4096
    frame, mask = wl.talking_head_frame(wl.SPEC_ROI)
    mu, chol, rgb, op, _ = oracle.init_roi(frame, mask, N, 11, 1.0, 4.0)
    g = wl.GaussianSet(mu, chol, rgb, op)
    fd = torch.as_tensor(frame).cuda()
    ctx = gs.Context(W, H, N)
    spec = wl.uniform_quant_spec(W, H)
    levels, lo, step, inv = spec
    runs, psnrs, codes = [], [], []
    for _ in range(3):
        p = gs.Params.from_numpy(g)
        rep = gs.gs_encode_iframe(ctx, fd, p, gs.AdamState.zeros(N), 300, lr=1e-2)
        assert rep.status == 0
        psnrs.append(rep.psnr)
        flat = _np(p.flat9()).astype(np.float64)
        runs.append(flat)
        q = _np(gs.gs_fake_quantize(ctx, p, spec).flat9()).astype(np.float64)
        on = levels > 0
        codes.append(np.rint((q[:, on] - lo[on].astype(np.float64)) / step[on].astype(np.float64)).astype(np.int64))
        assert torch.equal(gs.gs_decode(ctx, p), gs.gs_decode(ctx, p))
    assert max(psnrs) - min(psnrs) < 0.005, psnrs
    for k in (1, 2):
        dp = np.abs(runs[k] - runs[0])
        assert np.quantile(dp, 0.999) < 2e-3 and dp.max() < 1e-2, (float(np.quantile(dp, 0.999)), float(dp.max()))
        d = np.abs(codes[k] - codes[0])
        assert d.max() <= 1 and (d != 0).mean() < 0.01, (int(d.max()), float((d != 0).mean()))
    ctx.close()


# ------------------------------------------------------------------ deterministic mode (gs_set_deterministic)

def test_deterministic_mode_is_bit_reproducible_and_matches_the_oracle(gs):
    """gs_set_deterministic(ctx, 1): lists sorted before they are summed, per-pair moment slots added in tile order
    instead of binary32 atomics (SPEC.md "Determinism").  (1) Gradients of the L2 loss and of a given
    dL/dC keep the oracle's bar (DESIGN.md §3 #16), on lists beyond one chunk (team tiles, streamed lists) and on a
    frame without a tensor map; repeated calls return the same BITS.  (2) Two 300-iteration fits of configs[1] end
    in bit-identical parameters and moments, within 0.05 dB of the oracle's fit -- also with an active mask
    (selective refit) and with the quantisers in the loop.  (3) Call pattern and context history do not matter."""
    # (1) gradients
    W, H, N = 333, 95, 1500
    g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=6.0, opacity_range=(0.05, 0.3), config_index=93, margin=6.0)
    g.mu[:200] = np.array([72.0, 40.0]) + np.random.default_rng(7).uniform(-6, 6, (200, 2))
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 94))
    po = oracle.Params.from_f32(g)
    img_o = oracle.render(W, H, po)
    _, Go = oracle.loss(img_o, frame)
    gref = oracle.backward(W, H, po, Go)
    fd = torch.as_tensor(frame).cuda()
    ctx = gs.Context(W, H, N, max_pairs=400_000)
    gs.gs_set_deterministic(ctx, True)
    p = gs.Params.from_numpy(g)
    gs.gs_render(ctx, p)                                          # files the tiles under their classes
    ms = []
    for _ in range(3):                                            # (first launch: every tile by one warp; then teams)
        st = gs.AdamState.zeros(N)
        gs.gs_fit_steps(ctx, fd, p, st, 1, t0=1, lr=0.0)
        assert gs.gs_status(ctx) == 0
        _assert_grads(_np(st.m) / (1.0 - np.float32(0.9)), gref)
        ms.append(st.m.clone())
    assert torch.equal(ms[1], ms[2])
    Gt = torch.as_tensor(Go.astype(np.float32)).cuda()
    g1 = gs.gs_render_backward(ctx, p, Gt).flat9().clone()
    g2 = gs.gs_render_backward(ctx, p, Gt).flat9().clone()
    _assert_grads(_np(g1), gref)
    assert torch.equal(g1, g2)
    ctx.close()

    # (2) fits of configs[1]: plain, with an active mask, with quantisers
    W, H, N = 480, 272, 4096
    frame, mask = wl.talking_head_frame(wl.SPEC_ROI)
    mu, chol, rgb, op, _ = oracle.init_roi(frame, mask, N, 11, 1.0, 4.0)
    g = wl.GaussianSet(mu, chol, rgb, op)
    fd = torch.as_tensor(frame).cuda()
    rep_o = oracle.fit(W, H, oracle.Params.from_f32(g), frame, 300, lr=1e-2)
    act = torch.as_tensor((np.random.default_rng(5).uniform(size=N) < 0.4).astype(np.uint8)).cuda()
    for variant in ("plain", "masked", "qat"):
        ends = []
        for _ in range(2):
            ctx = gs.Context(W, H, N)
            gs.gs_set_deterministic(ctx, True)
            if variant == "qat":
                gs.gs_set_quantization(ctx, wl.uniform_quant_spec(W, H))
            p, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
            if variant == "masked":
                gs.gs_fit_steps(ctx, fd, p, st, 300, t0=1, lr=1e-2, active=act)
            else:
                rep = gs.gs_encode_iframe(ctx, fd, p, st, 300, lr=1e-2)
                assert rep.status == 0
                if variant == "plain":
                    assert abs(rep.psnr - rep_o.psnr) < 0.05, (rep.psnr, rep_o.psnr)
            assert gs.gs_status(ctx) == 0
            ends.append((p.flat9().clone(), st.m.clone(), st.v.clone()))
            ctx.close()
        for a, b in zip(ends[0], ends[1]):
            assert torch.equal(a, b), variant

    # (3) the bits do not depend on how the iterations are called or on what the context did before: resumed single
    # steps, non-resumed single steps (a standalone binning per call) and one call, on ONE context, one after the other
    # (the sort stage files every tile under the class of its current length: team or single warp follows the list)
    ctx = gs.Context(W, H, N)
    gs.gs_set_deterministic(ctx, True)
    runs = []
    for mode in ("one_call", "resume", "plain"):
        p, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
        if mode == "one_call":
            gs.gs_fit_steps(ctx, fd, p, st, 12, t0=1, lr=1e-2)
        else:
            for t in range(1, 13):
                gs.gs_fit_steps(ctx, fd, p, st, 1, t0=t, lr=1e-2, resume=(mode == "resume"))
        assert gs.gs_status(ctx) == 0
        runs.append(p.flat9().clone())
    assert torch.equal(runs[0], runs[1]) and torch.equal(runs[0], runs[2])
    ctx.close()


# ------------------------------------------------------------------ round-2 options at configs[2]'s size

def test_full_size_roi_loss_and_deterministic_mode(gs):
    """1920x1080, 50,000 Gaussians.  (1) gs_set_roi with the head + torso mask (22 % of the frame): loss and PSNR over
    the ROI against the oracle's c-16 on the initial set, and after 8 fit iterations on both sides (PSNR within
    0.05 dB, loss within 2 %).  (2) gs_set_deterministic: two 60-iteration fits end in identical bits, within 0.05 dB
    of a fit with the atomics."""
    W, H, N = 1920, 1080, 50_000
    frame, mask = wl.talking_head_frame(wl.SPEC_1080P, 0)
    mu, chol, rgb, op, _ = oracle.init_roi(frame, mask, N, 1, 1.0, 8.0)
    g = wl.GaussianSet(mu, chol, rgb, op)
    fd, md = torch.as_tensor(frame).cuda(), torch.as_tensor(mask).cuda()
    ctx = gs.Context(W, H, N, max_pairs=1_000_000)
    # (1)
    gs.gs_set_roi(ctx, md)
    p = gs.Params.from_numpy(g)
    po = oracle.Params.from_f32(g)
    img_o = oracle.render(W, H, po)
    L, _ = oracle.loss_roi(img_o, frame, mask)
    loss, psnr = gs.gs_loss_psnr(ctx, fd, p)
    assert abs(loss - L) <= 1e-5 * L and abs(psnr - oracle.psnr_roi(img_o, frame, mask)) < 1e-3
    rep = gs.gs_encode_iframe(ctx, fd, p, gs.AdamState.zeros(N), 8, lr=1e-2)
    rep_o = oracle.fit(W, H, po, frame, 8, lr=1e-2, roi=mask)
    assert rep.status == 0 and abs(rep.psnr - rep_o.psnr) < 0.05, (rep.psnr, rep_o.psnr)
    assert abs(rep.final_loss - rep_o.final_loss) < 2e-2 * rep_o.final_loss
    gs.gs_set_roi(ctx, None)
    # (2)
    ends = []
    for det in (True, True, False):
        gs.gs_set_deterministic(ctx, det)
        q, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
        r = gs.gs_encode_iframe(ctx, fd, q, st, 60, lr=1e-2)
        assert r.status == 0
        ends.append((q.flat9().clone(), st.m.clone(), r.psnr))
    assert torch.equal(ends[0][0], ends[1][0]) and torch.equal(ends[0][1], ends[1][1])
    assert abs(ends[0][2] - ends[2][2]) < 0.05
    ctx.close()
