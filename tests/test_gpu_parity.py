"""GPU parity: libgs2d (through its C-ABI binding) against the float64 oracle on the
same seeded inputs.  Tolerances are BASELINE.json's north_star: tile bins and index
lists bit-exact, pixels within 1e-4 absolute, gradients within 1e-3 relative
(reading DESIGN.md §3 #16: |g - g*| <= 1e-3 |g*| + 1e-4 max|g*| per parameter
group), PSNR after a fixed iteration count within 0.05 dB."""
import os

import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def gs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2505_09324_b200 as gs
    gs.lib()  # fail loudly if the extension is missing
    return gs


def _np(t):
    return t.detach().cpu().numpy()


def _scene(W, H, N, seed, **kw):
    return wl.random_gaussians(N, W, H, config_index=50 + seed, **kw)


def _assert_bins(gs, ctx, W, H, g):
    rect, rng_o, lst_o = oracle.bin(W, H, oracle.Params.from_f32(g))
    rng_g, lst_g = gs.gs_get_bins(ctx)
    assert np.array_equal(_np(rng_g), rng_o)
    assert np.array_equal(_np(lst_g), lst_o)
    return len(lst_o)


GROUPS = {"mu": slice(0, 2), "chol": slice(2, 5), "rgb": slice(5, 8), "opacity": slice(8, 9)}


def _assert_grads(g_gpu, g_ref, rel=1e-3, floor=1e-4):
    for name, sl in GROUPS.items():
        a, b = g_gpu[:, sl], g_ref[:, sl]
        scale = np.abs(b).max()
        tol = rel * np.abs(b) + floor * scale + 1e-30
        bad = np.abs(a - b) > tol
        assert not bad.any(), (name, int(bad.sum()), float(np.abs(a - b).max()), float(scale))


# --------------------------------------------------------------------------- bins + pixels

@pytest.mark.parametrize("W,H,N,seed,smax", [(64, 64, 256, 0, 4.0), (200, 120, 1500, 1, 8.0), (333, 95, 3000, 2, 16.0),
                                              (480, 272, 4096, 3, 4.0)])
def test_bins_bit_exact_and_pixels(gs, W, H, N, seed, smax):
    g = _scene(W, H, N, seed, s_min=1.0, s_max=smax, margin=20.0)
    ctx = gs.Context(W, H, N, max_pairs=64 * N)
    p = gs.Params.from_numpy(g)
    img = _np(gs.gs_render(ctx, p, clamp=False))
    P = _assert_bins(gs, ctx, W, H, g)
    assert P > N  # several tiles per Gaussian on average
    ref = oracle.render(W, H, oracle.Params.from_f32(g))
    assert np.abs(img - ref).max() < 1e-4
    dec = _np(gs.gs_decode(ctx, p))
    assert np.abs(dec - np.clip(ref, 0, 1)).max() < 1e-4
    assert dec.min() >= 0.0 and dec.max() <= 1.0
    ctx.close()


def test_render_is_deterministic(gs):
    W, H, N = 200, 120, 2000
    g = _scene(W, H, N, 7, s_max=8.0)
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    a = gs.gs_render(ctx, p).clone()
    for _ in range(3):
        assert torch.equal(a, gs.gs_render(ctx, p))  # sorted lists + fixed-order sums: bit-identical
    ctx.close()


def test_culled_and_degenerate_gaussians(gs):
    """Off-frame, non-finite and singular Gaussians are skipped by both sides; a Gaussian
    covering every tile and a tile list longer than the shared-memory sort limit work."""
    W, H = 160, 96
    g = _scene(W, H, 4000, 9, s_min=1.0, s_max=3.0)
    g.mu[:2600] = np.array([40.0, 40.0]) + np.random.default_rng(0).uniform(-3, 3, (2600, 2))  # one crowded tile
    g.mu[2600] = [-500.0, 10.0]          # off-frame
    g.mu[2601] = [np.nan, 10.0]          # non-finite
    g.chol[2602] = [0.0, 0.0, 1.0]       # singular
    g.chol[2603] = [1.0, 0.0, 0.0]
    g.chol[2604] = [np.inf, 0.0, 1.0]
    g.chol[2605] = [400.0, 30.0, 300.0]  # covers the whole frame
    g.chol[2606] = [-2.0, 0.5, -3.0]     # negative diagonal: Sigma = L L^T is still SPD
    g.opacity[:] = 0.01
    ctx = gs.Context(W, H, g.n, max_pairs=200 * g.n)
    p = gs.Params.from_numpy(g)
    img = _np(gs.gs_render(ctx, p))
    _, rng_o, lst_o = oracle.bin(W, H, oracle.Params.from_f32(g))
    assert (np.diff(rng_o) > 2048).any()  # exercises the long-segment sort
    _assert_bins(gs, ctx, W, H, g)
    for bad in (2600, 2601, 2602, 2603, 2604):
        assert bad not in set(lst_o.tolist())
    go = g.copy()
    go.mu[2601] = [-500.0, 10.0]  # the oracle's render loops only over listed ids; keep its inputs finite
    go.chol[2604] = [1.0, 0.0, 1.0]
    go.mu[2604] = [-500.0, 10.0]
    ref = oracle.render(W, H, oracle.Params.from_f32(go))
    assert np.isfinite(img).all()
    assert np.abs(img - ref).max() < 1e-4
    ctx.close()


def test_capacity_error_is_latched(gs):
    W, H, N = 128, 128, 500
    g = _scene(W, H, N, 11, s_min=4.0, s_max=8.0)
    ctx = gs.Context(W, H, N, max_pairs=600)  # far too small
    p = gs.Params.from_numpy(g)
    out = torch.full((H, W, 3), -7.0, device="cuda")
    gs.gs_render(ctx, p, out=out)
    assert gs.gs_status(ctx) == -4          # GS_ERR_CAPACITY
    assert gs.gs_status(ctx) == 0           # cleared
    assert (out == -7.0).all()              # outputs untouched
    with pytest.raises(gs.GsError):
        gs.gs_get_bins(ctx)
    ctx.close()
    with pytest.raises(gs.GsError):
        gs.Context(W, H, 0)
    with pytest.raises(gs.GsError):
        c2 = gs.Context(W, H, 10)
        gs.gs_render(c2, gs.Params.from_numpy(_scene(W, H, 11, 1)))  # n > max_gaussians


# --------------------------------------------------------------------------- gradients

@pytest.mark.parametrize("W,H,N,seed", [(64, 64, 256, 0), (200, 120, 1500, 1), (333, 95, 2000, 2)])
def test_backward_parity(gs, W, H, N, seed):
    g = _scene(W, H, N, seed, s_min=1.0, s_max=8.0, margin=10.0, opacity_range=(0.2, 1.0))
    G = wl.random_image_grad(W, H, 60 + seed)
    ctx = gs.Context(W, H, N, max_pairs=64 * N)
    p = gs.Params.from_numpy(g)
    gr = gs.gs_render_backward(ctx, p, torch.as_tensor(G).cuda())
    got = _np(gr.flat9())
    ref = oracle.backward(W, H, oracle.Params.from_f32(g), G.astype(np.float64))
    _assert_grads(got, ref)
    # Gaussians outside all tiles get exactly zero gradient (north_star invariant)
    rect, _, _ = oracle.bin(W, H, oracle.Params.from_f32(g))
    culled = rect[:, 2] < rect[:, 0]
    assert culled.any() and np.all(got[culled] == 0.0)
    # zero image gradient -> zero gradients
    z = gs.gs_render_backward(ctx, p, torch.zeros((H, W, 3), device="cuda"))
    assert float(z.flat9().abs().max()) == 0.0
    ctx.close()


def test_backward_of_l2_loss_matches_oracle(gs):
    """The loss path end to end: G from the oracle's own render differs from the GPU's by
    rounding only, so compare with G computed on each side's own image."""
    W, H, N = 96, 80, 400
    g = _scene(W, H, N, 5, s_min=1.5, s_max=6.0, opacity_range=(0.1, 0.5))
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 70))
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    img = gs.gs_render(ctx, p)
    Gg = (2.0 / (3 * W * H)) * (img - torch.as_tensor(frame).cuda())
    got = _np(gs.gs_render_backward(ctx, p, Gg.contiguous()).flat9())
    po = oracle.Params.from_f32(g)
    L, Go = oracle.loss(oracle.render(W, H, po), frame)
    ref = oracle.backward(W, H, po, Go)
    _assert_grads(got, ref)
    loss, psnr = gs.gs_loss_psnr(ctx, torch.as_tensor(frame).cuda(), p)
    assert abs(loss - L) <= 1e-5 * L
    assert abs(psnr - oracle.psnr(oracle.render(W, H, po), frame)) < 1e-3
    ctx.close()


# --------------------------------------------------------------------------- Adam

def test_adam_step_parity_mask_and_projection(gs):
    N = 3000
    r = np.random.default_rng(3)
    g = _scene(640, 480, N, 4)
    g.chol[:50, 0] = 0.1004  # will cross l_min
    g.chol[:50, 2] = 0.1004
    grad = (r.standard_normal((N, 9)) * 10.0 ** r.uniform(-7, 0, (N, 9))).astype(np.float32)
    grad[:50, 2] = 1.0
    grad[:50, 4] = 1.0
    m0 = (r.standard_normal((N, 9)) * 1e-3).astype(np.float32)
    v0 = (np.abs(r.standard_normal((N, 9))) * 1e-5).astype(np.float32)
    active = (r.uniform(size=N) < 0.6).astype(np.uint8)
    active[:50] = 1
    lr = [1e-2, 3e-3, 5e-3, 2e-3]
    ctx = gs.Context(640, 480, N)
    for t, act in ((1, None), (7, active)):
        p = gs.Params.from_numpy(g)
        st = gs.AdamState(torch.as_tensor(m0).cuda().clone(), torch.as_tensor(v0).cuda().clone())
        gp = gs.Params(*[torch.as_tensor(np.ascontiguousarray(grad[:, sl])).cuda() for sl in
                         (slice(0, 2), slice(2, 5), slice(5, 8))], torch.as_tensor(grad[:, 8].copy()).cuda())
        before = p.flat9().clone()
        gs.gs_adam_step(ctx, p, gp, st, lr, t, active=None if act is None else torch.as_tensor(act).cuda())
        po = oracle.Params.from_f32(g)
        mo, vo = m0.astype(np.float64), v0.astype(np.float64)
        # the C-ABI carries beta1, beta2, eps as binary32: give the oracle the same values
        oracle.adam(po, grad.astype(np.float64), mo, vo, lr, t, active=act, beta1=float(np.float32(0.9)),
                    beta2=float(np.float32(0.999)), eps=float(np.float32(1e-8)))
        got, ref = _np(p.flat9()), po.flat9()
        # the stored result is rounded to binary32 (|err| <= 0.6e-7 |theta|); the step itself to 1e-4
        step_o = ref - _np(before).astype(np.float64)
        tol = 1e-4 * np.abs(step_o) + 1.2e-7 * np.abs(ref) + 1e-12
        assert np.all(np.abs(got - ref) <= tol)
        # moments: a few binary32 roundings of the two terms that are added (they may cancel)
        g64 = np.abs(grad.astype(np.float64))
        assert np.all(np.abs(_np(st.m) - mo) <= 3e-7 * (0.9 * np.abs(m0) + 0.1 * g64) + 1e-37)
        assert np.all(np.abs(_np(st.v) - vo) <= 3e-7 * (0.999 * v0 + 0.001 * g64 * g64) + 1e-37)
        assert np.all(got[:50, 2] == np.float32(0.1)) and np.all(got[:50, 4] == np.float32(0.1))  # projection
        if act is not None:
            frozen = act == 0
            assert torch.equal(p.flat9()[torch.as_tensor(frozen).cuda()], before[torch.as_tensor(frozen).cuda()])
            assert np.array_equal(_np(st.m)[frozen], m0[frozen]) and np.array_equal(_np(st.v)[frozen], v0[frozen])
    ctx.close()


# --------------------------------------------------------------------------- fit loops

def test_iframe_fit_tiny_config_psnr_parity(gs):
    """configs[0]: 64x64, 256 Gaussians, lr 1e-2, 100 iterations; PSNR within 0.05 dB."""
    frame, _ = wl.talking_head_frame(wl.SPEC_TINY)
    g = wl.tiny_gaussians()
    po = oracle.Params.from_f32(g)
    rep_o = oracle.fit(64, 64, po, frame, 100, lr=1e-2)
    ctx = gs.Context(64, 64, g.n)
    p = gs.Params.from_numpy(g)
    st = gs.AdamState.zeros(g.n)
    rep = gs.gs_encode_iframe(ctx, torch.as_tensor(frame).cuda(), p, st, 100, lr=1e-2)
    assert rep.status == 0 and rep.iters_run == 100 and rep.first_nonfinite_iter == 0
    assert abs(rep.psnr - rep_o.psnr) < 0.05
    assert abs(rep.final_loss - rep_o.final_loss) < 2e-2 * rep_o.final_loss
    # the reported numbers describe the returned parameters
    img = oracle.render(64, 64, oracle.Params.from_f32(wl.GaussianSet(_np(p.mu), _np(p.chol), _np(p.rgb),
                                                                       _np(p.opacity))))
    assert abs(oracle.psnr(img, frame) - rep.psnr) < 1e-3
    ctx.close()


def test_fit_single_iteration_matches_oracle_step(gs):
    """One full iteration (bin, render, loss, backward, Adam) on identical inputs."""
    W, H, N = 120, 72, 600
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 71))
    g = _scene(W, H, N, 6, s_min=1.5, s_max=5.0, opacity_range=(0.3, 1.0))
    po = oracle.Params.from_f32(g)
    _, G0 = oracle.loss(oracle.render(W, H, po), frame)
    g0 = oracle.backward(W, H, po, G0)                       # the gradient the first step is taken along
    oracle.fit(W, H, po, frame, 1, lr=1e-2)
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    st = gs.AdamState.zeros(N)
    gs.gs_encode_iframe(ctx, torch.as_tensor(frame).cuda(), p, st, 1, lr=1e-2)
    got, ref = _np(p.flat9()), po.flat9()
    # The first Adam step is -lr g / (|g| + eps), eps = 1e-8.  A gradient error dg moves it by
    # lr eps |dg| / ((|g| + eps)(|g + dg| + eps)): with the gradient bar of DESIGN.md §3 #16 (1e-3 |g| + 1e-4 max|g|) that
    # is below 1e-6 wherever |g| >= 1e-5, so there the parameters agree to binary32 rounding; where |g| is
    # comparable with eps the step is ill-conditioned and only bounded by its size, 2 lr between the two sides.
    well = np.abs(g0) >= 1e-5
    assert well.mean() > 0.95
    assert np.all(np.abs(got - ref)[well] <= 1e-5 * np.maximum(1.0, np.abs(ref))[well])
    assert np.abs(got - ref).max() <= 2.0e-2 + 1e-5
    ctx.close()


def test_fit_fixed_point_and_nonfinite_flag(gs):
    W, H, N = 80, 64, 200
    g = _scene(W, H, N, 8, s_min=1.5, s_max=5.0)
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    target = gs.gs_render(ctx, p).clone()
    st = gs.AdamState.zeros(N)
    rep = gs.gs_encode_iframe(ctx, target, p, st, 5, lr=1e-6)
    assert rep.final_loss < 1e-10 and rep.status == 0
    # a non-finite target poisons the loss: flagged at iteration 1, parameters left as they were
    bad = target.clone()
    bad[3, 3, 0] = float("nan")
    q = gs.Params.from_numpy(g)
    before = q.flat9().clone()
    rep = gs.gs_encode_iframe(ctx, bad, q, st, 4, lr=1e-2)
    assert rep.status == -5 and rep.first_nonfinite_iter == 1 and rep.iters_run == 0
    assert torch.equal(q.flat9(), before)
    ctx.close()


def test_nonfinite_latch_is_cleared_and_stale_bins_are_dropped(gs):
    """After a non-finite loss has been latched by gs_fit_steps, reading it with gs_status re-arms the
    context: a following fit on fresh parameters moves them (the Adam kernel skips its step only while the
    latch is set).  And gs_adam_step, which rewrites the parameters in place, invalidates bins that a
    resumable gs_fit_steps left for the same arrays."""
    W, H, N = 96, 64, 300
    g = _scene(W, H, N, 21, s_min=1.5, s_max=5.0, opacity_range=(0.2, 0.8))
    frame = torch.as_tensor(wl.talking_head_frame(wl.scaled_spec(W, H, 22))[0]).cuda()
    ctx = gs.Context(W, H, N)
    bad = frame.clone()
    bad[5, 7, 1] = float("inf")
    p, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
    gs.gs_fit_steps(ctx, bad, p, st, 2, t0=1, lr=1e-2, resume=True)
    assert gs.gs_status(ctx) == -5                       # GS_ERR_NONFINITE, consumed by this call
    assert gs.gs_status(ctx) == 0
    q, st2 = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
    before = q.flat9().clone()
    gs.gs_fit_steps(ctx, frame, q, st2, 1, t0=5, lr=1e-2, resume=True)     # t0 != 1: only the consumed latch re-arms
    assert gs.gs_status(ctx) == 0
    assert not torch.equal(q.flat9(), before)
    # stale bins: the resumed step above left bins of q; gs_adam_step moves q; a resumed fit step must re-bin
    grad = gs.Params(torch.zeros_like(q.mu), torch.zeros_like(q.chol), torch.zeros_like(q.rgb),
                     torch.zeros_like(q.opacity))
    grad.mu += 1.0                                         # every centre moves by +lr / (1 + eps) in x and y
    st3 = gs.AdamState.zeros(N)
    gs.gs_adam_step(ctx, q, grad, st3, 4.0, 1)
    moved = wl.GaussianSet(_np(q.mu), _np(q.chol), _np(q.rgb), _np(q.opacity))
    img = _np(gs.gs_render(ctx, q))
    _assert_bins(gs, ctx, W, H, moved)
    assert np.abs(img - oracle.render(W, H, oracle.Params.from_f32(moved))).max() < 1e-4
    # a resumed step right after the in-place update consumes bins of the MOVED set: its gradients are the oracle's
    po = oracle.Params.from_f32(moved)
    _, Go = oracle.loss(oracle.render(W, H, po), _np(frame))
    gref = oracle.backward(W, H, po, Go)
    st4 = gs.AdamState.zeros(N)
    q2 = gs.Params.from_numpy(moved)
    gs.gs_fit_steps(ctx, frame, q2, st4, 1, t0=1, lr=1e-2, resume=True)    # leaves bins of q2 (updated)
    gs.gs_adam_step(ctx, q2, grad, gs.AdamState.zeros(N), 4.0, 1)           # ... which this call makes stale
    now = wl.GaussianSet(_np(q2.mu), _np(q2.chol), _np(q2.rgb), _np(q2.opacity))
    st5 = gs.AdamState.zeros(N)
    gs.gs_fit_steps(ctx, frame, q2, st5, 1, t0=1, lr=0.0, resume=True)
    pn = oracle.Params.from_f32(now)
    _, Gn = oracle.loss(oracle.render(W, H, pn), _np(frame))
    _assert_grads(_np(st5.m) / (1.0 - np.float32(0.9)), oracle.backward(W, H, pn, Gn))
    ctx.close()


def test_misaligned_parameter_views_are_rejected(gs):
    """The kernels move parameter arrays as float4 slabs: a contiguous but misaligned view (chol[1:]) is an
    invalid argument, not a misaligned-address fault."""
    W, H, N = 64, 64, 130
    g = _scene(W, H, N + 1, 23, s_min=1.5, s_max=4.0)
    ctx = gs.Context(W, H, N + 1)
    full = gs.Params.from_numpy(g)
    view = gs.Params(full.mu[1:], full.chol[1:], full.rgb[1:], full.opacity[1:])   # 8 / 12 / 12 / 4 bytes in
    with pytest.raises(gs.GsError) as e:
        gs.gs_render(ctx, view)
    assert e.value.code == -1
    assert gs.gs_status(ctx) == 0
    img = gs.gs_render(ctx, full)                          # the context is unharmed
    assert torch.isfinite(img).all()
    ctx.close()


def test_fit_steps_resume_leaves_exact_bins(gs):
    """gs_fit_steps(resume=1): the fused Adam kernel bins the parameters it has just updated.  The
    bins it leaves must be the oracle's bins of those parameters, bit for bit; resumed single
    steps, a non-resumed call and one multi-iteration call follow the same trajectory; a caller
    who edits the parameters and does NOT resume gets bins of the edited parameters."""
    W, H, N = 200, 120, 1500
    frame = torch.as_tensor(wl.talking_head_frame(wl.scaled_spec(W, H, 5))[0]).cuda()
    g = _scene(W, H, N, 12, s_min=1.0, s_max=8.0, margin=10.0, opacity_range=(0.3, 1.0))
    ctx = gs.Context(W, H, N)
    runs = {}
    for mode in ("resume", "plain", "one_call"):
        p, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
        if mode == "one_call":
            gs.gs_fit_steps(ctx, frame, p, st, 6, t0=1, lr=1e-2)
        else:
            for t in range(1, 7):
                gs.gs_fit_steps(ctx, frame, p, st, 1, t0=t, lr=1e-2, resume=(mode == "resume"))
        assert gs.gs_status(ctx) == 0
        runs[mode] = (p, _np(p.flat9()))
        if mode == "resume":  # bins left behind by the last fused Adam step == oracle bins of the result
            got = wl.GaussianSet(_np(p.mu), _np(p.chol), _np(p.rgb), _np(p.opacity))
            _assert_bins(gs, ctx, W, H, got)
    ref = runs["one_call"][1]
    for mode in ("resume", "plain"):
        # float atomics reorder the gradient sums; after 6 Adam steps of 1e-2 the paths stay together
        assert np.abs(runs[mode][1] - ref).max() < 2e-3, mode
    # edit the parameters behind the library's back, then a non-resumed step: it must bin the edit
    p, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
    gs.gs_fit_steps(ctx, frame, p, st, 1, t0=1, lr=1e-2, resume=True)
    p.mu += 5.0
    edited = wl.GaussianSet(_np(p.mu), _np(p.chol), _np(p.rgb), _np(p.opacity))
    img = _np(gs.gs_render(ctx, p))
    _assert_bins(gs, ctx, W, H, edited)
    assert np.abs(img - oracle.render(W, H, oracle.Params.from_f32(edited))).max() < 1e-4
    ctx.close()


def test_resumed_fit_rereads_frame_and_mask_rewritten_in_place(gs):
    """A streaming loop keeps ONE frame buffer and ONE mask buffer, overwrites both for the next frame and calls
    gs_fit_steps(active, resume=1) from t0 = 1 again.  The selective refit's derived target (frame minus the frozen
    Gaussians' render) and its active-only bins were made from the OLD contents; pointer identity must not make the
    library keep them (include/gs2d.h, gs_fit_opts.resume).  In deterministic mode fits are bit-reproducible whatever
    the call pattern, so the streaming loop must end in the same bits as a loop over separate buffers that never
    resumes -- also when a selection call sits between the two fits, and with an ROI set."""
    W, H, N = 200, 120, 1200
    fa = torch.as_tensor(wl.talking_head_frame(wl.scaled_spec(W, H, 5))[0]).cuda()
    fb = torch.as_tensor(wl.talking_head_frame(wl.scaled_spec(W, H, 6), 3)[0]).cuda()
    g = _scene(W, H, N, 14, s_min=1.0, s_max=8.0, margin=10.0, opacity_range=(0.3, 1.0))
    r = np.random.default_rng(5)
    ma = torch.as_tensor((r.uniform(size=N) < 0.4).astype(np.uint8)).cuda()
    mb = torch.as_tensor((r.uniform(size=N) < 0.4).astype(np.uint8)).cuda()
    roi = torch.zeros((H, W), dtype=torch.uint8, device="cuda")
    roi[20:100, 30:170] = 1
    assert float((fa - fb).abs().max()) > 0.05 and int((ma != mb).sum()) > N // 4
    for use_roi in (False, True):
        ends = {}
        for mode in ("separate", "in_place", "in_place_select_between"):
            ctx = gs.Context(W, H, N)
            gs.gs_set_deterministic(ctx, True)
            if use_roi:
                gs.gs_set_roi(ctx, roi)
            p, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
            if mode == "separate":
                gs.gs_fit_steps(ctx, fa, p, st, 5, t0=1, lr=1e-2, active=ma)
                st.m.zero_(), st.v.zero_()
                gs.gs_fit_steps(ctx, fb, p, st, 3, t0=1, lr=1e-2, active=mb)
                gs.gs_fit_steps(ctx, fb, p, st, 2, t0=4, lr=1e-2, active=mb)
            else:
                frame, mask = fa.clone(), ma.clone()
                gs.gs_fit_steps(ctx, frame, p, st, 5, t0=1, lr=1e-2, active=mask, resume=True)
                frame.copy_(fb), mask.copy_(mb)  # the next frame arrives in the same buffers
                st.m.zero_(), st.v.zero_()
                if mode == "in_place_select_between":
                    gs.gs_pframe_select(ctx, frame, p, 0.02)
                gs.gs_fit_steps(ctx, frame, p, st, 3, t0=1, lr=1e-2, active=mask, resume=True)
                gs.gs_fit_steps(ctx, frame, p, st, 2, t0=4, lr=1e-2, active=mask, resume=True)  # continues: may keep
            assert gs.gs_status(ctx) == 0
            ends[mode] = p.flat9().clone()
            ctx.close()
        moved = (ends["separate"] - gs.Params.from_numpy(g).flat9()).abs().amax(dim=1) > 0
        freed = (ma | mb) != 0
        # (Gaussians off the frame -- or, with an ROI, away from it -- have no gradient and rest)
        assert not bool((moved & ~freed).any()) and int(moved.sum()) > (0.4 if use_roi else 0.8) * int(freed.sum())
        for mode in ("in_place", "in_place_select_between"):
            assert torch.equal(ends[mode], ends["separate"]), (use_roi, mode)


def test_tile_beyond_its_bucket_renders_and_fits(gs):
    """One tile lists 3,000 Gaussians at 1080p with max_pairs = 1e6 (bucket: 512 ids per tile): the entries beyond
    the bucket go to the shared spill list, which every consumer walks for that tile.  Bins and index lists stay
    bit-exact, pixels within 1e-4 (relative to max(1, |C|): the crowded pixels sum 3,000 terms), gradients of the
    L2 loss per DESIGN.md §3 #16, decode and selections as the oracle's -- and a fit of 40 iterations tracks it."""
    W, H, N = 1920, 1080, 3600
    g = _scene(W, H, N, 13, s_min=1.0, s_max=3.0, opacity_range=(0.001, 0.004))
    r = np.random.default_rng(1)
    g.mu[:3000] = np.array([1000.0, 504.0]) + r.uniform(-3, 3, (3000, 2))   # tile (62, 31) and its neighbours
    frame, _ = wl.talking_head_frame(wl.SPEC_1080P, 0)
    fd = torch.as_tensor(frame).cuda()
    po = oracle.Params.from_f32(g)
    ctx = gs.Context(W, H, N, max_pairs=1_000_000)
    p = gs.Params.from_numpy(g)
    img = _np(gs.gs_render(ctx, p))
    assert gs.gs_status(ctx) == 0
    P = _assert_bins(gs, ctx, W, H, g)
    _, rng_o, _ = oracle.bin(W, H, po)
    assert np.diff(rng_o).max() >= 3000 and P < 100_000
    ref = oracle.render(W, H, po)
    assert np.all(np.abs(img - ref) <= 1e-4 * np.maximum(1.0, np.abs(ref)))
    # (2,488 spilled entries: beyond 766 per tile the batches follow the spill list's arrival order, so this tile
    # is reproducible to rounding only; every other tile bit for bit)
    again = _np(gs.gs_render(ctx, p))
    assert np.all(np.abs(again - img) <= 2e-5 * np.maximum(1.0, np.abs(img)))
    far = np.ones((H, W), bool)
    far[31 * 16 - 16:32 * 16 + 16, 62 * 16 - 16:63 * 16 + 16] = False
    assert np.array_equal(again[far], img[far])
    # gradients of the L2 loss, on the context's first fit launch (one warp walks the whole list) and on the
    # second (the tile is filed as a team tile)
    _, Go = oracle.loss(ref, frame)
    gref = oracle.backward(W, H, po, Go)
    for launch in (0, 1):
        st = gs.AdamState.zeros(N)
        q = gs.Params.from_numpy(g)
        gs.gs_fit_steps(ctx, fd, q, st, 1, t0=1, lr=0.0)
        assert gs.gs_status(ctx) == 0, launch
        _assert_grads(_np(st.m) / (1.0 - np.float32(0.9)), gref)
    loss, psnr = gs.gs_loss_psnr(ctx, fd, p)
    L, _ = oracle.loss(ref, frame)
    assert abs(loss - L) <= 1e-5 * L
    # tile-residual selection sees the spilled entries too
    resid_o, flag_o, act_o, na_o = oracle.pframe_select(W, H, po, frame, 0.02)
    _, _, act_g, na_g = gs.gs_pframe_select(ctx, fd, p, 0.02)
    assert np.array_equal(_np(act_g), act_o) and na_g == na_o
    # a short fit follows the oracle's
    st = gs.AdamState.zeros(N)
    q = gs.Params.from_numpy(g)
    rep = gs.gs_encode_iframe(ctx, fd, q, st, 40, lr=1e-2)
    rep_o = oracle.fit(W, H, oracle.Params.from_f32(g), frame, 40, lr=1e-2)
    assert rep.status == 0 and abs(rep.psnr - rep_o.psnr) < 0.05, (rep.psnr, rep_o.psnr)
    ctx.close()


def test_spill_list_overflow_is_a_capacity_error(gs):
    """The spill list holds max(4096, max_pairs / 4) entries: beyond that a binning is a capacity error (outputs
    untouched), and the context recovers for the next call."""
    W, H = 256, 256
    N = 6000
    g = _scene(W, H, N, 13, s_min=1.0, s_max=1.5)
    g.mu[:] = np.array([100.0, 100.0]) + np.random.default_rng(1).uniform(-2, 2, (N, 2))   # one crowded tile
    ctx = gs.Context(W, H, N, max_pairs=16000)  # bucket 512 + spill 4096 < 6000 entries of one tile
    p = gs.Params.from_numpy(g)
    out = torch.full((H, W, 3), -7.0, device="cuda")
    gs.gs_render(ctx, p, out=out)
    assert gs.gs_status(ctx) == -4 and gs.gs_status(ctx) == 0
    assert (out == -7.0).all()
    g2 = _scene(W, H, N, 14, s_min=1.0, s_max=2.0)
    img = _np(gs.gs_render(ctx, gs.Params.from_numpy(g2)))
    assert gs.gs_status(ctx) == 0
    _assert_bins(gs, ctx, W, H, g2)
    assert np.abs(img - oracle.render(W, H, oracle.Params.from_f32(g2))).max() < 1e-4
    ctx.close()


# --------------------------------------------------------------------------- ROI init

def test_init_roi_parity(gs):
    spec = wl.scaled_spec(480, 272, 1)
    frame, mask = wl.talking_head_frame(wl.SPEC_ROI)
    W, H, N, seed = 480, 272, 4096, 1234
    mu_o, chol_o, rgb_o, op_o, pix = oracle.init_roi(frame, mask, N, seed, 1.0, 4.0)
    ctx = gs.Context(W, H, N)
    p = gs.gs_init_roi(ctx, torch.as_tensor(frame).cuda(), torch.as_tensor(mask).cuda(), N, seed, 1.0, 4.0)
    assert np.array_equal(_np(p.mu), mu_o)        # sampled pixel + jitter: bit-exact
    assert np.array_equal(_np(p.rgb), rgb_o)      # copied colours: bit-exact
    assert np.array_equal(_np(p.opacity), op_o)
    # scales and rotation go through binary32 exp/sin/cos here and float64 in the oracle
    assert np.allclose(_np(p.chol), chol_o, rtol=1e-5, atol=1e-5)
    # edge cases: empty ROI is an error, full ROI puts everything inside
    with pytest.raises(gs.GsError) as e:
        gs.gs_init_roi(ctx, torch.as_tensor(frame).cuda(), torch.zeros((H, W), dtype=torch.uint8, device="cuda"), N,
                       seed, 1.0, 4.0)
    assert e.value.code == -3
    full = np.ones((H, W), dtype=np.uint8)
    mu_f = oracle.init_roi(frame, full, 500, 7, 1.0, 4.0)[0]
    pf = gs.gs_init_roi(ctx, torch.as_tensor(frame).cuda(), torch.as_tensor(full).cuda(), 500, 7, 1.0, 4.0)
    assert np.array_equal(_np(pf.mu), mu_f)
    ctx.close()
    del spec


# --------------------------------------------------------------------------- P-frames

def test_pframe_select_parity_and_freeze(gs):
    W, H, N = 160, 112, 900
    spec = wl.scaled_spec(W, H, 72)
    f0, mask = wl.talking_head_frame(spec, 0)
    f1, _ = wl.talking_head_frame(spec, 6)
    ctx = gs.Context(W, H, N)
    p = gs.gs_init_roi(ctx, torch.as_tensor(f0).cuda(), torch.as_tensor(mask).cuda(), N, 5, 1.5, 5.0)
    st = gs.AdamState.zeros(N)
    gs.gs_encode_iframe(ctx, torch.as_tensor(f0).cuda(), p, st, 150, lr=1e-2)
    gset = wl.GaussianSet(_np(p.mu), _np(p.chol), _np(p.rgb), _np(p.opacity))
    po = oracle.Params.from_f32(gset)
    # configs[3]'s tau = 0.02 sits at the noise floor of this small, briefly fitted scene (every
    # tile exceeds it), so the fixture takes tau in the gap at the 80th percentile of the
    # oracle's tile residuals: about a fifth of the tiles, the moving head, are selected
    resid_o = oracle.pframe_select(W, H, po, f1, 0.02)[0]
    srt = np.sort(resid_o)
    k = int(0.8 * len(srt))
    tau = float(0.5 * (srt[k - 1] + srt[k]))
    resid_o, flag_o, act_o, na_o = oracle.pframe_select(W, H, po, f1, tau)
    resid, flag, act, na = gs.gs_pframe_select(ctx, torch.as_tensor(f1).cuda(), p, tau)
    assert np.abs(_np(resid) - resid_o).max() < 1e-5
    border = np.abs(resid_o - tau) < 1e-6          # DESIGN.md §3 #15: borderline tiles are exempt
    assert np.array_equal(_np(flag)[~border], flag_o[~border])
    if not border.any():
        assert np.array_equal(_np(act), act_o) and na == na_o
    assert 0 < na < N
    # identical frame and render -> empty selection, nothing changes
    same = gs.gs_decode(ctx, p).clone()
    before = p.flat9().clone()
    a2, rep2 = gs.gs_encode_pframe(ctx, same, p, st, tau, 20, lr=1e-2)
    assert rep2.n_active == 0 and rep2.iters_run == 0 and int(a2.sum()) == 0
    assert torch.equal(p.flat9(), before)
    # refit: unselected Gaussians bit-identical, PSNR improves, close to the oracle's
    psnr_before = gs.gs_loss_psnr(ctx, torch.as_tensor(f1).cuda(), p)[1]
    a3, rep3 = gs.gs_encode_pframe(ctx, torch.as_tensor(f1).cuda(), p, st, tau, 60, lr=1e-2)
    frozen = a3 == 0
    assert torch.equal(p.flat9()[frozen], before[frozen]) and rep3.n_active == int(a3.sum()) == na
    assert rep3.psnr > psnr_before
    act_ref, rep_o = oracle.encode_pframe(W, H, po, f1, tau, 60, lr=1e-2)
    assert abs(rep3.psnr - rep_o.psnr) < 0.05
    ctx.close()


# --------------------------------------------------------------------------- superpixel init

@pytest.mark.parametrize("W,H,N,m,iters,cfg", [(96, 64, 40, 10, 10, 90), (480, 272, 4096, 10, 10, 1),
                                                (333, 95, 300, 25, 3, 2), (1920, 1080, 50_000, 10, 10, 0)])
def test_init_superpixel_parity(gs, W, H, N, m, iters, cfg):
    """The paper's initialiser: SLIC-style superpixels on the ROI, one Gaussian per
    segment.  The segmentation is integer arithmetic: labels, segment count and order are bit-exact
    with the oracle; means / Cholesky factors / colours agree to binary32 rounding."""
    if (W, H) == (1920, 1080):
        frame, mask = wl.talking_head_frame(wl.SPEC_1080P, 0)
    elif (W, H) == (480, 272):
        frame, mask = wl.talking_head_frame(wl.SPEC_ROI)
    else:
        frame, mask = wl.talking_head_frame(wl.scaled_spec(W, H, cfg))
    mu_o, chol_o, rgb_o, op_o, lab_o, S = oracle.init_superpixel(frame, mask, N, compactness=m, iters=iters)
    ctx = gs.Context(W, H, N)
    p, lab = gs.gs_init_superpixel(ctx, torch.as_tensor(frame).cuda(), torch.as_tensor(mask).cuda(), N, m, iters)
    assert p.n == len(mu_o) <= N
    assert np.array_equal(_np(lab), lab_o)
    assert np.allclose(_np(p.mu), mu_o, rtol=0, atol=2e-4)
    assert np.allclose(_np(p.chol), chol_o, rtol=2e-6, atol=2e-6)
    assert np.allclose(_np(p.rgb), rgb_o, rtol=0, atol=1e-6)
    assert np.array_equal(_np(p.opacity), op_o)
    # edge cases: empty ROI is an error; a full-frame ROI works; one segment takes everything
    with pytest.raises(gs.GsError) as e:
        gs.gs_init_superpixel(ctx, torch.as_tensor(frame).cuda(), torch.zeros((H, W), dtype=torch.uint8, device="cuda"), N)
    assert e.value.code == -3
    if W <= 480:
        full = np.ones((H, W), np.uint8)
        nf = min(N, 64)
        ref = oracle.init_superpixel(frame, full, nf, compactness=m, iters=2)
        pf, lf = gs.gs_init_superpixel(ctx, torch.as_tensor(frame).cuda(), torch.as_tensor(full).cuda(), nf, m, 2)
        assert np.array_equal(_np(lf), ref[4]) and pf.n == len(ref[0])
        one, l1 = gs.gs_init_superpixel(ctx, torch.as_tensor(frame).cuda(), torch.as_tensor(mask).cuda(), 1, m, 1)
        assert one.n == 1 and int(l1.max()) == 0
    # the set it returns fits: a short fit from it reaches a higher PSNR than from the sampled init
    if (W, H) == (480, 272):
        fd = torch.as_tensor(frame).cuda()
        st = gs.AdamState.zeros(p.n)
        q = gs.Params(p.mu.contiguous(), p.chol.contiguous(), p.rgb.contiguous(), p.opacity.contiguous())
        target = fd * torch.as_tensor(mask).cuda()[..., None].float()
        ra = gs.gs_encode_iframe(ctx, target.contiguous(), q, st, 100, lr=1e-2)
        inside = torch.as_tensor(np.ones((H, W), np.uint8)).cuda()
        s2 = gs.gs_init_roi(ctx, fd, torch.as_tensor(mask).cuda() * inside, q.n, 5, 1.0, 4.0)
        rb = gs.gs_encode_iframe(ctx, target.contiguous(), s2, gs.AdamState.zeros(q.n), 100, lr=1e-2)
        assert ra.psnr > rb.psnr, (ra.psnr, rb.psnr)
    ctx.close()


# --------------------------------------------------------------------------- lr schedule + early stop

def test_iframe_fit_schedule_and_early_stop_parity(gs):
    """gs_encode_iframe_sched (c-12): two-step lr decay and early stop at a target PSNR, against
    the oracle's scheduled loop on configs[0]'s inputs."""
    frame, _ = wl.talking_head_frame(wl.SPEC_TINY)
    g = wl.tiny_gaussians()
    fd = torch.as_tensor(frame).cuda()
    ctx = gs.Context(64, 64, g.n)
    po = oracle.Params.from_f32(g)
    ro = oracle.fit_sched(64, 64, po, frame, 100, lr=1e-2)
    p, st = gs.Params.from_numpy(g), gs.AdamState.zeros(g.n)
    r = gs.gs_encode_iframe_sched(ctx, fd, p, st, 100, lr=1e-2)
    assert r.status == 0 and r.iters_run == 100 and abs(r.psnr - ro.psnr) < 0.05
    plain = gs.gs_encode_iframe(ctx, fd, gs.Params.from_numpy(g), gs.AdamState.zeros(g.n), 100, lr=1e-2)
    assert abs(plain.psnr - r.psnr) > 1e-3                      # the decay changed the trajectory
    # early stop: same stopping iteration as the oracle for a target well inside a check interval
    target = ro.psnr - 1.5
    po2 = oracle.Params.from_f32(g)
    ro2 = oracle.fit_sched(64, 64, po2, frame, 100, lr=1e-2, target_psnr=target, check_every=10)
    p2, st2 = gs.Params.from_numpy(g), gs.AdamState.zeros(g.n)
    r2 = gs.gs_encode_iframe_sched(ctx, fd, p2, st2, 100, lr=1e-2, target_psnr=target, check_every=10)
    assert 0 < ro2.iters_run < 100
    assert r2.iters_run == ro2.iters_run and r2.psnr >= target and abs(r2.psnr - ro2.psnr) < 0.05
    # the report describes the returned parameters
    loss, psnr = gs.gs_loss_psnr(ctx, fd, p2)
    assert abs(psnr - r2.psnr) < 1e-6
    ctx.close()


# --------------------------------------------------------------------------- pixel-granular P-frame selection

@pytest.mark.parametrize("W,H,N,dilate", [(160, 112, 900, False), (480, 272, 4096, True)])
def test_pframe_select_pixels_parity(gs, W, H, N, dilate):
    """c-13: per-pixel change map against the clamped render, then the Gaussians that
    influence a changed pixel.  The change map agrees with the oracle's except at pixels whose
    residual is within rounding of tau; from the SAME change map the selected set equals the oracle's
    (float64 exp(-sigma) >= eps) except for knife-edge Gaussians whose largest weight over the changed
    pixels is within 1e-4 relative of eps (the kernel decides in binary32), which must be rare."""
    spec = wl.scaled_spec(W, H, 73)
    f0, mask = wl.talking_head_frame(spec, 0)
    f1, _ = wl.talking_head_frame(spec, 5)
    ctx = gs.Context(W, H, N)
    fd0, fd1 = torch.as_tensor(f0).cuda(), torch.as_tensor(f1).cuda()
    p = gs.gs_init_roi(ctx, fd0, torch.as_tensor(mask).cuda(), N, 5, 1.5, 5.0)
    st = gs.AdamState.zeros(N)
    gs.gs_encode_iframe(ctx, fd0, p, st, 150, lr=1e-2)
    po = oracle.Params.from_f32(wl.GaussianSet(_np(p.mu), _np(p.chol), _np(p.rgb), _np(p.opacity)))
    tau = 0.12
    ch_o, resid_o, act_o, na_o = oracle.pframe_select_pixels(W, H, po, f1, tau, eps=0.01, dilate=False)
    ch_g, act_g, na_g = gs.gs_pframe_select_pixels(ctx, fd1, p, tau, 0.01, dilate=False)
    border = np.abs(resid_o - tau) < 1e-5
    assert np.array_equal(_np(ch_g)[~border], ch_o[~border]) and 0 < ch_o.sum() < 0.5 * W * H
    # same change map in -> same selection out, bit for bit (with and without the dilation)
    ch_g2, act_g2, na_g2 = gs.gs_pframe_select_pixels(ctx, fd1, p, tau, 0.01, dilate=dilate)
    _, _, act_ref, na_ref, wmax = oracle.pframe_select_pixels(W, H, po, f1, tau, eps=float(np.float32(0.01)),
                                                              changed=_np(ch_g2), want_wmax=True)
    clear = np.abs(wmax / float(np.float32(0.01)) - 1.0) > 1e-4
    assert np.array_equal(_np(act_g2)[clear], act_ref[clear]) and 0 < na_ref < N
    assert (~clear).sum() <= 3 and abs(na_g2 - na_ref) <= (~clear).sum()
    if dilate:
        assert int(ch_g2.sum()) > int(ch_g.sum())
    # a caller-provided change map is used as it is
    given = torch.zeros((H, W), dtype=torch.uint8, device="cuda")
    given[H // 2 - 2:H // 2 + 2, W // 2 - 2:W // 2 + 2] = 1
    _, act_g3, na_g3 = gs.gs_pframe_select_pixels(ctx, fd1, p, tau, 0.02, changed=given)
    _, _, act_r3, na_r3, wmax3 = oracle.pframe_select_pixels(W, H, po, f1, tau, eps=float(np.float32(0.02)),
                                                             changed=_np(given), want_wmax=True)
    clear3 = np.abs(wmax3 / float(np.float32(0.02)) - 1.0) > 1e-4
    assert np.array_equal(_np(act_g3)[clear3], act_r3[clear3]) and abs(na_g3 - na_r3) <= (~clear3).sum()
    # fewer Gaussians than the tile rule selects for the same threshold on the tile mean
    _, _, act_tile, na_tile = gs.gs_pframe_select(ctx, fd1, p, 0.02)
    # refit: frozen Gaussians bit-identical, PSNR improves
    before = p.flat9().clone()
    psnr0 = gs.gs_loss_psnr(ctx, fd1, p)[1]
    act, rep = gs.gs_encode_pframe_pixels(ctx, fd1, p, st, tau, 60, eps=0.01, dilate=dilate)
    assert rep.status == 0 and rep.n_active == int(act.sum()) == na_g2 and rep.iters_run == 60
    frozen = act == 0
    assert torch.equal(p.flat9()[frozen], before[frozen]) and rep.psnr > psnr0
    ctx.close()


# --------------------------------------------------------------------------- quantisation (PTQ / QAT)

def test_fake_quantize_and_qat_fit_parity(gs):
    """c-14: the quantisers are defined in binary32, so gs_fake_quantize is
    bit-exact with the oracle; a render with quantisation set on the context equals the render of
    the pre-quantised set; the QAT fit (render and gradients at the quantised parameters,
    straight-through to the raw ones) ends within 0.05 dB of the oracle's."""
    W = H = 64
    spec = wl.uniform_quant_spec(W, H)
    frame, _ = wl.talking_head_frame(wl.SPEC_TINY)
    g = wl.tiny_gaussians()
    r = np.random.default_rng(8)
    g.chol[:, 1] = r.uniform(-1.0, 1.0, g.n).astype(np.float32)
    g.mu[:5] = [[-3.0, 70.0]] * 5                                     # out of range: clamps
    fd = torch.as_tensor(frame).cuda()
    ctx = gs.Context(W, H, g.n)
    p = gs.Params.from_numpy(g)
    po = oracle.Params.from_f32(g)
    q = gs.gs_fake_quantize(ctx, p, spec)
    qo = oracle.fake_quantize(po, spec)
    assert np.array_equal(_np(q.flat9()), qo.flat9().astype(np.float32))
    img_q = gs.gs_render(ctx, q).clone()
    gs.gs_set_quantization(ctx, spec)
    assert torch.equal(gs.gs_render(ctx, p), img_q)
    _assert_bins(gs, ctx, W, H, wl.GaussianSet(_np(q.mu), _np(q.chol), _np(q.rgb), _np(q.opacity)))
    # gradients are taken at the quantised parameters
    G = wl.random_image_grad(W, H, 64)
    got = _np(gs.gs_render_backward(ctx, p, torch.as_tensor(G).cuda()).flat9())
    _assert_grads(got, oracle.backward(W, H, qo, G.astype(np.float64)))
    # QAT fit
    g2 = wl.tiny_gaussians()
    p2, st = gs.Params.from_numpy(g2), gs.AdamState.zeros(g2.n)
    rep = gs.gs_encode_iframe(ctx, fd, p2, st, 100, lr=1e-2)
    po2 = oracle.Params.from_f32(g2)
    rep_o = oracle.fit_qat(W, H, po2, frame, 100, spec, lr=1e-2)
    assert rep.status == 0 and abs(rep.psnr - rep_o.psnr) < 0.05, (rep.psnr, rep_o.psnr)
    # the report is the PSNR of the quantised set, which is what a decoder renders
    gs.gs_set_quantization(ctx, None)
    dec = gs.gs_decode(ctx, gs.gs_fake_quantize(ctx, p2, spec))
    mse = float(((dec - fd) ** 2).mean())
    assert abs(10 * np.log10(1.0 / mse) - rep.psnr) < 1e-3
    # and differs from the unquantised render of the raw parameters
    assert abs(gs.gs_loss_psnr(ctx, fd, p2)[1] - rep.psnr) > 1e-4
    ctx.close()


# --------------------------------------------------------------------------- edge cases

def test_edge_cases_tiny_frames_single_gaussian_and_empty_lists(gs):
    """Ragged and degenerate inputs through the whole path: a frame smaller than one tile, a
    one-row frame, a single Gaussian, a set that is culled entirely (every tile list empty)."""
    for W, H, N in ((8, 5, 3), (40, 1, 6), (17, 33, 1)):
        g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=3.0, opacity_range=(0.3, 0.9), config_index=97)
        frame = np.random.default_rng(W).uniform(0, 1, (H, W, 3)).astype(np.float32)
        ctx = gs.Context(W, H, max(N, 1))
        p = gs.Params.from_numpy(g)
        po = oracle.Params.from_f32(g)
        img = _np(gs.gs_render(ctx, p))
        _assert_bins(gs, ctx, W, H, g)
        assert np.abs(img - oracle.render(W, H, po)).max() < 1e-4
        L, Go = oracle.loss(oracle.render(W, H, po), frame)
        st = gs.AdamState.zeros(N)
        gs.gs_fit_steps(ctx, torch.as_tensor(frame).cuda(), p, st, 1, t0=1, lr=0.0)
        _assert_grads(_np(st.m) / (1.0 - np.float32(0.9)), oracle.backward(W, H, po, Go))
        rep = gs.gs_encode_iframe(ctx, torch.as_tensor(frame).cuda(), p, st, 30, lr=1e-2)
        rep_o = oracle.fit(W, H, po, frame, 30, lr=1e-2)
        assert rep.status == 0 and abs(rep.psnr - rep_o.psnr) < 0.05
        ctx.close()
    # everything culled: empty lists everywhere, zero image, zero gradients, parameters only projected
    W, H, N = 64, 48, 20
    g = wl.random_gaussians(N, W, H, s_min=1.0, s_max=2.0, config_index=98)
    g.mu[:] += 1000.0
    frame = np.full((H, W, 3), 0.25, np.float32)
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    assert float(gs.gs_render(ctx, p).abs().max()) == 0.0
    rng, lst = gs.gs_get_bins(ctx)
    assert lst.numel() == 0 and int(rng.max()) == 0
    st = gs.AdamState.zeros(N)
    before = p.flat9().clone()
    rep = gs.gs_encode_iframe(ctx, torch.as_tensor(frame).cuda(), p, st, 5, lr=1e-2)
    assert rep.status == 0 and torch.equal(p.flat9(), before) and abs(rep.final_loss - 0.0625) < 1e-6
    act, rep2 = gs.gs_encode_pframe(ctx, torch.as_tensor(frame).cuda(), p, st, 0.02, 5)
    assert rep2.n_active == 0 and rep2.iters_run == 0       # changed tiles list nobody
    ctx.close()


# --------------------------------------------------------------------------- host-buffer entry points

def test_host_buffer_entry_points(gs):
    """gs_decode_host / gs_encode_iframe_host (the end-to-end path bench.py times): the same results
    as the device-pointer calls, with pinned and with pageable host memory."""
    W, H, N = 96, 80, 400
    g = _scene(W, H, N, 21, s_min=1.5, s_max=6.0, opacity_range=(0.1, 0.5))
    frame, _ = wl.talking_head_frame(wl.scaled_spec(W, H, 74))
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    dec = gs.gs_decode(ctx, p).cpu()
    for pin in (True, False):
        f = (lambda a: torch.as_tensor(a).pin_memory()) if pin else (lambda a: torch.as_tensor(a).clone())
        ph = gs.Params(f(g.mu), f(g.chol), f(g.rgb), f(g.opacity))
        out = gs.gs_decode_host(ctx, ph, torch.empty((H, W, 3), dtype=torch.float32).pin_memory() if pin else
                                torch.empty((H, W, 3), dtype=torch.float32))
        assert torch.equal(out, dec)
        rep_h = gs.gs_encode_iframe_host(ctx, f(frame), ph, 40, lr=1e-2)
        q, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
        rep_d = gs.gs_encode_iframe(ctx, torch.as_tensor(frame).cuda(), q, st, 40, lr=1e-2)
        assert rep_h.status == 0 and rep_h.iters_run == 40
        assert abs(rep_h.psnr - rep_d.psnr) < 0.02          # float atomics reorder the gradient sums
        assert np.abs(_np(q.flat9()) - torch.cat([ph.mu, ph.chol, ph.rgb, ph.opacity[:, None]], 1).numpy()).max() < 5e-2
        po = oracle.Params.from_f32(g)
        assert abs(oracle.fit(W, H, po, frame, 40, lr=1e-2).psnr - rep_h.psnr) < 0.05
    # in deterministic mode the two entry points return the same bits
    gs.gs_set_deterministic(ctx, True)
    ph = gs.Params(*[torch.as_tensor(a).pin_memory() for a in (g.mu, g.chol, g.rgb, g.opacity)])
    rep_h = gs.gs_encode_iframe_host(ctx, torch.as_tensor(frame).pin_memory(), ph, 40, lr=1e-2)
    q, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
    rep_d = gs.gs_encode_iframe(ctx, torch.as_tensor(frame).cuda(), q, st, 40, lr=1e-2)
    assert rep_h.psnr == rep_d.psnr and rep_h.final_loss == rep_d.final_loss
    assert torch.equal(q.flat9().cpu(), torch.cat([ph.mu, ph.chol, ph.rgb, ph.opacity[:, None]], 1))
    ctx.close()


# --------------------------------------------------------------------------- call-order fuzz

def test_random_call_sequences_keep_the_context_consistent(gs):
    """The context carries state between calls (fresh / consumed / sorted bins, binning epochs, the
    triple-buffered launch order, lazily allocated scratch).  Random sequences of calls on one context:
    after every call the status is clean, renders match the oracle, and gs_get_bins returns the
    oracle's bins of the parameters that were binned last."""
    W, H, N = 112, 80, 500
    frame, mask = wl.talking_head_frame(wl.scaled_spec(W, H, 75))
    fd = torch.as_tensor(frame).cuda()
    r = np.random.default_rng(int(os.environ.get("GS2D_FUZZ_SEED", "99")))   # (another seed: another sequence)
    ctx = gs.Context(W, H, N)
    g = _scene(W, H, N, 22, s_min=1.2, s_max=6.0, margin=6.0, opacity_range=(0.1, 0.6))
    p, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
    t = 1
    spec = wl.uniform_quant_spec(W, H)

    def host(pp):
        return wl.GaussianSet(_np(pp.mu), _np(pp.chol), _np(pp.rgb), _np(pp.opacity))

    roi = mask.copy()
    roi_d = torch.as_tensor(roi).cuda()
    roi_on = False
    for step in range(60):
        op = int(r.integers(0, 11))
        if op == 8:                                        # round-2 switches, toggled in the middle of everything
            gs.gs_set_deterministic(ctx, bool(r.integers(0, 2)))
        elif op == 9:
            roi_on = not roi_on
            gs.gs_set_roi(ctx, roi_d if roi_on else None)
            loss, _ = gs.gs_loss_psnr(ctx, fd, p)
            img_o = oracle.render(W, H, oracle.Params.from_f32(host(p)))
            L = oracle.loss_roi(img_o, frame, roi)[0] if roi_on else oracle.loss(img_o, frame)[0]
            assert abs(loss - L) <= 1e-5 * L
        elif op == 10:                                     # a masked refit: frozen rows stay bit-identical
            act = torch.as_tensor((r.uniform(size=N) < 0.3).astype(np.uint8)).cuda()
            before = p.flat9().clone()
            gs.gs_fit_steps(ctx, fd, p, st, 2, t0=t, lr=1e-2, active=act, resume=bool(r.integers(0, 2)))
            t += 2
            frozen = act == 0
            assert torch.equal(p.flat9()[frozen], before[frozen])
        elif op == 0:
            img = _np(gs.gs_render(ctx, p))
            assert np.abs(img - oracle.render(W, H, oracle.Params.from_f32(host(p)))).max() < 1e-4
            _assert_bins(gs, ctx, W, H, host(p))
        elif op == 1:
            k = int(r.integers(1, 4))
            gs.gs_fit_steps(ctx, fd, p, st, k, t0=t, lr=1e-2, resume=bool(r.integers(0, 2)))
            t += k
        elif op == 2:
            gs.gs_fit_steps(ctx, fd, p, st, 1, t0=t, lr=1e-2, resume=True)
            t += 1
            _assert_bins(gs, ctx, W, H, host(p))           # bins left by the fused Adam kernel
        elif op == 3:
            G = wl.random_image_grad(W, H, 65)
            got = _np(gs.gs_render_backward(ctx, p, torch.as_tensor(G).cuda()).flat9())
            _assert_grads(got, oracle.backward(W, H, oracle.Params.from_f32(host(p)), G.astype(np.float64)))
        elif op == 4:
            resid, _, act, na = gs.gs_pframe_select(ctx, fd, p, 0.05)
            assert na == int(act.sum())
            resid_o = oracle.pframe_select(W, H, oracle.Params.from_f32(host(p)), frame, 0.05, roi=roi if roi_on else None)[0]
            assert np.abs(_np(resid) - resid_o).max() < 1e-5
            _assert_bins(gs, ctx, W, H, host(p))
        elif op == 5:
            p.mu += float(r.uniform(-0.5, 0.5))            # the caller edits the parameters behind the library's back
            loss, _ = gs.gs_loss_psnr(ctx, fd, p)
            img_o = oracle.render(W, H, oracle.Params.from_f32(host(p)))
            L = oracle.loss_roi(img_o, frame, roi)[0] if roi_on else oracle.loss(img_o, frame)[0]
            assert abs(loss - L) <= 1e-5 * L
        elif op == 6:
            ch, act, na = gs.gs_pframe_select_pixels(ctx, fd, p, 0.1)
            if roi_on:
                assert int(_np(ch)[roi == 0].sum()) == 0
            _, _, act_ref, _, wmx = oracle.pframe_select_pixels(W, H, oracle.Params.from_f32(host(p)), frame, 0.1,
                                                                eps=float(np.float32(0.01)), changed=_np(ch),
                                                                want_wmax=True)
            clear = np.abs(wmx / float(np.float32(0.01)) - 1.0) > 1e-4
            assert np.array_equal(_np(act)[clear], act_ref[clear])
        else:
            gs.gs_set_quantization(ctx, spec)
            q = gs.gs_fake_quantize(ctx, p, spec)
            assert torch.equal(gs.gs_render(ctx, p), gs.gs_render(ctx, q))
            gs.gs_set_quantization(ctx, None)
        assert gs.gs_status(ctx) == 0, (step, op)
    gs.gs_set_roi(ctx, None)
    ctx.close()


# --------------------------------------------------------------------------- GoP loop over a sequence

@pytest.mark.parametrize("pixel_select", [False, True])
def test_gop_loop_parity(gs, pixel_select):
    """gs_encode_gop against oracle.encode_gop on 5 frames of the tiny
    config with K = 3 ([I,P,P,I,P]): frame types, the I-frames' bit-exact initial positions carried through the
    snapshots' row count, per-frame PSNR within 0.05 dB, selection counts within 2 % (tile rule; 5 % for the pixel rule, where single
    pixels sit on the threshold and flip with the last bits of the fitted set), frozen Gaussians bit-identical to the predecessor's snapshot."""
    W = H = 64
    N = 192
    fm = [wl.talking_head_frame(wl.SPEC_TINY, k) for k in range(5)]
    frames, masks = [f for f, _ in fm], [m for _, m in fm]
    kw = dict(seed=5, s_min=1.0, s_max=4.0, iframe_iters=40, pframe_iters=15, lr=1e-2,
              tau=0.35 if pixel_select else 0.15, pixel_select=pixel_select, influence_eps=0.01, dilate=False)
    ref = oracle.encode_gop(W, H, frames, masks, 3, N, **kw)
    ctx = gs.Context(W, H, N)
    fd = [torch.as_tensor(f).cuda() for f in frames]
    md = [torch.as_tensor(m).cuda() for m in masks]
    kw_g = dict(kw)
    kw_g["eps_adam"] = 1e-8
    outs, active, reps = gs.gs_encode_gop(ctx, fd, md, 3, N, **kw_g)
    assert [("I", "P")[t] for t, _ in reps] == [t for t, *_ in ref] == ["I", "P", "P", "I", "P"]
    some_partial = False
    for f, (ty, p_o, act_o, rep_o) in enumerate(ref):
        rep_g = reps[f][1]
        assert outs[f].n == p_o.n == N and rep_g.status == 0
        assert abs(rep_g.psnr - rep_o.psnr) < 0.05, (f, rep_g.psnr, rep_o.psnr)
        act_g = _np(active[f])
        if ty == "I":
            assert act_g.all() and rep_g.iters_run == 40 and rep_g.n_active == N
        else:
            assert abs(int(act_g.sum()) - int(act_o.sum())) <= (0.05 if pixel_select else 0.02) * N, (f, act_g.sum(), act_o.sum())
            assert rep_g.n_active == int(act_g.sum())
            some_partial |= 0 < int(act_g.sum()) < N
            frozen = torch.as_tensor(act_g == 0).cuda()
            assert torch.equal(outs[f].flat9()[frozen], outs[f - 1].flat9()[frozen])
        # the snapshot decodes to the reported PSNR
        assert abs(gs.gs_loss_psnr(ctx, fd[f], outs[f])[1] - rep_g.psnr) < 1e-6
    assert some_partial
    # K = 1: every frame an I-frame; zero frames: nothing to do
    outs1, _, reps1 = gs.gs_encode_gop(ctx, fd[:2], md[:2], 1, N, seed=5, s_min=1.0, s_max=4.0, iframe_iters=5)
    assert [t for t, _ in reps1] == [0, 0]
    assert gs.gs_encode_gop(ctx, [], [], 3, N)[2] == []
    ctx.close()


def test_gop_loop_superpixel_init_and_schedule(gs):
    """The loop with the paper's own I-frame recipe: superpixel initialiser (the set may hold fewer than the
    segments asked for), decaying learning rate, early stop at a target PSNR."""
    W = H = 64
    fm = [wl.talking_head_frame(wl.SPEC_TINY, k) for k in range(3)]
    frames = [f for f, _ in fm]
    ones = [np.ones((H, W), dtype=np.uint8)] * 3
    kw = dict(init="superpixel", compactness=10, kmeans_iters=5, iframe_iters=60, pframe_iters=10, lr=1e-2, decay=0.5,
              target_psnr=20.0, check_every=10, tau=0.05)
    ref = oracle.encode_gop(W, H, frames, ones, 2, 150, **kw)
    ctx = gs.Context(W, H, 150)
    outs, active, reps = gs.gs_encode_gop(ctx, [torch.as_tensor(f).cuda() for f in frames],
                                          [torch.as_tensor(m).cuda() for m in ones], 2, 150, **kw)
    assert [t for t, _ in reps] == [0, 1, 0]
    for f, (ty, p_o, act_o, rep_o) in enumerate(ref):
        assert outs[f].n == p_o.n <= 150
        assert reps[f][1].iters_run == rep_o.iters_run and abs(reps[f][1].psnr - rep_o.psnr) < 0.05
        assert not _np(active[f])[p_o.n:].any()
        assert abs(int(_np(active[f]).sum()) - int(act_o.sum())) <= 0.03 * 150
    assert ref[0][3].iters_run < 60  # the early stop took effect
    ctx.close()


# --------------------------------------------------------------------------- ROI-restricted loss (c-16)

def test_roi_restricted_loss_fit_and_selections(gs):
    """gs_set_roi (DESIGN.md c-16): loss, PSNR, gradients, a fit and both
    P-frame selections over the ROI's pixels only, against the oracle's c-16 functions, on a frame whose last
    tile row is partial and an ROI with holes; an empty mask is refused; None restores the full frame."""
    W, H, N = 200, 120, 1500
    spec = wl.scaled_spec(W, H, 75)
    frame, mask = wl.talking_head_frame(spec, 0)
    f1, _ = wl.talking_head_frame(spec, 6)
    roi = mask.copy()
    roi[np.random.default_rng(4).uniform(size=(H, W)) < 0.05] = 0
    g = _scene(W, H, N, 14, s_min=1.0, s_max=6.0, margin=8.0, opacity_range=(0.05, 0.3))
    po = oracle.Params.from_f32(g)
    fd, rd = torch.as_tensor(frame).cuda(), torch.as_tensor(roi).cuda()
    ctx = gs.Context(W, H, N)
    p = gs.Params.from_numpy(g)
    full = gs.gs_loss_psnr(ctx, fd, p)
    with pytest.raises(gs.GsError):
        gs.gs_set_roi(ctx, torch.zeros((H, W), dtype=torch.uint8, device="cuda"))
    assert gs.gs_loss_psnr(ctx, fd, p) == full                      # a refused mask changes nothing
    gs.gs_set_roi(ctx, rd)
    img_o = oracle.render(W, H, po)
    L, Go = oracle.loss_roi(img_o, frame, roi)
    loss, psnr = gs.gs_loss_psnr(ctx, fd, p)
    assert abs(loss - L) <= 1e-5 * L and abs(psnr - oracle.psnr_roi(img_o, frame, roi)) < 1e-3
    # gradients of the ROI loss: one iteration with lr = 0 leaves m = (1 - beta1) grad
    gref = oracle.backward(W, H, po, Go)
    for _ in range(2):                                              # (first launch: warps; second: teams)
        st = gs.AdamState.zeros(N)
        gs.gs_fit_steps(ctx, fd, p, st, 1, t0=1, lr=0.0)
        assert gs.gs_status(ctx) == 0
        _assert_grads(_np(st.m) / (1.0 - np.float32(0.9)), gref)
    # the render and a given dL/dC are untouched by the ROI
    assert np.abs(_np(gs.gs_render(ctx, p)) - img_o).max() < 1e-4
    # a fit
    q, st = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
    rep = gs.gs_encode_iframe(ctx, fd, q, st, 60, lr=1e-2)
    rep_o = oracle.fit(W, H, oracle.Params.from_f32(g), frame, 60, lr=1e-2, roi=roi)
    assert rep.status == 0 and abs(rep.psnr - rep_o.psnr) < 0.05, (rep.psnr, rep_o.psnr)
    assert abs(rep.final_loss - rep_o.final_loss) < 2e-2 * rep_o.final_loss
    # ... also with a mask of active Gaussians (selective refit: the frozen ones live in the target)
    act = (np.random.default_rng(6).uniform(size=N) < 0.5).astype(np.uint8)
    q2, st2 = gs.Params.from_numpy(g), gs.AdamState.zeros(N)
    gs.gs_fit_steps(ctx, fd, q2, st2, 40, t0=1, lr=1e-2, active=torch.as_tensor(act).cuda())
    qo = oracle.Params.from_f32(g)
    oracle.fit(W, H, qo, frame, 40, lr=1e-2, roi=roi, active=act)
    assert abs(gs.gs_loss_psnr(ctx, fd, q2)[1] - oracle.psnr_roi(oracle.render(W, H, qo), frame, roi)) < 0.05
    # tile-residual selection over the ROI's pixels
    qo = oracle.Params.from_f32(wl.GaussianSet(_np(q.mu), _np(q.chol), _np(q.rgb), _np(q.opacity)))
    resid_o = oracle.pframe_select(W, H, qo, f1, 0.0, roi=roi)[0]
    srt = np.sort(resid_o[resid_o > 0])
    k = int(0.6 * len(srt))
    tau = float(0.5 * (srt[k - 1] + srt[k]))
    resid_o, flag_o, act_o, na_o = oracle.pframe_select(W, H, qo, f1, tau, roi=roi)
    f1d = torch.as_tensor(f1).cuda()
    resid, flag, act_g, na = gs.gs_pframe_select(ctx, f1d, q, tau)
    assert np.abs(_np(resid) - resid_o).max() < 1e-5 and (resid_o == 0).any()
    border = np.abs(resid_o - tau) < 1e-6
    assert np.array_equal(_np(flag)[~border], flag_o[~border])
    if not border.any():
        assert np.array_equal(_np(act_g), act_o) and na == na_o
    # pixel-granular selection: the change map never leaves the ROI
    ch_g, act_p, na_p = gs.gs_pframe_select_pixels(ctx, f1d, q, 0.12, 0.01, dilate=False)
    ch_o, act_po, _ = oracle.pframe_select_pixels_roi(W, H, qo, f1, 0.12, roi)
    resid_px = oracle.pframe_select_pixels(W, H, qo, f1, 0.12)[1]
    edge = np.abs(resid_px - 0.12) < 1e-5
    assert np.array_equal(_np(ch_g)[~edge], ch_o[~edge]) and int(_np(ch_g)[roi == 0].sum()) == 0 and ch_o.sum() > 0
    # a non-finite frame value: outside the ROI it is not part of the loss; inside it poisons the loss at the first
    # iteration, exactly as without an ROI (the oracle's c-16 loss is NaN there) -- with and without
    # a mask of active Gaussians
    yo, xo = map(int, np.argwhere(roi == 0)[0])
    yi, xi = map(int, np.argwhere(roi != 0)[len(np.argwhere(roi != 0)) // 2])
    for bad_value in (float("nan"), float("inf")):
        f_out, f_in = fd.clone(), fd.clone()
        f_out[yo, xo, 1] = bad_value
        f_in[yi, xi, 1] = bad_value
        q3 = gs.Params.from_numpy(g)
        rep = gs.gs_encode_iframe(ctx, f_out, q3, gs.AdamState.zeros(N), 5, lr=1e-2)
        assert rep.status == 0 and rep.iters_run == 5 and np.isfinite(rep.final_loss)
        q3 = gs.Params.from_numpy(g)
        before = q3.flat9().clone()
        rep = gs.gs_encode_iframe(ctx, f_in, q3, gs.AdamState.zeros(N), 5, lr=1e-2)
        assert rep.status == -5 and rep.first_nonfinite_iter == 1 and rep.iters_run == 0
        assert torch.equal(q3.flat9(), before)
        fn = f_in.cpu().numpy()
        qo3 = oracle.Params.from_f32(g)
        assert oracle.fit(W, H, qo3, fn, 5, lr=1e-2, roi=roi).first_nonfinite_iter == 1
        assert np.array_equal(qo3.flat9(), oracle.Params.from_f32(g).flat9())  # the oracle stops there too
        gs.gs_fit_steps(ctx, f_in, q3, gs.AdamState.zeros(N), 3, t0=1, lr=1e-2, active=torch.as_tensor(act).cuda())
        assert gs.gs_status(ctx) == -5 and torch.equal(q3.flat9(), before)
    # None: the whole frame again
    gs.gs_set_roi(ctx, None)
    assert gs.gs_loss_psnr(ctx, fd, p) == full
    ctx.close()
