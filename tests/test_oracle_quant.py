"""Pins of the oracle's quantisers and QAT loop (c-14)."""
import numpy as np

import oracle
import workloads as wl


def _spec_one(col, lo, hi, bits):
    levels = np.zeros(9, np.int32)
    lo_a, step, inv = np.zeros(9, np.float32), np.ones(9, np.float32), np.ones(9, np.float32)
    levels[col] = (1 << bits) - 1
    lo_a[col] = lo
    step[col] = np.float32((hi - lo) / levels[col])
    inv[col] = np.float32(levels[col] / (hi - lo))
    return levels, lo_a, step, inv


def _params(col, values):
    flat = np.zeros((len(values), 9))
    flat[:, 2] = flat[:, 4] = 1.0
    flat[:, col] = values
    return oracle.Params(flat[:, 0:2].copy(), flat[:, 2:5].copy(), flat[:, 5:8].copy(), flat[:, 8].copy())


def test_spec_hand_example_and_round_trip():
    """Cholesky channel with range [0,4] at 6 bits: step 4/63; x = 1.0 -> index 16 ->
    16 * 4/63 = 1.01587; grid points survive; the error is at most half a step; out-of-range clamps."""
    spec = _spec_one(2, 0.0, 4.0, 6)
    x = np.array([1.0, 16 * 4 / 63, 0.0, 4.0, 2.03, -3.0, 9.0])
    q = oracle.fake_quantize(_params(2, x), spec).chol[:, 0]
    assert abs(q[0] - 16 * 4 / 63) < 1e-6 and abs(q[0] - 1.01587) < 1e-5
    assert abs(q[1] - x[1]) < 1e-6 and q[2] == 0.0 and abs(q[3] - 4.0) < 1e-6
    assert abs(q[4] - 2.03) <= 0.5 * 4 / 63 + 1e-6
    assert q[5] == 0.0 and abs(q[6] - 4.0) < 1e-6                      # clamped
    # other columns untouched
    p = _params(2, x)
    p.rgb[:] = 0.1234567
    assert np.array_equal(oracle.fake_quantize(p, spec).rgb.astype(np.float32), p.rgb.astype(np.float32))
    # idempotent
    pq = oracle.fake_quantize(_params(2, x), spec)
    assert np.array_equal(oracle.fake_quantize(pq, spec).flat9(), pq.flat9())


def test_round_half_to_even():
    """round-to-nearest-even.  Range [0, 255] at 8 bits has step exactly 1."""
    spec = _spec_one(5, 0.0, 255.0, 8)
    q = oracle.fake_quantize(_params(5, np.array([0.5, 1.5, 2.5, 3.5, 2.4999, 2.5001])), spec).rgb[:, 0]
    assert np.array_equal(q, [0.0, 2.0, 2.0, 4.0, 2.0, 3.0])


def test_default_spec_and_qat_loop():
    W = H = 64
    spec = wl.uniform_quant_spec(W, H)
    assert list(spec[0]) == [65535, 65535, 63, 63, 63, 255, 255, 255, 0]
    frame, _ = wl.talking_head_frame(wl.SPEC_TINY)
    g = wl.tiny_gaussians()
    p = oracle.Params.from_f32(g)
    pq = oracle.fake_quantize(p, spec)
    d = np.abs(pq.flat9() - p.flat9())
    assert np.all(d[:, :2] <= 0.5 * 64 / 65535 + 1e-6) and np.all(d[:, 5:8] <= 0.5 / 255 + 1e-7)
    assert np.array_equal(pq.opacity, p.opacity)
    # "loss evaluated at dequantized parameters equals loss of a manually quantized copy"
    man = p.flat9().astype(np.float32).copy()
    for j in range(8):
        idx = np.clip(np.rint((man[:, j].astype(np.float64) - spec[1][j]) * float(spec[3][j])), 0, spec[0][j])
        man[:, j] = spec[1][j] + idx * float(spec[2][j])
    manual = oracle.Params(man[:, 0:2].astype(np.float64), man[:, 2:5].astype(np.float64),
                           man[:, 5:8].astype(np.float64), man[:, 8].astype(np.float64))
    La = oracle.loss(oracle.render(W, H, pq), frame)[0]
    Lb = oracle.loss(oracle.render(W, H, manual), frame)[0]
    assert abs(La - Lb) <= 1e-5 * La                                  # (the manual copy is computed in float64)
    # the loop: the quantised set improves, and ends near the unquantised fit (8/6/16 bits are fine here)
    r0 = oracle.loss(oracle.render(W, H, pq), frame)[0]
    pa, pb = oracle.Params.from_f32(g), oracle.Params.from_f32(g)
    ra = oracle.fit_qat(W, H, pa, frame, 60, spec, lr=1e-2)
    rb = oracle.fit(W, H, pb, frame, 60, lr=1e-2)
    assert ra.final_loss < 0.5 * r0 and abs(ra.psnr - rb.psnr) < 1.0
    # straight-through: the raw parameters moved although single steps are far below a Cholesky step
    assert np.abs(pa.chol - g.chol).max() > 0.05


def test_fit_qat_single_step_is_straight_through_by_finite_differences():
    """Pin of oracle.fit_qat ("parameters pass through simulated quantize-dequantize with
    straight-through gradients before rendering") by what the mathematics fixes, not by its own
    building blocks.  With zero moments the first Adam step is  theta <- theta - lr sign(g)  (|g| >> eps), so one
    QAT iteration must move every RAW parameter by exactly one lr against the sign of dL/dtheta taken AT THE
    QUANTISED point -- obtained here by central differences of the rendered loss, not from oracle.backward.  The
    quantisers are coarse (3-bit Cholesky, 4-bit colour, 6-bit mean) so that the two plausible mistakes fail:
    differentiating at the raw point flips some signs, and stepping the quantised copy lands off the raw lattice
    p0 - lr sign(g).  The report must describe fake_quantize(result), not the raw result."""
    W = H = 16
    r = np.random.default_rng(3)
    n = 5
    mu = r.uniform(3, 13, (n, 2))
    chol = np.stack([r.uniform(1.5, 4.0, n), r.uniform(-1.0, 1.0, n), r.uniform(1.5, 4.0, n)], axis=1)
    g = wl.GaussianSet(mu.astype(np.float32), chol.astype(np.float32), r.uniform(0.2, 0.9, (n, 3)).astype(np.float32),
                       np.ones(n, dtype=np.float32))
    frame = r.uniform(0, 1, (H, W, 3)).astype(np.float32)
    spec = wl.uniform_quant_spec(W, H, mu_bits=6, chol_bits=3, rgb_bits=4)
    lr = 1e-3

    def loss_at(flat):
        q = oracle.Params(flat[:, 0:2].copy(), flat[:, 2:5].copy(), flat[:, 5:8].copy(), flat[:, 8].copy())
        return oracle.loss(oracle.render(W, H, q), frame)[0]

    def fd_grad(flat, h=1e-5):
        out = np.zeros_like(flat)
        for i in range(flat.shape[0]):
            for j in range(9):
                a, b = flat.copy(), flat.copy()
                a[i, j] += h
                b[i, j] -= h
                out[i, j] = (loss_at(a) - loss_at(b)) / (2 * h)
        return out

    p0 = oracle.Params.from_f32(g)
    raw0 = p0.flat9().copy()
    q0 = oracle.fake_quantize(p0, spec).flat9()
    assert np.abs(q0 - raw0)[:, 2:5].max() > 0.1                       # the quantised point is somewhere else
    g_q, g_raw = fd_grad(q0), fd_grad(raw0)
    sure = (np.abs(g_q) > 1e-5) & (np.abs(g_raw) > 1e-5)               # (Adam's eps is 1e-8)
    assert sure.sum() >= 35 and (np.sign(g_q) != np.sign(g_raw))[sure].sum() >= 2   # the pin can tell the two apart

    p = oracle.Params.from_f32(g)
    rep = oracle.fit_qat(W, H, p, frame, 1, spec, lr=lr)
    step = p.flat9() - raw0
    assert np.allclose(step[sure], (-lr * np.sign(g_q))[sure], rtol=1e-3, atol=1e-9)   # raw + straight-through
    assert not np.allclose(step[sure], (-lr * np.sign(g_raw))[sure], rtol=1e-3, atol=1e-9)
    assert not np.allclose((p.flat9() - q0)[sure], (-lr * np.sign(g_q))[sure], rtol=1e-3, atol=1e-9)
    # report at the quantised result
    L_q = loss_at(oracle.fake_quantize(p, spec).flat9())
    assert abs(rep.final_loss - L_q) <= 1e-12 * L_q and abs(L_q - loss_at(p.flat9())) > 1e-6 * L_q
