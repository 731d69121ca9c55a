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
