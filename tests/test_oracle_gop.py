"""The oracle's GoP loop (oracle.gop_frame_types / oracle.encode_gop, SURVEY.md §8(f)
next #4) against what the texts fix and against invariants of the loop: the frame-type sequences the
reference texts print (tests/golden/worked_values.txt), P-frames leave the unselected Gaussians of
their predecessor untouched, an I-frame owes nothing to the frames before it, K = 1 is a sequence of
independent I-frame fits."""
import os

import numpy as np
import pytest

import oracle
import workloads as wl


def _golden(golden_dir):
    out = []
    with open(os.path.join(golden_dir, "worked_values.txt")) as f:
        for line in f:
            if line.startswith("gop_types"):
                _, inp, exp, cite = [s.strip() for s in line.split("|")]
                kv = dict(tok.split("=") for tok in inp.split())
                out.append((int(kv["frames"]), int(kv["K"]), exp, cite))
    return out


def test_frame_types_printed_by_the_texts(golden_dir):
    rows = _golden(golden_dir)
    assert len(rows) >= 3
    for frames, K, exp, cite in rows:
        assert "".join(oracle.gop_frame_types(frames, K)) == exp, cite


@pytest.mark.parametrize("K", [1, 2, 4, 8])
def test_frame_type_rule_counts(K):
    """for every K the stream's frame types follow the K rule: every GoP opens with its only
    I-frame, so F frames hold ceil(F / K) of them and no two I-frames are closer than K."""
    for F in (0, 1, 7, 16, 17):
        ty = oracle.gop_frame_types(F, K)
        idx = [i for i, t in enumerate(ty) if t == "I"]
        assert len(ty) == F and len(idx) == (F + K - 1) // K
        assert all(b - a == K for a, b in zip(idx, idx[1:])) and (not idx or idx[0] == 0)
    with pytest.raises(ValueError):
        oracle.gop_frame_types(4, 0)


def _frames(n):
    fm = [wl.talking_head_frame(wl.SPEC_TINY, k) for k in range(n)]
    return [f for f, _ in fm], [m for _, m in fm]


def test_gop_loop_invariants():
    W = H = 64
    N = 192
    frames, masks = _frames(5)
    tau = 0.3
    out = oracle.encode_gop(W, H, frames, masks, 3, N, seed=5, s_min=1.0, s_max=4.0, iframe_iters=12, pframe_iters=6,
                            tau=tau)
    assert [t for t, *_ in out] == ["I", "P", "P", "I", "P"]
    for f in (1, 2, 4):  # P-frames: what was not selected is the predecessor's, bit for bit
        _, p, act, rep = out[f]
        prev = out[f - 1][1]
        frozen = act == 0
        assert 0 < int(act.sum()) < N and rep.n_active == int(act.sum()) and rep.iters_run == 6
        for a, b in ((p.mu, prev.mu), (p.chol, prev.chol), (p.rgb, prev.rgb), (p.opacity, prev.opacity)):
            assert np.array_equal(a[frozen], b[frozen]) and not np.array_equal(a[~frozen], b[~frozen])
    # an I-frame owes nothing to its predecessors: frame 3 alone gives the same set
    alone = oracle.encode_gop(W, H, frames[3:4], masks[3:4], 3, N, seed=5 + 3, s_min=1.0, s_max=4.0, iframe_iters=12,
                              pframe_iters=6, tau=tau)
    assert np.array_equal(alone[0][1].mu, out[3][1].mu) and np.array_equal(alone[0][1].rgb, out[3][1].rgb)
    assert out[3][3].iters_run == 12 and out[3][2].all()


def test_gop_length_one_is_independent_iframe_fits():
    W = H = 64
    N = 128
    frames, masks = _frames(2)
    out = oracle.encode_gop(W, H, frames, masks, 1, N, seed=9, s_min=1.0, s_max=4.0, iframe_iters=8)
    for f in range(2):
        mu, chol, rgb, op, _ = oracle.init_roi(frames[f], masks[f], N, 9 + f, 1.0, 4.0)
        p = oracle.Params(mu.astype(np.float64), chol.astype(np.float64), rgb.astype(np.float64), op.astype(np.float64))
        rep = oracle.fit(W, H, p, frames[f], 8, lr=1e-2)
        assert out[f][0] == "I" and np.array_equal(out[f][1].chol, p.chol) and out[f][3].psnr == rep.psnr


def test_gop_pixel_rule_and_schedule_compose():
    """The pixel-granular selection and the I-frame schedule in the loop: same calls, same results as made by hand."""
    W = H = 64
    N = 128
    frames, masks = _frames(2)
    out = oracle.encode_gop(W, H, frames, masks, 2, N, seed=2, s_min=1.0, s_max=4.0, iframe_iters=10, pframe_iters=5,
                            decay=0.5, tau=0.08, pixel_select=True, influence_eps=0.01, dilate=True)
    mu, chol, rgb, op, _ = oracle.init_roi(frames[0], masks[0], N, 2, 1.0, 4.0)
    p = oracle.Params(mu.astype(np.float64), chol.astype(np.float64), rgb.astype(np.float64), op.astype(np.float64))
    oracle.fit_sched(W, H, p, frames[0], 10, lr=1e-2, decay=0.5)
    assert np.array_equal(out[0][1].mu, p.mu)
    _, _, act, na = oracle.pframe_select_pixels(W, H, p, frames[1], 0.08, eps=0.01, dilate=True)
    assert np.array_equal(out[1][2], act) and out[1][3].n_active == na
    oracle.fit(W, H, p, frames[1], 5, lr=1e-2, active=act)
    assert np.array_equal(out[1][1].mu, p.mu)
