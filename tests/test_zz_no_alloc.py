"""gs_decode_static: the decode render for callers that cannot allocate device memory.

Some hosts of a decoder own every byte of the GPU themselves (a player or server that reserved the device for its own
pools), cannot take the device-wide stall of a cudaMalloc / cudaFree inside a real-time loop, or run under a rule that
forbids allocation once start-up is over.  They cannot use gs_create, which cudaMallocs a context.  For them
include/gs2d.h offers ONE call that needs no context: its scratch is a fixed array inside the library (at most 16 384
Gaussians, 4 096 tiles, 256 Gaussians per tile), shared by all calls on a GPU and never cleared between them.

What is checked here, against the existing context path (gs_decode) on the same inputs and to the pixel tolerance the
render tests use (1e-4 absolute):
  - two calls in a row on different scenes and frame sizes -- the second must not see what the first left in the
    shared scratch -- and the first scene again, which must give the same bits as before;
  - jobs beyond a limit are refused with GS_ERR_CAPACITY and leave the output untouched, and the call after a refused
    one works.
This file is named to be collected last: it must pass alone in a fresh process and after every other test.
"""
import ctypes as C

import numpy as np
import pytest

import workloads as wl

torch = pytest.importorskip("torch")

TOL = 1e-4  # pixels, absolute: the bar of tests/test_gpu_parity.py::test_bins_bit_exact_and_pixels
GS_ERR_INVALID_ARGUMENT, GS_ERR_CAPACITY = -1, -4
MAX_GAUSSIANS, MAX_TILES, TILE_CAP = 16384, 4096, 256


def test_limits_are_checked_before_any_device_work():
    """Sizes beyond the static scratch and malformed arguments are refused on the host: this needs no GPU."""
    import paper_2505_09324_b200 as gs
    f = gs.lib().gs_decode_static
    ok = 256  # any non-null, aligned address: these calls return before touching it
    p = lambda n: gs._Params(ok, ok, ok, ok, n)  # noqa: E731
    assert f(p(MAX_GAUSSIANS + 1), 64, 64, 3.0, ok, None) == GS_ERR_CAPACITY
    assert f(p(16), 16 * 65, 16 * 64, 3.0, ok, None) == GS_ERR_CAPACITY  # 65 x 64 tiles > 4096
    assert f(p(0), 64, 64, 3.0, ok, None) == GS_ERR_INVALID_ARGUMENT
    assert f(p(16), 0, 64, 3.0, ok, None) == GS_ERR_INVALID_ARGUMENT
    assert f(p(16), 64, 64, 0.0, ok, None) == GS_ERR_INVALID_ARGUMENT
    assert f(p(16), 64, 64, float("nan"), ok, None) == GS_ERR_INVALID_ARGUMENT
    assert f(p(16), 64, 64, 3.0, None, None) == GS_ERR_INVALID_ARGUMENT
    assert f(gs._Params(ok + 4, ok, ok, ok, 16), 64, 64, 3.0, ok, None) == GS_ERR_INVALID_ARGUMENT  # mu: 8 bytes
    with open(gs._build.INCLUDE + "/gs2d.h") as h:  # the header states the same limits
        text = h.read()
    for name, v in (("GS_STATIC_MAX_GAUSSIANS", MAX_GAUSSIANS), ("GS_STATIC_MAX_TILES", MAX_TILES),
                    ("GS_STATIC_TILE_CAP", TILE_CAP)):
        assert f"#define {name} {v}" in text


@pytest.fixture(scope="module")
def gs():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2505_09324_b200 as gs
    gs.lib()  # fail loudly if the extension is missing
    return gs


def _existing_path(gs, W, H, g):
    """The context path: gs_create (cudaMalloc) + gs_decode."""
    ctx = gs.Context(W, H, g.n, max_pairs=64 * g.n)
    img = gs.gs_decode(ctx, gs.Params.from_numpy(g)).cpu().numpy()
    assert gs.gs_status(ctx) == 0
    ctx.close()
    return img


def _static_path(gs, W, H, g):
    out = torch.full((H, W, 3), -7.0, dtype=torch.float32, device="cuda")  # the caller's buffer
    gs.gs_decode_static(gs.Params.from_numpy(g), W, H, out)
    return out.cpu().numpy()


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_context_path(gs):
    # several tiles, ragged right and bottom edges, Gaussians hanging over the frame; the second scene is larger in
    # both tile count and Gaussian count than the first, the third call returns to the first
    a = wl.random_gaussians(1200, 333, 95, config_index=91, s_min=1.0, s_max=8.0, margin=20.0)
    b = wl.random_gaussians(4096, 480, 272, config_index=92, s_min=1.0, s_max=4.0, margin=20.0)
    ref_a, ref_b = _existing_path(gs, 333, 95, a), _existing_path(gs, 480, 272, b)
    got_a = _static_path(gs, 333, 95, a)
    got_b = _static_path(gs, 480, 272, b)
    got_a2 = _static_path(gs, 333, 95, a)
    for got, ref in ((got_a, ref_a), (got_b, ref_b), (got_a2, ref_a)):
        assert got.min() >= 0.0 and got.max() <= 1.0  # every pixel written (the buffer held -7), clamped
        assert np.abs(got - ref).max() < TOL
    assert ref_a.max() > 0.5 and ref_b.max() > 0.5  # the scenes are not blank
    assert np.array_equal(got_a, got_a2)  # lists are summed in id order: nothing of call 2 leaks into call 3


@pytest.mark.gpu
def test_over_full_tile_is_refused_and_the_next_call_works(gs):
    W = H = 64
    n = TILE_CAP + 44  # all in one tile: more than a bucket of the static scratch holds
    g = wl.random_gaussians(n, W, H, config_index=93, s_min=0.5, s_max=0.6, margin=0.0)
    g.mu[:] = 8.0 + 0.01 * np.arange(n, dtype=np.float32)[:, None] / n  # tile (0, 0), footprints inside it
    out = torch.full((H, W, 3), -7.0, dtype=torch.float32, device="cuda")
    rc = gs.gs_decode_static(gs.Params.from_numpy(g), W, H, out, allow=(GS_ERR_CAPACITY,))
    assert rc == GS_ERR_CAPACITY
    assert bool((out == -7.0).all())  # refused, not truncated: nothing written
    # the flag and the counters of the refused call are still in the scratch; the next call clears them itself
    ok = wl.random_gaussians(256, W, H, config_index=94, s_min=1.0, s_max=4.0)
    assert np.abs(_static_path(gs, W, H, ok) - _existing_path(gs, W, H, ok)).max() < TOL
    # exactly a full bucket is still fine
    g2 = wl.random_gaussians(TILE_CAP, W, H, config_index=95, s_min=0.5, s_max=0.6, margin=0.0)
    g2.mu[:] = 8.0
    assert np.abs(_static_path(gs, W, H, g2) - _existing_path(gs, W, H, g2)).max() < TOL
