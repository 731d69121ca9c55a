"""Pins for the oracle's primitive math and binning rule.

Everything here checks ``oracle/`` against something other than itself: values
the reference texts print (tests/golden/worked_values.txt), numpy.linalg, and an
independently formulated brute force.
"""
import math
import os

import numpy as np
import pytest

import oracle
import workloads as wl


def _golden(golden_dir):
    rec = {}
    with open(os.path.join(golden_dir, "worked_values.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, inp, exp, cite = [s.strip() for s in line.split("|")]
            rec.setdefault(name, []).append((inp, exp, cite))
    return rec


def _l_of(inp):
    for tok in inp.split():
        if tok.startswith("l="):
            return [float(x) for x in tok[2:].split(",")]
    raise KeyError(inp)


def test_cov_and_inverse_worked_values(golden_dir):
    g = _golden(golden_dir)
    for inp, exp, cite in g["cov_from_chol"]:
        S = oracle.cov_from_chol(_l_of(inp)).ravel()
        assert np.allclose(S, [float(x) for x in exp.split(",")], atol=1e-15), cite
    for inp, exp, cite in g["inverse_cov"]:
        A = oracle.inverse_cov(_l_of(inp)).ravel()
        assert np.allclose(A, [float(x) for x in exp.split(",")], atol=1e-15), cite
    for inp, exp, cite in g["inverse_cov_x36"]:
        A = 36.0 * oracle.inverse_cov(_l_of(inp)).ravel()
        assert np.allclose(A, [float(x) for x in exp.split(",")], atol=1e-13), cite


def test_inverse_cov_against_numpy_linalg():
    r = np.random.default_rng(1)
    for _ in range(1000):  # SPEC.md:82-84 random set
        l = np.array([r.uniform(0.1, 10), r.uniform(-10, 10), r.uniform(0.1, 10)])
        L = np.array([[l[0], 0.0], [l[1], l[2]]])
        S = oracle.cov_from_chol(l)
        assert np.allclose(S, L @ L.T, rtol=1e-14)
        assert np.linalg.det(S) > 0 and np.trace(S) > 0
        A = oracle.inverse_cov(l)
        assert np.allclose(A @ S, np.eye(2), atol=1e-9)
        assert np.allclose(A, np.linalg.inv(S), rtol=1e-9, atol=1e-12)


def test_sigma_is_half_mahalanobis():
    """The whitened evaluation of sigma equals 1/2 d^T Sigma^-1 d with numpy's inverse."""
    r = np.random.default_rng(2)
    for _ in range(500):
        l = np.array([r.uniform(0.3, 8), r.uniform(-6, 6), r.uniform(0.3, 8)])
        d = r.uniform(-20, 20, 2)
        L = np.array([[l[0], 0.0], [l[1], l[2]]])
        ref = 0.5 * d @ np.linalg.inv(L @ L.T) @ d
        assert math.isclose(oracle.sigma(d[0], d[1], l), ref, rel_tol=1e-10, abs_tol=1e-14)
    # a sign flip of l2 or a transposed L would fail this one
    assert math.isclose(oracle.sigma(1.0, 0.0, [1.0, 2.0, 1.0]), 0.5 * (1 + 4), rel_tol=1e-14)
    assert math.isclose(oracle.sigma(0.0, 1.0, [1.0, 2.0, 1.0]), 0.5, rel_tol=1e-14)


def test_footprint_worked_values(golden_dir):
    g = _golden(golden_dir)
    (inp, exp, cite), = g["footprint_half"]
    hw = oracle.footprint_halfwidths(_l_of(inp), 3.0)
    assert list(hw) == [float(x) for x in exp.split(",")], cite
    # mu=(10,10), l=(1,0,1), cutoff 3 -> [7,13]^2 -> tile (0,0) only
    hw = oracle.footprint_halfwidths([1, 0, 1], 3.0)
    assert (10 - hw[0], 10 + hw[0], 10 - hw[1], 10 + hw[1]) == (7, 13, 7, 13)
    p = oracle.Params(np.array([[10.0, 10.0]]), np.array([[1.0, 0.0, 1.0]]), np.ones((1, 3)), np.ones(1))
    rect, rng, lst = oracle.bin(64, 64, p)
    assert rect.tolist() == [[0, 0, 0, 0]] and lst.tolist() == [0] and rng.tolist() == [0] + [1] * 16
    # footprint off-frame -> empty
    p.mu[0] = [-10.0, 10.0]
    rect, rng, lst = oracle.bin(64, 64, p)
    assert len(lst) == 0 and rng[-1] == 0
    # straddling a tile corner: mu=(16,16), radius 3 -> tiles (0..1, 0..1)
    p.mu[0] = [16.0, 16.0]
    rect, rng, lst = oracle.bin(64, 64, p)
    assert rect.tolist() == [[0, 0, 1, 1]] and len(lst) == 4


def _brute_bins(W, H, mu, chol, k=3.0):
    """Independent formulation: tile (tx,ty) lists n iff
    lo_x < 16(tx+1) and hi_x >= 16 tx (same in y), evaluated in float32."""
    f = np.float32
    TX, TY = (W + 15) // 16, (H + 15) // 16
    lists = [[] for _ in range(TX * TY)]
    for n in range(len(mu)):
        mx, my = f(mu[n, 0]), f(mu[n, 1])
        l1, l2, l3 = f(chol[n, 0]), f(chol[n, 1]), f(chol[n, 2])
        if not all(np.isfinite([mx, my, l1, l2, l3])) or l1 == 0 or l3 == 0:
            continue
        rx = f(k) * abs(l1)
        ry = f(k) * np.sqrt(f(f(l2 * l2) + f(l3 * l3)), dtype=np.float32)
        lox, hix, loy, hiy = f(mx - rx), f(mx + rx), f(my - ry), f(my + ry)
        for ty in range(TY):
            for tx in range(TX):
                if lox < 16 * (tx + 1) and hix >= 16 * tx and loy < 16 * (ty + 1) and hiy >= 16 * ty \
                        and hix >= 0 and lox < W and hiy >= 0 and loy < H:
                    lists[ty * TX + tx].append(n)
    return lists


@pytest.mark.parametrize("W,H,N,seed", [(64, 64, 256, 0), (100, 52, 300, 1), (33, 17, 64, 2)])
def test_bins_against_brute_force(W, H, N, seed):
    g = wl.random_gaussians(N, W, H, s_min=0.5, s_max=12.0, config_index=50 + seed, margin=30.0)
    # edge cases: exact tile boundaries, degenerate and non-finite inputs
    g.mu[0] = [16.0, 16.0]
    g.chol[0] = [1.0, 0.0, 1.0]
    g.mu[1] = [3.0, 3.0]
    g.chol[1] = [1.0, 0.0, 1.0]          # lo = 0 exactly, hi = 6
    g.mu[2] = [-3.0, 5.0]
    g.chol[2] = [1.0, 0.0, 1.0]          # hi_x = 0 exactly -> listed
    g.mu[3] = [W + 3.0, 5.0]
    g.chol[3] = [1.0, 0.0, 1.0]          # lo_x = W exactly -> culled
    g.chol[4] = [0.0, 0.0, 1.0]          # l1 = 0 -> culled
    g.mu[5] = [np.nan, 1.0]
    g.chol[6] = [np.inf, 0.0, 1.0]
    g.mu[7] = [8.0, 8.0]
    g.chol[7] = [-2.0, 1.0, -3.0]        # negative diagonal is a valid factor of a PSD Sigma
    p = oracle.Params.from_f32(g)
    rect, rng, lst = oracle.bin(W, H, p)
    lists = _brute_bins(W, H, g.mu, g.chol)
    T = len(lists)
    assert rng[0] == 0 and rng[T] == len(lst) == sum(len(x) for x in lists)
    for t in range(T):
        assert lst[rng[t]:rng[t + 1]].tolist() == lists[t], f"tile {t}"
    assert rect[3, 2] < rect[3, 0] and rect[4, 2] < rect[4, 0] and rect[5, 2] < rect[5, 0] and rect[6, 2] < rect[6, 0]
    assert 2 in lst and 7 in lst


def test_bins_cover_every_pixel_inside_the_cutoff_ellipse():
    """Coverage completeness: every pixel with sigma <= k^2/2 lies in
    a tile that lists the Gaussian.  float64 brute force over all pixels."""
    W, H, N = 96, 80, 120
    g = wl.random_gaussians(N, W, H, s_min=0.7, s_max=9.0, config_index=60, margin=10.0)
    p = oracle.Params.from_f32(g)
    rect, rng, lst = oracle.bin(W, H, p)
    TX = (W + 15) // 16
    ys, xs = np.meshgrid(np.arange(H) + 0.5, np.arange(W) + 0.5, indexing="ij")
    for n in range(N):
        l1, l2, l3 = p.chol[n]
        u = (xs - p.mu[n, 0]) / l1
        v = ((ys - p.mu[n, 1]) - l2 * u) / l3
        inside = 0.5 * (u * u + v * v) <= 4.5 * (1 - 1e-6)
        tiles = set((int(y) // 16) * TX + int(x) // 16 for y, x in zip(ys[inside], xs[inside]))
        for t in tiles:
            assert n in lst[rng[t]:rng[t + 1]]


def test_partial_tiles_1080p_shape():
    """1080 = 67.5 tiles: the last tile row exists and is listed."""
    W, H = 1920, 1080
    p = oracle.Params(np.array([[5.0, 1079.0]]), np.array([[2.0, 0.0, 2.0]]), np.ones((1, 3)), np.ones(1))
    rect, rng, lst = oracle.bin(W, H, p)
    assert len(rng) == 120 * 68 + 1
    assert rect.tolist() == [[0, 67, 0, 67]]
