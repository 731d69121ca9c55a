"""ORACLE -- test infrastructure only.

ctypes binding of ``oracle/gs_oracle.c``: a plain float64 CPU restatement of the
hot path of arXiv 2505.09324's 2D Gaussian Splatting codec (see the header of
the C file for the passage each function follows).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2505_09324_b200`` and the CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gs_oracle.c")
_LIB = os.path.join(_HERE, "_gs_oracle.so")

TILE = 16
CUTOFF = 3.0
L_MIN = 0.1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-ffp-contract=off keeps the binary32 binning
    rule single-rounded)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.gso_loss.restype = C.c_double
        _lib.gso_psnr.restype = C.c_double
        _lib.gso_sigma.restype = C.c_double
        _lib.gso_rnd64.restype = C.c_uint64
        _lib.gso_rnd64.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64]
        _lib.gso_get_threads.restype = C.c_int
    return _lib


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty)) if a is not None else None


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def set_threads(n: int) -> None:
    lib().gso_set_threads(C.c_int(int(n)))


def get_threads() -> int:
    return int(lib().gso_get_threads())


@dataclass
class Params:
    """float64 parameter set (the oracle's working precision)."""
    mu: np.ndarray
    chol: np.ndarray
    rgb: np.ndarray
    opacity: np.ndarray

    @staticmethod
    def from_f32(gs) -> "Params":
        return Params(_d(gs.mu).copy(), _d(gs.chol).copy(), _d(gs.rgb).copy(), _d(gs.opacity).copy())

    def copy(self) -> "Params":
        return Params(self.mu.copy(), self.chol.copy(), self.rgb.copy(), self.opacity.copy())

    @property
    def n(self) -> int:
        return int(self.mu.shape[0])

    def flat9(self) -> np.ndarray:
        return np.concatenate([self.mu, self.chol, self.rgb, self.opacity[:, None]], axis=1)


def cov_from_chol(l):
    S = np.zeros(4)
    lib().gso_cov_from_chol(_p(_d(l), C.c_double), _p(S, C.c_double))
    return S.reshape(2, 2)


def inverse_cov(l):
    abc = np.zeros(3)
    lib().gso_inverse_cov(_p(_d(l), C.c_double), _p(abc, C.c_double))
    return np.array([[abc[0], abc[1]], [abc[1], abc[2]]])


def sigma(dx, dy, l) -> float:
    return float(lib().gso_sigma(C.c_double(dx), C.c_double(dy), _p(_d(l), C.c_double)))


def footprint_halfwidths(l, cutoff=CUTOFF):
    out = np.zeros(2, dtype=np.float32)
    lib().gso_footprint_halfwidths(_p(_d(l), C.c_double), C.c_double(cutoff), _p(out, C.c_float))
    return out


def tiles_of(W, H):
    TX, TY = (W + TILE - 1) // TILE, (H + TILE - 1) // TILE
    return TX, TY, TX * TY


def bin(W, H, p: Params, cutoff=CUTOFF):
    """-> (rect4 [N,4] int32 {tx0,ty0,tx1,ty1}, range [T+1] int32, list [P] int32)."""
    _, _, T = tiles_of(W, H)
    N = p.n
    mu, chol = _d(p.mu), _d(p.chol)
    rect4 = np.zeros((max(N, 1), 4), dtype=np.int32)
    rng = np.zeros(T + 1, dtype=np.int32)
    P = C.c_longlong(0)
    lib().gso_bin(W, H, N, _p(mu, C.c_double), _p(chol, C.c_double), C.c_double(cutoff), _p(rect4, C.c_int),
                  _p(rng, C.c_int), None, C.c_longlong(0), C.byref(P))
    lst = np.zeros(max(P.value, 1), dtype=np.int32)
    rc = lib().gso_bin(W, H, N, _p(mu, C.c_double), _p(chol, C.c_double), C.c_double(cutoff), _p(rect4, C.c_int),
                       _p(rng, C.c_int), _p(lst, C.c_int), C.c_longlong(P.value), C.byref(P))
    assert rc == 0
    return rect4[:N], rng, lst[:P.value]


def render(W, H, p: Params, *, dense=False, cutoff=CUTOFF, tiles=None, out=None):
    """Unclamped image [H,W,3] float64.  ``tiles``: render only these tile ids."""
    img = out if out is not None else np.zeros((H, W, 3), dtype=np.float64)
    tl = None if tiles is None else np.ascontiguousarray(tiles, dtype=np.int32)
    lib().gso_render(W, H, p.n, _p(_d(p.mu), C.c_double), _p(_d(p.chol), C.c_double), _p(_d(p.rgb), C.c_double),
                     _p(_d(p.opacity), C.c_double), C.c_int(1 if dense else 0), C.c_double(cutoff),
                     _p(tl, C.c_int), C.c_int(0 if tl is None else len(tl)), _p(img, C.c_double))
    return img


def loss(image, target):
    """-> (L, G) with G = dL/dimage, float64."""
    H, W, _ = image.shape
    tgt = np.ascontiguousarray(target, dtype=np.float32)
    G = np.zeros_like(image, dtype=np.float64)
    L = lib().gso_loss(W, H, _p(_d(image), C.c_double), _p(tgt, C.c_float), _p(G, C.c_double))
    return float(L), G


def psnr(image, target) -> float:
    H, W, _ = image.shape
    tgt = np.ascontiguousarray(target, dtype=np.float32)
    return float(lib().gso_psnr(W, H, _p(_d(image), C.c_double), _p(tgt, C.c_float)))


def _roi(mask):
    return None if mask is None else np.ascontiguousarray(np.asarray(mask) != 0, dtype=np.uint8)


def loss_roi(image, target, roi):
    """c-16 -> (L, G): mean squared error over the ROI's pixels (roi None: c-4); G is zero outside the ROI."""
    H, W, _ = image.shape
    tgt = np.ascontiguousarray(target, dtype=np.float32)
    G = np.zeros_like(image, dtype=np.float64)
    f = lib().gso_loss_roi
    f.restype = C.c_double
    L = f(W, H, _p(_d(image), C.c_double), _p(tgt, C.c_float), _p(_roi(roi), C.c_ubyte), _p(G, C.c_double))
    if L != L:
        raise ValueError("empty ROI")
    return float(L), G


def psnr_roi(image, target, roi) -> float:
    H, W, _ = image.shape
    tgt = np.ascontiguousarray(target, dtype=np.float32)
    f = lib().gso_psnr_roi
    f.restype = C.c_double
    v = float(f(W, H, _p(_d(image), C.c_double), _p(tgt, C.c_float), _p(_roi(roi), C.c_ubyte)))
    if v != v:
        raise ValueError("empty ROI")
    return v


def backward(W, H, p: Params, G, *, dense=False, cutoff=CUTOFF, subset=None):
    """-> grad [N,9] float64, columns (mu_x, mu_y, l1, l2, l3, r, g, b, o).
    ``subset``: only these Gaussian ids are computed (other rows zero)."""
    grad = np.zeros((p.n, 9), dtype=np.float64)
    sub = None if subset is None else np.ascontiguousarray(subset, dtype=np.int32)
    lib().gso_backward(W, H, p.n, _p(_d(p.mu), C.c_double), _p(_d(p.chol), C.c_double), _p(_d(p.rgb), C.c_double),
                       _p(_d(p.opacity), C.c_double), _p(_d(G), C.c_double), C.c_int(1 if dense else 0),
                       C.c_double(cutoff), _p(sub, C.c_int), C.c_int(0 if sub is None else len(sub)),
                       _p(grad, C.c_double))
    return grad


def adam(p: Params, grad, m, v, lr, t, *, beta1=0.9, beta2=0.999, eps=1e-8, active=None, l_min=L_MIN):
    """In-place Adam step on p, m, v ([N,9] float64)."""
    lr4 = _d(np.broadcast_to(np.asarray(lr, dtype=np.float64), (4,)))
    act = None if active is None else np.ascontiguousarray(active, dtype=np.uint8)
    for a in (p.mu, p.chol, p.rgb, p.opacity, m, v):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    lib().gso_adam(p.n, _p(p.mu, C.c_double), _p(p.chol, C.c_double), _p(p.rgb, C.c_double),
                   _p(p.opacity, C.c_double), _p(_d(grad), C.c_double), _p(m, C.c_double), _p(v, C.c_double),
                   _p(lr4, C.c_double), C.c_double(beta1), C.c_double(beta2), C.c_double(eps), C.c_int(t),
                   _p(act, C.c_ubyte), C.c_double(l_min))


@dataclass
class FitReport:
    final_loss: float
    psnr: float
    iters_run: int
    first_nonfinite_iter: int
    n_active: int
    loss_trace: np.ndarray | None = None


def fit(W, H, p: Params, target, iters, lr=1e-2, *, beta1=0.9, beta2=0.999, eps=1e-8, active=None, l_min=L_MIN,
        cutoff=CUTOFF, trace=False, roi=None):
    """In-place fit of p to target.  -> FitReport (and m, v as attributes).  roi: the loss region of c-16."""
    N = p.n
    m = np.zeros((N, 9))
    v = np.zeros((N, 9))
    lr4 = _d(np.broadcast_to(np.asarray(lr, dtype=np.float64), (4,)))
    act = None if active is None else np.ascontiguousarray(active, dtype=np.uint8)
    tgt = np.ascontiguousarray(target, dtype=np.float32)
    tr = np.zeros(iters + 1) if trace else None
    fl, ps, nf = C.c_double(0), C.c_double(0), C.c_int(0)
    if roi is not None and not np.any(roi):
        raise ValueError("empty ROI")
    lib().gso_fit_roi(W, H, N, _p(p.mu, C.c_double), _p(p.chol, C.c_double), _p(p.rgb, C.c_double),
                      _p(p.opacity, C.c_double), _p(m, C.c_double), _p(v, C.c_double), _p(tgt, C.c_float),
                      _p(_roi(roi), C.c_ubyte), C.c_int(iters), _p(lr4, C.c_double), C.c_double(beta1),
                      C.c_double(beta2), C.c_double(eps), _p(act, C.c_ubyte), C.c_double(l_min), C.c_double(cutoff),
                      _p(tr, C.c_double), C.byref(fl), C.byref(ps), C.byref(nf))
    rep = FitReport(fl.value, ps.value, iters, nf.value, N if act is None else int(act.sum()), tr)
    rep.m, rep.v = m, v
    return rep


def lr_schedule(i, iters, base, decay=0.5, milestones=(0.6, 0.85)):
    """c-12 ("dynamic learning rate scheduler", read as SPEC.md:267-275): learning rate of
    iteration i (0-based) = base * decay^(number of milestones j with i >= round(milestone_j * iters));
    milestones and decay are binary32 values (they cross the C-ABI as floats)."""
    s = 1.0
    for ms in milestones:
        if float(i) >= math.floor(float(np.float32(ms)) * float(iters) + 0.5):
            s *= float(np.float32(decay))
    return base * s


def fit_sched(W, H, p: Params, target, iters, lr=1e-2, *, decay=0.5, milestones=(0.6, 0.85), target_psnr=0.0,
              check_every=50, beta1=0.9, beta2=0.999, eps=1e-8):
    """c-12: the c-7 loop with the lr schedule and an early stop once the PSNR of the clamped render,
    evaluated after every check_every-th iteration, reaches target_psnr.  A plain loop over
    the oracle's own steps.  In place; -> FitReport (iters_run = iterations done)."""
    N = p.n
    m = np.zeros((N, 9))
    v = np.zeros((N, 9))
    tgt = np.ascontiguousarray(target, dtype=np.float32)
    done = 0
    for k in range(1, iters + 1):
        img = render(W, H, p)
        _, G = loss(img, tgt)
        g = backward(W, H, p, G)
        adam(p, g, m, v, lr_schedule(k - 1, iters, lr, decay, milestones), k, beta1=beta1, beta2=beta2, eps=eps)
        done = k
        if target_psnr > 0 and k % check_every == 0 and psnr(render(W, H, p), tgt) >= target_psnr:
            break
    img = render(W, H, p)
    L, _ = loss(img, tgt)
    return FitReport(L, psnr(img, tgt), done, 0, N)


def fake_quantize(p: Params, spec) -> Params:
    """c-14: quantise-dequantise every parameter column with its
    uniform quantiser, in single-rounded binary32, ties to even:
        idx = clamp(rint((x - lo) * inv_step), 0, levels);  x_q = lo + idx * step.
    spec = (levels[9], lo[9], step[9], inv_step[9]); levels 0 = pass-through.  -> new Params (float64
    holding binary32 values)."""
    levels, lo, step, inv = spec
    flat = p.flat9().astype(np.float32)
    out = flat.copy()
    for j in range(9):
        if int(levels[j]) == 0:
            continue
        x = flat[:, j]
        t = (x - np.float32(lo[j])).astype(np.float32) * np.float32(inv[j])
        i = np.rint(t.astype(np.float32)).astype(np.float32)
        i = np.minimum(np.maximum(i, np.float32(0.0)), np.float32(levels[j]))
        out[:, j] = (np.float32(lo[j]) + (i * np.float32(step[j])).astype(np.float32)).astype(np.float32)
    o = out.astype(np.float64)
    return Params(o[:, 0:2].copy(), o[:, 2:5].copy(), o[:, 5:8].copy(), o[:, 8].copy())


def fit_qat(W, H, p: Params, target, iters, spec, lr=1e-2, *, beta1=0.9, beta2=0.999, eps=1e-8):
    """c-14: the c-7 loop with quantisation in it: render and gradients at fake_quantize(theta),
    the gradient applied to the raw theta (straight-through).  The raw parameters are kept in
    binary32 between steps (they are what a caller stores).  The report describes the QUANTISED set.
    In place; -> FitReport."""
    N = p.n
    m = np.zeros((N, 9))
    v = np.zeros((N, 9))
    tgt = np.ascontiguousarray(target, dtype=np.float32)
    for k in range(1, iters + 1):
        pq = fake_quantize(p, spec)
        _, G = loss(render(W, H, pq), tgt)
        g = backward(W, H, pq, G)
        adam(p, g, m, v, lr, k, beta1=beta1, beta2=beta2, eps=eps)
    pq = fake_quantize(p, spec)
    img = render(W, H, pq)
    L, _ = loss(img, tgt)
    return FitReport(L, psnr(img, tgt), iters, 0, N)


def rnd64(seed, i, k) -> int:
    return int(lib().gso_rnd64(C.c_uint64(seed), C.c_uint64(i), C.c_uint64(k)))


def roi_weights(frame, mask):
    H, W, _ = frame.shape
    fr = np.ascontiguousarray(frame, dtype=np.float32)
    mk = np.ascontiguousarray(mask, dtype=np.uint8)
    w_in = np.zeros((H, W), dtype=np.int32)
    w_out = np.zeros((H, W), dtype=np.int32)
    lib().gso_roi_weights(W, H, _p(fr, C.c_float), _p(mk, C.c_ubyte), _p(w_in, C.c_int), _p(w_out, C.c_int))
    return w_in, w_out


def init_roi(frame, mask, N, seed, s_min, s_max):
    """-> (mu, chol, rgb, opacity float32 arrays, pix int64 [N]); raises on empty ROI."""
    H, W, _ = frame.shape
    fr = np.ascontiguousarray(frame, dtype=np.float32)
    mk = np.ascontiguousarray(mask, dtype=np.uint8)
    mu = np.zeros((N, 2), dtype=np.float32)
    chol = np.zeros((N, 3), dtype=np.float32)
    rgb = np.zeros((N, 3), dtype=np.float32)
    op = np.zeros(N, dtype=np.float32)
    pix = np.zeros(N, dtype=np.int64)
    rc = lib().gso_init_roi(W, H, _p(fr, C.c_float), _p(mk, C.c_ubyte), C.c_int(N), C.c_uint64(seed),
                            C.c_double(s_min), C.c_double(s_max), _p(mu, C.c_float), _p(chol, C.c_float),
                            _p(rgb, C.c_float), _p(op, C.c_float), _p(pix, C.c_longlong))
    if rc != 0:
        raise ValueError(f"gso_init_roi failed with {rc} ({'empty ROI' if rc == -3 else 'bad argument'})")
    return mu, chol, rgb, op, pix


def init_superpixel(frame, mask, N, compactness=10, iters=10):
    """SLIC-style superpixel initialiser (c-11).  -> (mu, chol, rgb, opacity float32 [K,...],
    labels int32 [H,W] (-1 outside the ROI), (GX, GY) the cell grid); K <= N.  Raises on an empty ROI."""
    H, W, _ = frame.shape
    fr = np.ascontiguousarray(frame, dtype=np.float32)
    mk = np.ascontiguousarray(mask, dtype=np.uint8)
    mu = np.zeros((N, 2), dtype=np.float32)
    chol = np.zeros((N, 3), dtype=np.float32)
    rgb = np.zeros((N, 3), dtype=np.float32)
    op = np.zeros(N, dtype=np.float32)
    labels = np.zeros((H, W), dtype=np.int32)
    S = (C.c_int * 2)()
    k = lib().gso_init_superpixel(W, H, _p(fr, C.c_float), _p(mk, C.c_ubyte), C.c_int(N), C.c_int(compactness),
                                  C.c_int(iters), _p(mu, C.c_float), _p(chol, C.c_float), _p(rgb, C.c_float),
                                  _p(op, C.c_float), _p(labels, C.c_int), S)
    if k < 0:
        raise ValueError(f"gso_init_superpixel failed with {k} ({'empty ROI' if k == -3 else 'bad argument'})")
    return mu[:k], chol[:k], rgb[:k], op[:k], labels, (int(S[0]), int(S[1]))


def pframe_select(W, H, p: Params, frame, tau, cutoff=CUTOFF, roi=None):
    """-> (tile_resid [T] f64, tile_flag [T] u8, active [N] u8, n_active).  roi: residuals over the ROI's pixels (c-16)."""
    _, _, T = tiles_of(W, H)
    fr = np.ascontiguousarray(frame, dtype=np.float32)
    resid = np.zeros(T)
    flag = np.zeros(T, dtype=np.uint8)
    active = np.zeros(max(p.n, 1), dtype=np.uint8)
    na = C.c_int(0)
    lib().gso_pframe_select_roi(W, H, p.n, _p(_d(p.mu), C.c_double), _p(_d(p.chol), C.c_double),
                                _p(_d(p.rgb), C.c_double), _p(_d(p.opacity), C.c_double), _p(fr, C.c_float),
                                _p(_roi(roi), C.c_ubyte), C.c_double(tau), C.c_double(cutoff), _p(resid, C.c_double),
                                _p(flag, C.c_ubyte), _p(active, C.c_ubyte), C.byref(na))
    return resid, flag, active[:p.n], na.value


def pframe_select_pixels(W, H, p: Params, frame, tau, eps=0.01, dilate=False, changed=None, cutoff=CUTOFF,
                         want_wmax=False):
    """c-13 -> (changed [H,W] u8, resid [H,W] f64 max-channel residual (zeros when `changed` is given),
    active [N] u8, n_active); with want_wmax also wmax [N] f64, the largest exp(-sigma) of each Gaussian over
    the changed pixels of its listed tiles (active == wmax >= eps)."""
    fr = np.ascontiguousarray(frame, dtype=np.float32)
    ch_in = None if changed is None else np.ascontiguousarray(changed, dtype=np.uint8)
    ch_out = np.zeros((H, W), dtype=np.uint8)
    resid = np.zeros((H, W))
    active = np.zeros(max(p.n, 1), dtype=np.uint8)
    wmax = np.zeros(max(p.n, 1))
    na = C.c_int(0)
    lib().gso_pframe_select_pixels(W, H, p.n, _p(_d(p.mu), C.c_double), _p(_d(p.chol), C.c_double),
                                   _p(_d(p.rgb), C.c_double), _p(_d(p.opacity), C.c_double), _p(fr, C.c_float),
                                   C.c_double(tau), C.c_double(float(eps)), C.c_int(1 if dilate else 0),
                                   C.c_double(cutoff), _p(ch_in, C.c_ubyte), _p(ch_out, C.c_ubyte),
                                   _p(resid, C.c_double), _p(active, C.c_ubyte), _p(wmax, C.c_double), C.byref(na))
    if want_wmax:
        return ch_out, resid, active[:p.n], na.value, wmax[:p.n]
    return ch_out, resid, active[:p.n], na.value


def pframe_select_pixels_roi(W, H, p: Params, frame, tau, roi, eps=0.01, dilate=False, cutoff=CUTOFF):
    """c-13 with an ROI ("pixel marked changed iff max-channel |current - reference_render| > tau and
    pixel in ROI"): the raw change map is intersected with the ROI, THEN dilated; the influence test is c-13's.
    -> (changed [H,W] u8, active [N] u8, n_active)."""
    raw, _, _, _ = pframe_select_pixels(W, H, p, frame, tau, eps=eps, dilate=False, cutoff=cutoff)
    raw = (raw != 0) & (np.asarray(roi) != 0)
    ch = raw.copy()
    if dilate:
        pad = np.pad(raw, 1)
        for dy in range(3):
            for dx in range(3):
                ch |= pad[dy:dy + H, dx:dx + W]
    ch = ch.astype(np.uint8)
    _, _, active, na = pframe_select_pixels(W, H, p, frame, tau, eps=eps, changed=ch, cutoff=cutoff)
    return ch, active, na


def encode_pframe(W, H, p: Params, frame, tau, iters, lr=1e-2, *, beta1=0.9, beta2=0.999, eps=1e-8, l_min=L_MIN,
                  cutoff=CUTOFF):
    """In-place P-frame encode of p against frame.  -> (active [N] u8, FitReport)."""
    N = p.n
    m = np.zeros((N, 9))
    v = np.zeros((N, 9))
    lr4 = _d(np.broadcast_to(np.asarray(lr, dtype=np.float64), (4,)))
    fr = np.ascontiguousarray(frame, dtype=np.float32)
    active = np.zeros(max(N, 1), dtype=np.uint8)
    na, it, nf = C.c_int(0), C.c_int(0), C.c_int(0)
    fl, ps = C.c_double(0), C.c_double(0)
    lib().gso_encode_pframe(W, H, N, _p(p.mu, C.c_double), _p(p.chol, C.c_double), _p(p.rgb, C.c_double),
                            _p(p.opacity, C.c_double), _p(m, C.c_double), _p(v, C.c_double), _p(fr, C.c_float),
                            C.c_double(tau), C.c_int(iters), _p(lr4, C.c_double), C.c_double(beta1),
                            C.c_double(beta2), C.c_double(eps), C.c_double(l_min), C.c_double(cutoff),
                            _p(active, C.c_ubyte), C.byref(na), C.byref(it), C.byref(fl), C.byref(ps), C.byref(nf))
    return active[:N], FitReport(fl.value, ps.value, it.value, nf.value, na.value)


# ---- GoP loop over a sequence --------------

def gop_frame_types(n_frames: int, K: int):
    """"The codec determines whether to generate an I-frame or a P-frame based on a user-defined
    Group of Pictures (GoP) sequence length.  For example, a GoP length of 4 results in an I-frame every four
    P-frames", read as SPEC.md:439, 487 read it: frame f is an I-frame iff f % K == 0 ([I,P,P,P,I,...]; K = 1:
    all I).  -> list of 'I' / 'P'."""
    if K < 1 or n_frames < 0:
        raise ValueError("GoP length K >= 1, n_frames >= 0")
    return ["I" if f % K == 0 else "P" for f in range(n_frames)]


def encode_gop(W, H, frames, masks, K, N, *, init="roi", seed=1, s_min=1.0, s_max=8.0, compactness=10,
               kmeans_iters=10, iframe_iters=1000, pframe_iters=200, lr=1e-2, beta1=0.9, beta2=0.999, eps=1e-8,
               decay=1.0, milestones=(0.6, 0.85), target_psnr=0.0, check_every=25, tau=0.02, pixel_select=False,
               influence_eps=0.01, dilate=False):
    """The sequence loop, a plain composition of the single-frame steps above: an I-frame is initialised from
    its own frame and mask (init_roi with seed + f, or init_superpixel) and fitted from zeroed moments (c-7, with
    the c-12 schedule when one is asked for); a P-frame starts from the previous frame's fitted set, selects
    (c-9 tile rule or c-13 pixel rule) and refits the selected Gaussians from zeroed moments.
    -> list of (type, Params copy, active [n] uint8, FitReport), one per frame."""
    types = gop_frame_types(len(frames), K)
    out, p = [], None
    for f, frame in enumerate(frames):
        if types[f] == "I":
            if init == "roi":
                mu, chol, rgb, op, _ = init_roi(frame, masks[f], N, seed + f, s_min, s_max)
            else:
                mu, chol, rgb, op, _, _ = init_superpixel(frame, masks[f], N, compactness, kmeans_iters)
            p = Params(_d(mu).copy(), _d(chol).copy(), _d(rgb).copy(), _d(op).copy())
            if decay == 1.0 and not target_psnr > 0:
                rep = fit(W, H, p, frame, iframe_iters, lr=lr, beta1=beta1, beta2=beta2, eps=eps)
            else:
                rep = fit_sched(W, H, p, frame, iframe_iters, lr=lr, decay=decay, milestones=milestones,
                                target_psnr=target_psnr, check_every=check_every, beta1=beta1, beta2=beta2, eps=eps)
            active = np.ones(p.n, dtype=np.uint8)
        elif pixel_select:
            _, _, active, na = pframe_select_pixels(W, H, p, frame, tau, eps=influence_eps, dilate=dilate)
            if na == 0:
                img = render(W, H, p)
                rep = FitReport(loss(img, np.ascontiguousarray(frame, dtype=np.float32))[0], psnr(img, frame), 0, 0, 0)
            else:
                rep = fit(W, H, p, frame, pframe_iters, lr=lr, beta1=beta1, beta2=beta2, eps=eps, active=active)
        else:
            active, rep = encode_pframe(W, H, p, frame, tau, pframe_iters, lr=lr, beta1=beta1, beta2=beta2, eps=eps)
        out.append((types[f], p.copy(), np.array(active, dtype=np.uint8), rep))
    return out
