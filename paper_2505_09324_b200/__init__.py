"""paper_2505_09324_b200 -- Python binding of libgs2d (include/gs2d.h).

Argument marshalling only: every step of the hot path (tile binning, forward
rasterizer, backward, fused Adam, ROI init, P-frame selection) runs in the
hand-written sm_100a kernels of ``csrc/``.  PyTorch provides device memory and
streams.  There is no CPU fallback: if ``libgs2d.so`` cannot be loaded or built
the import of any compute entry point raises.

Functions carry the C names (``gs_render`` ...); ``Context`` is a small
convenience wrapper that owns a ``gs_ctx``.
"""
from __future__ import annotations

import ctypes as C
import math
from dataclasses import dataclass

from . import build as _build

__all__ = [
    "Params", "AdamState", "FitReport", "Context", "GsError", "lib",
    "gs_create", "gs_destroy", "gs_status", "gs_set_deterministic", "gs_set_roi", "gs_init_roi", "gs_init_superpixel", "gs_render", "gs_render_backward", "gs_adam_step",
    "gs_encode_iframe", "gs_encode_iframe_sched", "gs_encode_pframe", "gs_decode", "gs_set_quantization", "gs_fake_quantize", "gs_fit_steps", "gs_pframe_select", "gs_pframe_select_pixels", "gs_encode_pframe_pixels", "gs_loss_psnr",
    "gs_get_bins", "gs_get_tile_loss", "gs_decode_static", "gs_decode_host", "gs_encode_iframe_host", "gs_profile_fit_step", "gs_profile_decode", "FIT_KERNELS", "shard_units",
]

GS_OK = 0
# bytes the binning stores per (tile, Gaussian) pair: the id (include/gs2d.h, gs_config.max_pairs)
LIST_ENTRY_BYTES = 4
_ERR = {-1: "GS_ERR_INVALID_ARGUMENT", -2: "GS_ERR_INVALID_PARAMETER", -3: "GS_ERR_EMPTY_MASK",
        -4: "GS_ERR_CAPACITY", -5: "GS_ERR_NONFINITE", -6: "GS_ERR_CUDA", -7: "GS_ERR_UNSUPPORTED"}


class GsError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        detail = ""
        if code == -6:
            detail = ": " + lib().gs_last_cuda_error().decode()
        super().__init__(f"{where} -> {_ERR.get(code, code)}{detail}")


class _Config(C.Structure):
    _fields_ = [("width", C.c_int), ("height", C.c_int), ("tile", C.c_int), ("cutoff", C.c_float),
                ("l_min", C.c_float), ("max_gaussians", C.c_int), ("max_pairs", C.c_longlong)]


class _Params(C.Structure):
    _fields_ = [("mu", C.c_void_p), ("chol", C.c_void_p), ("rgb", C.c_void_p), ("opacity", C.c_void_p),
                ("n", C.c_int)]


class _AdamState(C.Structure):
    _fields_ = [("m", C.c_void_p), ("v", C.c_void_p)]


class _FitOpts(C.Structure):
    _fields_ = [("iters", C.c_int), ("lr", C.c_float * 4), ("beta1", C.c_float), ("beta2", C.c_float),
                ("eps", C.c_float), ("resume", C.c_int)]


class _QuantSpec(C.Structure):
    _fields_ = [("levels", C.c_int * 9), ("lo", C.c_float * 9), ("step", C.c_float * 9), ("inv_step", C.c_float * 9)]


def _qspec(spec) -> _QuantSpec:
    """spec: (levels[9] int, lo[9], step[9], inv_step[9] float32) -- e.g. workloads.uniform_quant_spec(...)"""
    levels, lo, step, inv = spec
    return _QuantSpec((C.c_int * 9)(*[int(x) for x in levels]), (C.c_float * 9)(*[float(x) for x in lo]),
                      (C.c_float * 9)(*[float(x) for x in step]), (C.c_float * 9)(*[float(x) for x in inv]))


class _FitSchedule(C.Structure):
    _fields_ = [("decay", C.c_float), ("milestone", C.c_float * 2), ("target_psnr", C.c_float),
                ("check_every", C.c_int)]


class _FitReport(C.Structure):
    _fields_ = [("final_loss", C.c_double), ("psnr", C.c_double), ("iters_run", C.c_int),
                ("first_nonfinite_iter", C.c_int), ("n_active", C.c_int), ("n_pairs", C.c_longlong)]


class _GopOpts(C.Structure):
    _fields_ = [("gop_length", C.c_int), ("init", C.c_int), ("n", C.c_int), ("seed", C.c_ulonglong),
                ("s_min", C.c_float), ("s_max", C.c_float), ("compactness", C.c_int), ("kmeans_iters", C.c_int),
                ("iframe", _FitOpts), ("sched", _FitSchedule), ("pframe", _FitOpts), ("pixel_select", C.c_int),
                ("tau", C.c_float), ("influence_eps", C.c_float), ("dilate", C.c_int)]


class _FrameReport(C.Structure):
    _fields_ = [("type", C.c_int), ("n", C.c_int), ("fit", _FitReport)]


_lib = None


def lib():
    """Load (building if stale) libgs2d.so.  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.is_stale():
        try:
            path = _build.build()
        except Exception as e:  # noqa: BLE001
            import os
            if not os.path.exists(_build.LIB):
                raise RuntimeError("libgs2d.so is missing and could not be built; there is no CPU fallback") from e
            path = _build.LIB  # a built library travelled with the tree; nvcc is absent here
    L = C.CDLL(path)
    vp, ci, cf, cll, cull = C.c_void_p, C.c_int, C.c_float, C.c_longlong, C.c_ulonglong
    sig = {
        "gs_create": [C.POINTER(_Config), C.POINTER(vp)],
        "gs_destroy": [vp],
        "gs_status": [vp, vp],
        "gs_set_deterministic": [vp, ci],
        "gs_set_roi": [vp, vp, vp],
        "gs_init_roi": [vp, vp, vp, ci, cull, cf, cf, _Params, vp],
        "gs_init_superpixel": [vp, vp, vp, ci, ci, ci, _Params, vp, C.POINTER(ci), vp],
        "gs_render": [vp, _Params, vp, ci, vp],
        "gs_render_backward": [vp, _Params, vp, _Params, vp],
        "gs_adam_step": [vp, _Params, _Params, _AdamState, C.POINTER(cf), cf, cf, cf, ci, vp, vp],
        "gs_encode_iframe": [vp, vp, _Params, _AdamState, C.POINTER(_FitOpts), C.POINTER(_FitReport), vp],
        "gs_encode_pframe": [vp, vp, _Params, _AdamState, cf, C.POINTER(_FitOpts), vp, C.POINTER(_FitReport), vp],
        "gs_encode_iframe_sched": [vp, vp, _Params, _AdamState, C.POINTER(_FitOpts), C.POINTER(_FitSchedule),
                                   C.POINTER(_FitReport), vp],
        "gs_decode": [vp, _Params, vp, vp],
        "gs_set_quantization": [vp, C.POINTER(_QuantSpec)],
        "gs_fake_quantize": [vp, _Params, C.POINTER(_QuantSpec), _Params, vp],
        "gs_pframe_select_pixels": [vp, vp, _Params, cf, cf, ci, vp, vp, vp, C.POINTER(ci), vp],
        "gs_encode_pframe_pixels": [vp, vp, _Params, _AdamState, cf, cf, ci, C.POINTER(_FitOpts), vp,
                                    C.POINTER(_FitReport), vp],
        "gs_fit_steps": [vp, vp, _Params, _AdamState, C.POINTER(_FitOpts), ci, vp, vp],
        "gs_pframe_select": [vp, vp, _Params, cf, vp, vp, vp, C.POINTER(ci), vp],
        "gs_profile_fit_step": [vp, vp, _Params, _AdamState, C.POINTER(_FitOpts), ci, vp, C.POINTER(cf), vp],
        "gs_loss_psnr": [vp, vp, _Params, C.POINTER(C.c_double), C.POINTER(C.c_double), vp],
        "gs_profile_decode": [vp, _Params, vp, C.POINTER(cf), vp],
        "gs_get_bins": [vp, vp, vp, cll, C.POINTER(cll), vp],
        "gs_get_tile_loss": [vp, vp, vp],
        "gs_decode_host": [vp, _Params, vp, vp],
        "gs_decode_static": [_Params, ci, ci, cf, vp, vp],
        "gs_encode_iframe_host": [vp, vp, _Params, C.POINTER(_FitOpts), C.POINTER(_FitReport), vp],
        "gs_encode_gop": [vp, C.POINTER(vp), C.POINTER(vp), ci, C.POINTER(_GopOpts), _Params, _AdamState,
                          C.POINTER(_Params), vp, C.POINTER(_FrameReport), vp],
    }
    for name, args in sig.items():
        fn = getattr(L, name)
        fn.argtypes = args
        fn.restype = ci
    L.gs_last_cuda_error.restype = C.c_char_p
    L.gs_last_cuda_error.argtypes = []
    _lib = L
    return L


def _torch():
    import torch
    return torch


def _stream():
    return C.c_void_p(_torch().cuda.current_stream().cuda_stream)


def _check(rc: int, where: str, allow=()):
    if rc != GS_OK and rc not in allow:
        raise GsError(rc, where)
    return rc


@dataclass
class Params:
    """Device SoA parameter set (float32 CUDA tensors); also the shape of a gradient."""
    mu: "object"       # [N,2]
    chol: "object"     # [N,3]
    rgb: "object"      # [N,3]
    opacity: "object"  # [N]

    @property
    def n(self) -> int:
        return int(self.mu.shape[0])

    @staticmethod
    def from_numpy(gs, device="cuda") -> "Params":
        t = _torch()
        f = lambda a: t.as_tensor(a, dtype=t.float32).contiguous().to(device)  # noqa: E731
        return Params(f(gs.mu), f(gs.chol), f(gs.rgb), f(gs.opacity))

    @staticmethod
    def empty(n: int, device="cuda") -> "Params":
        t = _torch()
        return Params(t.empty((n, 2), dtype=t.float32, device=device), t.empty((n, 3), dtype=t.float32, device=device),
                      t.empty((n, 3), dtype=t.float32, device=device), t.empty((n,), dtype=t.float32, device=device))

    def clone(self) -> "Params":
        return Params(self.mu.clone(), self.chol.clone(), self.rgb.clone(), self.opacity.clone())

    def flat9(self):
        t = _torch()
        return t.cat([self.mu, self.chol, self.rgb, self.opacity[:, None]], dim=1)

    def _c(self, cuda=True) -> _Params:
        t = _torch()
        for a, shape in ((self.mu, 2), (self.chol, 3), (self.rgb, 3)):
            assert a.dtype == t.float32 and a.is_contiguous() and a.dim() == 2 and a.shape[1] == shape
            assert a.is_cuda == cuda and a.shape[0] == self.n
        assert self.opacity.dtype == t.float32 and self.opacity.is_contiguous() and self.opacity.shape == (self.n,)
        assert self.opacity.is_cuda == cuda
        return _Params(self.mu.data_ptr(), self.chol.data_ptr(), self.rgb.data_ptr(), self.opacity.data_ptr(), self.n)


@dataclass
class AdamState:
    m: "object"  # [N,9]
    v: "object"

    @staticmethod
    def zeros(n: int, device="cuda") -> "AdamState":
        t = _torch()
        return AdamState(t.zeros((n, 9), dtype=t.float32, device=device),
                         t.zeros((n, 9), dtype=t.float32, device=device))

    def _c(self) -> _AdamState:
        t = _torch()
        for a in (self.m, self.v):
            assert a.dtype == t.float32 and a.is_contiguous() and a.is_cuda and a.shape[1] == 9
        return _AdamState(self.m.data_ptr(), self.v.data_ptr())


@dataclass
class FitReport:
    final_loss: float
    psnr: float
    iters_run: int
    first_nonfinite_iter: int
    n_active: int
    n_pairs: int
    status: int = 0


def _opts(iters, lr, beta1, beta2, eps, resume=False) -> _FitOpts:
    lr4 = [float(lr)] * 4 if not hasattr(lr, "__len__") else [float(x) for x in lr]
    assert len(lr4) == 4
    return _FitOpts(int(iters), (C.c_float * 4)(*lr4), float(beta1), float(beta2), float(eps), int(bool(resume)))


def _report(r: _FitReport, status=0) -> FitReport:
    return FitReport(r.final_loss, r.psnr, r.iters_run, r.first_nonfinite_iter, r.n_active, r.n_pairs, status)


def _img_ok(ctx, a, cuda=True):
    t = _torch()
    assert a.dtype == t.float32 and a.is_contiguous() and a.is_cuda == cuda
    assert tuple(a.shape) == (ctx.height, ctx.width, 3), (tuple(a.shape), (ctx.height, ctx.width, 3))


# ---- functions with the C names -----------------------------------------------------------------

def gs_create(width, height, max_gaussians, max_pairs, cutoff=3.0, l_min=0.1, tile=16) -> int:
    cfg = _Config(int(width), int(height), int(tile), float(cutoff), float(l_min), int(max_gaussians), int(max_pairs))
    h = C.c_void_p()
    _check(lib().gs_create(C.byref(cfg), C.byref(h)), "gs_create")
    return h.value


def gs_destroy(handle) -> None:
    if handle:
        lib().gs_destroy(C.c_void_p(handle))


def gs_set_deterministic(ctx, on: bool) -> None:
    """Bit-reproducible fits: sorted lists, per-pair moment slots instead of floating-point atomics (include/gs2d.h)."""
    _check(lib().gs_set_deterministic(ctx._h, 1 if on else 0), "gs_set_deterministic")


def gs_set_roi(ctx, roi_mask) -> None:
    """Loss, PSNR and P-frame residuals over the ROI's pixels only (DESIGN.md c-16); None: the whole frame.  The mask
    (uint8 [H,W] on the device) is kept alive by the context object while it is set."""
    if roi_mask is not None:
        t = _torch()
        assert roi_mask.dtype == t.uint8 and roi_mask.is_cuda and roi_mask.is_contiguous()
        assert tuple(roi_mask.shape) == (ctx.height, ctx.width)
    _check(lib().gs_set_roi(ctx._h, None if roi_mask is None else roi_mask.data_ptr(), _stream()), "gs_set_roi")
    ctx._roi = roi_mask


def gs_status(ctx) -> int:
    return lib().gs_status(ctx._h, _stream())


def gs_init_roi(ctx, frame, roi_mask, n, seed, s_min, s_max, out: Params | None = None) -> Params:
    t = _torch()
    _img_ok(ctx, frame)
    assert roi_mask.dtype == t.uint8 and roi_mask.is_cuda and roi_mask.is_contiguous()
    assert tuple(roi_mask.shape) == (ctx.height, ctx.width)
    out = out if out is not None else Params.empty(n, frame.device)
    _check(lib().gs_init_roi(ctx._h, frame.data_ptr(), roi_mask.data_ptr(), int(n), int(seed), float(s_min),
                             float(s_max), out._c(), _stream()), "gs_init_roi")
    return out


def gs_init_superpixel(ctx, frame, roi_mask, n_segments, compactness=10, kmeans_iters=10, want_labels=True):
    """-> (Params with K <= n_segments rows (views of an n_segments allocation), labels [H,W] int32 or None)"""
    t = _torch()
    _img_ok(ctx, frame)
    assert roi_mask.dtype == t.uint8 and roi_mask.is_cuda and roi_mask.is_contiguous()
    assert tuple(roi_mask.shape) == (ctx.height, ctx.width)
    out = Params.empty(n_segments, frame.device)
    labels = t.empty((ctx.height, ctx.width), dtype=t.int32, device=frame.device) if want_labels else None
    k = C.c_int(0)
    _check(lib().gs_init_superpixel(ctx._h, frame.data_ptr(), roi_mask.data_ptr(), int(n_segments), int(compactness),
                                    int(kmeans_iters), out._c(), labels.data_ptr() if want_labels else None,
                                    C.byref(k), _stream()), "gs_init_superpixel")
    kk = k.value
    return Params(out.mu[:kk], out.chol[:kk], out.rgb[:kk], out.opacity[:kk]), labels


def gs_render(ctx, params: Params, clamp: bool = False, out=None):
    t = _torch()
    out = out if out is not None else t.empty((ctx.height, ctx.width, 3), dtype=t.float32, device=params.mu.device)
    _img_ok(ctx, out)
    _check(lib().gs_render(ctx._h, params._c(), out.data_ptr(), int(bool(clamp)), _stream()), "gs_render")
    return out


def gs_decode(ctx, params: Params, out=None):
    t = _torch()
    out = out if out is not None else t.empty((ctx.height, ctx.width, 3), dtype=t.float32, device=params.mu.device)
    _img_ok(ctx, out)
    _check(lib().gs_decode(ctx._h, params._c(), out.data_ptr(), _stream()), "gs_decode")
    return out


def gs_decode_static(params: Params, width: int, height: int, out, cutoff: float = 3.0, allow=()) -> int:
    """gs_decode without a context and without any device allocation inside the library (include/gs2d.h): for hosts
    that own all GPU memory themselves or must not call cudaMalloc after start-up.  ``out`` ([height, width, 3]
    float32, CUDA) is the caller's -- this wrapper allocates nothing either.  The library's scratch is one fixed array
    per GPU shared by all calls: at most 16 384 Gaussians, 4 096 tiles, 256 Gaussians per tile (GsError -4 beyond), and
    calls on one device must not overlap.  Synchronises the current stream.  Returns the status code; codes listed in
    ``allow`` are returned instead of raised."""
    t = _torch()
    assert out.dtype == t.float32 and out.is_contiguous() and out.is_cuda and tuple(out.shape) == (height, width, 3)
    return _check(lib().gs_decode_static(params._c(), int(width), int(height), float(cutoff), out.data_ptr(),
                                         _stream()), "gs_decode_static", allow)


def gs_render_backward(ctx, params: Params, dL_dimage, grad_out: Params | None = None) -> Params:
    _img_ok(ctx, dL_dimage)
    g = grad_out if grad_out is not None else Params.empty(params.n, params.mu.device)
    _check(lib().gs_render_backward(ctx._h, params._c(), dL_dimage.data_ptr(), g._c(), _stream()),
           "gs_render_backward")
    return g


def gs_adam_step(ctx, params: Params, grad: Params, state: AdamState, lr, t, beta1=0.9, beta2=0.999, eps=1e-8,
                 active=None) -> None:
    lr4 = [float(lr)] * 4 if not hasattr(lr, "__len__") else [float(x) for x in lr]
    arr = (C.c_float * 4)(*lr4)
    act = None
    if active is not None:
        tt = _torch()
        assert active.dtype == tt.uint8 and active.is_cuda and active.is_contiguous() and active.numel() == params.n
        act = active.data_ptr()
    _check(lib().gs_adam_step(ctx._h, params._c(), grad._c(), state._c(), arr, float(beta1), float(beta2), float(eps),
                              int(t), act, _stream()), "gs_adam_step")


def gs_encode_iframe(ctx, frame, params: Params, state: AdamState, iters, lr=1e-2, beta1=0.9, beta2=0.999,
                     eps=1e-8) -> FitReport:
    _img_ok(ctx, frame)
    o, r = _opts(iters, lr, beta1, beta2, eps), _FitReport()
    rc = _check(lib().gs_encode_iframe(ctx._h, frame.data_ptr(), params._c(), state._c(), C.byref(o), C.byref(r),
                                       _stream()), "gs_encode_iframe", allow=(-5,))
    return _report(r, rc)


def gs_encode_iframe_sched(ctx, frame, params: Params, state: AdamState, iters, lr=1e-2, decay=0.5,
                           milestones=(0.6, 0.85), target_psnr=0.0, check_every=50, beta1=0.9, beta2=0.999,
                           eps=1e-8) -> FitReport:
    _img_ok(ctx, frame)
    o, r = _opts(iters, lr, beta1, beta2, eps), _FitReport()
    sc = _FitSchedule(float(decay), (C.c_float * 2)(float(milestones[0]), float(milestones[1])), float(target_psnr),
                      int(check_every))
    rc = _check(lib().gs_encode_iframe_sched(ctx._h, frame.data_ptr(), params._c(), state._c(), C.byref(o),
                                             C.byref(sc), C.byref(r), _stream()), "gs_encode_iframe_sched",
                allow=(-5,))
    return _report(r, rc)


def gs_encode_pframe(ctx, frame, params: Params, state: AdamState, tau, iters, lr=1e-2, beta1=0.9, beta2=0.999,
                     eps=1e-8):
    t = _torch()
    _img_ok(ctx, frame)
    active = t.zeros(params.n, dtype=t.uint8, device=frame.device)
    o, r = _opts(iters, lr, beta1, beta2, eps), _FitReport()
    rc = _check(lib().gs_encode_pframe(ctx._h, frame.data_ptr(), params._c(), state._c(), float(tau), C.byref(o),
                                       active.data_ptr(), C.byref(r), _stream()), "gs_encode_pframe", allow=(-5,))
    return active, _report(r, rc)


def gs_fit_steps(ctx, frame, params: Params, state: AdamState, iters, t0=1, lr=1e-2, beta1=0.9, beta2=0.999, eps=1e-8,
                 active=None, resume=False) -> None:
    _img_ok(ctx, frame)
    o = _opts(iters, lr, beta1, beta2, eps, resume)
    act = active.data_ptr() if active is not None else None
    _check(lib().gs_fit_steps(ctx._h, frame.data_ptr(), params._c(), state._c(), C.byref(o), int(t0), act, _stream()),
           "gs_fit_steps")


FIT_KERNELS = ("bin", "fit", "adam")


def gs_profile_fit_step(ctx, frame, params: Params, state: AdamState, t=1, lr=1e-2, beta1=0.9, beta2=0.999, eps=1e-8,
                        active=None) -> dict:
    """One fit iteration with CUDA events between its kernels -> {kernel: ms}."""
    _img_ok(ctx, frame)
    o = _opts(1, lr, beta1, beta2, eps)
    ms = (C.c_float * 3)()
    act = active.data_ptr() if active is not None else None
    _check(lib().gs_profile_fit_step(ctx._h, frame.data_ptr(), params._c(), state._c(), C.byref(o), int(t), act, ms,
                                     _stream()), "gs_profile_fit_step")
    return dict(zip(FIT_KERNELS, [float(x) for x in ms]))


def gs_profile_decode(ctx, params: Params, out) -> dict:
    """One gs_decode with CUDA events between its kernels -> {"bin": ms, "forward": ms}."""
    _img_ok(ctx, out)
    ms = (C.c_float * 2)()
    _check(lib().gs_profile_decode(ctx._h, params._c(), out.data_ptr(), ms, _stream()), "gs_profile_decode")
    return {"bin": float(ms[0]), "forward": float(ms[1])}


def gs_pframe_select(ctx, frame, params: Params, tau):
    """-> (tile_resid [T] f64, tile_flag [T] u8, active [N] u8, n_active)"""
    t = _torch()
    _img_ok(ctx, frame)
    dev = frame.device
    resid = t.empty(ctx.n_tiles, dtype=t.float64, device=dev)
    flag = t.empty(ctx.n_tiles, dtype=t.uint8, device=dev)
    active = t.zeros(params.n, dtype=t.uint8, device=dev)
    na = C.c_int(0)
    _check(lib().gs_pframe_select(ctx._h, frame.data_ptr(), params._c(), float(tau), resid.data_ptr(), flag.data_ptr(),
                                  active.data_ptr(), C.byref(na), _stream()), "gs_pframe_select")
    return resid, flag, active, na.value


def gs_pframe_select_pixels(ctx, frame, params: Params, tau, eps=0.01, dilate=False, changed=None):
    """-> (changed [H,W] u8, active [N] u8, n_active)"""
    t = _torch()
    _img_ok(ctx, frame)
    dev = frame.device
    ch_out = t.empty((ctx.height, ctx.width), dtype=t.uint8, device=dev)
    active = t.zeros(params.n, dtype=t.uint8, device=dev)
    na = C.c_int(0)
    if changed is not None:
        assert changed.dtype == t.uint8 and changed.is_cuda and changed.is_contiguous()
        assert tuple(changed.shape) == (ctx.height, ctx.width)
    _check(lib().gs_pframe_select_pixels(ctx._h, frame.data_ptr(), params._c(), float(tau), float(eps),
                                         int(bool(dilate)), changed.data_ptr() if changed is not None else None,
                                         ch_out.data_ptr(), active.data_ptr(), C.byref(na), _stream()),
           "gs_pframe_select_pixels")
    return ch_out, active, na.value


def gs_encode_pframe_pixels(ctx, frame, params: Params, state: AdamState, tau, iters, eps=0.01, dilate=False,
                            lr=1e-2, beta1=0.9, beta2=0.999, eps_adam=1e-8):
    t = _torch()
    _img_ok(ctx, frame)
    active = t.zeros(params.n, dtype=t.uint8, device=frame.device)
    o, r = _opts(iters, lr, beta1, beta2, eps_adam), _FitReport()
    rc = _check(lib().gs_encode_pframe_pixels(ctx._h, frame.data_ptr(), params._c(), state._c(), float(tau),
                                              float(eps), int(bool(dilate)), C.byref(o), active.data_ptr(),
                                              C.byref(r), _stream()), "gs_encode_pframe_pixels", allow=(-5,))
    return active, _report(r, rc)


def gs_encode_gop(ctx, frames, masks, gop_length, n, *, init="roi", seed=1, s_min=1.0, s_max=8.0, compactness=10,
                  kmeans_iters=10, iframe_iters=1000, pframe_iters=200, lr=1e-2, beta1=0.9, beta2=0.999, eps_adam=1e-8,
                  decay=1.0, milestones=(0.6, 0.85), target_psnr=0.0, check_every=25, tau=0.02, pixel_select=False,
                  influence_eps=0.01, dilate=False):
    """GoP loop over a sequence: frames / masks are lists of device tensors (masks[f] may be None
    for P-frames).  -> (list of Params, one per frame; active [F, n] uint8; list of (type, FitReport))."""
    t = _torch()
    F = len(frames)
    for f in frames:
        _img_ok(ctx, f)
    dev = frames[0].device if F else "cuda"
    work, state = Params.empty(n, dev), AdamState.zeros(n, dev)
    outs = [Params.empty(n, dev) for _ in range(F)]
    active = t.zeros((F, n), dtype=t.uint8, device=dev)
    fp = (C.c_void_p * max(F, 1))(*[f.data_ptr() for f in frames])
    mp = (C.c_void_p * max(F, 1))(*[(m.data_ptr() if m is not None else None) for m in masks])
    op = (_Params * max(F, 1))(*[o._c() for o in outs])
    rp = (_FrameReport * max(F, 1))()
    sch = _FitSchedule(float(decay), (C.c_float * 2)(*[float(x) for x in milestones]), float(target_psnr),
                       int(check_every))
    go = _GopOpts(int(gop_length), {"roi": 0, "superpixel": 1}[init], int(n), int(seed), float(s_min), float(s_max),
                  int(compactness), int(kmeans_iters), _opts(iframe_iters, lr, beta1, beta2, eps_adam), sch,
                  _opts(pframe_iters, lr, beta1, beta2, eps_adam), int(bool(pixel_select)), float(tau),
                  float(influence_eps), int(bool(dilate)))
    _check(lib().gs_encode_gop(ctx._h, fp, mp, F, C.byref(go), work._c(), state._c(), op, active.data_ptr(), rp,
                               _stream()), "gs_encode_gop")
    res = []
    for f in range(F):
        k = int(op[f].n)
        o = outs[f]
        res.append(Params(o.mu[:k], o.chol[:k], o.rgb[:k], o.opacity[:k]))
    return res, active, [(int(rp[f].type), _report(rp[f].fit)) for f in range(F)]


def gs_set_quantization(ctx, spec=None) -> None:
    """QAT: spec = (levels, lo, step, inv_step) arrays of 9, or None to switch it off."""
    _check(lib().gs_set_quantization(ctx._h, C.byref(_qspec(spec)) if spec is not None else None),
           "gs_set_quantization")


def gs_fake_quantize(ctx, params: Params, spec, out: Params | None = None) -> Params:
    out = out if out is not None else Params.empty(params.n, params.mu.device)
    _check(lib().gs_fake_quantize(ctx._h, params._c(), C.byref(_qspec(spec)), out._c(), _stream()), "gs_fake_quantize")
    return out


def gs_loss_psnr(ctx, frame, params: Params):
    _img_ok(ctx, frame)
    a, b = C.c_double(0), C.c_double(0)
    _check(lib().gs_loss_psnr(ctx._h, frame.data_ptr(), params._c(), C.byref(a), C.byref(b), _stream()),
           "gs_loss_psnr")
    return a.value, b.value


def gs_get_bins(ctx):
    """-> (range [T+1] int32, list [P] int32) device tensors of the last binning."""
    t = _torch()
    dev = t.device("cuda", t.cuda.current_device())
    rng = t.empty(ctx.n_tiles + 1, dtype=t.int32, device=dev)
    P = C.c_longlong(0)
    _check(lib().gs_get_bins(ctx._h, rng.data_ptr(), None, 0, C.byref(P), _stream()), "gs_get_bins")
    lst = t.empty(max(P.value, 1), dtype=t.int32, device=dev)
    _check(lib().gs_get_bins(ctx._h, rng.data_ptr(), lst.data_ptr(), lst.numel(), C.byref(P), _stream()),
           "gs_get_bins")
    return rng, lst[:P.value]


def gs_get_tile_loss(ctx):
    """-> [T] float64 device tensor: per-tile sum of (C - T)^2 left by the last fit iteration or statistics render."""
    t = _torch()
    out = t.empty(ctx.n_tiles, dtype=t.float64, device=t.device("cuda", t.cuda.current_device()))
    _check(lib().gs_get_tile_loss(ctx._h, out.data_ptr(), _stream()), "gs_get_tile_loss")
    return out


def gs_decode_host(ctx, params_host: Params, out_host=None):
    """params_host / out_host: CPU tensors (pinned for asynchronous copies)."""
    t = _torch()
    out_host = out_host if out_host is not None else t.empty((ctx.height, ctx.width, 3), dtype=t.float32).pin_memory()
    _img_ok(ctx, out_host, cuda=False)
    _check(lib().gs_decode_host(ctx._h, params_host._c(cuda=False), out_host.data_ptr(), _stream()), "gs_decode_host")
    return out_host


def gs_encode_iframe_host(ctx, frame_host, params_host: Params, iters, lr=1e-2, beta1=0.9, beta2=0.999,
                          eps=1e-8) -> FitReport:
    _img_ok(ctx, frame_host, cuda=False)
    o, r = _opts(iters, lr, beta1, beta2, eps), _FitReport()
    rc = _check(lib().gs_encode_iframe_host(ctx._h, frame_host.data_ptr(), params_host._c(cuda=False), C.byref(o),
                                            C.byref(r), _stream()), "gs_encode_iframe_host", allow=(-5,))
    return _report(r, rc)


def shard_units(n_units: int, rank: int, world_size: int) -> range:
    """Multi-GPU sharding of the path: the independent units -- I-frames, or GoPs
    (one I-frame plus its P-frames) -- are dealt out in contiguous, balanced blocks,
    rank r getting units [r*n/w, (r+1)*n/w).  No data-path collective: every rank runs the
    single-GPU library on its own units; only results (parameter sets, timings) are gathered."""
    if not (0 <= rank < world_size) or n_units < 0:
        raise ValueError("shard_units: need 0 <= rank < world_size and n_units >= 0")
    return range((rank * n_units) // world_size, ((rank + 1) * n_units) // world_size)


class Context:
    """Owns a gs_ctx for frames of ``width`` x ``height``."""

    def __init__(self, width: int, height: int, max_gaussians: int, max_pairs: int | None = None, cutoff: float = 3.0,
                 l_min: float = 0.1):
        t = _torch()
        if not t.cuda.is_available():
            raise RuntimeError("paper_2505_09324_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.width, self.height = int(width), int(height)
        self.tiles_x, self.tiles_y = math.ceil(width / 16), math.ceil(height / 16)
        self.n_tiles = self.tiles_x * self.tiles_y
        self.max_gaussians = int(max_gaussians)
        self.max_pairs = int(max_pairs) if max_pairs is not None else max(4096, 32 * int(max_gaussians))
        self._h = gs_create(width, height, max_gaussians, self.max_pairs, cutoff, l_min)

    def close(self):
        if getattr(self, "_h", None):
            gs_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:  # noqa: BLE001
            pass

    init_roi = gs_init_roi
    init_superpixel = gs_init_superpixel
    render = gs_render
    decode = gs_decode
    render_backward = gs_render_backward
    adam_step = gs_adam_step
    encode_iframe = gs_encode_iframe
    encode_iframe_sched = gs_encode_iframe_sched
    encode_pframe = gs_encode_pframe
    fit_steps = gs_fit_steps
    pframe_select = gs_pframe_select
    profile_fit_step = gs_profile_fit_step
    loss_psnr = gs_loss_psnr
    get_bins = gs_get_bins
    status = gs_status
    decode_host = gs_decode_host
    encode_iframe_host = gs_encode_iframe_host
