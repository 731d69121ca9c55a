"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This module holds NO arithmetic of the method (no rendering, no binning, no
gradients, no Adam, no ROI sampler).  It only draws the inputs that both the
float64 oracle (``oracle/``) and the CUDA library (``paper_2505_09324_b200``)
consume, so that the two sides are fed bit-identical arrays.  numpy only.

The frames stand in for the paper's talking-head videos (Microsoft VCD,
PAPER.md:146), which are not in the container: one subject (textured ellipse
"head" plus a rectangular "torso") over a static vertical-gradient background
with additive Gaussian noise, at the sizes BASELINE.json's ``configs`` name.
Recipe: SURVEY.md §8(d); restated in DESIGN.md §4.

Every random stream is ``numpy.random.default_rng([S0, config_index,
stream_index])`` with S0 = 250509324.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

S0 = 250509324

# stream indices inside one config
STREAM_COLOURS = 0      # head / torso base colours
STREAM_GAUSSIANS = 1    # Gaussian parameter sets drawn on the host
STREAM_NOISE0 = 100     # frame k uses STREAM_NOISE0 + k


def rng(config_index: int, stream_index: int) -> np.random.Generator:
    return np.random.default_rng([S0, int(config_index), int(stream_index)])


@dataclass(frozen=True)
class FrameSpec:
    """Geometry of one synthetic talking-head frame (pixels; origin top-left)."""
    width: int
    height: int
    centre: tuple          # head centre (cx, cy)
    axes: tuple            # head semi-axes (ax, ay)
    torso: bool
    config_index: int


# BASELINE.json configs[0..3]; SURVEY.md §8(d)
SPEC_TINY = FrameSpec(64, 64, (32.0, 28.0), (14.0, 18.0), False, 0)
SPEC_ROI = FrameSpec(480, 272, (240.0, 119.0), (59.5, 76.5), True, 1)
SPEC_1080P = FrameSpec(1920, 1080, (960.0, 472.5), (220.0, 300.0), True, 2)
SPEC_PSEQ = FrameSpec(1920, 1080, (960.0, 472.5), (220.0, 300.0), True, 3)


def scaled_spec(width: int, height: int, config_index: int, torso: bool = True) -> FrameSpec:
    """A frame of arbitrary size with the 1080p layout scaled to it (test sizes)."""
    sx = width / 1920.0
    sy = height / 1080.0
    s = min(sx, sy)
    return FrameSpec(width, height, (960.0 * sx, 472.5 * sy), (220.0 * s, 300.0 * s), torso, config_index)


def talking_head_frame(spec: FrameSpec, frame_index: int = 0, *, shift_px_per_frame: float = 2.0,
                       rot_deg_per_frame: float = 0.5, noise_sigma: float = 0.02):
    """Return (frame float32 [H,W,3] in [0,1], roi_mask uint8 [H,W]).

    Frame ``k`` has the head/torso translated ``k*shift`` px to the right and
    rotated ``k*rot`` degrees about the head centre; the background is static;
    the noise stream is fresh per frame (BASELINE.json configs[3]).
    """
    W, H = spec.width, spec.height
    ax, ay = spec.axes
    cx = spec.centre[0] + shift_px_per_frame * frame_index
    cy = spec.centre[1]
    theta = math.radians(rot_deg_per_frame * frame_index)

    cols = rng(spec.config_index, STREAM_COLOURS)
    head_colour = cols.uniform(0.0, 1.0, 3)
    torso_colour = cols.uniform(0.0, 1.0, 3)

    ys, xs = np.meshgrid(np.arange(H, dtype=np.float64) + 0.5,
                         np.arange(W, dtype=np.float64) + 0.5, indexing="ij")
    img = np.empty((H, W, 3), dtype=np.float64)
    img[:] = (0.2 + 0.6 * ys / H)[..., None]

    # local coordinates: rotate by -theta about the head centre
    dx = xs - cx
    dy = ys - cy
    ct, st = math.cos(theta), math.sin(theta)
    xl = ct * dx + st * dy
    yl = -st * dx + ct * dy

    lam = max(8.0, ay / 9.0)
    texture = 0.1 * np.sin(2.0 * math.pi * xl / lam) * np.sin(2.0 * math.pi * yl / lam)

    head = (xl / ax) ** 2 + (yl / ay) ** 2 <= 1.0
    mask = head.copy()
    if spec.torso:
        torso = (np.abs(xl) <= 1.8 * ax) & (yl >= 0.95 * ay) & ~head
        img[torso] = torso_colour[None, :] + texture[torso][:, None]
        mask |= torso
    img[head] = head_colour[None, :] + texture[head][:, None]

    noise = rng(spec.config_index, STREAM_NOISE0 + frame_index).normal(0.0, noise_sigma, img.shape)
    img = np.clip(img + noise, 0.0, 1.0)
    return img.astype(np.float32), mask.astype(np.uint8)


@dataclass
class GaussianSet:
    """Host-side SoA parameter set, float32, the layout that crosses the C-ABI."""
    mu: np.ndarray        # [N,2]
    chol: np.ndarray      # [N,3]  l1,l2,l3 with L=[[l1,0],[l2,l3]]
    rgb: np.ndarray       # [N,3]
    opacity: np.ndarray   # [N]

    @property
    def n(self) -> int:
        return int(self.mu.shape[0])

    def copy(self) -> "GaussianSet":
        return GaussianSet(self.mu.copy(), self.chol.copy(), self.rgb.copy(), self.opacity.copy())


def chol_from_scale_rotation(s1, s2, theta):
    """Input recipe only: lower-triangular factor of R diag(s1^2,s2^2) R^T."""
    c, s = np.cos(theta), np.sin(theta)
    s11 = c * c * s1 * s1 + s * s * s2 * s2
    s12 = c * s * (s1 * s1 - s2 * s2)
    s22 = s * s * s1 * s1 + c * c * s2 * s2
    l1 = np.sqrt(s11)
    l2 = s12 / l1
    l3 = np.sqrt(s22 - l2 * l2)
    return np.stack([l1, l2, l3], axis=-1)


def tiny_gaussians(n: int = 256, width: int = 64, height: int = 64, config_index: int = 0) -> GaussianSet:
    """configs[0]: positions U[0,W)x[0,H), l=(2,0,2), colours U[0,1]^3, opacity 1."""
    g = rng(config_index, STREAM_GAUSSIANS)
    mu = np.stack([g.uniform(0, width, n), g.uniform(0, height, n)], axis=-1)
    chol = np.tile(np.array([2.0, 0.0, 2.0]), (n, 1))
    rgb = g.uniform(0.0, 1.0, (n, 3))
    return GaussianSet(mu.astype(np.float32), chol.astype(np.float32), rgb.astype(np.float32),
                       np.ones(n, dtype=np.float32))


def random_gaussians(n: int, width: int, height: int, *, s_min: float = 1.0, s_max: float = 16.0,
                     opacity_range=(0.05, 0.25), config_index: int = 4, stream: int = STREAM_GAUSSIANS,
                     margin: float = 0.0) -> GaussianSet:
    """configs[4]: mu uniform over the frame (optionally spilling ``margin`` px
    outside it), scales log-uniform [s_min,s_max], rotation U[0,pi), colours
    U[0,1]^3, opacity U[opacity_range]."""
    g = rng(config_index, stream)
    mu = np.stack([g.uniform(-margin, width + margin, n), g.uniform(-margin, height + margin, n)], axis=-1)
    ls = math.log(s_max / s_min)
    s1 = s_min * np.exp(g.uniform(0.0, 1.0, n) * ls)
    s2 = s_min * np.exp(g.uniform(0.0, 1.0, n) * ls)
    theta = g.uniform(0.0, math.pi, n)
    chol = chol_from_scale_rotation(s1, s2, theta)
    rgb = g.uniform(0.0, 1.0, (n, 3))
    op = g.uniform(opacity_range[0], opacity_range[1], n)
    return GaussianSet(mu.astype(np.float32), chol.astype(np.float32), rgb.astype(np.float32),
                       op.astype(np.float32))


def random_image_grad(width: int, height: int, config_index: int, stream: int = 7, scale: float = 1.0):
    """A synthetic dL/dimage [H,W,3] float32 for backward parity at any size."""
    g = rng(config_index, stream)
    return (scale * g.standard_normal((height, width, 3))).astype(np.float32)


def uniform_quant_spec(width: int, height: int, *, mu_bits: int = 16, chol_bits: int = 6, rgb_bits: int = 8,
                       chol_range=((0.1, 12.0), (-8.0, 8.0), (0.1, 12.0)), rgb_range=(0.0, 1.0), opacity_bits: int = 0,
                       opacity_range=(0.0, 1.0)):
    """Input recipe only: the uniform quantisers of the 9 parameter columns (mu_x, mu_y, l1, l2, l3,
    r, g, b, o) as (levels int32[9], lo, step, inv_step float32[9]).  Bit widths follow the paper's
    compression section (PAPER.md:110 via SPEC.md:378-381: mean 16 bits over the frame, Cholesky 6
    bits per channel, colour 8 bits); the ranges stand in for the PTQ calibration, which needs the
    paper's dataset.  step = (hi - lo) / levels and inv_step = levels / (hi - lo), each computed in
    float64 and rounded to binary32 once; 0 bits = the column passes through."""
    bits = [mu_bits, mu_bits, chol_bits, chol_bits, chol_bits, rgb_bits, rgb_bits, rgb_bits, opacity_bits]
    rng_ = [(0.0, float(width)), (0.0, float(height)), *chol_range, rgb_range, rgb_range, rgb_range, opacity_range]
    levels = np.zeros(9, dtype=np.int32)
    lo = np.zeros(9, dtype=np.float32)
    step = np.ones(9, dtype=np.float32)
    inv = np.ones(9, dtype=np.float32)
    for j, (b, (a, z)) in enumerate(zip(bits, rng_)):
        if b <= 0:
            continue
        levels[j] = (1 << b) - 1
        lo[j] = np.float32(a)
        span = float(z) - float(np.float32(a))
        step[j] = np.float32(span / float(levels[j]))
        inv[j] = np.float32(float(levels[j]) / span)
    return levels, lo, step, inv
