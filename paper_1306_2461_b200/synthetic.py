"""Seeded synthetic particle-image pairs shaped like the paper's camera frames.

This module is the ONE piece shared by the oracle side (tests, bench cpu_baseline) and the CUDA
side (tests, bench): it only *makes inputs*.  It holds none of the method's arithmetic (no warp,
gradient, window sum, solve, pyramid) and imports neither `oracle/` nor the CUDA binding.

The paper measured on its own water-channel recordings (8-bit, ROI 1792x384), which
are not public; BASELINE.json names no dataset.  The pairs below take the shapes and statistics of
BASELINE.json `configs` (lines 7-11) and stand in for them.  Recipe (DESIGN.md
"Input recipe"):

* NumPy ``default_rng(seed)``, seed = 13062461*10 + config index.
* particle count round(ppp*(W+2m)*(H+2m)), positions uniform on [-m, W+m) x [-m, H+m), m = 24,
  so particles enter and leave the frame consistently;
* each particle is an analytic Gaussian  A*exp(-((x-xp)^2+(y-yp)^2)/(2 sigma^2))  summed in fp64
  (support truncated at ceil(5 sigma)+1 px: < 1e-3 DN);
* frame 2 is rendered from the displaced positions p + d(p) -- no image interpolation anywhere;
* then noise, clip, round-to-nearest to the integer type.
* flow convention: I2(x+u, y+v) ~= I1(x, y); ground truth at pixel x is d(x) (reported only).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

MARGIN = 24
SEED_BASE = 13062461 * 10

WINDOW_BOX = 0
WINDOW_GAUSSIAN = 1


@dataclass
class FlowCase:
    """One frame pair plus the solver parameters of its config."""
    name: str
    I1: np.ndarray            # (H, W) uint8 / uint16
    I2: np.ndarray
    width: int
    height: int
    levels: int
    window_radius: int
    iterations: int
    window_type: int
    truth_u: np.ndarray | None = None   # (H, W) float64, d(x) at pixel centres
    truth_v: np.ndarray | None = None
    meta: dict = field(default_factory=dict)

    @property
    def create_args(self):
        return (self.width, self.height, self.levels, self.window_radius, self.iterations,
                self.window_type)


# --------------------------------------------------------------------------------------------
# rendering
# --------------------------------------------------------------------------------------------

def seed_particles(rng, width, height, ppp, amp_lo, amp_hi, margin=MARGIN):
    n = int(round(ppp * (width + 2 * margin) * (height + 2 * margin)))
    xp = rng.uniform(-margin, width + margin, n)
    yp = rng.uniform(-margin, height + margin, n)
    amp = rng.uniform(amp_lo, amp_hi, n)
    return xp, yp, amp


def render_particles(xp, yp, amp, sigma, width, height):
    """Sum of analytic Gaussians on integer pixel centres, fp64, (H, W)."""
    rad = int(math.ceil(5.0 * sigma)) + 1
    ix = np.rint(xp).astype(np.int64)
    iy = np.rint(yp).astype(np.int64)
    keep = (ix >= -rad) & (ix < width + rad) & (iy >= -rad) & (iy < height + rad)
    xp, yp, amp, ix, iy = xp[keep], yp[keep], amp[keep], ix[keep], iy[keep]
    offs = np.arange(-rad, rad + 1)
    inv = 1.0 / (2.0 * sigma * sigma)
    img = np.zeros(width * height, dtype=np.float64)
    # chunk over particles to bound memory: chunk x (2rad+1)^2 entries
    side = 2 * rad + 1
    chunk = max(1, (1 << 22) // (side * side))
    for s in range(0, xp.size, chunk):
        sl = slice(s, s + chunk)
        xx = ix[sl, None] + offs[None, :]                      # (n, side)
        yy = iy[sl, None] + offs[None, :]
        gx = np.exp(-(xx - xp[sl, None]) ** 2 * inv)
        gy = np.exp(-(yy - yp[sl, None]) ** 2 * inv) * amp[sl, None]
        mx = (xx >= 0) & (xx < width)
        my = (yy >= 0) & (yy < height)
        val = gy[:, :, None] * gx[:, None, :]                  # (n, side_y, side_x)
        m = my[:, :, None] & mx[:, None, :]
        flat = (yy[:, :, None] * width + xx[:, None, :])
        img += np.bincount(flat[m], weights=val[m], minlength=width * height)
    return img.reshape(height, width)


def quantize(img, dtype, maxval):
    return np.clip(np.rint(img), 0, maxval).astype(dtype)


# --------------------------------------------------------------------------------------------
# displacement fields d(x, y) -> (dx, dy), vectorised over arrays of positions
# --------------------------------------------------------------------------------------------

def field_uniform(dx, dy):
    def d(x, y):
        return np.full_like(x, dx, dtype=np.float64), np.full_like(y, dy, dtype=np.float64)
    return d


def field_lamb_oseen(xc, yc, peak, core):
    """Tangential displacement peak*g(rho/core)/g_max, g(s) = (1-exp(-s^2))/s (counter-clockwise
    in (x right, y down) index coordinates)."""
    g_max = 0.6381726863389515     # max of g, at s = 1.1209064227...
    def d(x, y):
        rx, ry = x - xc, y - yc
        rho = np.hypot(rx, ry)
        s = np.maximum(rho / core, 1e-12)
        dth = peak * (-np.expm1(-s * s) / s) / g_max
        rho = np.maximum(rho, 1e-12)
        return -dth * ry / rho, dth * rx / rho
    return d


def field_backward_step(width, height):
    """tanh shear layer, +8 px free stream, -1 px recirculation upstream of x = 0.7 W
    (stand-in for the paper's backward-facing-step flow)."""
    def d(x, y):
        S = 0.5 * (1.0 + np.tanh((0.6 * height - y) / 24.0))
        B = 0.5 * (1.0 - np.tanh((x - 0.7 * width) / 64.0))
        u = 8.0 * S - (1.0 - S) * B
        v = 0.5 * np.sin(2.0 * np.pi * x / 320.0) / np.cosh((y - 0.6 * height) / 24.0) ** 2
        return u, v
    return d


def mask_backward_step(width, height):
    """Obstacle mask (uint8, 1 = fluid, 0 = obstacle) for the NEXT item f4 (PAPER.md:175 'masks to avoid
    computations over obstacles or side walls'): the step body (x < 0.25 W below the shear layer at
    y = 0.6 H) and two side-wall bands of 3 percent of the height.  About 14 percent of the frame."""
    m = np.ones((height, width), dtype=np.uint8)
    wall = max(1, int(round(0.03 * height)))
    m[:wall, :] = 0
    m[height - wall:, :] = 0
    m[int(round(0.6 * height)):, :int(round(0.25 * width))] = 0
    return m


def field_random_smooth(rng, width, height, filt_sigma, rms, pad=64):
    """Two independent white-noise fields, Gaussian-filtered (FFT) on a padded grid, jointly scaled
    to sqrt(mean(u^2+v^2)) = rms over the image; evaluated off-grid by cubic splines."""
    from scipy import ndimage
    gw, gh = width + 2 * pad, height + 2 * pad
    fy = np.fft.fftfreq(gh)[:, None]
    fx = np.fft.rfftfreq(gw)[None, :]
    H = np.exp(-2.0 * (np.pi * filt_sigma) ** 2 * (fx * fx + fy * fy))
    comps = []
    for _ in range(2):
        w = rng.standard_normal((gh, gw))
        comps.append(np.fft.irfft2(np.fft.rfft2(w) * H, s=(gh, gw)))
    gu, gv = comps
    core = (slice(pad, pad + height), slice(pad, pad + width))
    scale = rms / math.sqrt(np.mean(gu[core] ** 2 + gv[core] ** 2))
    gu *= scale
    gv *= scale
    def d(x, y):
        coords = np.stack([np.asarray(y, dtype=np.float64) + pad, np.asarray(x, dtype=np.float64) + pad])
        shp = coords.shape[1:]
        coords = coords.reshape(2, -1)
        u = ndimage.map_coordinates(gu, coords, order=3, mode="nearest").reshape(shp)
        v = ndimage.map_coordinates(gv, coords, order=3, mode="nearest").reshape(shp)
        return u, v
    return d


def _pixel_grid(width, height):
    y, x = np.mgrid[0:height, 0:width]
    return x.astype(np.float64), y.astype(np.float64)


def _pair_from_field(rng, width, height, ppp, sigma, amp_lo, amp_hi, dfield):
    xp, yp, amp = seed_particles(rng, width, height, ppp, amp_lo, amp_hi)
    dx, dy = dfield(xp, yp)
    f1 = render_particles(xp, yp, amp, sigma, width, height)
    f2 = render_particles(xp + dx, yp + dy, amp, sigma, width, height)
    gx, gy = _pixel_grid(width, height)
    tu, tv = dfield(gx, gy)
    return f1, f2, tu, tv


# --------------------------------------------------------------------------------------------
# the five configs of BASELINE.json (lines 7-11); width/height may be overridden for small tests
# --------------------------------------------------------------------------------------------

def config1(width=256, height=256):
    """BASELINE.json:7 -- 256x256, fp32-from-uint8, sigma 1.0, 0.02 ppp, A~U(150,255), uniform
    shift (1.3,-0.7), 1 level, box radius 8, 4 iterations."""
    rng = np.random.default_rng(SEED_BASE + 1)
    f1, f2, tu, tv = _pair_from_field(rng, width, height, 0.02, 1.0, 150.0, 255.0,
                                      field_uniform(1.3, -0.7))
    return FlowCase("config1", quantize(f1, np.uint8, 255), quantize(f2, np.uint8, 255),
                    width, height, 1, 8, 4, WINDOW_BOX, tu, tv, {"input": "f32-from-u8"})


def config2(width=1024, height=1024):
    """BASELINE.json:8 -- 1024x1024 uint8, sigma 1.2, 0.03 ppp, noise sigma 3 DN, Lamb-Oseen vortex
    (peak 4 px, core 80 px), 2 levels, box radius 7, 6 iterations."""
    rng = np.random.default_rng(SEED_BASE + 2)
    core = 80.0 * min(width, height) / 1024.0
    f1, f2, tu, tv = _pair_from_field(rng, width, height, 0.03, 1.2, 150.0, 255.0,
                                      field_lamb_oseen(0.5 * (width - 1), 0.5 * (height - 1), 4.0, core))
    f1 = f1 + rng.normal(0.0, 3.0, f1.shape)
    f2 = f2 + rng.normal(0.0, 3.0, f2.shape)
    return FlowCase("config2", quantize(f1, np.uint8, 255), quantize(f2, np.uint8, 255),
                    width, height, 2, 7, 6, WINDOW_BOX, tu, tv, {"input": "u8"})


def config3(width=1280, height=1024, seed_offset=0):
    """BASELINE.json:9 -- 1280x1024 uint8, 0.025 ppp, backward-facing-step-like field (tanh shear,
    8 px max, -1 px recirculation), 3 levels, Gaussian window sigma 4 (R = 12), 10 iterations."""
    rng = np.random.default_rng(SEED_BASE + 3 + 1000 * seed_offset)
    f1, f2, tu, tv = _pair_from_field(rng, width, height, 0.025, 1.2, 150.0, 255.0,
                                      field_backward_step(width, height))
    return FlowCase("config3", quantize(f1, np.uint8, 255), quantize(f2, np.uint8, 255),
                    width, height, 3, 12, 10, WINDOW_GAUSSIAN, tu, tv, {"input": "u8"})


def config4(width=2048, height=2048, filt_sigma=None):
    """BASELINE.json:10 -- 2048x2048 uint16 (12-bit), sigma 1.5, 0.02 ppp, Poisson noise, random
    smooth field (Gaussian-filtered white noise, RMS 3 px), 4 levels, box radius 10, 8 iterations."""
    rng = np.random.default_rng(SEED_BASE + 4)
    filt = filt_sigma if filt_sigma is not None else 48.0 * min(width, height) / 2048.0
    dfield = field_random_smooth(rng, width, height, filt, 3.0)
    f1, f2, tu, tv = _pair_from_field(rng, width, height, 0.02, 1.5, 1500.0, 4095.0, dfield)
    f1 = rng.poisson(f1 + 20.0).astype(np.float64)
    f2 = rng.poisson(f2 + 20.0).astype(np.float64)
    return FlowCase("config4", quantize(f1, np.uint16, 4095), quantize(f2, np.uint16, 4095),
                    width, height, 4, 10, 8, WINDOW_BOX, tu, tv, {"input": "u16"})


class Config5Stream:
    """BASELINE.json:11 -- consecutive 1280x1024 uint8 frames of a time-varying shear layer with
    convected sinusoidal vortices (0.5 px/frame); particles are advected frame to frame (one
    midpoint step) by the divergence-free field of the stream function
        psi = int U(y) dy + (A/k) sin(k (x - 0.5 t)) sech^2((y - 0.5 H)/40),
        U(y) = 2 + 3 tanh((0.5 H - y)/40) px/frame,  k = 2 pi 5/(W + 2 m),  A = 1 px,
    with periodic wrap in x on the padded domain (keeps the seeding uniform).
    3 levels, box radius 8, 10 iterations.  Frames are produced lazily, in order."""

    levels, window_radius, iterations, window_type = 3, 8, 10, WINDOW_BOX

    def __init__(self, n_frames=256, width=1280, height=1024):
        self.n_frames, self.width, self.height = n_frames, width, height
        self.rng = np.random.default_rng(SEED_BASE + 5)
        self.xp, self.yp, self.amp = seed_particles(self.rng, width, height, 0.025, 150.0, 255.0)
        self.t = 0
        self.k = 2.0 * np.pi * 5.0 / (width + 2 * MARGIN)

    @property
    def create_args(self):
        return (self.width, self.height, self.levels, self.window_radius, self.iterations,
                self.window_type)

    def velocity(self, x, y, t):
        """(u, v) = (d psi/dy, -d psi/dx) in px/frame at time t (frames)."""
        H = self.height
        eta = (y - 0.5 * H) / 40.0
        sech2 = 1.0 / np.cosh(eta) ** 2
        ph = self.k * (x - 0.5 * t)
        u = 2.0 + 3.0 * np.tanh(-eta) + (1.0 / self.k) * np.sin(ph) * (-2.0 * sech2 * np.tanh(eta) / 40.0)
        v = -np.cos(ph) * sech2
        return u, v

    def _advect(self):
        u1, v1 = self.velocity(self.xp, self.yp, self.t)
        u2, v2 = self.velocity(self.xp + 0.5 * u1, self.yp + 0.5 * v1, self.t + 0.5)
        self.xp = self.xp + u2
        self.yp = self.yp + v2
        span = self.width + 2 * MARGIN
        self.xp = (self.xp + MARGIN) % span - MARGIN
        self.t += 1

    def frames(self):
        for i in range(self.n_frames):
            if i > 0:
                self._advect()
            yield quantize(render_particles(self.xp, self.yp, self.amp, 1.2, self.width, self.height),
                           np.uint8, 255)


def make_case(index, **kw):
    return {1: config1, 2: config2, 3: config3, 4: config4}[index](**kw)


# --------------------------------------------------------------------------------------------
# analytic test images used to pin the oracle (BASELINE.json:5 self-checks; SURVEY.md 8(c) pins)
# --------------------------------------------------------------------------------------------

def bandlimited_pair(width=256, height=256, shift=(0.37, -0.21), n_waves=24, seed=SEED_BASE + 11,
                     lam_lo=10.0, lam_hi=24.0):
    """128 + 6*sum_k cos(2 pi (x cos th_k + y sin th_k)/lam_k + ph_k); I2 evaluated analytically at
    x - d, so that I2(x + d) = I1(x) exactly.  fp64, not quantised."""
    rng = np.random.default_rng(seed)
    th = rng.uniform(0.0, 2.0 * np.pi, n_waves)
    lam = rng.uniform(lam_lo, lam_hi, n_waves)
    ph = rng.uniform(0.0, 2.0 * np.pi, n_waves)
    x, y = _pixel_grid(width, height)

    def img(xs, ys):
        out = np.full_like(xs, 128.0)
        for k in range(n_waves):
            out += 6.0 * np.cos(2.0 * np.pi * (xs * math.cos(th[k]) + ys * math.sin(th[k])) / lam[k] + ph[k])
        return out

    return img(x, y), img(x - shift[0], y - shift[1])


def ramp_pair(width=64, height=64, grad=(0.8, 0.6), shift_along=0.25, c0=50.0):
    """I1 = c0 + a x + b y;  I2 = the same ramp shifted by d = shift_along*(a,b)/|(a,b)|."""
    a, b = grad
    n = math.hypot(a, b)
    d = (shift_along * a / n, shift_along * b / n)
    x, y = _pixel_grid(width, height)
    return c0 + a * x + b * y, c0 + a * (x - d[0]) + b * (y - d[1]), d
