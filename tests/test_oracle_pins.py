"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

Each test names the passage / reading it pins: PAPER.md:N = line of /root/reference/PAPER.md,
BASELINE.json:5 = the north_star's five self-checks, Dn = reading n of SURVEY.md 8(c) / DESIGN.md.
None of these tests touches the CUDA path.
"""
import math

import numpy as np
import pytest

from paper_1306_2461_b200 import synthetic as syn

BOX, GAUSS = 0, 1


def interior(a, m):
    return a[m:-m, m:-m]


# ------------------------------------------------------------------ BASELINE.json:5 check 1
def test_identical_images_give_exactly_zero_flow(oracle):
    """PAPER.md:61 'initial guess of zero displacement': It == 0 => p = q = 0 => du = dv = 0 bitwise."""
    c = syn.config1(96, 80)
    for levels, R, wt in ((1, 8, BOX), (2, 5, GAUSS)):
        r = oracle.solve(c.I1, c.I1, levels, R, 3, wt)
        assert np.all(r["u"] == 0.0) and np.all(r["v"] == 0.0)
        assert r["valid"].dtype == np.uint8 and r["valid"].max() == 1


# ------------------------------------------------------------------ BASELINE.json:5 check 2
def test_bandlimited_subpixel_shift_recovered_to_0p02_px(oracle):
    """Smooth band-limited image, known uniform shift (0.37,-0.21): max error <= 0.02 px
    (1 level, box R = 16, 6 iterations, margin 2R+4; SURVEY.md 8(c) pin table)."""
    I1, I2 = syn.bandlimited_pair(256, 256, (0.37, -0.21))
    r = oracle.solve(I1, I2, 1, 16, 6, BOX)
    m = 2 * 16 + 4
    eu = np.abs(interior(r["u"], m) - 0.37)
    ev = np.abs(interior(r["v"], m) + 0.21)
    assert max(eu.max(), ev.max()) <= 0.02
    assert abs(interior(r["u"], m).mean() - 0.37) < 5e-3
    assert abs(interior(r["v"], m).mean() + 0.21) < 5e-3


# ------------------------------------------------------------------ BASELINE.json:5 check 3
@pytest.mark.parametrize("eps", [1e-3, 1e-6])
def test_linear_ramp_closed_form_in_one_iteration(oracle, eps):
    """I1 = c0 + a x + b y, I2 = the ramp shifted by d || (a,b).  G is rank one, so the damped
    solve (D14) is the minimum-norm solve and one iteration gives u = d/(1+eps/2) in the interior;
    with eps -> 0 the ramp is 'solved exactly in one iteration'."""
    I1, I2, d = syn.ramp_pair(64, 64, (0.8, 0.6), 0.25)
    z = np.zeros_like(I1)
    u, v, *_ = oracle.iteration(I1, I2, z, z, 6, BOX, eps=eps)
    m = 8
    k = 1.0 / (1.0 + eps / 2.0)
    tol = 2e-15 / eps          # A*C - b^2 cancels to ~eps relative: rounding is amplified by 1/eps
    assert np.max(np.abs(interior(u, m) - d[0] * k)) < tol
    assert np.max(np.abs(interior(v, m) - d[1] * k)) < tol
    if eps == 1e-6:
        assert np.max(np.abs(interior(u, m) - d[0])) < 1e-6 * abs(d[0])


def test_ramp_three_iterations_converge_to_d(oracle):
    I1, I2, d = syn.ramp_pair(64, 64, (0.8, 0.6), 0.25)
    r = oracle.solve(I1, I2, 1, 6, 3, BOX)
    assert np.max(np.abs(interior(r["u"], 8) - d[0])) < 1e-9
    assert np.max(np.abs(interior(r["v"], 8) - d[1])) < 1e-9


# ------------------------------------------------------------------ BASELINE.json:5 check 4
def test_swapping_images_negates_flow(oracle):
    """D1 sign convention: I2(x+u) ~= I1(x); swapping the pair approximately negates the field."""
    I1, I2 = syn.bandlimited_pair(192, 192, (0.37, -0.21))
    a = oracle.solve(I1, I2, 1, 16, 6, BOX)
    b = oracle.solve(I2, I1, 1, 16, 6, BOX)
    m = 36
    assert np.max(np.abs(interior(a["u"] + b["u"], m))) <= 0.05
    assert np.max(np.abs(interior(a["v"] + b["v"], m))) <= 0.05
    assert interior(a["u"], m).mean() > 0.3 and interior(b["u"], m).mean() < -0.3


# ------------------------------------------------------------------ BASELINE.json:5 check 5
@pytest.mark.parametrize("wt,R", [(BOX, 3), (BOX, 8), (GAUSS, 6), (GAUSS, 12)])
def test_window_sums_match_brute_force_32x32(oracle, wt, R):
    """D11/D12: S(x,y) = sum w(dx) w(dy) f(x+dx,y+dy) over the in-image part of the window."""
    rng = np.random.default_rng(7)
    f = rng.standard_normal((32, 32))
    sigma = R / 3.0
    w = [1.0 if wt == BOX else math.exp(-(t * t) / (2.0 * sigma * sigma)) for t in range(-R, R + 1)]
    ref = np.zeros_like(f)
    for y in range(32):
        for x in range(32):
            s = 0.0
            for dy in range(-R, R + 1):
                for dx in range(-R, R + 1):
                    if 0 <= y + dy < 32 and 0 <= x + dx < 32:
                        s += w[dx + R] * w[dy + R] * f[y + dy, x + dx]
            ref[y, x] = s
    scale = np.abs(ref).max()
    assert np.max(np.abs(oracle.window_sum(f, R, wt) - ref)) <= 1e-12 * scale
    assert np.max(np.abs(oracle.window_sum(f, R, wt, direct=True) - ref)) <= 1e-12 * scale


def test_window_sum_nonsquare_and_weights(oracle):
    rng = np.random.default_rng(8)
    f = rng.standard_normal((20, 45))
    from scipy import ndimage
    R = 4
    ref = ndimage.uniform_filter(f, size=2 * R + 1, mode="constant") * (2 * R + 1) ** 2
    assert np.max(np.abs(oracle.window_sum(f, R, BOX) - ref)) < 1e-11
    # D11: Gaussian truncation radius R, sigma = R/3 (config 3: sigma 4 <=> R = 12, BASELINE.json:9)
    assert oracle.window_weight(0, 12, GAUSS) == 1.0
    assert abs(oracle.window_weight(4, 12, GAUSS) - math.exp(-0.5)) < 1e-15
    assert abs(oracle.window_weight(-12, 12, GAUSS) - math.exp(-4.5)) < 1e-15
    assert oracle.window_weight(5, 7, BOX) == 1.0


# ------------------------------------------------------------------ symmetries
def test_transpose_swaps_u_and_v(oracle):
    """x/y bookkeeping: transposing both images maps (u, v) -> (v^T, u^T)."""
    c = syn.config2(96, 64)
    a = oracle.solve(c.I1, c.I2, 2, 5, 3, BOX)
    b = oracle.solve(c.I1.T.copy(), c.I2.T.copy(), 2, 5, 3, BOX)
    assert np.max(np.abs(a["u"] - b["v"].T)) < 1e-10
    assert np.max(np.abs(a["v"] - b["u"].T)) < 1e-10
    assert np.array_equal(a["valid"], b["valid"].T)


def test_mirror_single_level(oracle):
    """Flip both images left-right (1 level only; even-pixel decimation breaks it for L > 1)."""
    c = syn.config2(96, 64)
    a = oracle.solve(c.I1, c.I2, 1, 5, 3, GAUSS)
    b = oracle.solve(c.I1[:, ::-1].copy(), c.I2[:, ::-1].copy(), 1, 5, 3, GAUSS)
    assert np.max(np.abs(a["u"] + b["u"][:, ::-1])) < 1e-10
    assert np.max(np.abs(a["v"] - b["v"][:, ::-1])) < 1e-10


def test_gain_offset_invariance(oracle):
    """D14: relative damping makes the solve invariant under I -> g I + c on both images."""
    c = syn.config1(80, 72)
    a = oracle.solve(c.I1, c.I2, 1, 6, 3, BOX)
    b = oracle.solve(3.5 * c.I1 + 40.0, 3.5 * c.I2 + 40.0, 1, 6, 3, BOX)
    assert np.max(np.abs(a["u"] - b["u"])) < 1e-9
    assert np.max(np.abs(a["v"] - b["v"])) < 1e-9


# ------------------------------------------------------------------ textbook reduction
def test_first_iteration_is_textbook_lucas_kanade(oracle):
    """1 level, 1 iteration, u = 0, eps -> 0: the classic Lucas-Kanade normal equations [28]
    (PAPER.md:57 'Lucas-Kanade family'), written independently with scipy.ndimage."""
    from scipy import ndimage
    I1, I2 = syn.bandlimited_pair(72, 60, (0.3, 0.2))
    R = 5
    z = np.zeros_like(I1)
    u, v, sums, valid, det = oracle.iteration(I1, I2, z, z, R, BOX, eps=0.0, max_step=1e9)
    P = np.pad(I1, 1, mode="edge")
    Ix = (P[1:-1, 2:] - P[1:-1, :-2]) / 2.0
    Iy = (P[2:, 1:-1] - P[:-2, 1:-1]) / 2.0
    It = I2 - I1
    box = lambda f: ndimage.uniform_filter(f, size=2 * R + 1, mode="constant") * (2 * R + 1) ** 2
    a, b, c, p, q = box(Ix * Ix), box(Ix * Iy), box(Iy * Iy), box(Ix * It), box(Iy * It)
    ref = np.empty(I1.shape + (2,))
    for y in range(I1.shape[0]):
        for x in range(I1.shape[1]):
            ref[y, x] = np.linalg.solve(np.array([[a[y, x], b[y, x]], [b[y, x], c[y, x]]]),
                                        -np.array([p[y, x], q[y, x]]))
    assert np.max(np.abs(u - ref[..., 0])) < 1e-9
    assert np.max(np.abs(v - ref[..., 1])) < 1e-9
    assert np.max(np.abs(sums[0] - a)) < 1e-9 * a.max() and np.max(np.abs(sums[4] - q)) < 1e-9 * np.abs(q).max()
    assert np.max(np.abs(det - (a * c - b * b))) < 1e-9 * det.max()
    assert valid.all()


def test_damped_solve_and_clamp_formula(oracle):
    """D14/D15 written out independently in NumPy for a non-zero current field (pins the
    -(p + a u + b v) right-hand side, the lam = eps tr/2 damping and the +-3 px clamp)."""
    from scipy import ndimage
    rng = np.random.default_rng(3)
    c = syn.config1(64, 56)
    I1 = c.I1.astype(np.float64)
    I2 = c.I2.astype(np.float64)
    u0 = rng.uniform(-1.5, 1.5, I1.shape)
    v0 = rng.uniform(-1.5, 1.5, I1.shape)
    R, eps = 4, 1e-3
    u, v, sums, valid, det = oracle.iteration(I1, I2, u0, v0, R, BOX, eps=eps, max_step=3.0)
    yy, xx = np.mgrid[0:I1.shape[0], 0:I1.shape[1]].astype(np.float64)
    I2w = ndimage.map_coordinates(I2, [yy + v0, xx + u0], order=1, mode="nearest")
    P = np.pad(I1, 1, mode="edge")
    Ix = (P[1:-1, 2:] - P[1:-1, :-2]) / 2.0
    Iy = (P[2:, 1:-1] - P[:-2, 1:-1]) / 2.0
    It = I2w - I1 - Ix * u0 - Iy * v0
    def box(f):       # sum of shifted zero-padded copies (no running sums: exact zeros stay zero)
        Z = np.pad(f, R)
        return sum(Z[R + dy:R + dy + f.shape[0], R + dx:R + dx + f.shape[1]]
                   for dy in range(-R, R + 1) for dx in range(-R, R + 1))
    a, b, cc, p, q = box(Ix * Ix), box(Ix * Iy), box(Iy * Iy), box(Ix * It), box(Iy * It)
    tr = a + cc
    ok = tr > 0
    lam = eps * tr / 2
    G = np.stack([np.stack([a + lam, b], -1), np.stack([b, cc + lam], -1)], -2)
    rhs = -np.stack([p + a * u0 + b * v0, q + b * u0 + cc * v0], -1)
    du = np.zeros(I1.shape + (2,))
    du[ok] = np.linalg.solve(G[ok], rhs[ok][..., None])[..., 0]
    du = np.clip(du, -3.0, 3.0)
    assert np.max(np.abs((u - u0)[ok] - du[ok][..., 0])) < 1e-8
    assert np.max(np.abs((v - v0)[ok] - du[ok][..., 1])) < 1e-8
    assert np.abs(du).max() == 3.0          # the clamp is exercised by this input
    assert np.array_equal(valid.astype(bool), sums[0] + sums[2] > 0)
    assert np.all((u - u0)[valid == 0] == 0)


def test_warp_matches_library_bilinear(oracle):
    """D8: bilinear with clamped indices == scipy map_coordinates(order=1, mode='nearest')."""
    from scipy import ndimage
    rng = np.random.default_rng(5)
    I2 = rng.uniform(0, 255, (40, 52))
    u = rng.uniform(-6, 6, I2.shape)
    v = rng.uniform(-6, 6, I2.shape)
    yy, xx = np.mgrid[0:40, 0:52].astype(np.float64)
    ref = ndimage.map_coordinates(I2, [yy + v, xx + u], order=1, mode="nearest")
    assert np.max(np.abs(oracle.warp(I2, u, v) - ref)) < 1e-10
    # integer displacements are exact (bilinear is exact at integer offsets)
    ui = np.full(I2.shape, 2.0)
    vi = np.full(I2.shape, -1.0)
    w = oracle.warp(I2, ui, vi)
    assert np.array_equal(w[1:, :-2], I2[:-1, 2:])


def test_gradients_central_difference_with_clamp(oracle):
    """D9: [-1/2, 0, 1/2] on I1, clamp-to-edge."""
    rng = np.random.default_rng(6)
    I = rng.uniform(0, 255, (17, 23))
    Ix, Iy = oracle.gradients(I)
    gy, gx = np.gradient(I)                      # central differences in the interior
    assert np.max(np.abs(Ix[:, 1:-1] - gx[:, 1:-1])) < 1e-12
    assert np.max(np.abs(Iy[1:-1, :] - gy[1:-1, :])) < 1e-12
    assert np.allclose(Ix[:, 0], (I[:, 1] - I[:, 0]) / 2) and np.allclose(Ix[:, -1], (I[:, -1] - I[:, -2]) / 2)
    assert np.allclose(Iy[0, :], (I[1, :] - I[0, :]) / 2) and np.allclose(Iy[-1, :], (I[-1, :] - I[-2, :]) / 2)
    # x runs along columns: a pure x-ramp has Iy == 0
    ramp = np.tile(np.arange(23.0), (17, 1))
    Ix, Iy = oracle.gradients(ramp)
    assert np.all(Iy == 0) and np.all(Ix[:, 1:-1] == 1.0)


def test_integer_shift_converges(oracle):
    """Particles re-rendered at an integer shift (2,-1): bilinear is exact there, so the fixed point
    is the shift itself on well-conditioned pixels."""
    rng = np.random.default_rng(9)
    xp, yp, amp = syn.seed_particles(rng, 128, 128, 0.03, 150, 255)
    I1 = syn.render_particles(xp, yp, amp, 1.2, 128, 128)
    I2 = syn.render_particles(xp + 2.0, yp - 1.0, amp, 1.2, 128, 128)
    r = oracle.solve(I1, I2, 2, 8, 8, BOX)
    S = r["det"] > 1e-3 * r["det"].max()
    S[:20] = S[-20:] = False
    S[:, :20] = S[:, -20:] = False
    assert np.median(np.abs(r["u"][S] - 2.0)) < 1e-4
    assert np.max(np.abs(r["u"][S] - 2.0)) < 5e-3 and np.max(np.abs(r["v"][S] + 1.0)) < 5e-3


# ------------------------------------------------------------------ pyramid / hand-down
def test_pyramid_filter_exact_on_constants_and_ramps(oracle):
    """D4/D5: [1 4 6 4 1]/16, even samples, clamp: constants stay constant (borders included);
    an interior ramp maps to a ramp with doubled slope per coarse pixel; sizes (W+1)/2."""
    c = np.full((21, 30), 7.25)
    d = oracle.downsample(c)
    assert d.shape == (11, 15) and np.all(d == 7.25)
    y, x = np.mgrid[0:40, 0:64].astype(np.float64)
    ramp = 3.0 + 0.5 * x - 0.25 * y
    d = oracle.downsample(ramp)
    Y, X = np.mgrid[0:20, 0:32].astype(np.float64)
    assert np.max(np.abs(d[1:-1, 1:-1] - (3.0 + 1.0 * X - 0.5 * Y)[1:-1, 1:-1])) < 1e-12
    # impulse response = outer product of the binomial taps at even phase
    imp = np.zeros((16, 16))
    imp[8, 8] = 256.0
    d = oracle.downsample(imp)
    assert np.array_equal(d[3:6, 3:6], np.outer([1, 6, 1], [1, 6, 1]).astype(float))
    imp = np.zeros((16, 16))
    imp[8, 9] = 256.0
    assert np.array_equal(oracle.downsample(imp)[3:6, 4:6], np.outer([1, 6, 1], [4, 4]).astype(float))


def test_upsample_doubles_and_reproduces_linear_fields(oracle):
    """D6: fine = 2 * bilinear(coarse; x/2, y/2)."""
    c = np.full((9, 12), 1.5)
    f = oracle.upsample_flow(c, 24, 18)
    assert np.all(f == 3.0)
    f = oracle.upsample_flow(c, 23, 17)           # odd fine sizes: (23+1)/2 = 12, (17+1)/2 = 9
    assert f.shape == (17, 23) and np.all(f == 3.0)
    Y, X = np.mgrid[0:10, 0:16].astype(np.float64)
    lin = 0.3 * X - 0.2 * Y + 1.0
    f = oracle.upsample_flow(lin, 32, 20)
    y, x = np.mgrid[0:20, 0:32].astype(np.float64)
    ref = 2.0 * (0.3 * x / 2 - 0.2 * y / 2 + 1.0)
    assert np.max(np.abs(f[:-1, :-1] - ref[:-1, :-1])) < 1e-12


def test_eq1_more_levels_needed_for_large_displacements(oracle):
    """eq. 1: (dx)max / 2^(n_lev-1) < 3 px.  A smooth field with ~10 px maximum
    needs n_lev >= 3: it fails with 1 and 2 levels and is recovered with 3."""
    rng = np.random.default_rng(123)
    W = H = 320
    d = syn.field_random_smooth(rng, W, H, 48.0, 6.0)
    I1, I2, tu, tv = syn._pair_from_field(rng, W, H, 0.03, 1.5, 150.0, 255.0, d)
    dmax = max(np.abs(tu).max(), np.abs(tv).max())
    assert dmax / 2 ** (3 - 1) < 3.0 <= dmax / 2 ** (2 - 1)
    m = 40
    err = {}
    for L in (1, 2, 3):
        r = oracle.solve(I1, I2, L, 10, 8, BOX)
        e = np.hypot(r["u"] - tu, r["v"] - tv)
        err[L] = math.sqrt(np.mean(interior(e, m) ** 2))
    assert err[1] > 3.0 and err[2] > 1.0 and err[3] < 0.4


def test_error_non_increasing_in_iterations_and_fixed_point(oracle):
    """Table 1 trend: error falls with n_iter; 'n_iter >= 10 is seldom needed'
    (PAPER.md:91): iterations 10 -> 14 move the field by < 1e-3 px on well-conditioned pixels."""
    c = syn.config2(256, 256)
    I1, I2 = c.I1.astype(np.float64), c.I2.astype(np.float64)
    m = 24
    errs, fields = [], {}
    for n in (1, 2, 4, 10, 14):
        r = oracle.solve(I1, I2, 2, 7, n, BOX)
        e = np.hypot(r["u"] - c.truth_u, r["v"] - c.truth_v)
        errs.append(math.sqrt(np.mean(interior(e, m) ** 2)))
        fields[n] = r
    assert errs[0] > errs[1] > errs[2] >= errs[3] - 1e-3
    S = fields[10]["det"] > 1e-3 * fields[10]["det"].max()
    assert np.max(np.abs(fields[10]["u"] - fields[14]["u"])[S]) < 1e-2
    assert math.sqrt(np.mean((fields[10]["u"] - fields[14]["u"])[S] ** 2)) < 1e-3


def test_levels_argument_counts_base_image(oracle):
    """D3: levels >= 1 includes the base; coarsest level smaller than the window is rejected."""
    c = syn.config1(64, 64)
    with pytest.raises(ValueError):
        oracle.solve(c.I1, c.I2, 3, 8, 1, BOX)        # 16x16 < 17
    r = oracle.solve(c.I1, c.I2, 2, 8, 1, BOX, return_levels=True)
    assert r["level_u"][1].shape == (32, 32) and r["level_u"][0].shape == (64, 64)
    assert np.array_equal(r["level_u"][0], r["u"])


def test_solve_equals_stepwise_composition(oracle):
    """oracle_solve is exactly pyramid -> (upsample -> iterations) per level, coarse to fine
    (PAPER.md:61), composed here from the primitives."""
    c = syn.config2(96, 80)
    I1, I2 = c.I1.astype(np.float64), c.I2.astype(np.float64)
    r = oracle.solve(I1, I2, 2, 5, 2, GAUSS)
    P1, P2 = oracle.downsample(I1), oracle.downsample(I2)
    u = np.zeros_like(P1)
    v = np.zeros_like(P1)
    for _ in range(2):
        u, v, *_ = oracle.iteration(P1, P2, u, v, 5, GAUSS)
    u, v = oracle.upsample_flow(u, 96, 80), oracle.upsample_flow(v, 96, 80)
    for _ in range(2):
        u, v, s, valid, det = oracle.iteration(I1, I2, u, v, 5, GAUSS)
    assert np.array_equal(u, r["u"]) and np.array_equal(v, r["v"])
    assert np.array_equal(valid, r["valid"]) and np.array_equal(det, r["det"])
    # direct (definition) window sums give the same field to rounding
    rd = oracle.solve(I1, I2, 2, 5, 2, GAUSS, direct=True)
    assert np.max(np.abs(rd["u"] - r["u"])) < 1e-9


def test_empty_windows_are_invalid_and_keep_zero_flow(oracle):
    """D14: valid <=> tr(G) > 0; texture-less windows get no update."""
    I1 = np.zeros((64, 64))
    I2 = np.zeros((64, 64))
    I1[30:34, 30:34] = 100.0
    I2[30:34, 31:35] = 100.0
    r = oracle.solve(I1, I2, 1, 4, 2, BOX)
    assert r["valid"][32, 32] == 1 and r["valid"][5, 5] == 0 and r["valid"][32, 50] == 0
    assert np.all(r["u"][r["valid"] == 0] == 0.0)
    # central differences of the 4x4 block are non-zero on a plus-shaped support inside rows/cols
    # 29..34 without its four corner pixels; dilated by the 9x9 window: 14x14 minus the 4 corners
    assert r["valid"].sum() == (6 + 8) ** 2 - 4


# ---------------------------------------------------------------------------- eq. 2 (NEXT item f1)
def test_equalise_matches_library_box_statistics_in_interior(oracle):
    """eq. 2: (I - local mean) / local std over an 11x11 box; in the interior the
    local moments are what scipy.ndimage.uniform_filter computes."""
    from scipy.ndimage import uniform_filter
    rng = np.random.default_rng(3)
    I = rng.integers(0, 256, (48, 64)).astype(np.float64)
    r = 5
    out = oracle.equalise(I, r)
    m = uniform_filter(I, 2 * r + 1, mode="constant")
    m2 = uniform_filter(I * I, 2 * r + 1, mode="constant")
    ref = (I - m) / np.sqrt(m2 - m * m)
    sl = (slice(r, -r), slice(r, -r))
    assert np.max(np.abs(out[sl] - ref[sl])) < 1e-10


def test_equalise_borders_use_the_in_image_part_of_the_box(oracle):
    rng = np.random.default_rng(4)
    I = rng.integers(0, 4096, (20, 23)).astype(np.float64)
    r = 3
    out = oracle.equalise(I, r)
    for (x, y) in ((0, 0), (22, 0), (0, 19), (22, 19), (1, 10), (11, 18)):
        win = I[max(0, y - r):y + r + 1, max(0, x - r):x + r + 1]
        ref = (I[y, x] - win.mean()) / win.std()
        assert abs(out[y, x] - ref) < 1e-10, (x, y)


def test_equalise_invariances_and_flat_guard(oracle):
    rng = np.random.default_rng(5)
    I = rng.integers(0, 256, (40, 40)).astype(np.float64)
    a = oracle.equalise(I, 5)
    b = oracle.equalise(3.5 * I + 17.0, 5)                    # illumination gain and offset drop out
    assert np.max(np.abs(a - b)) < 1e-9
    assert np.all(oracle.equalise(np.full((30, 30), 99.0), 5) == 0.0)     # flat -> 0, never NaN
    flat = I.copy()
    flat[10:30, 10:30] = 50.0
    out = oracle.equalise(flat, 5)
    assert np.isfinite(out).all() and np.all(out[15:25, 15:25] == 0.0)


def test_flow_is_unchanged_by_equalisation_of_an_unevenly_lit_pair(oracle):
    """Purpose of eq. 2: 'eliminate the influence of illumination inhomogeneities'.  A smooth
    multiplicative illumination change between the frames biases the raw solve; after equalisation the
    bias is gone (error vs the known shift drops)."""
    d = (0.37, -0.21)
    I1, I2 = syn.bandlimited_pair(192, 160, shift=d)
    yy, xx = np.mgrid[0:160, 0:192]
    lit = 1.0 + 0.4 * xx / 192.0 + 0.2 * yy / 160.0
    raw = oracle.solve(I1, I2 * lit, 1, 10, 4, BOX)
    eq = oracle.solve(oracle.equalise(I1, 5), oracle.equalise(I2 * lit, 5), 1, 10, 4, BOX)
    m = (slice(24, -24), slice(24, -24))
    err_raw = np.sqrt(np.mean((raw["u"][m] - d[0]) ** 2 + (raw["v"][m] - d[1]) ** 2))
    err_eq = np.sqrt(np.mean((eq["u"][m] - d[0]) ** 2 + (eq["v"][m] - d[1]) ** 2))
    assert err_eq < 0.5 * err_raw and err_eq < 0.05


# ---------------------------------------------------------------------------- eq. 3 (NEXT item f3)
def test_bubble_surface_definition_on_hand_worked_fields(oracle):
    """eq. 3: share of available vectors with v_x <= T_v, T_v = mid-range of the mean field."""
    mean = np.array([[-1.0, 0.0, 1.0], [2.0, 3.0, 7.0]])
    assert oracle.bubble_threshold(mean) == 3.0                       # (min -1 + max 7) / 2
    vx = np.array([[3.0, 3.5, -2.0], [2.9, 8.0, 3.0]])
    assert oracle.bubble_counts(vx, 3.0) == (4, 6)                    # 3.0, -2.0, 2.9, 3.0 (<= is inclusive)
    valid = np.array([[1, 1, 0], [1, 0, 1]], dtype=np.uint8)
    assert oracle.bubble_counts(vx, 3.0, valid) == (3, 4)             # only available vectors count
    assert oracle.bubble_threshold(mean, valid) == 3.0
    # a linear profile v_x = x over [0, W-1]: T_v = (W-1)/2 and exactly the lower half (inclusive) is below
    W = 11
    lin = np.tile(np.arange(W, dtype=np.float64), (4, 1))
    T = oracle.bubble_threshold(lin)
    assert T == 5.0 and oracle.bubble_counts(lin, T) == (4 * 6, 4 * W)


def test_bubble_surface_of_the_backward_step_like_truth_field(oracle):
    """The config-3 ground-truth field has a -1 px recirculation region upstream of x = 0.7 W below the shear
    layer: its bubble surface must be the area share of that region (cross-check of the definition with
    a thresholded-area count done independently with NumPy)."""
    c = syn.config3(320, 256)
    T = oracle.bubble_threshold(c.truth_u)
    below, total = oracle.bubble_counts(c.truth_u, T)
    assert total == 320 * 256 and below == int(np.count_nonzero(c.truth_u <= T))
    assert 0.15 < below / total < 0.45


# ---------------------------------------------------------------------------- masks (NEXT item f4)
# PAPER.md:175 "using masks to avoid computations over obstacles or side walls"; readings M1-M5
# (oracle/optflow_oracle.c above oracle_mask_downsample).
def _blob_mask(H, W):
    m = np.ones((H, W), dtype=np.uint8)
    m[20:44, 10:40] = 0          # an obstacle
    m[:, :3] = 0                 # a side wall
    m[50, 60] = 0                # a single dead pixel
    return m


def test_mask_of_ones_is_no_mask_bit_for_bit(oracle):
    c = syn.config2(96, 80)
    a = oracle.solve(c.I1, c.I2, 2, 5, 2, GAUSS)
    b = oracle.solve(c.I1, c.I2, 2, 5, 2, GAUSS, mask=np.ones((80, 96), dtype=np.uint8))
    for k in ("u", "v", "valid", "det"):
        assert np.array_equal(a[k], b[k])


def test_masked_pixels_carry_no_vector_at_any_level(oracle):
    """M3: u = v = 0, valid = 0, det = 0 over the obstacle, at every level (mask pyramid M4)."""
    c = syn.config2(96, 80)
    m0 = _blob_mask(80, 96)
    r = oracle.solve(c.I1, c.I2, 3, 4, 2, BOX, mask=m0, return_levels=True)
    m = m0
    for l in range(3):
        assert np.all(r["level_u"][l][m == 0] == 0.0) and np.all(r["level_v"][l][m == 0] == 0.0)
        assert np.any(r["level_u"][l][m == 1] != 0.0)
        m = oracle.mask_downsample(m)
    assert np.all(r["valid"][m0 == 0] == 0) and np.all(r["det"][m0 == 0] == 0.0)
    assert r["valid"][m0 == 1].min() == 1          # textured fluid pixels stay valid next to the obstacle


def test_mask_pyramid_is_the_or_of_the_children(oracle):
    """M4 against a plain Python loop, odd sizes (last column / row has fewer children)."""
    rng = np.random.default_rng(5)
    m = (rng.random((13, 17)) < 0.3).astype(np.uint8)
    got = oracle.mask_downsample(m)
    assert got.shape == (7, 9)
    for Y in range(7):
        for X in range(9):
            kids = [m[y, x] for y in (2 * Y, 2 * Y + 1) for x in (2 * X, 2 * X + 1) if y < 13 and x < 17]
            assert got[Y, X] == (1 if any(kids) else 0)
    assert oracle.mask_downsample(np.zeros((4, 6), np.uint8)).max() == 0
    assert oracle.mask_downsample(np.ones((5, 5), np.uint8)).min() == 1


@pytest.mark.parametrize("wt,R", [(BOX, 3), (GAUSS, 6)])
def test_masked_sums_are_brute_force_sums_of_mask_times_product(oracle, wt, R):
    """M2: a, b, c, p, q = sum over the window of w * mask * product, summed pixel by pixel here from
    the oracle's own warp / gradient primitives (32x32, zero extension outside the image)."""
    rng = np.random.default_rng(9)
    I1 = rng.random((32, 32)) * 100.0
    I2 = rng.random((32, 32)) * 100.0
    u = rng.normal(0.0, 0.7, (32, 32))
    v = rng.normal(0.0, 0.7, (32, 32))
    m = (rng.random((32, 32)) < 0.6).astype(np.uint8)
    _, _, sums, valid, _ = oracle.iteration(I1, I2, u, v, R, wt, mask=m)
    Ix, Iy = oracle.gradients(I1)
    It = oracle.warp(I2, u, v) - I1 - Ix * u - Iy * v
    prods = [Ix * Ix, Ix * Iy, Iy * Iy, Ix * It, Iy * It]
    w = [oracle.window_weight(t, R, wt) for t in range(-R, R + 1)]
    for (y, x) in [(0, 0), (5, 17), (31, 31), (16, 2), (30, 9)]:
        for f in range(5):
            acc = 0.0
            for dy in range(-R, R + 1):
                for dx in range(-R, R + 1):
                    yy, xx = y + dy, x + dx
                    if 0 <= yy < 32 and 0 <= xx < 32 and m[yy, xx]:
                        acc += w[dy + R] * w[dx + R] * prods[f][yy, xx]
            assert abs(sums[f, y, x] - acc) <= 1e-9 * max(1.0, abs(acc))
    assert np.all(valid[m == 0] == 0)


def test_ramp_is_still_solved_in_one_iteration_beside_an_obstacle(oracle):
    """Every pixel of a linear ramp satisfies the same linear equation, so dropping any subset of them
    from the window (M2) leaves the closed form u = d/(1+eps/2) at every fluid pixel whose window
    still holds a fluid pixel.  A mask applied to G but not to the right-hand side (or the reverse)
    fails this."""
    I1, I2, d = syn.ramp_pair(64, 64, (0.8, 0.6), 0.25)
    m = np.ones((64, 64), dtype=np.uint8)
    m[24:40, 20:50] = 0
    m[10, 10] = 0
    z = np.zeros_like(I1)
    eps = 1e-3
    u, v, _, valid, _ = oracle.iteration(I1, I2, z, z, 6, BOX, eps=eps, mask=m)
    k = 1.0 / (1.0 + eps / 2.0)
    fluid = interior(m, 8) == 1
    assert np.max(np.abs(interior(u, 8)[fluid] - d[0] * k)) < 2e-12
    assert np.max(np.abs(interior(v, 8)[fluid] - d[1] * k)) < 2e-12
    assert np.all(u[m == 0] == 0.0) and np.all(valid[m == 0] == 0) and np.all(valid[m == 1] == 1)


def test_image_content_deep_under_the_mask_reaches_no_fluid_vector(oracle):
    """M2 + M5 at one level: a fluid vector depends on the images only through fluid pixels of its
    window, their gradient stencils (1 px) and their warped samples (|u| <= iterations * 3 px, D15).
    Scribbling over the obstacle's deep interior leaves every fluid vector bit-identical with the mask
    and changes vectors near the obstacle without it."""
    c = syn.config1(96, 96)
    I1, I2 = c.I1.astype(np.float64), c.I2.astype(np.float64)
    m = np.ones((96, 96), dtype=np.uint8)
    m[20:76, 30:70] = 0
    J1, J2 = I1.copy(), I2.copy()
    rng = np.random.default_rng(3)
    J1[30:66, 40:60] = rng.random((36, 20)) * 255.0      # >= 10 px from any fluid pixel
    J2[30:66, 40:60] = rng.random((36, 20)) * 255.0
    a = oracle.solve(I1, I2, 1, 8, 2, BOX, mask=m)
    b = oracle.solve(J1, J2, 1, 8, 2, BOX, mask=m)
    assert np.array_equal(a["u"], b["u"]) and np.array_equal(a["v"], b["v"]) and np.array_equal(a["valid"], b["valid"])
    a0 = oracle.solve(I1, I2, 1, 8, 2, BOX)
    b0 = oracle.solve(J1, J2, 1, 8, 2, BOX)
    assert np.max(np.abs(a0["u"] - b0["u"])[m == 1]) > 1e-3


def test_masked_solve_equals_stepwise_composition(oracle):
    """Two levels with a mask: pyramid of images and of masks, masked iterations, hand-down, zero over
    the obstacle (M3), masked iterations -- composed from the primitives."""
    c = syn.config2(96, 80)
    I1, I2 = c.I1.astype(np.float64), c.I2.astype(np.float64)
    m0 = _blob_mask(80, 96)
    m1 = oracle.mask_downsample(m0)
    r = oracle.solve(I1, I2, 2, 5, 2, GAUSS, mask=m0)
    P1, P2 = oracle.downsample(I1), oracle.downsample(I2)
    u = np.zeros_like(P1)
    v = np.zeros_like(P1)
    for _ in range(2):
        u, v, *_ = oracle.iteration(P1, P2, u, v, 5, GAUSS, mask=m1)
    u, v = oracle.upsample_flow(u, 96, 80), oracle.upsample_flow(v, 96, 80)
    u[m0 == 0] = 0.0
    v[m0 == 0] = 0.0
    for _ in range(2):
        u, v, s, valid, det = oracle.iteration(I1, I2, u, v, 5, GAUSS, mask=m0)
    assert np.array_equal(u, r["u"]) and np.array_equal(v, r["v"]) and np.array_equal(valid, r["valid"])


# ------------------------------------------------------------------ D9 (what of_set_hoist relies on)
@pytest.mark.parametrize("wt,R", [(BOX, 4), (GAUSS, 6)])
def test_matrix_sums_do_not_depend_on_the_displacement(oracle, wt, R):
    """Reading D9: the gradients are taken on the unwarped I1, so the window sums a, b, c of IxIx, IxIy, IyIy (the 2x2
    matrix of the local least-squares problem) are the same for every displacement field, i.e. in every
    iteration of a level; only the sums of IxIt, IyIt follow the warp.  Pinned on the oracle itself: a, b, c with a zero
    field equal a, b, c with a rough random field bit for bit (also with an obstacle mask), p and q do not, and a, b, c
    equal the window sums of the gradient products formed here from np.gradient-style differences."""
    c = syn.config1(72, 56)
    I1, I2 = c.I1.astype(np.float64), c.I2.astype(np.float64)
    rng = np.random.default_rng(7)
    z = np.zeros_like(I1)
    u, v = rng.uniform(-3, 3, I1.shape), rng.uniform(-3, 3, I1.shape)
    mask = np.ones(I1.shape, np.uint8)
    mask[20:30, 10:40] = 0
    for m in (None, mask):
        s0 = oracle.iteration(I1, I2, z, z, R, wt, mask=m)[2]
        s1 = oracle.iteration(I1, I2, u, v, R, wt, mask=m)[2]
        assert np.array_equal(s0[:3], s1[:3])
        assert not np.array_equal(s0[3], s1[3]) and not np.array_equal(s0[4], s1[4])
    # independent formation of a, b, c: central differences with clamped borders, then the oracle's own window sum
    P = np.pad(I1, 1, mode="edge")
    Ix, Iy = 0.5 * (P[1:-1, 2:] - P[1:-1, :-2]), 0.5 * (P[2:, 1:-1] - P[:-2, 1:-1])
    s0 = oracle.iteration(I1, I2, u, v, R, wt)[2]
    for k, f in enumerate((Ix * Ix, Ix * Iy, Iy * Iy)):
        assert np.allclose(s0[k], oracle.window_sum(f, R, wt, direct=True), rtol=1e-12, atol=1e-9)


def test_backward_step_mask_recipe():
    m = syn.mask_backward_step(1280, 1024)
    assert m.dtype == np.uint8 and m.shape == (1024, 1280)
    assert 0.13 < 1.0 - m.mean() < 0.17
    assert m[512, 640] == 1 and m[0, 0] == 0 and m[1000, 100] == 0
