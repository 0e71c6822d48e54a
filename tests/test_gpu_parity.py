"""GPU parity: the CUDA path (through the C-ABI binding) against the fp64 oracle, element by element,
on the same seeded inputs.  Run on the B200 box with `pytest -m gpu`.

Tolerance (BASELINE.json:5, D23): max <= 1e-3 px, RMS <= 1e-4 px on pixels whose determinant exceeds
1e-3 of the field maximum; identical validity masks everywhere.
"""
import numpy as np
import pytest

from paper_1306_2461_b200 import synthetic as syn
from parity import assert_parity, compare_flow

pytestmark = pytest.mark.gpu

BOX, GAUSS = 0, 1


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    return t


@pytest.fixture(scope="module")
def B():
    from paper_1306_2461_b200 import binding
    binding.lib()          # fails loudly if liboptflow.so is missing
    return binding


def gpu_solve(torch, B, I1, I2, levels, R, iters, wt, as_float=False, graph=True):
    H, W = I1.shape
    with B.OpticalFlow(W, H, levels, R, iters, wt) as of:
        of.set_graph(graph)
        if as_float:
            d1 = torch.from_numpy(I1.astype(np.float32)).cuda()
            d2 = torch.from_numpy(I2.astype(np.float32)).cuda()
        elif I1.dtype == np.uint16:
            d1 = torch.from_numpy(I1.view(np.int16)).cuda()
            d2 = torch.from_numpy(I2.view(np.int16)).cuda()
        else:
            d1 = torch.from_numpy(I1).cuda()
            d2 = torch.from_numpy(I2).cuda()
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            u, v = of.compute(d1, d2)
            m = of.validity()
        s.synchronize()
        return u.cpu().numpy(), v.cpu().numpy(), m.cpu().numpy(), of.last_launch_count()


def run_case(torch, B, oracle, c, as_float=False):
    ref = oracle.solve(c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type)
    u, v, m, n = gpu_solve(torch, B, c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type, as_float)
    st = assert_parity(u, v, m, ref, c.name)
    print(c.name, c.width, c.height, st, "launches", n)
    return st


# ---------------------------------------------------------------------------- the five configs
def test_config1_256_uniform_shift(torch, B, oracle):
    """BASELINE.json:7: fp32-from-uint8, 1 level, box R 8, 4 iterations; expected flow (1.3,-0.7)."""
    c = syn.config1()
    run_case(torch, B, oracle, c, as_float=True)
    u, v, m, _ = gpu_solve(torch, B, c.I1, c.I2, 1, 8, 4, BOX, as_float=True)
    assert abs(np.median(u) - 1.3) < 0.05 and abs(np.median(v) + 0.7) < 0.05


def test_config2_small_ragged(torch, B, oracle):
    """config-2 statistics at a size that is no multiple of any tile (several tiles + ragged tail)."""
    run_case(torch, B, oracle, syn.config2(330, 214))


def test_config2_1024_vortex(torch, B, oracle):
    run_case(torch, B, oracle, syn.config2())


def test_config3_small_gaussian(torch, B, oracle):
    run_case(torch, B, oracle, syn.config3(400, 296))


def test_config3_1280x1024_gaussian(torch, B, oracle):
    """BASELINE.json:9 -- the bench workload, in the launch configuration bench.py times."""
    run_case(torch, B, oracle, syn.config3())


def test_config4_small_u16(torch, B, oracle):
    run_case(torch, B, oracle, syn.config4(400, 360, filt_sigma=48.0))


def test_config4_2048_u16(torch, B, oracle):
    run_case(torch, B, oracle, syn.config4())


def test_config5_streaming(torch, B, oracle):
    """BASELINE.json:11: consecutive frames through the pinned double-buffered pipeline.  Every field
    must equal (bitwise) the non-streaming call on the same pair; sampled pairs are checked against
    the oracle."""
    import os
    n_frames = int(os.environ.get("OF_TEST_STREAM_FRAMES", "256"))
    st = syn.Config5Stream(n_frames)
    W, H = st.width, st.height
    sample = sorted({0, (n_frames - 1) // 2, n_frames - 2})
    frames_kept = {}
    fields = {}
    with B.OpticalFlow(*st.create_args) as of, B.OpticalFlow(*st.create_args) as of2:
        of.stream_open(B.OF_DTYPE_U8, B.OF_STREAM_CONSECUTIVE, True)
        prev = None
        submitted = 0
        for k, f in enumerate(st.frames()):
            slot = of.stream_acquire()
            slot[...] = f
            of.stream_submit()
            submitted += 1
            if k >= 1:
                if (k - 1) in sample:
                    frames_kept[k - 1] = (prev.copy(), f.copy())
                # stay one field behind so upload k+1 overlaps solve k
                if k >= 2:
                    idx, u, v = of.stream_result()
                    assert idx == k - 2
                    if idx in sample or idx % 37 == 0:
                        fields[idx] = (u.copy(), v.copy())
            prev = f
        idx, u, v = of.stream_result()
        assert idx == n_frames - 2
        fields[idx] = (u.copy(), v.copy())
        of.stream_close()
        # non-streaming call on the kept pairs must agree bitwise; oracle parity on them
        for idx, (f1, f2) in frames_kept.items():
            d1, d2 = torch.from_numpy(f1).cuda(), torch.from_numpy(f2).cuda()
            u2, v2 = of2.compute(d1, d2)
            m2 = of2.validity()
            torch.cuda.synchronize()
            assert np.array_equal(u2.cpu().numpy(), fields[idx][0]), idx
            assert np.array_equal(v2.cpu().numpy(), fields[idx][1]), idx
            ref = oracle.solve(f1, f2, st.levels, st.window_radius, st.iterations, st.window_type)
            print("config5 pair", idx, assert_parity(fields[idx][0], fields[idx][1], m2.cpu().numpy(), ref, "config5"))
    # the convected shear layer moves right at ~2+-3 px/frame: sanity on the sign of the field
    u_last = fields[n_frames - 2][0]
    assert u_last[: H // 4].mean() > 3.0 and u_last[-H // 4:].mean() < 0.5


def test_stream_pairs_mode(torch, B, oracle):
    c = syn.config2(320, 256)
    ref = oracle.solve(c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type)
    with B.OpticalFlow(*c.create_args) as of:
        of.stream_open(B.OF_DTYPE_U8, B.OF_STREAM_PAIRS, True)
        for rep in range(5):
            slot = of.stream_acquire()
            slot[0] = c.I1
            slot[1] = c.I2
            of.stream_submit()
            idx, u, v = of.stream_result()
            assert idx == rep
            assert_parity(u, v, None, ref, "pairs-mode")
        # three fields may be in flight (include/optflow.h); a fourth uncollected one is refused, and the three come out right and in order
        for rep in range(3):
            slot = of.stream_acquire(); slot[0] = c.I1; slot[1] = c.I2; of.stream_submit()
        of.stream_acquire()
        with pytest.raises(B.OptflowError):
            of.stream_submit()
        held = []
        for rep in range(3):
            idx, u, v = of.stream_result()
            assert idx == 5 + rep
            held.append((u, v))
            assert_parity(u, v, None, ref, "pairs-mode, three in flight")
        # a returned field stays valid until the second-next of_stream_result call: the last two are still intact
        assert np.array_equal(held[1][0], held[2][0]) and np.array_equal(held[1][1], held[2][1])
        of.stream_submit()                                   # the slot acquired above
        idx, u, v = of.stream_result()
        assert idx == 8
        of.stream_close()


# ---------------------------------------------------------------------------- single steps
def test_pyramid_step_matches_oracle(torch, B, oracle):
    rng = np.random.default_rng(1)
    for (H, W) in ((64, 64), (37, 131), (5, 9), (1024, 1280)):
        img = rng.integers(0, 4096, (H, W)).astype(np.float32)
        ref = oracle.downsample(img)
        out = B.pyramid_down(torch.from_numpy(img).cuda()).cpu().numpy()
        assert out.shape == ref.shape
        assert np.max(np.abs(out - ref)) <= 1e-6 * 4096, (H, W)
        # integers < 2^12 with dyadic taps: one level is exact in fp32
        assert np.array_equal(out.astype(np.float64), ref), (H, W)


def test_upsample_step_matches_oracle(torch, B, oracle):
    rng = np.random.default_rng(2)
    for (H, W) in ((64, 64), (37, 131), (7, 10)):
        hc, wc = (H + 1) // 2, (W + 1) // 2
        uc = rng.uniform(-8, 8, (hc, wc)).astype(np.float32)
        vc = rng.uniform(-8, 8, (hc, wc)).astype(np.float32)
        u, v = B.upsample_flow(torch.from_numpy(uc).cuda(), torch.from_numpy(vc).cuda(), W, H)
        assert np.max(np.abs(u.cpu().numpy() - oracle.upsample_flow(uc, W, H))) < 2e-6
        assert np.max(np.abs(v.cpu().numpy() - oracle.upsample_flow(vc, W, H))) < 2e-6


def test_intermediates_per_level(torch, B, oracle):
    """Pyramid levels, the per-level fields (rule D23 applied at every level: element-wise on the pixels whose determinant exceeds
    1e-3 of the level's maximum) and det against the oracle's intermediates."""
    c = syn.config3(352, 288)
    ref = oracle.solve(c.I1, c.I2, 3, 6, 3, GAUSS, return_levels=True)
    with B.OpticalFlow(352, 288, 3, 6, 3, GAUSS) as of:
        u, v = of.compute(torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda())
        torch.cuda.synchronize()
        P1, P2 = c.I1.astype(np.float64), c.I2.astype(np.float64)
        for l in range(3):
            g = of.debug_plane(l, 0).cpu().numpy()
            assert np.max(np.abs(g - P1)) < 1e-4, l
            if l >= 1:
                gu = of.debug_plane(l, 2).cpu().numpy().astype(np.float64)
                gv = of.debug_plane(l, 3).cpu().numpy().astype(np.float64)
                det_l = oracle.iteration(P1, P2, np.zeros_like(P1), np.zeros_like(P1), 6, GAUSS)[4]     # iteration independent (D9)
                S = det_l > 1e-3 * det_l.max()
                du, dv = (gu - ref["level_u"][l])[S], (gv - ref["level_v"][l])[S]
                assert S.mean() > 0.5 and max(np.abs(du).max(), np.abs(dv).max()) <= 1e-3, (l, np.abs(du).max(), np.abs(dv).max())
                assert np.sqrt(np.mean(du * du + dv * dv)) <= 1e-4, l
            P1, P2 = oracle.downsample(P1), oracle.downsample(P2)
        det = of.debug_plane(0, 9).cpu().numpy()
        assert np.max(np.abs(det - ref["det"])) <= 1e-4 * ref["det"].max()


@pytest.mark.parametrize("W,H,R,wt", [(192, 160, 8, BOX), (203, 131, 12, GAUSS)])
def test_k2_planes_and_window_sums_elementwise(torch, B, oracle, W, H, R, wt):
    """K2 on its own: the five horizontally summed product planes (debug planes 4..8) after one stand-alone K2 pass from a non-zero
    field, element by element against the oracle's warp / gradients / products summed along x; and those planes summed along y
    against the oracle's window sums a, b, c, p, q (sums5).  Zero extension outside the image (D12) in both directions."""
    from scipy.ndimage import correlate1d
    c = syn.config1(W, H)
    I1, I2 = c.I1.astype(np.float64), c.I2.astype(np.float64)
    with B.OpticalFlow(W, H, 1, R, 2, wt) as of:
        of.compute(torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda())
        torch.cuda.synchronize()
        u0 = of.debug_plane(0, 2).cpu().numpy().astype(np.float64)
        v0 = of.debug_plane(0, 3).cpu().numpy().astype(np.float64)
        of.run_step(0, 0)
        torch.cuda.synchronize()
        planes = [of.debug_plane(0, 4 + f).cpu().numpy().astype(np.float64) for f in range(5)]
    I2w = oracle.warp(I2, u0, v0)
    Ix, Iy = oracle.gradients(I1)
    It = I2w - I1 - Ix * u0 - Iy * v0
    prods = [Ix * Ix, Ix * Iy, Iy * Iy, Ix * It, Iy * It]
    w = np.array([oracle.window_weight(t, R, wt) for t in range(-R, R + 1)])
    sums5 = oracle.iteration(I1, I2, u0, v0, R, wt)[2]
    for f in range(5):
        hs = correlate1d(prods[f], w, axis=1, mode="constant", cval=0.0)
        scale = max(np.abs(hs).max(), 1e-30)
        assert np.abs(planes[f] - hs).max() <= 1e-5 * scale, (f, np.abs(planes[f] - hs).max(), scale)
        ws = correlate1d(planes[f], w, axis=0, mode="constant", cval=0.0)
        scale = max(np.abs(sums5[f]).max(), 1e-30)
        assert np.abs(ws - sums5[f]).max() <= 1e-5 * scale, (f, np.abs(ws - sums5[f]).max(), scale)


def test_single_iteration_kernels_vs_oracle(torch, B, oracle):
    """K2 then K3 run once through of_run_step from a non-zero field equal one oracle iteration."""
    c = syn.config1(192, 160)
    I1, I2 = c.I1.astype(np.float64), c.I2.astype(np.float64)
    with B.OpticalFlow(192, 160, 1, 8, 2, BOX) as of:
        of.compute(torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda())
        torch.cuda.synchronize()
        u0 = of.debug_plane(0, 2).cpu().numpy().astype(np.float64)    # field after iteration 1
        v0 = of.debug_plane(0, 3).cpu().numpy().astype(np.float64)
        of.run_step(0, 0)
        of.run_step(0, 1)
        torch.cuda.synchronize()
        u1 = of.debug_plane(0, 2).cpu().numpy()
        v1 = of.debug_plane(0, 3).cpu().numpy()
    ru, rv, sums, valid, det = oracle.iteration(I1, I2, u0, v0, 8, BOX)
    S = det > 1e-3 * det.max()
    assert np.max(np.abs(u1 - ru)[S]) < 1e-4 and np.max(np.abs(v1 - rv)[S]) < 1e-4


# ---------------------------------------------------------------------------- edge cases
@pytest.mark.parametrize("W,H,L,R,it,wt", [
    (17, 17, 1, 8, 2, BOX),          # image == window
    (3, 3, 1, 1, 1, BOX),            # smallest legal
    (33, 65, 1, 16, 3, GAUSS),       # maximum radius
    (130, 70, 2, 4, 3, BOX),         # ragged, two levels, odd sizes downstream (65x35)
    (129, 67, 3, 2, 2, GAUSS),       # odd sizes at every level
    (1000, 36, 1, 1, 5, BOX),        # wide and flat
    (36, 1000, 2, 5, 2, BOX),        # tall and thin
])
def test_ragged_and_degenerate_sizes(torch, B, oracle, W, H, L, R, it, wt):
    rng = np.random.default_rng(W * 1000 + H)
    xp, yp, amp = syn.seed_particles(rng, W, H, 0.05, 100, 255)
    I1 = syn.quantize(syn.render_particles(xp, yp, amp, 1.2, W, H), np.uint8, 255)
    I2 = syn.quantize(syn.render_particles(xp + 0.6, yp - 0.4, amp, 1.2, W, H), np.uint8, 255)
    ref = oracle.solve(I1, I2, L, R, it, wt)
    u, v, m, _ = gpu_solve(torch, B, I1, I2, L, R, it, wt)
    if ref["det"].max() > 0:
        assert_parity(u, v, m, ref, (W, H, L, R))
    else:
        assert np.array_equal(m, ref["valid"])


def test_identical_images_exact_zero(torch, B):
    c = syn.config2(300, 200)
    u, v, m, _ = gpu_solve(torch, B, c.I1, c.I1, 2, 7, 4, BOX)
    assert np.all(u == 0.0) and np.all(v == 0.0)


def test_empty_images_all_invalid(torch, B, oracle):
    z = np.zeros((96, 128), dtype=np.uint8)
    u, v, m, _ = gpu_solve(torch, B, z, z, 2, 5, 2, BOX)
    assert np.all(u == 0) and np.all(v == 0) and np.all(m == 0)
    # sparse texture: most windows are empty -> masks must still agree exactly
    z1, z2 = z.copy(), z.copy()
    z1[40:44, 60:64] = 200
    z2[40:44, 61:65] = 200
    ref = oracle.solve(z1, z2, 1, 5, 3, BOX)
    u, v, m, _ = gpu_solve(torch, B, z1, z2, 1, 5, 3, BOX)
    assert np.array_equal(m, ref["valid"]) and 0 < m.sum() < m.size
    assert np.all(u[m == 0] == 0)


def test_saturated_and_large_displacements_stay_finite(torch, B, oracle):
    """Full-scale 16-bit values and displacements far beyond eq. 1's range: finite, clamped to
    +-3 px per iteration (D15), identical masks."""
    rng = np.random.default_rng(5)
    I1 = rng.integers(0, 65536, (120, 160)).astype(np.uint16)
    I2 = np.roll(I1, 25, axis=1)
    ref = oracle.solve(I1, I2, 1, 6, 4, BOX)
    u, v, m, _ = gpu_solve(torch, B, I1, I2, 1, 6, 4, BOX)
    assert np.isfinite(u).all() and np.isfinite(v).all()
    assert np.abs(u).max() <= 12.0 + 1e-4 and np.abs(v).max() <= 12.0 + 1e-4
    assert np.array_equal(m, ref["valid"])


def test_graph_and_plain_launches_agree_bitwise_and_repeat(torch, B):
    c = syn.config3(320, 256)
    a = gpu_solve(torch, B, c.I1, c.I2, 3, 12, 4, GAUSS, graph=True)
    b = gpu_solve(torch, B, c.I1, c.I2, 3, 12, 4, GAUSS, graph=False)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    assert a[3] == b[3] == 2 + 1                          # convert+pyramid, pyramid, 1 persistent solve
    H, W = c.I1.shape
    with B.OpticalFlow(W, H, 3, 12, 4, GAUSS) as of:
        d1, d2 = torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda()
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            u1, v1 = of.compute(d1, d2)
            u1 = u1.clone()
            u2, v2 = of.compute(d1, d2)      # graph replay with new output pointers
            u3, v3 = of.compute(d1, d2, u2, v2)   # same pointers: cached graph
        s.synchronize()
        assert torch.equal(u1, u2) and torch.equal(u1, u3) and np.array_equal(u1.cpu().numpy(), a[0])


@pytest.mark.parametrize("W,H,L,R,it,wt", [(320, 256, 3, 12, 4, GAUSS), (130, 70, 2, 4, 3, BOX), (1280, 1024, 3, 12, 10, GAUSS)])
def test_persistent_and_per_kernel_launches_agree_bitwise(torch, B, W, H, L, R, it, wt):
    """The persistent solve kernel runs the same passes as the stand-alone K2/K3/K4 launches, so the two
    modes must agree bit for bit (also pins the grid barrier and the cross-pass memory ordering)."""
    c = syn.config3(W, H)
    d1, d2 = torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda()
    out = []
    for persistent in (True, False):
        with B.OpticalFlow(W, H, L, R, it, wt) as of:
            of.set_persistent(persistent)
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                for _ in range(3):                      # repeat: barrier generation and ring parity carry over
                    u, v = of.compute(d1, d2)
                m = of.validity()
            s.synchronize()
            out.append((u.cpu().numpy(), v.cpu().numpy(), m.cpu().numpy(), of.last_launch_count()))
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1]) and np.array_equal(out[0][2], out[1][2])
    prep = 1 if L == 1 else L - 1                          # conversion is fused into the first pyramid step
    assert out[0][3] == prep + 1 and out[1][3] == prep + (L - 1) + 2 * L * it


@pytest.mark.parametrize("W,H,L,R,it,wt,persistent", [(320, 256, 3, 12, 4, GAUSS, True), (130, 70, 2, 4, 3, BOX, True),
                                                     (203, 131, 3, 8, 5, BOX, False), (256, 256, 4, 10, 3, BOX, True),
                                                     (37, 23, 1, 2, 1, BOX, True), (70, 67, 2, 16, 2, GAUSS, True),
                                                     (1280, 1024, 3, 12, 10, GAUSS, True)])
def test_hoisted_invariant_planes_agree_bitwise(torch, B, W, H, L, R, it, wt, persistent):
    """of_set_hoist (SURVEY.md 8(f) note f5, reading D9): IxIx, IxIy, IyIy depend on I1 alone, so forming them in the
    first iteration of a level only must not change a single bit of the result, with and without an obstacle mask."""
    c = syn.config3(W, H)
    d1, d2 = torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda()
    mask = np.ones((H, W), np.uint8)
    mask[H // 3: H // 2, : W // 2] = 0
    for use_mask in (False, True):
        out = []
        for hoist in (False, True):
            with B.OpticalFlow(W, H, L, R, it, wt) as of:
                of.set_persistent(persistent)
                of.set_hoist(hoist)
                if use_mask:
                    of.set_mask(mask)
                s = torch.cuda.Stream()
                with torch.cuda.stream(s):
                    for _ in range(2):                  # second solve: the planes of the previous pair must not leak in
                        u, v = of.compute(d2 if _ == 0 else d1, d1 if _ == 0 else d2)
                    m = of.validity()
                s.synchronize()
                out.append((u.cpu().numpy(), v.cpu().numpy(), m.cpu().numpy()))
        assert all(np.array_equal(a, b) for a, b in zip(out[0], out[1])), "hoist changed the result (mask=%s)" % use_mask


def test_large_image_crop_parity(torch, B, oracle):
    """4096x3072, one level: the result in a window depends only on a neighbourhood of radius
    iterations*(R+max|u|+2), so the oracle on a crop pins sampled outputs of the full-size run."""
    W, H, R, it = 4096, 3072, 8, 3
    rng = np.random.default_rng(77)
    xp, yp, amp = syn.seed_particles(rng, W, H, 0.03, 150, 255)
    I1 = syn.quantize(syn.render_particles(xp, yp, amp, 1.2, W, H), np.uint8, 255)
    I2 = syn.quantize(syn.render_particles(xp + 1.4, yp + 0.8, amp, 1.2, W, H), np.uint8, 255)
    u, v, m, _ = gpu_solve(torch, B, I1, I2, 1, R, it, BOX)
    margin = it * (R + 3 + 2) + 4
    for (x0, y0) in ((0, 0), (W - 300, H - 260), (1900, 1500), (W - 300, 0)):
        cw, ch = 300, 260
        ref = oracle.solve(I1[y0:y0 + ch, x0:x0 + cw], I2[y0:y0 + ch, x0:x0 + cw], 1, R, it, BOX)
        sl = (slice(margin, ch - margin), slice(margin, cw - margin))
        gsl = (slice(y0 + margin, y0 + ch - margin), slice(x0 + margin, x0 + cw - margin))
        sub = {k: ref[k][sl] for k in ("u", "v", "det", "valid")}
        assert_parity(u[gsl], v[gsl], m[gsl], sub, ("crop", x0, y0))


def test_errors_are_reported_not_thrown(B):
    assert B.lib().of_create(64, 64, 3, 8, 1, 0) in (None, 0)      # 16x16 < 17
    assert "coarsest" in B.last_error()
    assert B.lib().of_create(64, 64, 1, 17, 1, 0) in (None, 0)
    assert B.lib().of_create(64, 64, 1, 4, 0, 0) in (None, 0)
    assert B.lib().of_create(64, 64, 1, 4, 1, 7) in (None, 0)
    assert B.lib().of_compute(None, None, None, None, None, None) < 0
    B.lib().of_destroy(None)


# ---------------------------------------------------------------------------- eq. 2 pre-filter (NEXT item f1)
@pytest.mark.parametrize("dtype,W,H,r", [(np.uint8, 320, 256, 5), (np.uint16, 203, 131, 3), (np.float32, 130, 70, 5),
                                         (np.uint8, 64, 40, 16)])
def test_equalisation_kernel_matches_oracle(torch, B, oracle, dtype, W, H, r):
    """of_set_equalisation: the level-0 plane is eq. 2 of the raw frame; flat
    neighbourhoods give exactly 0 on both sides."""
    rng = np.random.default_rng(W + H + r)
    hi = {np.uint8: 256, np.uint16: 4096, np.float32: 256}[dtype]
    I1 = rng.integers(0, hi, (H, W)).astype(dtype)
    I2 = rng.integers(0, hi, (H, W)).astype(dtype)
    I1[H // 4:H // 2, W // 4:W // 2] = 7                      # a flat patch larger than the box
    ref1, ref2 = oracle.equalise(I1, r), oracle.equalise(I2, r)
    R = min(3, (min(W, H) - 1) // 2)
    with B.OpticalFlow(W, H, 1, R, 1, BOX) as of:
        of.set_equalisation(r)
        d1 = torch.from_numpy(I1.view(np.int16) if dtype == np.uint16 else I1).cuda()
        d2 = torch.from_numpy(I2.view(np.int16) if dtype == np.uint16 else I2).cuda()
        of.compute(d1, d2)
        torch.cuda.synchronize()
        g1, g2 = of.debug_plane(0, 0).cpu().numpy(), of.debug_plane(0, 1).cpu().numpy()
    assert np.max(np.abs(g1 - ref1)) < 2e-5 and np.max(np.abs(g2 - ref2)) < 2e-5
    assert np.array_equal(g1 == 0.0, ref1 == 0.0)


def test_solve_with_equalisation_matches_oracle(torch, B, oracle):
    """Whole path with the pre-filter on: unevenly lit config-3-like pair, parity at the usual bar."""
    c = syn.config3(352, 288)
    yy, xx = np.mgrid[0:288, 0:352]
    lit = 0.6 + 0.4 * xx / 352.0
    I2 = np.clip(np.rint(c.I2 * lit), 0, 255).astype(np.uint8)
    ref = oracle.solve(oracle.equalise(c.I1, 5), oracle.equalise(I2, 5), 3, 6, 4, GAUSS)
    with B.OpticalFlow(352, 288, 3, 6, 4, GAUSS) as of:
        of.set_equalisation(5)
        u, v = of.compute(torch.from_numpy(c.I1).cuda(), torch.from_numpy(I2).cuda())
        m = of.validity()
        torch.cuda.synchronize()
        st = assert_parity(u.cpu().numpy(), v.cpu().numpy(), m.cpu().numpy(), ref, "equalised")
        of.set_equalisation(0)
        u0, v0 = of.compute(torch.from_numpy(c.I1).cuda(), torch.from_numpy(I2).cuda())
        torch.cuda.synchronize()
    ref0 = oracle.solve(c.I1, I2, 3, 6, 4, GAUSS)
    assert_parity(u0.cpu().numpy(), v0.cpu().numpy(), None, ref0, "switched off again")


# ---------------------------------------------------------------------------- eq. 3 bubble surface (NEXT item f3)
def test_bubble_surface_counts_match_oracle_exactly(torch, B, oracle):
    """Mean field over 3 solves -> T_v -> thresholded count on the device; integer results, compared exactly
    with the oracle applied to the SAME fp32 fields (eq. 3)."""
    W, H = 320, 256
    with B.OpticalFlow(W, H, 2, 6, 3, BOX) as of:
        total = torch.zeros((H, W), dtype=torch.float32, device="cuda")
        fields = []
        for k in range(3):
            c = syn.config3(W, H, seed_offset=k)
            u, v = of.compute(torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda())
            of.field_accumulate(total, u)
            fields.append(u.clone())
        m = of.validity()
        mm = of.field_minmax(total, m)
        torch.cuda.synchronize()
        tot_h = fields[0].cpu().numpy().astype(np.float32)
        for f in fields[1:]:
            tot_h = tot_h + f.cpu().numpy()                       # same fp32 running sum, same order
        assert np.array_equal(total.cpu().numpy(), tot_h)
        mh = m.cpu().numpy()
        lo, hi = float(mm[0]), float(mm[1])
        assert lo == float(tot_h[mh != 0].min()) and hi == float(tot_h[mh != 0].max())
        T = np.float32(0.5) * (np.float32(lo) + np.float32(hi)) / np.float32(3.0)      # mid-range of the MEAN field
        assert abs(float(T) - oracle.bubble_threshold(tot_h.astype(np.float64) / 3.0, mh)) < 1e-5
        cnt = of.bubble_count(fields[2], float(T), m)
        cnt_all = of.bubble_count(fields[2], float(T))
        torch.cuda.synchronize()
        assert tuple(cnt.cpu().tolist()) == oracle.bubble_counts(fields[2].cpu().numpy(), float(T), mh)
        assert tuple(cnt_all.cpu().tolist()) == oracle.bubble_counts(fields[2].cpu().numpy(), float(T))
        assert 0 < cnt[0] < cnt[1] <= W * H
        # the same with the threshold kept on the device (no host value between the steps of eq. 3)
        thr_dev = of.bubble_threshold(total, 3, m)
        cnt_dev = of.bubble_count_dev(fields[2], thr_dev, m)
        torch.cuda.synchronize()
        assert np.float32(thr_dev.cpu().numpy()[0]) == T
        assert tuple(cnt_dev.cpu().tolist()) == tuple(cnt.cpu().tolist())


# ---------------------------------------------------------------------------- NEXT item f4: obstacle masks
def gpu_solve_masked(torch, B, c, mask, persistent=True, graph=True, then_clear=False):
    with B.OpticalFlow(c.width, c.height, c.levels, c.window_radius, c.iterations, c.window_type) as of:
        of.set_graph(graph)
        of.set_persistent(persistent)
        of.set_mask(mask)
        d1 = torch.from_numpy(c.I1.view(np.int16) if c.I1.dtype == np.uint16 else c.I1).cuda()
        d2 = torch.from_numpy(c.I2.view(np.int16) if c.I2.dtype == np.uint16 else c.I2).cuda()
        s = torch.cuda.Stream()
        out = []
        with torch.cuda.stream(s):
            for rep in range(2):                       # twice: the second solve starts from the fields the first one left
                u = torch.full((c.height, c.width), 7.0, dtype=torch.float32, device="cuda")   # stale values must be overwritten
                v = torch.full((c.height, c.width), -7.0, dtype=torch.float32, device="cuda")
                of.compute(d1, d2, u, v)
                out.append((u.cpu().numpy(), v.cpu().numpy(), of.validity().cpu().numpy()))
            if then_clear:
                of.set_mask(None)
                u, v = of.compute(d1, d2)
                out.append((u.cpu().numpy(), v.cpu().numpy(), of.validity().cpu().numpy()))
        s.synchronize()
        return out


def _blob_mask(H, W):
    m = np.ones((H, W), dtype=np.uint8)
    m[H // 4:H // 2, W // 8:W // 2] = 0
    m[:, :3] = 0
    m[(3 * H) // 4, (3 * W) // 4] = 0
    return m


@pytest.mark.parametrize("case,maskfn", [
    (lambda: syn.config1(), _blob_mask),
    (lambda: syn.config2(203, 157), _blob_mask),
    (lambda: syn.config3(320, 256), lambda H, W: syn.mask_backward_step(W, H)),
    (lambda: syn.config4(256, 192), _blob_mask),
    (lambda: syn.config3(), lambda H, W: syn.mask_backward_step(W, H)),
], ids=["config1", "config2-ragged", "config3-small-step", "config4-small-u16", "config3-1280x1024-step"])
def test_masked_solve_matches_oracle(torch, B, oracle, case, maskfn):
    """Readings M1-M5: parity on the fluid pixels, exactly no vector over the obstacle, identical validity;
    the persistent kernel and the per-kernel launches agree bit for bit; a repeat gives the same bits."""
    c = case()
    mask = maskfn(c.height, c.width)
    ref = oracle.solve(c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type, mask=mask)
    runs = gpu_solve_masked(torch, B, c, mask)
    u, v, m = runs[0]
    st = assert_parity(u, v, m, ref, c.name + "+mask")
    print(c.name, "masked", st)
    assert np.all(u[mask == 0] == 0.0) and np.all(v[mask == 0] == 0.0) and np.all(m[mask == 0] == 0)
    assert np.array_equal(runs[1][0], u) and np.array_equal(runs[1][1], v) and np.array_equal(runs[1][2], m)
    u2, v2, m2 = gpu_solve_masked(torch, B, c, mask, persistent=False, graph=False)[0]
    assert np.array_equal(u2, u) and np.array_equal(v2, v) and np.array_equal(m2, m)


def test_mask_of_ones_zeros_and_removal(torch, B):
    c = syn.config3(320, 256)
    plain = gpu_solve(torch, B, c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type)
    ones = gpu_solve_masked(torch, B, c, np.ones((c.height, c.width), np.uint8))[0]
    assert np.array_equal(ones[0], plain[0]) and np.array_equal(ones[1], plain[1]) and np.array_equal(ones[2], plain[2])
    runs = gpu_solve_masked(torch, B, c, np.zeros((c.height, c.width), np.uint8), then_clear=True)
    assert not runs[0][0].any() and not runs[0][1].any() and not runs[0][2].any()
    assert np.array_equal(runs[2][0], plain[0]) and np.array_equal(runs[2][1], plain[1]) and np.array_equal(runs[2][2], plain[2])


def test_mask_skips_work(torch, B):
    """The point of the mask (PAPER.md:175 'higher speeds'): the solve of a half-masked frame is faster."""
    c = syn.config3()
    mask = np.ones((c.height, c.width), np.uint8)
    mask[:, c.width // 2:] = 0
    with B.OpticalFlow(c.width, c.height, c.levels, c.window_radius, c.iterations, c.window_type) as of:
        d1, d2 = torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda()
        of.compute(d1, d2)
        def timed():
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            of.run_solve(5)
            a.record(); of.run_solve(20); b.record(); b.synchronize()
            return a.elapsed_time(b) / 20
        t_full = timed()
        of.set_mask(mask)
        of.compute(d1, d2)
        t_half = timed()
    print("solve ms: unmasked %.3f, right half masked %.3f" % (t_full, t_half))
    assert t_half < 0.9 * t_full


# ---------------------------------------------------------------------------- conditioning (D14, D15)
@pytest.mark.parametrize("eps,max_step", [(1e-2, 3.0), (1e-6, 3.0), (1e-3, 0.5)])
def test_conditioning_parity(torch, B, oracle, eps, max_step):
    """of_set_conditioning: relative damping 1e-2 / 1e-6 and a step limit of 0.5 px that is active (the images are 2.4 px apart and
    there is one level, so the first iterations are clamped) against the oracle run with the same constants."""
    W, H = 224, 160
    rng = np.random.default_rng(2461)
    xp, yp, amp = syn.seed_particles(rng, W, H, 0.04, 120, 255)
    I1 = syn.quantize(syn.render_particles(xp, yp, amp, 1.3, W, H), np.uint8, 255)
    I2 = syn.quantize(syn.render_particles(xp + 2.4, yp - 1.1, amp, 1.3, W, H), np.uint8, 255)
    ref = oracle.solve(I1, I2, 1, 9, 5, BOX, eps=eps, max_step=max_step)
    with B.OpticalFlow(W, H, 1, 9, 5, BOX) as of:
        of.set_conditioning(eps, max_step)
        u, v = of.compute(torch.from_numpy(I1).cuda(), torch.from_numpy(I2).cuda())
        m = of.validity()
        torch.cuda.synchronize()
        u, v, m = u.cpu().numpy(), v.cpu().numpy(), m.cpu().numpy()
    st = assert_parity(u, v, m, ref, "conditioning eps=%g max_step=%g" % (eps, max_step))
    if max_step < 1.0:                                  # the clamp was active: after 5 iterations nothing can exceed 5 x 0.5 px
        assert np.abs(ref["u"]).max() <= 5 * max_step + 1e-9 and np.abs(u).max() <= 5 * max_step + 1e-4
        assert np.abs(ref["u"]).max() > 4 * max_step
    print("conditioning", eps, max_step, st)


def test_fp32_frames_of_tiny_gain(torch, B, oracle):
    """Gain invariance of the fp32 path: the same pair scaled by 1e-6 (fp32 frames of very small gain).  The oracle is gain
    invariant to 4e-15 (pinned on the CPU side); here the fp32 kernels (approximate reciprocal of a determinant of ~1e-20) must
    still meet the parity bar and agree with the unscaled run."""
    c = syn.config2(320, 256)
    g = np.float32(1e-6)
    f1, f2 = c.I1.astype(np.float32) * g, c.I2.astype(np.float32) * g
    ref = oracle.solve(f1, f2, c.levels, c.window_radius, c.iterations, c.window_type)
    u, v, m, _ = gpu_solve(torch, B, f1, f2, c.levels, c.window_radius, c.iterations, c.window_type)
    st = assert_parity(u, v, m, ref, "tiny gain")
    u1, v1, m1, _ = gpu_solve(torch, B, c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type)
    S = ref["det"] > 1e-3 * ref["det"].max()
    assert np.abs(u - u1)[S].max() < 1e-3 and np.abs(v - v1)[S].max() < 1e-3 and np.array_equal(m, m1)
    print("tiny gain", st)


# ---------------------------------------------------------------------------- streaming variants
@pytest.mark.parametrize("dtype_name", ["u16", "f32"])
def test_stream_device_results_and_validity(torch, B, oracle, dtype_name):
    """of_stream_* with device-resident results (result_on_host = 0), 16-bit and fp32 frames, CONSECUTIVE mode: every field and its
    validity plane (of_stream_result_validity: one plane per slot of the result ring) equal the non-streaming call bit for bit."""
    W, H, n = 320, 256, 5
    rng = np.random.default_rng(77)
    xp, yp, amp = syn.seed_particles(rng, W, H, 0.03, 1500, 4095)
    frames = []
    for k in range(n):
        img = syn.render_particles(xp + 0.9 * k, yp + 0.3 * k, amp, 1.4, W, H)
        frames.append(syn.quantize(img, np.uint16, 4095) if dtype_name == "u16" else img.astype(np.float32))
    dt = B.OF_DTYPE_U16 if dtype_name == "u16" else B.OF_DTYPE_F32
    to_dev = (lambda a: torch.from_numpy(a.view(np.int16)).cuda()) if dtype_name == "u16" else (lambda a: torch.from_numpy(a).cuda())
    args = (W, H, 2, 7, 4, BOX)
    with B.OpticalFlow(*args) as of, B.OpticalFlow(*args) as of2:
        of.stream_open(dt, B.OF_STREAM_CONSECUTIVE, False)
        got = []
        for k, f in enumerate(frames):
            slot = of.stream_acquire()
            slot[...] = f
            of.stream_submit()
            if k >= 1:
                idx, pu, pv = of.stream_result()
                pm = of.stream_result_validity()
                assert idx == k - 1 and isinstance(pu, int) and isinstance(pm, int)
                got.append((B.device_to_numpy(pu, W * H, np.float32).reshape(H, W), B.device_to_numpy(pv, W * H, np.float32).reshape(H, W),
                            B.device_to_numpy(pm, W * H, np.uint8).reshape(H, W)))
        of.stream_close()
        for k in range(n - 1):
            u2, v2 = of2.compute(to_dev(frames[k]), to_dev(frames[k + 1]))
            m2 = of2.validity()
            torch.cuda.synchronize()
            assert np.array_equal(got[k][0], u2.cpu().numpy()) and np.array_equal(got[k][1], v2.cpu().numpy()), k
            assert np.array_equal(got[k][2], m2.cpu().numpy()), k
        ref = oracle.solve(frames[0], frames[1], 2, 7, 4, BOX)
        print("stream", dtype_name, assert_parity(got[0][0], got[0][1], got[0][2], ref, "stream device results"))


def test_stream_consecutive_with_mask_and_equalisation(torch, B, oracle):
    """CONSECUTIVE mode with an obstacle mask and the eq. 2 pre-filter set: the first frame of a stream takes a separate code path
    (conversion + pyramid only).  Host results and validity planes against the masked oracle on equalised frames."""
    W, H, n = 320, 256, 4
    rng = np.random.default_rng(78)
    xp, yp, amp = syn.seed_particles(rng, W, H, 0.03, 120, 255)
    frames = [syn.quantize(syn.render_particles(xp + 0.7 * k, yp - 0.4 * k, amp, 1.3, W, H) + 20.0 * (np.arange(W) / W)[None, :], np.uint8, 255)
              for k in range(n)]
    mask = syn.mask_backward_step(W, H)
    with B.OpticalFlow(W, H, 2, 6, 4, GAUSS) as of:
        of.set_equalisation(5)
        of.set_mask(mask)
        of.stream_open(B.OF_DTYPE_U8, B.OF_STREAM_CONSECUTIVE, True)
        out = []
        for k, f in enumerate(frames):
            slot = of.stream_acquire()
            slot[...] = f
            of.stream_submit()
            if k >= 1:
                idx, u, v = of.stream_result()
                out.append((u.copy(), v.copy(), of.stream_result_validity().copy()))
        of.stream_close()
    eq = [oracle.equalise(f.astype(np.float64), 5) for f in frames]
    for k in range(n - 1):
        ref = oracle.solve(eq[k], eq[k + 1], 2, 6, 4, GAUSS, mask=mask)
        st = assert_parity(out[k][0], out[k][1], out[k][2], ref, "stream mask+eq pair %d" % k)
        assert np.all(out[k][0][mask == 0] == 0.0) and np.all(out[k][2][mask == 0] == 0)
    print("stream mask+eq", st)


# ---------------------------------------------------------------------------- masked + hoisted against the oracle
@pytest.mark.parametrize("W,H,L,R,it,wt", [(256, 256, 4, 10, 3, BOX), (320, 256, 3, 12, 4, GAUSS)])
def test_masked_hoisted_solve_matches_oracle(torch, B, oracle, W, H, L, R, it, wt):
    """of_set_hoist together with of_set_mask against the masked oracle (the bitwise hoist test compares with the default kernel only)."""
    c = syn.config3(W, H)
    mask = np.ones((H, W), np.uint8)
    mask[H // 3: H // 2, : W // 2] = 0
    ref = oracle.solve(c.I1, c.I2, L, R, it, wt, mask=mask)
    with B.OpticalFlow(W, H, L, R, it, wt) as of:
        of.set_hoist(True)
        of.set_mask(mask)
        u, v = of.compute(torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda())
        m = of.validity()
        torch.cuda.synchronize()
        u, v, m = u.cpu().numpy(), v.cpu().numpy(), m.cpu().numpy()
    print("mask+hoist", assert_parity(u, v, m, ref, "mask+hoist"))
    assert np.all(u[mask == 0] == 0.0) and np.all(m[mask == 0] == 0)


def test_fused_and_two_pass_levels_agree_bitwise(torch, B):
    """of_set_fused (coarse levels iterated inside the CTA, of_fused.cuh) against the two-pass form in the same persistent kernel."""
    for (W, H, L, R, it, wt) in [(256, 256, 1, 8, 4, BOX), (640, 512, 3, 12, 3, GAUSS), (203, 131, 2, 5, 5, BOX)]:
        c = syn.config3(W, H)
        d1, d2 = torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda()
        out = []
        for fused in (True, False):
            with B.OpticalFlow(W, H, L, R, it, wt) as of:
                of.set_fused(fused)
                u, v = of.compute(d1, d2)
                m = of.validity()
                torch.cuda.synchronize()
                out.append((u.cpu().numpy(), v.cpu().numpy(), m.cpu().numpy()))
        assert all(np.array_equal(a, b) for a, b in zip(out[0], out[1])), (W, H, L, R)


def test_misaligned_field_pointers_are_rejected(torch, B):
    c = syn.config1()
    with B.OpticalFlow(*c.create_args) as of:
        d1, d2 = torch.from_numpy(c.I1.astype(np.float32)).cuda(), torch.from_numpy(c.I2.astype(np.float32)).cuda()
        big = torch.empty(c.width * c.height + 4, dtype=torch.float32, device="cuda")
        good = torch.empty(c.width * c.height, dtype=torch.float32, device="cuda")
        rc = B.lib().of_compute(of._h, d1.data_ptr(), d2.data_ptr(), big.data_ptr() + 4, good.data_ptr(), None)
        assert rc == B.OF_ERR_INVALID_ARG and "aligned" in B.last_error()


@pytest.mark.parametrize("W,H,L,R,it,wt,hoist,masked", [(320, 256, 3, 12, 4, GAUSS, False, False), (256, 256, 1, 8, 4, BOX, False, False),
                                                        (448, 320, 2, 7, 6, BOX, True, True), (1280, 1024, 3, 12, 10, GAUSS, False, False)])
def test_repeated_solves_are_bitwise_stable(torch, B, W, H, L, R, it, wt, hoist, masked):
    """Race evidence without a sanitizer (compute-sanitizer is closed on this GPU pool, profiles/r2_sanitizer.md): the grid barrier,
    the mbarrier rings, the proxy fences and the shared-memory union between the passes are all exercised by 60 back-to-back solves on
    one handle, alternating two different pairs, and every result must reproduce the first one of its pair bit for bit."""
    ca, cb = syn.config3(W, H, seed_offset=0), syn.config3(W, H, seed_offset=1)
    d = [(torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda()) for c in (ca, cb)]
    with B.OpticalFlow(W, H, L, R, it, wt) as of:
        of.set_hoist(hoist)
        if masked:
            mask = np.ones((H, W), np.uint8)
            mask[H // 3: H // 2, : W // 2] = 0
            of.set_mask(mask)
        first = [None, None]
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            outs = []
            for k in range(60):
                u, v = of.compute(d[k & 1][0], d[k & 1][1])
                outs.append((k & 1, u, v, of.validity()))
        s.synchronize()
        for k, u, v, m in outs:
            if first[k] is None:
                first[k] = (u, v, m)
            else:
                assert torch.equal(u, first[k][0]) and torch.equal(v, first[k][1]) and torch.equal(m, first[k][2])
        assert not torch.equal(first[0][0], first[1][0])


# ---------------------------------------------------------------------------- throughput mode: two pairs in one launch (of_compute_dual)
@pytest.mark.parametrize("W,H,L,R,it,wt,dt", [(320, 256, 3, 12, 4, GAUSS, "u8"), (256, 256, 1, 8, 4, BOX, "f32"), (130, 70, 2, 4, 3, BOX, "u8"),
                                              (203, 131, 2, 5, 5, GAUSS, "u8"), (1280, 1024, 3, 12, 10, GAUSS, "u8"), (1280, 1024, 3, 8, 10, BOX, "u8"),
                                              (1024, 1024, 2, 7, 6, BOX, "u16")])
def test_dual_launch_matches_single_solves_bitwise(torch, B, W, H, L, R, it, wt, dt):
    """of_compute_dual runs the passes of two different pairs alternately in one persistent kernel with split grid barriers
    (csrc/of_solve_dual.cuh).  Each pair must come out exactly as of_compute gives it (fields and validity masks), also on the
    second and third launch (barrier counters and ring parities carry over), and a single solve on the same handles afterwards
    must still be right (the counters are returned to zero)."""
    ca, cb = syn.config3(W, H, seed_offset=0), syn.config3(W, H, seed_offset=1)

    def dev(a):
        if dt == "f32":
            return torch.from_numpy(a.astype(np.float32)).cuda()
        if dt == "u16":
            return torch.from_numpy((a.astype(np.uint16) * 16).view(np.int16)).cuda()
        return torch.from_numpy(a).cuda()
    d = [(dev(c.I1), dev(c.I2)) for c in (ca, cb)]
    with B.OpticalFlow(W, H, L, R, it, wt) as ofa, B.OpticalFlow(W, H, L, R, it, wt) as ofb:
        ref = []
        for of, (i1, i2) in ((ofa, d[0]), (ofb, d[1])):
            u, v = of.compute(i1, i2)
            ref.append((u.clone(), v.clone(), of.validity().clone()))
        torch.cuda.synchronize()
        assert not torch.equal(ref[0][0], ref[1][0])
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            for rep in range(3):
                ua, va, ub, vb = B.compute_dual(ofa, ofb, d[0][0], d[0][1], d[1][0], d[1][1])
                ma, mb = ofa.validity(), ofb.validity()
        s.synchronize()
        assert ofa.last_launch_count() == 2 * (1 if L == 1 else L - 1) + 1
        assert torch.equal(ua, ref[0][0]) and torch.equal(va, ref[0][1]) and torch.equal(ma, ref[0][2])
        assert torch.equal(ub, ref[1][0]) and torch.equal(vb, ref[1][1]) and torch.equal(mb, ref[1][2])
        # pairs swapped between the handles, then a single solve on each handle
        with torch.cuda.stream(s):
            ub2, vb2, ua2, va2 = B.compute_dual(ofa, ofb, d[1][0], d[1][1], d[0][0], d[0][1])
            u1, v1 = ofb.compute(d[0][0], d[0][1])
        s.synchronize()
        assert torch.equal(ua2, ref[0][0]) and torch.equal(vb2, ref[1][1]) and torch.equal(u1, ref[0][0]) and torch.equal(v1, ref[0][1])


def test_dual_launch_against_oracle(torch, B, oracle):
    """The two fields of one of_compute_dual launch against the fp64 oracle, element by element (D23)."""
    W, H, L, R, it, wt = 448, 320, 3, 7, 5, BOX
    cs = [syn.config3(W, H, seed_offset=k) for k in (3, 4)]
    with B.OpticalFlow(W, H, L, R, it, wt) as ofa, B.OpticalFlow(W, H, L, R, it, wt) as ofb:
        ua, va, ub, vb = B.compute_dual(ofa, ofb, *[torch.from_numpy(x).cuda() for x in (cs[0].I1, cs[0].I2, cs[1].I1, cs[1].I2)])
        ma, mb = ofa.validity(), ofb.validity()
        torch.cuda.synchronize()
    for c, u, v, m in ((cs[0], ua, va, ma), (cs[1], ub, vb, mb)):
        ref = oracle.solve(c.I1, c.I2, L, R, it, wt)
        assert_parity(u.cpu().numpy(), v.cpu().numpy(), m.cpu().numpy(), ref, "dual")


def test_dual_launch_falls_back_and_rejects(torch, B):
    """Handles that cannot share a launch (a mask on one of them) are solved one after the other with the same results; the same
    handle twice is rejected."""
    W, H, L, R, it, wt = 320, 256, 2, 6, 3, BOX
    ca, cb = syn.config3(W, H, seed_offset=0), syn.config3(W, H, seed_offset=1)
    d = [torch.from_numpy(x).cuda() for x in (ca.I1, ca.I2, cb.I1, cb.I2)]
    mask = np.ones((H, W), np.uint8)
    mask[40:90, 100:200] = 0
    with B.OpticalFlow(W, H, L, R, it, wt) as ofa, B.OpticalFlow(W, H, L, R, it, wt) as ofb:
        ofb.set_mask(mask)
        ra = [t.clone() for t in ofa.compute(d[0], d[1])]
        rb = [t.clone() for t in ofb.compute(d[2], d[3])]
        ua, va, ub, vb = B.compute_dual(ofa, ofb, *d)
        torch.cuda.synchronize()
        assert torch.equal(ua, ra[0]) and torch.equal(va, ra[1]) and torch.equal(ub, rb[0]) and torch.equal(vb, rb[1])
        assert float(ub[60, 150]) == 0.0 and ofa.last_launch_count() == 2            # an ordinary solve: pyramid + solve kernel
        with pytest.raises(B.OptflowError):
            B.compute_dual(ofa, ofa, *d)
        with pytest.raises(B.OptflowError):
            B.run_solve_dual(ofa, ofb)


@pytest.mark.parametrize("W,H,L,R,it,wt", [(320, 256, 3, 12, 4, GAUSS), (640, 512, 2, 8, 5, BOX), (1280, 1024, 3, 12, 10, GAUSS)])
def test_dual_repeated_launches_are_bitwise_stable(torch, B, W, H, L, R, it, wt):
    """Race evidence for the split grid barrier of of_solve_dual (compute-sanitizer is closed on this pool): 40 two-pair launches in a
    row on the same two handles, the pairs swapping handles every launch and a single solve thrown in every eighth launch; every
    field must reproduce the first one of its pair bit for bit."""
    cs = [syn.config3(W, H, seed_offset=k) for k in (0, 1)]
    d = [(torch.from_numpy(c.I1).cuda(), torch.from_numpy(c.I2).cuda()) for c in cs]
    with B.OpticalFlow(W, H, L, R, it, wt) as ofa, B.OpticalFlow(W, H, L, R, it, wt) as ofb:
        outs = []
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            for k in range(40):
                p, q = (0, 1) if k % 2 == 0 else (1, 0)
                ua, va, ub, vb = B.compute_dual(ofa, ofb, d[p][0], d[p][1], d[q][0], d[q][1])
                outs += [(p, ua, va), (q, ub, vb)]
                if k % 8 == 7:
                    u1, v1 = ofa.compute(d[1][0], d[1][1])
                    outs.append((1, u1, v1))
        s.synchronize()
        first = [None, None]
        for p, u, v in outs:
            if first[p] is None:
                first[p] = (u, v)
            else:
                assert torch.equal(u, first[p][0]) and torch.equal(v, first[p][1])
        assert not torch.equal(first[0][0], first[1][0])
