"""Pins of the fp64 oracle (oracle/) against things OTHER than itself: closed forms, invariants,
library special cases, brute force in numpy, and a statistical expectation.  S-numbers refer to
DESIGN.md "Oracle pins".  CPU only."""
import math
import os

import numpy as np
import pytest
import scipy.ndimage as ndi

HERE = os.path.dirname(os.path.abspath(__file__))


# ------------------------------------------------------------------------------------ taps

CONFIG_SIGMAS = [1.0, 1.5, 2.0, 2.5, 3.0, 4.0, 8.0, 16.0, 24.0, 32.0]


@pytest.mark.parametrize("sigma", CONFIG_SIGMAS + [0.7, 5.3])
def test_S1_taps_invariants(oracle, sigma):
    g = oracle.taps(sigma)
    r = math.ceil(3.0 * sigma)
    assert len(g) == 2 * r + 1                                  # C-2: F = 2*ceil(3 sigma)+1
    assert np.array_equal(g, g[::-1])                           # symmetric
    assert abs(g.sum() - 1.0) < 1e-15                           # C-3: renormalised
    assert np.argmax(g) == r
    assert np.all(np.diff(g[: r + 1]) > 0)                      # monotone up to the centre
    # ratio of neighbouring taps is the Gaussian's, independent of the normalisation:
    # g[o+1]/g[o] = exp(-(2o+1)/(2 sigma^2))
    o = np.arange(0, r)
    np.testing.assert_allclose(g[r + 1:] / g[r:-1], np.exp(-(2 * o + 1) / (2 * sigma ** 2)), rtol=1e-13)


def test_S1_taps_golden_sigma1(oracle):
    """tests/golden/taps_sigma1.txt: hand-evaluated exp(-o^2/2)/sum for sigma=1, r=3
    (BASELINE.json configs[0]: 'taps truncated at radius ceil(3*sigma) and renormalised to sum 1')."""
    gold = np.loadtxt(os.path.join(HERE, "golden", "taps_sigma1.txt"), comments="#")
    np.testing.assert_allclose(oracle.taps(1.0), gold, rtol=0, atol=5e-9)


def test_S1_sigma_zero_is_identity(oracle):
    assert oracle.radius(0.0) == 0
    np.testing.assert_array_equal(oracle.taps(0.0), [1.0])
    d = np.random.default_rng(5).standard_normal((5, 6, 7)).astype(np.float32)
    np.testing.assert_array_equal(oracle.filter_full(d, (0, 0, 0)), d.astype(np.float64))


# ------------------------------------------------------------------------------------ filter

def test_S2_impulse_interior_is_outer_product(oracle):
    sig = (1.0, 1.5, 2.0)
    gx, gy, gz = (oracle.taps(s) for s in sig)
    rx, ry, rz = ((len(g) - 1) // 2 for g in (gx, gy, gz))
    nz, ny, nx = 2 * rz + 5, 2 * ry + 4, 2 * rx + 3
    c = (rx + 1, ry + 2, rz + 2)                        # (x,y,z) of the impulse
    d = np.zeros((nz, ny, nx), np.float32)
    d[c[2], c[1], c[0]] = 1.0
    expect = np.zeros(d.shape)
    # correlation (C-4): f[c - o] = g[o]; symmetric taps -> same thing
    expect[c[2] - rz: c[2] + rz + 1, c[1] - ry: c[1] + ry + 1, c[0] - rx: c[0] + rx + 1] = \
        gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
    for fn in (oracle.filter_direct, oracle.filter_full):
        np.testing.assert_allclose(fn(d, sig), expect, rtol=0, atol=1e-16)


def test_S2_asymmetric_probe_is_correlation_not_transposed(oracle):
    """Two impulses of different height at different offsets along each axis: catches a transposed
    axis or swapped sigma (x<->z) because the three sigmas differ."""
    sig = (1.0, 2.0, 3.0)
    d = np.zeros((40, 30, 20), np.float32)
    d[20, 15, 10] = 1.0
    f = oracle.filter_full(d, sig)
    gx, gy, gz = (oracle.taps(s) for s in sig)
    # profile through the impulse along each axis equals that axis' taps times the other centres
    np.testing.assert_allclose(f[20, 15, 10 - 3: 10 + 4], gx * gy[6] * gz[9], atol=1e-16)
    np.testing.assert_allclose(f[20, 15 - 6: 15 + 7, 10], gy * gx[3] * gz[9], atol=1e-16)
    np.testing.assert_allclose(f[20 - 9: 20 + 10, 15, 10], gz * gx[3] * gy[6], atol=1e-16)


def test_S3_impulse_at_corner_is_clipped_not_renormalised(oracle):
    sig = (1.0, 1.0, 2.0)
    gx, gy, gz = (oracle.taps(s) for s in sig)
    d = np.zeros((20, 12, 12), np.float32)
    d[0, 0, 0] = 2.0
    expect = np.zeros(d.shape)
    expect[:7, :4, :4] = 2.0 * gz[6:, None, None] * gy[None, 3:, None] * gx[None, None, 3:]
    for fn in (oracle.filter_direct, oracle.filter_full):
        np.testing.assert_allclose(fn(d, sig), expect, rtol=0, atol=1e-16)


def test_S4_constant_cube_interior_and_face_closed_form(oracle):
    sig = (1.0, 1.5, 2.0)
    c0 = 3.25
    d = np.full((30, 24, 20), c0, np.float32)
    f = oracle.filter_full(d, sig)
    taps = [oracle.taps(s) for s in sig]
    r = [(len(g) - 1) // 2 for g in taps]
    assert np.max(np.abs(f[r[2]: 30 - r[2], r[1]: 24 - r[1], r[0]: 20 - r[0]] - c0)) < 1e-14
    # faces: f = c0 * Px(x) Py(y) Pz(z), P = partial tap sum over the in-cube part (C-5)

    def partial(g, rr, n):
        return np.array([g[max(0, rr - i): min(2 * rr + 1, rr + n - i)].sum() for i in range(n)])
    px, py, pz = partial(taps[0], r[0], 20), partial(taps[1], r[1], 24), partial(taps[2], r[2], 30)
    expect = c0 * pz[:, None, None] * py[None, :, None] * px[None, None, :]
    np.testing.assert_allclose(f, expect, rtol=0, atol=1e-14)
    assert f[0, 0, 0] < 0.3 * c0          # corner really is attenuated (not renormalised)


@pytest.mark.parametrize("sig", [(1.0, 1.0, 2.0), (2.0, 1.0, 8.0), (0.0, 1.5, 0.0)])
def test_S5_separable_equals_direct_16cube(oracle, sig):
    """L1 (three 1-D passes) == L0 (Eq. 2 six-deep loop) incl. a radius larger than the cube
    (sigma_z = 8 -> r = 24 > 16)."""
    d = np.random.default_rng(11).standard_normal((16, 16, 16)).astype(np.float32)
    a = oracle.filter_direct(d, sig)
    b = oracle.filter_full(d, sig)
    assert np.max(np.abs(a - b)) < 1e-14


def test_S5b_direct_equals_numpy_einsum_definition(oracle):
    """L0 against an independent numpy evaluation of Eq. 2 on a zero-padded copy."""
    rng = np.random.default_rng(12)
    d = rng.standard_normal((9, 8, 7)).astype(np.float32)
    sig = (1.0, 1.5, 2.0)
    gx, gy, gz = (oracle.taps(s) for s in sig)
    rx, ry, rz = 3, 5, 6
    pad = np.zeros((9 + 2 * rz, 8 + 2 * ry, 7 + 2 * rx))
    pad[rz:rz + 9, ry:ry + 8, rx:rx + 7] = d
    win = np.lib.stride_tricks.sliding_window_view(pad, (2 * rz + 1, 2 * ry + 1, 2 * rx + 1))
    expect = np.einsum("zyxabc,a,b,c->zyx", win, gz, gy, gx)
    np.testing.assert_allclose(oracle.filter_direct(d, sig), expect, rtol=0, atol=1e-14)


def test_S6_flux_conservation_for_interior_support(oracle):
    sig = (1.0, 1.0, 2.0)
    rng = np.random.default_rng(13)
    d = np.zeros((40, 24, 24), np.float32)
    d[6:-6, 3:-3, 3:-3] = rng.standard_normal((28, 18, 18)).astype(np.float32)
    f = oracle.filter_full(d, sig)
    assert abs(f.sum() - d.astype(np.float64).sum()) < 1e-12 * np.abs(d).sum()


@pytest.mark.parametrize("sig", [(1.0, 1.0, 2.0), (3.0, 3.0, 8.0), (1.5, 2.5, 4.0)])
def test_S7_library_cross_check_scipy(oracle, sig):
    """scipy.ndimage.correlate1d(mode='constant', cval=0) per axis with the oracle's taps, and
    scipy's own gaussian_filter (truncate=3, mode='constant'; its radius int(3 sigma + .5) equals
    ceil(3 sigma) for every sigma in the configs)."""
    d = np.random.default_rng(14).standard_normal((40, 33, 29)).astype(np.float32)
    f = oracle.filter_full(d, sig)
    e = d.astype(np.float64)
    for ax, s in zip((2, 1, 0), sig):
        e = ndi.correlate1d(e, oracle.taps(s), axis=ax, mode="constant", cval=0.0)
    assert np.max(np.abs(f - e)) < 1e-14
    g = ndi.gaussian_filter(d.astype(np.float64), sigma=sig[::-1], truncate=3.0, mode="constant",
                            radius=[oracle.radius(s) for s in sig[::-1]])
    assert np.max(np.abs(f - g)) < 1e-13


def test_S8_gaussian_source_closed_form(oracle):
    """Continuous closed form (sanity, ~1 %): Gaussian source sigma_s filtered by sigma_f is a
    Gaussian of sqrt(ss^2+sf^2) with amplitude * prod ss/sqrt(ss^2+sf^2)."""
    ss, sf = (3.0, 3.0, 6.0), (2.0, 2.0, 4.0)
    nz, ny, nx = 96, 64, 64
    z, y, x = np.meshgrid(np.arange(nz) - 48, np.arange(ny) - 32, np.arange(nx) - 32, indexing="ij")
    d = np.exp(-0.5 * (x ** 2 / ss[0] ** 2 + y ** 2 / ss[1] ** 2 + z ** 2 / ss[2] ** 2)).astype(np.float32)
    f = oracle.filter_full(d, sf)
    amp = np.prod([a / math.sqrt(a * a + b * b) for a, b in zip(ss, sf)])
    assert abs(f[48, 32, 32] / amp - 1.0) < 0.015
    st = [math.sqrt(a * a + b * b) for a, b in zip(ss, sf)]
    assert abs(f[48, 32, 32 + 4] / f[48, 32, 32] - math.exp(-0.5 * 16 / st[0] ** 2)) < 0.01


def test_region_mode_equals_full(oracle):
    rng = np.random.default_rng(15)
    d = rng.standard_normal((50, 40, 30)).astype(np.float32)
    sig = (1.0, 2.0, 3.0)
    full = oracle.filter_full(d, sig)
    lo, hi = (5, 0, 20), (30, 17, 50)                # touches faces and interior
    (a, b) = oracle.required_input_box((30, 40, 50), [sig], (0, 0, 0), lo, hi)
    sub = d[a[2]:b[2], a[1]:b[1], a[0]:b[0]]
    reg = oracle.filter_region(sub, a, (30, 40, 50), sig, lo, hi)
    np.testing.assert_array_equal(reg, full[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]])
    with pytest.raises(ValueError):                  # sub too small must be refused, not zero-filled
        oracle.filter_region(d[25:, :, :], (0, 0, 25), (30, 40, 50), sig, lo, hi)


# ------------------------------------------------------------------------------------ statistics

@pytest.mark.parametrize("h", [(1, 2, 3), (4, 4, 8), (20, 3, 40), (0, 0, 0)])
def test_S9_box_sums_equal_brute_force(oracle, h):
    c = np.random.default_rng(21).standard_normal((14, 12, 10))
    a = oracle.threshold_brute(c, h, 1.5)
    b = oracle.threshold_full(c, h, 1.5)
    assert np.max(np.abs(a.mean - b.mean)) < 1e-13
    # compare variances: sqrt amplifies the 1e-16 rounding of the prefix sums where var ~ 0 (h = 0)
    assert np.max(np.abs(a.std ** 2 - b.std ** 2)) < 1e-13
    ok = a.std > 1e-3
    assert np.max(np.abs(a.std - b.std)[ok], initial=0.0) < 1e-12
    assert np.max(np.abs(a.thr - b.thr)[ok], initial=0.0) < 1e-11
    near = np.abs(c - a.thr) < 1e-6
    assert np.array_equal(a.mask[~near], b.mask[~near])


def test_S9b_brute_equals_library_box_sums(oracle):
    """L0 window scan vs scipy.ndimage.uniform_filter: zero-padded sums / clipped counts (C-7)."""
    c = np.random.default_rng(22).standard_normal((13, 11, 9))
    h = (2, 3, 4)
    size = (2 * h[2] + 1, 2 * h[1] + 1, 2 * h[0] + 1)
    nwin = np.prod(size)
    s1 = ndi.uniform_filter(c, size=size, mode="constant") * nwin
    s2 = ndi.uniform_filter(c * c, size=size, mode="constant") * nwin
    n = ndi.uniform_filter(np.ones_like(c), size=size, mode="constant") * nwin
    m = s1 / n
    sd = np.sqrt(np.maximum(s2 / n - m * m, 0.0))
    a = oracle.threshold_brute(c, h, 4.0)
    np.testing.assert_allclose(a.mean, m, atol=1e-12)
    np.testing.assert_allclose(a.std, sd, atol=1e-12)
    np.testing.assert_allclose(a.thr, m + 4.0 * sd, atol=1e-11)


def test_S10_linear_ramp_closed_form(oracle):
    """f = a*x: interior m = a x, var = a^2 h(h+1)/3 (population, C-8); at x=0 the clipped window
    has h+1 samples: m = a h/2, var = a^2 h(h+2)/12."""
    a_, h = 0.37, 5
    nx = 40
    c = np.broadcast_to(a_ * np.arange(nx, dtype=np.float64), (6, 7, nx)).copy()
    for fn in (oracle.threshold_brute, oracle.threshold_full):
        st = fn(c, (h, 2, 1), 4.0)
        xs = np.arange(h, nx - h)
        np.testing.assert_allclose(st.mean[3, 3, h: nx - h], a_ * xs, atol=1e-12)
        np.testing.assert_allclose(st.std[3, 3, h: nx - h], a_ * math.sqrt(h * (h + 1) / 3.0), atol=1e-12)
        assert abs(st.mean[0, 0, 0] - a_ * h / 2.0) < 1e-12
        assert abs(st.std[0, 0, 0] - a_ * math.sqrt(h * (h + 2) / 12.0)) < 1e-12
        # sample (n-1) variance would give a*sqrt(h(h+1)/3 * n/(n-1)): make sure we are not that
        n = 2 * h + 1
        assert abs(st.std[3, 3, 20] - a_ * math.sqrt(h * (h + 1) / 3.0 * n / (n - 1))) > 1e-3


def test_S11_single_spike_closed_form(oracle):
    """Spike A on zeros, window n: z = sqrt(n-1) at the spike, -1/sqrt(n-1) elsewhere in the window;
    set iff sqrt(n-1) > k (self-inclusion, population variance, strict >)."""
    h = (4, 4, 8)
    n = 9 * 9 * 17
    assert n == 1377
    c = np.zeros((40, 24, 24))
    A = 2.5
    c[20, 12, 12] = A
    for k, expect_set in ((4.0, True), (37.0, True), (37.2, False)):
        st = oracle.threshold_full(c, h, k)
        z = (c - st.mean) / np.where(st.std > 0, st.std, 1.0)
        assert abs(z[20, 12, 12] - math.sqrt(n - 1)) < 1e-9
        assert abs(z[20, 12, 13] + 1.0 / math.sqrt(n - 1)) < 1e-12
        assert abs(math.sqrt(n - 1) - 37.094) < 1e-3
        assert bool(st.mask[20, 12, 12]) == expect_set
        assert st.mask.sum() == (1 if expect_set else 0)
    # far from the spike: window all zeros -> std 0, nothing selected
    st = oracle.threshold_full(c, h, 4.0)
    assert st.std[0, 0, 0] == 0.0 and st.mask[0, 0, 0] == 0


def test_S12_constant_cube_selects_nothing(oracle):
    c = np.full((12, 10, 9), 0.1)              # 0.1 is inexact in binary: S2/n - m^2 may round < 0
    for fn in (oracle.threshold_brute, oracle.threshold_full):
        st = fn(c, (2, 2, 3), 4.0)
        assert np.all(st.std < 1e-8) and np.all(st.std >= 0)
    st = oracle.threshold_full(np.full((12, 10, 9), 0.5), (2, 2, 3), 4.0)
    assert st.mask.sum() == 0 and np.all(st.std == 0.0)


def test_S13_white_noise_false_positive_rate(oracle):
    """N(0,1) cube fed directly to the threshold stage, box (8,8,16), k = 4: expected set fraction
    Q(4) = 3.167e-5 (BASELINE.json north_star: 'near its Gaussian expectation')."""
    rng = np.random.default_rng(31)
    n = 160
    c = rng.standard_normal((n, n, n))
    st = oracle.threshold_full(c, (8, 8, 16), 4.0)
    q4 = 0.5 * math.erfc(4.0 / math.sqrt(2.0))
    expect = q4 * c.size
    got = int(st.mask.sum())
    assert abs(got - expect) < 4.0 * math.sqrt(expect) + 0.05 * expect, (got, expect)
    # local estimates themselves: mean ~ 0 +- 1/sqrt(n_win), std ~ 1
    nwin = 17 * 17 * 33
    inner = (slice(40, 120),) * 3
    assert abs(st.std[inner].mean() - 1.0) < 5e-3
    assert abs(st.mean[inner].std() - 1.0 / math.sqrt(nwin)) < 0.3 / math.sqrt(nwin)


def test_S14_power_of_two_scale_invariance(oracle):
    from paper_1507_04941_b200 import synth
    d = synth.make_cube((48, 32, 32), seed=7, n_sources=4, device="cpu").numpy()
    a = oracle.find_full(d, [(1, 1, 2)], (3, 3, 6), 3.0)
    b = oracle.find_full(2.0 * d, [(1, 1, 2)], (3, 3, 6), 3.0)
    np.testing.assert_array_equal(2.0 * a.scales[0].f, b.scales[0].f)
    np.testing.assert_array_equal(a.mask, b.mask)
    assert a.count == b.count and a.count > 0


def test_S15_multiscale_or_halo_and_count(oracle):
    from paper_1507_04941_b200 import synth
    d = synth.make_cube((64, 40, 40), seed=9, n_sources=6, device="cpu").numpy()
    sig = [(1, 1, 2), (2, 2, 4)]
    h, k = (3, 3, 6), 2.5
    full = oracle.find_full(d, sig, h, k)
    per = [oracle.find_full(d, [s], h, k) for s in sig]
    np.testing.assert_array_equal(full.mask, per[0].mask | per[1].mask)
    assert full.count == int(full.mask.sum()) and full.count > 0
    assert per[0].count != per[1].count                   # the two scales do differ
    halo = (4, 5, 6)
    hal = oracle.find_full(d, sig, h, k, halo=halo)
    core = (slice(6, -6), slice(5, -5), slice(4, -4))
    np.testing.assert_array_equal(hal.mask[core], full.mask[core])    # same standalone cube (C-11)
    hal.mask[core] = 0
    assert hal.mask.sum() == 0                                        # halo voxels forced to 0
    # region mode of the whole pipeline
    lo, hi = (8, 0, 10), (40, 25, 50)
    a, b = oracle.required_input_box((40, 40, 64), sig, h, lo, hi)
    reg = oracle.find_region(d[a[2]:b[2], a[1]:b[1], a[0]:b[0]], a, (40, 40, 64), sig, h, k, lo, hi, halo)
    ref = oracle.find_full(d, sig, h, k, halo=halo)
    sl = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
    np.testing.assert_array_equal(reg.mask, ref.mask[sl])
    # region mode with lo != 0 reproduces the full-cube VALUES too (filtered data, mean, std, threshold), not only
    # the mask: a window clipped to the brick instead of the cube, or a shifted origin, would show here
    for rs, fs in zip(reg.scales, ref.scales):
        np.testing.assert_allclose(rs.f, fs.f[sl], rtol=0, atol=1e-14)
        np.testing.assert_allclose(rs.stats.mean, fs.stats.mean[sl], rtol=0, atol=1e-14)
        np.testing.assert_allclose(rs.stats.std, fs.stats.std[sl], rtol=1e-12, atol=1e-15)
        np.testing.assert_allclose(rs.stats.thr, fs.stats.thr[sl], rtol=0, atol=1e-13)
        np.testing.assert_array_equal(rs.stats.mask, fs.stats.mask[sl])


# ---------------------------------------------------------------------------------- Eq. 1 (weighted), NEXT-1

def _wcube(shape, seed):
    rng = np.random.default_rng(seed)
    d = rng.standard_normal(shape).astype(np.float32)
    w = rng.uniform(0.25, 2.0, shape).astype(np.float32)
    return d, w


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("sigma3", [(1.0, 1.0, 2.0), (0.0, 1.5, 1.0), (1.0, 2.0, 5.0)])
def test_W1_weighted_separable_equals_direct(oracle, mode, sigma3):
    """L1 (separable numerator / box or filtered denominator) == L0 (Eq. 1 as a six-deep loop),
    including a radius larger than the cube (sigma_z = 5 -> r = 15 > 14)."""
    d, w = _wcube((14, 10, 12), 7)
    a = oracle.wfilter_full(d, w, sigma3, mode)
    b = oracle.wfilter_direct(d, w, sigma3, mode)
    assert np.max(np.abs(a - b)) <= 1e-13 * max(1.0, np.max(np.abs(b)))


def test_W2_unit_weights(oracle):
    """w == 1: the printed denominator counts the support voxels inside the cube, so c_w = c_u / n
    (n = 7*7*13 in the interior: the property reading C-16 notes); mode 1 divides by the partial tap sums
    instead, so c_w = c_u in the interior."""
    rng = np.random.default_rng(11)
    d = rng.standard_normal((30, 16, 18)).astype(np.float32)
    w = np.ones_like(d)
    sig = (1.0, 1.0, 2.0)
    cu = oracle.filter_full(d, sig)
    r = [oracle.radius(s) for s in sig]
    nz, ny, nx = d.shape
    cnt = [np.array([min(c + rr, n - 1) - max(c - rr, 0) + 1 for c in range(n)], dtype=np.float64)
           for n, rr in zip((nx, ny, nz), r)]
    n3 = cnt[2][:, None, None] * cnt[1][None, :, None] * cnt[0][None, None, :]
    c0 = oracle.wfilter_full(d, w, sig, 0)
    assert np.max(np.abs(c0 - cu / n3)) <= 1e-15
    assert n3[15, 8, 9] == 7 * 7 * 13
    c1 = oracle.wfilter_full(d, w, sig, 1)
    inner = (slice(r[2], nz - r[2]), slice(r[1], ny - r[1]), slice(r[0], nx - r[0]))
    assert np.max(np.abs(c1[inner] - cu[inner])) <= 1e-14
    # at a face mode 1 renormalises by the partial tap sum (closed form, cf. S4)
    g = [oracle.taps(s) for s in sig]
    px = np.array([g[0][max(0, r[0] - x):min(2 * r[0] + 1, r[0] + nx - x)].sum() for x in range(nx)])
    assert abs(c1[15, 8, 0] - cu[15, 8, 0] / px[0]) <= 1e-14


@pytest.mark.parametrize("mode", [0, 1])
def test_W3_weight_scale_invariance(oracle, mode):
    """Eq. 1 is a ratio that is homogeneous of degree 0 in w: w -> 4 w changes nothing (power of two: exactly)."""
    d, w = _wcube((12, 12, 12), 3)
    a = oracle.wfilter_full(d, w, (1.0, 1.0, 2.0), mode)
    b = oracle.wfilter_full(d, 4.0 * w, (1.0, 1.0, 2.0), mode)
    assert np.array_equal(a, b)


@pytest.mark.parametrize("mode", [0, 1])
def test_W4_zero_weight_removes_a_voxel(oracle, mode):
    """A voxel with w = 0 contributes to neither sum: a huge spike there is invisible, and the result
    equals the one with the spike removed from d."""
    d, w = _wcube((16, 12, 12), 5)
    w[8, 6, 5] = 0.0
    d2 = d.copy()
    d2[8, 6, 5] = 1e6
    a = oracle.wfilter_full(d, w, (1.0, 1.0, 2.0), mode)
    b = oracle.wfilter_full(d2, w, (1.0, 1.0, 2.0), mode)
    assert np.array_equal(a, b)
    # all-zero weights: 0 / 0 -> 0
    z = oracle.wfilter_full(d, np.zeros_like(w), (1.0, 1.0, 2.0), mode)
    assert not z.any()


@pytest.mark.parametrize("mode", [0, 1])
def test_W5_weighted_against_scipy(oracle, mode):
    """Library special case: numerator = correlate1d chain on d*w (mode='constant'), denominator =
    correlate1d chain on w with the taps (mode 1) or with ones (mode 0)."""
    from scipy import ndimage
    d, w = _wcube((20, 14, 16), 9)
    sig = (1.0, 2.0, 3.0)
    num = (d.astype(np.float64) * w.astype(np.float64))
    den = w.astype(np.float64)
    for ax, s in zip((2, 1, 0), sig):
        g = oracle.taps(s)
        num = ndimage.correlate1d(num, g, axis=ax, mode="constant", cval=0.0)
        den = ndimage.correlate1d(den, g if mode else np.ones_like(g), axis=ax, mode="constant", cval=0.0)
    ref = num / den
    a = oracle.wfilter_full(d, w, sig, mode)
    assert np.max(np.abs(a - ref)) <= 1e-13 * np.max(np.abs(ref))


def test_W6_constant_data_any_weights(oracle):
    """d == c: mode 1 returns c wherever any weight is positive (a weighted mean of a constant), for ANY
    weights; mode 0 returns c * sum f w / sum w."""
    rng = np.random.default_rng(2)
    w = rng.uniform(0.1, 3.0, (12, 10, 14)).astype(np.float32)
    d = np.full_like(w, 2.5)
    c1 = oracle.wfilter_full(d, w, (1.0, 1.0, 2.0), 1)
    assert np.max(np.abs(c1 - 2.5)) <= 1e-14


# ---------------------------------------------------------------------------------- Eq. 2, arbitrary filter (NEXT-2)

def test_G1_general_equals_outer_product_path(oracle):
    """With f = gz (x) gy (x) gx the general routine is the L0 routine of S5 (and hence the separable one)."""
    rng = np.random.default_rng(21)
    d = rng.standard_normal((14, 12, 16)).astype(np.float32)
    sig = (1.0, 1.5, 2.0)
    g = [oracle.taps(s) for s in sig]
    f = g[2][:, None, None] * g[1][None, :, None] * g[0][None, None, :]
    a = oracle.filter_general(d, f)
    b = oracle.filter_direct(d, sig)
    assert np.max(np.abs(a - b)) <= 1e-14


def test_G2_general_impulse_orientation(oracle):
    """Eq. 2 is printed as a correlation, c[v] = sum_o d[v+o] f[o]: an impulse at p gives c[p - o] = f[o],
    i.e. the FLIPPED filter around p.  An asymmetric random f tells correlation from convolution and
    catches transposed axes (unequal radii)."""
    rng = np.random.default_rng(22)
    f = rng.standard_normal((5, 3, 7))            # rz = 2, ry = 1, rx = 3
    d = np.zeros((11, 9, 13), np.float32)
    p = (5, 4, 6)
    d[p] = 1.0
    c = oracle.filter_general(d, f)
    for oz in range(-2, 3):
        for oy in range(-1, 2):
            for ox in range(-3, 4):
                assert c[p[0] - oz, p[1] - oy, p[2] - ox] == f[oz + 2, oy + 1, ox + 3]
    assert np.count_nonzero(c) == np.count_nonzero(f)


def test_G3_general_against_scipy_correlate(oracle):
    """Library special case: scipy.ndimage.correlate(mode='constant') is Eq. 2 with zero padding."""
    rng = np.random.default_rng(23)
    d = rng.standard_normal((12, 10, 15)).astype(np.float32)
    f = rng.standard_normal((7, 5, 3))
    ref = ndi.correlate(d.astype(np.float64), f, mode="constant", cval=0.0)
    a = oracle.filter_general(d, f)
    assert np.max(np.abs(a - ref)) <= 1e-13
    # a radius larger than the cube along z
    f2 = rng.standard_normal((29, 1, 3))
    ref2 = ndi.correlate(d.astype(np.float64), f2, mode="constant", cval=0.0)
    assert np.max(np.abs(oracle.filter_general(d, f2) - ref2)) <= 1e-13


# ------------------------------------------------------------------------------------ NEXT-4: object labelling (C-19)

def _mask(shape, voxels):
    m = np.zeros(shape, np.uint8)
    for z, y, x in voxels:
        m[z, y, x] = 1
    return m


def test_L1_hand_built_masks(oracle):
    """26-connectivity on masks whose components can be counted by eye; a wrong neighbourhood (6 or 18) or a wrong
    axis stride fails one of them."""
    sh = (5, 6, 7)
    lin = lambda z, y, x: x + 7 * (y + 6 * z)
    cases = [
        ([], 0),
        ([(0, 0, 0)], 1),
        ([(1, 1, 1), (2, 2, 2)], 1),                       # corner contact only: one object (two under 6 / 18)
        ([(1, 1, 1), (1, 2, 2)], 1),                       # edge contact only (two under 6-connectivity)
        ([(1, 1, 1), (1, 1, 3)], 2),                       # a gap of one voxel along x
        ([(0, 0, 6), (0, 1, 0)], 2),                       # end of one row / start of the next: adjacent in memory only
        ([(0, 5, 3), (1, 0, 3)], 2),                       # last row of a plane / first row of the next plane
        ([(0, 0, 0), (1, 1, 1), (2, 2, 2), (3, 3, 3), (4, 4, 4)], 1),          # a space diagonal
        ([(2, y, x) for y in range(1, 5) for x in range(1, 6) if y in (1, 4) or x in (1, 5)], 1),      # a ring
        ([(2, y, x) for y in range(1, 5) for x in range(1, 6) if y in (1, 4) or x in (1, 5)] + [(2, 2, 3)], 1),
        ([(4, 5, 6), (0, 0, 0), (2, 3, 3)], 3),
    ]
    for vox, expect in cases:
        m = _mask(sh, vox)
        labels, n = oracle.label26(m)
        assert n == expect, (vox, n)
        assert np.array_equal(labels != 0, m != 0)
        for z, y, x in vox:                                # label = 1 + smallest index of the voxel's component
            comp = np.argwhere(labels == labels[z, y, x])
            assert labels[z, y, x] == 1 + min(lin(*c) for c in comp)


def test_L2_scipy_label_partition(oracle):
    """Library cross-check: scipy.ndimage.label with the full 3 x 3 x 3 structure gives the same partition."""
    ndi = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(7)
    for shape, dens in [((9, 11, 13), 0.08), ((16, 16, 16), 0.15), ((3, 40, 5), 0.3), ((1, 1, 50), 0.5)]:
        m = (rng.random(shape) < dens).astype(np.uint8)
        labels, n = oracle.label26(m)
        ref, nref = ndi.label(m, structure=np.ones((3, 3, 3)))
        assert n == nref
        # same partition: the map oracle label -> scipy label is a bijection on the set voxels
        pairs = set(zip(labels[m != 0].tolist(), ref[m != 0].tolist()))
        assert len(pairs) == n and len({a for a, _ in pairs}) == n and len({b for _, b in pairs}) == n


def test_L3_brute_force_closure(oracle):
    """Definition level: components as the transitive closure of 'Chebyshev distance 1' on tiny masks."""
    rng = np.random.default_rng(11)
    for _ in range(20):
        shape = tuple(rng.integers(1, 6, 3))
        m = (rng.random(shape) < 0.35).astype(np.uint8)
        pts = np.argwhere(m != 0)
        comp = list(range(len(pts)))
        changed = True
        while changed:
            changed = False
            for i in range(len(pts)):
                for j in range(len(pts)):
                    if np.max(np.abs(pts[i] - pts[j])) <= 1 and comp[i] != comp[j]:
                        comp[i] = comp[j] = min(comp[i], comp[j])
                        changed = True
        labels, n = oracle.label26(m)
        assert n == len(set(comp))
        for i in range(len(pts)):
            for j in range(len(pts)):
                same = labels[tuple(pts[i])] == labels[tuple(pts[j])]
                assert same == (comp[i] == comp[j])


def test_L4_invariances(oracle):
    """The count is invariant under flips and axis permutations; a full cube is one object; an isolated-voxel lattice
    of spacing 2 has as many objects as voxels."""
    rng = np.random.default_rng(3)
    m = (rng.random((10, 12, 14)) < 0.1).astype(np.uint8)
    _, n = oracle.label26(m)
    for t in (m[::-1], m[:, ::-1], m[:, :, ::-1], m.transpose(2, 0, 1), m.transpose(1, 2, 0)):
        assert oracle.label26(np.ascontiguousarray(t))[1] == n
    assert oracle.label26(np.ones((4, 5, 6), np.uint8))[1] == 1
    lat = np.zeros((7, 7, 7), np.uint8)
    lat[::2, ::2, ::2] = 1
    assert oracle.label26(lat)[1] == 64
