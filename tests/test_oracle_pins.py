"""Pins for the CPU oracle: every step is checked against something other than
itself -- hand values from the paper's equations, closed forms, invariants,
library routines on special cases, and brute force on tiny inputs.

Citations are PAPER.md lines (arXiv:1510.01815).  Hand values used here are also
listed, with their derivations, in tests/golden/eq_hand_values.txt.
"""
import math
import os

import numpy as np
import pytest
from scipy import signal

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _row(xo=0.0, yo=0.0, pa=0.0, inc=0.0, vsys=0.0, vt=200.0, rt=3.0, sig=40.0, r0=4.0, i0=1.0):
    return [xo, yo, pa, inc, vsys, vt, rt, sig, r0, i0]


# ------------------------------------------------------------------ taps ----

def test_fwhm_sigma_closed_form(oracle):
    # FWHM = 2 sqrt(2 ln 2) sigma: a Gaussian of sigma 1 has FWHM 2.354820045...
    assert oracle.fwhm_to_sigma(2.3548200450309493) == pytest.approx(1.0, abs=1e-15)


def test_gaussian_taps(oracle):
    sigma = 1.2739827  # FWHM 3 px
    t = oracle.gaussian_taps(sigma)
    R = (t.size - 1) // 2
    assert R == math.ceil(4 * sigma) == 6                      # A10
    assert t.sum() == pytest.approx(1.0, abs=1e-15)            # A9
    assert np.array_equal(t, t[::-1])                          # symmetric
    # ratios of an unnormalised Gaussian survive the normalisation (eq. 9, :166)
    assert t[R + 1] / t[R] == pytest.approx(math.exp(-0.5 / sigma ** 2), rel=1e-14)
    assert t[R + 3] / t[R] == pytest.approx(math.exp(-4.5 / sigma ** 2), rel=1e-14)
    # sigma <= 0 is the delta kernel
    assert np.array_equal(oracle.gaussian_taps(0.0), [1.0])


def test_gaussian_psf_image_is_outer_product_with_fine_sigma(oracle):
    img = oracle.psf_gaussian_image(2.5, 2)          # A14: sigma_f = u * sigma
    t = oracle.gaussian_taps(2 * oracle.fwhm_to_sigma(2.5))
    assert img.shape == (t.size, t.size) and t.size == 2 * 9 + 1
    assert np.allclose(img, np.outer(t, t), rtol=0, atol=1e-18)
    assert img.sum() == pytest.approx(1.0, abs=1e-14)


def test_moffat_image(oracle):
    img = oracle.psf_moffat_image(4.0, 2.5, 15)
    assert img.sum() == pytest.approx(1.0, abs=1e-14)
    # half maximum at radius FWHM/2 = 2 fine pixels, by the definition of FWHM
    assert img[7, 9] / img[7, 7] == pytest.approx(0.5, rel=1e-13)
    assert img[5, 7] / img[7, 7] == pytest.approx(0.5, rel=1e-13)
    # profile value at (3,4) -> r = 5: [1 + 25/alpha^2]^-2.5, alpha = 2/sqrt(2^0.4 - 1)
    alpha2 = 4.0 / (2.0 ** 0.4 - 1.0)
    assert img[7 + 4, 7 + 3] / img[7, 7] == pytest.approx((1 + 25 / alpha2) ** -2.5, rel=1e-13)
    assert math.sqrt(alpha2) == pytest.approx(3.53826, abs=1e-5)
    assert np.allclose(img, img.T) and np.allclose(img, img[::-1, ::-1])
    # the shared input generator makes the same image up to its float32 storage
    from paper_1510_01815_b200 import workloads
    w = workloads.moffat_image(4.0, 2.5, 15).astype(np.float64)
    assert np.allclose(w / w.sum(), img, rtol=2e-7)


# -------------------------------------------------- geometry, eq. 1-8 ----

def test_geometry_pa0_major_axis_is_plus_y(oracle):
    # eq. 1-2 with PA = 0: x_e = (y - y_o), y_e = -(x - x_o)
    # arctan curve at r = r_t: V_rot = (2/pi) V_t atan(1) = V_t / 2 (eq. 6, :120)
    # V_t = 200, i = 30 deg, on the major axis (cos theta = 1): v - V_sys = 100 * 0.5 = 50
    p = _row(xo=10, yo=10, pa=0, inc=30, vsys=7, vt=200, rt=3, r0=4, i0=2.5)
    I, v = oracle.disc_point(p, oracle.RC_ARCTAN, 10.0, 13.0)
    assert v == pytest.approx(7 + 50.0, abs=1e-12)
    assert I == pytest.approx(2.5 * math.exp(-3.0 / 4.0), rel=1e-14)     # eq. 5 (:110)
    I, v = oracle.disc_point(p, oracle.RC_ARCTAN, 10.0, 7.0)             # receding/approaching
    assert v == pytest.approx(7 - 50.0, abs=1e-12)
    # minor axis: x_e = 0 => cos theta = 0 => v = V_sys; r = |dx| / cos i (eq. 3, :92)
    I, v = oracle.disc_point(p, oracle.RC_ARCTAN, 12.0, 10.0)
    assert v == pytest.approx(7.0, abs=1e-12)
    assert I == pytest.approx(2.5 * math.exp(-(2.0 / math.cos(math.radians(30))) / 4.0), rel=1e-14)
    # I(r0) = I0 / e
    I, _ = oracle.disc_point(p, oracle.RC_ARCTAN, 10.0, 14.0)
    assert I == pytest.approx(2.5 / math.e, rel=1e-14)


def test_geometry_general_pa_hand_points(oracle):
    # PA = 30 deg.  Sky offset a*(-sin PA, cos PA): eq. 1 gives x_e = a, eq. 2 gives y_e = 0.
    # Sky offset b*(-cos PA, -sin PA): x_e = 0, y_e = b  => r = b / cos i.
    pa, inc = 30.0, 60.0
    s, c = math.sin(math.radians(pa)), math.cos(math.radians(pa))
    p = _row(xo=5, yo=-2, pa=pa, inc=inc, vsys=0, vt=100, rt=2, r0=3, i0=1)
    a = 2.0
    I, v = oracle.disc_point(p, oracle.RC_ARCTAN, 5 - s * a, -2 + c * a)
    assert I == pytest.approx(math.exp(-a / 3.0), rel=1e-13)
    assert v == pytest.approx(100 * 0.5 * math.sin(math.radians(60)), rel=1e-13)  # r = r_t, cos th = 1
    b = 1.5
    I, v = oracle.disc_point(p, oracle.RC_ARCTAN, 5 - c * b, -2 - s * b)
    assert I == pytest.approx(math.exp(-(b / 0.5) / 3.0), rel=1e-13)     # cos 60 = 0.5
    assert abs(v) < 1e-12
    # sign of the x_e term: opposite side of the major axis flips the velocity
    _, v2 = oracle.disc_point(p, oracle.RC_ARCTAN, 5 + s * a, -2 - c * a)
    assert v2 == pytest.approx(-100 * 0.5 * math.sin(math.radians(60)), rel=1e-13)
    # 45 deg off the major axis in the disc plane, face-on-corrected: x_e = y_e/cos i
    # => cos theta = 1/sqrt 2, r = sqrt 2 * x_e
    xe = 1.0
    ye = xe * 0.5
    x = 5 - s * xe - c * ye
    y = -2 + c * xe - s * ye
    I, v = oracle.disc_point(p, oracle.RC_ARCTAN, x, y)
    r = math.sqrt(2.0)
    assert I == pytest.approx(math.exp(-r / 3.0), rel=1e-13)
    assert v == pytest.approx((2 / math.pi) * 100 * math.atan(r / 2.0)
                              * math.sin(math.radians(60)) / math.sqrt(2.0), rel=1e-13)


def test_ramp_curve_and_centre(oracle):
    # A7: V_t min(r/r_t, 1); A8: r = 0 -> v = V_sys
    p = _row(xo=0, yo=0, pa=0, inc=30, vsys=3, vt=120, rt=4)
    _, v = oracle.disc_point(p, oracle.RC_RAMP, 0.0, 2.0)
    assert v == pytest.approx(3 + 120 * 0.5 * 0.5, abs=1e-12)
    _, v = oracle.disc_point(p, oracle.RC_RAMP, 0.0, 4.0)
    assert v == pytest.approx(3 + 120 * 0.5, abs=1e-12)
    _, v = oracle.disc_point(p, oracle.RC_RAMP, 0.0, 9.0)
    assert v == pytest.approx(3 + 120 * 0.5, abs=1e-12)
    for rc in (oracle.RC_ARCTAN, oracle.RC_RAMP):
        I, v = oracle.disc_point(p, rc, 0.0, 0.0)
        assert v == 3.0 and I == 1.0


def test_grid_conventions(oracle):
    # A1: u = 1 sample sits on the integer; u = 2 samples at j -+ 0.25
    assert oracle.fine_coord(5, 1) == 5.0
    assert oracle.fine_coord(10, 2) == 4.75 and oracle.fine_coord(11, 2) == 5.25
    assert oracle.fine_coord(-1, 2) == -0.75
    # A2: band symmetric about v_center
    g = oracle.Grid(nx=1, ny=1, nv=4, dv=10.0, v_center=100.0)
    assert np.array_equal(g.channel_velocities(), [85.0, 95.0, 105.0, 115.0])


def test_domain_rule(oracle):
    ok = _row(inc=40)
    assert oracle.row_valid(ok)
    for ix, bad in ((7, 0.0), (7, -1.0), (8, 0.0), (6, 0.0), (9, 0.0), (3, 90.0), (0, math.nan),
                    (5, math.inf)):
        p = list(ok)
        p[ix] = bad
        assert not oracle.row_valid(p)


# ----------------------------------------- line + moments, delta kernels ----

def test_delta_kernels_give_eq8_sigma0_and_eq5(oracle):
    """PSF and LSF deltas, u = 1: m1 = eq. 8, m2 = sigma0, m0 = I(r) for a line that is narrow
    relative to the band but resolved by the channels (sigma0/dv = 1.33)."""
    g = oracle.Grid(nx=12, ny=9, nv=96, dv=30.0, v_center=5.0)
    p = _row(xo=5.3, yo=4.1, pa=37, inc=55, vsys=12, vt=200, rt=3, sig=40, r0=4, i0=1.7)
    m0, m1, m2 = oracle.model_maps(g, p)
    for y in range(9):
        for x in range(12):
            I, v = oracle.disc_point(p, 0, x, y)
            assert m1[y, x] == pytest.approx(v, abs=1e-9)
            assert m2[y, x] == pytest.approx(40.0, abs=1e-8)
            assert m0[y, x] == pytest.approx(I, rel=1e-8)


def test_line_is_flux_normalised_gaussian(oracle):
    # A3: cube value at channel c = I dv /(sigma0 sqrt(2 pi)) exp(-(v_c - v_los)^2/(2 sigma0^2))
    g = oracle.Grid(nx=1, ny=1, nv=5, dv=20.0, v_center=0.0)
    p = _row(xo=0, yo=0, vsys=10.0, sig=25.0, i0=3.0)
    cube = oracle.model_cube(g, p)[:, 0, 0]
    peak = 3.0 * 20.0 / (25.0 * math.sqrt(2 * math.pi))
    vel = [-40.0, -20.0, 0.0, 20.0, 40.0]
    for c, v in zip(cube, vel):
        assert c == pytest.approx(peak * math.exp(-0.5 * ((v - 10.0) / 25.0) ** 2), rel=1e-14)


def test_lsf_adds_variance(oracle):
    """Discrete convolution adds variances exactly: m2^2 = Var(line) + Var(L taps) dv^2."""
    dv, sig0, sig_l = 30.0, 40.0, 25.0
    taps = oracle.gaussian_taps(sig_l / dv)
    R = (taps.size - 1) // 2
    var_taps = float(np.sum(taps * (np.arange(-R, R + 1) ** 2))) * dv * dv
    g0 = oracle.Grid(nx=3, ny=3, nv=128, dv=dv)
    g1 = oracle.Grid(nx=3, ny=3, nv=128, dv=dv, lsf=taps)
    p = _row(xo=1, yo=1, pa=20, inc=40, vsys=-8)
    a0, a1, a2 = oracle.model_maps(g0, p)
    b0, b1, b2 = oracle.model_maps(g1, p)
    assert np.allclose(b2 ** 2, a2 ** 2 + var_taps, rtol=1e-11)
    assert np.allclose(b1, a1, atol=1e-9) and np.allclose(b0, a0, rtol=1e-12)
    # and close to the continuum value sqrt(sigma0^2 + sigma_LSF^2) (tap truncation ~ 6e-5)
    assert b2[1, 1] == pytest.approx(math.hypot(sig0, sig_l), rel=2e-5)


# ----------------------------------------------------------- convolution ----

def _brute_full_conv3d(vol, ker):
    """Definition of the 3-D convolution, zero boundary, full output: six nested loops."""
    Z, Y, X = vol.shape
    kz, ky, kx = ker.shape
    out = np.zeros((Z + kz - 1, Y + ky - 1, X + kx - 1))
    for z in range(Z):
        for y in range(Y):
            for x in range(X):
                for a in range(kz):
                    for b in range(ky):
                        for c in range(kx):
                            out[z + a, y + b, x + c] += vol[z, y, x] * ker[a, b, c]
    return out


def test_convolution_against_brute_force_8x8x8(oracle):
    rng = np.random.default_rng(7)
    vol = rng.random((8, 8, 8))
    L = rng.random(3)                 # asymmetric on purpose (A11: true convolution)
    Pk = rng.random((5, 5))
    ker = L[:, None, None] * Pk[None, :, :]   # PSF kernel = LSF x PSF
    want = _brute_full_conv3d(vol, ker)
    pad = np.pad(vol, ((2, 2), (4, 4), (4, 4)))
    got = oracle.conv_psf(oracle.conv_lsf(pad, L), Pk)
    assert got.shape == want.shape == (10, 12, 12)
    assert np.allclose(got, want, rtol=0, atol=1e-13)
    assert got.sum() == pytest.approx(vol.sum() * ker.sum(), rel=1e-13)


def test_impulse_response_is_the_kernel(oracle):
    rng = np.random.default_rng(8)
    L, Pk = rng.random(5), rng.random((3, 3))
    imp = np.zeros((9, 7, 7))
    imp[4, 3, 3] = 1.0
    out = oracle.conv_psf(oracle.conv_lsf(imp, L), Pk)      # valid: (5, 5, 5)
    # out[k, b, a] = L[k + 4 - 4]... impulse at (4,3,3): out[k,b,a] = L[4-k] * P[2+... ]
    # A true convolution centred on the impulse reproduces the kernel itself around it.
    full = oracle.conv_psf(oracle.conv_lsf(np.pad(imp, ((4, 4), (2, 2), (2, 2))), L), Pk)
    assert np.allclose(full[4:9, 3:6, 3:6], L[:, None, None] * Pk[None], atol=1e-15)
    assert np.count_nonzero(full) == 5 * 9
    assert out.shape == (5, 5, 5)


def test_convolution_matches_library_routines(oracle):
    rng = np.random.default_rng(9)
    cube = rng.random((6, 11, 13))
    Pk = rng.random((5, 5))
    L = rng.random(3)
    got = oracle.conv_psf(cube, Pk)
    for c in range(6):
        assert np.allclose(got[c], signal.convolve2d(cube[c], Pk, mode="valid"), atol=1e-13)
    got = oracle.conv_lsf(cube, L)
    for y in range(11):
        for x in range(13):
            assert np.allclose(got[:, y, x], np.convolve(cube[:, y, x], L, mode="valid"),
                               atol=1e-14)


# ----------------------------------------- down-sample, moments, chi^2 ----

def test_downsample(oracle):
    const = np.full((2, 6, 6), 3.25)
    assert np.array_equal(oracle.downsample(const, 3), np.full((2, 2, 2), 3.25))
    yy, xx = np.mgrid[0:4, 0:6].astype(float)
    ramp = (10 * yy + xx)[None]
    out = oracle.downsample(ramp, 2)
    # block (Y, X) averages x in {2X, 2X+1} -> 2X + 0.5 and y likewise
    want = 10 * (2 * np.arange(2)[:, None] + 0.5) + (2 * np.arange(3)[None, :] + 0.5)
    assert np.allclose(out[0], want, atol=1e-14)


def test_moments_two_spikes(oracle):
    vel = np.array([-30.0, -10.0, 10.0, 30.0, 50.0])
    spec = np.zeros((5, 1))
    a, b = 2.0, 6.0
    spec[1, 0], spec[4, 0] = a, b
    m0, m1, m2 = oracle.moments(spec, vel)
    assert m0[0] == 8.0
    assert m1[0] == pytest.approx((a * -10 + b * 50) / 8.0)
    assert m2[0] == pytest.approx(math.sqrt(a * b) / (a + b) * 60.0)
    # empty spectrum: 0/0
    z0, z1, z2 = oracle.moments(np.zeros((5, 1)), vel)
    assert z0[0] == 0.0 and math.isnan(z1[0]) and math.isnan(z2[0])


def test_chi2_by_hand(oracle):
    m0 = np.ones((2, 2))
    m1 = np.array([[10.0, 20.0], [30.0, 40.0]])
    m2 = np.array([[5.0, 6.0], [7.0, 8.0]])
    vobs = np.array([[11.0, 18.0], [30.0, 0.0]], dtype=np.float32)
    verr = np.array([[1.0, 2.0], [4.0, 1.0]], dtype=np.float32)
    sobs = np.array([[5.0, 9.0], [6.0, 0.0]], dtype=np.float32)
    serr = np.array([[1.0, 3.0], [0.5, 1.0]], dtype=np.float32)
    mask = np.array([[1, 1], [1, 0]], dtype=np.uint8)
    # eq. 11: (1)^2 + (1)^2 + 0 + [0 + (1)^2 + (2)^2] = 7
    val, resid = oracle.chi2(m0, m1, m2, vobs, verr, sobs, serr, mask, want_resid=True)
    assert val == pytest.approx(7.0)
    assert np.allclose(resid[0], [[-1, 1], [0, 0]]) and np.allclose(resid[1], [[0, -1], [2, 0]])
    # no mask: the fourth spaxel counts: + 40^2 + 8^2
    assert oracle.chi2(m0, m1, m2, vobs, verr, sobs, serr) == pytest.approx(7 + 1600 + 64)
    # no dispersion map: second term dropped
    assert oracle.chi2(m0, m1, m2, vobs, verr, None, None, mask) == pytest.approx(2.0)
    # W folded into the error: serr / sqrt(W) scales the second term by W
    W = 0.2
    val_w = oracle.chi2(m0, m1, m2, vobs, verr, sobs, (serr / math.sqrt(W)).astype(np.float32),
                        mask)
    assert val_w == pytest.approx(2.0 + W * 5.0, rel=1e-6)
    # A15: model-dark or non-finite unmasked spaxel -> +INF; masked ones are ignored
    dark = m0.copy()
    dark[1, 1] = 0.0
    assert oracle.chi2(dark, m1, m2, vobs, verr, sobs, serr, mask, dark_level=1e-30) == \
        pytest.approx(7.0)
    dark[0, 0] = 1e-31
    assert math.isinf(oracle.chi2(dark, m1, m2, vobs, verr, sobs, serr, mask, dark_level=1e-30))
    nan1 = m1.copy()
    nan1[0, 1] = math.nan
    assert math.isinf(oracle.chi2(m0, nan1, m2, vobs, verr, sobs, serr, mask))


# --------------------------------------------------------- whole pipeline ----

def _cfg1_grid(oracle, **kw):
    d = dict(nx=32, ny=32, nv=64, u=1, v_center=0.0, dv=30.0,
             psf=oracle.psf_gaussian_image(2.5, 1), lsf=oracle.gaussian_taps(25.0 / 30.0))
    d.update(kw)
    return oracle.Grid(**d)


def test_face_on_disc_has_m1_equal_vsys(oracle):
    g = _cfg1_grid(oracle)
    p = _row(xo=16.3, yo=15.8, pa=37, inc=0.0, vsys=12, vt=200, rt=3, sig=40, r0=4)
    m0, m1, m2 = oracle.model_maps(g, p)
    assert np.allclose(m1, 12.0, atol=1e-10)
    assert np.ptp(m2) < 1e-9
    assert m2[0, 0] == pytest.approx(math.hypot(40.0, 25.0), rel=1e-4)


def test_point_symmetry_and_axis_symmetries(oracle):
    # centre on the grid's symmetry point, symmetric PSF
    g = _cfg1_grid(oracle, nx=31, ny=31)
    p = _row(xo=15, yo=15, pa=37, inc=55, vsys=12, vt=200, rt=3, sig=40, r0=4)
    m0, m1, m2 = oracle.model_maps(g, p)
    assert np.allclose(m1 + m1[::-1, ::-1], 24.0, atol=1e-9)
    assert np.allclose(m0, m0[::-1, ::-1], rtol=1e-12)
    assert np.allclose(m2, m2[::-1, ::-1], atol=1e-9)
    # PA = 0: major axis along y.  Mirror in x (across the major axis): v symmetric.
    # Mirror in y (across the minor axis): v - V_sys antisymmetric (eq. 1, 4, 8).
    p = _row(xo=15, yo=15, pa=0, inc=55, vsys=12, vt=200, rt=3, sig=40, r0=4)
    m0, m1, m2 = oracle.model_maps(g, p)
    assert np.allclose(m1, m1[:, ::-1], atol=1e-9)
    assert np.allclose((m1 - 12.0), -(m1 - 12.0)[::-1, :], atol=1e-9)
    assert np.allclose(m1[15, :], 12.0, atol=1e-9)        # the minor axis itself
    assert np.allclose(m2, m2[::-1, :], atol=1e-9) and np.allclose(m2, m2[:, ::-1], atol=1e-9)
    assert m1[20, 15] > 12.0 > m1[10, 15]


def test_flux_conservation_under_normalised_psf_and_lsf(oracle):
    # compact disc well inside the field: nothing leaks through the border
    base = dict(nx=41, ny=41, nv=96, dv=30.0)
    p = _row(xo=20, yo=20, pa=25, inc=35, vsys=0, vt=150, rt=2, sig=40, r0=0.8, i0=2.0)
    sharp = oracle.Grid(**base)
    smooth = oracle.Grid(**base, psf=oracle.psf_gaussian_image(2.5, 1),
                         lsf=oracle.gaussian_taps(25.0 / 30.0))
    f_sharp = oracle.model_maps(sharp, p)[0].sum()
    f_smooth = oracle.model_maps(smooth, p)[0].sum()
    assert f_smooth == pytest.approx(f_sharp, rel=1e-9)
    # total flux of an inclined exponential disc: 2 pi r0^2 I0 cos i; with fine sampling the
    # Riemann sum approaches it (cusp at r = 0 limits the rate)
    fine = oracle.Grid(**base, u=4)
    f_fine = oracle.model_maps(fine, p)[0].sum()
    analytic = 2 * math.pi * 0.8 ** 2 * 2.0 * math.cos(math.radians(35))
    assert f_fine == pytest.approx(analytic, rel=1e-3)
    assert abs(f_fine - analytic) < abs(f_sharp - analytic)


def test_halo_reading_changes_only_the_border(oracle):
    # A6: interior spaxels (farther than R_p from the edge) do not see the halo switch
    g = _cfg1_grid(oracle)
    gz = _cfg1_grid(oracle, halo_zero=True)
    p = _row(xo=16.3, yo=15.8, pa=37, inc=55, vsys=12, vt=200, rt=3, sig=40, r0=4)
    a = oracle.model_maps(g, p)
    b = oracle.model_maps(gz, p)
    R = 5
    for ma, mb in zip(a, b):
        assert np.array_equal(ma[R:-R, R:-R], mb[R:-R, R:-R])
    assert not np.allclose(a[0], b[0], rtol=1e-3)


def test_moment_first_identity_with_library_convolution(oracle):
    """Independent second derivation (lives here, not in the oracle): the three un-normalised
    moments are linear in the cube, so PSF-convolving three 2-D maps of LSF-folded channel
    weights must reproduce the literal pipeline."""
    u = 2
    psf = oracle.psf_gaussian_image(2.0, u)
    lsf = oracle.gaussian_taps(20.0 / 30.0)
    g = oracle.Grid(nx=10, ny=8, nv=40, u=u, dv=30.0, v_center=4.0, psf=psf, lsf=lsf)
    p = _row(xo=4.6, yo=3.7, pa=110, inc=50, vsys=9, vt=180, rt=2.5, sig=35, r0=3)
    m0, m1, m2 = oracle.model_maps(g, p)
    cube = oracle.model_cube(g, p)                     # [nv + 2Rv, eh, ew]
    Rv = (lsf.size - 1) // 2
    vel = g.channel_velocities()
    w = np.zeros((3, cube.shape[0]))
    for c in range(cube.shape[0]):                      # extended channel index
        for k in range(g.nv):                           # in-band output channel
            t = (c - Rv) - k                            # out[k] = sum_t L[t'] in[k + Rv*2 - t']
            j = Rv - t
            if 0 <= j < lsf.size:
                for q in range(3):
                    w[q, c] += lsf[j] * vel[k] ** q
    S = np.tensordot(w, cube, axes=(1, 0))              # [3, eh, ew]
    Sc = np.stack([signal.convolve2d(S[q], psf, mode="valid") for q in range(3)])
    Sd = Sc.reshape(3, g.ny, u, g.nx, u).mean(axis=(2, 4))
    assert np.allclose(Sd[0], m0, rtol=1e-12)
    assert np.allclose(Sd[1] / Sd[0], m1, atol=1e-9)
    assert np.allclose(np.sqrt(np.maximum(0, Sd[2] / Sd[0] - (Sd[1] / Sd[0]) ** 2)), m2, atol=1e-8)


def test_upsampling_changes_maps_smoothly(oracle):
    # Fig. 1: a finer cube removes sampling artefacts; u=2 and u=4 agree
    # better with each other than u=1 and u=2 do
    maps = {}
    for u in (1, 2, 4):
        g = _cfg1_grid(oracle, nx=16, ny=16, u=u, psf=oracle.psf_gaussian_image(2.5, u))
        maps[u] = oracle.model_maps(g, _row(xo=7.3, yo=7.8, pa=37, inc=55, vsys=12, r0=4))
    d12 = np.abs(maps[1][1] - maps[2][1]).max()
    d24 = np.abs(maps[2][1] - maps[4][1]).max()
    assert d24 < d12 and d12 < 5.0


def test_eval_rows_matches_steps_and_domain_rule(oracle):
    from paper_1510_01815_b200 import workloads as wl
    g = _cfg1_grid(oracle, nx=12, ny=10, nv=48)
    rng = np.random.default_rng(3)
    w = wl.config(1).scaled(nx=12, ny=10, nv=48)
    true = _row(xo=5.5, yo=4.5, pa=30, inc=50, vsys=5, r0=3)
    m0, m1, m2 = oracle.model_maps(g, true)
    obs = wl.observe(w, m0, m1, m2, rng)
    rows = np.array([true, _row(xo=5.0, yo=4.0, pa=40, inc=45, vsys=0, r0=3),
                     _row(sig=-1.0), _row(inc=90.0)], dtype=np.float32)
    out = oracle.eval_rows(g, obs.vobs, obs.verr, obs.sobs, obs.serr, obs.mask, rows,
                           want_maps=True, want_resid=True, nthreads=2)
    for k in range(2):
        a0, a1, a2 = oracle.model_maps(g, rows[k].astype(np.float64))
        assert np.array_equal(out["m1"][k], a1)
        want = oracle.chi2(a0, a1, a2, obs.vobs[...], obs.verr, obs.sobs, obs.serr, obs.mask,
                           dark_level=1e-30)
        assert out["chi2"][k] == want
    n_ok = int(obs.mask.sum())
    # chi^2 of the true row is ~ 2 per unmasked spaxel (unit-variance residuals, two terms)
    assert 0.6 * 2 * n_ok < out["chi2"][0] < 1.4 * 2 * n_ok
    assert out["chi2"][1] > out["chi2"][0]
    assert np.isinf(out["chi2"][2]) and np.isinf(out["chi2"][3])
    assert np.isnan(out["m1"][2]).all() and np.isnan(out["resid"][3]).all()
    assert np.all(out["resid"][0][:, obs.mask[...] == 0] == 0)


def test_golden_hand_values_file(oracle):
    """tests/golden/eq_hand_values.txt: hand-derived values of eq. 1-8 (with derivations)."""
    n = 0
    with open(os.path.join(GOLDEN, "eq_hand_values.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            tok = line.split()
            rc = {"arctan": 0, "ramp": 1, "epinat": 2}[tok[0]]
            npar = oracle.row_len(rc)                      # 12 columns for the Epinat curve (a, g last)
            p = [float(t) for t in tok[1:1 + npar]]
            x, y, I_want, v_want = (float(t) for t in tok[1 + npar:5 + npar])
            I, v = oracle.disc_point(p, rc, x, y)
            assert I == pytest.approx(I_want, rel=1e-9), line
            assert v == pytest.approx(v_want, abs=1e-7), line
            n += 1
    assert n >= 8


# ------------------------------------------------ velocity-field strategy ----

def _vf_grid(oracle, nx, ny, rc=0):
    return oracle.Grid(nx=nx, ny=ny, nv=8, u=1, v_center=0.0, dv=10.0, rc_model=rc,
                       psf=np.ones((1, 1)), lsf=np.ones(1))


def test_vfield_map_equals_the_golden_hand_values(oracle):
    """vmap[y][x] of the velocity-field oracle = the hand-derived eq. 8 values of the golden file
    (spaxel j is centred on coordinate j, reading A1), for every golden point on the pixel grid."""
    n = 0
    with open(os.path.join(GOLDEN, "eq_hand_values.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            tok = line.split()
            rc = {"arctan": 0, "ramp": 1, "epinat": 2}[tok[0]]
            npar = oracle.row_len(rc)
            p = np.array([float(t) for t in tok[1:1 + npar]], dtype=np.float32)
            x, y, _, v_want = (float(t) for t in tok[1 + npar:5 + npar])
            if x < 0 or y < 0 or x != int(x) or y != int(y):
                continue
            g = _vf_grid(oracle, 20, 20, rc)
            z = np.zeros((20, 20), np.float32)
            out = oracle.vfield_rows(g, z, z + 1, None, p[None], want_maps=True)
            assert out["vmap"][0, int(y), int(x)] == pytest.approx(v_want, abs=1e-5), line
            n += 1
    assert n >= 11


def test_vfield_chi2_by_hand_masks_and_domain(oracle):
    g = _vf_grid(oracle, 2, 2)
    # face-on disc: v = V_sys = 12 everywhere (eq. 8 with sin i = 0)
    p = np.array([[0.5, 0.5, 30.0, 0.0, 12.0, 200.0, 3.0, np.nan, np.nan, np.nan]], dtype=np.float32)
    vobs = np.array([[10.0, 12.0], [15.0, 0.0]], np.float32)
    verr = np.array([[1.0, 2.0], [3.0, 4.0]], np.float32)
    out = oracle.vfield_rows(g, vobs, verr, None, p, want_maps=True, want_resid=True)
    assert np.allclose(out["vmap"][0], 12.0, atol=1e-12)
    assert out["chi2"][0] == pytest.approx(2.0 ** 2 + 0.0 + 1.0 ** 2 + 3.0 ** 2)      # 4 + 0 + 1 + 9
    assert np.allclose(out["resid"][0], [[2.0, 0.0], [-1.0, 3.0]])
    mask = np.array([[1, 1], [1, 0]], np.uint8)
    out = oracle.vfield_rows(g, vobs, verr, mask, p, want_resid=True)
    assert out["chi2"][0] == pytest.approx(5.0) and out["resid"][0, 1, 1] == 0.0
    # sigma_0, r_0, I_0 are not part of eq. 8 (NaN above was harmless); the kinematic ones are
    for j, bad in ((6, 0.0), (3, 90.0), (5, np.inf), (0, np.nan)):
        q = p.copy()
        q[0, j] = bad
        assert np.isinf(oracle.vfield_rows(g, vobs, verr, None, q)["chi2"][0]), j


def test_vfield_is_antisymmetric_about_the_centre_and_equals_delta_kernel_m1(oracle):
    """v(c + d) + v(c - d) = 2 V_sys (eq. 1, 4, 8), and the velocity field is the m1 map of the cube
    strategy with delta PSF and LSF (the strategies differ only in steps 2.2.2-2.2.5)."""
    p = np.array([[7.0, 6.0, 123.0, 50.0, 8.0, 180.0, 2.5, 40.0, 3.0, 1.5]], dtype=np.float32)
    for rc in (0, 1):
        g = oracle.Grid(nx=15, ny=13, nv=96, u=1, v_center=0.0, dv=12.0, rc_model=rc,
                        psf=np.ones((1, 1)), lsf=np.ones(1))
        z = np.zeros((13, 15), np.float32)
        v = oracle.vfield_rows(g, z, z + 1, None, p, want_maps=True)["vmap"][0]
        assert np.allclose(v + v[::-1, ::-1], 16.0, atol=1e-10)
        m0, m1, m2 = oracle.model_maps(g, p[0].astype(np.float64))
        assert np.max(np.abs(m1 - v)) < 1e-6


def test_vfield_epinat_plateaus_and_domain(oracle):
    """Eq. 7: a = g gives a flat plateau V -> V_t, a < g rises, a > g declines
    (PAPER.md:129); slopes must be > 0."""
    g = _vf_grid(oracle, 400, 1, rc=2)
    z = np.zeros((1, 400), np.float32)
    def curve(a, gg):
        p = np.array([[0.0, 0.0, 90.0, 90.0 - 1e-3, 0.0, 100.0, 2.0, np.nan, np.nan, np.nan, a, gg]],
                     dtype=np.float32)                  # sigma_0, r_0, I_0 are not part of eq. 8
        # PA = 90: x_e = -(x - x_o); i ~ 90: sin i = 1 -> v(x) = -V_rot(|x|) on this row
        return -oracle.vfield_rows(g, z, z + 1, None, p, want_maps=True)["vmap"][0, 0]
    flat, rising, falling = curve(1.5, 1.5), curve(1.0, 1.5), curve(1.5, 1.0)
    assert flat[-1] == pytest.approx(100.0, rel=2e-3) and flat[2] == pytest.approx(50.0, rel=1e-9)
    assert rising[-1] > rising[200] > 100.0 and falling[-1] < falling[200] < falling[4]
    p = np.array([[0.0, 0.0, 0.0, 30.0, 0.0, 100.0, 2.0, 40.0, 4.0, 1.0, 1.0, 1.0]], dtype=np.float32)
    assert np.isfinite(oracle.vfield_rows(g, z, z + 1, None, p)["chi2"][0])
    for j, bad in ((10, 0.0), (11, 0.0), (10, -1.0), (11, np.nan)):
        q = p.copy()
        q[0, j] = bad
        assert np.isinf(oracle.vfield_rows(g, z, z + 1, None, q)["chi2"][0]), (j, bad)


# ------------------------- Epinat curve and a tabulated profile in the cube ----

def test_cube_with_the_epinat_curve_delta_kernels(oracle):
    """Eq. 7 inside the intensity-cube strategy: with delta PSF and LSF the m1 map
    is eq. 8 with V_rot = V_t q^g / (1 + q^a), q = r / r_t -- written out here for every spaxel -- m2
    is sigma_0 and m0 the exponential disc of eq. 5; a = g = 1 at r = r_t gives V_t / 2 by hand."""
    g = oracle.Grid(nx=17, ny=15, nv=160, u=1, v_center=0.0, dv=12.0, rc_model=oracle.RC_EPINAT,
                    psf=np.ones((1, 1)), lsf=np.ones(1))
    xo, yo, pa, inc, vsys, vt, rt, sig, r0, i0, a, gg = 8.0, 7.0, 0.0, 30.0, 7.0, 200.0, 3.0, 40.0, 4.0, 2.5, 1.7, 0.8
    p = np.array([xo, yo, pa, inc, vsys, vt, rt, sig, r0, i0, a, gg])
    m0, m1, m2 = oracle.model_maps(g, p)
    yy, xx = np.mgrid[0:15, 0:17].astype(float)
    xe = (yy - yo)                                    # PA = 0: eq. 1 gives x_e = y - y_o
    ye = -(xx - xo)                                   # eq. 2
    r = np.sqrt(xe ** 2 + (ye / np.cos(np.radians(inc))) ** 2)
    with np.errstate(invalid="ignore", divide="ignore"):
        cos_t = np.where(r > 0, xe / r, 0.0)
    q = r / rt
    v = vsys + vt * q ** gg / (1.0 + q ** a) * np.sin(np.radians(inc)) * cos_t
    assert np.max(np.abs(m1 - v)) < 1e-6
    assert np.max(np.abs(m2 - sig)) < 1e-6
    assert np.max(np.abs(m0 / (i0 * np.exp(-r / r0)) - 1.0)) < 1e-8
    p1 = p.copy()
    p1[10:] = 1.0
    _, m1b, _ = oracle.model_maps(g, p1)
    assert m1b[10, 8] == pytest.approx(7.0 + 100.0 * 0.5, abs=1e-6)      # (x, y) = (8, 10): r = r_t, on the major axis
    for j, bad in ((10, 0.0), (11, -2.0), (10, np.nan)):                    # slopes must be finite and > 0
        pb = p.copy()
        pb[j] = bad
        assert not oracle.row_valid_rc(pb, oracle.RC_EPINAT)
        assert np.isnan(oracle.model_maps(g, pb)[0]).all()


def test_tabulated_profile_by_hand(oracle):
    """The tabulated radial profile (reading A22): linear interpolation between the
    nodes x_j = j dx, the last value beyond them."""
    tab = np.array([4.0, 2.0, 1.0, 0.25])
    assert oracle.table_profile(tab, 0.5, 0.0) == 4.0
    assert oracle.table_profile(tab, 0.5, 0.25) == pytest.approx(3.0)           # half way 4 -> 2
    assert oracle.table_profile(tab, 0.5, 0.5) == 2.0
    assert oracle.table_profile(tab, 0.5, 1.2) == pytest.approx(1.0 - 0.4 * 0.75)   # 40 % of the way 1 -> 0.25
    assert oracle.table_profile(tab, 0.5, 1.5) == 0.25
    assert oracle.table_profile(tab, 0.5, 7.0) == 0.25


def test_cube_with_a_tabulated_intensity_profile(oracle):
    """I(r) = I_0 T(r / r_0) replaces eq. 5 in the cube: (1) a constant table gives a uniform disc,
    m0 = I_0 c; (2) a table of exp(-x) on a fine mesh reproduces the exponential model to the
    interpolation error dx^2/8; (3) a linear table gives hand-computable m0 at spaxels of known r;
    the velocity and dispersion maps do not depend on the profile when the kernels are deltas."""
    base = dict(nx=13, ny=11, nv=128, u=1, v_center=0.0, dv=15.0, rc_model=0, psf=np.ones((1, 1)),
                lsf=np.ones(1))
    p = np.array([6.0, 5.0, 0.0, 60.0, 3.0, 150.0, 2.0, 35.0, 3.0, 1.5])
    g_exp = oracle.Grid(**base)
    m0e, m1e, m2e = oracle.model_maps(g_exp, p)
    # (1) uniform disc
    m0, m1, m2 = oracle.model_maps(oracle.Grid(**base, tab=np.array([0.7, 0.7]), tab_dx=1.0), p)
    assert np.max(np.abs(m0 / (1.5 * 0.7) - 1.0)) < 1e-8
    assert np.max(np.abs(m1 - m1e)) < 1e-9 and np.max(np.abs(m2 - m2e)) < 1e-9
    # (2) exp(-x) on a mesh of 0.01 out to x = 12
    dx = 0.01
    tab = np.exp(-dx * np.arange(1201))
    m0, _, _ = oracle.model_maps(oracle.Grid(**base, tab=tab, tab_dx=dx), p)
    rel = np.abs(m0 / m0e - 1.0)
    assert rel.max() < 1.3 * dx * dx / 8.0 and rel.max() > 0.0       # chord above a convex curve: <= dx^2/8
    # (3) T(x) = 1 - x/4 on [0, 4] (two nodes), 0 beyond is not reached here: r_0 = 3, r <= 12
    m0, _, _ = oracle.model_maps(oracle.Grid(**base, tab=np.array([1.0, 0.0]), tab_dx=4.0), p)
    # PA = 0, i = 60: spaxel (x, y) = (6, 8) lies on the major axis at r = 3 => x = 1, T = 0.75;
    # spaxel (8, 5) lies on the minor axis: r = 2 / cos 60 = 4 => x = 4/3, T = 2/3
    assert m0[8, 6] == pytest.approx(1.5 * 0.75, rel=1e-8)
    assert m0[5, 8] == pytest.approx(1.5 * (1.0 - (4.0 / 3.0) / 4.0), rel=1e-8)
    assert m0[5, 6] == pytest.approx(1.5, rel=1e-8)                      # the centre: r = 0


# ---------------- Gaussian-profile extraction ----

def _gauss(v, A, mu, s):
    return A * np.exp(-0.5 * ((v - mu) / s) ** 2)


def test_gaussfit_recovers_an_exact_sampled_gaussian(oracle):
    """A spectrum that IS a sampled Gaussian is fitted exactly, whether the centre sits on a channel,
    between channels, or close to the band edge with a third of the line cut off (where the moments
    are biased: the reason the paper gives for the method's "superior accuracy")."""
    v = (np.arange(48) - 23.5) * 12.0
    cases = [(3.0, 6.0, 30.0), (0.7, -41.3, 17.0), (5.0, 100.0, 55.0), (1.0, 250.0, 40.0), (2.0, -275.0, 25.0)]
    cube = np.stack([_gauss(v, *c) for c in cases], axis=1)[:, None, :]      # [nv, 1, ncase]
    m0, mu, sg = oracle.gaussfit(cube, v)
    mm0, m1, m2 = oracle.moments(cube, v)
    for i, (A, mu_t, s_t) in enumerate(cases):
        assert mu[0, i] == pytest.approx(mu_t, abs=1e-6) and sg[0, i] == pytest.approx(s_t, abs=1e-6), i
        assert m0[0, i] == pytest.approx(mm0[0, i], rel=1e-14)              # flux stays the plain sum
    assert abs(m1[0, 3] - 250.0) > 5.0 and abs(m1[0, 4] + 275.0) > 5.0       # the truncated lines bias the moments
    assert abs(m1[0, 0] - 6.0) < 1e-6 and abs(m2[0, 0] - 30.0) < 1e-3        # ... not the complete ones


def test_gaussfit_minimises_the_sum_of_squares_and_matches_scipy(oracle):
    """For a spectrum that is NOT a Gaussian (two components, a skewed line) the result is the
    least-squares Gaussian: the gradient of the sum of squares vanishes there (central differences
    taken here), and scipy.optimize.least_squares from the same start lands on the same point."""
    from scipy.optimize import least_squares
    v = (np.arange(64) - 31.5) * 10.0
    specs = [_gauss(v, 2.0, -30.0, 25.0) + _gauss(v, 1.2, 40.0, 35.0),
             _gauss(v, 1.0, 10.0, 20.0) * (1.0 + 0.4 * np.tanh((v - 10.0) / 30.0)),
             _gauss(v, 3.0, 0.0, 12.0) + 0.02]
    cube = np.stack(specs, axis=1)[:, None, :]
    m0, mu, sg = oracle.gaussfit(cube, v)
    _, m1, m2 = oracle.moments(cube, v)
    for i, c in enumerate(specs):
        sse = lambda p: float(np.sum((c - _gauss(v, *p)) ** 2))
        start = [c.sum() * 10.0 / (max(m2[0, i], 5.0) * np.sqrt(2 * np.pi)), m1[0, i], max(m2[0, i], 5.0)]
        sol = least_squares(lambda p: c - _gauss(v, *p), start, xtol=1e-14, ftol=1e-14, gtol=1e-14).x
        assert mu[0, i] == pytest.approx(sol[1], abs=1e-4) and sg[0, i] == pytest.approx(abs(sol[2]), abs=1e-4), i
        A = np.sum(c * _gauss(v, 1.0, mu[0, i], sg[0, i])) / np.sum(_gauss(v, 1.0, mu[0, i], sg[0, i]) ** 2)
        p0 = np.array([A, mu[0, i], sg[0, i]])
        for j, h in ((1, 1e-3), (2, 1e-3)):
            e = np.zeros(3)
            e[j] = h
            grad = (sse(p0 + e) - sse(p0 - e)) / (2 * h)
            assert abs(grad) < 1e-6 * sse(p0) + 1e-9, (i, j, grad)


def test_gaussfit_in_the_pipeline_and_failures(oracle):
    """extract = 1 in the whole pipeline: with delta kernels and a line well inside the band the fitted
    velocity is eq. 8 and the fitted dispersion sigma_0 (the spectrum is an exact Gaussian), as with the
    moments; a dark spectrum (m0 = 0) gives NaN."""
    kw = dict(nx=9, ny=8, nv=96, u=1, v_center=0.0, dv=12.0, rc_model=0, psf=np.ones((1, 1)), lsf=np.ones(1))
    p = np.array([4.0, 3.5, 25.0, 50.0, 5.0, 150.0, 2.0, 35.0, 3.0, 1.5])
    m0a, m1a, m2a = oracle.model_maps(oracle.Grid(**kw), p)
    m0b, m1b, m2b = oracle.model_maps(oracle.Grid(**kw, extract=1), p)
    assert np.array_equal(m0a, m0b)
    assert np.max(np.abs(m1a - m1b)) < 1e-6 and np.max(np.abs(m2b - 35.0)) < 1e-6
    z = np.zeros((8, 1, 2))
    m0, mu, sg = oracle.gaussfit(z, np.arange(8.0))
    assert np.isnan(mu).all() and np.isnan(sg).all() and (m0 == 0).all()
    # beam smearing: with a wide PSF the two extractions differ near the centre (Fig. 14)
    psf = oracle.psf_gaussian_image(4.0, 1)
    g1 = oracle.Grid(**{**kw, "psf": psf})
    g2 = oracle.Grid(**{**kw, "psf": psf}, extract=1)
    _, v1, s1 = oracle.model_maps(g1, p)
    _, v2, s2 = oracle.model_maps(g2, p)
    assert 0.05 < np.nanmax(np.abs(s1 - s2)) < 20.0
