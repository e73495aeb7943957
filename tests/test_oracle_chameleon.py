"""Pins for the oracle's Chameleon light profile (Eq. 47, light part) and for the `kinds`
switch of the lensing half.  None retypes Eq. 47 as a whole: total flux in closed form, the single cored-isothermal limit,
the profile's own symmetries, and the image pipeline checked against a pipeline-free evaluation."""
import math

import numpy as np
import pytest
from scipy import integrate

import oracle


@pytest.fixture(scope="module", autouse=True)
def _build():
    oracle.build()


def test_total_flux_closed_form():
    """int [1/sqrt(R^2+a) - 1/sqrt(R^2+b)] R dR = sqrt(b) - sqrt(a), area element 2 pi q R dR for R^2 = x^2 + y^2/q^2:
    F = 2 pi q I_0/(1+q) * 2 (w_t - w_c)/(1+q).  Each term alone diverges: a wrong sign or a missing q would show."""
    for I0, wc, wt, q in ((1.3, 0.05, 0.9, 0.8), (0.4, 0.3, 0.31, 0.55), (2.0, 0.01, 3.0, 1.0)):
        f = lambda R: oracle.chameleon(R, 0.0, I0, wc, wt, q, 0.0) * 2 * math.pi * q * R
        # the difference decays like R^-3: integrate to 1e5 and add the analytic tail (b - a)/(2 R) * 2 pi q I0/(1+q)
        num, _ = integrate.quad(f, 0.0, 1e4, limit=2000, epsabs=0, epsrel=1e-10, points=[wc, wt, 10 * wt])
        a, b = 4 * wc * wc / (1 + q) ** 2, 4 * wt * wt / (1 + q) ** 2
        num += 2 * math.pi * q * I0 / (1 + q) * (b - a) / (2 * 1e4)
        want = 2 * math.pi * q * I0 / (1 + q) * 2 * (wt - wc) / (1 + q)
        assert num == pytest.approx(want, rel=1e-6)


def test_single_cored_isothermal_limit_and_axes():
    """w_t -> infinity leaves I_0/(1+q) / sqrt(R^2 + 4 w_c^2/(1+q)^2); on the minor axis R = y/q."""
    I0, wc, q = 0.9, 0.2, 0.7
    for x, y in ((0.5, 0.0), (0.0, 0.5), (0.3, -0.4)):
        R2 = x * x + y * y / (q * q)
        want = I0 / (1 + q) / math.sqrt(R2 + 4 * wc * wc / (1 + q) ** 2)
        assert oracle.chameleon(x, y, I0, wc, 1e9, q, 0.0) == pytest.approx(want, rel=1e-8)
    # centre value: I_0/2 (1/w_c - 1/w_t)
    assert oracle.chameleon(0, 0, I0, wc, 1.1, q, 0.3) == pytest.approx(I0 / 2 * (1 / wc - 1 / 1.1), rel=1e-12)


def test_symmetries_and_rotation():
    I0, wc, wt, q = 1.0, 0.1, 0.8, 0.6
    v = oracle.chameleon(0.4, 0.25, I0, wc, wt, q, 0.0)
    assert oracle.chameleon(-0.4, 0.25, I0, wc, wt, q, 0.0) == pytest.approx(v, rel=1e-14)
    assert oracle.chameleon(0.4, -0.25, I0, wc, wt, q, 0.0) == pytest.approx(v, rel=1e-14)
    phi = 0.7                      # rotating the point with the profile changes nothing (angles counter-clockwise from +x)
    xr, yr = 0.4 * math.cos(phi) - 0.25 * math.sin(phi), 0.4 * math.sin(phi) + 0.25 * math.cos(phi)
    assert oracle.chameleon(xr, yr, I0, wc, wt, q, phi) == pytest.approx(v, rel=1e-12)
    assert oracle.chameleon(0.4, 0.25, I0, wc, wt, 1.0, 1.234) == pytest.approx(oracle.chameleon(0.25, 0.4, I0, wc, wt, 1.0, 0.0), rel=1e-12)
    assert oracle.chameleon(0.4, 0.25, I0, wt, wc, q, 0.0) == pytest.approx(-v, rel=1e-12)      # swapping the cores flips the sign
    assert oracle.chameleon(3.0, 0.0, I0, wc, wt, q, 0.0) > 0 and v > oracle.chameleon(0.8, 0.5, I0, wc, wt, q, 0.0)


def _grid(n=24, pix=0.1, s=1):
    return dict(nx=n, ny=n, supersample=s, pix=pix, x0=-(n - 1) / 2 * pix, y0=-(n - 1) / 2 * pix)


def test_image_pipeline_with_chameleon_lens_light_and_source():
    """No mass (theta_E = 0, no shear, no BH), delta PSF: the image is the profile at the pixel centres, lens light at theta
    and source at beta = theta; supersampling = mean of the finer grid; Sersic components are untouched by the switch."""
    g = _grid()
    p = np.zeros((1, 26), np.float32)
    p[0, 0:6] = [0.03, -0.02, 0.0, 2.0, 0.8, 0.3]
    p[0, 9:16] = [0.2, 0.1, 0.7, 0.05, 0.5, 0.9, 1.0]            # source as Chameleon {x,y,I0,wc,wt,q,phi}
    p[0, 16:21] = [1.1, 0.08, 0.9, 0.7, 0.3]                      # lens light 1 as Chameleon
    p[0, 21:26] = [0.5, 0.6, 2.0, 0.8, 0.3]                       # lens light 2 stays a Sersic
    psf = np.zeros((3, 3), np.float32); psf[1, 1] = 1.0
    img = oracle.lens_image_batch(p, g, psf, kinds=[1, 1, 0])["images"][0]
    pd = p[0].astype(np.float64)
    for iy, ix in ((0, 0), (11, 12), (23, 5)):
        x, y = g["x0"] + ix * g["pix"], g["y0"] + iy * g["pix"]
        want = (oracle.chameleon(x - pd[9], y - pd[10], *pd[11:16]) + oracle.chameleon(x - pd[0], y - pd[1], *pd[16:21])
                + oracle.sersic(x - pd[0], y - pd[1], *pd[21:26]))
        assert img[iy, ix] == pytest.approx(want, rel=1e-12)
    # all-Sersic kinds == the plain call
    a = oracle.lens_image_batch(p, g, psf, kinds=[0, 0, 0])["images"]
    b = oracle.lens_image_batch(p, g, psf)["images"]
    assert np.array_equal(a, b)
    # supersampling: mean of the 3x finer grid
    g3, gf = _grid(8, 0.3, 3), _grid(24, 0.1, 1)
    fine = oracle.lens_image_batch(p, gf, psf, kinds=[1, 1, 0])["images"][0]
    coarse = oracle.lens_image_batch(p, g3, psf, kinds=[1, 1, 0])["images"][0]
    assert np.allclose(coarse, fine.reshape(8, 3, 8, 3).mean(axis=(1, 3)), rtol=1e-12)


def test_validity_and_bad_kinds():
    g = _grid(8)
    psf = np.ones((1, 1), np.float32)
    p = np.zeros((3, 26), np.float32)
    p[:, 0:6] = [0, 0, 1.0, 2.0, 0.8, 0.0]
    p[:, 16:21] = [1.0, 0.1, 0.8, 0.7, 0.0]
    p[1, 17:19] = [0.8, 0.1]                                      # w_t < w_c: negative profile -> invalid
    p[2, 17] = 0.0                                                # w_c = 0 -> invalid (1/R cusp)
    out = oracle.lens_image_batch(p, g, psf, kinds=[0, 1, 0])
    assert list(out["flags"]) == [0, oracle.FLAG_LENS_INVALID, oracle.FLAG_LENS_INVALID]
    assert np.isnan(out["images"][1]).all() and np.isfinite(out["images"][0]).all()
    with pytest.raises(ValueError):
        oracle.lens_image_batch(p, g, psf, kinds=[0, 2, 0])
