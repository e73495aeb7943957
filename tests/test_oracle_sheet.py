"""Pins for the internal mass sheet of the oracle (Eq. 5-9, Eq. 50-51, "multiply by
the dPIE sheet"; readings R-S1..3; CPU only).  The mass-sheet degeneracy itself is the pin: with a flat sheet the lensed image
of a source scaled by lam (Eq. 5), the predicted image positions and lam x the time delays (Eq. 9) are unchanged."""
import math

import numpy as np
import pytest

from quasar_util import RXJ_LIKE, mock_quasar
from test_oracle_lens import grid, lens_vec
from test_oracle_quasar import d5

RC, RT = 45.0, 45.09
FLAT = (4.5e4, 4.509e4)         # a sheet flat to 1e-9 over the image: the exact transformation of Eq. 6


def s_paper(R, rc, rt):
    """Eq. 50 normalised to its central value (Eq. 51): the profile that stands for the constant sheet."""
    return (1 / math.sqrt(R * R + rc * rc) - 1 / math.sqrt(R * R + rt * rt)) / (1 / rc - 1 / rt)


@pytest.mark.parametrize("rc,rt", [(RC, RT), (3.0, 7.0), (0.5, 0.6)])
def test_sheet_deflection_potential_hessian_are_consistent_with_eq50(oracle, rc, rt):
    rng = np.random.default_rng(3)
    p = lens_vec(thetaE=0.0, xl=0.03, yl=-0.02)          # sheet alone
    for _ in range(12):
        lam = rng.uniform(0.5, 1.5)
        x, y = rng.uniform(-3, 3, 2)
        dx, dy = x - p[0], y - p[1]
        kap = oracle.sheet_kappa(lam, rc, rt, dx, dy)
        assert kap == pytest.approx((1 - lam) * s_paper(math.hypot(dx, dy), rc, rt), rel=1e-9, abs=1e-15)
        ax, ay = oracle.deflection(p, x, y, lam, (rc, rt))
        gx = d5(lambda t: oracle.potential(p, t, y, lam, (rc, rt)), x, 1e-3)
        gy = d5(lambda t: oracle.potential(p, x, t, lam, (rc, rt)), y, 1e-3)
        assert gx == pytest.approx(ax, rel=1e-7, abs=1e-10) and gy == pytest.approx(ay, rel=1e-7, abs=1e-10)
        h = oracle.hessian(p, x, y, lam, (rc, rt))
        assert h[0] == pytest.approx(d5(lambda t: oracle.deflection(p, t, y, lam, (rc, rt))[0], x, 1e-3), rel=1e-7, abs=1e-10)
        assert h[1] == pytest.approx(d5(lambda t: oracle.deflection(p, x, t, lam, (rc, rt))[0], y, 1e-3), rel=1e-7, abs=1e-10)
        assert h[2] == pytest.approx(d5(lambda t: oracle.deflection(p, x, t, lam, (rc, rt))[1], y, 1e-3), rel=1e-7, abs=1e-10)
        assert 0.5 * (h[0] + h[2]) == pytest.approx(kap, rel=1e-12, abs=1e-16)      # Poisson, Eq. 7
        # radial, and alpha = (1 - lam) theta for a flat sheet (R << rc)
        assert ax * dy == pytest.approx(ay * dx, rel=1e-12, abs=1e-15)
    ax, ay = oracle.deflection(p, 1.03, -0.02, 0.8, FLAT)
    assert ax == pytest.approx(0.2, rel=1e-8) and abs(ay) < 1e-15
    assert oracle.potential(p, p[0], p[1], 0.8, (RC, RT)) == 0.0


def test_lambda_one_is_no_sheet(oracle):
    p = lens_vec(bh=0.01, **RXJ_LIKE)
    for xy in ((1.2, 0.4), (-0.3, 1.9)):
        assert oracle.deflection(p, *xy, 1.0, (RC, RT)) == oracle.deflection(p, *xy)
        assert oracle.potential(p, *xy, 1.0, (RC, RT)) == oracle.potential(p, *xy)
        assert np.array_equal(oracle.hessian(p, *xy, 1.0, (RC, RT)), oracle.hessian(p, *xy))


def test_mass_sheet_degeneracy_of_the_extended_image(oracle):
    """Eq. 5-6: kappa -> (1-lam) + lam kappa maps beta -> lam beta, so a source shrunk by lam about the origin gives the
    same image (surface brightness is conserved).  The external shear is a separate free parameter outside kappa_int
    (reading R-S2), so the transformation of the whole potential (Eq. 8) has gamma_ext -> lam gamma_ext."""
    g = grid(40, 0.1, s=2)
    base = lens_vec(Ies=1.0, Res=0.25, ns=1.5, qs=0.7, phis=0.4, xs=0.1, ys=-0.06, **RXJ_LIKE)
    psf = np.ones((1, 1), np.float32)
    ref = oracle.lens_image_batch(base[None], g, psf)["images"][0]
    for lam in (0.7, 1.3):
        p = base.copy()
        p[9:11] *= lam
        p[12] *= lam
        p[6] *= lam
        img = oracle.lens_image_batch(p[None], g, psf, lam=[lam], sheet=FLAT)["images"][0]
        assert np.max(np.abs(img - ref)) < 2e-6 * ref.max()          # float32 rounding of the scaled vector
        # ... and without rescaling the source the image does change: the pin can see a missing sheet
        img2 = oracle.lens_image_batch(base[None], g, psf, lam=[lam], sheet=FLAT)["images"][0]
        assert np.max(np.abs(img2 - ref)) > 1e-2 * ref.max()
    # the paper's radii: flat to (R/rc)^2/2 ~ 1e-3 over a 2" arc
    p = base.copy(); p[9:11] *= 0.8; p[12] *= 0.8; p[6] *= 0.8
    img = oracle.lens_image_batch(p[None], g, psf, lam=[0.8], sheet=(RC, RT))["images"][0]
    assert 1e-7 * ref.max() < np.max(np.abs(img - ref)) < 2e-2 * ref.max()


def test_mass_sheet_degeneracy_of_positions_and_delays(oracle):
    """Image positions are invariant, beta -> lam beta, and Delta t -> lam Delta t at fixed D_dt, i.e. D_dt,int = D_dt/lam (Eq. 9)."""
    p = lens_vec(**RXJ_LIKE).astype(np.float32).astype(np.float64)
    q = mock_quasar(oracle, p, np.array([0.08, -0.05]), 1823.0, seed=4)
    a = oracle.quasar_batch(p[None], [1823.0], q)
    for lam in (0.6, 1.4):
        lf = float(np.float32(lam))
        pl = p.copy()
        pl[6] = np.float32(p[6] * lf)           # gamma_ext -> lam gamma_ext (see the image test)
        p1 = p.copy()
        p1[6] = pl[6] / lf                      # ... so that the comparison vector is exactly the float32 one divided by lam
        a = oracle.quasar_batch(p1[None], [1823.0], q)
        b = oracle.quasar_batch(pl[None], [1823.0], q, lam=[lam], sheet=FLAT)
        np.testing.assert_allclose(b["theta_pre"], a["theta_pre"], atol=1e-8)
        np.testing.assert_allclose(b["beta"], lf * a["beta"], rtol=1e-7, atol=1e-9)
        np.testing.assert_allclose(b["dt_pre"], lf * a["dt_pre"], rtol=1e-6, atol=1e-7)
        assert b["chi2_img"][0] == pytest.approx(a["chi2_img"][0], rel=1e-5)
        c = oracle.quasar_batch(pl[None], [1823.0 / lf], q, lam=[lam], sheet=FLAT)
        np.testing.assert_allclose(c["dt_pre"], a["dt_pre"], rtol=1e-6, atol=1e-7)
        assert c["chi2_tmd"][0] == pytest.approx(a["chi2_tmd"][0], rel=1e-4)


def test_model_tables_with_the_sheet(oracle):
    """Sigma_int = Sigma_crit [lam kappa_epl + (1 - lam) S(R)]: lam x the EPL rows, then round rows that sum back to the sheet."""
    lens = lens_vec(Ie1=0.02, Re1=1.85, n1=4.0, q1=0.8, **RXJ_LIKE)[None].astype(np.float32)
    dyn = np.array([[1.4, 775.0, 0.0, 1.0]], np.float32)
    sheet = dict(rc=RC, rt=RT, n=12, sigma_lo=6.0, sigma_hi=2000.0)
    _, lum0, m0 = oracle.model_tables(lens, dyn, [1823.0], 0.295, 12, 16, (0.02, 10.0), (0.02, 50.0))
    for lam in (0.75, 1.25):
        lf = float(np.float32(lam))
        _, lum, m = oracle.model_tables(lens, dyn, [1823.0], 0.295, 12, 16, (0.02, 10.0), (0.02, 50.0), lam=[lam], sheet=sheet)
        assert m.shape == (1, 28, 3) and np.array_equal(lum, lum0)
        np.testing.assert_allclose(m[0, :16, 0], lf * m0[0, :, 0], rtol=2e-7)
        assert np.array_equal(m[0, :16, 1:], m0[0, :, 1:]) and np.all(m[0, 16:, 2] == 1.0)
        sc = oracle.sigma_crit(1823.0, 775.0, 0.295)
        for R in (0.0, 1.0, 5.0, 20.0, 40.0):
            tot = np.sum(m[0, 16:, 0].astype(np.float64) * np.exp(-R * R / (2 * m[0, 16:, 1].astype(np.float64) ** 2)))
            assert tot == pytest.approx(sc * (1 - lf) * s_paper(R, RC, RT), rel=0.02)
