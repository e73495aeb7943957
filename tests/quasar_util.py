"""Test-side helpers for the quasar terms (Eq. 35-36): find the images of a point source by a route that does NOT
go through the oracle's own Newton iteration -- scipy.optimize.root (MINPACK hybrid, numerical Jacobian) on the lens
equation built from oracle.deflection, started from a polar grid -- and make seeded mock "observed" positions / delays.
Test infrastructure (imports oracle/), never imported by the product."""
import numpy as np
from scipy.optimize import root

RXJ_LIKE = dict(xl=0.0, yl=0.0, thetaE=1.65, gamma=2.0, q=0.8, pa=np.radians(30.0), gext=0.09, phiext=1.42)


def find_images(oracle, p, beta, rmax=3.5, nr=14, nphi=24, rmin=0.15):
    """All solutions of theta - alpha(theta) = beta with |theta - centre| > rmin (the central, demagnified image of a
    singular lens is excluded), deduplicated, sorted by polar angle."""
    p = np.asarray(p, np.float64)

    def f(t):
        ax, ay = oracle.deflection(p, t[0], t[1])
        return [t[0] - ax - beta[0], t[1] - ay - beta[1]]

    sols = []
    for r in np.linspace(0.3, rmax, nr):
        for ph in np.linspace(0, 2 * np.pi, nphi, endpoint=False):
            s = root(f, [p[0] + r * np.cos(ph), p[1] + r * np.sin(ph)], tol=1e-14)
            if not s.success or np.hypot(*f(s.x)) > 1e-11:
                continue
            if np.hypot(s.x[0] - p[0], s.x[1] - p[1]) < rmin:
                continue
            if all(np.hypot(*(s.x - o)) > 1e-6 for o in sols):
                sols.append(s.x.copy())
    sols.sort(key=lambda t: np.arctan2(t[1] - p[1], t[0] - p[0]))
    return np.array(sols)


def fermat(oracle, p, theta, beta):
    """Eq. 2."""
    return 0.5 * ((theta[0] - beta[0]) ** 2 + (theta[1] - beta[1]) ** 2) - oracle.potential(p, theta[0], theta[1])


def mock_quasar(oracle, p, beta, ddt, seed=0, sigma_theta=0.004, frac_dt=0.03, noise=True):
    """Observed image positions / delays of a point source at beta seen through lens vector p (Eq. 33, Eq. 3-4),
    reference image = the first arrival; positions + N(0, sigma_theta), delays * (1 + N(0, frac_dt))."""
    th = find_images(oracle, p, beta)
    assert len(th) in (2, 4), f"expected a double or a quad, found {len(th)} images"
    phi = np.array([fermat(oracle, p, t, beta) for t in th])
    ref = int(np.argmin(phi))
    dt = oracle.tdelay_const() * ddt * (phi - phi[ref])
    rng = np.random.default_rng(seed)
    if noise:
        th = th + rng.normal(0.0, sigma_theta, th.shape)
        dt = dt * (1.0 + rng.normal(0.0, frac_dt, dt.shape))
    sd = np.maximum(frac_dt * np.abs(dt), 0.25)
    sd[ref] = 0.0
    return dict(theta=th, sigma_theta=np.full(len(th), sigma_theta), ref=ref, dt_obs=dt, sigma_dt=sd)
