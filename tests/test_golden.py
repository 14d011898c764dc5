"""Pins from tests/golden/: closed-form / ODE values (cited there) against the independent evaluators and the oracle."""
import os

import numpy as np
import pytest

import analytic
from paper_1608_06577_b200 import inputs

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
HB = inputs.HBARC


def table(name):
    return np.loadtxt(os.path.join(GOLD, name), comments="#", ndmin=2)


def test_riemann_plateau_fixture():
    for eL, eR, ep, vp, Vs in table("riemann_plateau.txt"):
        g = analytic.riemann_plateau(eL, eR)
        assert g[0] / eR == pytest.approx(ep, rel=1e-8) and g[1] == pytest.approx(vp, rel=1e-7) and g[2] == pytest.approx(Vs, rel=1e-7)


def test_gubser_ode_fixture():
    That, pibar = inputs.gubser_ode(0.2, 5.0)
    t = table("gubser_ode.txt")
    assert That(t[:, 0]) == pytest.approx(t[:, 1], rel=2e-7)
    assert pibar(t[:, 0]) == pytest.approx(t[:, 2], rel=2e-6, abs=1e-12)


def test_bjorken_fixture_against_ode_and_oracle(vo):
    t = table("bjorken_ode.txt")
    T0 = 0.6 / HB
    e0 = 13.8 * T0**4
    tau0 = 0.25
    pi0 = 4.0 / 3.0 * 0.2 * (4.0 / 3.0 * e0 / T0) / tau0
    eos = lambda e: (e / 3, 1 / 3, (e / 13.8) ** 0.25)
    tr = lambda e, p, cs2, T: (T / (5 * 0.2), (e + p) / 5, 0.0, 0.0)
    co = dict(delta_pipi=4 / 3, tau_pipi=10 / 7, lambda_piPi=6 / 5, delta_PiPi=2 / 3, lambda_Pipi_coef=8 / 5)
    ref = analytic.bjorken_ode(e0, pi0, 0.0, tau0, list(t[:, 0]), eos, tr, co)
    assert ref[0] / e0 == pytest.approx(t[:, 1], rel=1e-6)
    assert ref[1] / e0 == pytest.approx(t[:, 2], rel=1e-6)
    # the 3+1d oracle on a homogeneous 3^3 grid lands on the fixture (tau = 0.5, 1.0): pins G_c^tau, theta, sigma^{eta eta}, Eq. 40
    prm = inputs.base_params(nx=3, ny=3, nz=3, tau0=tau0, dtau=0.0025, eos=0, physics=1, zeta_model=0, rho_max=1e30,
                             tau_relax_floor_over_dtau=0.0)
    shp = (1, 3, 3, 3)
    pi = np.zeros((10,) + shp)
    pi[4] = pi0 / 2; pi[7] = pi0 / 2; pi[9] = -pi0 / tau0**2      # pi^xx = pi^yy = pi/2, tau^2 pi^{eta eta} = -pi (Eq. 78 convention)
    o = vo.Oracle(prm)
    o.set_initial(np.full(shp, e0), inputs.rest_velocity(shp), pi, None)
    done = 0
    for tau, ee, pp in t[:2]:
        n = int(round((tau - tau0) / prm["dtau"]))
        o.step(n - done); done = n
        f = o.get_fields()
        assert f["e"][0, 1, 1, 1] / e0 == pytest.approx(ee, rel=2e-4)
        assert -tau * tau * f["q"][13][0, 1, 1, 1] / e0 == pytest.approx(pp, rel=2e-3)
