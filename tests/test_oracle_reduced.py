"""Pins of the oracle's reduced-storage mode (storage = 1; PAPER.md:476 with Eqs. 47-51, :318-331; reading R22 of DESIGN.md): only
pi^xx, pi^xy, pi^xeta, pi^yy, pi^yeta and u^x, u^y, u^eta are state, the rest is algebraic.

What fixes it without reference to the oracle: (1) the same exact / semi-analytic solutions that pin the full mode are solutions of the
reduced scheme too - their pi^{mu nu} is traceless and transverse - so the reduced run must converge to them at the same rate;
(2) Eqs. 47-51 are the constraints pi^{mu nu} u_nu = 0 and g_{mu nu} pi^{mu nu} = 0: after any evolution the exported tensor must satisfy
them to rounding (checked with a dense metric in numpy), as must u.u = 1; (3) the implicit inversion must return the (e, u) a state was
built from; (4) the reduced and the full mode differ by truncation error only: their distance falls with the resolution."""
import math

import numpy as np
import pytest

from paper_1608_06577_b200 import inputs
from test_oracle_flows import boosted_static_state

SLOT = [[4, 5, 6, 7], [5, 8, 9, 10], [6, 9, 11, 12], [7, 10, 12, 13]]


def constraints(f, tau):
    g = np.array([1.0, -1.0, -1.0, -tau * tau])
    pi = np.array([[f["q"][SLOT[m][n]] for n in range(4)] for m in range(4)])
    u = f["u"]
    trace = np.einsum("m,mm...->...", g, pi)
    orth = np.einsum("lm...,m,m...->l...", pi, g, u)
    orth[3] *= tau
    norm = np.einsum("m,m...->...", g, u * u) - 1.0
    scale = np.max(np.abs(pi))
    return np.max(np.abs(trace)) / scale, np.max(np.abs(orth)) / scale, np.max(np.abs(norm))


def test_reduced_mode_keeps_the_constraints_to_rounding_and_tracks_the_full_mode(vo):
    # a generic 3+1d evolution (vorticity, u^eta != 0, bulk on) on two grids whose cell centres coincide (8 and 24 cells per side).
    # The two modes solve the same continuum equations; their distance must be a small fraction of the discretisation error itself
    # (measured as the change of the full-mode solution between the two grids; on a 72-cell grid the distance falls by another 3-6x).
    out = {}
    for n in (8, 24):
        prm = inputs.base_params(nx=n, ny=n, nz=n // 2, dx=2.4 / n, dy=2.4 / n, dz=1.2 / n, tau0=0.9, dtau=0.24 / n, physics=3, xi0=1e9)
        st = inputs.smooth_random_state(prm, seed=13)
        # common initial state: the reduced mode's own projection of the random pi^{mu nu} onto Eqs. 47-51
        o1 = vo.Oracle(dict(prm, storage=1))
        o1.set_initial(st["e"], st["u"], st["pi"], st["Pi"])
        f0 = o1.get_fields()
        assert max(constraints(f0, prm["tau0"])) < 1e-13
        o0 = vo.Oracle(prm)
        o0.set_initial(st["e"], f0["u"], f0["q"][4:14], st["Pi"])
        ns = n // 4
        o0.step(ns); o1.step(ns)
        fa, fb = o0.get_fields(), o1.get_fields()
        tau = o1.status()["tau"]
        c_full, c_red = constraints(fa, tau), constraints(fb, tau)
        assert max(c_red) < 1e-13                      # algebraic: to rounding
        assert max(c_full[:2]) > 1e-7                  # propagated: to truncation error only (:333)
        assert o1.status()["n_inversion_failures"] == 0
        out[n] = (fa, fb)
    on8 = lambda f, k: f["q"][k][0][1::3, 1::3, 1::3]   # the 24-grid sampled at the centres of the 8-grid
    for k in (0, 1, 8, 9, 12, 14):
        S = np.max(np.abs(out[24][0]["q"][k]))
        disc = np.max(np.abs(out[8][0]["q"][k][0] - on8(out[24][0], k))) / S
        dist = np.max(np.abs(out[24][0]["q"][k] - out[24][1]["q"][k])) / S
        assert dist < 0.1 * disc, (k, dist, disc)


def test_reduced_mode_viscous_gubser(vo):
    # PAPER.md 5.7 (config 2 physics): same bounds and convergence as the full mode in tests/test_oracle_flows.py
    def run(n, d, dt, ns):
        prm, init, _, (x, That, pibar) = inputs.config_gubser(n=n, d=d, eta_over_s=0.2, theta=1.8)
        prm.update(rho_max=1e30, dtau=dt, storage=1)
        o = vo.Oracle(prm)
        o.set_initial(init["e"], init["u"], init["pi"])
        o.step(ns)
        tau = o.status()["tau"]
        f = o.get_fields()
        X, Y = np.meshgrid(x, x, indexing="xy")
        ea, ua, pia = inputs.gubser_fields(tau, X, Y, That, pibar)
        m = np.sqrt(X * X + Y * Y) < 3.0
        l2 = lambda a, b: np.sqrt(np.sum((a[m] - b[m]) ** 2) / np.sum(b[m] ** 2))
        assert o.status()["n_inversion_failures"] == 0
        return dict(e=l2(f["e"][0, 0], ea), ux=l2(f["u"][1][0, 0], ua[1]), pinn=l2(f["q"][13][0, 0], pia[9]), pixx=l2(f["q"][8][0, 0], pia[4]),
                    pixy=l2(f["q"][9][0, 0], pia[5]), pitt=l2(f["q"][4][0, 0], pia[0]), pitx=l2(f["q"][5][0, 0], pia[1]))
    e2 = run(61, 0.2, 0.025, 20)
    e1 = run(121, 0.1, 0.0125, 40)
    bound = dict(e=2e-2, ux=1.2e-2, pinn=2e-2, pixx=6e-2, pixy=0.13, pitt=7e-2, pitx=7e-2)
    for k in e1:
        assert e1[k] < bound[k], (k, e1[k])
        assert e1[k] < 0.62 * e2[k], (k, e1[k], e2[k])


def test_reduced_mode_boosted_static_exact_solution(vo):
    # the exact solution of tests/test_oracle_flows.py (u^eta != 0: every Christoffel term, and Eq. 50 / 51 with v_eta != 0) in reduced mode
    nz = 41
    prm = inputs.base_params(nx=3, ny=3, nz=nz, dz=0.025, tau0=2.0, dtau=0.002, eos=0, physics=1, zeta_model=0, rho_max=1e30,
                             tau_relax_floor_over_dtau=0.0, storage=1)
    e0 = 30.0
    amp = 0.05 * e0
    tau0 = prm["tau0"]
    itp = (e0 / 13.8) ** 0.25 / (5 * 0.2)
    eta = inputs.centred_axis(nz, prm["dz"])
    t0 = tau0 * np.cosh(eta)

    def state(tau):
        dec = np.exp(-(tau * np.cosh(eta) - t0.min()) * itp)[:, None, None]
        e, u, pi = boosted_static_state(prm, 1.0, 0.6, -0.3, 0.4, tau, e0)
        return e, u, pi * amp * dec[None, None]

    e, u, pi = state(tau0)
    o = vo.Oracle(prm)
    o.set_initial(e, u, pi)
    o.set_uprev(state(tau0 - prm["dtau"])[1])
    o.step(10)
    tau = o.status()["tau"]
    f = o.get_fields()
    ee, uu, pp = state(tau)
    k = slice(nz // 2 - 6, nz // 2 + 7)
    np.testing.assert_allclose(f["e"][0, k], ee[0, k], rtol=2e-5)
    np.testing.assert_allclose(f["u"][3][0, k], uu[3][0, k], rtol=1e-5, atol=2e-7)
    for n in range(10):
        np.testing.assert_allclose(f["q"][4 + n][0, k], pp[n][0, k], rtol=1e-4, atol=1e-5 * amp)


def test_implicit_inversion_returns_the_state_it_was_built_from(vo):
    # one cell: q from (e, u, the five independent components, Pi) by Eqs. 32-33 with the algebraic pi^{tau mu}; post() must give back e, u
    # although pi^{tau mu} (hence E and M_i of Eq. 72) depend on the velocity it is solving for.  Start far from the answer (guess = rest).
    tau = 1.7
    prm = inputs.base_params(nx=1, ny=1, nz=1, tau0=tau, physics=3, storage=1, rho_max=1e30)
    shp = (1, 1, 1, 1)
    e0 = 9.0
    ui = np.array([0.5, -0.3, 0.2])
    ut = math.sqrt(1 + ui[0] ** 2 + ui[1] ** 2 + tau * tau * ui[2] ** 2)
    u = np.array([ut, *ui]).reshape((4,) + shp)
    pi = np.zeros((10,) + shp)
    pi[4], pi[5], pi[6], pi[7], pi[8] = 0.8, -0.5, 0.3, -0.6, 0.2          # large: |pi| ~ 0.1 (e + p)
    o = vo.Oracle(prm)
    o.set_initial(np.full(shp, e0), u, pi, np.full(shp, -0.4))
    f0 = o.get_fields()
    assert max(constraints(f0, tau)) < 1e-14
    # overwrite u (the fixed point's starting velocity) with the rest frame and e (Newton's guess) with something else
    for m in range(1, 4):
        o.raw("u", m)[...] = 0.0
    o.raw("u", 0)[...] = 1.0
    o.raw("e")[...] = 3.0
    o.ghost()
    o.step(0)
    import ctypes
    o.L.vho_post_guess.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double]
    o.L.vho_post_guess(o.h, 0, tau)
    f1 = o.get_fields()
    assert f1["e"][0, 0, 0, 0] == pytest.approx(e0, rel=1e-11)
    assert np.allclose(f1["u"][:, 0, 0, 0, 0], [ut, *ui], rtol=1e-11)
    assert np.allclose(f1["q"][:, 0, 0, 0, 0], f0["q"][:, 0, 0, 0, 0], rtol=1e-10, atol=1e-13)
    assert o.status()["n_inversion_failures"] == 0


def test_reduced_mode_normalises_u_prev_at_its_own_time_level(vo):
    """Pin of Solver::set_uprev in reduced mode (R22: u^tau of a stored velocity is the normalisation u.u = 1 with the metric of the
    time level the velocity belongs to - for u^{n-1} that is tau0 - dtau, g_{eta eta} = -(tau0 - dtau)^2, Eq. 27).  The exact boosted-static
    solution fixes it: D u^tau = (u^tau_n - u^tau_{n-1})/dtau enters sigma^{mu nu} at the first step (A.5-A.12, :424), and a u^tau_{n-1}
    normalised with tau0 instead is off by ~ tau0 (u^eta)^2 dtau / u^tau - an O(1) error in that derivative, which drives pi^{mu nu} away
    from the solution ninety times faster than the truncation error does.  The u^tau handed to set_uprev is deliberately wrong (zero):
    in reduced mode it is not state and must not be used."""
    nz = 41
    e0 = 30.0
    amp = 0.05 * e0

    def first_step_error(storage, u_tau_prev):
        prm = inputs.base_params(nx=3, ny=3, nz=nz, dz=0.025, tau0=2.0, dtau=0.002, eos=0, physics=1, zeta_model=0, rho_max=1e30,
                                 tau_relax_floor_over_dtau=0.0, storage=storage)
        tau0 = prm["tau0"]
        itp = (e0 / 13.8) ** 0.25 / (5 * 0.2)
        eta = inputs.centred_axis(nz, prm["dz"])
        t0 = tau0 * np.cosh(eta)

        def state(tau):
            dec = np.exp(-(tau * np.cosh(eta) - t0.min()) * itp)[:, None, None]
            e, u, pi = boosted_static_state(prm, 1.0, 0.6, -0.3, 0.4, tau, e0)
            return e, u, pi * amp * dec[None, None]

        e, u, pi = state(tau0)
        up = state(tau0 - prm["dtau"])[1].copy()
        if u_tau_prev == "zero":
            up[0] = 0.0
        elif u_tau_prev == "normalised at tau0":
            up[0] = np.sqrt(1.0 + up[1] ** 2 + up[2] ** 2 + tau0 ** 2 * up[3] ** 2)
        o = vo.Oracle(prm)
        o.set_initial(e, u, pi)
        o.set_uprev(up)
        o.step(1)
        f, pp = o.get_fields(), state(o.status()["tau"])[2]
        k = slice(nz // 2 - 6, nz // 2 + 7)
        return max(np.max(np.abs(f["q"][4 + n][0, k] - pp[n][0, k])) for n in range(10)) / amp

    bar = 2e-6
    assert first_step_error(1, "zero") < bar                       # measured 5.2e-7: truncation error of one step
    # what the bar would catch - the full mode takes u^tau_{n-1} as given, so the mistake can be fed to it from outside:
    assert first_step_error(0, "exact") < bar
    assert first_step_error(0, "normalised at tau0") > 10 * bar    # measured 4.6e-5
