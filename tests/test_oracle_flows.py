"""T2-T6: the oracle against the Bjorken ODEs (Eqs. 77-81), ideal Gubser flow (Eqs. 82-85), the semi-analytic
viscous Gubser solution, the boosted-static exact solution and the invariants of
Eqs. 47-51 / :489.  Regularisation is switched off (rho_max = 1e30) where a comparator is an exact solution of the
un-regularised equations: with rho_max = 1 tanh(rho)/rho differs from 1 at O(rho^2/3), rho ~ |pi|/e."""
import math

import numpy as np
import pytest

import analytic
from paper_1608_06577_b200 import inputs

HB = inputs.HBARC


def bjorken_run(vo, prm, e0, pi0, Pi0, taus):
    shp = (1, prm["nz"], prm["ny"], prm["nx"])
    tau0 = prm["tau0"]
    pi = np.zeros((10,) + shp)
    pi[4] = pi0 / 2; pi[7] = pi0 / 2; pi[9] = -pi0 / tau0**2      # pi^xx = pi^yy = pi/2, tau^2 pi^{eta eta} = -pi
    o = vo.Oracle(prm)
    o.set_initial(np.full(shp, e0), inputs.rest_velocity(shp), pi, np.full(shp, Pi0))
    out = []
    for t in taus:
        n = int(round((t - o.status()["tau"]) / prm["dtau"]))
        o.step(n)
        f = o.get_fields()
        tau = o.status()["tau"]
        c = (0, prm["nz"] // 2, prm["ny"] // 2, prm["nx"] // 2)
        out.append((f["e"][c], -tau * tau * f["q"][13][c], f["q"][14][c], f["q"][8][c], f["q"][11][c]))
    return np.array(out), o


def test_conformal_bjorken_values_of_the_paper_setup(vo):
    # PAPER.md section 5.4 / Fig. 10: T0 = 0.6 GeV, tau0 = 0.25 fm, eta/s = 0.2, pi0 = Navier-Stokes (4/3) eta/tau0
    T0 = 0.6 / HB
    e0 = 13.8 * T0**4
    tau0 = 0.25
    pi0 = 4.0 / 3.0 * 0.2 * (4.0 / 3.0 * e0 / T0) / tau0
    assert pi0 / e0 == pytest.approx(0.46773803, rel=1e-7)
    prm = inputs.base_params(nx=3, ny=3, nz=3, tau0=tau0, dtau=0.0025, eos=0, physics=1, zeta_model=0, rho_max=1e30,
                             tau_relax_floor_over_dtau=0.0)
    taus = [0.5, 1.0, 2.0]
    got, o = bjorken_run(vo, prm, e0, pi0, 0.0, taus)
    # independent ODE solve of Eqs. 77-78
    eos = lambda e: (e / 3, 1 / 3, (e / 13.8) ** 0.25)
    tr = lambda e, p, cs2, T: (T / (5 * 0.2), (e + p) / 5, 0.0, 0.0)
    co = dict(delta_pipi=4 / 3, tau_pipi=10 / 7, lambda_piPi=6 / 5, delta_PiPi=2 / 3, lambda_Pipi_coef=8 / 5)
    ref = analytic.bjorken_ode(e0, pi0, 0.0, tau0, taus, eos, tr, co)
    # SURVEY T2 values (derived there from the same ODEs)
    assert ref[0] / e0 == pytest.approx([0.50719836, 0.23350857, 0.10179714], rel=1e-6)
    assert ref[1] / e0 == pytest.approx([0.13611997, 0.039452114, 0.010843441], rel=1e-6)
    np.testing.assert_allclose(got[:, 0], ref[0], rtol=2e-4)
    np.testing.assert_allclose(got[:, 1], ref[1], rtol=2e-3)
    # pi^xx = pi^yy = pi/2 stays (pins the xx/yy rows of sigma and I_4), no inversion failure, homogeneous
    # (the two are separate discrete equations, xx without and eta-eta with G_pi and tau^2: equal up to truncation error)
    np.testing.assert_allclose(got[:, 3], got[:, 1] / 2, rtol=1e-3)
    np.testing.assert_allclose(got[:, 4], got[:, 3], rtol=1e-13)
    assert o.status()["n_inversion_failures"] == 0
    f = o.get_fields()
    assert np.ptp(f["e"]) <= 1e-12 * f["e"].mean()
    assert np.max(np.abs(f["u"][1:])) < 1e-14


def test_bjorken_is_second_order_in_dtau(vo):
    # reading R7: stage 2 and the first Post at tau^n + dtau.  Heun is 2nd order only then.
    T0 = 0.6 / HB
    e0 = 13.8 * T0**4
    pi0 = 0.3 * e0
    eos = lambda e: (e / 3, 1 / 3, (e / 13.8) ** 0.25)
    tr = lambda e, p, cs2, T: (T / (5 * 0.2), (e + p) / 5, 0.0, 0.0)
    co = dict(delta_pipi=4 / 3, tau_pipi=10 / 7, lambda_piPi=6 / 5, delta_PiPi=2 / 3, lambda_Pipi_coef=8 / 5)
    ref = analytic.bjorken_ode(e0, pi0, 0.0, 0.5, [1.0], eos, tr, co)
    errs = []
    for dt in (0.02, 0.01, 0.005):
        prm = inputs.base_params(nx=1, ny=1, nz=1, tau0=0.5, dtau=dt, eos=0, physics=1, zeta_model=0, rho_max=1e30,
                                 tau_relax_floor_over_dtau=0.0)
        got, _ = bjorken_run(vo, prm, e0, pi0, 0.0, [1.0])
        errs.append(abs(got[0, 0] - ref[0][0]) / ref[0][0])
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.15) and errs[1] / errs[2] == pytest.approx(4.0, rel=0.15)


def test_nonconformal_bjorken_with_bulk(vo):
    # PAPER.md section 5.5, Eqs. 79-81, with the EOS and zeta/s of BASELINE.json configs 3-5 (the lattice EOS is NEXT-1)
    prm = inputs.base_params(nx=2, ny=2, nz=2, tau0=0.5, dtau=0.0025, rho_max=1e30)
    e0 = 12.0 / HB
    p = lambda e: (e / 3) * (1 - 0.4 * np.exp(-e / prm["eos_e0"]))
    cs2 = lambda e: (1 / 3) * (1 - 0.4 * np.exp(-e / prm["eos_e0"]) * (1 - e / prm["eos_e0"]))
    eos = lambda e: (p(e), cs2(e), (e / 13.8) ** 0.25)
    clamp = 1.0 / (5 * prm["dtau"])

    def tr(e, pp, c2, T):
        zs = 0.1 * math.exp(-(((T * HB) - 0.18) / 0.03) ** 2)
        itP = min(T * (1 / 3 - c2) ** 2 / (5 * zs), clamp)
        return (T / (5 * 0.2), (e + pp) / 5, itP, zs * (e + pp) / T * itP)

    co = dict(delta_pipi=4 / 3, tau_pipi=10 / 7, lambda_piPi=6 / 5, delta_PiPi=2 / 3, lambda_Pipi_coef=8 / 5)
    taus = [1.0, 3.0, 6.0]
    pi0, Pi0 = 0.1 * e0, -0.01 * e0
    ref = analytic.bjorken_ode(e0, pi0, Pi0, 0.5, taus, eos, tr, co)
    got, o = bjorken_run(vo, prm, e0, pi0, Pi0, taus)
    np.testing.assert_allclose(got[:, 0], ref[0], rtol=3e-4)
    np.testing.assert_allclose(got[:, 1], ref[1], rtol=3e-3)
    np.testing.assert_allclose(got[:, 2], ref[2], rtol=5e-3, atol=1e-6 * e0)
    assert abs(ref[2][-1]) > 1e-5 * ref[0][-1]       # the bulk channel is actually exercised
    assert o.status()["n_inversion_failures"] == 0


def test_ideal_gubser_flow(vo):
    # PAPER.md section 5.6 (Eqs. 82-85): tau0 = 1, T0hat = 1.2, q = 1; compare at tau = 1.5 inside the causal interior
    n, d = 101, 0.1
    prm, init, _, (x, That, pibar) = inputs.config_gubser(n=n, d=d, eta_over_s=0.0, theta=1.8)
    prm["dtau"] = 0.0125
    # the initial profile itself is Eq. 82 and Eqs. 83-85 with outward flow (R16)
    c = n // 2
    r = np.abs(x)
    np.testing.assert_allclose((init["e"][0, 0, c] / 13.8) ** 0.25, analytic.gubser_ideal_T(1.0, r), rtol=1e-12)
    np.testing.assert_allclose(init["u"][1][0, 0, c], np.sign(x) * np.sinh(analytic.gubser_kappa(1.0, r)), rtol=1e-12, atol=1e-15)
    o = vo.Oracle(prm)
    o.set_initial(init["e"], init["u"])
    o.step(40)
    tau = o.status()["tau"]
    assert tau == pytest.approx(1.5)
    f = o.get_fields()
    m = r < 3.0
    T = (f["e"][0, 0, c] / 13.8) ** 0.25
    np.testing.assert_allclose(T[m], analytic.gubser_ideal_T(tau, r[m]), rtol=8e-3)   # dx = 0.1 (twice the paper's)
    np.testing.assert_allclose(f["u"][1][0, 0, c][m], np.sign(x[m]) * np.sinh(analytic.gubser_kappa(tau, r[m])), rtol=2e-2, atol=2e-3)
    # cylindrical symmetry on the Cartesian grid (:718): x <-> y transpose and reflections
    np.testing.assert_allclose(f["e"][0, 0], f["e"][0, 0].T, rtol=1e-12)
    np.testing.assert_allclose(f["e"][0, 0], f["e"][0, 0][::-1, ::-1], rtol=1e-12)
    np.testing.assert_allclose(f["u"][1][0, 0], f["u"][2][0, 0].T, rtol=1e-11, atol=1e-13)
    assert o.status()["n_inversion_failures"] == 0


def test_viscous_gubser_flow(vo):
    # PAPER.md section 5.7: eta/s = 0.2, tau_pipi = 0, theta = 1.8; ODE pair re-derived in SURVEY 8(c) T4
    n, d = 121, 0.1
    prm, init, _, (x, That, pibar) = inputs.config_gubser(n=n, d=d, eta_over_s=0.2, theta=1.8)
    prm["rho_max"] = 1e30
    # ODE pins (derived there)
    assert That(np.array([-5.0, -2.0, -1.0, 1.0, 2.0])) == pytest.approx([0.13267347, 0.55515668, 0.90881844, 0.90438090, 0.52109399], rel=2e-7)
    assert pibar(np.array([-5.0, -2.0, -1.0, 1.0, 2.0])) == pytest.approx([0.52766587, 0.48509728, 0.16527408, 0.082379481, 0.19829894], rel=2e-6)
    # ideal limit of the ODE is Eq. 82 on the centre line
    Ti, _ = inputs.gubser_ode(0.0, 5.0)
    e_, u_, _ = inputs.gubser_fields(2.0, np.array([0.0, 1.0]), np.array([0.0, 0.5]), Ti, lambda r: np.zeros_like(r))
    np.testing.assert_allclose((e_ / 13.8) ** 0.25, analytic.gubser_ideal_T(2.0, np.array([0.0, math.sqrt(1.25)])), rtol=1e-12)
    # generated pi^{mu nu}: traceless and orthogonal to u (Eqs. 47-51)
    pi, u = init["pi"][:, 0, 0], init["u"][:, 0, 0]
    tau0 = 1.0
    tr = pi[0] - pi[4] - pi[7] - tau0**2 * pi[9]
    assert np.max(np.abs(tr)) < 1e-13
    assert np.max(np.abs(pi[0] * u[0] - pi[1] * u[1] - pi[2] * u[2])) < 1e-13
    assert np.max(np.abs(pi[1] * u[0] - pi[4] * u[1] - pi[5] * u[2])) < 1e-13
    def run(n, d, dt, ns):
        prm, init, _, (x, That, pibar) = inputs.config_gubser(n=n, d=d, eta_over_s=0.2, theta=1.8)
        prm["rho_max"] = 1e30
        prm["dtau"] = dt
        o = vo.Oracle(prm)
        o.set_initial(init["e"], init["u"], init["pi"])
        o.step(ns)
        tau = o.status()["tau"]
        f = o.get_fields()
        X, Y = np.meshgrid(x, x, indexing="xy")
        ea, ua, pia = inputs.gubser_fields(tau, X, Y, That, pibar)
        m = np.sqrt(X * X + Y * Y) < 3.0
        l2 = lambda a, b: np.sqrt(np.sum((a[m] - b[m]) ** 2) / np.sum(b[m] ** 2))
        errs = dict(e=l2(f["e"][0, 0], ea), ux=l2(f["u"][1][0, 0], ua[1]), uy=l2(f["u"][2][0, 0], ua[2]),
                    pinn=l2(f["q"][13][0, 0], pia[9]), pixx=l2(f["q"][8][0, 0], pia[4]), piyy=l2(f["q"][11][0, 0], pia[7]),
                    pixy=l2(f["q"][9][0, 0], pia[5]), pitt=l2(f["q"][4][0, 0], pia[0]), pitx=l2(f["q"][5][0, 0], pia[1]))
        return errs, f, o, tau

    # relative L2 errors inside r < 3 (the outflow boundary of the box is not Gubser-symmetric) at dx = 0.2 and 0.1
    # (the paper uses 0.05): every field converges towards the semi-analytic solution at between 1st and 2nd order
    # (theta = 1.8 limiter; the pointwise error peaks in the ring r ~ 1.2-1.6 where pibar changes sign)
    e2, _, _, _ = run(61, 0.2, 0.025, 20)
    e1, f, o, tau = run(121, 0.1, 0.0125, 40)
    bound = dict(e=2e-2, ux=1.2e-2, uy=1.2e-2, pinn=2e-2, pixx=6e-2, piyy=6e-2, pixy=0.13, pitt=7e-2, pitx=7e-2)
    for k in e1:
        assert e1[k] < bound[k], (k, e1[k])
        assert e1[k] < 0.62 * e2[k], (k, e1[k], e2[k])
    n = 121
    # centre-line values: (tau=1.5, r=0) T = 0.75862052 fm^-1, tau^2 pi^{eta eta} = 0.11160348 fm^-4
    c = n // 2
    assert (f["e"][0, 0, c, c] / 13.8) ** 0.25 == pytest.approx(0.75862052, rel=2e-3)
    assert tau * tau * f["q"][13][0, 0, c, c] == pytest.approx(0.11160348, rel=2e-2)
    assert o.status()["n_inversion_failures"] == 0


def boosted_static_state(prm, pizz, pixz, pixx, pixy, tau, e0):
    """homogeneous fluid at rest in Minkowski space seen from Milne coordinates."""
    nx, ny, nz = prm["nx"], prm["ny"], prm["nz"]
    eta = inputs.centred_axis(nz, prm["dz"])[:, None, None] * np.ones((1, ny, nx))
    ch, sh = np.cosh(eta), np.sinh(eta)
    shp = (1, nz, ny, nx)
    u = np.zeros((4,) + shp)
    u[0, 0] = ch; u[3, 0] = -sh / tau
    pi = np.zeros((10,) + shp)
    piyz = 0.7 * pixz
    piyy = -(pixx + pizz)                              # traceless in Minkowski: pi^xx + pi^yy + pi^zz = 0 (pi^{tt}=0 at rest)
    pi[0, 0] = sh * sh * pizz
    pi[1, 0] = -sh * pixz
    pi[2, 0] = -sh * piyz
    pi[3, 0] = -sh * ch * pizz / tau
    pi[4, 0] = pixx
    pi[5, 0] = pixy
    pi[6, 0] = ch * pixz / tau
    pi[7, 0] = piyy
    pi[8, 0] = ch * piyz / tau
    pi[9, 0] = ch * ch * pizz / tau**2
    return np.full(shp, e0), u, pi


def test_boosted_static_exact_solution(vo):
    # pi^{ij}(t) = pi0^{ij} exp(-t/tau_pi), e constant, in Minkowski; t = tau cosh(eta).  Every Christoffel term with
    # u^eta != 0 (G_c, G_pi, the Gamma pieces of sigma, theta, Du) must cancel against flux / time-derivative terms.
    nz = 41
    prm = inputs.base_params(nx=3, ny=3, nz=nz, dz=0.025, tau0=2.0, dtau=0.002, eos=0, physics=1, zeta_model=0,
                             rho_max=1e30, tau_relax_floor_over_dtau=0.0)
    e0 = 30.0
    amp = 0.05 * e0      # exact at any amplitude; large enough that the O(d eta^2) error of sigma (times eta/tau_pi) is relatively small
    tau0 = prm["tau0"]
    T = (e0 / 13.8) ** 0.25
    itp = T / (5 * 0.2)
    eta = inputs.centred_axis(nz, prm["dz"])
    t0 = tau0 * np.cosh(eta)

    def state(tau):
        dec = np.exp(-(tau * np.cosh(eta) - t0.min()) * itp)[:, None, None]
        e, u, pi = boosted_static_state(prm, 1.0, 0.6, -0.3, 0.4, tau, e0)
        return e, u, pi * amp * dec[None, None]

    e, u, pi = state(tau0)
    o = vo.Oracle(prm)
    o.set_initial(e, u, pi)
    _, um, _ = state(tau0 - prm["dtau"])
    o.set_uprev(um)                                   # exact u^{n-1}: u depends on tau here
    ns = 10
    o.step(ns)
    tau = o.status()["tau"]
    f = o.get_fields()
    ee, uu, pp = state(tau)
    k = slice(nz // 2 - 6, nz // 2 + 7)               # interior, outside the domain of influence of the eta boundary
    np.testing.assert_allclose(f["e"][0, k], ee[0, k], rtol=2e-5)
    np.testing.assert_allclose(f["u"][0][0, k], uu[0][0, k], rtol=2e-6)
    np.testing.assert_allclose(f["u"][3][0, k], uu[3][0, k], rtol=1e-5, atol=2e-7)
    assert np.max(np.abs(f["u"][1][0, k])) < 1e-6 and np.max(np.abs(f["u"][2][0, k])) < 1e-6
    for n in range(10):
        ref = pp[n][0, k]
        np.testing.assert_allclose(f["q"][4 + n][0, k], ref, rtol=1e-4, atol=1e-5 * amp)
    # error is truncation error: it falls when dtau and d(eta) are halved together
    def err(dz, dt, ns):
        prm2 = dict(prm, nz=nz if dz == 0.025 else 2 * nz - 1, dz=dz, dtau=dt)
        eta2 = inputs.centred_axis(prm2["nz"], dz)
        def st(tau):
            dec = np.exp(-(tau * np.cosh(eta2) - tau0) * itp)[:, None, None]
            e, u, pi = boosted_static_state(prm2, 1.0, 0.6, -0.3, 0.4, tau, e0)
            return e, u, pi * amp * dec[None, None]
        e, u, pi = st(tau0)
        o = vo.Oracle(prm2); o.set_initial(e, u, pi); o.set_uprev(st(tau0 - dt)[1]); o.step(ns)
        f = o.get_fields(); _, _, pr = st(o.status()["tau"])
        c = prm2["nz"] // 2
        kk = slice(c - 3, c + 4)
        return max(np.max(np.abs(f["q"][4 + n][0, kk] - pr[n][0, kk])) for n in range(10)) / amp
    e1, e2 = err(0.025, 0.002, 10), err(0.0125, 0.001, 20)
    assert e2 < 0.6 * e1


def test_invariants_on_a_generic_evolution(vo):
    # T5: starting from a state that satisfies Eqs. 47-51, the trace and pi.u stay at truncation-error level; u.u = 1 (:489)
    prm, init, _ = inputs.config_3d(12, 10, 8, n_hot=3, width=0.4, seed=11, rho_max=1e30)
    o = vo.Oracle(prm)
    o.set_initial(init["e"], init["u"])
    o.step(6)
    f = o.get_fields()
    st = o.status()
    tau = st["tau"]
    q, u = f["q"], f["u"]
    uu = u[0] ** 2 - u[1] ** 2 - u[2] ** 2 - tau**2 * u[3] ** 2
    assert np.max(np.abs(uu - 1)) < 1e-12
    assert st["n_inversion_failures"] == 0 and st["n_nonfinite"] == 0
    scale = np.max(np.abs(q[4:14]))
    assert scale > 0
    tr = q[4] - q[8] - q[11] - tau**2 * q[13]
    assert np.max(np.abs(tr)) < 0.05 * scale
    piu = q[4] * u[0] - q[5] * u[1] - q[6] * u[2] - tau**2 * q[7] * u[3]
    assert np.max(np.abs(piu)) < 0.05 * scale
    # Landau matching: T^{tau mu} rebuilt from the primitives (Eqs. 32-33) reproduces q (regularisation off here: pi is
    # rescaled AFTER the inversion, steps 2-3 / reading R8, which breaks this identity by (1 - tanh(rho)/rho) |pi|)
    P = f["p"] + q[14]
    np.testing.assert_allclose((f["e"] + P) * u[0] ** 2 - P + q[4], q[0], rtol=1e-12)
    for i in (1, 2, 3):
        np.testing.assert_allclose((f["e"] + P) * u[0] * u[i] + q[4 + i], q[i], rtol=1e-9, atol=1e-13)


def test_2plus1d_is_eta_independent_limit_of_3plus1d(vo):
    # PAPER.md:474 / SURVEY T7: an eta-independent 3+1d run reproduces the nz = 1 run
    prm2, init2, _ = inputs.config_batched2d(n_batch=1, n=14, n_hot=3, seed=5)
    o2 = vo.Oracle(prm2); o2.set_initial(init2["e"], init2["u"]); o2.step(4)
    prm3 = dict(prm2, nz=3)
    e3 = np.repeat(init2["e"], 3, axis=1)
    o3 = vo.Oracle(prm3); o3.set_initial(e3, inputs.rest_velocity(e3.shape)); o3.step(4)
    f2, f3 = o2.get_fields(), o3.get_fields()
    for k in range(3):
        np.testing.assert_allclose(f3["q"][:, 0, k], f2["q"][:, 0, 0], rtol=1e-13, atol=1e-15)
        np.testing.assert_allclose(f3["e"][0, k], f2["e"][0, 0], rtol=1e-13)
    assert np.max(np.abs(f3["q"][3])) == 0.0 and np.max(np.abs(f3["u"][3])) == 0.0
