"""Pins for the scalar pieces of the oracle (oracle/vh_oracle.hpp): minmod (Eqs. 67-68), EOS, transport
coefficients (Eqs. 10-16), Newton inversion (Eqs. 52-54, 72 and the closed form of PAPER.md:339),
Heun combination (Eqs. 69-71), ghost cells (Eqs. 75-76), q^0 construction (Eqs. 32-33)."""
import math

import numpy as np
import pytest

from paper_1608_06577_b200 import inputs


def test_minmod_definition_cases(vo):
    # Eq. 68 with sgn(0)=0 (reading R10): 0 unless all three share a strict sign, then the smallest magnitude
    assert vo.minmod3(1.0, 2.0, 3.0) == 1.0
    assert vo.minmod3(3.0, 2.0, 0.5) == 0.5
    assert vo.minmod3(-1.0, -2.0, -3.0) == -1.0
    assert vo.minmod3(-4.0, -2.0, -3.0) == -2.0
    assert vo.minmod3(1.0, -2.0, 3.0) == 0.0
    assert vo.minmod3(1.0, 2.0, -3.0) == 0.0
    assert vo.minmod3(-1.0, 2.0, 3.0) == 0.0
    assert vo.minmod3(0.0, 2.0, 3.0) == 0.0
    assert vo.minmod3(1.0, 0.0, 3.0) == 0.0
    assert vo.minmod3(1.0, 2.0, 0.0) == 0.0


def test_minmod_brute_force(vo):
    rng = np.random.default_rng(1)
    for _ in range(2000):
        x, y, z = rng.normal(size=3) * rng.choice([0.0, 1.0, 1e-3], size=3)
        if x > 0 and y > 0 and z > 0:
            ref = min(x, y, z)
        elif x < 0 and y < 0 and z < 0:
            ref = max(x, y, z)
        else:
            ref = 0.0
        assert vo.minmod3(x, y, z) == ref


def test_limited_slope_linear_data_and_tvd(vo):
    # on linear data the limited slope (Eq. 67) is the exact slope for every theta in [1,2]; at an extremum it is 0
    for theta in (1.0, 1.5, 2.0):
        s, d = 0.37, 0.1
        qm, q0, qp = 1.0 - s * d, 1.0, 1.0 + s * d
        got = vo.minmod3(theta * (q0 - qm) / d, (qp - qm) / (2 * d), theta * (qp - q0) / d)
        assert got == pytest.approx(s, rel=1e-12)
        assert vo.minmod3(theta * (1.0 - 0.5) / d, (0.7 - 0.5) / (2 * d), theta * (0.7 - 1.0) / d) == 0.0


def test_eos_cs2_is_dp_de(vo):
    prm = inputs.base_params()
    for e in (0.05, 0.3, 1.0, 5.0677, 20.0, 150.0):
        h = 1e-5 * e
        num = (vo.eos(prm, e + h)["p"] - vo.eos(prm, e - h)["p"]) / (2 * h)
        assert vo.eos(prm, e)["cs2"] == pytest.approx(num, rel=1e-8)
    # limits of p(e) = (e/3)(1 - 0.4 exp(-e/e0)): p/e -> 0.2 (e->0), 1/3 (e->inf); cs2 = 1/3 exactly at e = e0
    assert vo.eos(prm, 1e-9)["p"] / 1e-9 == pytest.approx(0.2, rel=1e-6)
    assert vo.eos(prm, 1e4)["p"] / 1e4 == pytest.approx(1 / 3, rel=1e-12)
    assert vo.eos(prm, prm["eos_e0"])["cs2"] == pytest.approx(1 / 3, abs=1e-15)
    # temperature: e = a T^4
    assert vo.eos(prm, 13.8 * 2.0**4)["T"] == pytest.approx(2.0, rel=1e-14)
    conf = inputs.base_params(eos=0)
    assert vo.eos(conf, 7.0)["p"] == pytest.approx(7.0 / 3, rel=1e-15)
    assert vo.eos(conf, 7.0)["cs2"] == pytest.approx(1 / 3, rel=1e-15)


def test_transport_coefficients_match_paper_equations(vo):
    # Eq. 13: eta/tau_pi = (e+p)/5 ; tau_pi = 5 eta/(e+p) = 5 (eta/s)/T.  Bulk in the BASELINE.json form
    # tau_Pi = 5 zeta/((e+p)(1/3-cs2)^2): zeta/tau_Pi = (e+p)(1/3-cs2)^2/5 when unclamped; Eq. 12: (8/5)(1/3-cs2)
    prm = inputs.base_params(tau_relax_floor_over_dtau=0.0)
    e = 0.3 / inputs.HBARC
    th = vo.eos(prm, e)
    tc = vo.transport(prm, e)
    assert tc["eta_over_tau_pi"] == pytest.approx((e + th["p"]) / 5, rel=1e-14)
    assert tc["inv_tau_pi"] == pytest.approx(th["T"] / (5 * 0.2), rel=1e-14)
    b = 1 / 3 - th["cs2"]
    assert tc["zeta_over_tau_Pi"] == pytest.approx((e + th["p"]) * b * b / 5, rel=1e-12)
    zs = 0.1 * math.exp(-(((th["T"] * inputs.HBARC) - 0.18) / 0.03) ** 2)
    assert tc["inv_tau_Pi"] == pytest.approx(th["T"] * b * b / (5 * zs), rel=1e-12)
    assert tc["lambda_Pipi_over_tau_Pi"] == pytest.approx(1.6 * b, rel=1e-14)
    # SURVEY 8(c) stiffness table (config form, derived there): 1/tau_Pi = 0.73 fm^-1 at 0.3 GeV/fm^3
    assert tc["inv_tau_Pi"] == pytest.approx(0.73, rel=0.02)
    # Eq. 10 form: zeta/tau_Pi = 15 (1/3-cs2)^2 (e+p)  <=>  c_tau_Pi = 1/15
    prm10 = inputs.base_params(tau_relax_floor_over_dtau=0.0, c_tau_Pi=1 / 15)
    assert vo.transport(prm10, e)["zeta_over_tau_Pi"] == pytest.approx(15 * b * b * (e + th["p"]), rel=1e-12)
    # clamp (reading R14): 1/tau_Pi <= 1/(5 dtau), and zeta/tau_Pi keeps the Navier-Stokes target zeta = (zeta/s) s
    prmc = inputs.base_params()
    ec = 0.1 / inputs.HBARC
    tcc = vo.transport(prmc, ec)
    thc = vo.eos(prmc, ec)
    assert tcc["inv_tau_Pi"] == pytest.approx(1 / (5 * 0.025), rel=1e-14)
    zsc = 0.1 * math.exp(-(((thc["T"] * inputs.HBARC) - 0.18) / 0.03) ** 2)
    assert tcc["zeta_over_tau_Pi"] == pytest.approx(zsc * (ec + thc["p"]) / thc["T"] * 8.0, rel=1e-12)
    # vanishing zeta/s: finite clamp, vanishing source; zeta_model 0 (zeta/s == 0 exactly) gives exactly zero
    cold = vo.transport(prmc, 1e-4 / inputs.HBARC)
    assert cold["inv_tau_Pi"] == pytest.approx(8.0) and 0.0 <= cold["zeta_over_tau_Pi"] < 1e-14
    none = vo.transport(inputs.base_params(zeta_model=0), 1.0)
    assert none["inv_tau_Pi"] == pytest.approx(8.0) and none["zeta_over_tau_Pi"] == 0.0


def test_zeta_over_s_of_eq17(vo):
    # PAPER.md Eq. 17 (:174-186), zeta_model 3: what the paper prints about the curve pins the branches and their constants -
    # "(zeta/s)_norm = 3 has a peak value of 1" (:190), the floors 0.001 (hot) and 0.03 (cold), T_c = 200 MeV - plus the
    # near-continuity of the three pieces at 0.995 T_c and 1.05 T_c that an interpolating parametrisation must have
    HB = inputs.HBARC
    Tc = 0.2 / HB

    def zs(T_gev, norm=1.0):
        prm = inputs.base_params(zeta_model=3, zeta_amp=norm, zeta_T0=Tc, tau_relax_floor_over_dtau=0.0)
        T = T_gev / HB
        e = prm["eos_a"] * T**4
        th, tc = vo.eos(prm, e), vo.transport(prm, e)
        s = (e + th["p"]) / th["T"]
        return tc["zeta_over_tau_Pi"] / tc["inv_tau_Pi"] / s      # zeta/s recovered from zeta/tau_Pi and 1/tau_Pi

    grid = np.linspace(0.05, 0.32, 1081)      # (hotter, exp(-e/e0) of EOS 1 underflows, 1/tau_Pi = 0 and the ratio below is 0/0)
    vals = np.array([zs(t) for t in grid])
    ok = np.isfinite(vals)      # (1/tau_Pi vanishes where c_s^2 = 1/3, e = e0 of EOS 1: the ratio is 0/0 at that one temperature)
    assert ok.sum() >= len(grid) - 2
    grid, vals = grid[ok], vals[ok]
    assert vals.max() == pytest.approx(0.33, abs=2e-3) and abs(grid[vals.argmax()] - 0.2) < 2e-3      # peak -13.45 + 27.55 - 13.77 at T_c
    assert zs(0.2, norm=3.0) == pytest.approx(0.99, abs=1e-12)                                        # "peak value of 1" for norm 3
    assert zs(0.05) == pytest.approx(0.03, rel=1e-6)                                                  # cold floor (hot floor 0.001: formula check below)
    for Tj in (0.995 * 0.2, 1.05 * 0.2):                                                              # joins continuous to ~1.5 %
        assert zs(Tj * (1 - 1e-9)) == pytest.approx(zs(Tj * (1 + 1e-9)), rel=1.5e-2)
    assert zs(0.19) == pytest.approx(0.9 * math.exp(-20.0) + 0.22 * math.exp(-0.05 / 0.022) + 0.03, rel=1e-12)
    assert zs(0.3) == pytest.approx(0.9 * math.exp(-20.0) + 0.25 * math.exp(-0.5 / 0.13) + 0.001, rel=1e-12)
    assert np.all(vals > 0) and np.all(np.diff(vals[grid > 0.2105]) < 0) and np.all(np.diff(vals[grid < 0.1985]) > 0)


def test_newton_vs_conformal_closed_form(vo):
    # e = sqrt(4E^2 - 3M^2) - E for p = e/3, Pi = 0
    prm = inputs.base_params(eos=0)
    rng = np.random.default_rng(5)
    worst = 0.0
    for _ in range(3000):
        E = 10 ** rng.uniform(-3, 3)
        M2 = (rng.uniform(0, 0.999) * E) ** 2
        guess = E * 10 ** rng.uniform(-2, 1)
        e, it, fail = vo.invert(prm, E, M2, 0.0, guess)
        ref = math.sqrt(4 * E * E - 3 * M2) - E
        assert fail == 0 and it <= 50
        worst = max(worst, abs(e - ref) / ref)
    assert worst < 5e-12


def test_newton_round_trip_nonconformal_with_bulk(vo):
    # forward map Eqs. 32-33 written out here; the oracle must recover e from (E, M^2, Pi)
    prm = inputs.base_params()
    rng = np.random.default_rng(6)
    for _ in range(2000):
        e = 10 ** rng.uniform(-1.5, 2.3)
        p0 = (e / 3) * (1 - 0.4 * math.exp(-e / prm["eos_e0"]))
        Pi = rng.uniform(-0.3, 0.3) * p0
        tau = rng.uniform(0.3, 3.0)
        ux, uy, un = rng.normal(size=3) * np.array([0.8, 0.8, 0.8 / tau])
        ut = math.sqrt(1 + ux * ux + uy * uy + tau * tau * un * un)
        P = p0 + Pi
        E = (e + P) * ut * ut - P
        M2 = ((e + P) * ut) ** 2 * (ux * ux + uy * uy + tau * tau * un * un)
        got, it, fail = vo.invert(prm, E, M2, Pi, E)
        assert fail == 0
        assert got == pytest.approx(e, rel=2e-11)


def test_newton_failure_is_reported_not_hidden(vo):
    prm = inputs.base_params(eos=0)
    e, it, fail = vo.invert(prm, 1.0, 4.0, 0.0, 1.0)     # |M| > E: no positive root (f(0) >= 0), reading R6
    assert fail == 1 and e == 1.0
    e, it, fail = vo.invert(prm, -1.0, 0.0, 0.0, 1.0)
    assert fail == 1


def test_set_initial_builds_q0_from_eqs_32_33_and_ghosts(vo):
    prm = inputs.base_params(nx=3, ny=4, nz=2, tau0=0.7)
    st = inputs.smooth_random_state(prm, seed=3)
    o = vo.Oracle(prm)
    o.set_initial(st["e"], st["u"], st["pi"], st["Pi"])
    f = o.get_fields()
    e, u, pi, Pi = st["e"], st["u"], st["pi"], st["Pi"]
    p0 = (e / 3) * (1 - 0.4 * np.exp(-e / prm["eos_e0"]))
    P = p0 + Pi
    np.testing.assert_allclose(f["q"][0], (e + P) * u[0] ** 2 - P + pi[0], rtol=1e-14)
    for i in (1, 2, 3):
        np.testing.assert_allclose(f["q"][i], (e + P) * u[0] * u[i] + pi[i], rtol=1e-14, atol=1e-15)
    np.testing.assert_array_equal(f["q"][4:14], pi)
    np.testing.assert_array_equal(f["q"][14], Pi)
    np.testing.assert_allclose(f["p"], p0, rtol=1e-15)
    # ghost faces replicate the outermost physical cell in both layers (Eqs. 75-76)
    for name, comp in (("q", 0), ("q", 9), ("q", 14), ("e", 0), ("p", 0), ("u", 1)):
        a = o.raw(name, comp)
        inner = a[2:-2, 2:-2, 2:-2]
        np.testing.assert_array_equal(a[2:-2, 2:-2, 0], inner[:, :, 0]); np.testing.assert_array_equal(a[2:-2, 2:-2, 1], inner[:, :, 0])
        np.testing.assert_array_equal(a[2:-2, 2:-2, -1], inner[:, :, -1]); np.testing.assert_array_equal(a[2:-2, 2:-2, -2], inner[:, :, -1])
        np.testing.assert_array_equal(a[2:-2, 0, 2:-2], inner[:, 0, :]); np.testing.assert_array_equal(a[2:-2, -1, 2:-2], inner[:, -1, :])
        np.testing.assert_array_equal(a[0, 2:-2, 2:-2], inner[0]); np.testing.assert_array_equal(a[1, 2:-2, 2:-2], inner[0])
        np.testing.assert_array_equal(a[-1, 2:-2, 2:-2], inner[-1]); np.testing.assert_array_equal(a[-2, 2:-2, 2:-2], inner[-1])
    # u^{-1} = u^0 (footnote 4)
    np.testing.assert_array_equal(o.get_fields(with_uprev=True)["up"], st["u"])


def test_heun_on_pure_relaxation(vo):
    # Homogeneous fluid at rest at very large tau (geometric terms ~1/tau negligible): d pi^{xy}/d tau = -pi^{xy}/tau_pi.
    # One Heun step (Eqs. 69-71, beta_1 = 1/2) multiplies by 1 - z + z^2/2, z = dtau/tau_pi.
    prm = inputs.base_params(nx=2, ny=2, nz=2, tau0=1e9, dtau=0.05, eos=0, physics=1, zeta_model=0, rho_max=1e30,
                             tau_relax_floor_over_dtau=0.0)
    shp = (1, 2, 2, 2)
    e0 = 20.0
    pi = np.zeros((10,) + shp)
    pi[5] = 1e-3   # pi^{xy}
    o = vo.Oracle(prm)
    o.set_initial(np.full(shp, e0), inputs.rest_velocity(shp), pi)
    o.step(1)
    T = (e0 / 13.8) ** 0.25
    z = 0.05 * T / (5 * 0.2)
    got = o.get_fields()["q"][9] / 1e-3
    np.testing.assert_allclose(got, 1 - z + z * z / 2, rtol=1e-7)


def test_regularisation_factor_values(vo):
    # Eqs. 73-74 at rest, pi = diag-free single component, Pi = 0: rho = sqrt(pi.pi)/sqrt(e^2+3p^2) (first entry of the max;
    # the trace and pi.u entries vanish for pi^{xy} only), factor tanh(rho)/rho.  Reading R9.
    prm = inputs.base_params(nx=1, ny=1, nz=1, tau0=1.3, eos=0, physics=1, zeta_model=0)
    o = vo.Oracle(prm)
    shp = (1, 1, 1, 1)
    e0 = 9.0
    for amp in (1e-12, 0.5, 3.0, 40.0):
        pi = np.zeros((10,) + shp)
        pi[5] = amp
        o.set_initial(np.full(shp, e0), inputs.rest_velocity(shp), pi)
        o.post(1.3)
        rho = math.sqrt(2 * amp * amp) / math.sqrt(e0 * e0 + 3 * (e0 / 3) ** 2)
        fac = 1.0 if rho < 1e-8 else math.tanh(rho) / rho
        assert o.raw("q", 9)[2, 2, 2] == pytest.approx(amp * fac, rel=1e-14)
    # a pure trace violation (pi^{xx} only, |g_{mu nu} pi^{mu nu}| = |pi^{xx}|) is caught by the xi0 entry: rho >= 1/xi0 = 10
    pi = np.zeros((10,) + shp)
    pi[4] = 1e-6
    o.set_initial(np.full(shp, e0), inputs.rest_velocity(shp), pi)
    o.post(1.3)
    assert o.raw("q", 8)[2, 2, 2] == pytest.approx(1e-6 * math.tanh(10.0) / 10.0, rel=1e-12)


def test_diagnostics_against_their_definitions(vo):
    # the maxima of the oracle's diagnostics() re-derived with numpy from the exported fields - T from e = a T^4,
    # u.u with g = diag(1,-1,-1,-tau^2) (:243), the constraints of Eqs. 47-51, the inverse Reynolds numbers of Eq. 89
    prm = inputs.base_params(nx=12, ny=8, nz=6, tau0=0.6, dtau=0.02)
    st = inputs.smooth_random_state(prm, seed=3)
    o = vo.Oracle(prm)
    o.set_initial(st["e"], st["u"], st["pi"], st["Pi"])
    o.step(3)
    d, f, tau = o.diagnostics(), o.get_fields(), o.status()["tau"]
    g = np.array([1.0, -1.0, -1.0, -tau * tau])
    u, e, p = f["u"], f["e"], f["p"]
    slot = [[4, 5, 6, 7], [5, 8, 9, 10], [6, 9, 11, 12], [7, 10, 12, 13]]
    pi = np.array([[f["q"][slot[m][n]] for n in range(4)] for m in range(4)])
    assert d["max_T"] == pytest.approx(np.max((e / prm["eos_a"]) ** 0.25), rel=1e-14)
    assert d["max_norm_violation"] == pytest.approx(np.max(np.abs(np.einsum("m,m...->...", g, u * u) - 1)), abs=1e-15)
    assert d["max_trace_violation"] == pytest.approx(np.max(np.abs(np.einsum("m,mm...->...", g, pi)) / (e + p)), rel=1e-12)
    c = np.abs(np.einsum("lm...,m,m...->l...", pi, g, u))
    c[3] *= tau
    assert d["max_transversality_violation"] == pytest.approx(np.max(c.max(axis=0) / (e + p)), rel=1e-12)
    pipi = np.einsum("mn...,m,n,mn...->...", pi, g, g, pi)
    assert d["max_inv_reynolds_shear"] == pytest.approx(np.max(np.sqrt(np.abs(pipi)) / p), rel=1e-12)
    assert d["max_inv_reynolds_bulk"] == pytest.approx(np.max(np.abs(f["q"][14]) / p), rel=1e-14)
    # Knudsen numbers (:830): theta of A.11 from the exported u^n, u^{n-1} with numpy differences (ghost = copy of the boundary cell)
    fu = o.get_fields(with_uprev=True)
    pad = lambda a, ax: np.concatenate([np.take(a, [0], axis=ax), a, np.take(a, [-1], axis=ax)], axis=ax)
    cd = lambda a, ax, h: (np.take(pad(a, ax), range(2, a.shape[ax] + 2), axis=ax) - np.take(pad(a, ax), range(0, a.shape[ax]), axis=ax)) / (2 * h)
    theta = u[0] / tau + (u[0] - fu["up"][0]) / prm["dtau"] + cd(u[1], 3, prm["dx"]) + cd(u[2], 2, prm["dy"]) + cd(u[3], 1, prm["dz"])
    it_pi = np.vectorize(lambda ee: vo.transport(prm, ee)["inv_tau_pi"])(e)
    it_Pi = np.vectorize(lambda ee: vo.transport(prm, ee)["inv_tau_Pi"])(e)
    assert d["max_knudsen_shear"] == pytest.approx(np.max(np.abs(theta) / it_pi), rel=1e-12)
    assert d["max_knudsen_bulk"] == pytest.approx(np.max(np.abs(theta) / it_Pi), rel=1e-12)
    # the per-cell maps (Figs. 15-17 are slices of such maps) against the same numpy expressions, cell by cell
    m = o.diagnostic_maps()[:, 0]
    ref = [(e / prm["eos_a"]) ** 0.25, np.abs(np.einsum("m,m...->...", g, u * u) - 1), np.abs(np.einsum("m,mm...->...", g, pi)) / (e + p),
           c.max(axis=0) / (e + p), np.sqrt(np.abs(pipi)) / p, np.abs(f["q"][14]) / p, np.abs(theta) / it_pi, np.abs(theta) / it_Pi]
    for k, r in enumerate(ref):
        np.testing.assert_allclose(m[k], r[0], rtol=1e-11, atol=1e-13 * max(np.max(r), 1e-3), err_msg=str(k))
        assert np.max(m[k]) == list(d.values())[k]
    assert d["max_norm_violation"] < 1e-14 and 0 < d["max_trace_violation"] < 0.05      # u.u = 1 after inversion (:489); constraints drift slowly (:333)


def test_second_order_reynolds_numbers_in_bjorken_flow(vo):
    # Eq. 90 (:831) with J, J^{mu nu} of Eq. 5 at n^mu = 0.  Closed form for a uniform fluid at rest in Milne coordinates (Bjorken flow):
    # theta = 1/tau, sigma^{mu nu} = (2/(3 tau)) d^{mu nu}, pi^{mu nu} = pi d^{mu nu} with d = diag(0, 1/2, 1/2, -1/tau^2); no vorticity;
    # pi^{lambda<mu} sigma^{nu>}_lambda = (pi/(3 tau)) d^{mu nu}; pi^{mu nu} sigma_{mu nu} = pi/tau.  Hence
    #   (R_pi^(2))^-1 = |-(delta_pipi + tau_pipi/3) pi + (2/3) lambda_piPi Pi| / ((4/3) eta/tau_pi)     (coefficients in units of tau_pi)
    #   (R_Pi^(2))^-1 = |-delta_PiPi Pi + (lambda_Pipi/tau_Pi) pi| / (zeta/tau_Pi)
    tau0, e0, pi0, Pi0 = 0.7, 9.0, 0.31, -0.12
    prm = inputs.base_params(nx=6, ny=5, nz=4, tau0=tau0, dtau=0.01, eos=1, zeta_model=1)
    shape = (1, 4, 5, 6)
    e = np.full(shape, e0)
    pi = np.zeros((10,) + shape)
    pi[4], pi[7], pi[9] = 0.5 * pi0, 0.5 * pi0, -pi0 / tau0 ** 2
    o = vo.Oracle(prm)
    o.set_initial(e, inputs.rest_velocity(shape), pi, np.full(shape, Pi0))
    d, m, tc = o.diagnostics(), o.diagnostic_maps(), vo.transport(prm, e0)
    r2s = abs(-(prm["delta_pipi"] + prm["tau_pipi"] / 3) * pi0 + (2.0 / 3.0) * prm["lambda_piPi"] * Pi0) / ((4.0 / 3.0) * tc["eta_over_tau_pi"])
    r2b = abs(-prm["delta_PiPi"] * Pi0 + tc["lambda_Pipi_over_tau_Pi"] * pi0) / tc["zeta_over_tau_Pi"]
    assert tc["zeta_over_tau_Pi"] > 0 and r2s > 0.01 and r2b > 0.01
    assert d["max_inv_reynolds2_shear"] == pytest.approx(r2s, rel=1e-12)
    assert d["max_inv_reynolds2_bulk"] == pytest.approx(r2b, rel=1e-12)
    np.testing.assert_allclose(m[8], r2s, rtol=1e-12)
    np.testing.assert_allclose(m[9], r2b, rtol=1e-12)
    assert d["max_knudsen_shear"] == pytest.approx(1.0 / tau0 / tc["inv_tau_pi"], rel=1e-12)
    # a state without gradients and without tau-expansion (Cartesian geometry is ideal-only, so: sectors off -> zeros)
    o2 = vo.Oracle(dict(prm, physics=0))
    o2.set_initial(e, inputs.rest_velocity(shape))
    d2 = o2.diagnostics()
    assert d2["max_inv_reynolds2_shear"] == 0.0 and d2["max_inv_reynolds2_bulk"] == 0.0


def test_regulation_map_records_the_applied_factor(vo):
    # Fig. 17 (:820): the map of tanh(rho)/rho.  The recorded factor must be the one by which the regularisation scaled pi^{mu nu} and
    # Pi at that cell (Eq. 73): ratio of the exported fields after / before program-flow step 3, cell by cell
    prm = inputs.base_params(nx=9, ny=7, nz=5, tau0=0.9, dtau=0.02)
    st = inputs.smooth_random_state(prm, seed=11)
    o = vo.Oracle(prm)
    o.set_initial(st["e"], st["u"], 6.0 * st["pi"], 6.0 * st["Pi"])
    assert np.all(o.regulation_map() == 1.0)
    before = o.get_fields()["q"].copy()
    o.post(0.9)
    after, m = o.get_fields()["q"], o.regulation_map()
    assert m.shape == (1, 5, 7, 9) and 0.0 < m.min() < 0.9 and m.max() <= 1.0 and np.ptp(m) > 0.05
    for n in range(4, 15):
        np.testing.assert_allclose(after[n], m * before[n], rtol=1e-14, atol=0)
    np.testing.assert_allclose(after[:4], before[:4], rtol=0, atol=0)
    # after a full step the map is that of the step's last regularisation: never below the run's minimum
    o.step(2)
    assert o.regulation_map().min() >= o.status()["min_reg_factor"]
