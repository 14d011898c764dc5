"""Pin of the oracle's dissipative source terms (Eqs. 39-46, B.10-B.12, App. A) against an independent,
fully generic covariant evaluation of the governing relaxation equations, Eq. 8 (:147-149):

  * Christoffel symbols from the metric by the general formula, dense 4x4x4 - not the Milne shortcuts;
  * theta, sigma^{mu nu}, omega^{mu nu}, Du_lambda from their covariant definitions (A.1-A.4 first forms, :122) with the
    rank-4 projector Delta^{mu nu}_{alpha beta} - not the expanded forms the oracle uses;
  * angular brackets of Eq. 8 applied literally with that projector;
  * flow field analytic and exactly normalised, derivatives analytic (sympy).

The oracle gets the same flow sampled on a tiny grid (central differences, spacing 1e-4; backward time difference 1e-7), so
the two agree to truncation error ~1e-7.  The vorticity term enters with the sign of Eq. 8 (reading R4).
The same evaluation pins the second-order inverse Reynolds numbers of Eq. 90 (J^{mu nu}, J of Eq. 5 written out with the projector)."""
import numpy as np
import pytest
import sympy as sp

from paper_1608_06577_b200 import inputs


def generic_rhs(prm, point, coeffs, pi_seed, Pi):
    tau, x, y, eta = sp.symbols("tau x y eta", positive=True)
    X = [tau, x, y, eta]
    ux = 0.30 * sp.sin(0.7 * x + 0.4 * y - 0.5 * eta + 0.9 * tau) + 0.10
    uy = -0.25 * sp.cos(0.3 * x - 0.8 * y + 0.6 * eta - 0.4 * tau) + 0.05
    un = (0.20 * sp.sin(0.5 * x + 0.2 * y + 0.9 * eta + 0.3 * tau) - 0.05) / tau
    ut = sp.sqrt(1 + ux**2 + uy**2 + tau**2 * un**2)
    U = [ut, ux, uy, un]
    g = sp.diag(1, -1, -1, -tau**2)
    gi = g.inv()
    Gam = [[[sum(gi[l, n] * (sp.diff(g[a, n], X[b]) + sp.diff(g[n, b], X[a]) - sp.diff(g[a, b], X[n])) for n in range(4)) / 2
             for b in range(4)] for a in range(4)] for l in range(4)]
    sub = dict(zip(X, point))
    f = lambda ex: float(sp.N(sp.sympify(ex).subs(sub), 30))
    u = np.array([f(c) for c in U])
    du = np.array([[f(sp.diff(U[n], X[a])) for n in range(4)] for a in range(4)])        # du[a][n] = partial_a u^n
    divv = sum(f(sp.diff(U[i] / U[0], X[i])) for i in (1, 2, 3))
    G = np.array([[[f(Gam[l][a][b]) for b in range(4)] for a in range(4)] for l in range(4)])   # G[l,a,b]
    gl = np.array([[f(g[a, b]) for b in range(4)] for a in range(4)])
    gu = np.linalg.inv(gl)
    ufun = sp.lambdify(X, U, "mpmath")

    cov = du + np.einsum("nal,l->an", G, u)                    # cov[a,n] = d_a u^n          (Eq. 25)
    theta = np.trace(cov)                                      # A.2
    Dl = gu - np.outer(u, u)                                   # Delta^{mu nu}
    Dm = Dl @ gl                                               # Delta^mu_nu
    Dll = gl @ Dl @ gl                                         # Delta_{mu nu}
    P4 = 0.5 * (np.einsum("ma,nb->mnab", Dm, Dm) + np.einsum("na,mb->mnab", Dm, Dm)) - np.einsum("mn,ab->mnab", Dl, Dll) / 3.0
    dup = gu @ cov                                             # d^a u^n
    sig = np.einsum("mnab,ab->mn", P4, dup)                    # sigma^{mu nu} = Delta^{mu nu}_{ab} d^a u^b
    nab = Dl @ cov                                             # nabla^mu u^nu = Delta^{mu a} d_a u^nu
    om = 0.5 * (nab - nab.T)                                   # omega^{mu nu}  (:122)
    Du_up = u @ cov
    Du_lo = gl @ Du_up
    # a shear tensor satisfying the constraints: project a seeded symmetric matrix
    rng = np.random.default_rng(pi_seed)
    A = rng.normal(size=(4, 4)); A = 0.5 * (A + A.T)
    pi = np.einsum("mnab,ab->mn", P4, A) * 0.7
    assert abs(np.einsum("mn,mn->", gl, pi)) < 1e-12 and np.max(np.abs(pi @ gl @ u)) < 1e-12
    itp, eotp, itP, zotP, lPp = coeffs
    br = lambda T: np.einsum("mnab,ab->mn", P4, T)
    pi_lo1 = pi @ gl                                           # pi^mu_lambda
    t_om = br(np.einsum("ml,nl->mn", pi_lo1, om))              # pi^{<mu}_lambda omega^{nu>lambda}
    sig_lo1 = sig @ gl                                         # sigma^nu_lambda
    t_ps = br(np.einsum("lm,nl->mn", pi, sig_lo1))             # pi^{lambda<mu} sigma^{nu>}_lambda
    # Eq. 8 divided by tau_pi, solved for D pi^{<mu nu>}
    Dpi_br = -pi * itp + 2 * eotp * sig + 2 * t_om - prm["delta_pipi"] * pi * theta - prm["tau_pipi"] * t_ps + prm["lambda_piPi"] * Pi * sig
    Dpi = Dpi_br - (np.einsum("lm,n,l->mn", pi, u, Du_lo) + np.einsum("ln,m,l->mn", pi, u, Du_lo))
    Gpi = np.einsum("a,mab,bn->mn", u, G, pi) + np.einsum("a,nab,bm->mn", u, G, pi)     # :300
    J_pi = (Dpi - Gpi) / u[0] + pi * divv                      # B.9, B.11
    pisig = np.einsum("mn,ma,nb,ab->", pi, gl, gl, sig)
    DPi = -zotP * theta - Pi * itP - prm["delta_PiPi"] * Pi * theta + lPp * pisig      # Eq. 8 first line / tau_Pi
    J_Pi = DPi / u[0] + Pi * divv
    # Eq. 90 (:831) with J^{mu nu}, J of Eq. 5 (:116-120) at n^mu = 0, both divided by their relaxation time
    J2 = 2 * t_om - prm["delta_pipi"] * pi * theta - prm["tau_pipi"] * t_ps + prm["lambda_piPi"] * Pi * sig
    J0 = -prm["delta_PiPi"] * Pi * theta + lPp * pisig
    con = lambda T: np.einsum("mn,ma,nb,ab->", T, gl, gl, T)
    r2_shear = np.sqrt(abs(con(J2))) / (2 * eotp * np.sqrt(abs(con(sig))))
    r2_bulk = abs(J0) / (zotP * abs(theta))
    return dict(u=u, ufun=ufun, pi=pi, J_pi=J_pi, J_Pi=J_Pi, theta=theta, sig=sig, om=om, r2_shear=r2_shear, r2_bulk=r2_bulk, t_om=t_om)


@pytest.mark.parametrize("pi_seed", [1, 2])
def test_dissipative_sources_against_generic_covariant_evaluation(vo, pi_seed):
    h, dt = 1e-4, 1e-7
    point = (1.3, 0.4, -0.2, 0.6)
    prm = inputs.base_params(nx=1, ny=1, nz=1, dx=h, dy=h, dz=h, tau0=point[0], dtau=dt, rho_max=1e30)
    e0 = 2.0 / inputs.HBARC
    tc = vo.transport(prm, e0)
    coeffs = (tc["inv_tau_pi"], tc["eta_over_tau_pi"], tc["inv_tau_Pi"], tc["zeta_over_tau_Pi"], tc["lambda_Pipi_over_tau_Pi"])
    Pi = -0.3
    ref = generic_rhs(prm, point, coeffs, pi_seed, Pi)
    o = vo.Oracle(prm)
    shp = (1, 1, 1, 1)
    slot = [[4, 5, 6, 7], [5, 8, 9, 10], [6, 9, 11, 12], [7, 10, 12, 13]]
    pi10 = np.zeros((10,) + shp)
    for m in range(4):
        for n in range(m, 4):
            pi10[slot[m][n] - 4] = ref["pi"][m, n]
    o.set_initial(np.full(shp, e0), ref["u"].reshape((4,) + shp), pi10, np.full(shp, Pi))
    # overwrite the padded velocity arrays with the analytic flow (ghost cells hold the true neighbours here)
    for kk in range(5):
        for jj in range(5):
            for ii in range(5):
                xx = (point[0], point[1] + (ii - 2) * h, point[2] + (jj - 2) * h, point[3] + (kk - 2) * h)
                uu = [float(c) for c in ref["ufun"](*xx)]
                for m in range(4):
                    o.raw("u", m)[kk, jj, ii] = uu[m]
    um = [float(c) for c in ref["ufun"](point[0] - dt, *point[1:])]
    for m in range(4):
        o.raw("up", m)[2, 2, 2] = um[m]
    J = o.sources_at(2, 2, 2, point[0])
    scale = np.max(np.abs(ref["J_pi"]))
    for m in range(4):
        for n in range(m, 4):
            assert J[slot[m][n]] == pytest.approx(ref["J_pi"][m, n], abs=3e-6 * scale), (m, n)
    assert J[14] == pytest.approx(ref["J_Pi"], rel=3e-6)
    # second-order inverse Reynolds numbers of Eq. 90 (reading R21) at the same cell, vorticity term included
    m10 = o.diagnostic_maps()[:, 0, 0, 0, 0]
    assert m10[8] == pytest.approx(ref["r2_shear"], rel=3e-6) and m10[9] == pytest.approx(ref["r2_bulk"], rel=3e-6)
    assert m10[6] == pytest.approx(abs(ref["theta"]) / tc["inv_tau_pi"], rel=3e-6)
    assert np.max(np.abs(ref["t_om"])) > 0.02 * np.max(np.abs(ref["pi"])) and ref["r2_shear"] > 0.05 and ref["r2_bulk"] > 0.05
    # the terms being pinned are all present at a comparable size (a vanishing term would pin nothing)
    assert np.max(np.abs(ref["om"])) > 0.05 and np.max(np.abs(ref["sig"])) > 0.05 and abs(ref["theta"]) > 0.05
