"""Closed-form / ODE comparators used to pin the oracle (never used by the product path).

  * ideal relativistic Riemann problem for p = e/3 with both sides at rest (PAPER.md :577-579, :634; Ref. [34])
  * 0+1d Bjorken ODEs, Eqs. 77-78 and 79-81
  * ideal Gubser flow, Eqs. 82-85
  * boosted-static exact solution
"""
import math

import numpy as np
from scipy.integrate import solve_ivp
from scipy.optimize import brentq

CS = 1.0 / math.sqrt(3.0)


def riemann_plateau(eL, eR):
    """Plateau state and shock speed.  Rarefaction invariant: artanh v = (sqrt3/4) ln(eL/e);
    Taub adiabat for p=e/3, upstream at rest: v^2 = 3 (ep-eR)^2 / ((3eR+ep)(3ep+eR)); Vs^2 = (3ep+eR)/(3(3eR+ep))."""

    def f(ep):
        v_r = math.tanh(math.sqrt(3.0) / 4.0 * math.log(eL / ep))
        v_s = math.sqrt(3.0 * (ep - eR) ** 2 / ((3 * eR + ep) * (3 * ep + eR)))
        return v_r - v_s

    ep = brentq(f, eR * (1 + 1e-12), eL * (1 - 1e-12), xtol=1e-14 * eR, rtol=1e-15)
    vp = math.tanh(math.sqrt(3.0) / 4.0 * math.log(eL / ep))
    Vs = math.sqrt((3 * ep + eR) / (3 * (3 * eR + ep)))
    return ep, vp, Vs


def riemann_solution(x, t, eL, eR):
    """e(x,t), v(x,t) of the shock tube (membrane at x=0)."""
    ep, vp, Vs = riemann_plateau(eL, eR)
    xi = np.asarray(x, dtype=float) / t
    e = np.empty_like(xi)
    v = np.empty_like(xi)
    head = -CS
    tail = (vp - CS) / (1 - vp * CS)
    left = xi <= head
    fan = (xi > head) & (xi < tail)
    plat = (xi >= tail) & (xi < Vs)
    right = xi >= Vs
    e[left] = eL; v[left] = 0.0
    vf = (xi[fan] + CS) / (1 + CS * xi[fan])
    v[fan] = vf
    e[fan] = eL * ((1 - vf) / (1 + vf)) ** (2.0 / math.sqrt(3.0))
    e[plat] = ep; v[plat] = vp
    e[right] = eR; v[right] = 0.0
    return e, v


def bjorken_ode(e0, pi0, Pi0, tau0, taus, eos, transport, coeffs):
    """PAPER.md Eqs. 79-81 (77-78 when Pi == 0 and zeta == 0), pi = -tau^2 pi^{eta eta}.
    eos(e) -> (p, cs2, T); transport(e, p, cs2, T) -> (1/tau_pi, eta/tau_pi, 1/tau_Pi, zeta/tau_Pi)
    coeffs: dict delta_pipi, tau_pipi, lambda_piPi, delta_PiPi, lambda_Pipi_coef (in units of the relaxation times)."""

    def rhs(tau, y):
        e, pi, Pi = y
        p, cs2, T = eos(e)
        itp, eotp, itP, zotP = transport(e, p, cs2, T)
        de = -(e + p + Pi - pi) / tau
        dpi = -pi * itp + (4.0 / 3.0) * eotp / tau - (coeffs["tau_pipi"] / 3.0 + coeffs["delta_pipi"]) * pi / tau \
            + (2.0 / 3.0) * coeffs["lambda_piPi"] * Pi / tau
        dPi = -Pi * itP - zotP / tau - coeffs["delta_PiPi"] * Pi / tau + coeffs["lambda_Pipi_coef"] * (1.0 / 3.0 - cs2) * pi / tau
        return [de, dpi, dPi]

    sol = solve_ivp(rhs, [tau0, max(taus)], [e0, pi0, Pi0], method="DOP853", rtol=1e-12, atol=1e-14, t_eval=taus)
    return sol.y


def gubser_ideal_T(tau, r, T0hat=1.2, q=1.0):
    """PAPER.md Eq. 82."""
    return T0hat * (2 * q * tau) ** (2.0 / 3.0) / (tau * (1 + 2 * q * q * (tau * tau + r * r) + q**4 * (tau * tau - r * r) ** 2) ** (1.0 / 3.0))


def gubser_kappa(tau, r, q=1.0):
    """PAPER.md Eq. 85."""
    return np.arctanh(2 * q * q * tau * r / (1 + q * q * tau * tau + q * q * r * r))
