"""Pins of the oracle's VISCOUS Cartesian mode (geometry = 1 with shear on) and of the multi-dimensional Cartesian
test problems of PAPER.md 5.2-5.3 (:696-718).

(1) Damped sound wave.  Linearising the equations the solver integrates (Eqs. 30-31 with Eq. 40, Cartesian, conformal, shear only)
    around a fluid at rest gives, for a plane wave exp(i(kx - wt)) along x,
        -i w de + (e+p) i k du = 0,   -i w (e+p) du + cs2 i k de + i k dpi = 0,   (1 - i w tau_pi) dpi = -(4/3) eta i k du
    (pi^{xx}_NS = 2 eta sigma^{xx} = -(4/3) eta d_x u^x in the mostly-minus metric; every second-order term of Eq. 42 is quadratic in the
    perturbation), i.e. the cubic  -i tau_pi w^3 + w^2 + i (cs2 tau_pi + nu) k^2 w - cs2 k^2 = 0,  nu = (4/3) eta/(e+p).
    The right-moving root and its eigenvector are started on a long 1-d grid; after a time T the oracle's wave in the middle of the grid
    must equal the eigenmode times exp(-i w T): damping rate and phase velocity from numpy.roots, nothing from the oracle.
    A wrong sign or factor in 2 eta sigma^{mu nu}, in 1/tau_pi, in the pi^{xx} gradient of the momentum equation, or a Christoffel term
    left on, changes the complex amplitude by far more than the tolerance.  Run along x and along the third axis (tau^2 -> 1).
(2) 2+1d diagonal shock tube (:696-704): the discontinuity runs along x + y = 0; the solution must be symmetric under x <-> y and, in
    rotated coordinates, reproduce the plateau of the analytic Riemann solution (tests/analytic.py).
(3) Cylindrical blast (:706-718): "cylindrical symmetry preserved on a Cartesian grid" - the four-fold and diagonal mirror symmetries
    must hold to rounding, and the radial profile sampled along the axis and along the diagonal must agree to truncation error.
"""
import math

import numpy as np
import pytest

import analytic
from paper_1608_06577_b200 import inputs


def sound_mode(k, T0, a, eta_s, c_tau_pi):
    e0 = a * T0 ** 4
    w_enth = 4.0 * e0 / 3.0                      # e + p
    cs2 = 1.0 / 3.0
    tau_pi = c_tau_pi * eta_s / T0               # tau_pi = c eta/(e+p), eta = (eta/s) s, s = (e+p)/T   (Eq. 13)
    nu = (4.0 / 3.0) * eta_s / T0                # (4/3) eta/(e+p)
    roots = np.roots([-1j * tau_pi, 1.0, 1j * (cs2 * tau_pi + nu) * k * k, -cs2 * k * k])
    w = [r for r in roots if r.real > 1e-9][0]
    assert w.imag < 0
    de = w_enth * k / w                          # per unit du
    dpi = -nu * w_enth * 1j * k / (1.0 - 1j * w * tau_pi)
    return e0, w, de, dpi


@pytest.mark.parametrize("axis", [0, 2])
def test_damped_sound_wave_viscous_cartesian(vo, axis):
    n, d = 768, 0.025
    lam = 128 * d                                # 128 cells per wavelength
    k = 2.0 * math.pi / lam
    T0, eta_s = 1.0, 0.5
    dims = [1, 1, 1]
    dims[axis] = n
    dt = 0.2 * d
    prm = inputs.base_params(nx=dims[0], ny=dims[1], nz=dims[2], dx=d, dy=d, dz=d, tau0=1.0, dtau=dt, geometry=1, physics=1, eos=0, eta_over_s=eta_s,
                             zeta_model=0, minmod_theta=2.0, tau_relax_floor_over_dtau=0.0)
    e0, w, de, dpi = sound_mode(k, T0, prm["eos_a"], eta_s, prm["c_tau_pi"])
    A = 1e-5
    x = inputs.centred_axis(n, d)
    ph = np.exp(1j * k * x)
    shp = (1, dims[2], dims[1], dims[0])
    line = lambda z: np.real(z).reshape(shp)
    u = np.zeros((4,) + shp)
    u[1 + axis] = line(A * ph)
    u[0] = np.sqrt(1.0 + u[1 + axis] ** 2)
    e = e0 + line(A * de * ph)
    pl = line(A * dpi * ph)                      # pi^{rr} along the wave
    v = u[1 + axis] / u[0]
    pi = np.zeros((10,) + shp)
    slot_rr = {0: 4, 2: 9}[axis]                 # xx / nn
    slot_tr = {0: 1, 2: 3}[axis]                 # tx / tn
    others = {0: (7, 9), 2: (4, 7)}[axis]        # the two transverse diagonal components: -pi^{rr}/2 each (traceless in the rest frame)
    pi[slot_rr] = pl
    pi[slot_tr] = pl * v                         # transversality pi^{mu nu} u_nu = 0 (second order in A)
    pi[0] = pl * v * v
    for s in others:
        pi[s] = -0.5 * pl * (1.0 - v * v)        # keeps g_{mu nu} pi^{mu nu} = 0 to second order
    o = vo.Oracle(prm)
    o.set_initial(e, u, pi)
    n_steps = 400                                # T = 2 fm: boundary effects (outflow ghosts) travel 2 fm at most; the grid is 19.2 fm long
    o.step(n_steps)
    T_end = n_steps * dt
    f = o.get_fields()
    mid = slice(n // 2 - 128, n // 2 + 128)      # two wavelengths in the middle
    proj = lambda arr: 2.0 * np.mean(arr.reshape(-1)[mid] * np.exp(-1j * k * x[mid]))
    got_u = proj(f["u"][1 + axis])
    got_e = proj(f["e"] - e0)
    got_pi = proj(f["q"][4 + slot_rr])
    exp_u = A * np.exp(-1j * w * T_end)
    # the eigenmode decays by a factor that a first-order (Navier-Stokes) estimate or a missing relaxation time would get wrong
    decay = abs(exp_u) / A
    assert 0.2 < decay < 0.9
    assert abs(got_u - exp_u) / abs(exp_u) < 0.01
    assert abs(got_e - de * exp_u) / abs(de * exp_u) < 0.01
    assert abs(got_pi - dpi * exp_u) / abs(dpi * exp_u) < 0.01
    assert o.status()["n_inversion_failures"] == 0
    # the transverse components follow -pi^{rr}/2
    assert abs(proj(f["q"][4 + others[0]]) + 0.5 * got_pi) / abs(got_pi) < 1e-3


def test_diagonal_shock_tube_2plus1d(vo):
    # PAPER.md 5.2: membrane along y = x.  (a) mirror symmetry about the line y = -x, which maps the problem onto itself:
    # e(x, y) = e(-y, -x), (v_x, v_y) -> (-v_y, -v_x);  (b) along the normal through the origin the plateau of the analytic 1-d solution
    n = 101
    prm, init, xn = inputs.config_diagonal_shocktube(n=n)
    o = vo.Oracle(prm)
    o.set_initial(init["e"], init["u"])
    n_steps = 100                                   # t = 2.5 fm
    o.step(n_steps)
    f = o.get_fields()
    assert o.status()["n_inversion_failures"] == 0
    e = f["e"][0, 0]
    ux, uy, ut = f["u"][1][0, 0], f["u"][2][0, 0], f["u"][0][0, 0]
    mirror = lambda a: a[::-1, ::-1].T               # (x, y) -> (-y, -x) on the centred grid
    assert np.max(np.abs(e - mirror(e))) <= 1e-12 * np.max(e)
    assert np.max(np.abs(ux + mirror(uy))) <= 1e-12
    # (b) cells on the anti-diagonal j = n-1-i lie on the normal through the origin: x' = (x - y)/sqrt2 = sqrt2 x
    t = n_steps * prm["dtau"]
    idx = np.arange(n)
    xprime = xn[n - 1 - idx, idx]
    e_line = e[n - 1 - idx, idx]
    vn_line = ((ux - uy) / math.sqrt(2.0) / ut)[n - 1 - idx, idx]
    eL, eR = init["e"].max(), init["e"].min()
    ep, vp, Vs = analytic.riemann_plateau(eL, eR)
    tail = (vp - analytic.CS) / (1 - vp * analytic.CS)
    plat = (xprime > tail * t + 0.6) & (xprime < Vs * t - 0.45)
    assert plat.sum() >= 4
    assert np.max(np.abs(e_line[plat] / ep - 1)) < 0.01
    assert np.max(np.abs(vn_line[plat] / vp - 1)) < 0.01
    # the whole profile against the analytic solution in the L1 sense (first-order accurate at the shock)
    inner = np.abs(xprime) < 3.5
    ea, va = analytic.riemann_solution(xprime[inner], t, eL, eR)
    assert np.mean(np.abs(e_line[inner] - ea)) / eL < 0.02
    # the flow is along the normal: the tangential velocity vanishes
    assert np.max(np.abs((ux + uy)[n - 1 - idx, idx][inner])) < 1e-12


def test_cylindrical_blast_keeps_its_symmetry(vo):
    # PAPER.md 5.3 (:718): cylindrical symmetry on the Cartesian grid.  The discrete problem is invariant under the symmetry group of the
    # square (x -> -x, y -> -y, x <-> y): these hold to rounding; the radial profile along an axis and along the diagonal agree to
    # truncation error, the shock runs outwards and the centre rarefies.
    n = 101
    prm, init, r = inputs.config_blast(n=n)
    o = vo.Oracle(prm)
    o.set_initial(init["e"], init["u"])
    o.step(80)                                      # t = 2 fm
    f = o.get_fields()
    assert o.status()["n_inversion_failures"] == 0
    e, ux, uy, ut = f["e"][0, 0], f["u"][1][0, 0], f["u"][2][0, 0], f["u"][0][0, 0]
    tol = 1e-12 * np.max(e)
    assert np.max(np.abs(e - e[:, ::-1])) <= tol and np.max(np.abs(e - e[::-1, :])) <= tol and np.max(np.abs(e - e.T)) <= tol
    assert np.max(np.abs(ux + ux[:, ::-1])) <= 1e-12 and np.max(np.abs(ux - uy.T)) <= 1e-12
    c = n // 2
    # radial velocity is outward and the tangential one vanishes on the axis and on the diagonal
    x = inputs.centred_axis(n, prm["dx"])
    vr_axis = (ux / ut)[c, c:]
    vr_diag = np.array([((ux[c + m, c + m] + uy[c + m, c + m]) / math.sqrt(2.0)) / ut[c + m, c + m] for m in range(0, 36)])
    assert np.min(vr_axis) > -1e-12 and np.max(np.abs(uy[c, :])) <= 1e-12
    # same radial profile along the axis and along the diagonal (interpolated to the same radii), to truncation error of the scheme
    r_axis, r_diag = x[c:], math.sqrt(2.0) * x[c:c + 36]
    e_axis = e[c, c:]
    e_diag = np.array([e[c + m, c + m] for m in range(0, 36)])
    e_diag_on_axis = np.interp(r_axis[r_axis < r_diag[-1]], r_diag, e_diag)
    sel = r_axis < r_diag[-1]
    assert np.max(np.abs(e_diag_on_axis - e_axis[sel])) / np.max(e_axis) < 0.10      # 7 % at r = 0.3 fm = 3 cells
    vr_on_axis = np.interp(r_axis[sel], r_diag, vr_diag)
    assert np.max(np.abs(vr_on_axis - vr_axis[sel])) < 0.10
    # the blast has expanded: the centre is below its initial value and the shock sits between 1.5 and 3 fm
    assert e[c, c] < 0.5 * init["e"].max()
    front = r_axis[np.nonzero(e_axis > 1.05 * init["e"].min())[0][-1]]      # outermost cell the shock has reached
    assert 1.8 < front < 3.0
