"""Pins of the oracle's regularisation (Eqs. 73-74; reading R9) and of the order invert -> regulate
(program-flow steps 2-3, :510-511; reading R8) for a MOVING fluid, tau != 1 and a pi^{mu nu} that violates the constraints of
Eqs. 47-51 in a chosen way.

The expected rho never retypes the component sums of regulate_cell().  The states are BUILT from their Lorentz-invariant content:
in an orthonormal local rest frame pi_T = diag(0, a, b, -(a+b)) is traceless and transverse with pi_T:pi_T = a^2 + b^2 + (a+b)^2;
a violation c (u^mu z^nu + z^mu u^nu) with a unit spacelike z orthogonal to u has zero trace, contracts with u_nu to c z^mu and
adds -2 c^2 to the invariant; a violation c u^mu u^nu has trace c, contracts to c u^mu and adds c^2.  The rest frame is carried to
the Milne components by a textbook Lorentz boost in the orthonormal basis (tau, x, y, tau*eta), so each entry of the max of
Eq. 74 is known in closed form.  A dense-metric numpy evaluation of Eq. 74 is checked beside it.
"""
import math

import numpy as np
import pytest

from paper_1608_06577_b200 import inputs

SLOT = [[0, 1, 2, 3], [1, 4, 5, 6], [2, 5, 7, 8], [3, 6, 8, 9]]      # pi10 order tt tx ty tn xx xy xn yy yn nn


def boost(vx, vy, vz):
    """Lorentz boost matrix (orthonormal basis) that takes the rest frame to the frame where the fluid moves with velocity v."""
    v2 = vx * vx + vy * vy + vz * vz
    gam = 1.0 / math.sqrt(1.0 - v2)
    L = np.eye(4)
    v = np.array([vx, vy, vz])
    L[0, 0] = gam
    L[0, 1:] = gam * v
    L[1:, 0] = gam * v
    if v2 > 0:
        L[1:, 1:] += (gam - 1.0) * np.outer(v, v) / v2
    return L


def milne_components(X_orth, tau):
    """contravariant Milne components of a tensor given in the orthonormal basis (tau, x, y, tau*eta): each eta index divides by tau"""
    s = np.array([1.0, 1.0, 1.0, 1.0 / tau])
    return X_orth * np.outer(s, s)


def pack10(X):
    out = np.zeros(10)
    for m in range(4):
        for n in range(m, 4):
            out[SLOT[m][n]] = X[m, n]
    return out


def run_post(vo, prm, e0, u_milne, pi_milne, Pi, tau):
    shp = (1, 1, 1, 1)
    o = vo.Oracle(prm)
    o.set_initial(np.full(shp, e0), u_milne.reshape((4,) + shp), pack10(pi_milne).reshape((10,) + shp), np.full(shp, Pi))
    q_before = np.array([o.raw("q", n)[2, 2, 2] for n in range(15)])
    o.post(tau)
    q_after = np.array([o.raw("q", n)[2, 2, 2] for n in range(15)])
    e_after = o.raw("e")[2, 2, 2]
    u_after = np.array([o.raw("u", m)[2, 2, 2] for m in range(4)])
    return q_before, q_after, e_after, u_after


def eq74_dense(pi_milne, Pi, u_milne, e0, p0, tau, xi0, rho_max):
    """Eq. 74 written with the full 4x4 metric matrix (no diagonal shortcuts); returns rho and the five constraint entries."""
    g = np.diag([1.0, -1.0, -1.0, -tau * tau])
    u_lo = g @ u_milne
    pi_lo = g @ pi_milne @ g
    PP = math.sqrt(abs(np.sum(pi_milne * pi_lo) + 3.0 * Pi * Pi))
    trace = np.trace(g @ pi_milne)
    pu = pi_milne @ u_lo
    pu[3] *= tau
    entries = np.abs(np.concatenate(([trace], pu))) / (xi0 * rho_max * PP)
    return max(PP / (rho_max * math.sqrt(e0 * e0 + 3.0 * p0 * p0)), entries.max()), entries


@pytest.mark.parametrize("case", ["z_eta", "z_x", "z_y", "uu"])
def test_transversality_entries_of_eq74_for_a_moving_fluid(vo, case):
    tau = 2.0
    prm = inputs.base_params(nx=1, ny=1, nz=1, tau0=tau, eos=0, physics=3, zeta_model=0)
    e0, Pi = 7.0, 0.0
    p0 = e0 / 3.0
    a, b = 0.30, -0.11                                  # rest-frame eigenvalues of the transverse traceless part
    inv_T = a * a + b * b + (a + b) ** 2                # pi_T : pi_T (Lorentz invariant)
    # fluid moving along the direction of z (boost along one axis): u = gamma (1, v), z = gamma (v, 1) in the orthonormal basis
    axis = {"z_eta": 3, "z_x": 1, "z_y": 2, "uu": 3}[case]
    v = 0.55
    vel = [0.0, 0.0, 0.0]
    vel[axis - 1] = v
    L = boost(*vel)
    gam = 1.0 / math.sqrt(1 - v * v)
    u_orth = L @ np.array([1.0, 0, 0, 0])
    z_rest = np.zeros(4)
    z_rest[axis] = 1.0
    z_orth = L @ z_rest
    piT_rest = np.diag([0.0, a, b, -(a + b)])
    piT_orth = L @ piT_rest @ L.T
    c = 0.02
    if case == "uu":
        X_orth = c * np.outer(u_orth, u_orth)
        inv = inv_T + c * c
        # trace entry |c|; transversality entries |c u^lambda| (eta entry times tau = orthonormal component): the largest is c u^tau
        expect_entry = abs(c) * gam
    else:
        X_orth = c * (np.outer(u_orth, z_orth) + np.outer(z_orth, u_orth))
        inv = inv_T - 2.0 * c * c
        # entries |c z^lambda| in the orthonormal basis: (gamma v, ..., gamma at the axis): the axis entry wins since gamma > gamma v
        expect_entry = abs(c) * gam
    u_milne = u_orth * np.array([1, 1, 1, 1 / tau])
    pi_milne = milne_components(piT_orth + X_orth, tau)
    rho_expected = expect_entry / (prm["xi0"] * prm["rho_max"] * math.sqrt(abs(inv)))
    assert rho_expected > 0.5                              # the constraint entry, not the first entry, decides (first entry ~ 0.05)
    rho_dense, entries = eq74_dense(pi_milne, Pi, u_milne, e0, p0, tau, prm["xi0"], prm["rho_max"])
    assert rho_dense == pytest.approx(rho_expected, rel=1e-12)
    # which entry of the max is it?  (0 trace, 1..4 lambda = tau, x, y, eta)
    win = int(np.argmax(entries))
    assert win == (1 if case == "uu" else 1 + axis)
    if case == "z_eta":
        # without the factor tau on the lambda = eta entry (Eq. 74 in the units of the other entries, R9) the lambda = tau entry would win
        assert entries[4] / tau < entries[1]
    qb, qa, e_after, u_after = run_post(vo, prm, e0, u_milne, pi_milne, Pi, tau)
    fac = math.tanh(rho_expected) / rho_expected
    for n in range(4, 14):
        assert qa[n] == pytest.approx(qb[n] * fac, rel=1e-11, abs=1e-15)
    # R8: e and u come from the UN-regulated q (E = T^{tau tau} - pi^{tau tau} with the pi of before the scaling): they equal the
    # values the state was built from, although pi^{tau mu} changed by the factor
    assert abs(qb[4]) > 1e-3 and fac < 0.95
    assert e_after == pytest.approx(e0, rel=1e-12)
    assert np.allclose(u_after, u_milne, rtol=1e-12, atol=1e-14)
    # T^{tau mu} themselves are not touched by the regularisation
    assert np.array_equal(qa[:4], qb[:4])


def test_trace_entry_of_eq74(vo):
    # pi = pi_T + c Delta^{mu nu}: transverse, trace 3c, invariant pi_T:pi_T + 3 c^2 -> rho = 3|c| / (xi0 rho_max sqrt(...))
    tau = 0.7
    prm = inputs.base_params(nx=1, ny=1, nz=1, tau0=tau, eos=0, physics=3, zeta_model=0)
    e0 = 4.0
    a, b, c = 0.2, 0.05, 0.004
    L = boost(0.3, -0.4, 0.5)
    u_orth = L @ np.array([1.0, 0, 0, 0])
    eta_mink = np.diag([1.0, -1.0, -1.0, -1.0])
    Delta = eta_mink - np.outer(u_orth, u_orth)
    piT_orth = L @ np.diag([0.0, a, b, -(a + b)]) @ L.T
    u_milne = u_orth * np.array([1, 1, 1, 1 / tau])
    pi_milne = milne_components(piT_orth + c * Delta, tau)
    inv = a * a + b * b + (a + b) ** 2 + 3.0 * c * c
    rho_expected = 3.0 * abs(c) / (prm["xi0"] * prm["rho_max"] * math.sqrt(inv))
    rho_dense, entries = eq74_dense(pi_milne, 0.0, u_milne, e0, e0 / 3, tau, prm["xi0"], prm["rho_max"])
    assert int(np.argmax(entries)) == 0 and rho_dense == pytest.approx(rho_expected, rel=1e-11)
    qb, qa, e_after, u_after = run_post(vo, prm, e0, u_milne, pi_milne, 0.0, tau)
    fac = math.tanh(rho_expected) / rho_expected
    for n in range(4, 14):
        assert qa[n] == pytest.approx(qb[n] * fac, rel=1e-10, abs=1e-15)
    assert e_after == pytest.approx(e0, rel=1e-12) and np.allclose(u_after, u_milne, rtol=1e-12, atol=1e-14)


def test_first_entry_of_eq74_uses_the_equilibrium_pressure(vo):
    # exactly transverse, traceless pi_T (the constraint entries vanish to rounding) with a large amplitude and Pi != 0, EOS 1 near e0
    # where P0 is far from e/3: rho = sqrt(pi_T:pi_T + 3 Pi^2) / (rho_max sqrt(e^2 + 3 P0^2)) with the EQUILIBRIUM pressure (R9)
    tau = 1.6
    prm = inputs.base_params(nx=1, ny=1, nz=1, tau0=tau, eos=1, physics=3)
    e0 = 1.2 * prm["eos_e0"]
    p0 = (e0 / 3.0) * (1.0 - prm["eos_alpha"] * math.exp(-e0 / prm["eos_e0"]))      # EOS of BASELINE.json config 3
    assert abs(p0 - e0 / 3) / (e0 / 3) > 0.1
    a, b = 0.9 * e0, -0.2 * e0
    Pi = -0.25 * e0
    L = boost(-0.35, 0.2, 0.6)
    u_orth = L @ np.array([1.0, 0, 0, 0])
    piT_orth = L @ np.diag([0.0, a, b, -(a + b)]) @ L.T
    u_milne = u_orth * np.array([1, 1, 1, 1 / tau])
    pi_milne = milne_components(piT_orth, tau)
    inv = a * a + b * b + (a + b) ** 2 + 3.0 * Pi * Pi
    rho_expected = math.sqrt(inv) / (prm["rho_max"] * math.sqrt(e0 * e0 + 3.0 * p0 * p0))
    rho_wrong_pressure = math.sqrt(inv) / (prm["rho_max"] * math.sqrt(e0 * e0 + 3.0 * (p0 + Pi) ** 2))
    rho_conformal = math.sqrt(inv) / (prm["rho_max"] * math.sqrt(e0 * e0 + 3.0 * (e0 / 3) ** 2))
    assert abs(rho_wrong_pressure / rho_expected - 1) > 0.02 and abs(rho_conformal / rho_expected - 1) > 0.005
    _, entries = eq74_dense(pi_milne, Pi, u_milne, e0, p0, tau, prm["xi0"], prm["rho_max"])
    assert entries.max() < 1e-12                                                     # pi_T is transverse and traceless by construction
    qb, qa, e_after, u_after = run_post(vo, prm, e0, u_milne, pi_milne, Pi, tau)
    fac = math.tanh(rho_expected) / rho_expected
    assert 0.5 < fac < 0.9
    for n in range(4, 15):                                                           # Pi is scaled by the same factor (R9)
        assert qa[n] == pytest.approx(qb[n] * fac, rel=1e-11, abs=1e-15)
    # R8 with a Pi that the scaling changes: the bulk pressure in Eq. 72 is the un-regulated one
    assert e_after == pytest.approx(e0, rel=1e-11)
    assert np.allclose(u_after, u_milne, rtol=1e-11, atol=1e-13)
