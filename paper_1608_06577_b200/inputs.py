"""Seeded synthetic inputs and parameter sets for the workloads of BASELINE.json (configs 1-5).

This module serves BOTH the CUDA path and the test oracle and therefore holds none of the method's
arithmetic (no KT scheme, no sources, no inversion): only parameter dictionaries, a counter-based
random generator, and closed-form / ODE initial profiles.  numpy (+ scipy for the Gubser ODE) only.

Units (reading R13): natural units inside the solver, e in fm^-4, T in fm^-1,
hbar*c = 0.1973269804 GeV fm converts GeV/fm^3 -> fm^-4 and GeV -> fm^-1.

Stand-in statement: the paper's benchmark event is a Monte-Carlo Glauber profile
which is not available; seeded Gaussian hotspots of the shapes given in BASELINE.json configs 3-5 stand in for it.
"""
import math

import numpy as np

HBARC = 0.1973269804  # GeV fm
BASE_SEED = 20160823


def base_params(**over):
    """Parameter dictionary with the paper's transport coefficients (Eqs. 10-16) and the survey's defaults."""
    d = dict(
        nx=1, ny=1, nz=1, n_batch=1,
        dx=0.1, dy=0.1, dz=0.1, tau0=0.5, dtau=0.025,
        geometry=0, physics=3, eos=1,
        eos_a=13.8, eos_alpha=0.4, eos_e0=1.0 / HBARC,
        eta_over_s=0.2,
        zeta_model=1, zeta_amp=0.1, zeta_T0=0.18 / HBARC, zeta_width=0.03 / HBARC,
        c_tau_pi=5.0, c_tau_Pi=5.0,
        delta_pipi=4.0 / 3.0, tau_pipi=10.0 / 7.0, lambda_piPi=6.0 / 5.0,
        delta_PiPi=2.0 / 3.0, lambda_Pipi_coef=8.0 / 5.0,
        minmod_theta=1.0, xi0=0.1, rho_max=1.0,
        newton_max_iter=50, newton_rtol=1e-13,
        tau_relax_floor_over_dtau=5.0,
        storage=0,
    )
    for k, v in over.items():
        if k not in d:
            raise KeyError(k)
        d[k] = v
    return d


# ------------------------------------------------------------------ counter-based RNG (SplitMix64)
class SplitMix64:
    MASK = (1 << 64) - 1

    def __init__(self, seed):
        self.s = seed & self.MASK

    def next_u64(self):
        self.s = (self.s + 0x9E3779B97F4A7C15) & self.MASK
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & self.MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & self.MASK
        return z ^ (z >> 31)

    def uniform(self):
        return (self.next_u64() >> 11) * (1.0 / 9007199254740992.0)  # 2^-53


def centred_axis(n, d):
    return (np.arange(n) - 0.5 * (n - 1)) * d


def hotspots_energy(nx, ny, nz, dx, dy, dz, n_hot, width, seed, three_d, pedestal_gev=0.05, radius=5.0, eta_half=2.0):
    """e(x,y,eta) [fm^-4] = pedestal + sum_h A_h exp(-|x-x_h|^2/(2 w^2)); draw order per hotspot: A, r, phi, (eta).
    Centres uniform in a disc of `radius` fm (5 fm in BASELINE.json) and in |eta| < eta_half (2); small test grids shrink both."""
    rng = SplitMix64(seed)
    A = np.empty(n_hot); xh = np.empty(n_hot); yh = np.empty(n_hot); zh = np.zeros(n_hot)
    for h in range(n_hot):
        A[h] = 5.0 + 25.0 * rng.uniform()
        r = radius * math.sqrt(rng.uniform())
        ph = 2.0 * math.pi * rng.uniform()
        xh[h] = r * math.cos(ph); yh[h] = r * math.sin(ph)
        if three_d:
            zh[h] = eta_half * (-1.0 + 2.0 * rng.uniform())
    x = centred_axis(nx, dx); y = centred_axis(ny, dy); z = centred_axis(nz, dz)
    gx = np.exp(-((x[None, :] - xh[:, None]) ** 2) / (2 * width * width))          # [h, nx]
    gy = np.exp(-((y[None, :] - yh[:, None]) ** 2) / (2 * width * width))          # [h, ny]
    if three_d:
        gz = np.exp(-((z[None, :] - zh[:, None]) ** 2) / (2 * width * width))      # [h, nz]
    else:
        gz = np.ones((n_hot, nz))
    M = (A[:, None, None] * gz[:, :, None] * gy[:, None, :]).reshape(n_hot, nz * ny)  # [h, nz*ny]
    e = (M.T @ gx).reshape(nz, ny, nx) + pedestal_gev
    return e / HBARC


def rest_velocity(shape):
    u = np.zeros((4,) + tuple(shape))
    u[0] = 1.0
    return u


# ------------------------------------------------------------------ config 1: 1d ideal shock tube (PAPER.md :577-579, :634, :684)
def config_shocktube(n=200, axis=0, theta=1.8, cfl=0.5, length=10.0, T_L=0.4, T_R=0.2):
    """BASELINE.json configs[0].  axis 0/1/2 puts the tube along x / y / eta(z)."""
    d = length / n
    dims = [1, 1, 1]
    dims[axis] = n
    prm = base_params(nx=dims[0], ny=dims[1], nz=dims[2], dx=d, dy=d, dz=d, tau0=0.0, dtau=cfl * d, geometry=1, physics=0,
                      eos=0, zeta_model=0, minmod_theta=theta, tau_relax_floor_over_dtau=0.0)
    x = centred_axis(n, d)
    a = prm["eos_a"]
    e1 = np.where(x < 0, a * (T_L / HBARC) ** 4, a * (T_R / HBARC) ** 4)
    shp = (1, dims[2], dims[1], dims[0])
    e = np.empty(shp)
    bshape = [1, 1, 1, 1]
    bshape[3 - axis] = n
    e[...] = e1.reshape(bshape)
    return prm, dict(e=e, u=rest_velocity(shp), pi=None, Pi=None), 100, x


def config_diagonal_shocktube(n=101, d=0.1, cfl=0.25, theta=1.0, e_hi=0.0246, e_lo=0.0015):
    """PAPER.md 5.2 (:696-704): the Sod membrane of section 5.1 placed along the main diagonal y = x of the transverse grid; energy
    densities of :634 in GeV/fm^3, p = e/3, ideal, Cartesian.  High side: y > x.  Returns the coordinate x' = (x - y)/sqrt2 normal
    to the membrane as the last item."""
    prm = base_params(nx=n, ny=n, nz=1, dx=d, dy=d, dz=d, tau0=0.0, dtau=cfl * d, geometry=1, physics=0, eos=0, zeta_model=0,
                      minmod_theta=theta, tau_relax_floor_over_dtau=0.0)
    x = centred_axis(n, d)
    X, Y = np.meshgrid(x, x, indexing="xy")            # [y, x]
    xn = (X - Y) / math.sqrt(2.0)
    shp = (1, 1, n, n)
    e = np.where(xn < -1e-12, e_hi / HBARC, e_lo / HBARC).reshape(shp)
    return prm, dict(e=e, u=rest_velocity(shp), pi=None, Pi=None), xn


def config_blast(n=101, d=0.1, cfl=0.25, theta=1.0, radius=1.0, e_in=0.0246, e_out=0.0015):
    """PAPER.md 5.3 (:706-718): cylindrical explosion - e = 0.0246 GeV/fm^3 inside r <= R = 1 fm, 0.0015 GeV/fm^3 outside, in a
    10 x 10 fm^2 box, p = e/3, ideal, Cartesian.  Returns r(x, y) as the last item."""
    prm = base_params(nx=n, ny=n, nz=1, dx=d, dy=d, dz=d, tau0=0.0, dtau=cfl * d, geometry=1, physics=0, eos=0, zeta_model=0,
                      minmod_theta=theta, tau_relax_floor_over_dtau=0.0)
    x = centred_axis(n, d)
    X, Y = np.meshgrid(x, x, indexing="xy")
    r = np.sqrt(X * X + Y * Y)
    shp = (1, 1, n, n)
    e = np.where(r <= radius, e_in / HBARC, e_out / HBARC).reshape(shp)
    return prm, dict(e=e, u=rest_velocity(shp), pi=None, Pi=None), r


# ------------------------------------------------------------------ config 2: Gubser flow (PAPER.md :757-779)
def gubser_ode(eta_over_s, c_tau_pi, T0hat=1.2, rho_lo=-12.0, rho_hi=6.0):
    """Conformal Israel-Stewart under Gubser symmetry (tau_pipi = 0), with pibar = pihat^eta_eta/(ehat+phat):
         (1/T) dT/drho + (2/3) tanh(rho) = (1/3) pibar tanh(rho)
         (c (eta/s)/T) [dpibar/drho + (4/3) pibar^2 tanh(rho)] + pibar = (4/3)(eta/s) tanh(rho)/T
       (the equations PAPER.md:775 refers to; re-derived in SURVEY.md 8(c) T4).  Data at rho=0: T=T0hat, pibar=0.
       Returns callables That(rho), pibar(rho)."""
    from scipy.integrate import solve_ivp

    if eta_over_s <= 0:
        return (lambda rho: T0hat / np.cosh(rho) ** (2.0 / 3.0)), (lambda rho: np.zeros_like(np.asarray(rho, dtype=float)))

    def rhs(rho, y):
        T, pb = y
        th = math.tanh(rho)
        dT = T * (pb * th / 3.0 - 2.0 * th / 3.0)
        dpb = (4.0 / 3.0 * eta_over_s * th / T - pb) * T / (c_tau_pi * eta_over_s) - 4.0 / 3.0 * pb * pb * th
        return [dT, dpb]

    kw = dict(method="DOP853", rtol=1e-12, atol=1e-14, dense_output=True)
    fw = solve_ivp(rhs, [0.0, rho_hi], [T0hat, 0.0], **kw)
    bw = solve_ivp(rhs, [0.0, rho_lo], [T0hat, 0.0], **kw)

    def ev(rho, k):
        rho = np.asarray(rho, dtype=float)
        out = np.empty_like(rho)
        m = rho >= 0
        if m.any():
            out[m] = fw.sol(rho[m])[k]
        if (~m).any():
            out[~m] = bw.sol(rho[~m])[k]
        return out

    return (lambda rho: ev(rho, 0)), (lambda rho: ev(rho, 1))


def gubser_fields(tau, X, Y, That, pibar, a=13.8, q=1.0):
    """Milne-frame (e, u^mu, pi^{mu nu}) of the Gubser solution at proper time tau on the transverse points X, Y."""
    r = np.sqrt(X * X + Y * Y)
    rho = np.arcsinh(-(1.0 - q * q * tau * tau + q * q * r * r) / (2.0 * q * tau))
    T = That(rho) / tau
    e = a * T ** 4
    p = e / 3.0
    kap = np.arctanh(2.0 * q * q * tau * r / (1.0 + q * q * tau * tau + q * q * r * r))
    ch, sh = np.cosh(kap), np.sinh(kap)
    with np.errstate(invalid="ignore", divide="ignore"):
        cx = np.where(r > 0, X / r, 0.0)
        cy = np.where(r > 0, Y / r, 0.0)
    u = np.stack([ch, sh * cx, sh * cy, np.zeros_like(r)])       # outward flow (reading R16)
    pb = pibar(rho) * (e + p)
    prr = -0.5 * pb                                              # LRF pi = diag(-1/2,-1/2,+1) pibar (e+p) in (r, phi, eta)
    pff = -0.5 * pb
    ptt = prr * sh * sh
    ptr = prr * sh * ch
    prr_b = prr * ch * ch
    pi = np.stack([
        ptt, ptr * cx, ptr * cy, np.zeros_like(r),
        prr_b * cx * cx + pff * cy * cy, (prr_b - pff) * cx * cy, np.zeros_like(r),
        prr_b * cy * cy + pff * cx * cx, np.zeros_like(r), pb / (tau * tau)])
    # at r = 0 the transverse tensor is isotropic: pi^xx = pi^yy = -pb/2 (cx=cy=0 above would give 0)
    z = r == 0
    if z.any():
        pi[4][z] = prr[z]; pi[7][z] = prr[z]
    return e, u, pi


def config_gubser(n=201, d=0.05, eta_over_s=0.2, n_steps=400, theta=1.8):
    """BASELINE.json configs[1]; ideal Gubser (Eqs. 82-85) when eta_over_s == 0."""
    viscous = eta_over_s > 0
    prm = base_params(nx=n, ny=n, nz=1, dx=d, dy=d, dz=1.0, tau0=1.0, dtau=0.0125, geometry=0,
                      physics=1 if viscous else 0, eos=0, zeta_model=0, eta_over_s=eta_over_s if viscous else 0.2,
                      tau_pipi=0.0, minmod_theta=theta, tau_relax_floor_over_dtau=0.0)
    That, pibar = gubser_ode(eta_over_s, prm["c_tau_pi"])
    x = centred_axis(n, d)
    X, Y = np.meshgrid(x, x, indexing="xy")          # [ny, nx]
    e, u, pi = gubser_fields(prm["tau0"], X, Y, That, pibar, a=prm["eos_a"])
    shp = (1, 1, n, n)
    init = dict(e=e.reshape(shp), u=u.reshape((4,) + shp), pi=pi.reshape((10,) + shp) if viscous else None, Pi=None)
    return prm, init, n_steps, (x, That, pibar)


# ------------------------------------------------------------------ configs 3-5: seeded hotspots
def config_3d(nx=128, ny=128, nz=128, dx=0.1, dy=0.1, dz=0.1, n_hot=40, width=0.5, seed=BASE_SEED, n_steps=100, radius=5.0, eta_half=2.0,
              **over):
    """BASELINE.json configs[2] (defaults) and configs[4] (512,512,128, dx=dy=0.05, n_hot=200, n_steps=50)."""
    prm = base_params(nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, tau0=0.5, dtau=0.025, **over)
    e = hotspots_energy(nx, ny, nz, dx, dy, dz, n_hot, width, seed, three_d=True, radius=radius, eta_half=eta_half)
    shp = (1, nz, ny, nx)
    return prm, dict(e=e.reshape(shp), u=rest_velocity(shp), pi=None, Pi=None), n_steps


def config_batched2d(n_batch=256, n=201, d=0.1, n_hot=20, width=0.4, seed=BASE_SEED, n_steps=200, radius=5.0, **over):
    """BASELINE.json configs[3]: n_batch independent 2+1d events, event b seeded with seed+b."""
    prm = base_params(nx=n, ny=n, nz=1, n_batch=n_batch, dx=d, dy=d, dz=1.0, tau0=0.5, dtau=0.025, **over)
    e = np.empty((n_batch, 1, n, n))
    for b in range(n_batch):
        e[b] = hotspots_energy(n, n, 1, d, d, 1.0, n_hot, width, seed + b, three_d=False, radius=radius)
    shp = (n_batch, 1, n, n)
    return prm, dict(e=e, u=rest_velocity(shp), pi=None, Pi=None), n_steps


def config_large3d():
    return config_3d(512, 512, 128, 0.05, 0.05, 0.1, n_hot=200, n_steps=50)


def smooth_random_state(prm, seed=7, amp_v=0.3, amp_pi=0.05):
    """A generic smooth state with non-zero flow in all directions, shear stress and bulk pressure, for parity tests
    that must exercise every term (vorticity, u^eta != 0, all ten pi components).  Sum of a few seeded Fourier modes."""
    nx, ny, nz, nb = prm["nx"], prm["ny"], prm["nz"], prm["n_batch"]
    rng = SplitMix64(seed)
    x = (np.arange(nx) + 0.5) / nx; y = (np.arange(ny) + 0.5) / ny; z = (np.arange(nz) + 0.5) / nz
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")

    def field():
        f = np.zeros((nb, nz, ny, nx))
        for b in range(nb):
            for _ in range(3):
                kx, ky, kz = (int(3 * rng.uniform()) for _ in range(3))
                ph = 2 * math.pi * rng.uniform()
                am = rng.uniform() - 0.5
                f[b] += am * np.cos(2 * math.pi * (kx * X + ky * Y + (kz * Z if nz > 1 else 0.0)) + ph)
        return f

    e = (2.0 + 1.0 * field()) * 5.0
    ux = amp_v * field(); uy = amp_v * field()
    un = (amp_v * field() if nz > 1 else np.zeros_like(ux)) / prm["tau0"]
    t2 = prm["tau0"] ** 2 if prm["geometry"] == 0 else 1.0
    ut = np.sqrt(1.0 + ux * ux + uy * uy + t2 * un * un)
    u = np.stack([ut, ux, uy, un])
    pi = np.stack([amp_pi * field() for _ in range(10)])
    pi[3] /= prm["tau0"]; pi[6] /= prm["tau0"]; pi[8] /= prm["tau0"]; pi[9] /= prm["tau0"] ** 2
    Pi = amp_pi * field()
    return dict(e=e, u=u, pi=pi, Pi=Pi)
