// vh_device.cuh -- device-side arithmetic of the KT / Heun step (product path; shares nothing with oracle/).
// Citations are PAPER.md lines / equations.  Component forms (App. A, A.12, A.14-A.19, B.12) are used here; the
// test oracle uses index forms.  Readings R1..R18 are listed in DESIGN.md.
#pragma once
#include "vh_real.cuh"

namespace vh {

constexpr int NQ = 15;
// q slots
enum { TTT = 0, TTX, TTY, TTN, PTT, PTX, PTY, PTN, PXX, PXY, PXN, PYY, PYN, PNN, BPI };

constexpr real kVorticitySign = -real(1.0);   // R4: Eq. 8 (:149) with omega^{mu nu} of :122

struct DevParams {
  int nx, ny, nz, n_batch;
  int NXp, NYp, NZp;            // padded extents (NXp is the row pitch, multiple of 16 doubles = 128 B)
  long long plane;              // NXp*NYp
  long long bstride;            // NXp*NYp*NZp   (one event)
  long long fstride;            // bstride*n_batch (one field)
  int zoff;                     // 2 (3+1d) or 0 (2+1d: no eta ghost planes are stored)
  real dx, dy, dz, dtau;
  real inv_dx, inv_dy, inv_dz, inv_dtau;
  int shear, bulk;              // physics bits
  real eos_a_inv, eos_alpha, eos_e0_inv;
  // EOS 2 (lattice, Eqs. 19-20; R19, R20): table of kN + 1 nodes uniform in x = e^{1/4}, node k = (P, h dP/dx, T, h dT/dx)
  const real2* eos_tab; int eos_n; real eos_x0, eos_xN, eos_inv_h, eos_lo_slope, eos_pN, eos_eN, eos_T0_over_x0, eos_TN_over_xN;
  real inv_ctaupi_etas;       // 1/(c_tau_pi * eta/s)
  real inv_ctaupi;            // 1/c_tau_pi
  int zeta_model; real zeta_amp, zeta_T0, zeta_inv_width, inv_ctauPi;
  real delta_pipi, tau_pipi, lambda_piPi, delta_PiPi, lambda_Pipi_coef;
  real theta;                 // minmod theta
  real inv_rho_max, xi0_rho_max;
  int newton_max_iter; real newton_rtol;
  real newton_stop;             // convergence test of the product kernels: |de| <= newton_stop |e| guarantees |next de| <= newton_rtol |e| (see fill_dev_params)
  real relax_clamp;           // 1/(c*dtau) or +inf
};

// (rcp_fast, rcp_half, rsqrt_fast, sqrt_fast, exp_neg, sign_differs: vh_real.cuh, one overload per precision)

// ---------------------------------------------------------------- EOS (BASELINE.json configs) and transport (Eqs. 10-16)
template <int EOS> __device__ __forceinline__ void eos_p_cs2(const DevParams& P, real e, real& p, real& cs2) {
  if (EOS == 0) {
    p = e * (real(1.0) / real(3.0));
    cs2 = real(1.0) / real(3.0);
  } else {
    real x = e * P.eos_e0_inv;
    real aex = P.eos_alpha * exp_neg(x);
    p = (e * (real(1.0) / real(3.0))) * (real(1.0) - aex);
    cs2 = (real(1.0) / real(3.0)) * (real(1.0) - aex * (real(1.0) - x));
  }
}
// EOS 2: cubic Hermite interpolation in x = e^{1/4} of the tabulated lattice pressure and temperature (R20); c_s^2 is the
// derivative of the pressure interpolant.  Below the table P = (P_0/e_0) e, T = (T_0/x_0) x; above it P = P_N + (e - e_N)/3.
__device__ __forceinline__ void eos_lattice(const DevParams& P, real e, real& p, real& cs2, real& T) {
  // x = e^{1/4} as rsqrt(rsqrt(e)), y = e^{-1/2}: two MUFU seeds with two Newton steps each, no IEEE square-root slow path, and
  // 1/x^3 = x y^2 comes for free (e <= 0 or NaN falls into the first branch below)
  const real y = rsqrt_fast(e);
  const real x = (e > real(0.0)) ? rsqrt_fast(y) : real(0.0);
  if (!(x >= P.eos_x0)) { p = P.eos_lo_slope * e; cs2 = P.eos_lo_slope; T = P.eos_T0_over_x0 * x; return; }
  if (x >= P.eos_xN) { p = fma(e - P.eos_eN, real(1.0) / real(3.0), P.eos_pN); cs2 = real(1.0) / real(3.0); T = P.eos_TN_over_xN * x; return; }
  const real u = (x - P.eos_x0) * P.eos_inv_h;
  const int k = min((int)u, P.eos_n - 1);
  const real s = u - (real)k, s2 = s * s, s3 = s2 * s;
  const real2 ap = __ldg(P.eos_tab + 2 * k), at = __ldg(P.eos_tab + 2 * k + 1), bp = __ldg(P.eos_tab + 2 * k + 2), bt = __ldg(P.eos_tab + 2 * k + 3);
  const real h00 = real(2.0) * s3 - real(3.0) * s2 + real(1.0), h10 = s3 - real(2.0) * s2 + s, h01 = real(3.0) * s2 - real(2.0) * s3, h11 = s3 - s2;
  p = h00 * ap.x + h10 * ap.y + h01 * bp.x + h11 * bp.y;
  T = h00 * at.x + h10 * at.y + h01 * bt.x + h11 * bt.y;
  const real d00 = real(6.0) * (s2 - s), d10 = real(3.0) * s2 - real(4.0) * s + real(1.0), d11 = real(3.0) * s2 - real(2.0) * s;
  const real dpdx = (d00 * (ap.x - bp.x) + d10 * ap.y + d11 * bp.y) * P.eos_inv_h;
  cs2 = dpdx * (real(0.25) * x) * (y * y);
}
template <> __device__ __forceinline__ void eos_p_cs2<2>(const DevParams& P, real e, real& p, real& cs2) {
  real T;
  eos_lattice(P, e, p, cs2, T);
}
// temperature for the transport coefficients: T = (e/a)^{1/4} for the analytic EOS, T(e) of the table for EOS 2
template <int EOS> __device__ __forceinline__ real eos_temperature(const DevParams& P, real e) {
  if (EOS == 2) { real p, c, T; eos_lattice(P, e, p, c, T); return T; }
  const real y = e * P.eos_a_inv;
  return sqrt(sqrt(y));
}
template <int EOS> __device__ __forceinline__ real eos_p(const DevParams& P, real e) {
  real p, c;
  eos_p_cs2<EOS>(P, e, p, c);
  return p;
}

// ---------------------------------------------------------------- zeta/s(T)
// zeta_model 0: none; 1: Gaussian amp exp(-((T - T0)/width)^2) (BASELINE.json configs 3-5); 2: constant amp;
// 3: the paper's parametrisation, Eq. 17 (:174-186), times (zeta/s)_norm = zeta_amp, with T_c = zeta_T0 and the ranges read as
//    T < 0.995 T_c, 0.995 T_c <= T <= 1.05 T_c, T > 1.05 T_c (the printed inequalities are reversed, reading R3).
__device__ __forceinline__ real zeta_over_s(const DevParams& P, real T) {
  if (P.zeta_model == 1) { const real d = (T - P.zeta_T0) * P.zeta_inv_width; return P.zeta_amp * exp_neg(d * d); }
  if (P.zeta_model == 2) return P.zeta_amp;
  if (P.zeta_model == 3) {
    const real x = T * P.zeta_inv_width;      // T / T_c (zeta_inv_width holds 1/T_c for this model)
    real z;
    if (x > real(1.05)) z = real(0.9) * exp_neg((x - real(1.0)) * (real(1.0) / real(0.025))) + real(0.25) * exp_neg((x - real(1.0)) * (real(1.0) / real(0.13))) + real(0.001);
    else if (x < real(0.995)) z = real(0.9) * exp_neg((real(1.0) - x) * (real(1.0) / real(0.0025))) + real(0.22) * exp_neg((real(1.0) - x) * (real(1.0) / real(0.022))) + real(0.03);
    else z = -real(13.45) + x * (real(27.55) - real(13.77) * x);
    return P.zeta_amp * z;
  }
  return real(0.0);
}

// ---------------------------------------------------------------- Newton-Raphson on Eq. 72 (R6)
// returns e; fail is set when no acceptable root was found (then e = max(E, tiny)).
template <int EOS> __device__ __forceinline__ real invert_energy(const DevParams& P, real E, real M2, real Pi, real guess, bool& fail) {
  bool bad = !(E > real(0.0)) || !isfinite(E) || !isfinite(M2) || !isfinite(Pi);
  real e = (guess > real(0.0) && isfinite(guess)) ? guess : E;
  bool done = bad, conv = false;
  for (int it = 0; it < P.newton_max_iter; ++it) {
    if (__all_sync(0xffffffffu, done)) break;     // warp-level convergence vote; every caller is warp-converged
    if (!done) {
      real p, cs2;
      eos_p_cs2<EOS>(P, e, p, cs2);
      real den = E + p + Pi;
      real rden = real(1.0) / den;
      real f = e - E + M2 * rden;
      real fp = real(1.0) - M2 * cs2 * rden * rden;
      real de = f / fp;
      e = e - de;
      if (fabs(de) <= P.newton_rtol * fabs(e)) { conv = true; done = true; }
    }
  }
  fail = bad || !conv || !(e > real(0.0)) || !isfinite(e);
  if (fail) e = (tiny_e() > E) ? tiny_e() : E;      // max(E, tiny) that keeps a NaN E visible to n_nonfinite
  return e;
}

// minmod limited half-slope:  (dr/2) * minmod(theta (q0-qm)/dr, (qp-qm)/(2 dr), theta (qp-q0)/dr)   (Eqs. 67-68, R10)
__device__ __forceinline__ real half_slope(real qm, real q0, real qp, real theta) {
  real a = theta * (q0 - qm), b = real(0.5) * (qp - qm), c = theta * (qp - q0);
  real m = fmin(fmin(fabs(a), fabs(b)), fabs(c));
  bool pos = (a > real(0.0)) && (b > real(0.0)) && (c > real(0.0));
  bool neg = (a < real(0.0)) && (b < real(0.0)) && (c < real(0.0));
  real s = pos ? m : (neg ? -m : real(0.0));
  return real(0.5) * s;
}

// velocity v_r of a reconstructed state along direction r (Alg. 3 :667-672, :424): v^i = M_i/(E + P0(e) + Pi)
template <int EOS, bool MILNE>
__device__ __forceinline__ real state_velocity(const DevParams& P, real E, real Mx, real My, real Mn, real Pi, real t2,
                                                 real guess, int r, bool count, unsigned long long& nfail) {
  real M2 = Mx * Mx + My * My + (MILNE ? t2 : real(1.0)) * Mn * Mn;     // :339
  bool fail;
  real e = invert_energy<EOS>(P, E, M2, Pi, guess, fail);
  real p = eos_p<EOS>(P, e);
  real Mr = (r == 0) ? Mx : ((r == 1) ? My : Mn);
  real v = Mr / (E + p + Pi);
  if (fail) {
    if (count) ++nfail;
    if (!(fabs(v) < real(1.0))) v = (v > real(0.0)) ? clip_one() : ((v < real(0.0)) ? -clip_one() : real(0.0));
  }
  return v;
}

struct Kin {            // kinematic scalars / tensors at a cell (App. A)
  real theta;
  real Du[4];         // covariant Du_lambda (A.9-A.10)
  real sig[10];       // sigma^{mu nu} in the order tt tx ty tn xx xy xn yy yn nn (A.12)
  real W[6];          // W^{tx} W^{ty} W^{tn} W^{xy} W^{xn} W^{yn} (A.14-A.19)
};

// u = (ut,ux,uy,un); dt,dx,dy,dn = partial derivatives of the four components (:424).
// MILNE = false is the Cartesian mode (R12): metric factors tau^2 -> 1 (t2, g2i) and every Christoffel symbol -> 0 (ch = Gamma^eta_{eta tau}
// = 1/tau, ct = Gamma^tau_{eta eta} = tau), kept apart so that each falls out at compile time.
template <bool MILNE>
__device__ __forceinline__ void kinematics(const real u[4], const real dt[4], const real dx[4], const real dy[4], const real dn[4],
                                           real t, Kin& K) {
  const real ut = u[0], ux = u[1], uy = u[2], un = u[3];
  const real t2 = MILNE ? t * t : real(1.0), g2i = MILNE ? real(1.0) / (t * t) : real(1.0);
  const real ch = MILNE ? real(1.0) / t : real(0.0), ct = MILNE ? t : real(0.0);
  // convective derivatives (A.5-A.8)
  real dut = ut * dt[0] + ux * dx[0] + uy * dy[0] + un * dn[0];
  real dux = ut * dt[1] + ux * dx[1] + uy * dy[1] + un * dn[1];
  real duy = ut * dt[2] + ux * dx[2] + uy * dy[2] + un * dn[2];
  real dun = ut * dt[3] + ux * dx[3] + uy * dy[3] + un * dn[3];
  real th = ut * ch + dt[0] + dx[1] + dy[2] + dn[3];                 // A.11
  real th3 = th * (real(1.0) / real(3.0));
  K.theta = th;
  K.Du[0] = dut + ct * un * un;                                         // A.9
  K.Du[1] = -dux;
  K.Du[2] = -duy;
  K.Du[3] = -t2 * (dun + real(2.0) * ch * ut * un);                           // A.10
  real un2 = un * un;
  // A.12 (D(.) read as the convective derivative of the contravariant component, reading in DESIGN.md)
  K.sig[0] = -ct * ut * un2 + dt[0] - ut * dut + (ut * ut - real(1.0)) * th3;
  K.sig[1] = -real(0.5) * ct * un2 * ux + real(0.5) * (dt[1] - dx[0]) - real(0.5) * (ut * dux + ux * dut) + ut * ux * th3;
  K.sig[2] = -real(0.5) * ct * un2 * uy + real(0.5) * (dt[2] - dy[0]) - real(0.5) * (ut * duy + uy * dut) + ut * uy * th3;
  K.sig[3] = -real(0.5) * un * (real(2.0) * ch * ut * ut + ct * un2) + real(0.5) * (dt[3] - dn[0] * g2i) - real(0.5) * (ut * dun + un * dut) + ut * un * th3;
  K.sig[4] = -dx[1] - ux * dux + (real(1.0) + ux * ux) * th3;
  K.sig[5] = -real(0.5) * (dx[2] + dy[1]) - real(0.5) * (ux * duy + uy * dux) + ux * uy * th3;
  K.sig[6] = -ut * ux * un * ch - real(0.5) * (dx[3] + dn[1] * g2i) - real(0.5) * (ux * dun + un * dux) + ux * un * th3;
  K.sig[7] = -dy[2] - uy * duy + (real(1.0) + uy * uy) * th3;
  K.sig[8] = -ut * uy * un * ch - real(0.5) * (dy[3] + dn[2] * g2i) - real(0.5) * (uy * dun + un * duy) + uy * un * th3;
  K.sig[9] = -ut * g2i * ch * (real(1.0) + real(2.0) * un2 * t2) - dn[3] * g2i - un * dun + (g2i + un2) * th3;
  // A.14-A.19 divided by the metric factors so that W^{mu nu} is the contravariant antisymmetric tensor of :122
  K.W[0] = real(0.5) * (dt[1] + dx[0]) + real(0.5) * (ux * dut - ut * dux) + real(0.5) * ct * un2 * ux;
  K.W[1] = real(0.5) * (dt[2] + dy[0]) + real(0.5) * (uy * dut - ut * duy) + real(0.5) * ct * un2 * uy;
  K.W[2] = un * ch + real(0.5) * dt[3] + real(0.5) * dn[0] * g2i + real(0.5) * (un * dut - ut * dun) - ut * ut * un * ch + real(0.5) * ct * un2 * un;
  K.W[3] = real(0.5) * (dy[1] - dx[2]) + real(0.5) * (uy * dux - ux * duy);
  K.W[4] = real(0.5) * dn[1] * g2i - real(0.5) * dx[3] + real(0.5) * (un * dux - ux * dun) - ux * ut * un * ch;
  K.W[5] = real(0.5) * dn[2] * g2i - real(0.5) * dy[3] + real(0.5) * (un * duy - uy * dun) - uy * ut * un * ch;
}

// symmetric-slot lookup for 4x4 symmetric tensors stored as 10 (tt tx ty tn xx xy xn yy yn nn)
__device__ __forceinline__ constexpr int sym(int m, int n) {
  // not recursive: a recursive form is not always folded and then costs a real call plus a dynamically indexed local array
  const int a = (m < n) ? m : n, b = (m < n) ? n : m;
  return (a == 0) ? b : ((a == 1) ? 3 + b : ((a == 2) ? 5 + b : 9));
}

// Dissipative source terms J = S + G for the 10 pi components and Pi (B.10-B.12, Eqs. 39-46).
// pi[10] in slot order; returns Jpi[10], JPi.
template <int EOS, bool MILNE>
__device__ __forceinline__ void dissipative_sources(const DevParams& P, real t, const real u[4], const Kin& K, const real pi[10], real Pi,
                                                    real e, real p, real cs2, real divv, real Jpi[10], real& JPi) {
  const real t2 = MILNE ? t * t : real(1.0), g2i = MILNE ? real(1.0) / (t * t) : real(1.0);      // metric factors
  const real it = MILNE ? real(1.0) / t : real(0.0), ct = MILNE ? t : real(0.0);                  // Christoffel symbols (0 in the Cartesian mode, R12)
  const real g[4] = {real(1.0), -real(1.0), -real(1.0), -t2};
  // transport coefficients (Eqs. 10-16; R14)
  real T = eos_temperature<EOS>(P, e);
  real itp = fmin(T * P.inv_ctaupi_etas, P.relax_clamp);
  real eotp = (e + p) * P.inv_ctaupi;
  const real zs = zeta_over_s(P, T);
  real b = (real(1.0) / real(3.0)) - cs2;
  real itP = (zs > real(0.0)) ? T * b * b * P.inv_ctauPi / zs : inf_r();
  itP = fmin(itP, P.relax_clamp);
  real zotP = (zs > real(0.0)) ? zs * ((e + p) / T) * itP : real(0.0);
  real lPp = P.lambda_Pipi_coef * b;

  // full symmetric / antisymmetric tables
  real S[4][4], W[4][4], Pm[4][4];
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = 0; n < 4; ++n) { S[m][n] = K.sig[sym(m, n)]; Pm[m][n] = pi[sym(m, n)]; }
  W[0][0] = W[1][1] = W[2][2] = W[3][3] = real(0.0);
  W[0][1] = K.W[0]; W[0][2] = K.W[1]; W[0][3] = K.W[2]; W[1][2] = K.W[3]; W[1][3] = K.W[4]; W[2][3] = K.W[5];
  W[1][0] = -K.W[0]; W[2][0] = -K.W[1]; W[3][0] = -K.W[2]; W[2][1] = -K.W[3]; W[3][1] = -K.W[4]; W[3][2] = -K.W[5];

  // A^mu = pi^{lambda mu} Du_lambda ;  B^{mu nu} = pi^{mu l} g_l W^{l nu} ;  C^{mu nu} = g_l pi^{mu l} sigma^{nu l}
  real A[4], B[4][4], C[4][4];
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    A[m] = Pm[0][m] * K.Du[0] + Pm[1][m] * K.Du[1] + Pm[2][m] * K.Du[2] + Pm[3][m] * K.Du[3];
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      real bb = real(0.0), cc = real(0.0);
#pragma unroll
      for (int l = 0; l < 4; ++l) { bb += Pm[m][l] * g[l] * W[l][n]; cc += g[l] * Pm[m][l] * S[n][l]; }
      B[m][n] = bb; C[m][n] = cc;
    }
  }
  real pisig = g[0] * C[0][0] + g[1] * C[1][1] + g[2] * C[2][2] + g[3] * C[3][3];      // pi^{mu nu} sigma_{mu nu}
  const real gi[4] = {real(1.0), -real(1.0), -real(1.0), -g2i};
  const real iut = real(1.0) / u[0];
  // G_pi = u^a Gamma^mu_{ab} pi^{b nu} + (mu<->nu)  (:300; R1, R2)
  real G[10];
  const real ut = u[0], un = u[3];
  G[0] = real(2.0) * ct * un * pi[3];
  G[1] = ct * un * pi[6];
  G[2] = ct * un * pi[8];
  G[3] = ct * un * pi[9] + (ut * pi[3] + un * pi[0]) * it;
  G[4] = real(0.0); G[5] = real(0.0);
  G[6] = (ut * pi[6] + un * pi[1]) * it;
  G[7] = real(0.0);
  G[8] = (ut * pi[8] + un * pi[2]) * it;
  G[9] = real(2.0) * (ut * pi[9] + un * pi[3]) * it;
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = m; n < 4; ++n) {
      const int s = sym(m, n);
      real Dmn = ((m == n) ? gi[m] : real(0.0)) - u[m] * u[n];
      real I1 = u[n] * A[m] + u[m] * A[n];                                   // Eq. 43
      real I2 = K.theta * pi[s];                                             // Eq. 44
      real I3 = kVorticitySign * (B[m][n] + B[n][m]);                        // Eq. 45 (R4)
      real I4 = real(0.5) * (C[m][n] + C[n][m]) - (real(1.0) / real(3.0)) * Dmn * pisig;       // Eq. 46
      real Ipi = I1 + P.delta_pipi * I2 - I3 + P.tau_pipi * I4 - P.lambda_piPi * Pi * K.sig[s];   // Eq. 42
      Jpi[s] = (real(2.0) * eotp * K.sig[s] - pi[s] * itp - Ipi - G[s]) * iut + pi[s] * divv;              // B.11, B.9
    }
  real IPi = P.delta_PiPi * Pi * K.theta - lPp * pisig;                                             // Eq. 41
  JPi = (-zotP * K.theta - Pi * itP - IPi) * iut + Pi * divv;                                         // B.10
}

// Regularisation factor tanh(rho)/rho (Eqs. 73-74, R9)
template <bool MILNE>
__device__ __forceinline__ real regulation_factor(const DevParams& P, const real q[NQ], real e, real p0, const real u[4], real t) {
  const real t2 = MILNE ? t * t : real(1.0);
  const real* pi = q + PTT;
  real Pi = q[BPI];
  real pipi = pi[0] * pi[0] - real(2.0) * (pi[1] * pi[1] + pi[2] * pi[2] + t2 * pi[3] * pi[3]) + pi[4] * pi[4] + real(2.0) * pi[5] * pi[5] +
                real(2.0) * t2 * pi[6] * pi[6] + pi[7] * pi[7] + real(2.0) * t2 * pi[8] * pi[8] + t2 * t2 * pi[9] * pi[9];
  real tr = pi[0] - pi[4] - pi[7] - t2 * pi[9];
  real PP = sqrt(fabs(pipi + real(3.0) * Pi * Pi));
  real rho = PP * P.inv_rho_max / sqrt(e * e + real(3.0) * p0 * p0);
  real den1 = P.xi0_rho_max * PP;
  if (PP > real(0.0) && isfinite(den1)) {
    real id = real(1.0) / den1;
    // pi^{l mu} u_mu, u_mu = (ut,-ux,-uy,-t2 un)
    real c0 = pi[0] * u[0] - pi[1] * u[1] - pi[2] * u[2] - t2 * pi[3] * u[3];
    real c1 = pi[1] * u[0] - pi[4] * u[1] - pi[5] * u[2] - t2 * pi[6] * u[3];
    real c2 = pi[2] * u[0] - pi[5] * u[1] - pi[7] * u[2] - t2 * pi[8] * u[3];
    real c3 = (pi[3] * u[0] - pi[6] * u[1] - pi[8] * u[2] - t2 * pi[9] * u[3]) * sqrt(t2);
    rho = fmax(rho, fabs(tr) * id);
    rho = fmax(rho, fabs(c0) * id);
    rho = fmax(rho, fabs(c1) * id);
    rho = fmax(rho, fabs(c2) * id);
    rho = fmax(rho, fabs(c3) * id);
  }
  if (!isfinite(rho)) rho = real(0.0);
  return (rho < real(1e-8)) ? real(1.0) : tanh(rho) / rho;
}

}  // namespace vh
