// vh_device.cuh -- device-side arithmetic of the KT / Heun step (product path; shares nothing with oracle/).
// Citations are PAPER.md lines / equations.  Component forms (App. A, A.12, A.14-A.19, B.12) are used here; the
// test oracle uses index forms.  Readings R1..R18 are listed in DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

namespace vh {

constexpr int NQ = 15;
// q slots
enum { TTT = 0, TTX, TTY, TTN, PTT, PTX, PTY, PTN, PXX, PXY, PXN, PYY, PYN, PNN, BPI };

constexpr double kVorticitySign = -1.0;   // R4: Eq. 8 (:149) with omega^{mu nu} of :122

struct DevParams {
  int nx, ny, nz, n_batch;
  int NXp, NYp, NZp;            // padded extents (NXp is the row pitch, multiple of 16 doubles = 128 B)
  long long plane;              // NXp*NYp
  long long bstride;            // NXp*NYp*NZp   (one event)
  long long fstride;            // bstride*n_batch (one field)
  int zoff;                     // 2 (3+1d) or 0 (2+1d: no eta ghost planes are stored)
  double dx, dy, dz, dtau;
  double inv_dx, inv_dy, inv_dz, inv_dtau;
  int shear, bulk;              // physics bits
  double eos_a_inv, eos_alpha, eos_e0_inv;
  // EOS 2 (lattice, Eqs. 19-20; R19, R20): table of kN + 1 nodes uniform in x = e^{1/4}, node k = (P, h dP/dx, T, h dT/dx)
  const double2* eos_tab; int eos_n; double eos_x0, eos_xN, eos_inv_h, eos_lo_slope, eos_pN, eos_eN, eos_T0_over_x0, eos_TN_over_xN;
  double inv_ctaupi_etas;       // 1/(c_tau_pi * eta/s)
  double inv_ctaupi;            // 1/c_tau_pi
  int zeta_model; double zeta_amp, zeta_T0, zeta_inv_width, inv_ctauPi;
  double delta_pipi, tau_pipi, lambda_piPi, delta_PiPi, lambda_Pipi_coef;
  double theta;                 // minmod theta
  double inv_rho_max, xi0_rho_max;
  int newton_max_iter; double newton_rtol;
  double relax_clamp;           // 1/(c*dtau) or +inf
};

// ---------------------------------------------------------------- branch-free reciprocal / square roots on the MUFU seeds
// 1/x to ~1 ulp: MUFU.RCP64H seed (~20 bits) + two Newton steps.  No denormal / overflow slow path: callers pass
// well-scaled positive quantities; inf/NaN/0 propagate as NaN/inf and are caught by the callers' finiteness checks.
__device__ __forceinline__ double rcp_fast(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double t = fma(-x, y, 1.0);
  y = fma(y, t, y);
  t = fma(-x, y, 1.0);
  return fma(y, t, y);
}
// one Newton step only (~40 bits): enough wherever the quotient only steers an iteration
__device__ __forceinline__ double rcp_half(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double t = fma(-x, y, 1.0);
  return fma(y, t, y);
}
// 1/sqrt(x) to ~1 ulp: MUFU.RSQ64H seed + two Newton steps
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double hx = 0.5 * x;
  double t = fma(-hx * y, y, 0.5);
  y = fma(y, t, y);
  t = fma(-hx * y, y, 0.5);
  return fma(y, t, y);
}
// sqrt(x) for x > 0 (x = 0 gives 0): x * rsqrt(x) with one correction step
__device__ __forceinline__ double sqrt_fast(double x) {
  double r = rsqrt_fast(x);
  double s = x * r;
  double d = fma(-s, s, x);
  s = fma(0.5 * r, d, s);
  return (x > 0.0) ? s : 0.0;
}

// ---------------------------------------------------------------- exp(-x) for the EOS and zeta/s(T)
// exp(-x) with the argument clamped to [-700, 700] (beyond: 1e304 / 1e-304 instead of inf / 0, never reached by a state
// that passes the finiteness checks).  -x = k ln2 + r, |r| <= ln2/2, Taylor polynomial of degree 13 (truncation 4e-18), 2^k
// added into the exponent field.  The coefficients sit in constant memory so that each Horner step is ONE DFMA with a
// constant-bank operand; the library exp() materialises its 64-bit immediates with two moves per coefficient, which made
// half of its instructions moves (profiles/r01b_ncu_summary.md).  About 1 ulp, like the library routine.
static __constant__ double kExpTaylor[14] = {1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320, 1.0 / 362880,
                                             1.0 / 3628800, 1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0};
static __constant__ double kExpRed[4] = {1.4426950408889634, 6755399441055744.0, 6.93147180369123816490e-01, 1.90821492927058770002e-10};
__device__ __forceinline__ double exp_neg(double x) {
  x = (fabs(x) < 700.0) ? x : copysign(700.0, x);      // one compare and a select (fmin/fmax with their NaN rules cost four times that); NaN -> 700
  const double t = fma(-x, kExpRed[0], kExpRed[1]);      // 1.5 * 2^52 + rint(-x log2 e): the integer sits in the low word
  const int k = __double2loint(t);
  const double kd = t - kExpRed[1];
  double r = fma(-kd, kExpRed[2], -x);
  r = fma(-kd, kExpRed[3], r);
  double p = kExpTaylor[13];
#pragma unroll
  for (int i = 12; i >= 0; --i) p = fma(p, r, kExpTaylor[i]);
  return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}

// ---------------------------------------------------------------- EOS (BASELINE.json configs) and transport (Eqs. 10-16)
template <int EOS> __device__ __forceinline__ void eos_p_cs2(const DevParams& P, double e, double& p, double& cs2) {
  if (EOS == 0) {
    p = e * (1.0 / 3.0);
    cs2 = 1.0 / 3.0;
  } else {
    double x = e * P.eos_e0_inv;
    double aex = P.eos_alpha * exp_neg(x);
    p = (e * (1.0 / 3.0)) * (1.0 - aex);
    cs2 = (1.0 / 3.0) * (1.0 - aex * (1.0 - x));
  }
}
// EOS 2: cubic Hermite interpolation in x = e^{1/4} of the tabulated lattice pressure and temperature (R20); c_s^2 is the
// derivative of the pressure interpolant.  Below the table P = (P_0/e_0) e, T = (T_0/x_0) x; above it P = P_N + (e - e_N)/3.
__device__ __forceinline__ void eos_lattice(const DevParams& P, double e, double& p, double& cs2, double& T) {
  // x = e^{1/4} as rsqrt(rsqrt(e)), y = e^{-1/2}: two MUFU seeds with two Newton steps each, no IEEE square-root slow path, and
  // 1/x^3 = x y^2 comes for free (e <= 0 or NaN falls into the first branch below)
  const double y = rsqrt_fast(e);
  const double x = (e > 0.0) ? rsqrt_fast(y) : 0.0;
  if (!(x >= P.eos_x0)) { p = P.eos_lo_slope * e; cs2 = P.eos_lo_slope; T = P.eos_T0_over_x0 * x; return; }
  if (x >= P.eos_xN) { p = fma(e - P.eos_eN, 1.0 / 3.0, P.eos_pN); cs2 = 1.0 / 3.0; T = P.eos_TN_over_xN * x; return; }
  const double u = (x - P.eos_x0) * P.eos_inv_h;
  const int k = min((int)u, P.eos_n - 1);
  const double s = u - (double)k, s2 = s * s, s3 = s2 * s;
  const double2 ap = __ldg(P.eos_tab + 2 * k), at = __ldg(P.eos_tab + 2 * k + 1), bp = __ldg(P.eos_tab + 2 * k + 2), bt = __ldg(P.eos_tab + 2 * k + 3);
  const double h00 = 2.0 * s3 - 3.0 * s2 + 1.0, h10 = s3 - 2.0 * s2 + s, h01 = 3.0 * s2 - 2.0 * s3, h11 = s3 - s2;
  p = h00 * ap.x + h10 * ap.y + h01 * bp.x + h11 * bp.y;
  T = h00 * at.x + h10 * at.y + h01 * bt.x + h11 * bt.y;
  const double d00 = 6.0 * (s2 - s), d10 = 3.0 * s2 - 4.0 * s + 1.0, d11 = 3.0 * s2 - 2.0 * s;
  const double dpdx = (d00 * (ap.x - bp.x) + d10 * ap.y + d11 * bp.y) * P.eos_inv_h;
  cs2 = dpdx * (0.25 * x) * (y * y);
}
template <> __device__ __forceinline__ void eos_p_cs2<2>(const DevParams& P, double e, double& p, double& cs2) {
  double T;
  eos_lattice(P, e, p, cs2, T);
}
// temperature for the transport coefficients: T = (e/a)^{1/4} for the analytic EOS, T(e) of the table for EOS 2
template <int EOS> __device__ __forceinline__ double eos_temperature(const DevParams& P, double e) {
  if (EOS == 2) { double p, c, T; eos_lattice(P, e, p, c, T); return T; }
  const double y = e * P.eos_a_inv;
  return sqrt(sqrt(y));
}
template <int EOS> __device__ __forceinline__ double eos_p(const DevParams& P, double e) {
  double p, c;
  eos_p_cs2<EOS>(P, e, p, c);
  return p;
}

// ---------------------------------------------------------------- zeta/s(T)
// zeta_model 0: none; 1: Gaussian amp exp(-((T - T0)/width)^2) (BASELINE.json configs 3-5); 2: constant amp;
// 3: the paper's parametrisation, Eq. 17 (:174-186), times (zeta/s)_norm = zeta_amp, with T_c = zeta_T0 and the ranges read as
//    T < 0.995 T_c, 0.995 T_c <= T <= 1.05 T_c, T > 1.05 T_c (the printed inequalities are reversed, reading R3).
__device__ __forceinline__ double zeta_over_s(const DevParams& P, double T) {
  if (P.zeta_model == 1) { const double d = (T - P.zeta_T0) * P.zeta_inv_width; return P.zeta_amp * exp_neg(d * d); }
  if (P.zeta_model == 2) return P.zeta_amp;
  if (P.zeta_model == 3) {
    const double x = T * P.zeta_inv_width;      // T / T_c (zeta_inv_width holds 1/T_c for this model)
    double z;
    if (x > 1.05) z = 0.9 * exp_neg((x - 1.0) * (1.0 / 0.025)) + 0.25 * exp_neg((x - 1.0) * (1.0 / 0.13)) + 0.001;
    else if (x < 0.995) z = 0.9 * exp_neg((1.0 - x) * (1.0 / 0.0025)) + 0.22 * exp_neg((1.0 - x) * (1.0 / 0.022)) + 0.03;
    else z = -13.45 + x * (27.55 - 13.77 * x);
    return P.zeta_amp * z;
  }
  return 0.0;
}

// ---------------------------------------------------------------- Newton-Raphson on Eq. 72 (R6)
// returns e; fail is set when no acceptable root was found (then e = max(E, tiny)).
template <int EOS> __device__ __forceinline__ double invert_energy(const DevParams& P, double E, double M2, double Pi, double guess, bool& fail) {
  bool bad = !(E > 0.0) || !isfinite(E) || !isfinite(M2) || !isfinite(Pi);
  double e = (guess > 0.0 && isfinite(guess)) ? guess : E;
  bool done = bad, conv = false;
  for (int it = 0; it < P.newton_max_iter; ++it) {
    if (__all_sync(0xffffffffu, done)) break;     // warp-level convergence vote; every caller is warp-converged
    if (!done) {
      double p, cs2;
      eos_p_cs2<EOS>(P, e, p, cs2);
      double den = E + p + Pi;
      double rden = 1.0 / den;
      double f = e - E + M2 * rden;
      double fp = 1.0 - M2 * cs2 * rden * rden;
      double de = f / fp;
      e = e - de;
      if (fabs(de) <= P.newton_rtol * fabs(e)) { conv = true; done = true; }
    }
  }
  fail = bad || !conv || !(e > 0.0) || !isfinite(e);
  if (fail) e = (1e-300 > E) ? 1e-300 : E;      // max(E, tiny) that keeps a NaN E visible to n_nonfinite
  return e;
}

// minmod limited half-slope:  (dr/2) * minmod(theta (q0-qm)/dr, (qp-qm)/(2 dr), theta (qp-q0)/dr)   (Eqs. 67-68, R10)
__device__ __forceinline__ double half_slope(double qm, double q0, double qp, double theta) {
  double a = theta * (q0 - qm), b = 0.5 * (qp - qm), c = theta * (qp - q0);
  double m = fmin(fmin(fabs(a), fabs(b)), fabs(c));
  bool pos = (a > 0.0) && (b > 0.0) && (c > 0.0);
  bool neg = (a < 0.0) && (b < 0.0) && (c < 0.0);
  double s = pos ? m : (neg ? -m : 0.0);
  return 0.5 * s;
}

// velocity v_r of a reconstructed state along direction r (Alg. 3 :667-672, :424): v^i = M_i/(E + P0(e) + Pi)
template <int EOS, bool MILNE>
__device__ __forceinline__ double state_velocity(const DevParams& P, double E, double Mx, double My, double Mn, double Pi, double t2,
                                                 double guess, int r, bool count, unsigned long long& nfail) {
  double M2 = Mx * Mx + My * My + (MILNE ? t2 : 1.0) * Mn * Mn;     // :339
  bool fail;
  double e = invert_energy<EOS>(P, E, M2, Pi, guess, fail);
  double p = eos_p<EOS>(P, e);
  double Mr = (r == 0) ? Mx : ((r == 1) ? My : Mn);
  double v = Mr / (E + p + Pi);
  if (fail) {
    if (count) ++nfail;
    if (!(fabs(v) < 1.0)) v = (v > 0.0) ? 1.0 - 1e-12 : ((v < 0.0) ? -1.0 + 1e-12 : 0.0);
  }
  return v;
}

struct Kin {            // kinematic scalars / tensors at a cell (App. A)
  double theta;
  double Du[4];         // covariant Du_lambda (A.9-A.10)
  double sig[10];       // sigma^{mu nu} in the order tt tx ty tn xx xy xn yy yn nn (A.12)
  double W[6];          // W^{tx} W^{ty} W^{tn} W^{xy} W^{xn} W^{yn} (A.14-A.19)
};

// u = (ut,ux,uy,un); dt,dx,dy,dn = partial derivatives of the four components (:424).
// MILNE = false is the Cartesian mode (R12): metric factors tau^2 -> 1 (t2, g2i) and every Christoffel symbol -> 0 (ch = Gamma^eta_{eta tau}
// = 1/tau, ct = Gamma^tau_{eta eta} = tau), kept apart so that each falls out at compile time.
template <bool MILNE>
__device__ __forceinline__ void kinematics(const double u[4], const double dt[4], const double dx[4], const double dy[4], const double dn[4],
                                           double t, Kin& K) {
  const double ut = u[0], ux = u[1], uy = u[2], un = u[3];
  const double t2 = MILNE ? t * t : 1.0, g2i = MILNE ? 1.0 / (t * t) : 1.0;
  const double ch = MILNE ? 1.0 / t : 0.0, ct = MILNE ? t : 0.0;
  // convective derivatives (A.5-A.8)
  double dut = ut * dt[0] + ux * dx[0] + uy * dy[0] + un * dn[0];
  double dux = ut * dt[1] + ux * dx[1] + uy * dy[1] + un * dn[1];
  double duy = ut * dt[2] + ux * dx[2] + uy * dy[2] + un * dn[2];
  double dun = ut * dt[3] + ux * dx[3] + uy * dy[3] + un * dn[3];
  double th = ut * ch + dt[0] + dx[1] + dy[2] + dn[3];                 // A.11
  double th3 = th * (1.0 / 3.0);
  K.theta = th;
  K.Du[0] = dut + ct * un * un;                                         // A.9
  K.Du[1] = -dux;
  K.Du[2] = -duy;
  K.Du[3] = -t2 * (dun + 2.0 * ch * ut * un);                           // A.10
  double un2 = un * un;
  // A.12 (D(.) read as the convective derivative of the contravariant component, reading in DESIGN.md)
  K.sig[0] = -ct * ut * un2 + dt[0] - ut * dut + (ut * ut - 1.0) * th3;
  K.sig[1] = -0.5 * ct * un2 * ux + 0.5 * (dt[1] - dx[0]) - 0.5 * (ut * dux + ux * dut) + ut * ux * th3;
  K.sig[2] = -0.5 * ct * un2 * uy + 0.5 * (dt[2] - dy[0]) - 0.5 * (ut * duy + uy * dut) + ut * uy * th3;
  K.sig[3] = -0.5 * un * (2.0 * ch * ut * ut + ct * un2) + 0.5 * (dt[3] - dn[0] * g2i) - 0.5 * (ut * dun + un * dut) + ut * un * th3;
  K.sig[4] = -dx[1] - ux * dux + (1.0 + ux * ux) * th3;
  K.sig[5] = -0.5 * (dx[2] + dy[1]) - 0.5 * (ux * duy + uy * dux) + ux * uy * th3;
  K.sig[6] = -ut * ux * un * ch - 0.5 * (dx[3] + dn[1] * g2i) - 0.5 * (ux * dun + un * dux) + ux * un * th3;
  K.sig[7] = -dy[2] - uy * duy + (1.0 + uy * uy) * th3;
  K.sig[8] = -ut * uy * un * ch - 0.5 * (dy[3] + dn[2] * g2i) - 0.5 * (uy * dun + un * duy) + uy * un * th3;
  K.sig[9] = -ut * g2i * ch * (1.0 + 2.0 * un2 * t2) - dn[3] * g2i - un * dun + (g2i + un2) * th3;
  // A.14-A.19 divided by the metric factors so that W^{mu nu} is the contravariant antisymmetric tensor of :122
  K.W[0] = 0.5 * (dt[1] + dx[0]) + 0.5 * (ux * dut - ut * dux) + 0.5 * ct * un2 * ux;
  K.W[1] = 0.5 * (dt[2] + dy[0]) + 0.5 * (uy * dut - ut * duy) + 0.5 * ct * un2 * uy;
  K.W[2] = un * ch + 0.5 * dt[3] + 0.5 * dn[0] * g2i + 0.5 * (un * dut - ut * dun) - ut * ut * un * ch + 0.5 * ct * un2 * un;
  K.W[3] = 0.5 * (dy[1] - dx[2]) + 0.5 * (uy * dux - ux * duy);
  K.W[4] = 0.5 * dn[1] * g2i - 0.5 * dx[3] + 0.5 * (un * dux - ux * dun) - ux * ut * un * ch;
  K.W[5] = 0.5 * dn[2] * g2i - 0.5 * dy[3] + 0.5 * (un * duy - uy * dun) - uy * ut * un * ch;
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
__device__ __forceinline__ void dissipative_sources(const DevParams& P, double t, const double u[4], const Kin& K, const double pi[10], double Pi,
                                                    double e, double p, double cs2, double divv, double Jpi[10], double& JPi) {
  const double t2 = MILNE ? t * t : 1.0, g2i = MILNE ? 1.0 / (t * t) : 1.0;      // metric factors
  const double it = MILNE ? 1.0 / t : 0.0, ct = MILNE ? t : 0.0;                  // Christoffel symbols (0 in the Cartesian mode, R12)
  const double g[4] = {1.0, -1.0, -1.0, -t2};
  // transport coefficients (Eqs. 10-16; R14)
  double T = eos_temperature<EOS>(P, e);
  double itp = fmin(T * P.inv_ctaupi_etas, P.relax_clamp);
  double eotp = (e + p) * P.inv_ctaupi;
  const double zs = zeta_over_s(P, T);
  double b = (1.0 / 3.0) - cs2;
  double itP = (zs > 0.0) ? T * b * b * P.inv_ctauPi / zs : CUDART_INF;
  itP = fmin(itP, P.relax_clamp);
  double zotP = (zs > 0.0) ? zs * ((e + p) / T) * itP : 0.0;
  double lPp = P.lambda_Pipi_coef * b;

  // full symmetric / antisymmetric tables
  double S[4][4], W[4][4], Pm[4][4];
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = 0; n < 4; ++n) { S[m][n] = K.sig[sym(m, n)]; Pm[m][n] = pi[sym(m, n)]; }
  W[0][0] = W[1][1] = W[2][2] = W[3][3] = 0.0;
  W[0][1] = K.W[0]; W[0][2] = K.W[1]; W[0][3] = K.W[2]; W[1][2] = K.W[3]; W[1][3] = K.W[4]; W[2][3] = K.W[5];
  W[1][0] = -K.W[0]; W[2][0] = -K.W[1]; W[3][0] = -K.W[2]; W[2][1] = -K.W[3]; W[3][1] = -K.W[4]; W[3][2] = -K.W[5];

  // A^mu = pi^{lambda mu} Du_lambda ;  B^{mu nu} = pi^{mu l} g_l W^{l nu} ;  C^{mu nu} = g_l pi^{mu l} sigma^{nu l}
  double A[4], B[4][4], C[4][4];
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    A[m] = Pm[0][m] * K.Du[0] + Pm[1][m] * K.Du[1] + Pm[2][m] * K.Du[2] + Pm[3][m] * K.Du[3];
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      double bb = 0.0, cc = 0.0;
#pragma unroll
      for (int l = 0; l < 4; ++l) { bb += Pm[m][l] * g[l] * W[l][n]; cc += g[l] * Pm[m][l] * S[n][l]; }
      B[m][n] = bb; C[m][n] = cc;
    }
  }
  double pisig = g[0] * C[0][0] + g[1] * C[1][1] + g[2] * C[2][2] + g[3] * C[3][3];      // pi^{mu nu} sigma_{mu nu}
  const double gi[4] = {1.0, -1.0, -1.0, -g2i};
  const double iut = 1.0 / u[0];
  // G_pi = u^a Gamma^mu_{ab} pi^{b nu} + (mu<->nu)  (:300; R1, R2)
  double G[10];
  const double ut = u[0], un = u[3];
  G[0] = 2.0 * ct * un * pi[3];
  G[1] = ct * un * pi[6];
  G[2] = ct * un * pi[8];
  G[3] = ct * un * pi[9] + (ut * pi[3] + un * pi[0]) * it;
  G[4] = 0.0; G[5] = 0.0;
  G[6] = (ut * pi[6] + un * pi[1]) * it;
  G[7] = 0.0;
  G[8] = (ut * pi[8] + un * pi[2]) * it;
  G[9] = 2.0 * (ut * pi[9] + un * pi[3]) * it;
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = m; n < 4; ++n) {
      const int s = sym(m, n);
      double Dmn = ((m == n) ? gi[m] : 0.0) - u[m] * u[n];
      double I1 = u[n] * A[m] + u[m] * A[n];                                   // Eq. 43
      double I2 = K.theta * pi[s];                                             // Eq. 44
      double I3 = kVorticitySign * (B[m][n] + B[n][m]);                        // Eq. 45 (R4)
      double I4 = 0.5 * (C[m][n] + C[n][m]) - (1.0 / 3.0) * Dmn * pisig;       // Eq. 46
      double Ipi = I1 + P.delta_pipi * I2 - I3 + P.tau_pipi * I4 - P.lambda_piPi * Pi * K.sig[s];   // Eq. 42
      Jpi[s] = (2.0 * eotp * K.sig[s] - pi[s] * itp - Ipi - G[s]) * iut + pi[s] * divv;              // B.11, B.9
    }
  double IPi = P.delta_PiPi * Pi * K.theta - lPp * pisig;                                             // Eq. 41
  JPi = (-zotP * K.theta - Pi * itP - IPi) * iut + Pi * divv;                                         // B.10
}

// Regularisation factor tanh(rho)/rho (Eqs. 73-74, R9)
template <bool MILNE>
__device__ __forceinline__ double regulation_factor(const DevParams& P, const double q[NQ], double e, double p0, const double u[4], double t) {
  const double t2 = MILNE ? t * t : 1.0;
  const double* pi = q + PTT;
  double Pi = q[BPI];
  double pipi = pi[0] * pi[0] - 2.0 * (pi[1] * pi[1] + pi[2] * pi[2] + t2 * pi[3] * pi[3]) + pi[4] * pi[4] + 2.0 * pi[5] * pi[5] +
                2.0 * t2 * pi[6] * pi[6] + pi[7] * pi[7] + 2.0 * t2 * pi[8] * pi[8] + t2 * t2 * pi[9] * pi[9];
  double tr = pi[0] - pi[4] - pi[7] - t2 * pi[9];
  double PP = sqrt(fabs(pipi + 3.0 * Pi * Pi));
  double rho = PP * P.inv_rho_max / sqrt(e * e + 3.0 * p0 * p0);
  double den1 = P.xi0_rho_max * PP;
  if (PP > 0.0 && isfinite(den1)) {
    double id = 1.0 / den1;
    // pi^{l mu} u_mu, u_mu = (ut,-ux,-uy,-t2 un)
    double c0 = pi[0] * u[0] - pi[1] * u[1] - pi[2] * u[2] - t2 * pi[3] * u[3];
    double c1 = pi[1] * u[0] - pi[4] * u[1] - pi[5] * u[2] - t2 * pi[6] * u[3];
    double c2 = pi[2] * u[0] - pi[5] * u[1] - pi[7] * u[2] - t2 * pi[8] * u[3];
    double c3 = (pi[3] * u[0] - pi[6] * u[1] - pi[8] * u[2] - t2 * pi[9] * u[3]) * sqrt(t2);
    rho = fmax(rho, fabs(tr) * id);
    rho = fmax(rho, fabs(c0) * id);
    rho = fmax(rho, fabs(c1) * id);
    rho = fmax(rho, fabs(c2) * id);
    rho = fmax(rho, fabs(c3) * id);
  }
  if (!isfinite(rho)) rho = 0.0;
  return (rho < 1e-8) ? 1.0 : tanh(rho) / rho;
}

}  // namespace vh
