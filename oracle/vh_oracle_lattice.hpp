// =====================================================================================
// vh_oracle_lattice.hpp -- TEST INFRASTRUCTURE ONLY (part of the CPU oracle, see vh_oracle.hpp).
// Equation of state "eos = 2": the lattice-QCD parametrisation of PAPER.md section 2.3.
//
//   I(T)/T^4 = [ h0/(1 + alpha t^2) + f0 (tanh(f1 t + f2) + 1)/(1 + g1 t + g2 t^2) ] exp(-h1/t - h2/t^2),  t = T/(0.2 GeV)   (Eq. 19, :206; sign: R19)
//   P(T)/T^4 = int_0^T dT'/T' I(T')/T'^4                                                                       (Eq. 20, :211)
//   e = 3 P + I;  "construct the inverse function T(e) and c_s^2 = dP/de" (:214)
//
// The paper does not say HOW the inverse is constructed.  Reading ("EOS 2"), identical on both sides but coded
// independently: a table with N = 2048 intervals, uniform in x = e^{1/4} between T = 0.03 GeV and T = 2 GeV, holding at every
// node the exact (quadrature + Newton) values of P, T and their x-derivatives; between nodes cubic Hermite interpolation in x
// for P and T, and c_s^2 = (dP/dx of the interpolant)/(4 x^3).  Below / above the table: P = P_0 e/e_0, T = T_0 x/x_0 and
// P = P_N + (e - e_N)/3, T = T_N x/x_N.  Natural units: T in fm^-1, e, P in fm^-4 (hbar c = 0.1973269804 GeV fm).
// Pins: tests/test_oracle_lattice.py (Eq. 20 re-evaluated with scipy.integrate.quad, thermodynamic identities, limits).
// =====================================================================================
#pragma once
#include <cmath>
#include <vector>

namespace vho {
namespace lattice {

constexpr double kHbarC = 0.1973269804;          // GeV fm
constexpr double kTc = 0.2 / kHbarC;             // the 0.2 GeV of Eq. 19, in fm^-1
constexpr double kTlo = 0.03 / kHbarC, kThi = 2.0 / kHbarC, kTcut = 0.004 / kHbarC;
constexpr int kN = 2048;
constexpr double kH1Sign = -1.0;                // sign of h1/t in the exponent of Eq. 19 (reading R19, see trace_anomaly)

// Eq. 19 and its t-derivative
inline void trace_anomaly(double t, double& A, double& dAdt) {
  const double h0 = 0.1396, h1 = -0.1800, h2 = 0.0350, f0 = 2.76, f1 = 6.79, f2 = -5.29, g1 = -0.47, g2 = 1.04, alpha = 0.01;
  const double B = h0 / (1.0 + alpha * t * t);
  const double dB = -2.0 * alpha * t * h0 / ((1.0 + alpha * t * t) * (1.0 + alpha * t * t));
  const double u = f1 * t + f2, th = std::tanh(u), D = 1.0 + g1 * t + g2 * t * t;
  const double C = f0 * (th + 1.0) / D;
  const double dC = f0 * (f1 * (1.0 - th * th) * D - (th + 1.0) * (g1 + 2.0 * g2 * t)) / (D * D);
  // exponent: reading R19 - PAPER.md :206 prints exp(h1/t - h2/t^2); with h1 = -0.18 that caps P/T^4 at 63 % of the
  // Stefan-Boltzmann value, against the paper's own statement (:216, footnote 2) that the pressure approaches that limit.  The
  // parametrisation it quotes (its Ref. [14]) has exp(-h1/t - h2/t^2): 87 % of SB at high T, e/T^4 = 12 at 400 MeV.  One constant.
  const double E = std::exp(kH1Sign * h1 / t - h2 / (t * t));
  const double dE = E * (-kH1Sign * h1 / (t * t) + 2.0 * h2 / (t * t * t));
  A = (B + C) * E;
  dAdt = (dB + dC) * E + (B + C) * dE;
}

// Gauss-Legendre nodes and weights on [-1, 1] (Newton iteration on the Legendre recurrence)
inline void gauss_legendre(int n, std::vector<double>& x, std::vector<double>& w) {
  x.assign(n, 0.0); w.assign(n, 0.0);
  const double pi = 3.14159265358979323846;
  for (int i = 0; i < n; ++i) {
    double z = std::cos(pi * (i + 0.75) / (n + 0.5)), dp = 1.0;
    for (int it = 0; it < 100; ++it) {
      double p0 = 1.0, p1 = z;
      for (int k = 2; k <= n; ++k) { const double p2 = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k; p0 = p1; p1 = p2; }
      dp = n * (z * p1 - p0) / (z * z - 1.0);
      const double dz = p1 / dp;
      z -= dz;
      if (std::fabs(dz) < 1e-16) break;
    }
    x[i] = z; w[i] = 2.0 / ((1.0 - z * z) * dp * dp);
  }
}

struct Table {
  double x0 = 0, h = 0;
  std::vector<double> p, dpdx, T, dTdx;      // kN + 1 nodes
  std::vector<double> glx, glw;

  // int_{Ta}^{Tb} dT/T I/T^4 = int A(e^s) ds, s = ln T: 16-point Gauss-Legendre on panels no wider than 0.05 in s
  double F_between(double Ta, double Tb) const {
    const double sa = std::log(Ta), sb = std::log(Tb);
    const int m = (int)std::ceil(std::fabs(sb - sa) / 0.05);
    if (m == 0) return 0.0;
    const double ds = (sb - sa) / m;
    double sum = 0.0;
    for (int j = 0; j < m; ++j) {
      const double c = sa + (j + 0.5) * ds;
      for (size_t i = 0; i < glx.size(); ++i) {
        double A, dA;
        trace_anomaly(std::exp(c + 0.5 * ds * glx[i]) / kTc, A, dA);
        sum += 0.5 * ds * glw[i] * A;
      }
    }
    return sum;
  }
  // thermodynamics at temperature T given F = P/T^4
  static void thermo(double T, double F, double& e, double& P, double& dPdT, double& dedT) {
    double A, dA;
    trace_anomaly(T / kTc, A, dA);
    const double T4 = T * T * T * T;
    P = T4 * F;
    const double I = T4 * A;
    e = 3.0 * P + I;
    dPdT = (4.0 * P + I) / T;                           // entropy density
    dedT = 3.0 * dPdT + 4.0 * I / T + T4 * dA / kTc;
  }
  void build() {
    gauss_legendre(16, glx, glw);
    p.assign(kN + 1, 0.0); dpdx = p; T = p; dTdx = p;
    const double F0 = F_between(kTcut, kTlo);
    const double FN = F0 + F_between(kTlo, kThi);
    double e, P, dP, de;
    thermo(kTlo, F0, e, P, dP, de);
    x0 = std::sqrt(std::sqrt(e));
    double eN, PN, dPN, deN;
    thermo(kThi, FN, eN, PN, dPN, deN);
    h = (std::sqrt(std::sqrt(eN)) - x0) / kN;
    double Tprev = kTlo, Fprev = F0;
    for (int k = 0; k <= kN; ++k) {
      const double x = x0 + k * h, ek = x * x * x * x;
      double Tk = Tprev, Fk = Fprev;
      if (k == kN) { Tk = kThi; Fk = FN; thermo(Tk, Fk, e, P, dP, de); }
      else {
        for (int it = 0; it < 60; ++it) {                 // Newton on e(T) = e_k, F carried from the previous node
          Fk = Fprev + F_between(Tprev, Tk);
          thermo(Tk, Fk, e, P, dP, de);
          const double dT = (e - ek) / de;
          Tk -= dT;
          if (std::fabs(dT) <= 1e-15 * Tk) break;
        }
        Fk = Fprev + F_between(Tprev, Tk);
        thermo(Tk, Fk, e, P, dP, de);
      }
      const double dedx = 4.0 * x * x * x;
      p[k] = P; dpdx[k] = (dP / de) * dedx; T[k] = Tk; dTdx[k] = dedx / de;
      Tprev = Tk; Fprev = Fk;
    }
  }
  void eval(double e, double& P, double& cs2, double& Tout) const {
    const double x = std::sqrt(std::sqrt(e));
    const double xN = x0 + kN * h;
    if (!(x >= x0)) {                                     // below the table (also e <= 0, NaN)
      const double e0 = x0 * x0 * x0 * x0;
      P = p[0] * (e / e0); cs2 = p[0] / e0; Tout = T[0] * (x / x0);
      return;
    }
    if (x >= xN) {
      const double eN = xN * xN * xN * xN;
      P = p[kN] + (e - eN) / 3.0; cs2 = 1.0 / 3.0; Tout = T[kN] * (x / xN);
      return;
    }
    int k = (int)((x - x0) / h);
    if (k > kN - 1) k = kN - 1;
    const double s = (x - (x0 + k * h)) / h, s2 = s * s, s3 = s2 * s;
    const double h00 = 2 * s3 - 3 * s2 + 1, h10 = s3 - 2 * s2 + s, h01 = -2 * s3 + 3 * s2, h11 = s3 - s2;
    const double d00 = 6 * s2 - 6 * s, d10 = 3 * s2 - 4 * s + 1, d01 = -6 * s2 + 6 * s, d11 = 3 * s2 - 2 * s;
    P = h00 * p[k] + h10 * h * dpdx[k] + h01 * p[k + 1] + h11 * h * dpdx[k + 1];
    const double dPdx = (d00 * p[k] + d01 * p[k + 1]) / h + d10 * dpdx[k] + d11 * dpdx[k + 1];
    cs2 = dPdx / (4.0 * x * x * x);
    Tout = h00 * T[k] + h10 * h * dTdx[k] + h01 * T[k + 1] + h11 * h * dTdx[k + 1];
  }
};

inline const Table& table() {
  static const Table t = [] { Table x; x.build(); return x; }();
  return t;
}

}  // namespace lattice
}  // namespace vho
