// vh_eos_lattice.hpp -- host-side builder of the EOS 2 table (product path; shares nothing with oracle/).
//
// PAPER.md section 2.3: trace anomaly I(T)/T^4 (Eq. 19, :206; exponent read as exp(-h1/t - h2/t^2), R19),
// P(T)/T^4 = int_0^T dT'/T' I/T'^4 (Eq. 20, :211), e = 3P + I, and "the inverse function T(e) and c_s^2" (:214) as the table of
// DESIGN.md R20: VH_EOS_N intervals uniform in x = e^{1/4} from T = 0.03 GeV to T = 2 GeV; node k holds (P, h dP/dx, T, h dT/dx).
// Quadrature here: 12-point Gauss-Legendre in ln T on panels of at most 0.1, carried from node to node; root of e(T) = e_k by a
// bracketed Newton iteration.  Natural units (T in fm^-1, e and P in fm^-4).
#pragma once
#include <cmath>
#include <vector>

namespace vh_eos {

constexpr int VH_EOS_N = 2048;
constexpr double kHbarc = 0.1973269804;      // GeV fm
constexpr double kSignH1 = -1.0;             // R19

struct Anomaly { double a, dadt; };           // I/T^4 and its derivative with respect to t = T/(0.2 GeV)

inline Anomaly anomaly(double t) {
  const double h0 = 0.1396, h1 = -0.1800, h2 = 0.0350, f0 = 2.76, f1 = 6.79, f2 = -5.29, g1 = -0.47, g2 = 1.04, al = 0.01;
  const double it = 1.0 / t, q = 1.0 + al * t * t, den = 1.0 + t * (g1 + g2 * t);
  const double th = std::tanh(f1 * t + f2);
  const double first = h0 / q, second = f0 * (1.0 + th) / den;
  const double dfirst = -first * (2.0 * al * t) / q;
  const double dsecond = (f0 * f1 * (1.0 - th * th) - second * (g1 + 2.0 * g2 * t)) / den;
  const double ex = std::exp(it * (kSignH1 * h1 - h2 * it));
  const double dlog = it * it * (-kSignH1 * h1 + 2.0 * h2 * it);      // d/dt of the exponent
  Anomaly r;
  r.a = (first + second) * ex;
  r.dadt = (dfirst + dsecond) * ex + r.a * dlog;
  return r;
}

struct LatticeTable {
  std::vector<double> node;      // 4 * (VH_EOS_N + 1): P, h dP/dx, T, h dT/dx
  double x0 = 0, xN = 0, h = 0;
};

class Builder {
 public:
  Builder() {
    // nodes and weights of the 12-point rule: roots of P_12 by Newton from the Chebyshev guess
    const int n = 12;
    gx_.resize(n); gw_.resize(n);
    for (int i = 0; i < n; ++i) {
      double z = std::cos(3.14159265358979323846 * (4.0 * i + 3.0) / (4.0 * n + 2.0));
      double d = 0.0;
      for (int it = 0; it < 50; ++it) {
        double pm = 1.0, pc = z;
        for (int k = 1; k < n; ++k) { const double pn = ((2.0 * k + 1.0) * z * pc - k * pm) / (k + 1.0); pm = pc; pc = pn; }
        d = n * (pm - z * pc) / (1.0 - z * z);
        const double step = pc / d;
        z -= step;
        if (std::fabs(step) < 1e-16) break;
      }
      gx_[i] = z; gw_[i] = 2.0 / ((1.0 - z * z) * d * d);
    }
  }
  // int_{Ta}^{Tb} (I/T^4) dT/T, T in fm^-1
  double integral(double Ta, double Tb) const {
    const double a = std::log(Ta), b = std::log(Tb), tc = 0.2 / kHbarc;
    const int panels = std::max(1, (int)std::ceil(std::fabs(b - a) / 0.1));
    const double w = (b - a) / panels;
    double acc = 0.0;
    for (int p = 0; p < panels; ++p) {
      const double mid = a + (p + 0.5) * w;
      double s = 0.0;
      for (size_t i = 0; i < gx_.size(); ++i) s += gw_[i] * anomaly(std::exp(mid + 0.5 * w * gx_[i]) / tc).a;
      acc += 0.5 * w * s;
    }
    return acc;
  }
  struct State { double e, P, s, dedT; };      // s = dP/dT (entropy density)
  static State state(double T, double F) {
    const double tc = 0.2 / kHbarc;
    const Anomaly A = anomaly(T / tc);
    const double T3 = T * T * T, T4 = T3 * T;
    State r;
    r.P = F * T4;
    r.e = T4 * (3.0 * F + A.a);
    r.s = T3 * (4.0 * F + A.a);
    r.dedT = 3.0 * r.s + 4.0 * T3 * A.a + T4 * A.dadt / tc;
    return r;
  }
  LatticeTable build() const {
    LatticeTable tab;
    tab.node.resize(4 * (VH_EOS_N + 1));
    const double Tlo = 0.03 / kHbarc, Thi = 2.0 / kHbarc, Tcut = 0.004 / kHbarc;
    const double Flo = integral(Tcut, Tlo), Fhi = Flo + integral(Tlo, Thi);
    tab.x0 = std::pow(state(Tlo, Flo).e, 0.25);
    tab.xN = std::pow(state(Thi, Fhi).e, 0.25);
    tab.h = (tab.xN - tab.x0) / VH_EOS_N;
    double Tref = Tlo, Fref = Flo;
    for (int k = 0; k <= VH_EOS_N; ++k) {
      const double x = tab.x0 + k * tab.h, target = x * x * x * x;
      double T = Tref, F = Fref;
      if (k == VH_EOS_N) { T = Thi; F = Fhi; }
      else if (k > 0) {
        double lo = Tref, hi = Thi;                     // e(T) is monotonic: bracket [previous node, top of the table]
        for (int it = 0; it < 80; ++it) {
          F = Fref + integral(Tref, T);
          const State st = state(T, F);
          if (st.e > target) hi = T; else lo = T;
          double Tn = T - (st.e - target) / st.dedT;
          if (!(Tn > lo && Tn < hi)) Tn = 0.5 * (lo + hi);
          const double change = std::fabs(Tn - T);
          T = Tn;
          if (change <= 1e-15 * T) break;
        }
        F = Fref + integral(Tref, T);
      }
      const State st = state(T, F);
      const double dedx = 4.0 * x * x * x;
      double* n4 = &tab.node[4 * k];
      n4[0] = st.P;
      n4[1] = tab.h * (st.s / st.dedT) * dedx;          // h dP/dx = h c_s^2 de/dx
      n4[2] = T;
      n4[3] = tab.h * dedx / st.dedT;                   // h dT/dx
      Tref = T; Fref = F;
    }
    return tab;
  }

 private:
  std::vector<double> gx_, gw_;
};

}  // namespace vh_eos
