// =====================================================================================
// vh_oracle.hpp -- TEST INFRASTRUCTURE ONLY.  Plain, slow, serial CPU oracle (FP64) for
// one Heun/RK2 Kurganov-Tadmor step of 3+1d second-order viscous hydrodynamics in Milne
// coordinates, written from /root/reference/PAPER.md (arXiv 1608.06577).
//
//   * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
//     legs may build, link or call anything in oracle/.  The product (CUDA) path never
//     does, shares no code with this file and does not import it.
//   * It follows the paper's algorithm in the paper's order: Euler step (Eq. 59, :375),
//     inversion (Eqs. 52-54, 72), regularisation (Eqs. 73-74), ghost cells (Eqs. 75-76),
//     two-stage RK program flow steps 1-9 (:503-529).  Tensor algebra is in 4x4 INDEX
//     form (Eqs. 39-46, A.3, :122) - deliberately not the unrolled component lists.
//   * Readings of silent / garbled passages are listed in DESIGN.md ("Readings"), and
//     are referred to below as R1..R18 (numbering of SURVEY.md section 8(c)).
//   * Parity status: every function is pinned by tests/test_oracle_*.py (Riemann solution, Bjorken ODEs, ideal and
//     viscous Gubser flow, boosted-static exact solution, a generic covariant evaluation of Eq. 8, closed-form
//     inversion, invariants).  The vorticity sign (R4) is pinned to the governing equation, Eq. 8, by
//     tests/test_oracle_covariant.py (the appendix list A.25-A.29 has the opposite sign).  The regularisation
//     (Eqs. 73-74, reading R9) and the order invert -> regulate (R8) are pinned by tests/test_oracle_regulation.py: every entry of the
//     max of Eq. 74 for a moving fluid at tau != 1 from states built out of Lorentz-invariant pieces, the equilibrium pressure in the
//     first entry, and e, u returned from the un-regulated state; the rest-frame values by tests/test_oracle_units.py.  Applied literally it makes
//     the discrete Gubser run ill-conditioned ("config 2").  The lattice EOS (eos = 2, vh_oracle_lattice.hpp,
//     readings R19, R20) is pinned by tests/test_oracle_lattice.py, zeta/s of Eq. 17, diagnostics() (incl. Eq. 90, reading R21, also tests/test_oracle_covariant.py) and regulation_map() by tests/test_oracle_units.py.  The viscous Cartesian mode (geometry = 1 with physics != 0) is pinned by the damped
//     sound wave of the linearised equations, the 2+1d diagonal shock tube and the cylindrical blast (tests/test_oracle_cartesian.py).  No function is "parity unpinned".
//     Solver<float> (vho_create_f32) is the same code with a float scalar: comparator of the single-precision build, pinned against Solver<double> (tests/test_f32.py).
//
// The scalar type is a template parameter so that an operation-counting type can be
// substituted (oracle/vh_oracle_capi.cpp instantiates double and a counting type).
// =====================================================================================
#pragma once
#ifndef VHO_COUNTING_SECTION
#define VHO_COUNTING_SECTION(x) ((void)0)     // used only by vh_oracle_count.cpp (operation counting)
#endif
#include <cmath>
#include <cstddef>
#include <limits>
#include <vector>

#include "vh_oracle_lattice.hpp"

namespace vho {

using std::exp; using std::pow; using std::sqrt; using std::tanh;

// Sign s_omega of the vorticity coupling, R4: I_3^{mu nu} = s_omega (pi^{mu l} g_{lk} W^{k nu} + (mu<->nu)),
// W^{mu nu} = (1/2)(nabla^mu u^nu - nabla^nu u^mu) (:122).  -1 reproduces Eq. 8 (:149).
constexpr int kVorticitySign = -1;

struct Params {
  int nx, ny, nz, n_batch;     // physical cells; nz==1 -> 2+1d; n_batch independent events
  double dx, dy, dz;           // fm, fm, rapidity
  double tau0, dtau;           // fm
  int geometry;                // 0 Milne, 1 Cartesian (R12: the paper uses it for its ideal tests; the viscous terms work too, pinned by tests/test_oracle_cartesian.py)
  int physics;                 // bit0 shear, bit1 bulk; 0 ideal
  int eos;                     // 0: p=e/3; 1: p=(e/3)(1-alpha*exp(-e/e0)), T=(e/a)^(1/4) for both; 2: lattice EOS (Eqs. 19-20), T(e) from its table
  double eos_a, eos_alpha, eos_e0;
  double eta_over_s;
  int zeta_model;              // 0: zeta/s=0; 1: Gaussian amp*exp(-((T-T0)/width)^2); 2: constant amp; 3: Eq. 17 x amp, T_c = T0
  double zeta_amp, zeta_T0, zeta_width;     // T0, width in fm^-1 (R13)
  double c_tau_pi;             // tau_pi = c_tau_pi*eta/(e+p)                 (Eq. 13 -> 5)
  double c_tau_Pi;             // tau_Pi = c_tau_Pi*zeta/((e+p)(1/3-cs2)^2)   (configs 5; Eq. 10 -> 1/15)
  double delta_pipi, tau_pipi, lambda_piPi;   // in units of tau_pi: 4/3, 10/7, 6/5 (Eqs. 14-16)
  double delta_PiPi, lambda_Pipi_coef;        // 2/3, 8/5 (Eqs. 11-12)
  double minmod_theta;         // Eq. 67
  double xi0, rho_max;         // Eq. 74 (:445)
  int newton_max_iter; double newton_rtol;    // R6
  double tau_relax_floor_over_dtau;           // R14; 0 disables
  int storage;                                // 0: all ten pi^{mu nu} and four u^mu are propagated (the paper's choice, :333); 1: reduced storage
                                              //    (:476, Eqs. 47-51): only pi^xx, pi^xy, pi^xeta, pi^yy, pi^yeta and u^x, u^y, u^eta are state, reading R22
};

// field order of q (Eqs. 56-58 with the lost pi^{y eta} restored, R2):
//  0 T^tt 1 T^tx 2 T^ty 3 T^tn | 4 pi^tt 5 pi^tx 6 pi^ty 7 pi^tn 8 pi^xx 9 pi^xy 10 pi^xn 11 pi^yy 12 pi^yn 13 pi^nn | 14 Pi
constexpr int NQ = 15;
// symmetric index -> storage slot of pi^{mu nu} inside q
constexpr int PI_SLOT[4][4] = {{4, 5, 6, 7}, {5, 8, 9, 10}, {6, 9, 11, 12}, {7, 10, 12, 13}};

template <class R> inline R sgn(R x) { return (x > R(0)) ? R(1) : ((x < R(0)) ? R(-1) : R(0)); }  // R10: sgn(0)=0
template <class R> inline R absr(R x) { return (x < R(0)) ? -x : x; }
template <class R> inline R minr(R a, R b) { return (b < a) ? b : a; }
template <class R> inline R maxr(R a, R b) { return (b > a) ? b : a; }

// minmod(x,y) = [sgn x + sgn y] min(|x|,|y|)/2 ; minmod(x,y,z) = minmod(x, minmod(y,z))   (Eq. 68 and :411)
template <class R> inline R minmod2(R x, R y) { return (sgn(x) + sgn(y)) * minr(absr(x), absr(y)) / R(2); }
template <class R> inline R minmod3(R x, R y, R z) { return minmod2(x, minmod2(y, z)); }

// ---------------------------------------------------------------- equation of state / transport
template <class R> struct Thermo { R p, cs2, T; };

// BASELINE.json configs: eos 0  p=e/3 ; eos 1  p=(e/3)(1-alpha exp(-e/e0)); T=(e/a)^{1/4} for both.
template <class R> inline Thermo<R> eos(const Params& P, R e) {
  Thermo<R> t;
  if (P.eos == 0) {
    t.p = e / R(3);
    t.cs2 = R(1) / R(3);
  } else if (P.eos == 2) {
    // lattice EOS of section 2.3 (Eqs. 19-20): table + cubic Hermite interpolation, vh_oracle_lattice.hpp (evaluated in double)
    double pp, cc, TT;
    lattice::table().eval((double)e, pp, cc, TT);
    t.p = R(pp);
    t.cs2 = R(cc);
  } else {
    R x = e / R(P.eos_e0);
    R ex = exp(-x);
    t.p = (e / R(3)) * (R(1) - R(P.eos_alpha) * ex);
    t.cs2 = (R(1) / R(3)) * (R(1) - R(P.eos_alpha) * ex * (R(1) - x));   // dp/de
  }
  t.T = R(0);     // filled by temperature() where it is needed (transport coefficients only)
  return t;
}
template <class R> inline R temperature(const Params& P, R e) {
  if (P.eos == 2) { double pp, cc, TT; lattice::table().eval((double)e, pp, cc, TT); return R(TT); }      // T(e) of the lattice EOS
  return pow(e / R(P.eos_a), R(0.25));                                                                    // e = a T^4
}

template <class R> struct Transport {
  R inv_tau_pi, eta_over_tau_pi;        // 1/tau_pi, eta/tau_pi
  R inv_tau_Pi, zeta_over_tau_Pi;       // 1/tau_Pi, zeta/tau_Pi
  R lambda_Pipi_over_tau_Pi;            // (8/5)(1/3-cs2)  (Eq. 12)
};

// Eqs. 10-16 in the parametrisation of BASELINE.json configs; stiffness clamp R14.
template <class R> inline Transport<R> transport(const Params& P, R e, const Thermo<R>& th) {
  Transport<R> c;
  const R inf = std::numeric_limits<double>::infinity();
  R clamp = (P.tau_relax_floor_over_dtau > 0) ? R(1) / (R(P.tau_relax_floor_over_dtau) * R(P.dtau)) : inf;
  // shear: tau_pi = c_tau_pi (eta/s) / T  =>  1/tau_pi = T/(c_tau_pi eta/s);  eta/tau_pi = (e+p)/c_tau_pi   (Eq. 13)
  c.inv_tau_pi = minr(th.T / (R(P.c_tau_pi) * R(P.eta_over_s)), clamp);
  c.eta_over_tau_pi = (e + th.p) / R(P.c_tau_pi);
  // bulk
  R zs = R(0);
  if (P.zeta_model == 1) {
    R d = (th.T - R(P.zeta_T0)) / R(P.zeta_width);
    zs = R(P.zeta_amp) * exp(-d * d);
  } else if (P.zeta_model == 2) {
    zs = R(P.zeta_amp);
  } else if (P.zeta_model == 3) {
    // Eq. 17 (:174-186) times (zeta/s)_norm = zeta_amp, x = T/T_c with T_c = zeta_T0; ranges T < 0.995 T_c, in between, T > 1.05 T_c (R3)
    R x = th.T / R(P.zeta_T0);
    if (x > R(1.05)) zs = R(0.9) * exp(-(x - R(1)) / R(0.025)) + R(0.25) * exp(-(x - R(1)) / R(0.13)) + R(0.001);
    else if (x < R(0.995)) zs = R(0.9) * exp((x - R(1)) / R(0.0025)) + R(0.22) * exp((x - R(1)) / R(0.022)) + R(0.03);
    else zs = R(-13.45) + R(27.55) * x + R(-13.77) * x * x;
    zs = R(P.zeta_amp) * zs;
  }
  R b = R(1) / R(3) - th.cs2;
  R it = (zs > R(0)) ? th.T * b * b / (R(P.c_tau_Pi) * zs) : inf;
  c.inv_tau_Pi = minr(it, clamp);
  R s = (e + th.p) / th.T;                                // entropy density
  c.zeta_over_tau_Pi = (zs > R(0)) ? zs * s * c.inv_tau_Pi : R(0);
  c.lambda_Pipi_over_tau_Pi = R(P.lambda_Pipi_coef) * b;
  return c;
}

// ---------------------------------------------------------------- primitive inversion (Eqs. 52-54, 72; R6)
// Solves f(e) = e - E + M2/(E + P0(e) + Pi) = 0 by Newton-Raphson from `guess`.
template <class R> inline R invert_energy(const Params& P, R E, R M2, R Pi, R guess, int* iters, int* failed) {
  *failed = 0;
  *iters = 0;
  const R tiny = R(1e-300);
  bool bad = !(E > R(0)) || !std::isfinite((double)E) || !std::isfinite((double)M2) || !std::isfinite((double)Pi);
  R e = (guess > R(0) && std::isfinite((double)guess)) ? guess : E;
  bool conv = false;
  if (!bad) {
    for (int it = 0; it < P.newton_max_iter; ++it) {
      Thermo<R> th = eos(P, e);
      R den = E + th.p + Pi;
      R f = e - E + M2 / den;
      R fp = R(1) - M2 * th.cs2 / (den * den);
      R de = f / fp;
      R en = e - de;
      *iters = it + 1;
      e = en;
      if (absr(de) <= R(P.newton_rtol) * absr(en)) { conv = true; break; }
    }
  }
  if (bad || !conv || !(e > R(0)) || !std::isfinite((double)e)) {
    *failed = 1;
    e = maxr(E, tiny);
  }
  return e;
}

// ---------------------------------------------------------------- the solver
template <class R> class Solver {
 public:
  explicit Solver(const Params& prm) : P(prm) {
    NX = P.nx + 4; NY = P.ny + 4; NZ = P.nz + 4;
    N = (size_t)NX * NY * NZ;
    tau = P.tau0;
    for (int n = 0; n < NQ; ++n) { q[n].assign(N, R(0)); qS[n].assign(N, R(0)); Q[n].assign(N, R(0)); }
    for (int m = 0; m < 4; ++m) { u[m].assign(N, R(0)); up[m].assign(N, R(0)); uS[m].assign(N, R(0)); }
    reg_factor.assign(N, 1.0);
    e.assign(N, R(0)); p.assign(N, R(0));
  }

  Params P;
  int NX, NY, NZ;
  size_t N;
  double tau;
  long long n_steps = 0, n_fail = 0, n_nonfinite = 0;
  double min_reg_factor = 1.0;
  std::vector<double> reg_factor;         // tanh(rho)/rho that the most recent regularisation applied at each cell (Fig. 17); 1 before the first
  double last_fail[4] = {0, 0, 0, 0};     // E, M2, Pi, guess of the most recent failed inversion (diagnostics)
  std::vector<R> q[NQ], qS[NQ], Q[NQ];   // :470  q, qS, Q
  std::vector<R> u[4], up[4], uS[4];     // :470  u, up, uS
  std::vector<R> e, p;                   // :501  single copies

  size_t idx(int i, int j, int k) const { return (size_t)i + (size_t)NX * ((size_t)j + (size_t)NY * (size_t)k); }  // :472
  bool milne() const { return P.geometry == 0; }
  R tau2(R t) const { return milne() ? t * t : R(1); }

  // Program flow step 4 (:490): q^0 from (e,u,pi,Pi) via Eqs. 32-33; u^{-1}=u^0 (footnote 4 :519).
  // Arrays are physical cells only, x fastest.
  void set_initial(const double* e_in, const double* u_in, const double* pi_in, const double* Pi_in) {
    size_t np = (size_t)P.nx * P.ny * P.nz;
    for (int k = 0; k < P.nz; ++k) for (int j = 0; j < P.ny; ++j) for (int i = 0; i < P.nx; ++i) {
      size_t c = (size_t)i + (size_t)P.nx * ((size_t)j + (size_t)P.ny * k);
      size_t s = idx(i + 2, j + 2, k + 2);
      R ee = e_in[c];
      Thermo<R> th = eos(P, ee);
      R Pi = (Pi_in && (P.physics & 2)) ? R(Pi_in[c]) : R(0);
      R Pt = th.p + Pi;
      R uu[4];
      for (int m = 0; m < 4; ++m) uu[m] = u_in[m * np + c];
      R pi[10];
      for (int n = 0; n < 10; ++n) pi[n] = (pi_in && (P.physics & 1)) ? R(pi_in[n * np + c]) : R(0);
      if (reduced()) {     // the dependent components that were passed in are not state: replace them before T^{tau mu} is built
        const R t2i = tau2(R(P.tau0));
        uu[0] = sqrt(R(1) + uu[1] * uu[1] + uu[2] * uu[2] + t2i * uu[3] * uu[3]);
        R v[3] = {uu[1] / uu[0], uu[2] / uu[0], uu[3] / uu[0]}, d[5];
        dependent_pi(v, t2i, pi[4], pi[5], pi[6], pi[7], pi[8], d);
        pi[0] = d[0]; pi[1] = d[1]; pi[2] = d[2]; pi[3] = d[3]; pi[9] = d[4];
      }
      q[0][s] = (ee + Pt) * uu[0] * uu[0] - Pt + pi[0];                 // Eq. 32
      for (int m = 1; m < 4; ++m) q[m][s] = (ee + Pt) * uu[0] * uu[m] + pi[m];   // Eq. 33
      for (int n = 0; n < 10; ++n) q[4 + n][s] = pi[n];
      q[14][s] = Pi;
      e[s] = ee; p[s] = th.p;
      for (int m = 0; m < 4; ++m) { u[m][s] = uu[m]; up[m][s] = uu[m]; }
    }
    ghost(q, e, p, u);
    tau = P.tau0; n_steps = 0; n_fail = 0; n_nonfinite = 0; min_reg_factor = 1.0;
    reg_factor.assign((size_t)NX * NY * NZ, 1.0);
  }

  // optional: overwrite u^{n-1} (bit-exact restart)
  void set_uprev(const double* up_in) {
    size_t np = (size_t)P.nx * P.ny * P.nz;
    for (int k = 0; k < P.nz; ++k) for (int j = 0; j < P.ny; ++j) for (int i = 0; i < P.nx; ++i) {
      size_t c = (size_t)i + (size_t)P.nx * ((size_t)j + (size_t)P.ny * k);
      size_t s = idx(i + 2, j + 2, k + 2);
      for (int m = 0; m < 4; ++m) up[m][s] = up_in[m * np + c];
      // reduced storage: u^tau is not state - it is always the normalisation at the time level the velocity belongs to (here tau0 - dtau;
    // pinned by tests/test_oracle_reduced.py::test_reduced_mode_normalises_u_prev_at_its_own_time_level)
      if (reduced()) up[0][s] = sqrt(R(1) + up[1][s] * up[1][s] + up[2][s] * up[2][s] + tau2(R(P.tau0 - P.dtau)) * up[3][s] * up[3][s]);
    }
  }

  void get_fields(double* q_out, double* e_out, double* p_out, double* u_out, double* up_out) const {
    size_t np = (size_t)P.nx * P.ny * P.nz;
    for (int k = 0; k < P.nz; ++k) for (int j = 0; j < P.ny; ++j) for (int i = 0; i < P.nx; ++i) {
      size_t c = (size_t)i + (size_t)P.nx * ((size_t)j + (size_t)P.ny * k);
      size_t s = idx(i + 2, j + 2, k + 2);
      if (q_out) for (int n = 0; n < NQ; ++n) q_out[n * np + c] = (double)q[n][s];
      if (e_out) e_out[c] = (double)e[s];
      if (p_out) p_out[c] = (double)p[s];
      if (u_out) for (int m = 0; m < 4; ++m) u_out[m * np + c] = (double)u[m][s];
      if (up_out) for (int m = 0; m < 4; ++m) up_out[m * np + c] = (double)up[m][s];
    }
  }

  // ------------------------------------------------------------ diagnostics, maxima over the physical cells
  // out[0] max T (freeze-out test "T < T_f everywhere", program-flow step 8, :494);  out[1] max |u.u - 1| (:489);
  // out[2] max |g_{mu nu} pi^{mu nu}|/(e+p), out[3] max_lambda |pi^{lambda mu} u_mu|/(e+p) (Eqs. 47-51, :318-331; the lambda = eta
  // entry times tau);  out[8], out[9]: second-order inverse Reynolds numbers of Eq. 90 (see cell_diagnostics);  out[4] max R_pi^-1 = sqrt(pi^{mu nu} pi_{mu nu})/P0, out[5] max R_Pi^-1 = |Pi|/P0 (Eq. 89, :826);
  // out[6] max Kn_{theta pi} = tau_pi |theta|, out[7] max Kn_{theta Pi} = tau_Pi |theta| (:830) with theta of A.11 discretised as in the
  // sources (backward difference in time, central in space, :424) and the relaxation times the solver uses (R14); a cell whose
  // quotient is not finite (1/tau = 0) does not count; 0 when the sector is switched off
  void cell_diagnostics(size_t s, double v[10]) {      // the ten quantities at one cell (see diagnostics())
    const size_t stride[3] = {1, (size_t)NX, (size_t)NX * NY};
    const double dr[3] = {P.dx, P.dy, P.dz};
    const double t = (double)tau, t2 = (double)tau2(tau);
    const double g[4] = {1.0, -1.0, -1.0, -t2};
    const double ee = (double)e[s], pp = (double)p[s];
    const double T = (double)temperature(P, e[s]);
    double uu[4], pim[4][4];
    for (int m = 0; m < 4; ++m) uu[m] = (double)u[m][s];
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) pim[m][n] = (double)q[PI_SLOT[m][n]][s];
    double norm = 0.0, tr = 0.0, pipi = 0.0, orth = 0.0;
    for (int m = 0; m < 4; ++m) { norm += g[m] * uu[m] * uu[m]; tr += g[m] * pim[m][m]; }
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) pipi += g[m] * g[n] * pim[m][n] * pim[m][n];
    for (int l = 0; l < 4; ++l) {
      double c = 0.0;
      for (int m = 0; m < 4; ++m) c += pim[l][m] * g[m] * uu[m];
      if (l == 3 && milne()) c *= t;
      orth = std::fmax(orth, std::fabs(c));
    }
    v[0] = T;
    v[1] = std::fabs(norm - 1.0);
    v[2] = std::fabs(tr) / (ee + pp);
    v[3] = orth / (ee + pp);
    v[4] = std::sqrt(std::fabs(pipi)) / pp;
    v[5] = std::fabs((double)q[14][s]) / pp;
    double theta = (milne() ? uu[0] / t : 0.0) + (uu[0] - (double)up[0][s]) / P.dtau;
    for (int d = 0; d < 3; ++d) theta += ((double)u[d + 1][s + stride[d]] - (double)u[d + 1][s - stride[d]]) / (2.0 * dr[d]);
    Thermo<double> th = eos<double>(P, ee);
    th.T = T;
    const Transport<double> tc = transport<double>(P, ee, th);
    const double kp = std::fabs(theta) / tc.inv_tau_pi, kP = std::fabs(theta) / tc.inv_tau_Pi;
    v[6] = ((P.physics & 1) && std::isfinite(kp)) ? kp : 0.0;
    v[7] = ((P.physics & 2) && std::isfinite(kP)) ? kP : 0.0;
    // second-order inverse Reynolds numbers (Eq. 90, :831) from the terms of the source routine; 0 where 0/0 or the sector is off
    R J[NQ], second[2];
    sources(q, e, p, u, up, s, tau, J, second);
    v[8] = std::isfinite((double)second[0]) ? (double)second[0] : 0.0;
    v[9] = std::isfinite((double)second[1]) ? (double)second[1] : 0.0;
  }
  void diagnostics(double out[10]) {
    for (int i = 0; i < 10; ++i) out[i] = 0.0;
    for (int k = 2; k < NZ - 2; ++k) for (int j = 2; j < NY - 2; ++j) for (int i = 2; i < NX - 2; ++i) {
      double v[10];
      cell_diagnostics(idx(i, j, k), v);
      for (int m = 0; m < 10; ++m) out[m] = std::fmax(out[m], v[m]);
    }
  }
  // the factor of Eqs. 73-74 that the last regularisation (program-flow step 8 of the last time step) applied, physical cells, x fastest
  void regulation_map(double* out) const {
    size_t c = 0;
    for (int k = 2; k < NZ - 2; ++k) for (int j = 2; j < NY - 2; ++j) for (int i = 2; i < NX - 2; ++i, ++c) out[c] = reg_factor[idx(i, j, k)];
  }
  // the same ten quantities cell by cell (Figs. 15-17 of the paper are such maps): maps[m * np + c], physical cells, x fastest
  void diagnostic_maps(double* maps, size_t np, size_t offset) {
    size_t c = offset;
    for (int k = 2; k < NZ - 2; ++k) for (int j = 2; j < NY - 2; ++j) for (int i = 2; i < NX - 2; ++i, ++c) {
      double v[10];
      cell_diagnostics(idx(i, j, k), v);
      for (int m = 0; m < 10; ++m) maps[m * np + c] = v[m];
    }
  }

  // ------------------------------------------------------------ reduced storage (PAPER.md:476 with Eqs. 47-51, :318-331; reading R22)
  // "it can be reduced by simply propagating only the independent components of pi^{mu nu} (five) and u^mu (three), with the remaining
  // components determined algebraically."  The five are the paper's example (:316): pi^xx, pi^xy, pi^xeta, pi^yy, pi^yeta.  In this mode the
  // other five components and u^tau are NOT state: wherever the algorithm reads them (at any stencil cell) they are the algebraic values
  // below, evaluated with the velocity of that cell; what the Euler step computes for them is discarded.
  bool reduced() const { return P.storage == 1 && (P.physics & 1); }
  // Eqs. 48-51 then 47 (Eq. 49 with its typo fixed, R3: the last term is tau^2 pi^{y eta} v_eta) from v^i = u^i/u^tau
  void dependent_pi(const R v[3], R t2, R pxx, R pxy, R pxn, R pyy, R pyn, R out[5]) const {     // out: pi^tt, pi^tx, pi^ty, pi^tn, pi^nn
    const R vx = v[0], vy = v[1], vn = v[2];
    R pnn = (pxx * (vx * vx - R(1)) + pyy * (vy * vy - R(1)) + R(2) * pxy * vx * vy + R(2) * t2 * (pxn * vx * vn + pyn * vy * vn)) /
            (t2 * (R(1) - t2 * vn * vn));                                        // Eq. 51
    R ptx = pxx * vx + pxy * vy + t2 * pxn * vn;                                // Eq. 48
    R pty = pxy * vx + pyy * vy + t2 * pyn * vn;                                // Eq. 49
    R ptn = pxn * vx + pyn * vy + t2 * pnn * vn;                                // Eq. 50
    R ptt = ptx * vx + pty * vy + t2 * ptn * vn;                                // Eq. 47
    out[0] = ptt; out[1] = ptx; out[2] = pty; out[3] = ptn; out[4] = pnn;
  }
  // u^tau from u.u = 1 (:489) and the five dependent components, at every cell incl. ghosts (ghost cells are copies of q and u alike)
  void expand_all(std::vector<R>* qq, std::vector<R>* uu, R t) {
    const R t2 = tau2(t);
    for (size_t s = 0; s < N; ++s) {
      uu[0][s] = sqrt(R(1) + uu[1][s] * uu[1][s] + uu[2][s] * uu[2][s] + t2 * uu[3][s] * uu[3][s]);
      R v[3] = {uu[1][s] / uu[0][s], uu[2][s] / uu[0][s], uu[3][s] / uu[0][s]}, d[5];
      dependent_pi(v, t2, qq[8][s], qq[9][s], qq[10][s], qq[11][s], qq[12][s], d);
      qq[4][s] = d[0]; qq[5][s] = d[1]; qq[6][s] = d[2]; qq[7][s] = d[3]; qq[13][s] = d[4];
    }
  }

  // ------------------------------------------------------------ ghost cells, Eqs. 75-76 (:459-466)
  void ghost_one(std::vector<R>& a) {
    for (int k = 2; k < NZ - 2; ++k) for (int j = 2; j < NY - 2; ++j) {
      a[idx(0, j, k)] = a[idx(1, j, k)] = a[idx(2, j, k)];
      a[idx(NX - 1, j, k)] = a[idx(NX - 2, j, k)] = a[idx(NX - 3, j, k)];
    }
    for (int k = 2; k < NZ - 2; ++k) for (int i = 2; i < NX - 2; ++i) {
      a[idx(i, 0, k)] = a[idx(i, 1, k)] = a[idx(i, 2, k)];
      a[idx(i, NY - 1, k)] = a[idx(i, NY - 2, k)] = a[idx(i, NY - 3, k)];
    }
    for (int j = 2; j < NY - 2; ++j) for (int i = 2; i < NX - 2; ++i) {
      a[idx(i, j, 0)] = a[idx(i, j, 1)] = a[idx(i, j, 2)];
      a[idx(i, j, NZ - 1)] = a[idx(i, j, NZ - 2)] = a[idx(i, j, NZ - 3)];
    }
  }
  void ghost(std::vector<R>* qq, std::vector<R>& ee, std::vector<R>& pp, std::vector<R>* uu) {
    for (int n = 0; n < NQ; ++n) ghost_one(qq[n]);
    ghost_one(ee); ghost_one(pp);
    for (int m = 0; m < 4; ++m) ghost_one(uu[m]);
  }

  // ------------------------------------------------------------ interface state -> v_r   (:424, Alg. 3 :667-672; R5, R6)
  // qs: a reconstructed conserved state; returns the three v^i = M_i/(E+P) of that state.
  void state_velocity(const R* qs, R t, R guess, bool count, R v[3]) {
    R E = qs[0] - qs[4];
    R M[3] = {qs[1] - qs[5], qs[2] - qs[6], qs[3] - qs[7]};
    R M2 = M[0] * M[0] + M[1] * M[1] + tau2(t) * M[2] * M[2];          // :339
    int it, fail;
    R ee = invert_energy(P, E, M2, qs[14], guess, &it, &fail);
    Thermo<R> th = eos(P, ee);
    R den = E + th.p + qs[14];
    for (int i = 0; i < 3; ++i) v[i] = M[i] / den;
    if (fail) {
      if (count) ++n_fail;
      last_fail[0] = (double)E; last_fail[1] = (double)M2; last_fail[2] = (double)qs[14]; last_fail[3] = (double)guess;
      for (int i = 0; i < 3; ++i) {                                      // R6: clip |v|<1
        if (!(absr(v[i]) < R(1))) v[i] = (v[i] > R(0)) ? R(1) - R(1e-12) : ((v[i] < R(0)) ? R(-1) + R(1e-12) : R(0));
      }
    }
  }

  // Numerical flux H at the interface between stencil cells c and c+1 (Eq. 61), direction r.
  // I[n][0..4] = q_n at i-2..i+2 ; eI = e at the same cells ; c = 2 -> H_{i+1/2}, c = 1 -> H_{i-1/2}.
  void flux(const R I[NQ][5], const R eI[5], int c, int r, R dr, R t, bool count, R H[NQ]) {
    R qm[NQ], qp[NQ];
    R th = R(P.minmod_theta);
    for (int n = 0; n < NQ; ++n) {
      // Eq. 67 slopes of cell c and of cell c+1
      VHO_COUNTING_SECTION(3);
      R sc = minmod3(th * (I[n][c] - I[n][c - 1]) / dr, (I[n][c + 1] - I[n][c - 1]) / (R(2) * dr), th * (I[n][c + 1] - I[n][c]) / dr);
      R sn = minmod3(th * (I[n][c + 1] - I[n][c]) / dr, (I[n][c + 2] - I[n][c]) / (R(2) * dr), th * (I[n][c + 2] - I[n][c + 1]) / dr);
      VHO_COUNTING_SECTION(1);
      qm[n] = I[n][c] + (dr / R(2)) * sc;         // q^-: Eq. 64 / 66
      qp[n] = I[n][c + 1] - (dr / R(2)) * sn;     // q^+: Eq. 63 / 65
    }
    R vm[3], vp[3];
    VHO_COUNTING_SECTION(2);
    state_velocity(qm, t, eI[c], count, vm);      // guess: e of the cell the state was extrapolated from (R6)
    state_velocity(qp, t, eI[c + 1], count, vp);
    VHO_COUNTING_SECTION(1);
    R a = maxr(absr(vp[r]), absr(vm[r]));         // Eq. 62 with rho = |v_r| (:388)
    for (int n = 0; n < NQ; ++n) H[n] = (vp[r] * qp[n] + vm[r] * qm[n]) / R(2) - a * (qp[n] - qm[n]) / R(2);   // Eq. 61
  }

  // ------------------------------------------------------------ sources J = S + G  (App. B; Eqs. 39-46; App. A index forms)
  void sources(const std::vector<R>* qi, const std::vector<R>& ei, const std::vector<R>& pi_, const std::vector<R>* ui,
               const std::vector<R>* uprev, size_t s, R t, R J[NQ], R* second = nullptr) {
    const size_t stride[3] = {1, (size_t)NX, (size_t)NX * NY};
    const R dr[3] = {R(P.dx), R(P.dy), R(P.dz)};
    const bool mil = milne();
    const R t2 = tau2(t);
    R g[4] = {R(1), R(-1), R(-1), -t2};              // g_{mu mu}  (Eq. 27)
    R gi[4] = {R(1), R(-1), R(-1), R(-1) / t2};      // g^{mu mu}
    for (int n = 0; n < NQ; ++n) J[n] = R(0);

    R uc[4]; for (int m = 0; m < 4; ++m) uc[m] = ui[m][s];
    R pic[4][4]; for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) pic[m][n] = qi[PI_SLOT[m][n]][s];
    R Pic = qi[14][s];
    R ec = ei[s], pc = pi_[s];
    R Ptc = pc + Pic;

    // ---- conservation rows.  S_c^nu = -d_i A^{i nu},  A^{i nu} = P (v^i delta^nu_tau - g^{i nu}) - v^i pi^{tau nu} + pi^{i nu}
    //      (B.2-B.5 :1002-1009, from Eqs. 33-34), central differences of the products at the neighbours (R11, :424)
    for (int i = 0; i < 3; ++i) {
      R A[2][4];
      for (int sd = 0; sd < 2; ++sd) {
        size_t sn = (sd == 0) ? s - stride[i] : s + stride[i];
        R vi = ui[i + 1][sn] / ui[0][sn];
        R Pt = pi_[sn] + qi[14][sn];
        for (int nu = 0; nu < 4; ++nu) {
          R gin = (nu == i + 1) ? gi[nu] : R(0);
          R dl = (nu == 0) ? R(1) : R(0);
          A[sd][nu] = Pt * (vi * dl - gin) - vi * qi[PI_SLOT[0][nu]][sn] + qi[PI_SLOT[i + 1][nu]][sn];
        }
      }
      for (int nu = 0; nu < 4; ++nu) J[nu] -= (A[1][nu] - A[0][nu]) / (R(2) * dr[i]);
    }
    // G_c (:1013) with T^{eta eta} = (e+P)(u^eta)^2 + P/tau^2 + pi^{eta eta}  (Eq. 34)
    if (mil) {
      R Tnn = (ec + Ptc) * uc[3] * uc[3] + Ptc / t2 + pic[3][3];
      J[0] -= (qi[0][s] + t2 * Tnn) / t;
      J[1] -= qi[1][s] / t;
      J[2] -= qi[2][s] / t;
      J[3] -= R(3) * qi[3][s] / t;
    }
    if (second) second[0] = second[1] = R(0);
    if ((P.physics & 3) == 0) return;     // ideal mode: pi, Pi stay zero

    // ---- velocity gradients: backward difference in time, central in space (:424)
    R du[4][4];                            // du[a][n] = partial_a u^n
    for (int n = 0; n < 4; ++n) du[0][n] = (uc[n] - uprev[n][s]) / R(P.dtau);
    R divv = R(0);                         // partial_i v^i
    for (int i = 0; i < 3; ++i) {
      size_t sm = s - stride[i], sp = s + stride[i];
      for (int n = 0; n < 4; ++n) du[i + 1][n] = (ui[n][sp] - ui[n][sm]) / (R(2) * dr[i]);
      divv += (ui[i + 1][sp] / ui[0][sp] - ui[i + 1][sm] / ui[0][sm]) / (R(2) * dr[i]);
    }
    // Christoffel symbols (Eq. 29), sparse list (l; a b)
    struct Chr { int l, a, b; R v; };
    Chr G3[3] = {{3, 0, 3, R(1) / t}, {3, 3, 0, R(1) / t}, {0, 3, 3, t}};
    int nG = mil ? 3 : 0;

    R conv[4], Dup[4], Dlo[4];             // du^n = u^a d_a u^n (A.5-A.8);  Du^n;  Du_l (A.9-A.10)
    for (int n = 0; n < 4; ++n) { conv[n] = R(0); for (int a = 0; a < 4; ++a) conv[n] += uc[a] * du[a][n]; }
    for (int n = 0; n < 4; ++n) Dup[n] = conv[n];
    for (int c = 0; c < nG; ++c) Dup[G3[c].l] += G3[c].v * uc[G3[c].a] * uc[G3[c].b];
    for (int l = 0; l < 4; ++l) Dlo[l] = g[l] * Dup[l];
    // theta = d_mu u^mu + Gamma^l_{l mu} u^mu   (A.2, A.11)
    R theta = R(0);
    for (int a = 0; a < 4; ++a) theta += du[a][a];
    for (int c = 0; c < nG; ++c) if (G3[c].l == G3[c].a) theta += G3[c].v * uc[G3[c].b];
    R Delta[4][4];
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) Delta[m][n] = ((m == n) ? gi[m] : R(0)) - uc[m] * uc[n];
    // sigma^{mu nu}: A.3, second form (:912-913)
    R sig[4][4];
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) {
      R a1 = gi[m] * du[m][n] - uc[m] * conv[n] + gi[n] * du[n][m] - uc[n] * conv[m];
      R a2 = R(0);
      for (int c = 0; c < nG; ++c) {
        if (G3[c].l == n) a2 += Delta[m][G3[c].a] * uc[G3[c].b] * G3[c].v;
        if (G3[c].l == m) a2 += Delta[n][G3[c].a] * uc[G3[c].b] * G3[c].v;
      }
      sig[m][n] = a1 / R(2) + a2 / R(2) - (theta / R(3)) * Delta[m][n];
    }
    // W^{mu nu} = (1/2)(nabla^mu u^nu - nabla^nu u^mu), nabla^mu = Delta^{mu a} d_a  (:122)
    R cov[4][4];                           // cov[a][n] = d_a u^n = partial_a u^n + Gamma^n_{a l} u^l  (Eq. 25)
    for (int a = 0; a < 4; ++a) for (int n = 0; n < 4; ++n) cov[a][n] = du[a][n];
    for (int c = 0; c < nG; ++c) cov[G3[c].a][G3[c].l] += G3[c].v * uc[G3[c].b];
    R nab[4][4];
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) { nab[m][n] = R(0); for (int a = 0; a < 4; ++a) nab[m][n] += Delta[m][a] * cov[a][n]; }
    R W[4][4];
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) W[m][n] = (nab[m][n] - nab[n][m]) / R(2);

    Thermo<R> th = eos(P, ec);
    th.T = temperature(P, ec);
    Transport<R> tc = transport(P, ec, th);

    R pisig = R(0);                        // pi^{mu nu} sigma_{mu nu}
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) pisig += g[m] * g[n] * pic[m][n] * sig[m][n];

    R JJ = R(0), sigsig = R(0);            // J^{mu nu} J_{mu nu} / tau_pi^2 and sigma^{mu nu} sigma_{mu nu}  (Eq. 90)
    if (P.physics & 1) {
      for (int m = 0; m < 4; ++m) for (int n = m; n < 4; ++n) {
        R I1 = R(0), I3 = R(0), I4 = R(0);
        for (int l = 0; l < 4; ++l) {
          I1 += (pic[l][m] * uc[n] + pic[l][n] * uc[m]) * Dlo[l];                                  // Eq. 43
          I3 += pic[m][l] * g[l] * W[l][n] + pic[n][l] * g[l] * W[l][m];                           // Eq. 45, R4
          I4 += g[l] * (pic[m][l] * sig[n][l] + pic[n][l] * sig[m][l]) / R(2);                     // Eq. 46
        }
        I3 *= R(kVorticitySign);
        I4 -= Delta[m][n] * pisig / R(3);
        R I2 = theta * pic[m][n];                                                                 // Eq. 44
        R Ipi = I1 + R(P.delta_pipi) * I2 - I3 + R(P.tau_pipi) * I4 - R(P.lambda_piPi) * Pic * sig[m][n];   // Eq. 42
        // Eq. 5 with n^mu = 0: J^{mu nu}/tau_pi = -(Ipi - I1)  (I1 belongs to the projected time derivative, not to J)
        if (second) {                      // diagnostics only: never part of a time step (nor of its operation count)
          const R w = g[m] * g[n] * ((m == n) ? R(1) : R(2));
          JJ += w * (Ipi - I1) * (Ipi - I1);
          sigsig += w * sig[m][n] * sig[m][n];
        }
        R Gpi = R(0);                                                                             // :300, R1, R2
        for (int c = 0; c < nG; ++c) {
          if (G3[c].l == m) Gpi += uc[G3[c].a] * G3[c].v * pic[G3[c].b][n];
          if (G3[c].l == n) Gpi += uc[G3[c].a] * G3[c].v * pic[G3[c].b][m];
        }
        // B.11 + G_pi/u^tau  (B.9)
        J[PI_SLOT[m][n]] = (R(2) * tc.eta_over_tau_pi * sig[m][n] - pic[m][n] * tc.inv_tau_pi - Ipi - Gpi) / uc[0] + pic[m][n] * divv;
      }
    }
    if (P.physics & 2) {
      R IPi = R(P.delta_PiPi) * Pic * theta - tc.lambda_Pipi_over_tau_Pi * pisig;                 // Eq. 41
      J[14] = (-tc.zeta_over_tau_Pi * theta - Pic * tc.inv_tau_Pi - IPi) / uc[0] + Pic * divv;    // B.10
      if (second) second[1] = absr(IPi) / (tc.zeta_over_tau_Pi * absr(theta));                   // Eq. 90: |J|/(zeta |theta|), J/tau_Pi = -IPi
    }
    if (second && (P.physics & 1)) second[0] = sqrt(absr(JJ)) / (R(2) * tc.eta_over_tau_pi * sqrt(absr(sigsig)));   // Eq. 90
  }

  // ------------------------------------------------------------ forward Euler step E[w] = w + dtau C[w]  (Eq. 59, :413)
  void euler(const std::vector<R>* qi, const std::vector<R>& ei, const std::vector<R>& pi_, const std::vector<R>* ui,
             const std::vector<R>* uprev, R t, std::vector<R>* qo) {
    const size_t stride[3] = {1, (size_t)NX, (size_t)NX * NY};
    const R dr[3] = {R(P.dx), R(P.dy), R(P.dz)};
    for (int k = 2; k < NZ - 2; ++k) for (int j = 2; j < NY - 2; ++j) for (int i = 2; i < NX - 2; ++i) {
      size_t s = idx(i, j, k);
      R C[NQ];
      sources(qi, ei, pi_, ui, uprev, s, t, C);
      for (int r = 0; r < 3; ++r) {
        R I[NQ][5], eI[5];
        for (int d = 0; d < 5; ++d) {
          size_t sn = s + (size_t)d * stride[r] - 2 * stride[r];
          for (int n = 0; n < NQ; ++n) I[n][d] = qi[n][sn];
          eI[d] = ei[sn];
        }
        R Hp[NQ], Hm[NQ];
        // diagnostics only: each interface state is counted once in n_fail (H_{+1/2} by this cell, H_{-1/2} only by the first
        // cell of the row) and not at all along a direction of extent 1, where H_{+1/2} - H_{-1/2} vanishes identically
        const int ext[3] = {P.nx, P.ny, P.nz};
        const int pos[3] = {i, j, k};
        VHO_COUNTING_SECTION(1);
        flux(I, eI, 2, r, dr[r], t, ext[r] > 1, Hp);
        flux(I, eI, 1, r, dr[r], t, ext[r] > 1 && pos[r] == 2, Hm);
        VHO_COUNTING_SECTION(0);
        for (int n = 0; n < NQ; ++n) C[n] -= (Hp[n] - Hm[n]) / dr[r];
      }
      for (int n = 0; n < NQ; ++n) qo[n][s] = qi[n][s] + R(P.dtau) * C[n];
      if (!(P.physics & 1)) for (int n = 4; n < 14; ++n) qo[n][s] = R(0);
      if (!(P.physics & 2)) qo[14][s] = R(0);
    }
  }

  // ------------------------------------------------------------ steps 2-4 / 8 (:510-512, :528): invert, regulate, ghost
  R regulate_cell(std::vector<R>* qq, size_t s, R ee, R p0, const R* uu, R t) {
    const R t2 = tau2(t);
    R g[4] = {R(1), R(-1), R(-1), -t2};
    R pic[4][4]; for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) pic[m][n] = qq[PI_SLOT[m][n]][s];
    R Pic = qq[14][s];
    R pipi = R(0), tr = R(0);
    for (int m = 0; m < 4; ++m) { tr += g[m] * pic[m][m]; for (int n = 0; n < 4; ++n) pipi += g[m] * g[n] * pic[m][n] * pic[m][n]; }
    R PP = sqrt(absr(pipi + R(3) * Pic * Pic));                      // sqrt(Pi^{mu nu} Pi_{mu nu}), R9
    R den0 = R(P.rho_max) * sqrt(ee * ee + R(3) * p0 * p0);
    R rho = PP / den0;
    R den1 = R(P.xi0) * R(P.rho_max) * PP;
    if (PP > R(0) && std::isfinite((double)den1)) {
      rho = maxr(rho, absr(tr) / den1);
      for (int l = 0; l < 4; ++l) {
        R pu = R(0);
        for (int m = 0; m < 4; ++m) pu += pic[l][m] * g[m] * uu[m];   // pi^{l mu} u_mu
        if (l == 3) pu *= sqrt(t2);                                   // eta component in units of the others, R9
        rho = maxr(rho, absr(pu) / den1);
      }
    }
    if (!std::isfinite((double)rho)) rho = R(0);
    R fac = (rho < R(1e-8)) ? R(1) : tanh(rho) / rho;                 // Eq. 73
    for (int n = 4; n < NQ; ++n) qq[n][s] *= fac;
    return fac;
  }

  // Reduced storage: pi^{tau mu} in E = T^{tau tau} - pi^{tau tau}, M_i = T^{tau i} - pi^{tau i} depend on the unknown velocity (Eqs. 47-50),
  // so Eqs. 52-54 become implicit.  Reading R22: fixed point on v - start from the velocity of the same cell at the stage's input,
  // v <- M(v)/(E(v) + P(e)) with e from Eq. 72 at every sweep (guess: previous sweep's e), until max_i |dv_i| <= newton_rtol (eta
  // component in units of the others) or newton_max_iter sweeps (then a failure is counted).  Returns the converged dependent components.
  void implicit_inversion(std::vector<R>* qq, size_t s, R t, const R vguess[3], R eguess, R& ee, R M[3], R& E, int& fail) {
    const R t2 = tau2(t), rt = sqrt(t2);
    R v[3] = {vguess[0], vguess[1], vguess[2]};
    R d[5];
    bool conv = false;
    fail = 0;
    ee = eguess;
    for (int sweep = 0; sweep < P.newton_max_iter && !conv; ++sweep) {
      dependent_pi(v, t2, qq[8][s], qq[9][s], qq[10][s], qq[11][s], qq[12][s], d);
      E = qq[0][s] - d[0];
      M[0] = qq[1][s] - d[1]; M[1] = qq[2][s] - d[2]; M[2] = qq[3][s] - d[3];
      R M2 = M[0] * M[0] + M[1] * M[1] + t2 * M[2] * M[2];
      int it, f1;
      ee = invert_energy(P, E, M2, qq[14][s], ee, &it, &f1);
      if (f1) { fail = 1; break; }
      Thermo<R> th = eos(P, ee);
      R den = E + th.p + qq[14][s];
      R vn[3] = {M[0] / den, M[1] / den, M[2] / den};
      R dv = maxr(maxr(absr(vn[0] - v[0]), absr(vn[1] - v[1])), rt * absr(vn[2] - v[2]));
      v[0] = vn[0]; v[1] = vn[1]; v[2] = vn[2];
      if (dv <= R(P.newton_rtol)) conv = true;
    }
    if (!conv) fail = 1;
    // the state that is kept: dependent components of the converged velocity (and E, M consistent with them)
    dependent_pi(v, t2, qq[8][s], qq[9][s], qq[10][s], qq[11][s], qq[12][s], d);
    qq[4][s] = d[0]; qq[5][s] = d[1]; qq[6][s] = d[2]; qq[7][s] = d[3]; qq[13][s] = d[4];
    E = qq[0][s] - d[0];
    M[0] = qq[1][s] - d[1]; M[1] = qq[2][s] - d[2]; M[2] = qq[3][s] - d[3];
  }

  // ug: velocity of the stage's input (used only by the reduced-storage mode as the starting point of its fixed point)
  void post(std::vector<R>* qq, std::vector<R>* uo, R t, const std::vector<R>* ug = nullptr) {
    for (int k = 2; k < NZ - 2; ++k) for (int j = 2; j < NY - 2; ++j) for (int i = 2; i < NX - 2; ++i) {
      size_t s = idx(i, j, k);
      if (reduced()) {
        R vg[3] = {ug[1][s] / ug[0][s], ug[2][s] / ug[0][s], ug[3][s] / ug[0][s]};
        R ee, M[3], E;
        int fail;
        implicit_inversion(qq, s, t, vg, e[s], ee, M, E, fail);
        if (fail) ++n_fail;
        R Pic = qq[14][s];
        Thermo<R> th = eos(P, ee);
        R Pt = th.p + Pic;
        R ut = sqrt((E + Pt) / (ee + Pt));                              // Eq. 53
        R uu[4] = {ut, M[0] / ((ee + Pt) * ut), M[1] / ((ee + Pt) * ut), M[2] / ((ee + Pt) * ut)};   // Eq. 54
        e[s] = ee; p[s] = th.p;
        for (int m = 1; m < 4; ++m) uo[m][s] = uu[m];
        uo[0][s] = sqrt(R(1) + uu[1] * uu[1] + uu[2] * uu[2] + tau2(t) * uu[3] * uu[3]);      // u^tau is not state: always from u.u = 1
        if (!(std::isfinite((double)ee) && std::isfinite((double)ut))) ++n_nonfinite;
        R fac = regulate_cell(qq, s, ee, th.p, uu, t);                  // step 3 (:511): all ten components scale alike, so Eqs. 47-51 keep holding
        if ((double)fac < min_reg_factor) min_reg_factor = (double)fac;
        reg_factor[s] = (double)fac;
        continue;
      }
      R E = qq[0][s] - qq[4][s];
      R M[3] = {qq[1][s] - qq[5][s], qq[2][s] - qq[6][s], qq[3][s] - qq[7][s]};
      R M2 = M[0] * M[0] + M[1] * M[1] + tau2(t) * M[2] * M[2];
      R Pic = qq[14][s];
      int it, fail;
      R ee = invert_energy(P, E, M2, Pic, e[s], &it, &fail);           // guess: e of the previous stage (R6)
      if (fail) { ++n_fail; last_fail[0] = (double)E; last_fail[1] = (double)M2; last_fail[2] = (double)Pic; last_fail[3] = (double)e[s]; }
      Thermo<R> th = eos(P, ee);
      R Pt = th.p + Pic;
      R ut = sqrt((E + Pt) / (ee + Pt));                                // Eq. 53
      R uu[4] = {ut, M[0] / ((ee + Pt) * ut), M[1] / ((ee + Pt) * ut), M[2] / ((ee + Pt) * ut)};   // Eq. 54
      e[s] = ee; p[s] = th.p;
      for (int m = 0; m < 4; ++m) uo[m][s] = uu[m];
      bool fin = std::isfinite((double)ee) && std::isfinite((double)ut);
      if (!fin) ++n_nonfinite;
      if (P.physics & 3) {                                              // step 3 (:511), after the inversion (R8)
        R fac = regulate_cell(qq, s, ee, th.p, uu, t);
        if ((double)fac < min_reg_factor) min_reg_factor = (double)fac;
        reg_factor[s] = (double)fac;
      }
    }
    ghost(qq, e, p, uo);                                                // step 4 (:512)
  }

  // ------------------------------------------------------------ one full RK step, program-flow steps 1-9 (:503-529)
  void step() {
    R t = tau, dt = P.dtau;
    if (reduced()) expand_all(q, u, t);           // (reduced storage: the dependent components of the state are their algebraic values)
    euler(q, e, p, u, up, t, qS);                 // 1. q* = E[q^n; e,p,u^n,u^{n-1}] at tau^n
    post(qS, uS, t + dt, u);                      // 2-4. e*,p*,u* ; regulate q* ; ghosts      (R7: tau^n + dtau)
    euler(qS, e, p, uS, u, t + dt, Q);            // 5. q** = E[q*; e*,p*,u*,u^n] at tau^n + dtau
    for (int k = 2; k < NZ - 2; ++k) for (int j = 2; j < NY - 2; ++j) for (int i = 2; i < NX - 2; ++i) {
      size_t s = idx(i, j, k);
      for (int n = 0; n < NQ; ++n) Q[n][s] = (q[n][s] + Q[n][s]) / R(2);   // 6. convex combination
    }
    for (int m = 0; m < 4; ++m) up[m].swap(u[m]); // 7. up <-> u
    post(Q, u, t + dt, uS);                       // 8. e,p,u^{n+1}; regulate; ghosts
    for (int n = 0; n < NQ; ++n) q[n].swap(Q[n]); // 9. q <-> Q
    ++n_steps;
    tau = P.tau0 + (double)n_steps * P.dtau;      // :493  tau = tau_0 + n dtau
  }
};

}  // namespace vho
