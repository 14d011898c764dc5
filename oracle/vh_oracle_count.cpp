// TEST INFRASTRUCTURE ONLY (see vh_oracle.hpp).  Instantiates the oracle with an operation-counting scalar to measure
// the ALGORITHMIC floating-point work of one KT/RK2 step ("replace the estimate by a measured count").
// Operations whose operands are all compile-time / per-run constants are not counted (a compiler hoists them), and neither is
// an addition of an exact constant 0 or a multiplication / division by an exact constant 0 or +-1 (the index-form loops of the
// oracle multiply by Kronecker deltas and metric signs; that is notation, not work the method needs).  Compares are their own
// class and carry no flop weight.  Work the oracle repeats is counted in sections of its own so that it can be charged once:
// every interface is evaluated from both adjacent cells (Alg. 2), and every limited slope (Eq. 67) four times.
#include <cmath>
#include <cstring>

namespace vho_cnt {
enum { ADD = 0, MUL, DIV, CMP, SQRT, EXP, POW, TANH, NCLASS };
static long long g_counts[4][NCLASS];
static int g_section = 0;     // 0: everything else, 1: inside flux(): half-cell extrapolation + Eq. 61, 2: the interface-state inversions inside flux(), 3: the limited slopes inside flux()
static bool g_on = false;
inline void tick(int cls, bool live) { if (g_on && live) ++g_counts[g_section][cls]; }

struct Cnt {
  double v;
  bool k;      // true: derived from constants only
  Cnt() : v(0), k(true) {}
  Cnt(double x) : v(x), k(true) {}
  Cnt(int x) : v(x), k(true) {}
  Cnt(double x, bool kk) : v(x), k(kk) {}
  explicit operator double() const { return v; }
};
inline bool zero(Cnt a) { return a.k && a.v == 0.0; }
inline bool unit(Cnt a) { return a.k && (a.v == 1.0 || a.v == -1.0); }
inline Cnt operator+(Cnt a, Cnt b) { bool k = a.k && b.k; tick(ADD, !k && !zero(a) && !zero(b)); return Cnt(a.v + b.v, k); }
inline Cnt operator-(Cnt a, Cnt b) { bool k = a.k && b.k; tick(ADD, !k && !zero(a) && !zero(b)); return Cnt(a.v - b.v, k); }
inline Cnt operator*(Cnt a, Cnt b) {
  bool k = a.k && b.k;
  if (!k && (zero(a) || zero(b))) return Cnt(a.v * b.v, true);      // x * 0 is the constant 0: nothing downstream of it is work either
  tick(MUL, !k && !unit(a) && !unit(b));
  return Cnt(a.v * b.v, k);
}
inline Cnt operator/(Cnt a, Cnt b) {      // x / const = x * (1/const)
  bool k = a.k && b.k;
  if (!k && zero(a)) return Cnt(a.v / b.v, true);
  tick(b.k ? MUL : DIV, !k && !unit(b));
  return Cnt(a.v / b.v, k);
}
inline Cnt operator-(Cnt a) { return Cnt(-a.v, a.k); }
inline Cnt& operator+=(Cnt& a, Cnt b) { a = a + b; return a; }
inline Cnt& operator-=(Cnt& a, Cnt b) { a = a - b; return a; }
inline Cnt& operator*=(Cnt& a, Cnt b) { a = a * b; return a; }
inline bool operator<(Cnt a, Cnt b) { tick(CMP, !(a.k && b.k)); return a.v < b.v; }
inline bool operator>(Cnt a, Cnt b) { tick(CMP, !(a.k && b.k)); return a.v > b.v; }
inline bool operator<=(Cnt a, Cnt b) { tick(CMP, !(a.k && b.k)); return a.v <= b.v; }
inline bool operator>=(Cnt a, Cnt b) { tick(CMP, !(a.k && b.k)); return a.v >= b.v; }
inline Cnt sqrt(Cnt a) { tick(SQRT, !a.k); return Cnt(std::sqrt(a.v), a.k); }
inline Cnt exp(Cnt a) { tick(EXP, !a.k); return Cnt(std::exp(a.v), a.k); }
inline Cnt tanh(Cnt a) { tick(TANH, !a.k); return Cnt(std::tanh(a.v), a.k); }
inline Cnt pow(Cnt a, Cnt b) { tick(POW, !(a.k && b.k)); return Cnt(std::pow(a.v, b.v), a.k && b.k); }
}  // namespace vho_cnt

namespace vho { using vho_cnt::sqrt; using vho_cnt::exp; using vho_cnt::tanh; using vho_cnt::pow; }
#define VHO_COUNTING_SECTION(x) (vho_cnt::g_section = (x))
#include "vh_oracle.hpp"

extern "C" {
// Runs `warm` uncounted steps (so that no array holds constant-flagged data), then counts `n` steps.
// counts: [4][8] = {other, flux, interface inversions, slopes} x {add, mul, div, cmp, sqrt, exp, pow, tanh}; totals over all cells and steps.
int vho_count_ops(const vho::Params* P, const double* e, const double* u4, const double* pi10, const double* Pi, int warm, int n,
                  long long* counts) {
  if (P->n_batch != 1) return -1;
  vho::Solver<vho_cnt::Cnt> s(*P);
  vho_cnt::g_on = false;
  s.set_initial(e, u4, pi10, Pi);
  for (int i = 0; i < warm; ++i) s.step();
  // the state arrays are data, not constants
  for (int f = 0; f < vho::NQ; ++f) for (auto& x : s.q[f]) x.k = false;
  for (int m = 0; m < 4; ++m) { for (auto& x : s.u[m]) x.k = false; for (auto& x : s.up[m]) x.k = false; }
  for (auto& x : s.e) x.k = false;
  for (auto& x : s.p) x.k = false;
  std::memset(vho_cnt::g_counts, 0, sizeof(vho_cnt::g_counts));
  vho_cnt::g_on = true;
  for (int i = 0; i < n; ++i) s.step();
  vho_cnt::g_on = false;
  std::memcpy(counts, vho_cnt::g_counts, sizeof(vho_cnt::g_counts));
  return (int)s.n_fail;
}
}
