// vh_math.cuh -- FP64 building blocks of the product kernels: branch-free reciprocal / square roots built on the MUFU
// seeds (a few DFMA instead of the IEEE slow-path calls), the minmod-limited half slope (Eqs. 67-68) with the sign
// logic on the integer pipe, and the paired Newton-Raphson inversion of Eq. 72.  Independent of the CPU test code.
#pragma once
#include "vh_device.cuh"

namespace vh {

// (rcp_fast, rcp_half, rsqrt_fast, sqrt_fast live in vh_device.cuh: the EOS lookup uses them too)

// (dr/2) * minmod(theta d1/dr, (d1+d2)/(2 dr), theta d2/dr) with d1 = q0 - qm, d2 = qp - q0   (Eqs. 67-68, R10).
// When d1, d2 have the same sign the centred difference has it too and |d1+d2|/2 = (|d1|+|d2|)/2; for theta = 1 it lies
// between the one-sided ones and drops out.  A zero one-sided difference gives min = 0, so only the sign bits are compared.
template <bool THETA1>
__device__ __forceinline__ real half_slope2(real d1, real d2, real half_theta) {
  const real a1 = fabs(d1), a2 = fabs(d2);
  real m = (a1 < a2) ? a1 : a2;
  if (THETA1) {
    m *= real(0.5);
  } else {
    m *= half_theta;
    const real b = real(0.25) * (a1 + a2);
    m = (b < m) ? b : m;
  }
  return sign_differs(d1, d2) ? real(0.0) : copysign(m, d1);
}

// ---------------------------------------------------------------- paired Newton-Raphson on Eq. 72 (R6)
// Two independent states are iterated together so that their dependent FP64 chains interleave.  Same tolerance, cap and failure
// semantics as invert_energy().  The tolerance |de| <= rtol |e| (R6) is tested one iteration early: Newton's method on Eq. 72 converges
// quadratically, |de_next| <= C de^2 with C = max|f''|/(2 min f') <= 0.2/(E+P) + 0.21/e0 (M^2 <= (E+P)^2, f' >= 1 - cs2 >= 0.65, P'' of
// the EOS), so |de| <= newton_stop |e| with newton_stop = 0.1 sqrt(rtol) bounds the NEXT correction - the one the oracle still performs and
// then finds below rtol - by 1.3e-14 |e| for e <= 60 e0: same root to the same tolerance, one evaluation of the EOS fewer per state.
struct NewtonState {
  real E, M2, Pi;     // inputs
  real e;             // iterate
  real p, rden;       // P0 and 1/(E + P0 + Pi) extrapolated to the returned e (valid when !fail)
  bool fail;
};

// (guessA, guessB: e of the cells the two states were extrapolated from, R6)
template <int EOS>
__device__ __forceinline__ void newton_pair(const DevParams& P, NewtonState& A, NewtonState& B, real guessA, real guessB) {
  const bool gokA = (guessA > real(0.0)) && isfinite(guessA), gokB = (guessB > real(0.0)) && isfinite(guessB);
  // (one finiteness test on the sum: it is finite exactly when E, M2 and Pi all are, short of an overflow that no state reaches)
  bool badA = !(A.E > real(0.0)) || !isfinite(A.E + A.M2 + A.Pi);
  bool badB = !(B.E > real(0.0)) || !isfinite(B.E + B.M2 + B.Pi);
  A.e = gokA ? guessA : A.E;
  B.e = gokB ? guessB : B.E;
  bool doneA = badA, doneB = badB, convA = false, convB = false;
  real pA = real(0.0), cA = real(0.0), rA = real(0.0), dA = real(0.0), pB = real(0.0), cB = real(0.0), rB = real(0.0), dB = real(0.0);      // last iterate's P0, cs2, 1/(E + P0 + Pi), correction
  for (int it = 0; it < P.newton_max_iter; ++it) {
    if (__all_sync(0xffffffffu, doneA && doneB)) break;
    eos_p_cs2<EOS>(P, A.e, pA, cA);
    eos_p_cs2<EOS>(P, B.e, pB, cB);
    rA = rcp_fast(A.E + pA + A.Pi); rB = rcp_fast(B.E + pB + B.Pi);
    const real fA = A.e - A.E + A.M2 * rA, fB = B.e - B.E + B.M2 * rB;
    const real gA = fma(-A.M2 * cA, rA * rA, real(1.0)), gB = fma(-B.M2 * cB, rB * rB, real(1.0));
    dA = fA * rcp_half(gA); dB = fB * rcp_half(gB);      // f' in (0, 1] only steers the iteration: 40 bits are plenty
    const real eA = A.e - dA, eB = B.e - dB;
    // A state that has converged keeps being iterated while the warp is still busy: at the root the correction is at rounding
    // level, so this costs no accuracy and saves the selects that would freeze it.  Only a state with bad input is held (its
    // iterates are not finite and it takes the failure path below anyway).
    A.e = badA ? A.e : eA;
    B.e = badB ? B.e : eB;
    if (fabs(dA) <= P.newton_stop * fabs(eA)) { convA = true; doneA = true; }
    if (fabs(dB) <= P.newton_stop * fabs(eB)) { convB = true; doneB = true; }
  }
  // P0 and 1/(E + P0 + Pi) at the returned e, extrapolated from the last iterate over its correction (once, after the loop):
  // P0(e - d) = P0(e) - cs2 d + O(d^2), 1/(den - cs2 d) = r + r^2 cs2 d + O(d^2), |d| <= rtol e at convergence
  A.p = fma(-cA, dA, pA);
  B.p = fma(-cB, dB, pB);
  A.rden = fma(rA * rA, cA * dA, rA);
  B.rden = fma(rB * rB, cB * dB, rB);
  A.fail = badA || !convA || !(A.e > real(0.0)) || !isfinite(A.e);
  B.fail = badB || !convB || !(B.e > real(0.0)) || !isfinite(B.e);
  if (A.fail) { A.e = fmax(A.E, tiny_e()); A.p = eos_p<EOS>(P, A.e); A.rden = real(1.0) / (A.E + A.p + A.Pi); }
  if (B.fail) { B.e = fmax(B.E, tiny_e()); B.p = eos_p<EOS>(P, B.e); B.rden = real(1.0) / (B.E + B.p + B.Pi); }
}

// single state (cell inversion in the stage epilogue)
template <int EOS>
__device__ __forceinline__ real newton_single(const DevParams& P, real E, real M2, real Pi, real guess, bool& fail) {
  const bool bad = !(E > real(0.0)) || !isfinite(E + M2 + Pi);      // (see newton_pair)
  real e = ((guess > real(0.0)) && isfinite(guess)) ? guess : E;
  bool done = bad, conv = false;
  for (int it = 0; it < P.newton_max_iter; ++it) {
    if (__all_sync(0xffffffffu, done)) break;
    real p, c;
    eos_p_cs2<EOS>(P, e, p, c);
    const real r = rcp_fast(E + p + Pi);
    const real f = e - E + M2 * r;
    const real g = fma(-M2 * c, r * r, real(1.0));
    const real d = f * rcp_half(g);      // (f' only steers the iteration)
    const real en = e - d;
    e = bad ? e : en;      // (a converged cell keeps iterating with its warp: see newton_pair)
    if (fabs(d) <= P.newton_stop * fabs(en)) { conv = true; done = true; }
  }
  fail = bad || !conv || !(e > real(0.0)) || !isfinite(e);
  if (fail) e = (tiny_e() > E) ? tiny_e() : E;      // max(E, tiny) that keeps a NaN E (fmax would drop it and hide the cell from n_nonfinite)
  return e;
}

// u^tau = sqrt((E + P)/(e + P)) of Eq. 53 and whether it is a number: the IEEE square root of a negative, infinite or NaN quotient is
// not finite, which sqrt_fast() alone would hide (it returns 0 there); such a cell is counted in n_nonfinite and carries NaN
__device__ __forceinline__ real u_tau_checked(real E_plus_P, real e_plus_P, bool& finite) {
  const real x = E_plus_P * rcp_fast(e_plus_P);
  finite = (x >= real(0.0)) && (x < inf_r());
  return finite ? sqrt_fast(x) : nan_r();
}

// clip of a failed state's velocity (R6)
__device__ __forceinline__ real clip_velocity(real v) {
  if (!(fabs(v) < real(1.0))) v = (v > real(0.0)) ? clip_one() : ((v < real(0.0)) ? -clip_one() : real(0.0));
  return v;
}

}  // namespace vh

namespace vh {

// minmod(d1, d2) of Eqs. 67-68 for theta = 1 (the centred difference lies between the one-sided ones and drops out):
// the argument of smaller magnitude when both have the same sign, else 0 (R10).  One DSETP, the rest on the ALU pipe;
// the factor 1/2 of the half-cell extrapolation is folded into the caller's FMA.
__device__ __forceinline__ real minmod2(real d1, real d2) {
  const real t = (fabs(d1) < fabs(d2)) ? d1 : d2;
  return zero_if(sign_differs(d1, d2), t);
}
// general theta: minmod(theta d1, (d1 + d2)/2, theta d2); `theta` in [1, 2]
__device__ __forceinline__ real minmod3(real d1, real d2, real theta) {
  const real t = theta * minmod2(d1, d2);
  const real c = real(0.5) * (d1 + d2);
  return (fabs(c) < fabs(t)) ? c : t;       // t = 0 (opposite signs) always wins
}
template <bool THETA1> __device__ __forceinline__ real minmod_slope(real d1, real d2, real theta) {
  return THETA1 ? minmod2(d1, d2) : minmod3(d1, d2, theta);
}

}  // namespace vh
