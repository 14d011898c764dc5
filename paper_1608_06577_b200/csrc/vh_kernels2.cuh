// vh_kernels2.cuh -- default stage pipeline ("split"): two kernels per Euler stage.
//
//   velocity_kernel : per cell and direction, the two reconstructed states the cell owns (q^+_{c-1/2} = q_c - h_c and
//                     q^-_{c+1/2} = q_c + h_c, Eqs. 63-66) are inverted (Eq. 72) ONCE, as a pair, and their propagation
//                     velocities v_r = M_r/(E+P) are stored (6 doubles per cell).  Alg. 3 (:667-672) does this inversion in
//                     every thread for both of its interfaces, i.e. twice per state.
//   stage_kernel    : KT flux divergence for the 15 fields from those velocities (Eqs. 59-62), all source terms (App. B),
//                     the Euler update / convex combination (Eqs. 69-71), the cell inversion (Eqs. 52-54), the
//                     regularisation (Eqs. 73-74) and the ghost-cell replicas (Eqs. 75-76) in one pass; each field is
//                     written once.
// See DESIGN.md "Kernels" for the instruction budget that led to this split.
#pragma once
#include "vh_kernels.cuh"
#include "vh_math.cuh"

namespace vh {

struct VelArgs {
  const real* q; const real* e;
  real* vL; real* vR;        // [3][fstride]: velocity of the state at the cell's low / high face, per direction
  Counters* cnt;
  real t;
};

struct Stage2Args {
  const real* q_in; const real* e_in; const real* p_in; const real* u_in; const real* u_prev;
  const real* q_n;
  const real* vL; const real* vR;
  real* q_out; real* e_out; real* p_out; real* u_out;
  Counters* cnt;
  real t, t_post;
  real* regfac;      // see StageArgs
};

template <int BX, int BY, int BZ>
__device__ __forceinline__ bool cell_index(const DevParams& P, int& i, int& j, int& k, long long& c) {
  i = blockIdx.x * BX + threadIdx.x;
  j = blockIdx.y * BY + threadIdx.y;
  const int nzb = (P.nz + BZ - 1) / BZ;
  const int b = blockIdx.z / nzb;
  k = (blockIdx.z % nzb) * BZ + threadIdx.z;
  const bool valid = (i < P.nx) && (j < P.ny) && (k < P.nz);
  i = min(i, P.nx - 1); j = min(j, P.ny - 1); k = min(k, P.nz - 1);
  c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  return valid;
}

// ------------------------------------------------------------------------------------------------ velocity kernel
template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1, int BX, int BY, int BZ>
__global__ void __launch_bounds__(BX* BY* BZ, 4) velocity_kernel(const __grid_constant__ DevParams P, const __grid_constant__ VelArgs A) {
  int i, j, k;
  long long c;
  const bool valid = cell_index<BX, BY, BZ>(P, i, j, k, c);
  const long long fs = P.fstride;
  const real t2 = MILNE ? A.t * A.t : real(1.0);
  const real ht = real(0.5) * P.theta;
  const real guess = A.e[c];
  unsigned long long nfail = 0;
  constexpr int ND = TWO_D ? 2 : 3;
#pragma unroll 1
  for (int d = 0; d < ND; ++d) {
    const long long s = (d == 0) ? 1 : ((d == 1) ? (long long)P.NXp : P.plane);
    const int pos = (d == 0) ? i : ((d == 1) ? j : k);
    const int ext = (d == 0) ? P.nx : ((d == 1) ? P.ny : P.nz);
    const real* __restrict__ q = A.q + c;
    // L = state at the low face (q^+_{c-1/2}), R = state at the high face (q^-_{c+1/2})
    real wL[5], wR[5];     // E, Mx, My, Mn, Pi
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const real* f = q + m * fs;
      const real a0 = f[-s], a1 = f[0], a2 = f[s];
      const real h = half_slope2<THETA1>(a1 - a0, a2 - a1, ht);
      wL[m] = a1 - h; wR[m] = a1 + h;
    }
    wL[4] = real(0.0); wR[4] = real(0.0);
    if (VISC) {
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        const real* f = q + (PTT + m) * fs;
        const real a0 = f[-s], a1 = f[0], a2 = f[s];
        const real h = half_slope2<THETA1>(a1 - a0, a2 - a1, ht);
        wL[m] -= a1 - h; wR[m] -= a1 + h;
      }
      const real* f = q + BPI * fs;
      const real a0 = f[-s], a1 = f[0], a2 = f[s];
      const real h = half_slope2<THETA1>(a1 - a0, a2 - a1, ht);
      wL[4] = a1 - h; wR[4] = a1 + h;
    }
    NewtonState SL, SR;
    SL.E = wL[0]; SL.Pi = wL[4]; SL.M2 = wL[1] * wL[1] + wL[2] * wL[2] + t2 * wL[3] * wL[3];     // :339
    SR.E = wR[0]; SR.Pi = wR[4]; SR.M2 = wR[1] * wR[1] + wR[2] * wR[2] + t2 * wR[3] * wR[3];
    newton_pair<EOS>(P, SL, SR, guess, guess);
    real vl = wL[d + 1] * SL.rden, vr = wR[d + 1] * SR.rden;      // v^r = M_r/(E + P0 + Pi)  (Eqs. 53-54)
    if (SL.fail) vl = clip_velocity(vl);
    if (SR.fail) vr = clip_velocity(vr);
    // status counter: every state of every interface once.  The states of the two outermost interfaces that belong to ghost
    // cells repeat the boundary cell's own state (outflow ghosts, Eqs. 75-76, give a zero slope there), so the boundary cell
    // counts twice; nothing is counted along a direction of extent 1.
    if (ext > 1) {
      nfail += (SL.fail ? 1u : 0u) + (SR.fail ? 1u : 0u);
      if (pos == 0 && SL.fail) ++nfail;
      if (pos == ext - 1 && SR.fail) ++nfail;
    }
    if (valid) {
      real* vL = A.vL + d * fs + c;
      real* vR = A.vR + d * fs + c;
      vL[0] = vl; vR[0] = vr;
      if (pos == 0) vR[-s] = vl;            // state q^-_{-1/2} of the ghost cell equals this cell's low-face state
      if (pos == ext - 1) vL[s] = vr;
    }
  }
  if (valid && nfail) atomicAdd(&A.cnt->n_fail, nfail);
}

// ------------------------------------------------------------------------------------------------ flux divergence
// acc[n] -= dtau/dr (H_{+1/2} - H_{-1/2}) for direction of stride s, with H = cp q^+ + cm q^- where
// cp = (v^+ - a)/2, cm = (v^- + a)/2, a = max(|v^+|,|v^-|)   (Eqs. 61-62 regrouped; dtau/dr folded into cp, cm).
template <bool VISC, bool THETA1>
__device__ __forceinline__ void flux_dir2(const DevParams& P, const real* __restrict__ q, const real* __restrict__ vL,
                                          const real* __restrict__ vR, long long s, real w, real* acc) {
  constexpr int NF = VISC ? NQ : 4;
  const long long fs = P.fstride;
  const real ht = real(0.5) * P.theta;
  real cph, cmh, cpl, cml;
  {
    const real vm_lo = vR[-s], vp_lo = vL[0], vm_hi = vR[0], vp_hi = vL[s];
    const real a_lo = fmax(fabs(vm_lo), fabs(vp_lo)), a_hi = fmax(fabs(vm_hi), fabs(vp_hi));
    const real hw = real(0.5) * w;
    cph = hw * (a_hi - vp_hi); cmh = -hw * (vm_hi + a_hi);      // -dtau/dr * (cp, cm) of the high face
    cpl = hw * (vp_lo - a_lo); cml = hw * (vm_lo + a_lo);       // +dtau/dr * (cp, cm) of the low face
  }
#pragma unroll
  for (int n = 0; n < NF; ++n) {
    const real* f = q + n * fs;
    const real a0 = f[-2 * s], a1 = f[-s], a2 = f[0], a3 = f[s], a4 = f[2 * s];
    const real d0 = a1 - a0, d1 = a2 - a1, d2 = a3 - a2, d3 = a4 - a3;
    const real hm = half_slope2<THETA1>(d0, d1, ht), h0 = half_slope2<THETA1>(d1, d2, ht), hp = half_slope2<THETA1>(d2, d3, ht);
    real r = acc[n];
    r = fma(cph, a3 - hp, r);      // q^+_{+1/2} (Eq. 63)
    r = fma(cmh, a2 + h0, r);      // q^-_{+1/2} (Eq. 64)
    r = fma(cpl, a2 - h0, r);      // q^+_{-1/2} (Eq. 65)
    r = fma(cml, a1 + hm, r);      // q^-_{-1/2} (Eq. 66)
    acc[n] = r;
  }
}

// ------------------------------------------------------------------------------------------------ conservation sources
// acc[0..3] += dtau (S_c + G_c) (B.2-B.5, :1013) and the velocity gradients du[a][n] = partial_a u^n, div v (:424).
template <bool VISC, bool MILNE, bool TWO_D>
__device__ __forceinline__ void conservation_sources2(const DevParams& P, const Stage2Args& A, long long c, real t, const real* uc,
                                                      real* acc, real du[4][4], real& divv) {
  const real* __restrict__ q = A.q_in;
  const real* __restrict__ pp = A.p_in;
  const real* __restrict__ uu = A.u_in;
  const long long fs = P.fstride;
  const real t2 = MILNE ? t * t : real(1.0);
  const real it = MILNE ? rcp_fast(t) : real(1.0);
  const real it2 = it * it;
  const real dt = P.dtau;
  const long long strides[3] = {1, (long long)P.NXp, P.plane};
  const real hinv[3] = {real(0.5) * P.inv_dx, real(0.5) * P.inv_dy, real(0.5) * P.inv_dz};
  divv = real(0.0);
#pragma unroll
  for (int n = 0; n < 4; ++n) du[0][n] = VISC ? (uc[n] - A.u_prev[n * fs + c]) * P.inv_dtau : real(0.0);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (TWO_D && d == 2) {
#pragma unroll
      for (int n = 0; n < 4; ++n) du[3][n] = real(0.0);
      continue;
    }
    const long long s = strides[d];
    real Am[4], Ap[4], um[4], up[4];
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      const long long cn = side ? c + s : c - s;
      real* un_ = side ? up : um;
#pragma unroll
      for (int n = 0; n < 4; ++n) un_[n] = (VISC || n == 0 || n == d + 1) ? uu[n * fs + cn] : real(0.0);
      const real vi = un_[d + 1] * rcp_fast(un_[0]);
      real Pt = pp[cn];
      real* Ax = side ? Ap : Am;
      if (VISC) {
        Pt += q[BPI * fs + cn];
        const real ptt = q[PTT * fs + cn], ptx = q[PTX * fs + cn], pty = q[PTY * fs + cn], ptn = q[PTN * fs + cn];
        // A^{i nu} = P (v^i delta^nu_tau - g^{i nu}) - v^i pi^{tau nu} + pi^{i nu}   (B.2-B.5)
        if (d == 0) {
          Ax[0] = fma(vi, Pt - ptt, ptx);
          Ax[1] = fma(-vi, ptx, Pt + q[PXX * fs + cn]);
          Ax[2] = fma(-vi, pty, q[PXY * fs + cn]);
          Ax[3] = fma(-vi, ptn, q[PXN * fs + cn]);
        } else if (d == 1) {
          Ax[0] = fma(vi, Pt - ptt, pty);
          Ax[1] = fma(-vi, ptx, q[PXY * fs + cn]);
          Ax[2] = fma(-vi, pty, Pt + q[PYY * fs + cn]);
          Ax[3] = fma(-vi, ptn, q[PYN * fs + cn]);
        } else {
          Ax[0] = fma(vi, Pt - ptt, ptn);
          Ax[1] = fma(-vi, ptx, q[PXN * fs + cn]);
          Ax[2] = fma(-vi, pty, q[PYN * fs + cn]);
          Ax[3] = fma(-vi, ptn, fma(Pt, it2, q[PNN * fs + cn]));
        }
      } else {
        Ax[0] = vi * Pt;
        Ax[1] = (d == 0) ? Pt : real(0.0);
        Ax[2] = (d == 1) ? Pt : real(0.0);
        Ax[3] = (d == 2) ? Pt * it2 : real(0.0);
      }
      divv = fma(side ? vi : -vi, hinv[d], divv);
    }
    const real wd = dt * hinv[d];
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      acc[n] = fma(Am[n] - Ap[n], wd, acc[n]);
      du[d + 1][n] = (up[n] - um[n]) * hinv[d];
    }
  }
  if (MILNE) {     // G_c (:1013), T^{eta eta} from Eq. 34
    const real ec = A.e_in[c], pc = pp[c];
    const real Ptc = pc + (VISC ? q[BPI * fs + c] : real(0.0));
    const real Tnn = fma((ec + Ptc) * uc[3], uc[3], fma(Ptc, it2, VISC ? q[PNN * fs + c] : real(0.0)));
    const real wt = dt * it;
    acc[0] = fma(-wt, fma(t2, Tnn, q[TTT * fs + c]), acc[0]);
    acc[1] = fma(-wt, q[TTX * fs + c], acc[1]);
    acc[2] = fma(-wt, q[TTY * fs + c], acc[2]);
    acc[3] = fma(-real(3.0) * wt, q[TTN * fs + c], acc[3]);
  }
}

// ------------------------------------------------------------------------------------------------ dissipative sources
// J = S + G for pi^{mu nu} (10) and Pi (B.10-B.12, Eqs. 39-46), one component at a time: emit(slot, J).
template <int EOS, bool MILNE, class Emit>
__device__ __forceinline__ void dissipative_sources2(const DevParams& P, real t, const real u[4], const Kin& K, const real pi[10], real Pi,
                                                     real e, real divv, Emit emit) {
  const real t2 = MILNE ? t * t : real(1.0);                                       // metric factor
  const real it = MILNE ? rcp_fast(t) : real(0.0), ct = MILNE ? t : real(0.0);           // Christoffel symbols (0 in the Cartesian mode, R12)
  // transport coefficients (Eqs. 10-16; R14)
  real p, cs2;
  eos_p_cs2<EOS>(P, e, p, cs2);
  const real T = (EOS == 2) ? eos_temperature<EOS>(P, e) : sqrt_fast(sqrt_fast(e * P.eos_a_inv));
  const real itp = fmin(T * P.inv_ctaupi_etas, P.relax_clamp);
  const real eotp2 = real(2.0) * (e + p) * P.inv_ctaupi;
  const real zs = zeta_over_s(P, T);
  const real b = (real(1.0) / real(3.0)) - cs2;
  real itP = (zs > real(0.0)) ? T * b * b * P.inv_ctauPi / zs : inf_r();
  itP = fmin(itP, P.relax_clamp);
  const real zotP = (zs > real(0.0)) ? zs * ((e + p) / T) * itP : real(0.0);
  const real lPp = P.lambda_Pipi_coef * b;
  const real iut = rcp_fast(u[0]);
  const real ut = u[0], un = u[3];

  // pi^{mu nu} sigma_{mu nu}: symmetric double contraction with the metric weights of g = diag(1,-1,-1,-t2)
  const real* S = K.sig;
  const real pisig = pi[0] * S[0] - real(2.0) * (pi[1] * S[1] + pi[2] * S[2]) + pi[4] * S[4] + real(2.0) * pi[5] * S[5] + pi[7] * S[7] +
                       t2 * (real(2.0) * (pi[6] * S[6] + pi[8] * S[8] - pi[3] * S[3]) + t2 * pi[9] * S[9]);
  // A^mu = pi^{lambda mu} Du_lambda (Eq. 43)
  real Av[4];
#pragma unroll
  for (int m = 0; m < 4; ++m)
    Av[m] = pi[sym(0, m)] * K.Du[0] + pi[sym(1, m)] * K.Du[1] + pi[sym(2, m)] * K.Du[2] + pi[sym(3, m)] * K.Du[3];
  // g_l W^{l n} and g_l sigma^{l n} (rows scaled by the metric)
  real gW[4][4], gS[4][4];
  {
    const real W01 = K.W[0], W02 = K.W[1], W03 = K.W[2], W12 = K.W[3], W13 = K.W[4], W23 = K.W[5];
    gW[0][0] = real(0.0);      gW[0][1] = W01;       gW[0][2] = W02;       gW[0][3] = W03;
    gW[1][0] = W01;      gW[1][1] = real(0.0);       gW[1][2] = -W12;      gW[1][3] = -W13;
    gW[2][0] = W02;      gW[2][1] = W12;       gW[2][2] = real(0.0);       gW[2][3] = -W23;
    gW[3][0] = t2 * W03; gW[3][1] = t2 * W13;  gW[3][2] = t2 * W23;  gW[3][3] = real(0.0);
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      gS[0][n] = S[sym(0, n)]; gS[1][n] = -S[sym(1, n)]; gS[2][n] = -S[sym(2, n)]; gS[3][n] = -t2 * S[sym(3, n)];
    }
  }
  const real gi[4] = {real(1.0), -real(1.0), -real(1.0), MILNE ? -it * it : -real(1.0)};
  const real third_pisig = (real(1.0) / real(3.0)) * pisig;
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = m; n < 4; ++n) {
      const int s = sym(m, n);
      real B = real(0.0), C = real(0.0);     // B = pi^{m l} g_l W^{l n} + (m<->n) ; C = pi^{m l} g_l sigma^{l n} + (m<->n)
#pragma unroll
      for (int l = 0; l < 4; ++l) {
        if (l != n) B = fma(pi[sym(m, l)], gW[l][n], B);
        if (l != m) B = fma(pi[sym(n, l)], gW[l][m], B);
        C = fma(pi[sym(m, l)], gS[l][n], C);
        C = fma(pi[sym(n, l)], gS[l][m], C);
      }
      const real Dmn = ((m == n) ? gi[m] : real(0.0)) - u[m] * u[n];
      const real I1 = u[n] * Av[m] + u[m] * Av[n];                          // Eq. 43
      const real I4 = real(0.5) * C - Dmn * third_pisig;                          // Eq. 46
      // Eq. 42: I1 + delta_pipi theta pi - I3 + tau_pipi I4 - lambda_piPi Pi sigma ; I3 = kVorticitySign * B (Eq. 45, R4)
      real Ipi = I1 + P.delta_pipi * K.theta * pi[s] - kVorticitySign * B + P.tau_pipi * I4 - P.lambda_piPi * Pi * S[s];
      // G_pi = u^a Gamma^mu_{ab} pi^{b nu} + (mu<->nu)  (:300; R1, R2)
      real G = real(0.0);
      if (s == 0) G = real(2.0) * ct * un * pi[3];
      if (s == 1) G = ct * un * pi[6];
      if (s == 2) G = ct * un * pi[8];
      if (s == 3) G = ct * un * pi[9] + (ut * pi[3] + un * pi[0]) * it;
      if (s == 6) G = (ut * pi[6] + un * pi[1]) * it;
      if (s == 8) G = (ut * pi[8] + un * pi[2]) * it;
      if (s == 9) G = real(2.0) * (ut * pi[9] + un * pi[3]) * it;
      emit(PTT + s, fma(fma(eotp2, S[s], -fma(pi[s], itp, Ipi + G)), iut, pi[s] * divv));      // B.11, B.9
    }
  const real IPi = P.delta_PiPi * Pi * K.theta - lPp * pisig;                                // Eq. 41
  emit(BPI, fma(-fma(zotP, K.theta, fma(Pi, itP, IPi)), iut, Pi * divv));                       // B.10
}

// ------------------------------------------------------------------------------------------------ stage kernel
// Per-thread phases: (1) flux divergence, (2) conservation sources + velocity gradients, (3) kinematics + dissipative
// sources, (4) cell inversion + regularisation, (5) stores with ghost replicas.  The 15 running values q + dtau C[q] are
// parked in shared memory (one conflict-free slot per thread and field) between phases so that the register file holds
// two blocks per SM.
template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1, int STAGE, int BX, int BY, int BZ, int MINB>
__global__ void __launch_bounds__(BX* BY* BZ, MINB) stage_kernel(const __grid_constant__ DevParams P, const __grid_constant__ Stage2Args A) {
  constexpr int NT = BX * BY * BZ;
  constexpr int NF = VISC ? NQ : 4;
  __shared__ real park[NF][NT];
  const int tid = threadIdx.x + BX * (threadIdx.y + BY * threadIdx.z);
  int i, j, k;
  long long c;
  const bool valid = cell_index<BX, BY, BZ>(P, i, j, k, c);
  const long long fs = P.fstride;
  const real t = A.t;
  unsigned long long nfail = 0, nnonf = 0;
  real minfac = real(1.0);

  real uc[4];
#pragma unroll
  for (int n = 0; n < 4; ++n) uc[n] = A.u_in[n * fs + c];
  {
    real acc[NF];
#pragma unroll
    for (int n = 0; n < NF; ++n) acc[n] = A.q_in[n * fs + c];
    // E[w] = w + dtau C[w]  (:413): flux divergence of every direction of extent > 1
    if (P.nx > 1) flux_dir2<VISC, THETA1>(P, A.q_in + c, A.vL + c, A.vR + c, 1, P.dtau * P.inv_dx, acc);
    if (P.ny > 1) flux_dir2<VISC, THETA1>(P, A.q_in + c, A.vL + fs + c, A.vR + fs + c, P.NXp, P.dtau * P.inv_dy, acc);
    if (!TWO_D) flux_dir2<VISC, THETA1>(P, A.q_in + c, A.vL + 2 * fs + c, A.vR + 2 * fs + c, P.plane, P.dtau * P.inv_dz, acc);
    if (VISC) {
#pragma unroll
      for (int n = 4; n < NF; ++n) park[n][tid] = acc[n];
    }
    real du[4][4], divv;
    conservation_sources2<VISC, MILNE, TWO_D>(P, A, c, t, uc, acc, du, divv);
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      real v = acc[n];
      if (STAGE == 2) v = real(0.5) * (A.q_n[n * fs + c] + v);           // Eq. 70, beta = 1/2
      park[n][tid] = v;
    }
    if (VISC) {
      Kin K;
      kinematics<MILNE>(uc, du[0], du[1], du[2], du[3], t, K);
      real pi[10];
#pragma unroll
      for (int n = 0; n < 10; ++n) pi[n] = A.q_in[(PTT + n) * fs + c];
      const real Pi = A.q_in[BPI * fs + c];
      const real ec = A.e_in[c];
      dissipative_sources2<EOS, MILNE>(P, t, uc, K, pi, Pi, ec, divv, [&](int slot, real J) {
        const bool on = (slot == BPI) ? (P.bulk != 0) : (P.shear != 0);
        real v = fma(P.dtau, J, park[slot][tid]);
        if (STAGE == 2) v = real(0.5) * (A.q_n[slot * fs + c] + v);      // Eq. 70
        park[slot][tid] = on ? v : real(0.0);
      });
    }
  }

  // Post: Eqs. 52-54, 72 then 73-74 (R8: regulate after the inversion)
  const real tp = A.t_post;
  const real tp2 = MILNE ? tp * tp : real(1.0);
  const real E = park[TTT][tid] - (VISC ? park[PTT][tid] : real(0.0));
  const real Mx = park[TTX][tid] - (VISC ? park[PTX][tid] : real(0.0)), My = park[TTY][tid] - (VISC ? park[PTY][tid] : real(0.0)),
               Mn = park[TTN][tid] - (VISC ? park[PTN][tid] : real(0.0));
  const real Pi = VISC ? park[BPI][tid] : real(0.0);
  const real M2 = Mx * Mx + My * My + tp2 * Mn * Mn;
  bool fail;
  const real e = newton_single<EOS>(P, E, M2, Pi, A.e_in[c], fail);
  if (fail) ++nfail;
  const real p0 = eos_p<EOS>(P, e);
  const real Pt = p0 + Pi;
  bool ut_ok;
  const real ut = u_tau_checked(E + Pt, e + Pt, ut_ok);        // Eq. 53
  const real inv = rcp_fast((e + Pt) * ut);                    // Eq. 54
  const real u[4] = {ut, Mx * inv, My * inv, Mn * inv};
  if (!(isfinite(e) && ut_ok)) ++nnonf;
  real fac = real(1.0);
  if (VISC) {
    real qo[NQ];
#pragma unroll
    for (int n = PTT; n < NQ; ++n) qo[n] = park[n][tid];
    fac = regulation_factor<MILNE>(P, qo, e, p0, u, tp);
    minfac = fmin(minfac, fac);
    if (A.regfac && valid) A.regfac[c] = fac;
  }

  if (valid) {
    // ghost replicas (Eqs. 75-76): the outermost physical cell is copied into both ghost layers of its face
    const bool edge = (i == 0) | (i == P.nx - 1) | (j == 0) | (j == P.ny - 1) | (!TWO_D && ((k == 0) | (k == P.nz - 1)));
    const long long sy = P.NXp, sz = P.plane;
    auto put = [&](real* a, real v) {
      a[c] = v;
      if (edge) {
        if (i == 0) { a[c - 1] = v; a[c - 2] = v; }
        if (i == P.nx - 1) { a[c + 1] = v; a[c + 2] = v; }
        if (j == 0) { a[c - sy] = v; a[c - 2 * sy] = v; }
        if (j == P.ny - 1) { a[c + sy] = v; a[c + 2 * sy] = v; }
        if (!TWO_D) {
          if (k == 0) { a[c - sz] = v; a[c - 2 * sz] = v; }
          if (k == P.nz - 1) { a[c + sz] = v; a[c + 2 * sz] = v; }
        }
      }
    };
#pragma unroll
    for (int n = 0; n < NQ; ++n) put(A.q_out + n * fs, (n < NF) ? ((n >= PTT) ? park[n][tid] * fac : park[n][tid]) : real(0.0));
    put(A.e_out, e);
    put(A.p_out, p0);
#pragma unroll
    for (int n = 0; n < 4; ++n) put(A.u_out + n * fs, u[n]);
  }
  flush_counters(A.cnt, valid ? nfail : 0ull, valid ? nnonf : 0ull, valid ? minfac : real(1.0), *(volatile unsigned long long*)&A.cnt->min_reg_bits);
}

}  // namespace vh
