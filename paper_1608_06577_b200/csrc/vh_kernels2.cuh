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
  const double* q; const double* e;
  double* vL; double* vR;        // [3][fstride]: velocity of the state at the cell's low / high face, per direction
  Counters* cnt;
  double t;
};

struct Stage2Args {
  const double* q_in; const double* e_in; const double* p_in; const double* u_in; const double* u_prev;
  const double* q_n;
  const double* vL; const double* vR;
  double* q_out; double* e_out; double* p_out; double* u_out;
  Counters* cnt;
  double t, t_post;
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
  c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + 2);
  return valid;
}

// ------------------------------------------------------------------------------------------------ velocity kernel
template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1, int BX, int BY, int BZ>
__global__ void __launch_bounds__(BX* BY* BZ) velocity_kernel(const __grid_constant__ DevParams P, const __grid_constant__ VelArgs A) {
  int i, j, k;
  long long c;
  const bool valid = cell_index<BX, BY, BZ>(P, i, j, k, c);
  const long long fs = P.fstride;
  const double t2 = MILNE ? A.t * A.t : 1.0;
  const double ht = 0.5 * P.theta;
  const double guess = A.e[c];
  unsigned long long nfail = 0;
  constexpr int ND = TWO_D ? 2 : 3;
#pragma unroll 1
  for (int d = 0; d < ND; ++d) {
    const long long s = (d == 0) ? 1 : ((d == 1) ? (long long)P.NXp : P.plane);
    const int pos = (d == 0) ? i : ((d == 1) ? j : k);
    const int ext = (d == 0) ? P.nx : ((d == 1) ? P.ny : P.nz);
    const double* __restrict__ q = A.q + c;
    // L = state at the low face (q^+_{c-1/2}), R = state at the high face (q^-_{c+1/2})
    double wL[5], wR[5];     // E, Mx, My, Mn, Pi
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const double* f = q + m * fs;
      const double a0 = f[-s], a1 = f[0], a2 = f[s];
      const double h = half_slope2<THETA1>(a1 - a0, a2 - a1, ht);
      wL[m] = a1 - h; wR[m] = a1 + h;
    }
    wL[4] = 0.0; wR[4] = 0.0;
    if (VISC) {
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        const double* f = q + (PTT + m) * fs;
        const double a0 = f[-s], a1 = f[0], a2 = f[s];
        const double h = half_slope2<THETA1>(a1 - a0, a2 - a1, ht);
        wL[m] -= a1 - h; wR[m] -= a1 + h;
      }
      const double* f = q + BPI * fs;
      const double a0 = f[-s], a1 = f[0], a2 = f[s];
      const double h = half_slope2<THETA1>(a1 - a0, a2 - a1, ht);
      wL[4] = a1 - h; wR[4] = a1 + h;
    }
    NewtonState SL, SR;
    SL.E = wL[0]; SL.Pi = wL[4]; SL.M2 = wL[1] * wL[1] + wL[2] * wL[2] + t2 * wL[3] * wL[3];     // :339
    SR.E = wR[0]; SR.Pi = wR[4]; SR.M2 = wR[1] * wR[1] + wR[2] * wR[2] + t2 * wR[3] * wR[3];
    newton_pair<EOS>(P, SL, SR, guess);
    double vl = wL[d + 1] * SL.rden, vr = wR[d + 1] * SR.rden;      // v^r = M_r/(E + P0 + Pi)  (Eqs. 53-54)
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
      double* vL = A.vL + d * fs + c;
      double* vR = A.vR + d * fs + c;
      vL[0] = vl; vR[0] = vr;
      if (pos == 0) vR[-s] = vl;            // state q^-_{-1/2} of the ghost cell equals this cell's low-face state
      if (pos == ext - 1) vL[s] = vr;
    }
  }
  if (valid && nfail) atomicAdd(&A.cnt->n_fail, nfail);
}

// ------------------------------------------------------------------------------------------------ flux divergence
// acc[n] -= dtau/dr (H_{+1/2} - H_{-1/2}) for direction of stride s, with H = cp q^+ + cm q^- where
// cp = (v^+ - a)/2, cm = (v^- + a)/2, a = max(|v^+|,|v^-|)   (Eqs. 61-62 regrouped).
template <bool VISC, bool THETA1>
__device__ __forceinline__ void flux_dir2(const DevParams& P, const double* __restrict__ q, const double* __restrict__ vL,
                                          const double* __restrict__ vR, long long s, double w, double* acc) {
  constexpr int NF = VISC ? NQ : 4;
  const long long fs = P.fstride;
  const double ht = 0.5 * P.theta;
  double cph, cmh, cpl, cml;
  {
    const double vm_lo = vR[-s], vp_lo = vL[0], vm_hi = vR[0], vp_hi = vL[s];
    const double a_lo = fmax(fabs(vm_lo), fabs(vp_lo)), a_hi = fmax(fabs(vm_hi), fabs(vp_hi));
    const double hw = 0.5 * w;
    cph = hw * (vp_hi - a_hi); cmh = hw * (vm_hi + a_hi);
    cpl = hw * (vp_lo - a_lo); cml = hw * (vm_lo + a_lo);
  }
#pragma unroll
  for (int n = 0; n < NF; ++n) {
    const double* f = q + n * fs;
    const double a0 = f[-2 * s], a1 = f[-s], a2 = f[0], a3 = f[s], a4 = f[2 * s];
    const double d0 = a1 - a0, d1 = a2 - a1, d2 = a3 - a2, d3 = a4 - a3;
    const double hm = half_slope2<THETA1>(d0, d1, ht), h0 = half_slope2<THETA1>(d1, d2, ht), hp = half_slope2<THETA1>(d2, d3, ht);
    const double Hhi = fma(cph, a3 - hp, cmh * (a2 + h0));      // q^+_{+1/2} (Eq. 63), q^-_{+1/2} (Eq. 64)
    const double Hlo = fma(cpl, a2 - h0, cml * (a1 + hm));      // q^+_{-1/2} (Eq. 65), q^-_{-1/2} (Eq. 66)
    acc[n] -= Hhi - Hlo;
  }
}

// ------------------------------------------------------------------------------------------------ sources (App. B)
// Adds dtau * J to acc.
template <int EOS, bool VISC, bool MILNE, bool TWO_D>
__device__ __forceinline__ void sources2(const DevParams& P, const Stage2Args& A, long long c, double t, const double* qc, double ec, double pc,
                                         const double* uc, double* acc) {
  const double* __restrict__ q = A.q_in;
  const double* __restrict__ pp = A.p_in;
  const double* __restrict__ uu = A.u_in;
  const long long fs = P.fstride;
  const double t2 = MILNE ? t * t : 1.0;
  const double it = MILNE ? 1.0 / t : 1.0;
  const double it2 = it * it;
  const double dt = P.dtau;
  const long long strides[3] = {1, (long long)P.NXp, P.plane};
  const double hinv[3] = {0.5 * P.inv_dx, 0.5 * P.inv_dy, 0.5 * P.inv_dz};
  double du[4][4];     // du[a][n] = partial_a u^n ; a = 0 is time (backward difference, :424)
  double divv = 0.0;
#pragma unroll
  for (int n = 0; n < 4; ++n) du[0][n] = VISC ? (uc[n] - A.u_prev[n * fs + c]) * P.inv_dtau : 0.0;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (TWO_D && d == 2) {
#pragma unroll
      for (int n = 0; n < 4; ++n) du[3][n] = 0.0;
      continue;
    }
    const long long s = strides[d];
    double Am[4], Ap[4], um[4], up[4];
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      const long long cn = side ? c + s : c - s;
      double* un_ = side ? up : um;
#pragma unroll
      for (int n = 0; n < 4; ++n) un_[n] = (VISC || n == 0 || n == d + 1) ? uu[n * fs + cn] : 0.0;
      const double vi = un_[d + 1] * rcp_fast(un_[0]);
      double Pt = pp[cn];
      double* Ax = side ? Ap : Am;
      if (VISC) {
        Pt += q[BPI * fs + cn];
        const double ptt = q[PTT * fs + cn], ptx = q[PTX * fs + cn], pty = q[PTY * fs + cn], ptn = q[PTN * fs + cn];
        // A^{i nu} = P (v^i delta^nu_tau - g^{i nu}) - v^i pi^{tau nu} + pi^{i nu}   (B.2-B.5)
        if (d == 0) {
          Ax[0] = vi * (Pt - ptt) + ptx;
          Ax[1] = Pt - vi * ptx + q[PXX * fs + cn];
          Ax[2] = -vi * pty + q[PXY * fs + cn];
          Ax[3] = -vi * ptn + q[PXN * fs + cn];
        } else if (d == 1) {
          Ax[0] = vi * (Pt - ptt) + pty;
          Ax[1] = -vi * ptx + q[PXY * fs + cn];
          Ax[2] = Pt - vi * pty + q[PYY * fs + cn];
          Ax[3] = -vi * ptn + q[PYN * fs + cn];
        } else {
          Ax[0] = vi * (Pt - ptt) + ptn;
          Ax[1] = -vi * ptx + q[PXN * fs + cn];
          Ax[2] = -vi * pty + q[PYN * fs + cn];
          Ax[3] = Pt * it2 - vi * ptn + q[PNN * fs + cn];
        }
      } else {
        Ax[0] = vi * Pt;
        Ax[1] = (d == 0) ? Pt : 0.0;
        Ax[2] = (d == 1) ? Pt : 0.0;
        Ax[3] = (d == 2) ? Pt * it2 : 0.0;
      }
      divv += (side ? vi : -vi) * hinv[d];
    }
    const double wd = dt * hinv[d];
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      acc[n] -= (Ap[n] - Am[n]) * wd;
      du[d + 1][n] = (up[n] - um[n]) * hinv[d];
    }
  }
  if (MILNE) {     // G_c (:1013), T^{eta eta} from Eq. 34
    const double Ptc = pc + (VISC ? qc[BPI] : 0.0);
    const double Tnn = (ec + Ptc) * uc[3] * uc[3] + Ptc * it2 + (VISC ? qc[PNN] : 0.0);
    const double wt = dt * it;
    acc[0] -= (qc[TTT] + t2 * Tnn) * wt;
    acc[1] -= qc[TTX] * wt;
    acc[2] -= qc[TTY] * wt;
    acc[3] -= 3.0 * qc[TTN] * wt;
  }
  if (VISC) {
    Kin K;
    kinematics(uc, du[0], du[1], du[2], du[3], t, K);
    double p0, cs2;
    eos_p_cs2<EOS>(P, ec, p0, cs2);
    double Jpi[10], JPi;
    dissipative_sources<EOS>(P, t, uc, K, qc + PTT, qc[BPI], ec, p0, cs2, divv, Jpi, JPi);
    if (P.shear) {
#pragma unroll
      for (int n = 0; n < 10; ++n) acc[PTT + n] = fma(dt, Jpi[n], acc[PTT + n]);
    }
    if (P.bulk) acc[BPI] = fma(dt, JPi, acc[BPI]);
  }
}

// ------------------------------------------------------------------------------------------------ stage kernel
template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1, int STAGE, int BX, int BY, int BZ>
__global__ void __launch_bounds__(BX* BY* BZ) stage_kernel(const __grid_constant__ DevParams P, const __grid_constant__ Stage2Args A) {
  int i, j, k;
  long long c;
  const bool valid = cell_index<BX, BY, BZ>(P, i, j, k, c);
  const long long fs = P.fstride;
  constexpr int NF = VISC ? NQ : 4;
  const double t = A.t;
  unsigned long long nfail = 0, nnonf = 0;
  double minfac = 1.0;

  double qc[NQ], acc[NQ];
#pragma unroll
  for (int n = 0; n < NQ; ++n) { qc[n] = (n < NF) ? A.q_in[n * fs + c] : 0.0; acc[n] = qc[n]; }
  const double ec = A.e_in[c], pc = A.p_in[c];
  double uc[4];
#pragma unroll
  for (int n = 0; n < 4; ++n) uc[n] = A.u_in[n * fs + c];

  // E[w] = w + dtau C[w]  (:413): flux divergence of every direction of extent > 1, then the sources
  if (P.nx > 1) flux_dir2<VISC, THETA1>(P, A.q_in + c, A.vL + c, A.vR + c, 1, P.dtau * P.inv_dx, acc);
  if (P.ny > 1) flux_dir2<VISC, THETA1>(P, A.q_in + c, A.vL + fs + c, A.vR + fs + c, P.NXp, P.dtau * P.inv_dy, acc);
  if (!TWO_D) flux_dir2<VISC, THETA1>(P, A.q_in + c, A.vL + 2 * fs + c, A.vR + 2 * fs + c, P.plane, P.dtau * P.inv_dz, acc);
  sources2<EOS, VISC, MILNE, TWO_D>(P, A, c, t, qc, ec, pc, uc, acc);

  double qo[NQ];
#pragma unroll
  for (int n = 0; n < NQ; ++n) {
    double v = 0.0;
    if (n < NF) {
      v = acc[n];
      if (STAGE == 2) v = 0.5 * (A.q_n[n * fs + c] + v);           // Eq. 70, beta = 1/2
    }
    if (VISC && n >= PTT && n < BPI && !P.shear) v = 0.0;
    if (VISC && n == BPI && !P.bulk) v = 0.0;
    qo[n] = v;
  }

  // Post: Eqs. 52-54, 72 then 73-74 (R8: regulate after the inversion)
  const double tp = A.t_post;
  const double tp2 = MILNE ? tp * tp : 1.0;
  const double E = qo[TTT] - (VISC ? qo[PTT] : 0.0);
  const double Mx = qo[TTX] - (VISC ? qo[PTX] : 0.0), My = qo[TTY] - (VISC ? qo[PTY] : 0.0), Mn = qo[TTN] - (VISC ? qo[PTN] : 0.0);
  const double Pi = VISC ? qo[BPI] : 0.0;
  const double M2 = Mx * Mx + My * My + tp2 * Mn * Mn;
  bool fail;
  const double e = newton_single<EOS>(P, E, M2, Pi, ec, fail);
  if (fail) ++nfail;
  const double p0 = eos_p<EOS>(P, e);
  const double Pt = p0 + Pi;
  const double ut = sqrt_fast((E + Pt) * rcp_fast(e + Pt));      // Eq. 53
  const double inv = rcp_fast((e + Pt) * ut);                    // Eq. 54
  const double u[4] = {ut, Mx * inv, My * inv, Mn * inv};
  if (!(isfinite(e) && isfinite(ut))) ++nnonf;
  if (VISC) {
    const double fac = regulation_factor<MILNE>(P, qo, e, p0, u, tp);
    minfac = fmin(minfac, fac);
#pragma unroll
    for (int n = PTT; n < NQ; ++n) qo[n] *= fac;
  }

  if (valid) {
    // ghost replicas (Eqs. 75-76): the outermost physical cell is copied into both ghost layers of its face
    const bool edge = (i == 0) | (i == P.nx - 1) | (j == 0) | (j == P.ny - 1) | (!TWO_D && ((k == 0) | (k == P.nz - 1)));
    const long long sy = P.NXp, sz = P.plane;
    auto put = [&](double* a, double v) {
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
    for (int n = 0; n < NQ; ++n) put(A.q_out + n * fs, qo[n]);
    put(A.e_out, e);
    put(A.p_out, p0);
#pragma unroll
    for (int n = 0; n < 4; ++n) put(A.u_out + n * fs, u[n]);
  }
  flush_counters(A.cnt, valid ? nfail : 0ull, valid ? nnonf : 0ull, valid ? minfac : 1.0);
}

}  // namespace vh
