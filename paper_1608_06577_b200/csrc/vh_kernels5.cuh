// vh_kernels5.cuh -- reduced-storage mode (vh_params.storage = 1; PAPER.md:476 with Eqs. 47-51, :318-331; reading R22).
//
// "[The global memory] can be reduced by simply propagating only the independent components of pi^{mu nu} (five) and u^mu (three), with the
// remaining components determined algebraically."  State arrays per time level: ten conserved fields
//     T^{tau tau}, T^{tau x}, T^{tau y}, T^{tau eta}, pi^{xx}, pi^{xy}, pi^{x eta}, pi^{yy}, pi^{y eta}, Pi
// and u^x, u^y, u^eta (43 padded arrays instead of 61 + 6).  Wherever the step reads pi^{tau tau}, pi^{tau i}, pi^{eta eta} or u^tau - at
// ANY stencil cell - they are evaluated from that cell's stored values: u^tau from u.u = 1, then Eqs. 51, 48-50, 47 with v^i = u^i/u^tau.
// What the Euler step would compute for the dependent components is not computed.  Eqs. 52-54 become implicit (pi^{tau mu} depends on the
// velocity being solved for): fixed point on v as in the oracle.
// One thread per cell, stencils through L1/L2 (the layout of variant 1): this is the memory-saving mode, not the fast path.
#pragma once
#include "vh_kernels.cuh"
#include "vh_math.cuh"

namespace vh {

constexpr int NQR = 10;      // stored conserved fields
// slot of a full-mode field in the reduced set (-1: dependent, not stored)
__device__ __forceinline__ constexpr int red_slot(int n) { return (n < 4) ? n : ((n >= PXX && n <= PYN) ? n - 4 : ((n == BPI) ? 9 : -1)); }

struct RedArgs {
  const real* q_in; const real* e_in; const real* p_in; const real* u_in; const real* u_prev;      // q: 10 arrays, u: 3 arrays
  const real* q_n;                                                                                   // stage 2: q^n (10 arrays)
  real* q_out; real* e_out; real* p_out; real* u_out;
  Counters* cnt;
  real t, t_post, t_prev;      // tau of C[q], of the inversion of the result, and of the time level u_prev belongs to (its u^tau is normalised there)
};

// Eqs. 51, 48-50, 47 (Eq. 49 with its typo fixed, R3): out = pi^tt, pi^tx, pi^ty, pi^tn, pi^nn
__device__ __forceinline__ void dependent_pi(const real v[3], real t2, real pxx, real pxy, real pxn, real pyy, real pyn, real out[5]) {
  const real vx = v[0], vy = v[1], vn = v[2];
  const real pnn = (pxx * (vx * vx - real(1.0)) + pyy * (vy * vy - real(1.0)) + real(2.0) * pxy * vx * vy + real(2.0) * t2 * (pxn * vx * vn + pyn * vy * vn)) *
                   rcp_fast(t2 * (real(1.0) - t2 * vn * vn));
  const real ptx = pxx * vx + pxy * vy + t2 * pxn * vn;
  const real pty = pxy * vx + pyy * vy + t2 * pyn * vn;
  const real ptn = pxn * vx + pyn * vy + t2 * pnn * vn;
  const real ptt = ptx * vx + pty * vy + t2 * ptn * vn;
  out[0] = ptt; out[1] = ptx; out[2] = pty; out[3] = ptn; out[4] = pnn;
}

// the full 15 fields and u^mu of one cell from its stored values
__device__ __forceinline__ void load_expanded(const DevParams& P, const real* __restrict__ q, const real* __restrict__ u, long long c, real t2, real qf[NQ],
                                              real uf[4]) {
  const long long fs = P.fstride;
  uf[1] = u[c]; uf[2] = u[fs + c]; uf[3] = u[2 * fs + c];
  uf[0] = sqrt_fast(real(1.0) + uf[1] * uf[1] + uf[2] * uf[2] + t2 * uf[3] * uf[3]);
  const real iut = rcp_fast(uf[0]);
  const real v[3] = {uf[1] * iut, uf[2] * iut, uf[3] * iut};
#pragma unroll
  for (int n = 0; n < 4; ++n) qf[n] = q[n * fs + c];
#pragma unroll
  for (int n = PXX; n <= PYN; ++n) qf[n] = q[(n - 4) * fs + c];
  qf[BPI] = q[9 * fs + c];
  real d[5];
  dependent_pi(v, t2, qf[PXX], qf[PXY], qf[PXN], qf[PYY], qf[PYN], d);
  qf[PTT] = d[0]; qf[PTX] = d[1]; qf[PTY] = d[2]; qf[PTN] = d[3]; qf[PNN] = d[4];
}

// ------------------------------------------------------------------------------------------------ the kernel
// grid: (ceil(nx/32), ceil(ny/4), nz*n_batch), block (32, 4)
template <int EOS, bool MILNE, bool TWO_D, int STAGE>
__global__ void __launch_bounds__(128) stage_reduced_kernel(const __grid_constant__ DevParams P, const __grid_constant__ RedArgs A) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z % P.nz, b = blockIdx.z / P.nz;
  const bool valid = (i < P.nx) && (j < P.ny);
  i = min(i, P.nx - 1);
  j = min(j, P.ny - 1);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  const long long fs = P.fstride;
  const real t = A.t;
  const real t2 = MILNE ? t * t : real(1.0);
  const real it2 = real(1.0) / t2;
  const real th = P.theta;
  unsigned long long nfail = 0, nnonf = 0;
  real minfac = real(1.0);

  real qc[NQ], uc[4];
  load_expanded(P, A.q_in, A.u_in, c, t2, qc, uc);
  const real ec = A.e_in[c], pc = A.p_in[c];
  real C[NQ];
#pragma unroll
  for (int n = 0; n < NQ; ++n) C[n] = real(0.0);
  real du[4][4];
  real divv = real(0.0);
  {      // backward difference in time (:424); u^tau of u_prev from u.u = 1 at its own time level
    const real tp2 = MILNE ? A.t_prev * A.t_prev : real(1.0);
    const real x = A.u_prev[c], y = A.u_prev[fs + c], z = A.u_prev[2 * fs + c];
    const real up4[4] = {sqrt(real(1.0) + x * x + y * y + tp2 * z * z), x, y, z};
#pragma unroll
    for (int n = 0; n < 4; ++n) du[0][n] = (uc[n] - up4[n]) * P.inv_dtau;
  }
  const long long strides[3] = {1, (long long)P.NXp, P.plane};
  const real inv_dr[3] = {P.inv_dx, P.inv_dy, P.inv_dz};
  const int ext[3] = {P.nx, P.ny, P.nz};
  const int pos[3] = {i, j, k};
#pragma unroll 1
  for (int d = 0; d < 3; ++d) {
    if (TWO_D && d == 2) {
#pragma unroll
      for (int n = 0; n < 4; ++n) du[3][n] = real(0.0);
      continue;
    }
    const long long s = strides[d];
    // the five stencil cells of this direction, expanded (Alg. 2: "I[5N]"), and e, p, u where they are needed
    real Q5[5][NQ], u5[5][4];
#pragma unroll
    for (int m = 0; m < 5; ++m) load_expanded(P, A.q_in, A.u_in, c + (m - 2) * s, t2, Q5[m], u5[m]);
    const real e5[3] = {A.e_in[c - s], ec, A.e_in[c + s]};
    const real p5[2] = {A.p_in[c - s], A.p_in[c + s]};
    // ---- KT flux of the ten evolved fields (Eqs. 59-68); each reconstructed state inverted for its velocity (Alg. 3 :667-672)
    auto recon4 = [&](int n, real out[4]) {
      const real a0 = Q5[0][n], a1 = Q5[1][n], a2 = Q5[2][n], a3 = Q5[3][n], a4 = Q5[4][n];
      const real hm = half_slope(a0, a1, a2, th), h0 = half_slope(a1, a2, a3, th), hp = half_slope(a2, a3, a4, th);
      out[0] = a2 + h0; out[1] = a3 - hp; out[2] = a1 + hm; out[3] = a2 - h0;      // q^-_{+1/2}, q^+_{+1/2}, q^-_{-1/2}, q^+_{-1/2}
    };
    real E[4], Mx[4], My[4], Mn[4], Pi4[4], w[4], w2[4];
    recon4(TTT, w); recon4(PTT, w2);
#pragma unroll
    for (int m = 0; m < 4; ++m) E[m] = w[m] - w2[m];
    recon4(TTX, w); recon4(PTX, w2);
#pragma unroll
    for (int m = 0; m < 4; ++m) Mx[m] = w[m] - w2[m];
    recon4(TTY, w); recon4(PTY, w2);
#pragma unroll
    for (int m = 0; m < 4; ++m) My[m] = w[m] - w2[m];
    recon4(TTN, w); recon4(PTN, w2);
#pragma unroll
    for (int m = 0; m < 4; ++m) Mn[m] = w[m] - w2[m];
    recon4(BPI, Pi4);
    const bool count_hi = ext[d] > 1, count_lo = ext[d] > 1 && pos[d] == 0;
    real v[4];
    {      // the four states as two pairs through the paired Newton iteration of the default path (same root, cap and tolerance, R6)
      const real* Mr = (d == 0) ? Mx : ((d == 1) ? My : Mn);
      NewtonState S[4];
#pragma unroll
      for (int m = 0; m < 4; ++m) { S[m].E = E[m]; S[m].Pi = Pi4[m]; S[m].M2 = Mx[m] * Mx[m] + My[m] * My[m] + t2 * Mn[m] * Mn[m]; }
      newton_pair<EOS>(P, S[0], S[1], e5[1], e5[2]);      // the upper interface: state from this cell, state from the next one
      newton_pair<EOS>(P, S[2], S[3], e5[0], e5[1]);      // the lower interface
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        v[m] = Mr[m] * S[m].rden;
        if (S[m].fail) { v[m] = clip_velocity(v[m]); if (m < 2 ? count_hi : count_lo) ++nfail; }
      }
    }
    const real ap = fmax(fabs(v[1]), fabs(v[0])), am = fmax(fabs(v[3]), fabs(v[2]));      // Eq. 62
#pragma unroll
    for (int n = 0; n < NQ; ++n) {
      if (red_slot(n) < 0) continue;
      recon4(n, w);
      const real Hp = real(0.5) * (v[1] * w[1] + v[0] * w[0]) - real(0.5) * ap * (w[1] - w[0]);      // Eq. 61
      const real Hm = real(0.5) * (v[3] * w[3] + v[2] * w[2]) - real(0.5) * am * (w[3] - w[2]);
      C[n] -= (Hp - Hm) * inv_dr[d];
    }
    // ---- conservation-law sources of this direction: -d_i A^{i nu}, A^{i nu} = P (v^i delta^nu_tau - g^{i nu}) - v^i pi^{tau nu} + pi^{i nu} (B.2-B.5)
    real Ax[2][4];
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      const real* qn = Q5[side ? 3 : 1];
      const real* un_ = u5[side ? 3 : 1];
      const real vi = un_[d + 1] / un_[0];
      const real Pt = p5[side] + qn[BPI];
      const int pin[3][4] = {{PTX, PXX, PXY, PXN}, {PTY, PXY, PYY, PYN}, {PTN, PXN, PYN, PNN}};      // pi^{i nu}
      Ax[side][0] = vi * (Pt - qn[PTT]) + qn[pin[d][0]];
#pragma unroll
      for (int nu = 1; nu < 4; ++nu) {
        const real g = (nu == d + 1) ? ((nu == 3) ? it2 : real(1.0)) : real(0.0);      // -g^{i nu}
        Ax[side][nu] = Pt * g - vi * qn[PTT + nu] + qn[pin[d][nu]];
      }
      divv += (side ? vi : -vi) * real(0.5) * inv_dr[d];
    }
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      C[n] -= (Ax[1][n] - Ax[0][n]) * real(0.5) * inv_dr[d];
      du[d + 1][n] = (u5[3][n] - u5[1][n]) * real(0.5) * inv_dr[d];
    }
  }
  if (MILNE) {      // G_c (:1013), T^{eta eta} from Eq. 34
    const real itau = real(1.0) / t;
    const real Ptc = pc + qc[BPI];
    const real Tnn = (ec + Ptc) * uc[3] * uc[3] + Ptc * it2 + qc[PNN];
    C[0] -= (qc[TTT] + t2 * Tnn) * itau;
    C[1] -= qc[TTX] * itau;
    C[2] -= qc[TTY] * itau;
    C[3] -= real(3.0) * qc[TTN] * itau;
  }
  {      // relaxation sources (Eqs. 39-46) at the centre with the expanded tensor; only the evolved components are kept
    Kin K;
    kinematics<MILNE>(uc, du[0], du[1], du[2], du[3], t, K);
    real p0, cs2;
    eos_p_cs2<EOS>(P, ec, p0, cs2);
    real Jpi[10], JPi;
    dissipative_sources<EOS, MILNE>(P, t, uc, K, qc + PTT, qc[BPI], ec, p0, cs2, divv, Jpi, JPi);
#pragma unroll
    for (int n = PXX; n <= PYN; ++n) C[n] += Jpi[n - PTT];
    if (P.bulk) C[BPI] += JPi;
  }
  // ---- stage result of the ten evolved fields (Eqs. 69-71)
  real qo[NQ];
#pragma unroll
  for (int n = 0; n < NQ; ++n) {
    qo[n] = real(0.0);
    const int r = red_slot(n);
    if (r < 0) continue;
    real v = qc[n] + P.dtau * C[n];
    if (STAGE == 2) v = real(0.5) * (A.q_n[r * fs + c] + v);
    if (n == BPI && !P.bulk) v = real(0.0);
    qo[n] = v;
  }
  // ---- Post (R22): Eqs. 52-54 with pi^{tau mu}(v) of Eqs. 47-50 - fixed point on v from the velocity of the stage's input, Eq. 72 at every sweep
  const real tq = A.t_post;
  const real tq2 = MILNE ? tq * tq : real(1.0);
  const real rt = MILNE ? tq : real(1.0);
  real vv[3] = {uc[1] / uc[0], uc[2] / uc[0], uc[3] / uc[0]};
  real ee = ec, Eo = real(0.0), M[3] = {real(0.0), real(0.0), real(0.0)};
  bool done = false, conv = false, failed = false;
  for (int sweep = 0; sweep < P.newton_max_iter; ++sweep) {
    if (__all_sync(0xffffffffu, done)) break;      // warp-uniform loop: invert_energy votes across the warp
    real dpi[5];
    dependent_pi(vv, tq2, qo[PXX], qo[PXY], qo[PXN], qo[PYY], qo[PYN], dpi);
    const real E1 = qo[TTT] - dpi[0];
    const real M1[3] = {qo[TTX] - dpi[1], qo[TTY] - dpi[2], qo[TTN] - dpi[3]};
    const real M2 = M1[0] * M1[0] + M1[1] * M1[1] + tq2 * M1[2] * M1[2];
    bool f1;
    const real e1 = invert_energy<EOS>(P, E1, M2, qo[BPI], ee, f1);
    if (!done) {
      Eo = E1; M[0] = M1[0]; M[1] = M1[1]; M[2] = M1[2];
      ee = e1;
      if (f1) { failed = true; done = true; }
      else {
        const real den = E1 + eos_p<EOS>(P, e1) + qo[BPI];
        const real vn[3] = {M1[0] / den, M1[1] / den, M1[2] / den};
        const real dv = fmax(fmax(fabs(vn[0] - vv[0]), fabs(vn[1] - vv[1])), rt * fabs(vn[2] - vv[2]));
        vv[0] = vn[0]; vv[1] = vn[1]; vv[2] = vn[2];
        if (dv <= P.newton_rtol) { conv = true; done = true; }
      }
    }
  }
  if (!conv) failed = true;
  if (failed) ++nfail;
  {      // the dependent components that go with the converged velocity, and E, M consistent with them
    real dpi[5];
    dependent_pi(vv, tq2, qo[PXX], qo[PXY], qo[PXN], qo[PYY], qo[PYN], dpi);
    qo[PTT] = dpi[0]; qo[PTX] = dpi[1]; qo[PTY] = dpi[2]; qo[PTN] = dpi[3]; qo[PNN] = dpi[4];
    Eo = qo[TTT] - dpi[0]; M[0] = qo[TTX] - dpi[1]; M[1] = qo[TTY] - dpi[2]; M[2] = qo[TTN] - dpi[3];
  }
  const real p0 = eos_p<EOS>(P, ee);
  const real Pt = p0 + qo[BPI];
  const real ut = sqrt((Eo + Pt) / (ee + Pt));          // Eq. 53
  const real inv = real(1.0) / ((ee + Pt) * ut);        // Eq. 54
  const real u[4] = {ut, M[0] * inv, M[1] * inv, M[2] * inv};
  if (!(isfinite(ee) && isfinite(ut))) ++nnonf;
  const real fac = regulation_factor<MILNE>(P, qo, ee, p0, u, tq);      // Eqs. 73-74; all ten components scale alike, so Eqs. 47-51 keep holding
  minfac = fmin(minfac, fac);
  if (valid) {
#pragma unroll
    for (int n = 0; n < NQ; ++n) {
      const int r = red_slot(n);
      if (r >= 0) A.q_out[r * fs + c] = (n >= PTT) ? qo[n] * fac : qo[n];
    }
    A.e_out[c] = ee;
    A.p_out[c] = p0;
#pragma unroll
    for (int n = 0; n < 3; ++n) A.u_out[n * fs + c] = u[n + 1];
  }
  flush_counters(A.cnt, valid ? nfail : 0ull, valid ? nnonf : 0ull, valid ? minfac : real(1.0), *(volatile unsigned long long*)&A.cnt->min_reg_bits);
}

// ------------------------------------------------------------------------------------------------ initial condition / export in reduced storage
// q^0 from (e, u, pi, Pi) by Eqs. 32-33 with the dependent pi^{tau mu}, pi^{eta eta} replaced by their algebraic values first (they are not state)
template <int EOS, bool MILNE>
__global__ void __launch_bounds__(256) init_reduced_kernel(const __grid_constant__ DevParams P, const double* __restrict__ e_in, const double* __restrict__ u_in,
                                                           const double* __restrict__ pi_in, const double* __restrict__ Pi_in, real t, real* q, real* e,
                                                           real* p, real* u, real* uprev) {
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= np) return;
  const int i = (int)(w % P.nx);
  long long r = w / P.nx;
  const int j = (int)(r % P.ny); r /= P.ny;
  const int k = (int)(r % P.nz);
  const int b = (int)(r / P.nz);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  const long long fs = P.fstride;
  const real t2 = MILNE ? t * t : real(1.0);
  const real ee = e_in[w];
  const real p0 = eos_p<EOS>(P, ee);
  const real Pi = (Pi_in && P.bulk) ? (real)Pi_in[w] : real(0.0);
  const real Pt = p0 + Pi;
  real uu[4];
#pragma unroll
  for (int n = 1; n < 4; ++n) uu[n] = u_in[n * np + w];
  uu[0] = sqrt(real(1.0) + uu[1] * uu[1] + uu[2] * uu[2] + t2 * uu[3] * uu[3]);
  real pi[10];
#pragma unroll
  for (int n = 0; n < 10; ++n) pi[n] = pi_in ? (real)pi_in[n * np + w] : real(0.0);
  const real v[3] = {uu[1] / uu[0], uu[2] / uu[0], uu[3] / uu[0]};
  real d[5];
  dependent_pi(v, t2, pi[4], pi[5], pi[6], pi[7], pi[8], d);
  q[0 * fs + c] = (ee + Pt) * uu[0] * uu[0] - Pt + d[0];
#pragma unroll
  for (int n = 1; n < 4; ++n) q[n * fs + c] = (ee + Pt) * uu[0] * uu[n] + d[n];
#pragma unroll
  for (int n = 0; n < 5; ++n) q[(4 + n) * fs + c] = pi[4 + n];
  q[9 * fs + c] = Pi;
  e[c] = ee;
  p[c] = p0;
#pragma unroll
  for (int n = 0; n < 3; ++n) { u[n * fs + c] = uu[n + 1]; uprev[n * fs + c] = uu[n + 1]; }
}

// compact (caller-side, double) full fields from the reduced state: q15 and / or u4 (either may be null); t = time level of the state
template <bool MILNE>
__global__ void __launch_bounds__(256) export_reduced_kernel(const __grid_constant__ DevParams P, const real* __restrict__ q, const real* __restrict__ u, real t,
                                                             double* q15, double* u4) {
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= np) return;
  const int i = (int)(w % P.nx);
  long long r = w / P.nx;
  const int j = (int)(r % P.ny); r /= P.ny;
  const int k = (int)(r % P.nz);
  const int b = (int)(r / P.nz);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  const real t2 = MILNE ? t * t : real(1.0);
  real qf[NQ], uf[4];
  if (q) {
    load_expanded(P, q, u, c, t2, qf, uf);
  } else {
    const long long fs = P.fstride;
    uf[1] = u[c]; uf[2] = u[fs + c]; uf[3] = u[2 * fs + c];
    uf[0] = sqrt(real(1.0) + uf[1] * uf[1] + uf[2] * uf[2] + t2 * uf[3] * uf[3]);
  }
  if (q15) {
#pragma unroll
    for (int n = 0; n < NQ; ++n) q15[n * np + w] = (double)qf[n];
  }
  if (u4) {
#pragma unroll
    for (int n = 0; n < 4; ++n) u4[n * np + w] = (double)uf[n];
  }
}

// compact full q15 / u4 (caller side) -> the stored subset
static __global__ void __launch_bounds__(256) import_reduced_kernel(const __grid_constant__ DevParams P, const double* __restrict__ q15, const double* __restrict__ u4,
                                                             real* q, real* u) {
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= np) return;
  const int i = (int)(w % P.nx);
  long long r = w / P.nx;
  const int j = (int)(r % P.ny); r /= P.ny;
  const int k = (int)(r % P.nz);
  const int b = (int)(r / P.nz);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  const long long fs = P.fstride;
  if (q15) {
#pragma unroll
    for (int n = 0; n < NQ; ++n) { const int s = red_slot(n); if (s >= 0) q[s * fs + c] = (real)q15[n * np + w]; }
  }
  if (u4) {
#pragma unroll
    for (int n = 0; n < 3; ++n) u[n * fs + c] = (real)u4[(n + 1) * np + w];
  }
}

}  // namespace vh
