// vh_kernels.cuh -- kernels of the KT / Heun step.  Variant 1 ("cell"): one thread per cell, stencils through L1/L2,
// both interfaces of every direction evaluated by the owning thread (Alg. 2-3 fused with Alg. 1 and with the
// "set inferred variables" / "regulate" kernels of Fig. 5).  See DESIGN.md "Kernels".
#pragma once
#include "vh_device.cuh"

namespace vh {

struct Counters {
  unsigned long long n_fail;        // failed Newton inversions (interface states + cells)
  unsigned long long n_nonfinite;   // cells with non-finite e or u^tau after inversion
  unsigned long long min_reg_bits;  // bit pattern of the smallest regularisation factor (positive doubles order as integers)
};

struct StageArgs {
  const real* q_in;  const real* e_in;  const real* p_in;  const real* u_in;  const real* u_prev;
  const real* q_n;   // stage 2: q^n for the convex combination (Eq. 70)
  real* q_out; real* e_out; real* p_out; real* u_out;
  Counters* cnt;
  real t;            // tau at which C[q] is evaluated (R7)
  real t_post;       // tau used by the inversion / regularisation of the result
  real* regfac;      // padded array receiving tanh(rho)/rho of every cell (Fig. 17), or nullptr (the default: nothing is stored)
};

// ------------------------------------------------------------------------------------------------ flux part, variant 1
// Adds -(H_{+1/2} - H_{-1/2})/dr of direction r (stride s) to C[0..NF).  Eqs. 59-68.
template <int EOS, bool VISC, bool MILNE>
__device__ __forceinline__ void flux_dir_cell(const DevParams& P, const real* __restrict__ q, const real* __restrict__ e_in, long long c,
                                              long long s, int r, real inv_dr, real t2, bool count_hi, bool count_lo, real* C,
                                              unsigned long long& nfail) {
  constexpr int NF = VISC ? NQ : 4;
  const real th = P.theta;
  // reconstructed primary combinations of the four states:
  //   0: q^-_{+1/2} (from cell c)   1: q^+_{+1/2} (from c+s)   2: q^-_{-1/2} (from c-s)   3: q^+_{-1/2} (from c)
  real E[4], Mx[4], My[4], Mn[4], Pi[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) { E[k] = 0; Mx[k] = 0; My[k] = 0; Mn[k] = 0; Pi[k] = 0; }
  auto recon4 = [&](int n, real out[4]) {
    const real* f = q + (long long)n * P.fstride + c;
    real a0 = f[-2 * s], a1 = f[-s], a2 = f[0], a3 = f[s], a4 = f[2 * s];
    real hm = half_slope(a0, a1, a2, th), h0 = half_slope(a1, a2, a3, th), hp = half_slope(a2, a3, a4, th);
    out[0] = a2 + h0;   // Eq. 64
    out[1] = a3 - hp;   // Eq. 63
    out[2] = a1 + hm;   // Eq. 66
    out[3] = a2 - h0;   // Eq. 65
  };
  {
    real w[4];
    recon4(TTT, w);
#pragma unroll
    for (int k = 0; k < 4; ++k) E[k] = w[k];
    recon4(TTX, w);
#pragma unroll
    for (int k = 0; k < 4; ++k) Mx[k] = w[k];
    recon4(TTY, w);
#pragma unroll
    for (int k = 0; k < 4; ++k) My[k] = w[k];
    recon4(TTN, w);
#pragma unroll
    for (int k = 0; k < 4; ++k) Mn[k] = w[k];
    if (VISC) {
      recon4(PTT, w);
#pragma unroll
      for (int k = 0; k < 4; ++k) E[k] -= w[k];
      recon4(PTX, w);
#pragma unroll
      for (int k = 0; k < 4; ++k) Mx[k] -= w[k];
      recon4(PTY, w);
#pragma unroll
      for (int k = 0; k < 4; ++k) My[k] -= w[k];
      recon4(PTN, w);
#pragma unroll
      for (int k = 0; k < 4; ++k) Mn[k] -= w[k];
      recon4(BPI, w);
#pragma unroll
      for (int k = 0; k < 4; ++k) Pi[k] = w[k];
    }
  }
  const real e0 = e_in[c], em = e_in[c - s], ep = e_in[c + s];
  real v[4];
  // failure counter: every interface state once (the +1/2 interface by its lower cell; the -1/2 interface only by the first
  // cell of the row), none along a direction of extent 1
  v[0] = state_velocity<EOS, MILNE>(P, E[0], Mx[0], My[0], Mn[0], Pi[0], t2, e0, r, count_hi, nfail);
  v[1] = state_velocity<EOS, MILNE>(P, E[1], Mx[1], My[1], Mn[1], Pi[1], t2, ep, r, count_hi, nfail);
  v[2] = state_velocity<EOS, MILNE>(P, E[2], Mx[2], My[2], Mn[2], Pi[2], t2, em, r, count_lo, nfail);
  v[3] = state_velocity<EOS, MILNE>(P, E[3], Mx[3], My[3], Mn[3], Pi[3], t2, e0, r, count_lo, nfail);
  const real ap = fmax(fabs(v[1]), fabs(v[0]));     // Eq. 62, a = |v_r| (:388)
  const real am = fmax(fabs(v[3]), fabs(v[2]));
#pragma unroll
  for (int n = 0; n < NF; ++n) {
    real w[4];
    recon4(n, w);
    real Hp = real(0.5) * (v[1] * w[1] + v[0] * w[0]) - real(0.5) * ap * (w[1] - w[0]);   // Eq. 61
    real Hm = real(0.5) * (v[3] * w[3] + v[2] * w[2]) - real(0.5) * am * (w[3] - w[2]);
    C[n] -= (Hp - Hm) * inv_dr;
  }
}

// ------------------------------------------------------------------------------------------------ sources, variant 1
// J = S + G (App. B).  Adds to C.
template <int EOS, bool VISC, bool MILNE, bool TWO_D>
__device__ __forceinline__ void sources_cell(const DevParams& P, const StageArgs& A, long long c, real t, const real* qc, real ec, real pc,
                                             const real* uc, real* C) {
  const real* __restrict__ q = A.q_in;
  const real* __restrict__ pp = A.p_in;
  const real* __restrict__ uu = A.u_in;
  const long long fs = P.fstride;
  const real t2 = MILNE ? t * t : real(1.0);
  const real it2 = real(1.0) / t2;
  const long long strides[3] = {1, (long long)P.NXp, P.plane};
  const real hinv[3] = {real(0.5) * P.inv_dx, real(0.5) * P.inv_dy, real(0.5) * P.inv_dz};
  real du[4][4];     // du[a][n] = partial_a u^n ; a = 0 is time
  real divv = real(0.0);
#pragma unroll
  for (int n = 0; n < 4; ++n) du[0][n] = (uc[n] - A.u_prev[n * fs + c]) * P.inv_dtau;
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
      for (int n = 0; n < 4; ++n) un_[n] = uu[n * fs + cn];
      real vi = un_[d + 1] / un_[0];
      real Pt = pp[cn];
      real* Ax = side ? Ap : Am;
      if (VISC) {
        Pt += q[BPI * fs + cn];
        real ptt = q[PTT * fs + cn], ptx = q[PTX * fs + cn], pty = q[PTY * fs + cn], ptn = q[PTN * fs + cn];
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
        Ax[1] = (d == 0) ? Pt : real(0.0);
        Ax[2] = (d == 1) ? Pt : real(0.0);
        Ax[3] = (d == 2) ? Pt * it2 : real(0.0);
      }
      divv += (side ? vi : -vi) * hinv[d];
    }
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      C[n] -= (Ap[n] - Am[n]) * hinv[d];
      du[d + 1][n] = (up[n] - um[n]) * hinv[d];
    }
  }
  if (MILNE) {     // G_c (:1013), T^{eta eta} from Eq. 34
    const real itau = real(1.0) / t;
    real Ptc = pc + (VISC ? qc[BPI] : real(0.0));
    real Tnn = (ec + Ptc) * uc[3] * uc[3] + Ptc * it2 + (VISC ? qc[PNN] : real(0.0));
    C[0] -= (qc[TTT] + t2 * Tnn) * itau;
    C[1] -= qc[TTX] * itau;
    C[2] -= qc[TTY] * itau;
    C[3] -= real(3.0) * qc[TTN] * itau;
  }
  if (VISC) {
    Kin K;
    kinematics<MILNE>(uc, du[0], du[1], du[2], du[3], t, K);
    real p0, cs2;
    eos_p_cs2<EOS>(P, ec, p0, cs2);
    real Jpi[10], JPi;
    dissipative_sources<EOS, MILNE>(P, t, uc, K, qc + PTT, qc[BPI], ec, p0, cs2, divv, Jpi, JPi);
    if (P.shear) {
#pragma unroll
      for (int n = 0; n < 10; ++n) C[PTT + n] += Jpi[n];
    }
    if (P.bulk) C[BPI] += JPi;
  }
}

// ------------------------------------------------------------------------------------------------ Post: Eqs. 52-54, 72-74
// Inverts the cell state q (in registers), regulates pi, Pi in place, writes q,e,p,u.  (Fig. 5 "set inferred variables" +
// "regulate dissipative currents" fused into the stage epilogue.)
template <int EOS, bool VISC, bool MILNE>
__device__ __forceinline__ void post_cell(const DevParams& P, const StageArgs& A, long long c, real* q, real guess, bool valid,
                                          unsigned long long& nfail, unsigned long long& nnonf, real& minfac) {
  const real t = A.t_post;
  const real t2 = MILNE ? t * t : real(1.0);
  real E = q[TTT] - (VISC ? q[PTT] : real(0.0));
  real Mx = q[TTX] - (VISC ? q[PTX] : real(0.0)), My = q[TTY] - (VISC ? q[PTY] : real(0.0)), Mn = q[TTN] - (VISC ? q[PTN] : real(0.0));
  real Pi = VISC ? q[BPI] : real(0.0);
  real M2 = Mx * Mx + My * My + t2 * Mn * Mn;
  bool fail;
  real e = invert_energy<EOS>(P, E, M2, Pi, guess, fail);
  if (fail) ++nfail;
  real p0 = eos_p<EOS>(P, e);
  real Pt = p0 + Pi;
  real ut = sqrt((E + Pt) / (e + Pt));          // Eq. 53
  real inv = real(1.0) / ((e + Pt) * ut);             // Eq. 54
  real u[4] = {ut, Mx * inv, My * inv, Mn * inv};
  if (!(isfinite(e) && isfinite(ut))) ++nnonf;
  if (VISC) {
    real fac = regulation_factor<MILNE>(P, q, e, p0, u, t);
    minfac = fmin(minfac, fac);
    if (A.regfac && valid) A.regfac[c] = fac;
#pragma unroll
    for (int n = PTT; n < NQ; ++n) q[n] *= fac;
  }
  if (valid) {
    const long long fs = P.fstride;
#pragma unroll
    for (int n = 0; n < NQ; ++n) A.q_out[n * fs + c] = q[n];
    A.e_out[c] = e;
    A.p_out[c] = p0;
#pragma unroll
    for (int n = 0; n < 4; ++n) A.u_out[n * fs + c] = u[n];
  }
}

// `record` is the value of cnt->min_reg_bits the caller read earlier (any earlier value works: the record only ever falls, so a
// stale one lets a few redundant atomics through but never loses a minimum); reading it at kernel start hides the load latency.
__device__ __forceinline__ void flush_counters(Counters* cnt, unsigned long long nfail, unsigned long long nnonf, real minfac_r,
                                               unsigned long long record = ~0ull) {
  if (nfail) atomicAdd(&cnt->n_fail, nfail);
  if (nnonf) atomicAdd(&cnt->n_nonfinite, nnonf);
  // warp minimum of the regularisation factor, then at most one atomic per warp (skipped when it cannot lower the record)
  // (positive doubles order like their bit patterns: two integer warp reductions, high word then low word among the ties)
  double minfac = (double)minfac_r;      // the record is kept as the bit pattern of a double in both precisions
  const unsigned hi = (unsigned)__double2hiint(minfac), lo = (unsigned)__double2loint(minfac);
  const unsigned hmin = __reduce_min_sync(0xffffffffu, hi);
  const unsigned lmin = __reduce_min_sync(0xffffffffu, (hi == hmin) ? lo : 0xffffffffu);
  minfac = __hiloint2double((int)hmin, (int)lmin);
  if ((threadIdx.x + blockDim.x * threadIdx.y) % 32 == 0 && minfac < real(1.0)) {
    unsigned long long bits = (unsigned long long)__double_as_longlong(minfac);
    if (bits < record) atomicMin(&cnt->min_reg_bits, bits);
  }
}

// ------------------------------------------------------------------------------------------------ stage kernel, variant 1
// grid: (ceil(nx/32), ceil(ny/BY), nz*n_batch), block (32, BY).
template <int EOS, bool VISC, bool MILNE, bool TWO_D, int STAGE>
__global__ void __launch_bounds__(256) stage_cell_kernel(const __grid_constant__ DevParams P, const __grid_constant__ StageArgs A) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int j = blockIdx.y * blockDim.y + threadIdx.y;
  int k = blockIdx.z % P.nz, b = blockIdx.z / P.nz;
  bool valid = (i < P.nx) && (j < P.ny);
  i = min(i, P.nx - 1);
  j = min(j, P.ny - 1);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  const long long fs = P.fstride;
  constexpr int NF = VISC ? NQ : 4;
  const real t = A.t;
  const real t2 = MILNE ? t * t : real(1.0);
  unsigned long long nfail = 0, nnonf = 0;
  real minfac = real(1.0);

  real qc[NQ], C[NQ];
#pragma unroll
  for (int n = 0; n < NQ; ++n) { qc[n] = (n < NF) ? A.q_in[n * fs + c] : real(0.0); C[n] = real(0.0); }
  const real ec = A.e_in[c], pc = A.p_in[c];
  real uc[4];
#pragma unroll
  for (int n = 0; n < 4; ++n) uc[n] = A.u_in[n * fs + c];

  flux_dir_cell<EOS, VISC, MILNE>(P, A.q_in, A.e_in, c, 1, 0, P.inv_dx, t2, P.nx > 1, P.nx > 1 && i == 0, C, nfail);
  flux_dir_cell<EOS, VISC, MILNE>(P, A.q_in, A.e_in, c, P.NXp, 1, P.inv_dy, t2, P.ny > 1, P.ny > 1 && j == 0, C, nfail);
  if (!TWO_D) flux_dir_cell<EOS, VISC, MILNE>(P, A.q_in, A.e_in, c, P.plane, 2, P.inv_dz, t2, P.nz > 1, P.nz > 1 && k == 0, C, nfail);
  sources_cell<EOS, VISC, MILNE, TWO_D>(P, A, c, t, qc, ec, pc, uc, C);

  real qo[NQ];
#pragma unroll
  for (int n = 0; n < NQ; ++n) {
    real v = real(0.0);
    if (n < NF) {
      v = qc[n] + P.dtau * C[n];                                   // E[w] = w + dtau C[w]  (:413)
      if (STAGE == 2) v = real(0.5) * (A.q_n[n * fs + c] + v);           // Eq. 70, beta = 1/2
    }
    if (VISC && n >= PTT && n < BPI && !P.shear) v = real(0.0);
    if (VISC && n == BPI && !P.bulk) v = real(0.0);
    qo[n] = v;
  }
  post_cell<EOS, VISC, MILNE>(P, A, c, qo, ec, valid, nfail, nnonf, minfac);
  flush_counters(A.cnt, valid ? nfail : 0ull, valid ? nnonf : 0ull, valid ? minfac : real(1.0), *(volatile unsigned long long*)&A.cnt->min_reg_bits);
}

// ------------------------------------------------------------------------------------------------ ghost cells (Eqs. 75-76)
struct GhostArgs { real* q; real* e; real* p; real* u; int nq; };      // nq conserved arrays (15, or 10 in reduced storage), then e, p, then the u arrays

// grid: (ceil(W/256), nq + 2 + nu, n_batch); W = ny*nz + nx*nz + nx*ny (3+1d) or ny + nx (2+1d)
template <bool TWO_D>
__global__ void __launch_bounds__(256) ghost_kernel(const __grid_constant__ DevParams P, const GhostArgs G) {
  const int a = blockIdx.y;
  real* f = (a < G.nq) ? G.q + (long long)a * P.fstride : (a == G.nq ? G.e : (a == G.nq + 1 ? G.p : G.u + (long long)(a - G.nq - 2) * P.fstride));
  f += (long long)blockIdx.z * P.bstride;
  const long long Wx = (long long)P.ny * P.nz, Wy = (long long)P.nx * P.nz, Wz = TWO_D ? 0 : (long long)P.nx * P.ny;
  long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long NXp = P.NXp, pl = P.plane;
  if (w < Wx) {
    int j = (int)(w % P.ny), k = (int)(w / P.ny);
    real* row = f + (long long)(k + P.zoff) * pl + (long long)(j + 2) * NXp;
    real lo = row[XOFF], hi = row[P.nx + XOFF - 1];
    row[XOFF - 2] = lo; row[XOFF - 1] = lo; row[P.nx + XOFF] = hi; row[P.nx + XOFF + 1] = hi;
  } else if (w < Wx + Wy) {
    w -= Wx;
    int i = (int)(w % P.nx), k = (int)(w / P.nx);
    real* col = f + (long long)(k + P.zoff) * pl + (i + XOFF);
    real lo = col[2 * NXp], hi = col[(long long)(P.ny + 1) * NXp];
    col[0] = lo; col[NXp] = lo; col[(long long)(P.ny + 2) * NXp] = hi; col[(long long)(P.ny + 3) * NXp] = hi;
  } else if (w < Wx + Wy + Wz) {
    w -= Wx + Wy;
    int i = (int)(w % P.nx), j = (int)(w / P.nx);
    real* col = f + (long long)(j + 2) * NXp + (i + XOFF);
    real lo = col[2 * pl], hi = col[(long long)(P.nz + 1) * pl];
    col[0] = lo; col[pl] = lo; col[(long long)(P.nz + 2) * pl] = hi; col[(long long)(P.nz + 3) * pl] = hi;
  }
}

// ------------------------------------------------------------------------------------------------ initial condition / export
// q^0 from (e,u,pi,Pi): Eqs. 32-33 (:267-269).  Compact arrays: physical cells, x fastest.
template <int EOS>
__global__ void __launch_bounds__(256) init_kernel(const __grid_constant__ DevParams P, const double* __restrict__ e_in, const double* __restrict__ u_in,
                                                   const double* __restrict__ pi_in, const double* __restrict__ Pi_in, real* q, real* e,
                                                   real* p, real* u, real* uprev) {
  const long long ncell = (long long)P.nx * P.ny * P.nz;
  const long long np = ncell * P.n_batch;
  long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= np) return;
  int i = (int)(w % P.nx);
  long long r = w / P.nx;
  int j = (int)(r % P.ny); r /= P.ny;
  int k = (int)(r % P.nz);
  int b = (int)(r / P.nz);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  const long long fs = P.fstride;
  real ee = e_in[w];
  real p0 = eos_p<EOS>(P, ee);
  real Pi = (Pi_in && P.bulk) ? Pi_in[w] : real(0.0);
  real Pt = p0 + Pi;
  real uu[4];
#pragma unroll
  for (int n = 0; n < 4; ++n) uu[n] = u_in[n * np + w];
  real pi[10];
#pragma unroll
  for (int n = 0; n < 10; ++n) pi[n] = (pi_in && P.shear) ? pi_in[n * np + w] : real(0.0);
  q[TTT * fs + c] = (ee + Pt) * uu[0] * uu[0] - Pt + pi[0];
#pragma unroll
  for (int n = 1; n < 4; ++n) q[n * fs + c] = (ee + Pt) * uu[0] * uu[n] + pi[n];
#pragma unroll
  for (int n = 0; n < 10; ++n) q[(PTT + n) * fs + c] = pi[n];
  q[BPI * fs + c] = Pi;
  e[c] = ee;
  p[c] = p0;
#pragma unroll
  for (int n = 0; n < 4; ++n) { u[n * fs + c] = uu[n]; uprev[n * fs + c] = uu[n]; }
}

// padded SoA (ncomp fields, the library's precision) <-> compact (the caller's arrays: always double)
template <bool TO_COMPACT>
__global__ void __launch_bounds__(256) pack_kernel(const __grid_constant__ DevParams P, real* padded, double* compact, int ncomp) {
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= np) return;
  int i = (int)(w % P.nx);
  long long r = w / P.nx;
  int j = (int)(r % P.ny); r /= P.ny;
  int k = (int)(r % P.nz);
  int b = (int)(r / P.nz);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  for (int n = 0; n < ncomp; ++n) {
    if (TO_COMPACT) compact[n * np + w] = (double)padded[n * P.fstride + c];
    else padded[n * P.fstride + c] = (real)compact[n * np + w];
  }
}

// p = P0(e) on every physical cell (used by vh_set_state)
template <int EOS>
__global__ void __launch_bounds__(256) pressure_kernel(const __grid_constant__ DevParams P, const real* __restrict__ e, real* p) {
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= np) return;
  int i = (int)(w % P.nx);
  long long r = w / P.nx;
  int j = (int)(r % P.ny); r /= P.ny;
  int k = (int)(r % P.nz);
  int b = (int)(r / P.nz);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  p[c] = eos_p<EOS>(P, e[c]);
}

// ------------------------------------------------------------------------------------------------ diagnostics
// Maxima over the physical cells, accumulated with atomicMax on the bit patterns (non-negative doubles order like integers):
// out[0] max T (freeze-out test "T < T_f everywhere", program-flow step 8, :494); out[1] max |u.u - 1| (:489);
// out[2] max |g_{mu nu} pi^{mu nu}|/(e+p), out[3] max_lambda |pi^{lambda mu} u_mu|/(e+p) (Eqs. 47-51, :318-331; lambda = eta entry
// times tau); out[4] max R_pi^-1 = sqrt(pi^{mu nu} pi_{mu nu})/P0, out[5] max R_Pi^-1 = |Pi|/P0 (Eq. 89, :826); out[6], out[7] max Knudsen
// numbers tau_pi |theta|, tau_Pi |theta| (:830): theta of A.11 with the differences of the sources (:424) and the solver's relaxation
// times (R14); cells with a non-finite quotient do not count, a switched-off sector gives 0.
// Second-order inverse Reynolds numbers (Eq. 90, :831): sqrt(J^{mu nu} J_{mu nu})/(2 eta sqrt(sigma^{mu nu} sigma_{mu nu})) and |J|/(zeta |theta|) with
// J^{mu nu}, J of Eq. 5 at n^mu = 0.  In the notation of Eqs. 41-46: J^{mu nu}/tau_pi = -(delta_pipi I2 - I3 + tau_pipi I4 - lambda_piPi Pi sigma^{mu nu}),
// J/tau_Pi = -(delta_PiPi Pi theta - lambda_Pipi pi^{mu nu} sigma_{mu nu}); eta/tau_pi and zeta/tau_Pi are the ratios the solver uses.
template <int EOS, bool MILNE>
__device__ __forceinline__ void second_order_reynolds(const DevParams& P, real t, const real u[4], const Kin& K, const real pi[10], real Pi,
                                                      real e, real& r2_shear, real& r2_bulk) {
  const real t2 = MILNE ? t * t : real(1.0);
  const real g[4] = {real(1.0), -real(1.0), -real(1.0), -t2};
  const real gi[4] = {real(1.0), -real(1.0), -real(1.0), -real(1.0) / t2};
  real p0, cs2;
  eos_p_cs2<EOS>(P, e, p0, cs2);
  const real T = eos_temperature<EOS>(P, e);
  const real eotp = (e + p0) * P.inv_ctaupi;
  const real zs = zeta_over_s(P, T), b = (real(1.0) / real(3.0)) - cs2;
  const real itP = fmin((zs > real(0.0)) ? T * b * b * P.inv_ctauPi / zs : inf_r(), P.relax_clamp);
  const real zotP = (zs > real(0.0)) ? zs * ((e + p0) / T) * itP : real(0.0);
  real S[4][4], W[4][4], Pm[4][4];
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = 0; n < 4; ++n) { S[m][n] = K.sig[sym(m, n)]; Pm[m][n] = pi[sym(m, n)]; }
  W[0][0] = W[1][1] = W[2][2] = W[3][3] = real(0.0);
  W[0][1] = K.W[0]; W[0][2] = K.W[1]; W[0][3] = K.W[2]; W[1][2] = K.W[3]; W[1][3] = K.W[4]; W[2][3] = K.W[5];
  W[1][0] = -K.W[0]; W[2][0] = -K.W[1]; W[3][0] = -K.W[2]; W[2][1] = -K.W[3]; W[3][1] = -K.W[4]; W[3][2] = -K.W[5];
  real B[4][4], C[4][4];      // B^{mu nu} = pi^{mu l} g_l W^{l nu};  C^{mu nu} = g_l pi^{mu l} sigma^{nu l}
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      real bb = real(0.0), cc = real(0.0);
#pragma unroll
      for (int l = 0; l < 4; ++l) { bb += Pm[m][l] * g[l] * W[l][n]; cc += g[l] * Pm[m][l] * S[n][l]; }
      B[m][n] = bb; C[m][n] = cc;
    }
  const real pisig = g[0] * C[0][0] + g[1] * C[1][1] + g[2] * C[2][2] + g[3] * C[3][3];
  real JJ = real(0.0), ss = real(0.0);
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = m; n < 4; ++n) {
      const int s = sym(m, n);
      const real Dmn = ((m == n) ? gi[m] : real(0.0)) - u[m] * u[n];
      const real I2 = K.theta * pi[s];
      const real I3 = kVorticitySign * (B[m][n] + B[n][m]);
      const real I4 = real(0.5) * (C[m][n] + C[n][m]) - (real(1.0) / real(3.0)) * Dmn * pisig;
      const real Jh = P.delta_pipi * I2 - I3 + P.tau_pipi * I4 - P.lambda_piPi * Pi * K.sig[s];
      const real w = g[m] * g[n] * ((m == n) ? real(1.0) : real(2.0));
      JJ += w * Jh * Jh;
      ss += w * K.sig[s] * K.sig[s];
    }
  const real IPi = P.delta_PiPi * Pi * K.theta - P.lambda_Pipi_coef * b * pisig;
  r2_shear = sqrt(fabs(JJ)) / (real(2.0) * eotp * sqrt(fabs(ss)));
  r2_bulk = fabs(IPi) / (zotP * fabs(K.theta));
}

template <int EOS, bool MILNE>
__global__ void __launch_bounds__(256) diagnostics_kernel(const __grid_constant__ DevParams P, const real* __restrict__ q, const real* __restrict__ e,
                                                          const real* __restrict__ p, const real* __restrict__ u, const real* __restrict__ u_prev,
                                                          real t, unsigned long long* __restrict__ out, double* __restrict__ maps) {
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const long long fs = P.fstride;
  const real t2 = MILNE ? t * t : real(1.0);
  real m[10] = {real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0)};
  for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < np; n += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(n % P.nx);
    const int j = (int)((n / P.nx) % P.ny);
    const int k = (int)((n / ((long long)P.nx * P.ny)) % P.nz);
    const int b = (int)(n / ((long long)P.nx * P.ny * P.nz));
    const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
    const real ee = e[c], pp = p[c];
    const real ut = u[c], ux = u[fs + c], uy = u[2 * fs + c], un = u[3 * fs + c];
    real pi[10];
#pragma unroll
    for (int s = 0; s < 10; ++s) pi[s] = q[(PTT + s) * fs + c];
    const real Pi = q[BPI * fs + c];
    const real norm = ut * ut - ux * ux - uy * uy - t2 * un * un;
    const real tr = pi[0] - pi[4] - pi[7] - t2 * pi[9];
    const real pipi = pi[0] * pi[0] - real(2.0) * (pi[1] * pi[1] + pi[2] * pi[2] + t2 * pi[3] * pi[3]) + pi[4] * pi[4] + real(2.0) * pi[5] * pi[5] +
                        real(2.0) * t2 * pi[6] * pi[6] + pi[7] * pi[7] + real(2.0) * t2 * pi[8] * pi[8] + t2 * t2 * pi[9] * pi[9];
    const real c0 = pi[0] * ut - pi[1] * ux - pi[2] * uy - t2 * pi[3] * un;
    const real c1 = pi[1] * ut - pi[4] * ux - pi[5] * uy - t2 * pi[6] * un;
    const real c2 = pi[2] * ut - pi[5] * ux - pi[7] * uy - t2 * pi[8] * un;
    const real c3 = (pi[3] * ut - pi[6] * ux - pi[8] * uy - t2 * pi[9] * un) * (MILNE ? t : real(1.0));
    const real iw = real(1.0) / (ee + pp), ip = real(1.0) / pp;
    real v[10];
    v[1] = fabs(norm - real(1.0));
    v[2] = fabs(tr) * iw;
    v[3] = fmax(fmax(fabs(c0), fabs(c1)), fmax(fabs(c2), fabs(c3))) * iw;
    v[4] = sqrt(fabs(pipi)) * ip;
    v[5] = fabs(Pi) * ip;
    // Knudsen numbers: theta = u^tau/tau + d_tau u^tau + d_i u^i (A.11), backward in time, central in space (:424)
    real theta = (MILNE ? ut / t : real(0.0)) + (ut - u_prev[c]) * P.inv_dtau;
    theta += (u[fs + c + 1] - u[fs + c - 1]) * (real(0.5) * P.inv_dx) + (u[2 * fs + c + P.NXp] - u[2 * fs + c - P.NXp]) * (real(0.5) * P.inv_dy);
    if (P.NZp > 1) theta += (u[3 * fs + c + P.plane] - u[3 * fs + c - P.plane]) * (real(0.5) * P.inv_dz);
    v[8] = real(0.0); v[9] = real(0.0);
    {
      if (P.shear || P.bulk) {       // Eq. 90: velocity gradients as in the source terms (:424), kinematics of App. A
        const real uc[4] = {ut, ux, uy, un};
        real dt[4], dx[4], dy[4], dn[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) {
          const real* ua = u + a * fs + c;
          dt[a] = (ua[0] - u_prev[a * fs + c]) * P.inv_dtau;
          dx[a] = (ua[1] - ua[-1]) * (real(0.5) * P.inv_dx);
          dy[a] = (ua[P.NXp] - ua[-P.NXp]) * (real(0.5) * P.inv_dy);
          dn[a] = (P.NZp > 1) ? (ua[P.plane] - ua[-P.plane]) * (real(0.5) * P.inv_dz) : real(0.0);
        }
        Kin K;
        kinematics<MILNE>(uc, dt, dx, dy, dn, t, K);
        real r2s, r2b;
        second_order_reynolds<EOS, MILNE>(P, t, uc, K, pi, Pi, ee, r2s, r2b);
        v[8] = (P.shear && isfinite(r2s)) ? r2s : real(0.0);
        v[9] = (P.bulk && isfinite(r2b)) ? r2b : real(0.0);
      }
    }
    const real T = eos_temperature<EOS>(P, ee);
    v[0] = T;
    real p0, cs2;
    eos_p_cs2<EOS>(P, ee, p0, cs2);
    const real itp = fmin(T * P.inv_ctaupi_etas, P.relax_clamp);
    const real zs = zeta_over_s(P, T), bb = (real(1.0) / real(3.0)) - cs2;
    const real itP = fmin((zs > real(0.0)) ? T * bb * bb * P.inv_ctauPi / zs : inf_r(), P.relax_clamp);
    const real kp = fabs(theta) / itp, kP = fabs(theta) / itP;
    v[6] = (P.shear && isfinite(kp)) ? kp : real(0.0);
    v[7] = (P.bulk && isfinite(kP)) ? kP : real(0.0);
#pragma unroll
    for (int s = 0; s < 10; ++s) m[s] = fmax(m[s], v[s]);
    if (maps) {                      // the same quantities cell by cell: maps[s * np + n], physical cells, x fastest
#pragma unroll
      for (int s = 0; s < 10; ++s) maps[s * np + n] = v[s];
    }
  }
#pragma unroll
  for (int s = 0; s < 10; ++s) {
    real v = m[s];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0 && v > real(0.0)) atomicMax(out + s, (unsigned long long)__double_as_longlong((double)v));
  }
}

// Whole padded eta planes of up to 21 arrays <-> a contiguous buffer of doubles (vh_halo_export / vh_halo_import: the exchange of an eta-slab
// decomposition).  buf[(a * n_planes + pl) * plane + w]; z0 = first padded plane index.
struct PlaneArgs { real* arr[21]; int n_arr; int z0; int n_planes; };
template <bool EXPORT>
__global__ void __launch_bounds__(256) plane_kernel(const __grid_constant__ DevParams P, const __grid_constant__ PlaneArgs G, double* __restrict__ buf) {
  const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= P.plane) return;
  const int pl = blockIdx.y % G.n_planes, a = blockIdx.y / G.n_planes;
  real* f = G.arr[a] + (long long)(G.z0 + pl) * P.plane + w;
  double* b = buf + ((long long)a * G.n_planes + pl) * P.plane + w;
  if (EXPORT) *b = (double)*f; else *f = (real)*b;
}

static __global__ void __launch_bounds__(256) fill_kernel(real* __restrict__ a, long long n, real v) {
  for (long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x; w < n; w += (long long)gridDim.x * blockDim.x) a[w] = v;
}

}  // namespace vh
