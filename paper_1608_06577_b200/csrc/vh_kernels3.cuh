// vh_kernels3.cuh -- default stage kernel ("tile"): one CTA per TX x TY x TZ tile of cells, one thread per cell.
//
// Every array with a stencil (u^mu, p, the 15 q fields) is STREAMED through shared memory, one array at a time, by TMA
// tensor-map loads (cp.async.bulk.tensor, SASS UTMALDG) into an NSTAGE-deep ring of slots, each slot guarded by an
// mbarrier ("full") that the loads complete with their byte count.  A slot holds the star-shaped neighbourhood of the
// tile for one array: box A = (TX+4) x (TY+4) x TZ (the tile with its +-2 halo in x and y) plus, in 3+1d, two boxes of
// TX x TY x 2 planes below and above the tile (the +-2 halo in eta); ghost edges / corners are never loaded (:453).
// While array s is consumed the loads of arrays s+1 .. s+NSTAGE-1 are in flight, so no thread ever waits on a global load
// in the stencil part.  Per array the thread reads its 13-point star from the slot and accumulates
//   * the KT flux divergence of that field in x, y, eta (Eqs. 59-68) and
//   * that field's contribution to the central-difference sources of the four conservation laws (B.2-B.5),
// so each neighbour value is read once.  The running values q + dtau C[q] are parked in shared memory (one slot per
// thread and field) until the epilogue: cell inversion (Eqs. 52-54, 72), regularisation (Eqs. 73-74), the stores and
// the ghost-cell replicas (Eqs. 75-76).  See DESIGN.md "Kernels".
#pragma once
#include <cuda.h>
#include <stdint.h>
#include "vh_kernels2.cuh"

namespace vh {

// ------------------------------------------------------------------------------------------------ tile geometry
template <bool TWO_D> struct Tile {
  static constexpr int TX = 32;
  static constexpr int TY = TWO_D ? 16 : 4;
  static constexpr int TZ = TWO_D ? 1 : 4;
  static constexpr int NT = TX * TY * TZ;                       // 512 threads
  static constexpr int AX = TX + 4, AY = TY + 4;
  static constexpr int A_SIZE = AX * AY * TZ;                   // doubles in box A
  static constexpr int Z_SIZE = TWO_D ? 0 : TX * TY * 2;        // doubles in one eta-halo box
  static constexpr int SLOT = A_SIZE + 2 * Z_SIZE;              // doubles per ring slot (13312 B / 5760 B: multiples of 128)
  static constexpr int NSTAGE = 4;
};

struct TileArgs {
  const double* q_in; const double* e_in; const double* p_in; const double* u_in; const double* u_prev;
  const double* q_n;
  const double* vL; const double* vR;
  double* q_out; double* e_out; double* p_out; double* u_out;
  Counters* cnt;
  double t, t_post;
  int a_q, a_u, a_p;      // index of q_in / u_in / p_in in the pool of padded arrays (outermost tensor-map coordinate)
};

// ------------------------------------------------------------------------------------------------ PTX: mbarrier + TMA
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "VH_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra VH_DONE_%=;\n"
      "bra VH_WAIT_%=;\n"
      "VH_DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2, int c3, int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
      : "memory");
}

// ------------------------------------------------------------------------------------------------ flux of one field, one direction
// r -= dtau/dr (H_{+1/2} - H_{-1/2}) from the five values a0..a4 along the direction (Eqs. 61-68; same grouping as flux_dir2)
template <bool THETA1>
__device__ __forceinline__ double flux_line(double a0, double a1, double a2, double a3, double a4, double cph, double cmh, double cpl,
                                            double cml, double ht, double r) {
  const double d0 = a1 - a0, d1 = a2 - a1, d2 = a3 - a2, d3 = a4 - a3;
  const double hm = half_slope2<THETA1>(d0, d1, ht), h0 = half_slope2<THETA1>(d1, d2, ht), hp = half_slope2<THETA1>(d2, d3, ht);
  r = fma(cph, a3 - hp, r);      // q^+_{+1/2} (Eq. 63)
  r = fma(cmh, a2 + h0, r);      // q^-_{+1/2} (Eq. 64)
  r = fma(cpl, a2 - h0, r);      // q^+_{-1/2} (Eq. 65)
  r = fma(cml, a1 + hm, r);      // q^-_{-1/2} (Eq. 66)
  return r;
}

// face coefficients of one direction from the four state velocities (Eq. 62; dtau/dr folded in, see flux_dir2)
__device__ __forceinline__ void face_coefficients(double vm_lo, double vp_lo, double vm_hi, double vp_hi, double w, double& cph, double& cmh,
                                                  double& cpl, double& cml) {
  const double a_lo = fmax(fabs(vm_lo), fabs(vp_lo)), a_hi = fmax(fabs(vm_hi), fabs(vp_hi));
  const double hw = 0.5 * w;
  cph = hw * (a_hi - vp_hi); cmh = -hw * (vm_hi + a_hi);
  cpl = hw * (vp_lo - a_lo); cml = hw * (vm_lo + a_lo);
}

// ------------------------------------------------------------------------------------------------ the kernel
template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1, int STAGE>
__global__ void __launch_bounds__(Tile<TWO_D>::NT, 1)
    stage_tile_kernel(const __grid_constant__ DevParams P, const __grid_constant__ TileArgs A, const __grid_constant__ CUtensorMap mapA,
                      const __grid_constant__ CUtensorMap mapZ) {
  using T = Tile<TWO_D>;
  constexpr int TX = T::TX, TY = T::TY, TZ = T::TZ, NT = T::NT, AX = T::AX, AY = T::AY, NSTAGE = T::NSTAGE;
  constexpr int NF = VISC ? NQ : 4;
  constexpr int NSTREAM = 5 + NF;                    // u^tau, u^x, u^y, u^eta, p, then the q fields
  constexpr unsigned SLOT_BYTES = T::SLOT * sizeof(double);

  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* ring = reinterpret_cast<double*>(smem_raw);                       // [NSTAGE][SLOT]
  double* park = ring + NSTAGE * T::SLOT;                                   // [NF][NT]
  uint64_t* full = reinterpret_cast<uint64_t*>(park + NF * NT);             // [NSTAGE]

  const int tid = threadIdx.x;
  const int tx = tid % TX, ty = (tid / TX) % TY, tz = tid / (TX * TY);
  const int nzb = (P.nz + TZ - 1) / TZ;
  const int b = blockIdx.z / nzb;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY, k0 = (blockIdx.z % nzb) * TZ;
  int i = i0 + tx, j = j0 + ty, k = k0 + tz;
  const bool valid = (i < P.nx) && (j < P.ny) && (k < P.nz);
  i = min(i, P.nx - 1); j = min(j, P.ny - 1); k = min(k, P.nz - 1);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + 2);
  const long long fs = P.fstride;

  // ---- producer: thread 0 issues the loads of stream position s into slot s % NSTAGE
  auto issue = [&](int s) {
    const int arr = (s < 4) ? A.a_u + s : ((s == 4) ? A.a_p : A.a_q + (s - 5));
    uint64_t* bar = &full[s % NSTAGE];
    double* dst = ring + (s % NSTAGE) * T::SLOT;
    mbar_arrive_expect_tx(bar, SLOT_BYTES);
    // padded coordinates: physical cell (i0, j0, k0) sits at (i0+2, j0+2, k0+zoff); box A starts two cells before it in x, y
    tma_load_5d(dst, &mapA, bar, i0, j0, TWO_D ? 0 : k0 + 2, b, arr);
    if (!TWO_D) {
      tma_load_5d(dst + T::A_SIZE, &mapZ, bar, i0 + 2, j0 + 2, k0, b, arr);                     // planes k0-2, k0-1
      tma_load_5d(dst + T::A_SIZE + T::Z_SIZE, &mapZ, bar, i0 + 2, j0 + 2, k0 + 2 + TZ, b, arr);  // planes k0+TZ, k0+TZ+1
    }
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) mbar_init(&full[s], 1);
    fence_mbar_init();
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) issue(s);
  }
  // consumer side of the ring: wait for stream position s; after the reads, release() lets thread 0 refill the slot
  auto acquire = [&](int s) -> const double* {
    mbar_wait(&full[s % NSTAGE], (unsigned)((s / NSTAGE) & 1));
    return ring + (s % NSTAGE) * T::SLOT;
  };
  auto release = [&](int s) {
    __syncthreads();
    if (tid == 0 && s + NSTAGE < NSTREAM) issue(s + NSTAGE);
  };

  // ---- per-thread offsets into a slot: centre in box A, and the four eta neighbours (box A, or the halo boxes at the tile faces)
  const int oc = (tz * AY + (ty + 2)) * AX + (tx + 2);
  int ozm2 = 0, ozm1 = 0, ozp1 = 0, ozp2 = 0;
  if (!TWO_D) {
    const int zl = T::A_SIZE + ty * TX + tx;               // plane 0 of the low halo box
    const int zh = zl + T::Z_SIZE;                         // plane 0 of the high halo box
    constexpr int PA = AX * AY, PZ = TX * TY;
    ozm2 = (tz >= 2) ? oc - 2 * PA : zl + tz * PZ;
    ozm1 = (tz >= 1) ? oc - PA : zl + PZ;
    ozp1 = (tz + 1 < TZ) ? oc + PA : zh;
    ozp2 = (tz + 2 < TZ) ? oc + 2 * PA : zh + (tz + 2 - TZ) * PZ;
  }

  const double t = A.t;
  const double t2 = MILNE ? t * t : 1.0;
  const double it = MILNE ? rcp_fast(t) : 1.0;
  const double it2 = it * it;
  const double dt = P.dtau;
  const double hinv[3] = {0.5 * P.inv_dx, 0.5 * P.inv_dy, 0.5 * P.inv_dz};
  const double wd[3] = {dt * hinv[0], dt * hinv[1], dt * hinv[2]};
  constexpr int ND = TWO_D ? 2 : 3;
  unsigned long long nfail = 0, nnonf = 0;
  double minfac = 1.0;

  // ================================================================= phase 1: u^mu and p (velocity gradients, v^i, p terms)
  double uc[4], du[4][4], vm[3], vp[3], acc[4] = {0.0, 0.0, 0.0, 0.0}, divv = 0.0, pc;
  {
    double rm[3], rp[3];      // 1/u^tau at the six neighbours
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const double* s = acquire(m) + oc;
      uc[m] = s[0];
      const double xm = s[-1], xp = s[1], ym = s[-AX], yp = s[AX];
      double zm = 0.0, zp = 0.0;
      if (!TWO_D) { const double* sb = s - oc; zm = sb[ozm1]; zp = sb[ozp1]; }
      release(m);
      const double nm[3] = {xm, ym, zm}, np[3] = {xp, yp, zp};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if (d < ND) {
          du[d + 1][m] = (np[d] - nm[d]) * hinv[d];
          if (m == 0) { rm[d] = rcp_fast(nm[d]); rp[d] = rcp_fast(np[d]); }
          if (m == d + 1) { vm[d] = nm[d] * rm[d]; vp[d] = np[d] * rp[d]; divv = fma(vp[d] - vm[d], hinv[d], divv); }
        } else {
          du[d + 1][m] = 0.0;
          if (m == d + 1) { vm[d] = 0.0; vp[d] = 0.0; }
        }
      }
    }
    const double* s = acquire(4) + oc;
    pc = s[0];
    const double xm = s[-1], xp = s[1], ym = s[-AX], yp = s[AX];
    double zm = 0.0, zp = 0.0;
    if (!TWO_D) { const double* sb = s - oc; zm = sb[ozm1]; zp = sb[ozp1]; }
    release(4);
    // P (v^i delta^nu_tau - g^{i nu}) part of B.2-B.5 (the Pi part follows when Pi streams through)
    acc[0] = fma(wd[0], fma(vm[0], xm, -vp[0] * xp), acc[0]);
    acc[0] = fma(wd[1], fma(vm[1], ym, -vp[1] * yp), acc[0]);
    acc[1] = wd[0] * (xm - xp);
    acc[2] = wd[1] * (ym - yp);
    if (!TWO_D) {
      acc[0] = fma(wd[2], fma(vm[2], zm, -vp[2] * zp), acc[0]);
      acc[3] = wd[2] * it2 * (zm - zp);
    }
  }

  // ================================================================= phase 2: per-cell sources (G_c, S_pi + G_pi, S_Pi)
  {
    const double ec = A.e_in[c];
    if (MILNE) {     // G_c (:1013), T^{eta eta} from Eq. 34
      const double Ptc = pc + (VISC ? A.q_in[BPI * fs + c] : 0.0);
      const double Tnn = fma((ec + Ptc) * uc[3], uc[3], fma(Ptc, it2, VISC ? A.q_in[PNN * fs + c] : 0.0));
      const double wt = dt * it;
      acc[0] = fma(-wt, fma(t2, Tnn, A.q_in[TTT * fs + c]), acc[0]);
      acc[1] = fma(-wt, A.q_in[TTX * fs + c], acc[1]);
      acc[2] = fma(-wt, A.q_in[TTY * fs + c], acc[2]);
      acc[3] = fma(-3.0 * wt, A.q_in[TTN * fs + c], acc[3]);
    }
    if (VISC) {
#pragma unroll
      for (int n = 0; n < 4; ++n) du[0][n] = (uc[n] - A.u_prev[n * fs + c]) * P.inv_dtau;      // backward difference in time (:424)
      Kin K;
      kinematics(uc, du[0], du[1], du[2], du[3], t, K);
      double pi[10];
#pragma unroll
      for (int n = 0; n < 10; ++n) pi[n] = A.q_in[(PTT + n) * fs + c];
      const double Pi = A.q_in[BPI * fs + c];
      dissipative_sources2<EOS>(P, t, uc, K, pi, Pi, ec, divv, [&](int slot, double J) { park[slot * NT + tid] = dt * J; });
    }
  }

  // ================================================================= phase 3: the q fields (flux divergence + conservation sources)
  {
    double cf[3][4];      // face coefficients (cph, cmh, cpl, cml) per direction
    {
      const long long sd[3] = {1, (long long)P.NXp, P.plane};
      const double w[3] = {dt * P.inv_dx, dt * P.inv_dy, dt * P.inv_dz};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if (d < ND) {
          const double* vL = A.vL + d * fs + c;
          const double* vR = A.vR + d * fs + c;
          face_coefficients(vR[-sd[d]], vL[0], vR[0], vL[sd[d]], w[d], cf[d][0], cf[d][1], cf[d][2], cf[d][3]);
        } else {
          cf[d][0] = cf[d][1] = cf[d][2] = cf[d][3] = 0.0;
        }
      }
    }
    const double ht = 0.5 * P.theta;
    const bool fx = P.nx > 1, fy = P.ny > 1, fz = !TWO_D;
#pragma unroll 1
    for (int n = 0; n < NF; ++n) {
      const double* sb = acquire(5 + n);
      const double* s = sb + oc;
      const double a2 = s[0];
      const double x0 = s[-2], x1 = s[-1], x3 = s[1], x4 = s[2];
      const double y0 = s[-2 * AX], y1 = s[-AX], y3 = s[AX], y4 = s[2 * AX];
      double z0 = 0.0, z1 = 0.0, z3 = 0.0, z4 = 0.0;
      if (!TWO_D) { z0 = sb[ozm2]; z1 = sb[ozm1]; z3 = sb[ozp1]; z4 = sb[ozp2]; }
      release(5 + n);
      double r = a2;
      if (VISC && n >= PTT) r += park[n * NT + tid];
      if (fx) r = flux_line<THETA1>(x0, x1, a2, x3, x4, cf[0][0], cf[0][1], cf[0][2], cf[0][3], ht, r);
      if (fy) r = flux_line<THETA1>(y0, y1, a2, y3, y4, cf[1][0], cf[1][1], cf[1][2], cf[1][3], ht, r);
      if (fz) r = flux_line<THETA1>(z0, z1, a2, z3, z4, cf[2][0], cf[2][1], cf[2][2], cf[2][3], ht, r);
      park[n * NT + tid] = r;
      if (VISC && n >= PTT) {
        // this field's part of A^{i nu} = P (v^i delta^nu_tau - g^{i nu}) - v^i pi^{tau nu} + pi^{i nu}, differenced (B.2-B.5)
        const double gx = wd[0] * (x1 - x3), gy = wd[1] * (y1 - y3), gz = TWO_D ? 0.0 : wd[2] * (z1 - z3);
        if (n <= PTN || n == BPI) {
          double vt = wd[0] * fma(vp[0], x3, -vm[0] * x1);
          vt = fma(wd[1], fma(vp[1], y3, -vm[1] * y1), vt);
          if (!TWO_D) vt = fma(wd[2], fma(vp[2], z3, -vm[2] * z1), vt);
          if (n == BPI) { acc[0] -= vt; acc[1] += gx; acc[2] += gy; acc[3] = fma(gz, it2, acc[3]); }
          else if (n == PTT) acc[0] += vt;
          else if (n == PTX) { acc[1] += vt; acc[0] += gx; }
          else if (n == PTY) { acc[2] += vt; acc[0] += gy; }
          else { acc[3] += vt; acc[0] += gz; }
        } else if (n == PXX) acc[1] += gx;
        else if (n == PXY) { acc[2] += gx; acc[1] += gy; }
        else if (n == PXN) { acc[3] += gx; acc[1] += gz; }
        else if (n == PYY) acc[2] += gy;
        else if (n == PYN) { acc[3] += gy; acc[2] += gz; }
        else acc[3] += gz;       // PNN
      }
    }
  }

  // ================================================================= phase 4: stage result, inversion, regularisation, stores
  double qv[NQ];
#pragma unroll
  for (int n = 0; n < NQ; ++n) {
    double v = 0.0;
    if (n < NF) {
      v = park[n * NT + tid];
      if (n < 4) v += acc[n];
      if (STAGE == 2) v = 0.5 * (A.q_n[n * fs + c] + v);           // Eq. 70, beta = 1/2
      if (VISC && n >= PTT) { const bool on = (n == BPI) ? (P.bulk != 0) : (P.shear != 0); v = on ? v : 0.0; }
    }
    qv[n] = v;
  }
  // Post: Eqs. 52-54, 72 then 73-74 (R8: regulate after the inversion)
  const double tp = A.t_post;
  const double tp2 = MILNE ? tp * tp : 1.0;
  // threads outside the grid (ragged tiles) carry a benign state so that the warp-voted Newton loop is not held up by them
  const double E = valid ? qv[TTT] - qv[PTT] : 1.0;
  const double Mx = valid ? qv[TTX] - qv[PTX] : 0.0, My = valid ? qv[TTY] - qv[PTY] : 0.0, Mn = valid ? qv[TTN] - qv[PTN] : 0.0;
  const double Pi = valid ? qv[BPI] : 0.0;
  const double M2 = Mx * Mx + My * My + tp2 * Mn * Mn;
  bool fail;
  const double e = newton_single<EOS>(P, E, M2, Pi, A.e_in[c], fail);
  if (fail) ++nfail;
  const double p0 = eos_p<EOS>(P, e);
  const double Pt = p0 + Pi;
  const double ut = sqrt_fast((E + Pt) * rcp_fast(e + Pt));      // Eq. 53
  const double inv = rcp_fast((e + Pt) * ut);                    // Eq. 54
  const double u[4] = {ut, Mx * inv, My * inv, Mn * inv};
  if (!(isfinite(e) && isfinite(ut))) ++nnonf;
  if (VISC) {
    const double fac = regulation_factor<MILNE>(P, qv, e, p0, u, tp);
    minfac = fmin(minfac, fac);
#pragma unroll
    for (int n = PTT; n < NQ; ++n) qv[n] *= fac;
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
    for (int n = 0; n < NQ; ++n) put(A.q_out + n * fs, qv[n]);
    put(A.e_out, e);
    put(A.p_out, p0);
#pragma unroll
    for (int n = 0; n < 4; ++n) put(A.u_out + n * fs, u[n]);
  }
  flush_counters(A.cnt, valid ? nfail : 0ull, valid ? nnonf : 0ull, valid ? minfac : 1.0);
}

}  // namespace vh
