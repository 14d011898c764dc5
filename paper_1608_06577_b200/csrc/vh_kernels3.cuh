// vh_kernels3.cuh -- default stage kernel ("tile"): one CTA per TX x TY x TZ tile of cells, one thread per cell.
//
// Every array with a stencil (u^mu, p, the 15 q fields) is STREAMED through shared memory, one array at a time, by TMA
// tensor-map loads (cp.async.bulk.tensor, SASS UTMALDG) into an NSTAGE-deep ring of slots, each slot guarded by an
// mbarrier ("full") that the loads complete with their byte count.  A slot holds the star-shaped neighbourhood of the
// tile for one array: box A = (TX+4) x (TY+4) x TZ (the tile with its +-2 halo in x and y) plus, in 3+1d, two boxes of
// TX x TY x 2 planes below and above the tile (the +-2 halo in eta); ghost edges / corners are never loaded (:453).
// While array s is consumed the loads of arrays s+1 .. s+NSTAGE-1 are in flight.  A slot is handed back through a second
// mbarrier ("empty", NW arrivals): lane 0 of every warp arrives after the warp's reads, and the warp whose arrival was the
// last one pending re-arms "full" and issues the next loads into that slot - no block-wide barrier inside the stream.
// Per array the thread reads its 13-point star from the slot and accumulates
//   * the KT flux divergence of that field in x, y, eta (Eqs. 59-68) and
//   * that field's contribution to the sources of the four conservation laws (B.2-B.5 and G_c, :1013),
// so each neighbour value is read once.  The cell's own pi^{mu nu}, Pi (needed all at once by the relaxation sources,
// Eqs. 39-46) arrive by eleven more TMA boxes, in thread order.  The running values q + dtau C[q] are parked in shared
// memory (one slot per thread and field) until the epilogue: cell inversion (Eqs. 52-54, 72), regularisation
// (Eqs. 73-74), the stores and the ghost-cell replicas (Eqs. 75-76).  See DESIGN.md "Kernels".
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
  static constexpr int NW = NT / 32;                            // warps
  static constexpr int AX = TX + 2 * XOFF, AY = TY + 4;          // box A: the tile with XOFF (>= 2) cells on either side in x, 2 in y
  static constexpr int A_SIZE = AX * AY * TZ;                   // doubles in box A
  static constexpr int Z_SIZE = TWO_D ? 0 : TX * TY * 2;        // doubles in one eta-halo box
  static constexpr int SLOT = (A_SIZE + 2 * Z_SIZE + 31) / 32 * 32;   // elements per ring slot, padded so that every slot starts 128-byte aligned in either precision
  static constexpr int NSTAGE = 6;
  static constexpr int NCEN = 11;                               // centre rows: pi^{mu nu} (10), Pi
};
template <bool TWO_D, bool VISC> constexpr size_t tile_smem_bytes() {
  using T = Tile<TWO_D>;
  return (size_t)(T::NSTAGE * T::SLOT + (VISC ? NQ + T::NCEN : 4) * T::NT) * sizeof(real) + (2 * T::NSTAGE + 1) * sizeof(uint64_t) + T::NT * sizeof(int);
}

struct TileArgs {
  const real* q_in; const real* e_in; const real* p_in; const real* u_in; const real* u_prev;
  const real* q_n;
  const real* vL; const real* vR;
  real* q_out; real* e_out; real* p_out; real* u_out;
  Counters* cnt;
  real t, t_post;
  int a_q, a_u, a_p;      // index of q_in / u_in / p_in in the pool of padded arrays (outermost tensor-map coordinate)
  real* regfac;         // see StageArgs
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
// arrive on a barrier (release) and return the number of arrivals that were still pending BEFORE this one
__device__ __forceinline__ unsigned mbar_arrive_pending(uint64_t* bar) {
  uint64_t state;
  unsigned pending;
  asm volatile("mbarrier.arrive.shared::cta.b64 %0, [%1];" : "=l"(state) : "r"(smem_u32(bar)) : "memory");
  asm volatile("mbarrier.pending_count.b64 %0, %1;" : "=r"(pending) : "l"(state));
  return pending;
}

// ------------------------------------------------------------------------------------------------ flux of one field, one direction
// r -= dtau/dr (H_{+1/2} - H_{-1/2}) from the five values a0..a4 along the direction (Eqs. 61-68): H = cp q^+ + cm q^- with
// cp = (v^+ - a)/2, cm = (v^- + a)/2 (Eq. 61 regrouped), dtau/dr and the sign of the face folded into the coefficients.
template <bool THETA1>
__device__ __forceinline__ real flux_line(real a0, real a1, real a2, real a3, real a4, real cph, real cmh, real cpl,
                                            real cml, real theta, real r) {
  const real d0 = a1 - a0, d1 = a2 - a1, d2 = a3 - a2, d3 = a4 - a3;
  const real sm = minmod_slope<THETA1>(d0, d1, theta), s0 = minmod_slope<THETA1>(d1, d2, theta), sp = minmod_slope<THETA1>(d2, d3, theta);
  r = fma(cph, fma(-real(0.5), sp, a3), r);      // q^+_{+1/2} (Eq. 63)
  r = fma(cmh, fma(real(0.5), s0, a2), r);       // q^-_{+1/2} (Eq. 64)
  r = fma(cpl, fma(-real(0.5), s0, a2), r);      // q^+_{-1/2} (Eq. 65)
  r = fma(cml, fma(real(0.5), sm, a1), r);       // q^-_{-1/2} (Eq. 66)
  return r;
}

// face coefficients of one direction from the four state velocities (Eq. 62; w = dtau/dr)
__device__ __forceinline__ void face_coefficients(real vm_lo, real vp_lo, real vm_hi, real vp_hi, real w, real& cph, real& cmh,
                                                  real& cpl, real& cml) {
  const real a_lo = fmax(fabs(vm_lo), fabs(vp_lo)), a_hi = fmax(fabs(vm_hi), fabs(vp_hi));
  const real hw = real(0.5) * w;
  cph = hw * (a_hi - vp_hi); cmh = -hw * (vm_hi + a_hi);
  cpl = hw * (vp_lo - a_lo); cml = hw * (vm_lo + a_lo);
}

// ------------------------------------------------------------------------------------------------ relaxation sources, register-lean
// dtau * (S + G) for pi^{mu nu} (10) and Pi (B.10-B.12, Eqs. 39-46), one component at a time.  The terms of Eq. 42 are regrouped:
//   dtau J^{mn} = c_pi pi^{mn} + c_S sigma^{mn} - (u'^n A'^m + u'^m A'^n) - sum_l (pi^{ml} Y^{ln} + pi^{nl} Y^{lm}) + k3 g^{mn} - w G^{mn}
// with w = dtau/u^tau, u' = w u, A'^m = pi^{lm} Du_l + (tau_pipi pi:sigma / 6) u^m  (I_1 and the u u part of I_4's projector),
// Y^{ln} = w g_ll (0.5 tau_pipi sigma^{ln} - s_omega W^{ln})  (I_4 and -I_3 share the contraction with pi), k3 = w tau_pipi pi:sigma / 3,
// c_pi = dtau (div v - (1/tau_pi + delta_pipi theta)/u^tau), c_S = w (2 eta/tau_pi + lambda_piPi Pi).
// The evaluation is ordered so that few values are live at a time (the 128-register budget of a
// 512-thread CTA): (1) kinematic tensors sigma (10) and W (6) as scalars (A.5-A.19); (2) the pi-independent part
// c_pi pi^{mn} + c_S sigma^{mn} goes to the cell's park slot at once; (3) sigma, W are transformed IN PLACE into the 16
// entries of Y^{ln} (pair (l,n), l < n: Y^{ln} = g_l (b sigma + a W), Y^{nl} = g_n (b sigma - a W)); (4) the contraction with
// pi is added to the parked value.  pi(s) reads the cell's pi component from shared memory; ld/st access the park slot.
template <int EOS, bool MILNE, class PiGet, class ParkLd, class ParkSt>
__device__ __forceinline__ void relaxation_sources4(const DevParams& P, real t, const real (&u)[4], const real (&du)[4][4], PiGet pi,
                                                    real Pi, real e, real divv, real dt, ParkLd ld, ParkSt st) {
  const real ut = u[0], ux = u[1], uy = u[2], un = u[3];
  // Cartesian mode (R12): metric factors tau^2 -> 1 (t2, it2), Christoffel symbols -> 0 (it = Gamma^eta_{eta tau}, ct = Gamma^tau_{eta eta})
  const real t2 = MILNE ? t * t : real(1.0), it = MILNE ? rcp_fast(t) : real(0.0), it2 = MILNE ? it * it : real(1.0), ct = MILNE ? t : real(0.0);
  const real* dT = du[0]; const real* dX = du[1]; const real* dY = du[2]; const real* dN = du[3];
  // convective derivatives (A.5-A.8), expansion rate (A.11), covariant acceleration (A.9-A.10)
  const real dut = ut * dT[0] + ux * dX[0] + uy * dY[0] + un * dN[0];
  const real dux = ut * dT[1] + ux * dX[1] + uy * dY[1] + un * dN[1];
  const real duy = ut * dT[2] + ux * dX[2] + uy * dY[2] + un * dN[2];
  const real dun = ut * dT[3] + ux * dX[3] + uy * dY[3] + un * dN[3];
  const real th = ut * it + dT[0] + dX[1] + dY[2] + dN[3];
  const real th3 = th * (real(1.0) / real(3.0));
  const real un2 = un * un;
  const real Du0 = dut + ct * un2, Du1 = -dux, Du2 = -duy, Du3 = -t2 * (dun + real(2.0) * it * ut * un);
  // Z[0..9] = sigma^{mu nu} (A.12; slot order tt tx ty tn xx xy xn yy yn nn), Z[10..15] = W^{tx} W^{ty} W^{tn} W^{xy} W^{xn} W^{yn}
  real Z[16];
  Z[0] = -ct * ut * un2 + dT[0] - ut * dut + (ut * ut - real(1.0)) * th3;
  Z[1] = -real(0.5) * ct * un2 * ux + real(0.5) * (dT[1] - dX[0]) - real(0.5) * (ut * dux + ux * dut) + ut * ux * th3;
  Z[2] = -real(0.5) * ct * un2 * uy + real(0.5) * (dT[2] - dY[0]) - real(0.5) * (ut * duy + uy * dut) + ut * uy * th3;
  Z[3] = -real(0.5) * un * (real(2.0) * it * ut * ut + ct * un2) + real(0.5) * (dT[3] - dN[0] * it2) - real(0.5) * (ut * dun + un * dut) + ut * un * th3;
  Z[4] = -dX[1] - ux * dux + (real(1.0) + ux * ux) * th3;
  Z[5] = -real(0.5) * (dX[2] + dY[1]) - real(0.5) * (ux * duy + uy * dux) + ux * uy * th3;
  Z[6] = -ut * ux * un * it - real(0.5) * (dX[3] + dN[1] * it2) - real(0.5) * (ux * dun + un * dux) + ux * un * th3;
  Z[7] = -dY[2] - uy * duy + (real(1.0) + uy * uy) * th3;
  Z[8] = -ut * uy * un * it - real(0.5) * (dY[3] + dN[2] * it2) - real(0.5) * (uy * dun + un * duy) + uy * un * th3;
  Z[9] = -ut * it2 * it * (real(1.0) + real(2.0) * un2 * t2) - dN[3] * it2 - un * dun + (it2 + un2) * th3;
  Z[10] = real(0.5) * (dT[1] + dX[0]) + real(0.5) * (ux * dut - ut * dux) + real(0.5) * ct * un2 * ux;
  Z[11] = real(0.5) * (dT[2] + dY[0]) + real(0.5) * (uy * dut - ut * duy) + real(0.5) * ct * un2 * uy;
  Z[12] = un * it + real(0.5) * dT[3] + real(0.5) * dN[0] * it2 + real(0.5) * (un * dut - ut * dun) - ut * ut * un * it + real(0.5) * ct * un2 * un;
  Z[13] = real(0.5) * (dY[1] - dX[2]) + real(0.5) * (uy * dux - ux * duy);
  Z[14] = real(0.5) * dN[1] * it2 - real(0.5) * dX[3] + real(0.5) * (un * dux - ux * dun) - ux * ut * un * it;
  Z[15] = real(0.5) * dN[2] * it2 - real(0.5) * dY[3] + real(0.5) * (un * duy - uy * dun) - uy * ut * un * it;

  // transport coefficients (Eqs. 10-16; R14)
  real p, cs2;
  real T;
  if (EOS == 2) eos_lattice(P, e, p, cs2, T);      // one table lookup gives all three
  else { eos_p_cs2<EOS>(P, e, p, cs2); T = sqrt_fast(sqrt_fast(e * P.eos_a_inv)); }
  const real itp = fmin(T * P.inv_ctaupi_etas, P.relax_clamp);
  const real eotp2 = real(2.0) * (e + p) * P.inv_ctaupi;
  const real zs = zeta_over_s(P, T);
  const real b = (real(1.0) / real(3.0)) - cs2;
  real itP = (zs > real(0.0)) ? T * b * b * P.inv_ctauPi * rcp_fast(zs) : inf_r();
  itP = fmin(itP, P.relax_clamp);
  const real zotP = (zs > real(0.0)) ? zs * ((e + p) * rcp_fast(T)) * itP : real(0.0);
  const real iut = rcp_fast(ut);
  const real w = dt * iut;

  // pi^{mu nu} sigma_{mu nu}: symmetric double contraction with the metric weights of g = diag(1,-1,-1,-t2)
  const real pisig = pi(0) * Z[0] - real(2.0) * (pi(1) * Z[1] + pi(2) * Z[2]) + pi(4) * Z[4] + real(2.0) * pi(5) * Z[5] + pi(7) * Z[7] +
                       t2 * (real(2.0) * (pi(6) * Z[6] + pi(8) * Z[8] - pi(3) * Z[3]) + t2 * pi(9) * Z[9]);
  {     // Pi (B.10, Eq. 41): done first, its coefficients die here
    const real IPi = P.delta_PiPi * Pi * th - P.lambda_Pipi_coef * b * pisig;
    st(BPI, dt * fma(-fma(zotP, th, fma(Pi, itP, IPi)), iut, Pi * divv));
  }
  {     // (2) pi-independent part: c_pi pi^{mn} + c_S sigma^{mn}
    const real cpi = dt * fma(-iut, fma(P.delta_pipi, th, itp), divv);
    const real cS = w * fma(P.lambda_piPi, Pi, eotp2);
#pragma unroll
    for (int s = 0; s < 10; ++s) st(PTT + s, fma(cS, Z[s], cpi * pi(s)));
  }
  const real beta = P.tau_pipi * pisig * (real(1.0) / real(6.0));
  // A'^m = pi^{lm} Du_l + beta u^m;  u'^m = w u^m
  real Ap[4], up[4];
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    Ap[m] = fma(beta, u[m], pi(sym(0, m)) * Du0 + pi(sym(1, m)) * Du1 + pi(sym(2, m)) * Du2 + pi(sym(3, m)) * Du3);
    up[m] = w * u[m];
  }
  // (3) in place: Y[l][n] = g_l (bh sigma^{ln} + am W^{ln}), g = w (1,-1,-1,-t2), W antisymmetric
  real Y[4][4];
  {
    const real gl[4] = {w, -w, -w, -w * t2};
    const real bh = real(0.5) * P.tau_pipi, am = -kVorticitySign;
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      Y[l][l] = gl[l] * (bh * Z[sym(l, l)]);
#pragma unroll
      for (int n = l + 1; n < 4; ++n) {
        const int wi = (l == 0) ? 9 + n : ((l == 1) ? 11 + n : 15);      // 01 02 03 12 13 23 -> Z[10..15]
        const real c1 = bh * Z[sym(l, n)], c2 = am * Z[wi];
        Y[l][n] = gl[l] * (c1 + c2);
        Y[n][l] = gl[n] * (c1 - c2);
      }
    }
  }
  const real k3 = real(2.0) * w * beta;
  const real gi[4] = {real(1.0), -real(1.0), -real(1.0), -it2};
  const real g1 = w * ct * un, g2 = w * ut * it, g3 = w * un * it;      // Christoffel weights of G_pi (:300; R1, R2)
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = m; n < 4; ++n) {
      const int s = sym(m, n);
      real J = ld(PTT + s);
      J = fma(-up[n], Ap[m], J);
      J = fma(-up[m], Ap[n], J);
#pragma unroll
      for (int l = 0; l < 4; ++l) {
        J = fma(-pi(sym(m, l)), Y[l][n], J);
        J = fma(-pi(sym(n, l)), Y[l][m], J);
      }
      if (m == n) J = fma(k3, gi[m], J);
      // G_pi = u^a Gamma^mu_{ab} pi^{b nu} + (mu<->nu)
      if (s == 0) J = fma(-real(2.0) * g1, pi(3), J);
      if (s == 1) J = fma(-g1, pi(6), J);
      if (s == 2) J = fma(-g1, pi(8), J);
      if (s == 3) J = fma(-g1, pi(9), fma(-g2, pi(3), fma(-g3, pi(0), J)));
      if (s == 6) J = fma(-g2, pi(6), fma(-g3, pi(1), J));
      if (s == 8) J = fma(-g2, pi(8), fma(-g3, pi(2), J));
      if (s == 9) J = fma(-real(2.0) * g2, pi(9), fma(-real(2.0) * g3, pi(3), J));
      st(PTT + s, J);
    }
}

// ------------------------------------------------------------------------------------------------ regularisation factor
// tanh(rho)/rho of Eqs. 73-74 (R9) with the branch-free reciprocal / square roots of vh_math.cuh (the IEEE sqrt and division
// of regulation_factor() each cost a call-like slow path); same case analysis.
template <bool MILNE>
__device__ __forceinline__ real regulation_factor_fast(const DevParams& P, const real q[NQ], real e, real p0, const real u[4], real t) {
  const real t2 = MILNE ? t * t : real(1.0);
  const real* pi = q + PTT;
  const real Pi = q[BPI];
  const real pipi = pi[0] * pi[0] - real(2.0) * (pi[1] * pi[1] + pi[2] * pi[2] + t2 * pi[3] * pi[3]) + pi[4] * pi[4] + real(2.0) * pi[5] * pi[5] +
                      real(2.0) * t2 * pi[6] * pi[6] + pi[7] * pi[7] + real(2.0) * t2 * pi[8] * pi[8] + t2 * t2 * pi[9] * pi[9];
  const real tr = pi[0] - pi[4] - pi[7] - t2 * pi[9];
  const real PP = sqrt_fast(fabs(pipi + real(3.0) * Pi * Pi));
  real rho = PP * P.inv_rho_max * rsqrt_fast(e * e + real(3.0) * p0 * p0);
  const real den1 = P.xi0_rho_max * PP;
  if (PP > real(0.0) && isfinite(den1)) {
    const real id = rcp_fast(den1);
    // pi^{l mu} u_mu, u_mu = (ut,-ux,-uy,-t2 un); the l = eta entry is multiplied by tau
    const real c0 = pi[0] * u[0] - pi[1] * u[1] - pi[2] * u[2] - t2 * pi[3] * u[3];
    const real c1 = pi[1] * u[0] - pi[4] * u[1] - pi[5] * u[2] - t2 * pi[6] * u[3];
    const real c2 = pi[2] * u[0] - pi[5] * u[1] - pi[7] * u[2] - t2 * pi[8] * u[3];
    const real c3 = (pi[3] * u[0] - pi[6] * u[1] - pi[8] * u[2] - t2 * pi[9] * u[3]) * (MILNE ? t : real(1.0));
    const real m = fmax(fmax(fabs(tr), fabs(c0)), fmax(fmax(fabs(c1), fabs(c2)), fabs(c3)));
    rho = fmax(rho, m * id);
  }
  if (!isfinite(rho)) rho = real(0.0);
  return (rho < real(1e-8)) ? real(1.0) : tanh(rho) * rcp_fast(rho);
}

// ------------------------------------------------------------------------------------------------ the kernel
template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1, int STAGE, bool REGMAP = false>
__global__ void __launch_bounds__(Tile<TWO_D>::NT, kF32 ? 2 : 1)      // single precision: 64 registers, two CTAs per SM (8 % faster despite 48 bytes of spills)
    stage_tile_kernel(const __grid_constant__ DevParams P, const __grid_constant__ TileArgs A, const __grid_constant__ CUtensorMap mapA,
                      const __grid_constant__ CUtensorMap mapZ, const __grid_constant__ CUtensorMap mapC) {
  using T = Tile<TWO_D>;
  constexpr int TX = T::TX, TY = T::TY, TZ = T::TZ, NT = T::NT, AX = T::AX, AY = T::AY, NSTAGE = T::NSTAGE;
  constexpr int NF = VISC ? NQ : 4;
  constexpr int NSTREAM = 5 + NF;                    // u^tau, u^x, u^y, u^eta, p, then the q fields
  constexpr unsigned SLOT_BYTES = (T::A_SIZE + 2 * T::Z_SIZE) * sizeof(real);      // the bytes the boxes deliver (SLOT is padded)

  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* ring = reinterpret_cast<real*>(smem_raw);                       // [NSTAGE][SLOT]
  real* park = ring + NSTAGE * T::SLOT;                                   // [NF][NT]   running values
  real* cen = park + NF * NT;                                             // [NCEN][NT] the cell's own pi^{mu nu}, Pi (VISC)
  uint64_t* full = reinterpret_cast<uint64_t*>(cen + (VISC ? T::NCEN * NT : 0));   // [NSTAGE] ring slots, [NSTAGE] = centre rows
  uint64_t* empty = full + NSTAGE + 1;                                      // [NSTAGE] one arrival per warp that is done with the slot

  const int tid = threadIdx.x;
  const int tx = tid % TX, ty = (tid / TX) % TY, tz = tid / (TX * TY);
  const int nzb = (P.nz + TZ - 1) / TZ;
  const int b = blockIdx.z / nzb;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY, k0 = (blockIdx.z % nzb) * TZ;
  int i = i0 + tx, j = j0 + ty, k = k0 + tz;
  const bool valid = (i < P.nx) && (j < P.ny) && (k < P.nz);
  i = min(i, P.nx - 1); j = min(j, P.ny - 1); k = min(k, P.nz - 1);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  const long long fs = P.fstride;

  // ---- producer side: the loads of stream position s go into slot s % NSTAGE
  auto issue = [&](int s) {
    const int arr = (s < 4) ? A.a_u + s : ((s == 4) ? A.a_p : A.a_q + (s - 5));
    uint64_t* bar = &full[s % NSTAGE];
    real* dst = ring + (s % NSTAGE) * T::SLOT;
    mbar_arrive_expect_tx(bar, SLOT_BYTES);
    // padded coordinates: physical cell (i0, j0, k0) sits at (i0+XOFF, j0+2, k0+zoff); box A starts XOFF cells before it in x, two in y
    tma_load_5d(dst, &mapA, bar, i0, j0, TWO_D ? 0 : k0 + 2, b, arr);
    if (!TWO_D) {
      tma_load_5d(dst + T::A_SIZE, &mapZ, bar, i0 + XOFF, j0 + 2, k0, b, arr);                       // planes k0-2, k0-1
      tma_load_5d(dst + T::A_SIZE + T::Z_SIZE, &mapZ, bar, i0 + XOFF, j0 + 2, k0 + 2 + TZ, b, arr);  // planes k0+TZ, k0+TZ+1
    }
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s <= NSTAGE; ++s) mbar_init(&full[s], 1);
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) mbar_init(&empty[s], (unsigned)T::NW);
    fence_mbar_init();
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) issue(s);
    if (VISC) {      // the tile's own pi^{mu nu}, Pi: boxes of TX x TY x TZ land in thread order
      mbar_arrive_expect_tx(&full[NSTAGE], (unsigned)(T::NCEN * NT * sizeof(real)));
#pragma unroll 1
      for (int n = 0; n < T::NCEN; ++n) tma_load_5d(cen + n * NT, &mapC, &full[NSTAGE], i0 + XOFF, j0 + 2, TWO_D ? 0 : k0 + 2, b, A.a_q + PTT + n);
    }
  }
  // ---- consumer side: wait for stream position s; after the warp's reads, release(s) counts the warp out of the slot and the
  // warp that completes the count refills it (nobody waits for anybody here)
  auto acquire = [&](int s) -> const real* {
    mbar_wait(&full[s % NSTAGE], (unsigned)((s / NSTAGE) & 1));
    return ring + (s % NSTAGE) * T::SLOT;
  };
  const bool lane0 = (tid & 31) == 0;
  // `witness`: a word that depends on every value a lane loaded from the slot.  EVERY lane stores its word to shared memory (one conflict-free
  // store per warp) before the warp arrives: a lane's store cannot issue until its loads have written their registers, __syncwarp orders all
  // lanes' loads and stores before what lane 0 does next, and lane 0's arrival is a release - so no load of this warp is still in flight when
  // the arrival becomes visible.  (Issuing the loads before the arrival is not enough: an arrival does not wait for earlier loads to complete,
  // and the refill of an L2-resident halo can land within a few hundred cycles.  Found in round 2 with two resident CTAs per SM, where a queued
  // load of the refilling warp itself was overtaken about once per launch.)
  // The warp whose arrival completes the count refills the slot.  Its arrival is a read-modify-write of the barrier that has observed the
  // release-arrivals of all other warps (that is what "one arrival pending" says); the fence.acq_rel.cta after it turns that observation
  // into an acquire, so "every warp's reads of the slot, then the refill" rests on release / acquire, not on issue order.  Measured
  // alternatives for this acquire, per step at 128^3: none 1.2115 ms, this fence 1.214, mbarrier.try_wait.parity on the completed phase 1.2345,
  // mbarrier.test_wait.parity 1.277; a warp-wide xor (redux) of the witness instead of the per-lane stores costs another 0.012 ms.
  int* witness_sink = reinterpret_cast<int*>(empty + NSTAGE);      // [NT] one word per thread
  auto release = [&](int s, int witness) {
    if (s + NSTAGE < NSTREAM) {      // (uniform) a slot that is not used again needs no hand-back
      *reinterpret_cast<volatile int*>(witness_sink + tid) = witness;
      __syncwarp();
      // the arrival that finds one arrival pending is the last one of this use of the slot: that warp refills it
      if (lane0 && mbar_arrive_pending(&empty[s % NSTAGE]) == 1u) {
        __threadfence_block();
        issue(s + NSTAGE);
      }
    }
  };
  auto hi = [](real x) -> int { return kF32 ? __float_as_int((float)x) : __double2hiint((double)x); };

  // ---- per-thread offsets into a slot: centre in box A, and the four eta neighbours (box A, or the halo boxes at the tile faces)
  const int oc = (tz * AY + (ty + 2)) * AX + (tx + XOFF);
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

  const real t = A.t;
  const real t2 = MILNE ? t * t : real(1.0);
  const real it = MILNE ? rcp_fast(t) : real(1.0);
  const real it2 = it * it;
  const real dt = P.dtau;
  const real wt = MILNE ? dt * it : real(0.0);               // dtau/tau: weight of the geometric sources G_c (:1013)
  const real hinv[3] = {real(0.5) * P.inv_dx, real(0.5) * P.inv_dy, real(0.5) * P.inv_dz};
  const real wd[3] = {dt * hinv[0], dt * hinv[1], dt * hinv[2]};
  constexpr int ND = TWO_D ? 2 : 3;
  unsigned long long nfail = 0, nnonf = 0;
  real minfac = real(1.0);

  // centre-only operands: plain coalesced loads issued before the stream is consumed
  const unsigned long long record = *(volatile unsigned long long*)&A.cnt->min_reg_bits;      // filter of flush_counters
  const real ec = A.e_in[c];
  real upv[4] = {real(0.0), real(0.0), real(0.0), real(0.0)};
  if (VISC) {
#pragma unroll
    for (int n = 0; n < 4; ++n) upv[n] = A.u_prev[n * fs + c];
  }
  // ================================================================= phase 1: u^mu and p (velocity gradients, v^i, p terms)
  real uc[4], du[4][4], vm[3], vp[3], acc[4] = {real(0.0), real(0.0), real(0.0), real(0.0)}, divv = real(0.0), gPi = real(0.0);
  {
    real rm[3], rp[3];      // 1/u^tau at the six neighbours
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const real* s = acquire(m) + oc;
      uc[m] = s[0];
      const real xm = s[-1], xp = s[1], ym = s[-AX], yp = s[AX];
      real zm = real(0.0), zp = real(0.0);
      if (!TWO_D) { const real* sb = s - oc; zm = sb[ozm1]; zp = sb[ozp1]; }
      const real nm[3] = {xm, ym, zm}, np[3] = {xp, yp, zp};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if (d < ND) {
          du[d + 1][m] = (np[d] - nm[d]) * hinv[d];
          if (m == 0) { rm[d] = rcp_fast(nm[d]); rp[d] = rcp_fast(np[d]); }
          if (m == d + 1) { vm[d] = nm[d] * rm[d]; vp[d] = np[d] * rp[d]; divv = fma(vp[d] - vm[d], hinv[d], divv); }
        } else {
          du[d + 1][m] = real(0.0);
          if (m == d + 1) { vm[d] = real(0.0); vp[d] = real(0.0); }
        }
      }
      release(m, hi(uc[m]) ^ hi(du[1][m]) ^ hi(du[2][m]) ^ hi(du[3][m]));      // (the differences depend on all six neighbours)
    }
    const real* s = acquire(4) + oc;
    const real pc = s[0];
    const real xm = s[-1], xp = s[1], ym = s[-AX], yp = s[AX];
    real zm = real(0.0), zp = real(0.0);
    if (!TWO_D) { const real* sb = s - oc; zm = sb[ozm1]; zp = sb[ozp1]; }
    // P (v^i delta^nu_tau - g^{i nu}) part of B.2-B.5 (the Pi part follows when Pi streams through)
    acc[0] = fma(wd[0], fma(vm[0], xm, -vp[0] * xp), acc[0]);
    acc[0] = fma(wd[1], fma(vm[1], ym, -vp[1] * yp), acc[0]);
    acc[1] = wd[0] * (xm - xp);
    acc[2] = wd[1] * (ym - yp);
    if (!TWO_D) {
      acc[0] = fma(wd[2], fma(vm[2], zm, -vp[2] * zp), acc[0]);
      acc[3] = wd[2] * it2 * (zm - zp);
    }
    release(4, hi(pc) ^ hi(acc[0]) ^ hi(acc[1]) ^ hi(acc[2]) ^ hi(acc[3]));
    if (MILNE) {
      // G_c^tau = -(T^{tau tau} + tau^2 T^{eta eta})/tau with T^{eta eta} = (e + P)(u^eta)^2 + P/tau^2 + pi^{eta eta}, P = p + Pi (Eq. 34):
      // the e, p part here; the Pi, pi^{eta eta} and T^{tau mu} parts are added when those fields stream through
      const real g = t2 * uc[3] * uc[3];
      acc[0] = fma(-wt, fma(ec + pc, g, pc), acc[0]);
      gPi = wt * (g + real(1.0));
    }
  }

  // ================================================================= phase 2: relaxation sources (S_pi + G_pi, S_Pi) -> park
  if (VISC) {
#pragma unroll
    for (int n = 0; n < 4; ++n) du[0][n] = (uc[n] - upv[n]) * P.inv_dtau;      // backward difference in time (:424)
    mbar_wait(&full[NSTAGE], 0u);
    const real* mine = cen + tid;
    real* mypark = park + tid;
    relaxation_sources4<EOS, MILNE>(P, t, uc, du, [&](int s) { return mine[s * NT]; }, mine[10 * NT], ec, divv, dt,
                             [&](int slot) { return mypark[slot * NT]; }, [&](int slot, real J) { mypark[slot * NT] = J; });
  }

  // ================================================================= phase 3: the q fields (flux divergence + conservation sources)
  {
    real cf[3][4];      // face coefficients (cph, cmh, cpl, cml) per direction
    {
      const long long sd[3] = {1, (long long)P.NXp, P.plane};
      const real w[3] = {dt * P.inv_dx, dt * P.inv_dy, dt * P.inv_dz};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if (d < ND) {
          const real* vL = A.vL + d * fs + c;
          const real* vR = A.vR + d * fs + c;
          const int ext = (d == 0) ? P.nx : ((d == 1) ? P.ny : P.nz);
          face_coefficients(vR[-sd[d]], vL[0], vR[0], vL[sd[d]], (ext > 1) ? w[d] : real(0.0), cf[d][0], cf[d][1], cf[d][2], cf[d][3]);
        } else {
          cf[d][0] = cf[d][1] = cf[d][2] = cf[d][3] = real(0.0);
        }
      }
    }
    const real theta = P.theta;
    const real wt2 = wt * t2;
#pragma unroll
    for (int n = 0; n < NF; ++n) {
      const real* sb = acquire(5 + n);
      const real* s = sb + oc;
      const real a2 = s[0];
      const real x0 = s[-2], x1 = s[-1], x3 = s[1], x4 = s[2];
      const real y0 = s[-2 * AX], y1 = s[-AX], y3 = s[AX], y4 = s[2 * AX];
      real z0 = real(0.0), z1 = real(0.0), z3 = real(0.0), z4 = real(0.0);
      if (!TWO_D) { z0 = sb[ozm2]; z1 = sb[ozm1]; z3 = sb[ozp1]; z4 = sb[ozp2]; }
      real r = a2;
      if (VISC && n >= PTT) r += park[n * NT + tid];
      if (MILNE && n < 4) r = fma((n == 3) ? -real(3.0) * wt : -wt, a2, r);      // G_c (:1013): -T^{tau mu}/tau, -3 T^{tau eta}/tau
      // three independent chains (the coefficients of a direction of extent 1 are zero: no branch, the fluxes cancel identically)
      const real rx = flux_line<THETA1>(x0, x1, a2, x3, x4, cf[0][0], cf[0][1], cf[0][2], cf[0][3], theta, real(0.0));
      const real ry = flux_line<THETA1>(y0, y1, a2, y3, y4, cf[1][0], cf[1][1], cf[1][2], cf[1][3], theta, real(0.0));
      if (!TWO_D) r += flux_line<THETA1>(z0, z1, a2, z3, z4, cf[2][0], cf[2][1], cf[2][2], cf[2][3], theta, real(0.0));
      r += rx + ry;
      park[n * NT + tid] = r;
      release(5 + n, hi(r));      // r = the flux divergence of all three directions: it depends on every value of the star
      if (VISC && n >= PTT) {
        // this field's part of A^{i nu} = P (v^i delta^nu_tau - g^{i nu}) - v^i pi^{tau nu} + pi^{i nu}, differenced (B.2-B.5)
        const real gx = wd[0] * (x1 - x3), gy = wd[1] * (y1 - y3), gz = TWO_D ? real(0.0) : wd[2] * (z1 - z3);
        if (n <= PTN || n == BPI) {
          real vt = wd[0] * fma(vp[0], x3, -vm[0] * x1);
          vt = fma(wd[1], fma(vp[1], y3, -vm[1] * y1), vt);
          if (!TWO_D) vt = fma(wd[2], fma(vp[2], z3, -vm[2] * z1), vt);
          if (n == BPI) { acc[0] = fma(-gPi, a2, acc[0] - vt); acc[1] += gx; acc[2] += gy; acc[3] = fma(gz, it2, acc[3]); }
          else if (n == PTT) acc[0] += vt;
          else if (n == PTX) { acc[1] += vt; acc[0] += gx; }
          else if (n == PTY) { acc[2] += vt; acc[0] += gy; }
          else { acc[3] += vt; acc[0] += gz; }
        } else if (n == PXX) acc[1] += gx;
        else if (n == PXY) { acc[2] += gx; acc[1] += gy; }
        else if (n == PXN) { acc[3] += gx; acc[1] += gz; }
        else if (n == PYY) acc[2] += gy;
        else if (n == PYN) { acc[3] += gy; acc[2] += gz; }
        else { acc[3] += gz; acc[0] = fma(-wt2, a2, acc[0]); }       // PNN (with its part of tau^2 T^{eta eta} in G_c^tau)
      }
    }
  }

  // ================================================================= phase 4: stage result, inversion, regularisation, stores
  real qv[NQ];
#pragma unroll
  for (int n = 0; n < NQ; ++n) {
    real v = real(0.0);
    if (n < NF) {
      v = park[n * NT + tid];
      if (n < 4) v += acc[n];
      if (STAGE == 2) v = real(0.5) * (A.q_n[n * fs + c] + v);           // Eq. 70, beta = 1/2
      if (VISC && n >= PTT) { const bool on = (n == BPI) ? (P.bulk != 0) : (P.shear != 0); v = on ? v : real(0.0); }
    }
    qv[n] = v;
  }
  // Post: Eqs. 52-54, 72 then 73-74 (R8: regulate after the inversion).  Threads outside the grid (ragged tiles) carry a
  // benign state so that the warp-voted Newton loop is not held up by them.
  const real tp = A.t_post;
  const real tp2 = MILNE ? tp * tp : real(1.0);
  const real E = valid ? qv[TTT] - qv[PTT] : real(1.0);
  const real Mx = valid ? qv[TTX] - qv[PTX] : real(0.0), My = valid ? qv[TTY] - qv[PTY] : real(0.0), Mn = valid ? qv[TTN] - qv[PTN] : real(0.0);
  const real Pi = valid ? qv[BPI] : real(0.0);
  const real M2 = Mx * Mx + My * My + tp2 * Mn * Mn;
  bool fail;
  const real e = newton_single<EOS>(P, E, M2, Pi, ec, fail);
  if (fail) ++nfail;
  const real p0 = eos_p<EOS>(P, e);
  const real Pt = p0 + Pi;
  bool ut_ok;
  const real ut = u_tau_checked(E + Pt, e + Pt, ut_ok);        // Eq. 53
  const real inv = rcp_fast((e + Pt) * ut);                    // Eq. 54
  const real u[4] = {ut, Mx * inv, My * inv, Mn * inv};
  if (!(isfinite(e) && ut_ok)) ++nnonf;
  if (valid) {      // results that the regularisation does not touch go out first: their stores drain while rho is being computed
#pragma unroll
    for (int n = 0; n < 4; ++n) A.q_out[n * fs + c] = qv[n];
    A.e_out[c] = e;
    A.p_out[c] = p0;
#pragma unroll
    for (int n = 0; n < 4; ++n) A.u_out[n * fs + c] = u[n];
  }
  if (VISC) {
    const real fac = regulation_factor_fast<MILNE>(P, qv, e, p0, u, tp);
    minfac = fmin(minfac, fac);
    if constexpr (REGMAP) { if (valid) A.regfac[c] = fac; }      // Fig. 17 map (vh_enable_regulation_map): its own instantiation, the default kernel pays nothing
#pragma unroll
    for (int n = PTT; n < NQ; ++n) qv[n] *= fac;
  }
  if (valid) {
    const long long sy = P.NXp, sz = P.plane;
#pragma unroll
    for (int n = 4; n < NQ; ++n) A.q_out[n * fs + c] = qv[n];
    // ghost replicas (Eqs. 75-76): the outermost physical cell is copied into both ghost layers of its face (one rarely taken block)
    const bool edge = (i == 0) | (i == P.nx - 1) | (j == 0) | (j == P.ny - 1) | (!TWO_D && ((k == 0) | (k == P.nz - 1)));
    if (edge) {
      // one block per face, each testing its condition ONCE and then writing all 21 arrays: a warp on an x face (half of all warps
      // at 128^3) runs one block with one active lane and skips the other five
      auto replicate = [&](long long o1, long long o2) {
#pragma unroll
        for (int n = 0; n < NQ; ++n) { real* a = A.q_out + n * fs + c; a[o1] = qv[n]; a[o2] = qv[n]; }
        A.e_out[c + o1] = e; A.e_out[c + o2] = e;
        A.p_out[c + o1] = p0; A.p_out[c + o2] = p0;
#pragma unroll
        for (int n = 0; n < 4; ++n) { real* a = A.u_out + n * fs + c; a[o1] = u[n]; a[o2] = u[n]; }
      };
      if (i == 0) replicate(-1, -2);
      if (i == P.nx - 1) replicate(1, 2);
      if (j == 0) replicate(-sy, -2 * sy);
      if (j == P.ny - 1) replicate(sy, 2 * sy);
      if (!TWO_D) {
        if (k == 0) replicate(-sz, -2 * sz);
        if (k == P.nz - 1) replicate(sz, 2 * sz);
      }
    }
  }
  flush_counters(A.cnt, valid ? nfail : 0ull, valid ? nnonf : 0ull, valid ? minfac : real(1.0), record);
}

}  // namespace vh
