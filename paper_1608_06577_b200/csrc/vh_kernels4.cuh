// vh_kernels4.cuh -- default velocity kernel ("velocity tile"): the interface-state inversions of one Euler stage with the
// nine fields that enter Eq. 72 (T^{tau mu}, pi^{tau mu}, Pi) staged in shared memory by TMA.
//
// One CTA per VX x VY x VZ tile, one thread per cell.  Lane 0 of each warp issues, for one of the NV fields, one tensor-map box of the
// tile with a 1-cell halo in y (and the 2-cell halo in x that the 16-byte start alignment of a box forces) plus, in 3+1d, one
// plane below and one above the tile; all loads complete on ONE mbarrier, so the CTA waits once and then works from shared
// memory only.  With 3-4 KB per field six 128-thread CTAs (3+1d) are resident per SM and hide one another's load latency.
// Arithmetic as in velocity_kernel (vh_kernels2.cuh): per
// direction the two reconstructed states the cell owns are inverted once, as a pair (Eqs. 63-66, 72; Alg. 3 :667-672).
#pragma once
#include "vh_kernels3.cuh"

namespace vh {

template <bool TWO_D> struct VTile {
  static constexpr int VX = 32;
  static constexpr int VY = TWO_D ? 8 : 4;
  static constexpr int VZ = 1;                                  // one eta plane per CTA: small CTAs, many per SM
  static constexpr int NT = VX * VY * VZ;                       // 128 threads (3+1d), 256 (2+1d)
  static constexpr int AX = VX + 2 * XOFF, AY = VY + 2;
  static constexpr int A_SIZE = AX * AY * VZ;                   // doubles in box A (tile + halo in x, y)
  static constexpr int Z_SIZE = TWO_D ? 0 : VX * VY;            // doubles in one eta-halo plane
  static constexpr int A_PAD = (A_SIZE + 31) / 32 * 32;         // offset of the eta-halo planes: every TMA destination 128-byte aligned in either precision
  static constexpr int SLOT = (A_PAD + 2 * Z_SIZE + 31) / 32 * 32;   // elements per field
};
template <bool TWO_D, bool VISC> constexpr size_t vtile_smem_bytes() {
  return (size_t)((VISC ? 9 : 4) * VTile<TWO_D>::SLOT) * sizeof(real) + sizeof(uint64_t);
}

struct VelTileArgs {
  const real* e;               // Newton guess: e of the cell (R6)
  real* vL; real* vR;        // [3][fstride]: velocity of the state at the cell's low / high face, per direction
  Counters* cnt;
  real t;
  int a_q;                       // index of q_in in the pool of padded arrays (outermost tensor-map coordinate)
  int nb_lo, nb_hi;              // eta-slab decomposition: another slab owns the cells beyond the low / high eta face (it counts that interface's outer state)
};

template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1>
__global__ void __launch_bounds__(VTile<TWO_D>::NT, TWO_D ? 3 : 6)
    velocity_tile_kernel(const __grid_constant__ DevParams P, const __grid_constant__ VelTileArgs A, const __grid_constant__ CUtensorMap mapVA,
                         const __grid_constant__ CUtensorMap mapVZ) {
  using T = VTile<TWO_D>;
  constexpr int VX = T::VX, VY = T::VY, VZ = T::VZ, AX = T::AX, AY = T::AY;
  constexpr int NV = VISC ? 9 : 4;
  constexpr int ND = TWO_D ? 2 : 3;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* slots = reinterpret_cast<real*>(smem_raw);                      // [NV][SLOT]
  uint64_t* full = reinterpret_cast<uint64_t*>(slots + NV * T::SLOT);

  const int tid = threadIdx.x;
  const int tx = tid % VX, ty = (tid / VX) % VY, tz = tid / (VX * VY);
  const int nzb = (P.nz + VZ - 1) / VZ;
  const int b = blockIdx.z / nzb;
  const int i0 = blockIdx.x * VX, j0 = blockIdx.y * VY, k0 = (blockIdx.z % nzb) * VZ;
  int i = i0 + tx, j = j0 + ty, k = k0 + tz;
  const bool valid = (i < P.nx) && (j < P.ny) && (k < P.nz);
  i = min(i, P.nx - 1); j = min(j, P.ny - 1); k = min(k, P.nz - 1);
  const long long c = (long long)b * P.bstride + (long long)(k + P.zoff) * P.plane + (long long)(j + 2) * P.NXp + (i + XOFF);
  const long long fs = P.fstride;

  if (tid == 0) {
    mbar_init(full, 1);
    fence_mbar_init();
    mbar_arrive_expect_tx(full, (unsigned)(NV * (T::A_SIZE + 2 * T::Z_SIZE) * sizeof(real)));      // the bytes the boxes deliver (SLOT is padded)
  }
  const real guess = A.e[c];
  __syncthreads();                 // the barrier is initialised and armed before anybody issues a load or waits on it
  // lane 0 of every warp issues the boxes of one field (warp 0 also those of the ninth): the loads start in parallel
  if ((tid & 31) == 0) {
#pragma unroll 1
    for (int m = tid >> 5; m < NV; m += T::NT / 32) {
      const int arr = A.a_q + ((m < 4) ? m : ((m < 8) ? PTT + (m - 4) : BPI));
      real* dst = slots + m * T::SLOT;
      // padded coordinates: physical cell (i0, j0, k0) sits at (i0+XOFF, j0+2, k0+zoff)
      tma_load_5d(dst, &mapVA, full, i0, j0 + 1, TWO_D ? 0 : k0 + 2, b, arr);
      if (!TWO_D) {
        tma_load_5d(dst + T::A_PAD, &mapVZ, full, i0 + XOFF, j0 + 2, k0 + 1, b, arr);                   // plane k0-1
        tma_load_5d(dst + T::A_PAD + T::Z_SIZE, &mapVZ, full, i0 + XOFF, j0 + 2, k0 + 2 + VZ, b, arr);   // plane k0+VZ
      }
    }
  }

  // offsets into a field's slot: centre, and the two eta neighbours (box A, or a halo plane at the tile faces)
  const int oc = (tz * AY + (ty + 1)) * AX + (tx + XOFF);
  int ozm = oc, ozp = oc;
  if (!TWO_D) {
    const int zl = T::A_PAD + ty * VX + tx;
    ozm = (tz >= 1) ? oc - AX * AY : zl;
    ozp = (tz + 1 < VZ) ? oc + AX * AY : zl + T::Z_SIZE;
  }
  const real t2 = MILNE ? A.t * A.t : real(1.0);
  const real theta = P.theta;
  unsigned long long nfail = 0;
  mbar_wait(full, 0u);

#pragma unroll
  for (int d = 0; d < ND; ++d) {
    const int om = (d == 0) ? oc - 1 : ((d == 1) ? oc - AX : ozm);
    const int op = (d == 0) ? oc + 1 : ((d == 1) ? oc + AX : ozp);
    const long long s = (d == 0) ? 1 : ((d == 1) ? (long long)P.NXp : P.plane);
    const int pos = (d == 0) ? i : ((d == 1) ? j : k);
    const int ext = (d == 0) ? P.nx : ((d == 1) ? P.ny : P.nz);
    // L = state at the low face (q^+_{c-1/2}), R = state at the high face (q^-_{c+1/2})
    real wL[5], wR[5];     // E, Mx, My, Mn, Pi
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const real* f = slots + m * T::SLOT;
      const real a0 = f[om], a1 = f[oc], a2 = f[op];
      const real sl = minmod_slope<THETA1>(a1 - a0, a2 - a1, theta);      // Eqs. 67-68; the half-cell factor 1/2 sits in the FMAs
      wL[m] = fma(-real(0.5), sl, a1); wR[m] = fma(real(0.5), sl, a1);
    }
    wL[4] = real(0.0); wR[4] = real(0.0);
    if (VISC) {
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        const real* f = slots + (4 + m) * T::SLOT;
        const real a0 = f[om], a1 = f[oc], a2 = f[op];
        const real sl = minmod_slope<THETA1>(a1 - a0, a2 - a1, theta);
        wL[m] -= fma(-real(0.5), sl, a1); wR[m] -= fma(real(0.5), sl, a1);
      }
      const real* f = slots + 8 * T::SLOT;
      const real a0 = f[om], a1 = f[oc], a2 = f[op];
      const real sl = minmod_slope<THETA1>(a1 - a0, a2 - a1, theta);
      wL[4] = fma(-real(0.5), sl, a1); wR[4] = fma(real(0.5), sl, a1);
    }
    NewtonState SL, SR;
    SL.E = wL[0]; SL.Pi = wL[4]; SL.M2 = wL[1] * wL[1] + wL[2] * wL[2] + t2 * wL[3] * wL[3];     // :339
    SR.E = wR[0]; SR.Pi = wR[4]; SR.M2 = wR[1] * wR[1] + wR[2] * wR[2] + t2 * wR[3] * wR[3];
    newton_pair<EOS>(P, SL, SR, guess, guess);
    real vl = wL[d + 1] * SL.rden, vr = wR[d + 1] * SR.rden;      // v^r = M_r/(E + P0 + Pi)  (Eqs. 53-54)
    if (SL.fail) vl = clip_velocity(vl);
    if (SR.fail) vr = clip_velocity(vr);
    // status counter: every state of every interface once (see velocity_kernel); nothing along a direction of extent 1
    if (ext > 1) {
      nfail += (SL.fail ? 1u : 0u) + (SR.fail ? 1u : 0u);
      // the outer state of a boundary interface is the ghost cell's, equal to this one (Eqs. 75-76) - unless a neighbouring slab owns it
      if (pos == 0 && SL.fail && !(d == 2 && A.nb_lo)) ++nfail;
      if (pos == ext - 1 && SR.fail && !(d == 2 && A.nb_hi)) ++nfail;
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

}  // namespace vh
