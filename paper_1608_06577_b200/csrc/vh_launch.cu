// vh_launch.cu -- kernel launches of one Euler stage for ONE combination of (EOS, viscous, Milne); compiled once per
// combination with -DVH_COMBO=k so that the instantiations build in parallel (paper_1608_06577_b200/build.py).
#include "vh_internal.cuh"

using namespace vh;

#ifndef VH_COMBO
#error "compile with -DVH_COMBO=0..11"
#endif
#define debug_sync vh_debug_sync

template <int EOS, bool VISC, bool MILNE, bool TWO_D>
static cudaError_t launch_stage_t(vh_handle* h, int stage, const StageArgs& A) {
  const DevParams& P = h->P;
  dim3 block(32, 8);
  dim3 grid((P.nx + 31) / 32, (P.ny + 7) / 8, P.nz * P.n_batch);
  if (stage == 1) stage_cell_kernel<EOS, VISC, MILNE, TWO_D, 1><<<grid, block, 0, h->stream>>>(P, A);
  else stage_cell_kernel<EOS, VISC, MILNE, TWO_D, 2><<<grid, block, 0, h->stream>>>(P, A);
  h->launches++;
  return debug_sync(h, stage == 1 ? "stage 1 kernel" : "stage 2 kernel");
}
template <int EOS, bool VISC, bool MILNE>
static cudaError_t launch_stage_d(vh_handle* h, int stage, const StageArgs& A) {
  return h->two_d ? launch_stage_t<EOS, VISC, MILNE, true>(h, stage, A) : launch_stage_t<EOS, VISC, MILNE, false>(h, stage, A);
}

// ---- split pipeline (variant 0): velocity kernel + stage kernel (vh_kernels2.cuh)
template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1>
static cudaError_t launch_split_t(vh_handle* h, int stage, const StageArgs& S, cudaEvent_t mid) {
  const DevParams& P = h->P;
  constexpr int BX = 32, BY = TWO_D ? 8 : 4, BZ = TWO_D ? 1 : 2;
  dim3 block(BX, BY, BZ);
  dim3 grid((P.nx + BX - 1) / BX, (P.ny + BY - 1) / BY, ((P.nz + BZ - 1) / BZ) * P.n_batch);
  VelArgs V{S.q_in, S.e_in, h->vL, h->vR, S.cnt, S.t};
  velocity_kernel<EOS, VISC, MILNE, TWO_D, THETA1, BX, BY, BZ><<<grid, block, 0, h->stream>>>(P, V);
  h->launches++;
  cudaError_t e = debug_sync(h, "velocity kernel");
  if (e != cudaSuccess) return e;
  if (mid) cudaEventRecord(mid, h->stream);
  Stage2Args A{S.q_in, S.e_in, S.p_in, S.u_in, S.u_prev, S.q_n, h->vL, h->vR, S.q_out, S.e_out, S.p_out, S.u_out, S.cnt, S.t, S.t_post, S.regfac};
  if (stage == 1) stage_kernel<EOS, VISC, MILNE, TWO_D, THETA1, 1, BX, BY, BZ, VH_STAGE_MINB><<<grid, block, 0, h->stream>>>(P, A);
  else stage_kernel<EOS, VISC, MILNE, TWO_D, THETA1, 2, BX, BY, BZ, VH_STAGE_MINB><<<grid, block, 0, h->stream>>>(P, A);
  h->launches++;
  return debug_sync(h, stage == 1 ? "stage 1 kernel" : "stage 2 kernel");
}
template <int EOS, bool VISC, bool MILNE>
static cudaError_t launch_split_d(vh_handle* h, int stage, const StageArgs& A, cudaEvent_t mid) {
  const bool th1 = h->prm.minmod_theta == 1.0;
  if (h->two_d) return th1 ? launch_split_t<EOS, VISC, MILNE, true, true>(h, stage, A, mid) : launch_split_t<EOS, VISC, MILNE, true, false>(h, stage, A, mid);
  return th1 ? launch_split_t<EOS, VISC, MILNE, false, true>(h, stage, A, mid) : launch_split_t<EOS, VISC, MILNE, false, false>(h, stage, A, mid);
}

// ---- tile pipeline (variant 0): velocity kernel + TMA tile kernel (vh_kernels3.cuh)
template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1, int STAGE, bool REGMAP = false>
static cudaError_t launch_tile_kernel(vh_handle* h, const TileArgs& A) {
  using T = Tile<TWO_D>;
  constexpr size_t smem = tile_smem_bytes<TWO_D, VISC>();
  if constexpr (VISC && STAGE == 2 && !REGMAP) {      // the map of Fig. 17 is stored by an instantiation of its own
    if (A.regfac) return launch_tile_kernel<EOS, VISC, MILNE, TWO_D, THETA1, STAGE, true>(h, A);
  }
  auto kern = stage_tile_kernel<EOS, VISC, MILNE, TWO_D, THETA1, STAGE, REGMAP>;
  if (cudaError_t e = vh_opt_in_smem(h, (const void*)kern, smem); e != cudaSuccess) return e;
  const DevParams& P = h->P;
  dim3 grid((P.nx + T::TX - 1) / T::TX, (P.ny + T::TY - 1) / T::TY, ((P.nz + T::TZ - 1) / T::TZ) * P.n_batch);
  kern<<<grid, T::NT, smem, h->stream>>>(P, A, h->mapA, h->mapZ, h->mapC);
  h->launches++;
  return debug_sync(h, STAGE == 1 ? "stage 1 tile kernel" : "stage 2 tile kernel");
}
template <int EOS, bool VISC, bool MILNE, bool TWO_D, bool THETA1>
static cudaError_t launch_tile_t(vh_handle* h, int stage, const StageArgs& S, cudaEvent_t mid, int part) {
  const DevParams& P = h->P;
  const long long fs = P.fstride;
  if (part != 2) {      // part: 0 both kernels, 1 velocity kernel only, 2 stage kernel only (vh_step_part)
    using V = VTile<TWO_D>;
    constexpr size_t vsmem = vtile_smem_bytes<TWO_D, VISC>();
    auto vkern = velocity_tile_kernel<EOS, VISC, MILNE, TWO_D, THETA1>;
    if (cudaError_t e = vh_opt_in_smem(h, (const void*)vkern, vsmem); e != cudaSuccess) return e;
    dim3 grid((P.nx + V::VX - 1) / V::VX, (P.ny + V::VY - 1) / V::VY, ((P.nz + V::VZ - 1) / V::VZ) * P.n_batch);
    VelTileArgs VA{S.e_in, h->vL, h->vR, S.cnt, S.t, (int)((S.q_in - h->pool) / fs), h->slab_nb[0] ? 1 : 0, h->slab_nb[1] ? 1 : 0};
    vkern<<<grid, V::NT, vsmem, h->stream>>>(P, VA, h->mapVA, h->mapVZ);
    h->launches++;
    cudaError_t e = debug_sync(h, "velocity tile kernel");
    if (e != cudaSuccess) return e;
  }
  if (mid) cudaEventRecord(mid, h->stream);
  if (part == 1) return cudaSuccess;
  TileArgs A{S.q_in, S.e_in, S.p_in, S.u_in, S.u_prev, S.q_n, h->vL, h->vR, S.q_out, S.e_out, S.p_out, S.u_out, S.cnt, S.t, S.t_post,
             (int)((S.q_in - h->pool) / fs), (int)((S.u_in - h->pool) / fs), (int)((S.p_in - h->pool) / fs), S.regfac};
  return (stage == 1) ? launch_tile_kernel<EOS, VISC, MILNE, TWO_D, THETA1, 1>(h, A) : launch_tile_kernel<EOS, VISC, MILNE, TWO_D, THETA1, 2>(h, A);
}
template <int EOS, bool VISC, bool MILNE>
static cudaError_t launch_tile_d(vh_handle* h, int stage, const StageArgs& A, cudaEvent_t mid, int part) {
  const bool th1 = h->prm.minmod_theta == 1.0;
  if (h->two_d) return th1 ? launch_tile_t<EOS, VISC, MILNE, true, true>(h, stage, A, mid, part) : launch_tile_t<EOS, VISC, MILNE, true, false>(h, stage, A, mid, part);
  return th1 ? launch_tile_t<EOS, VISC, MILNE, false, true>(h, stage, A, mid, part) : launch_tile_t<EOS, VISC, MILNE, false, false>(h, stage, A, mid, part);
}

#define VH_CAT2(a, b) a##b
#define VH_CAT(a, b) VH_CAT2(a, b)
cudaError_t VH_CAT(vh_launch_stage_combo, VH_COMBO)(vh_handle* h, int stage, const StageArgs& A, cudaEvent_t mid, int part) {
  constexpr int EOS = VH_COMBO % 3;
  constexpr int G = VH_COMBO / 3;      // 0: viscous Milne, 1: ideal Milne, 2: ideal Cartesian, 3: viscous Cartesian
  constexpr bool VISC = (G == 0) || (G == 3), MILNE = (G < 2);
  if (h->variant == 0) return launch_tile_d<EOS, VISC, MILNE>(h, stage, A, mid, part);
  if (h->variant == 2) return launch_split_d<EOS, VISC, MILNE>(h, stage, A, mid);
  return launch_stage_d<EOS, VISC, MILNE>(h, stage, A);
}
