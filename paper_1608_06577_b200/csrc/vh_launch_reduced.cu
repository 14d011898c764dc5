// vh_launch_reduced.cu -- launches of the reduced-storage stage kernel (vh_kernels5.cuh) for every EOS / geometry / dimensionality.
#include "vh_internal.cuh"
#include "vh_kernels5.cuh"

using namespace vh;

template <int EOS, bool MILNE, bool TWO_D>
static cudaError_t launch_t(vh_handle* h, int stage, const RedArgs& A) {
  const DevParams& P = h->P;
  dim3 block(32, 4);
  dim3 grid((P.nx + 31) / 32, (P.ny + 3) / 4, P.nz * P.n_batch);
  if (stage == 1) stage_reduced_kernel<EOS, MILNE, TWO_D, 1><<<grid, block, 0, h->stream>>>(P, A);
  else stage_reduced_kernel<EOS, MILNE, TWO_D, 2><<<grid, block, 0, h->stream>>>(P, A);
  h->launches++;
  return vh_debug_sync(h, stage == 1 ? "reduced-storage stage 1 kernel" : "reduced-storage stage 2 kernel");
}
template <int EOS>
static cudaError_t launch_e(vh_handle* h, int stage, const RedArgs& A) {
  const bool milne = (h->prm.geometry == 0);
  if (h->two_d) return milne ? launch_t<EOS, true, true>(h, stage, A) : launch_t<EOS, false, true>(h, stage, A);
  return milne ? launch_t<EOS, true, false>(h, stage, A) : launch_t<EOS, false, false>(h, stage, A);
}
cudaError_t vh_launch_stage_reduced(vh_handle* h, int stage, const RedArgs& A) {
  switch (h->prm.eos) {
    case 0: return launch_e<0>(h, stage, A);
    case 1: return launch_e<1>(h, stage, A);
    default: return launch_e<2>(h, stage, A);
  }
}
