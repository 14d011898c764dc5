// vh_internal.cuh -- shared between vh_api.cu and the per-physics launch units (vh_launch.cu, compiled once per combination
// of EOS / viscous / Milne so that the units build in parallel): the handle and the launch entry points.
#pragma once
#include "../../include/vh.h"
#include "vh_kernels4.cuh"

#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>

#ifndef VH_STAGE_MINB
#define VH_STAGE_MINB 2      // resident blocks per SM the stage kernel is compiled for (register cap 65536/(256*MINB))
#endif

struct vh_handle {
  vh_params prm;
  vh::DevParams P;
  cudaStream_t stream = nullptr;
  int device = 0;                    // the device the handle was created on (its buffers, tensor maps and kernel attributes belong to it)
  std::vector<const void*> smem_opted_in;   // kernels whose dynamic shared-memory limit was raised on `device` for this handle
  vh::real* pool = nullptr;          // 67 padded arrays (real = the library's precision: double in libvh.so, float in libvh_f32.so)
  vh::real* q[3] = {nullptr, nullptr, nullptr};   // q^n, q*, q^{n+1}   (:470 q, qS, Q)
  vh::real* u[3] = {nullptr, nullptr, nullptr};   // u^n, u^{n-1}, u*   (:470 u, up, uS)
  vh::real* e[2] = {nullptr, nullptr};            // e^n / e^{n+1}, e*
  vh::real* p[2] = {nullptr, nullptr};
  vh::real* vL = nullptr;              // [3] velocity of the reconstructed state at each cell's low face, per direction
  vh::real* vR = nullptr;              // [3] ... high face
  vh::Counters* cnt = nullptr;
  unsigned long long* diag = nullptr;   // [10] maxima of vh_get_diagnostics (bit patterns)
  vh::real* eos_tab = nullptr;         // EOS 2: the lattice table (vh_eos_lattice.hpp) in global memory
  vh::real* regfac = nullptr;          // one padded array: tanh(rho)/rho applied by the last step's final regularisation (vh_enable_regulation_map), else null
  double* stage_in = nullptr;  size_t stage_in_bytes = 0;     // device staging for host-side set_initial
  double* stage_out = nullptr; size_t stage_out_bytes = 0;    // device staging for host-side get_fields
  long long n_steps = 0;
  long long launches = 0;
  bool initialised = false;
  bool two_d = false;
  vh::real* cur[4] = {nullptr, nullptr, nullptr, nullptr};   // q, e, p, u of the most recently written state (what vh_halo_export(what = 1) reads)
  int next_part = 0;                 // vh_step_part: the part of the RK2 step that comes next (0..3)
  bool slab_nb[2] = {false, false};  // a neighbouring eta-slab exists beyond the low / high face: set by vh_halo_import, cleared by vh_set_initial / vh_set_state
  bool reduced = false;              // vh_params.storage == 1: 10 q + 3 u arrays per time level (vh_kernels5.cuh), own stage kernel
  bool uprev_initial = true;         // u^{n-1} is the copy of u^0 made by vh_set_initial (reduced storage: its u^tau is normalised at tau0, not tau0 - dtau)
  int variant = 0;                   // 0: velocity kernel + TMA tile kernel; 1: one-thread-per-cell kernel + ghost kernel; 2: velocity + L1 stage kernel
  CUtensorMap mapVA, mapVZ;          // velocity tile kernel: tile + 1-cell y halo, one eta-halo plane
  CUtensorMap mapA, mapZ, mapC;      // TMA tensor maps over the whole pool (box A: tile + xy halo, box Z: two eta-halo planes, box C: the tile)
  std::string err;
};


// Launch check of every kernel.  A debugging build (nvcc -DVH_DEBUG_SYNC) also synchronises after each launch and names the kernel that
// faulted; the product build reads nothing from the environment.
inline cudaError_t vh_debug_sync(vh_handle* h, const char* what) {
  cudaError_t e = cudaGetLastError();
#ifdef VH_DEBUG_SYNC
  if (e == cudaSuccess) {
    e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) fprintf(stderr, "[vh] %s faulted at step %lld: %s\n", what, h->n_steps, cudaGetErrorString(e));
  }
#else
  (void)h; (void)what;
#endif
  return e;
}

// Raise a kernel's dynamic shared-memory limit once per handle.  The attribute is per device, and a handle belongs to one device, so
// nothing process-wide is cached.
inline cudaError_t vh_opt_in_smem(vh_handle* h, const void* kern, size_t smem) {
  for (const void* k : h->smem_opted_in) if (k == kern) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) h->smem_opted_in.push_back(kern);
  return e;
}

// One Euler stage (kernels of the handle's variant) for one combination of template parameters; defined in vh_launch.cu.
// part: 0 = both kernels of the stage, 1 = velocity kernel only, 2 = stage kernel only (default pipeline; vh_step_part).
// combo = eos + 3 * (0: viscous Milne, 1: ideal Milne, 2: ideal Cartesian, 3: viscous Cartesian), eos = 0, 1, 2.  mid (optional) is recorded between the two launches.
#define VH_DECLARE_COMBO(K) cudaError_t vh_launch_stage_combo##K(vh_handle* h, int stage, const vh::StageArgs& A, cudaEvent_t mid, int part);
VH_DECLARE_COMBO(0) VH_DECLARE_COMBO(1) VH_DECLARE_COMBO(2) VH_DECLARE_COMBO(3) VH_DECLARE_COMBO(4) VH_DECLARE_COMBO(5)
VH_DECLARE_COMBO(6) VH_DECLARE_COMBO(7) VH_DECLARE_COMBO(8) VH_DECLARE_COMBO(9) VH_DECLARE_COMBO(10) VH_DECLARE_COMBO(11)
#undef VH_DECLARE_COMBO
// reduced-storage stage (vh_launch_reduced.cu): one launch of stage_reduced_kernel; A is a vh::RedArgs
namespace vh { struct RedArgs; }
cudaError_t vh_launch_stage_reduced(vh_handle* h, int stage, const vh::RedArgs& A);
