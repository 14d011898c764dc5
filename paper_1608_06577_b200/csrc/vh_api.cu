// vh_api.cu -- C ABI (include/vh.h): handle, buffers, buffer rotation (PAPER.md program-flow steps 7, 9), kernel dispatch.
#include "vh_internal.cuh"
#include "vh_eos_lattice.hpp"
#include "vh_peaks.cuh"
#include "vh_kernels5.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <new>
#include <string>
#include <vector>

using namespace vh;

static thread_local std::string g_err;

static int fail(vh_handle* h, int code, const std::string& msg) {
  if (h) h->err = msg;
  g_err = msg;
  return code;
}
#define CUDA_TRY(h, call)                                                                              \
  do {                                                                                                 \
    cudaError_t _e = (call);                                                                           \
    if (_e != cudaSuccess) return fail(h, VH_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(_e)); \
  } while (0)

// every entry point that touches the device runs on the handle's device, whatever the caller's current device is - and hands the caller's
// device back when it returns (on every path: the guard lives on the entry point's stack frame), so that a host framework's notion of the
// current device (later allocations, its current stream) is not changed behind its back by a call on a handle of another GPU
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
static int enter(vh_handle* h, DeviceGuard& g) {
  int dev = -1;
  const bool known = (cudaGetDevice(&dev) == cudaSuccess);
  if (!known || dev != h->device) {
    cudaError_t e = cudaSetDevice(h->device);
    if (e != cudaSuccess) return fail(h, VH_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(e));
    if (known) { g.prev = dev; g.switched = true; }
  }
  return VH_OK;
}
#define VH_ENTER(h)                                   \
  DeviceGuard _vh_device_guard;                       \
  do {                                                \
    if (int _rc = enter(h, _vh_device_guard)) return _rc; \
  } while (0)

static long long round_up(long long a, long long m) { return (a + m - 1) / m * m; }

static int fill_dev_params(const vh_params& p, DevParams& P) {
  std::memset(&P, 0, sizeof(P));
  P.nx = p.nx; P.ny = p.ny; P.nz = p.nz; P.n_batch = p.n_batch;
  const bool two_d = (p.nz == 1);
  P.NXp = (int)round_up(p.nx + XOFF + 2, 16);      // XOFF cells before the first physical cell, two ghost cells after the last
  P.NYp = p.ny + 4;
  P.NZp = two_d ? 1 : p.nz + 4;
  P.zoff = two_d ? 0 : 2;
  P.plane = (long long)P.NXp * P.NYp;
  P.bstride = P.plane * P.NZp;
  P.fstride = P.bstride * p.n_batch;
  P.dx = p.dx; P.dy = p.dy; P.dz = p.dz; P.dtau = p.dtau;
  P.inv_dx = 1.0 / p.dx; P.inv_dy = 1.0 / p.dy; P.inv_dz = 1.0 / p.dz; P.inv_dtau = 1.0 / p.dtau;
  P.shear = (p.physics & 1) ? 1 : 0;
  P.bulk = (p.physics & 2) ? 1 : 0;
  P.eos_a_inv = 1.0 / p.eos_a; P.eos_alpha = p.eos_alpha; P.eos_e0_inv = (p.eos == 1) ? 1.0 / p.eos_e0 : 0.0;
  P.inv_ctaupi_etas = 1.0 / (p.c_tau_pi * p.eta_over_s);
  P.inv_ctaupi = 1.0 / p.c_tau_pi;
  P.zeta_model = p.zeta_model; P.zeta_amp = p.zeta_amp; P.zeta_T0 = p.zeta_T0;
  P.zeta_inv_width = (p.zeta_model == 1) ? 1.0 / p.zeta_width : ((p.zeta_model == 3) ? 1.0 / p.zeta_T0 : 0.0);      // model 3: 1/T_c
  P.inv_ctauPi = 1.0 / p.c_tau_Pi;
  P.delta_pipi = p.delta_pipi; P.tau_pipi = p.tau_pipi; P.lambda_piPi = p.lambda_piPi;
  P.delta_PiPi = p.delta_PiPi; P.lambda_Pipi_coef = p.lambda_Pipi_coef;
  P.theta = p.minmod_theta;
  P.inv_rho_max = 1.0 / p.rho_max; P.xi0_rho_max = p.xi0 * p.rho_max;
  P.newton_max_iter = p.newton_max_iter; P.newton_rtol = p.newton_rtol;
  P.newton_stop = std::max(p.newton_rtol, 0.1 * std::sqrt(p.newton_rtol));      // see newton_pair (vh_math.cuh)
  P.relax_clamp = (p.tau_relax_floor_over_dtau > 0.0) ? 1.0 / (p.tau_relax_floor_over_dtau * p.dtau) : std::numeric_limits<double>::infinity();
  return 0;
}

static int check_params(const vh_params* p, std::string& why) {
  if (!p) { why = "params is NULL"; return -1; }
  if (p->nx < 1 || p->ny < 1 || p->nz < 1 || p->n_batch < 1) { why = "grid extents and n_batch must be >= 1"; return -1; }
  if (!(p->dx > 0 && p->dy > 0 && p->dz > 0 && p->dtau > 0)) { why = "spacings and dtau must be > 0"; return -1; }
  if (p->geometry != 0 && p->geometry != 1) { why = "geometry must be 0 (Milne) or 1 (Cartesian)"; return -1; }
  if (p->geometry == 0 && !(p->tau0 > 0)) { why = "Milne geometry needs tau0 > 0"; return -1; }
  if (p->physics < 0 || p->physics > 3) { why = "physics must be a combination of bit0 (shear) and bit1 (bulk)"; return -1; }
  if (p->eos < 0 || p->eos > 2) { why = "eos must be 0, 1 or 2"; return -1; }
  if (p->eos != 2 && !(p->eos_a > 0)) { why = "eos_a must be > 0"; return -1; }
  if (p->eos == 1 && !(p->eos_e0 > 0)) { why = "eos_e0 must be > 0"; return -1; }
  if (p->physics != 0 && !(p->eta_over_s > 0 && p->c_tau_pi > 0 && p->c_tau_Pi > 0)) { why = "eta_over_s, c_tau_pi, c_tau_Pi must be > 0"; return -1; }
  if (p->zeta_model < 0 || p->zeta_model > 3) { why = "zeta_model must be 0, 1, 2 or 3"; return -1; }
  if (p->zeta_model == 3 && !(p->zeta_T0 > 0 && p->zeta_amp >= 0)) { why = "zeta_model 3 (Eq. 17) needs zeta_T0 = T_c > 0 and zeta_amp = (zeta/s)_norm >= 0"; return -1; }
  if (p->zeta_model == 1 && !(p->zeta_width > 0)) { why = "zeta_width must be > 0"; return -1; }
  if (!(p->minmod_theta >= 1.0 && p->minmod_theta <= 2.0)) { why = "minmod_theta must lie in [1,2] (Eq. 67)"; return -1; }
  if (!(p->rho_max > 0 && p->xi0 > 0)) { why = "xi0, rho_max must be > 0"; return -1; }
  if (p->newton_max_iter < 1 || !(p->newton_rtol > 0)) { why = "newton_max_iter >= 1 and newton_rtol > 0 required"; return -1; }
  if (p->storage != 0 && p->storage != 1) { why = "storage must be 0 (all components) or 1 (reduced, PAPER.md:476)"; return -1; }
  if (p->storage == 1 && !(p->physics & 1)) { why = "storage = 1 needs shear on: without pi^{mu nu} there is nothing to reduce"; return -1; }
  if (kF32 && p->newton_rtol < 1e-6) { why = "the single-precision library needs newton_rtol >= 1e-6 (a tighter stopping rule cannot be met in FP32)"; return -1; }
  if ((long long)p->nz * p->n_batch > 65535) { why = "nz*n_batch exceeds the grid z limit (65535)"; return -1; }
  return 0;
}

// ------------------------------------------------------------------------------------------------ dispatch
#define debug_sync vh_debug_sync
// one Euler stage with the handle's kernel variant: the launch units are compiled per (EOS, viscous, Milne) combination
static cudaError_t launch_stage_any(vh_handle* h, int stage, const StageArgs& A, cudaEvent_t mid, int part = 0) {
  const int phys = (h->prm.physics != 0) ? ((h->prm.geometry == 0) ? 0 : 3) : ((h->prm.geometry == 0) ? 1 : 2);
  switch (h->prm.eos + 3 * phys) {
    case 0: return vh_launch_stage_combo0(h, stage, A, mid, part);
    case 1: return vh_launch_stage_combo1(h, stage, A, mid, part);
    case 2: return vh_launch_stage_combo2(h, stage, A, mid, part);
    case 3: return vh_launch_stage_combo3(h, stage, A, mid, part);
    case 4: return vh_launch_stage_combo4(h, stage, A, mid, part);
    case 5: return vh_launch_stage_combo5(h, stage, A, mid, part);
    case 6: return vh_launch_stage_combo6(h, stage, A, mid, part);
    case 7: return vh_launch_stage_combo7(h, stage, A, mid, part);
    case 8: return vh_launch_stage_combo8(h, stage, A, mid, part);
    case 9: return vh_launch_stage_combo9(h, stage, A, mid, part);
    case 10: return vh_launch_stage_combo10(h, stage, A, mid, part);
    default: return vh_launch_stage_combo11(h, stage, A, mid, part);
  }
}

// One 5-d tensor map (x, y, eta, event, array) over the whole pool of padded arrays per box shape.  cuTensorMapEncodeTiled is a
// driver-API entry point; it is looked up through the runtime so that the library needs no link-time dependency on libcuda.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static int make_tensor_maps(vh_handle* h, int n_arrays) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qr;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess || !fn)
    return fail(h, VH_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
  EncodeTiledFn encode = (EncodeTiledFn)fn;
  const DevParams& P = h->P;
  const cuuint64_t dims[5] = {(cuuint64_t)P.NXp, (cuuint64_t)P.NYp, (cuuint64_t)P.NZp, (cuuint64_t)P.n_batch, (cuuint64_t)n_arrays};
  const cuuint64_t R = sizeof(real);
  const cuuint64_t strides[4] = {(cuuint64_t)P.NXp * R, (cuuint64_t)P.plane * R, (cuuint64_t)P.bstride * R, (cuuint64_t)P.fstride * R};
  const CUtensorMapDataType dtype = kF32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
  // L2 promotion no wider than a box row (32 or 36 elements: 256 / 288 bytes in double, 128 / 144 bytes in single precision)
  const CUtensorMapL2promotion promo = kF32 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_L2_256B;
  const cuuint32_t ones[5] = {1, 1, 1, 1, 1};
  const bool td = h->two_d;
  const cuuint32_t boxA[5] = {(cuuint32_t)(td ? Tile<true>::AX : Tile<false>::AX), (cuuint32_t)(td ? Tile<true>::AY : Tile<false>::AY),
                              (cuuint32_t)(td ? Tile<true>::TZ : Tile<false>::TZ), 1, 1};
  const cuuint32_t boxZ[5] = {(cuuint32_t)Tile<false>::TX, (cuuint32_t)Tile<false>::TY, 2, 1, 1};
  CUresult r = encode(&h->mapA, dtype, 5, h->pool, dims, strides, boxA, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                      CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(h, VH_ERR_CUDA, "cuTensorMapEncodeTiled(box A) failed with CUresult " + std::to_string((int)r));
  r = encode(&h->mapZ, dtype, 5, h->pool, dims, strides, boxZ, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(h, VH_ERR_CUDA, "cuTensorMapEncodeTiled(box Z) failed with CUresult " + std::to_string((int)r));
  const cuuint32_t boxC[5] = {(cuuint32_t)Tile<false>::TX, (cuuint32_t)(td ? Tile<true>::TY : Tile<false>::TY),
                              (cuuint32_t)(td ? Tile<true>::TZ : Tile<false>::TZ), 1, 1};
  r = encode(&h->mapC, dtype, 5, h->pool, dims, strides, boxC, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(h, VH_ERR_CUDA, "cuTensorMapEncodeTiled(box C) failed with CUresult " + std::to_string((int)r));
  const cuuint32_t boxVA[5] = {(cuuint32_t)(td ? VTile<true>::AX : VTile<false>::AX), (cuuint32_t)(td ? VTile<true>::AY : VTile<false>::AY),
                               (cuuint32_t)(td ? VTile<true>::VZ : VTile<false>::VZ), 1, 1};
  r = encode(&h->mapVA, dtype, 5, h->pool, dims, strides, boxVA, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(h, VH_ERR_CUDA, "cuTensorMapEncodeTiled(box VA) failed with CUresult " + std::to_string((int)r));
  const cuuint32_t boxVZ[5] = {(cuuint32_t)VTile<false>::VX, (cuuint32_t)VTile<false>::VY, 1, 1, 1};
  r = encode(&h->mapVZ, dtype, 5, h->pool, dims, strides, boxVZ, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(h, VH_ERR_CUDA, "cuTensorMapEncodeTiled(box VZ) failed with CUresult " + std::to_string((int)r));
  return VH_OK;
}

static cudaError_t launch_ghost(vh_handle* h, real* q, real* e, real* p, real* u) {
  const int nq = h->reduced ? NQR : NQ, nu = h->reduced ? 3 : 4;
  const DevParams& P = h->P;
  long long W = h->two_d ? (long long)P.ny + P.nx : (long long)P.ny * P.nz + (long long)P.nx * P.nz + (long long)P.nx * P.ny;
  dim3 grid((unsigned)((W + 255) / 256), nq + 2 + nu, P.n_batch);
  GhostArgs G{q, e, p, u, nq};
  if (h->two_d) ghost_kernel<true><<<grid, 256, 0, h->stream>>>(P, G);
  else ghost_kernel<false><<<grid, 256, 0, h->stream>>>(P, G);
  h->launches++;
  return debug_sync(h, "ghost kernel");
}

static cudaError_t reset_regulation_map(vh_handle* h) {
  if (!h->regfac) return cudaSuccess;
  fill_kernel<<<1024, 256, 0, h->stream>>>(h->regfac, h->P.fstride, real(1.0));
  h->launches++;
  return cudaGetLastError();
}

template <int EOS>
static void launch_diag(vh_handle* h, real t, double* maps) {
  const DevParams& P = h->P;
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const unsigned nb = (unsigned)std::min<long long>((np + 255) / 256, 2048LL);      // grid-stride loop
  if (h->prm.geometry == 0) diagnostics_kernel<EOS, true><<<nb, 256, 0, h->stream>>>(P, h->q[0], h->e[0], h->p[0], h->u[0], h->u[1], t, h->diag, maps);
  else diagnostics_kernel<EOS, false><<<nb, 256, 0, h->stream>>>(P, h->q[0], h->e[0], h->p[0], h->u[0], h->u[1], t, h->diag, maps);
  h->launches++;
}

static int reset_counters(vh_handle* h) {
  Counters c;
  c.n_fail = 0; c.n_nonfinite = 0;
  double one = 1.0;
  std::memcpy(&c.min_reg_bits, &one, sizeof(double));
  CUDA_TRY(h, cudaMemcpyAsync(h->cnt, &c, sizeof(c), cudaMemcpyHostToDevice, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));    // c lives on this stack frame
  return VH_OK;
}

// ------------------------------------------------------------------------------------------------ C ABI
extern "C" {

int vh_create(const vh_params* p, void* cuda_stream, vh_handle** out) {
  std::string why;
  if (!out) return fail(nullptr, VH_ERR_ARG, "out is NULL");
  if (check_params(p, why)) return fail(nullptr, VH_ERR_ARG, why);
  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev < 1) return fail(nullptr, VH_ERR_CUDA, std::string("no CUDA device: ") + cudaGetErrorString(ce));
  vh_handle* h = new (std::nothrow) vh_handle;
  if (!h) return fail(nullptr, VH_ERR_ALLOC, "host allocation failed");
  h->prm = *p;
  fill_dev_params(*p, h->P);
  h->two_d = (p->nz == 1);
  h->stream = (cudaStream_t)cuda_stream;
  cudaGetDevice(&h->device);
  const long long fs = h->P.fstride;
  h->reduced = (p->storage == 1);
  const int nq = h->reduced ? NQR : NQ, nu = h->reduced ? 3 : 4;
  const int n_arrays = 3 * nq + 3 * nu + 4 + (h->reduced ? 0 : 6);      // 67, or 43 in reduced storage (no state velocities: its kernel inverts in place)
  const size_t bytes = (size_t)n_arrays * fs * sizeof(real);
  ce = cudaMalloc((void**)&h->pool, bytes);
  if (ce != cudaSuccess) { cudaGetLastError(); delete h; return fail(nullptr, VH_ERR_ALLOC, std::string("cudaMalloc of ") + std::to_string(bytes) + " bytes: " + cudaGetErrorString(ce)); }
  ce = cudaMalloc((void**)&h->cnt, sizeof(Counters));
  if (ce != cudaSuccess) { cudaGetLastError(); cudaFree(h->pool); delete h; return fail(nullptr, VH_ERR_ALLOC, "cudaMalloc(counters) failed"); }
  real* w = h->pool;
  for (int i = 0; i < 3; ++i) { h->q[i] = w; w += nq * fs; }
  for (int i = 0; i < 3; ++i) { h->u[i] = w; w += nu * fs; }
  for (int i = 0; i < 2; ++i) { h->e[i] = w; w += fs; }
  for (int i = 0; i < 2; ++i) { h->p[i] = w; w += fs; }
  if (!h->reduced) { h->vL = w; w += 3 * fs; h->vR = w; w += 3 * fs; }
  ce = cudaMemsetAsync(h->pool, 0, bytes, h->stream);
  if (ce != cudaSuccess) { cudaFree(h->pool); cudaFree(h->cnt); delete h; return fail(nullptr, VH_ERR_CUDA, "cudaMemsetAsync failed"); }
  if (make_tensor_maps(h, n_arrays) != VH_OK) {
    std::string msg = h->err;
    cudaFree(h->pool); cudaFree(h->cnt); delete h;
    return fail(nullptr, VH_ERR_CUDA, msg);
  }
  if (p->eos == 2) {      // lattice EOS: build the table on the host (milliseconds), keep it in global memory
    const vh_eos::LatticeTable tab = vh_eos::Builder().build();
    const std::vector<real> nodes(tab.node.begin(), tab.node.end());      // the table in the library's precision
    const size_t tb = nodes.size() * sizeof(real);
    ce = cudaMalloc((void**)&h->eos_tab, tb);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(h->eos_tab, nodes.data(), tb, cudaMemcpyHostToDevice, h->stream);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(h->stream);      // tab lives on this stack frame
    if (ce != cudaSuccess) { cudaGetLastError(); cudaFree(h->eos_tab); cudaFree(h->pool); cudaFree(h->cnt); delete h; return fail(nullptr, VH_ERR_ALLOC, "EOS table upload failed"); }
    const int n = vh_eos::VH_EOS_N;
    const double* nd = tab.node.data();
    const double e0 = std::pow(tab.x0, 4), eN = std::pow(tab.xN, 4);
    h->P.eos_tab = reinterpret_cast<const real2*>(h->eos_tab);
    h->P.eos_n = n; h->P.eos_x0 = tab.x0; h->P.eos_xN = tab.xN; h->P.eos_inv_h = 1.0 / tab.h;
    h->P.eos_lo_slope = nd[0] / e0; h->P.eos_pN = nd[4 * n]; h->P.eos_eN = eN;
    h->P.eos_T0_over_x0 = nd[2] / tab.x0; h->P.eos_TN_over_xN = nd[4 * n + 2] / tab.xN;
  }
  if (reset_counters(h) != VH_OK) {      // vh_get_status before vh_set_initial reads zeros, not uninitialised memory
    std::string msg = h->err;
    cudaFree(h->eos_tab); cudaFree(h->pool); cudaFree(h->cnt); delete h;
    return fail(nullptr, VH_ERR_CUDA, msg);
  }
  *out = h;
  return VH_OK;
}

void vh_destroy(vh_handle* h) {
  if (!h) return;
  DeviceGuard guard;
  enter(h, guard);
  cudaStreamSynchronize(h->stream);
  cudaFree(h->pool);
  cudaFree(h->cnt);
  cudaFree(h->eos_tab);
  cudaFree(h->diag);
  cudaFree(h->regfac);
  cudaFree(h->stage_in);
  cudaFree(h->stage_out);
  delete h;
}

const char* vh_last_error(vh_handle* h) { return h ? h->err.c_str() : g_err.c_str(); }
long long vh_launch_count(vh_handle* h) { return h ? h->launches : 0; }

int vh_set_kernel_variant(vh_handle* h, int variant) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  if (variant < 0 || variant > 2) return fail(h, VH_ERR_ARG, "unknown kernel variant");
  if (h->reduced && variant != 0) return fail(h, VH_ERR_ARG, "reduced-storage mode has one kernel (variant 0)");
  if (h->next_part != 0) return fail(h, VH_ERR_STATE, "vh_set_kernel_variant in the middle of a step taken with vh_step_part");
  h->variant = variant;
  return VH_OK;
}

static int ensure_stage(vh_handle* h, double** buf, size_t* have, size_t need) {
  if (*have >= need) return VH_OK;
  cudaFree(*buf);
  *buf = nullptr; *have = 0;
  if (cudaMalloc((void**)buf, need) != cudaSuccess) { cudaGetLastError(); *buf = nullptr; return fail(h, VH_ERR_ALLOC, "cudaMalloc(staging) failed"); }
  *have = need;
  return VH_OK;
}

int vh_set_initial(vh_handle* h, const double* e, const double* u4, const double* pi10, const double* Pi, int mem_space) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (!e || !u4) return fail(h, VH_ERR_ARG, "e and u4 are required");
  if (mem_space != 0 && mem_space != 1) return fail(h, VH_ERR_ARG, "mem_space must be 0 (host) or 1 (device)");
  const DevParams& P = h->P;
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const double *de = e, *du = u4, *dpi = pi10, *dPi = Pi;
  if (mem_space == 0) {
    int rc = ensure_stage(h, &h->stage_in, &h->stage_in_bytes, (size_t)16 * np * sizeof(double));
    if (rc) return rc;
    double* s = h->stage_in;
    CUDA_TRY(h, cudaMemcpyAsync(s, e, np * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    CUDA_TRY(h, cudaMemcpyAsync(s + np, u4, 4 * np * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    if (pi10) CUDA_TRY(h, cudaMemcpyAsync(s + 5 * np, pi10, 10 * np * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    if (Pi) CUDA_TRY(h, cudaMemcpyAsync(s + 15 * np, Pi, np * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    de = s; du = s + np; dpi = pi10 ? s + 5 * np : nullptr; dPi = Pi ? s + 15 * np : nullptr;
  }
  unsigned nb = (unsigned)((np + 255) / 256);
  if (h->reduced) {
    const real t0 = (real)h->prm.tau0;
    const bool mil = (h->prm.geometry == 0);
#define VH_INIT_RED(E)                                                                                                                        \
  do {                                                                                                                                        \
    if (mil) init_reduced_kernel<E, true><<<nb, 256, 0, h->stream>>>(P, de, du, dpi, dPi, t0, h->q[0], h->e[0], h->p[0], h->u[0], h->u[1]);   \
    else init_reduced_kernel<E, false><<<nb, 256, 0, h->stream>>>(P, de, du, dpi, dPi, t0, h->q[0], h->e[0], h->p[0], h->u[0], h->u[1]);      \
  } while (0)
    if (h->prm.eos == 2) VH_INIT_RED(2); else if (h->prm.eos == 1) VH_INIT_RED(1); else VH_INIT_RED(0);
#undef VH_INIT_RED
  } else if (h->prm.eos == 2) init_kernel<2><<<nb, 256, 0, h->stream>>>(P, de, du, dpi, dPi, h->q[0], h->e[0], h->p[0], h->u[0], h->u[1]);
  else if (h->prm.eos == 1) init_kernel<1><<<nb, 256, 0, h->stream>>>(P, de, du, dpi, dPi, h->q[0], h->e[0], h->p[0], h->u[0], h->u[1]);
  else init_kernel<0><<<nb, 256, 0, h->stream>>>(P, de, du, dpi, dPi, h->q[0], h->e[0], h->p[0], h->u[0], h->u[1]);
  h->launches++;
  CUDA_TRY(h, cudaGetLastError());
  CUDA_TRY(h, launch_ghost(h, h->q[0], h->e[0], h->p[0], h->u[0]));
  h->n_steps = 0;
  h->next_part = 0;
  h->slab_nb[0] = h->slab_nb[1] = false;
  h->cur[0] = h->q[0]; h->cur[1] = h->e[0]; h->cur[2] = h->p[0]; h->cur[3] = h->u[0];
  h->uprev_initial = true;
  int rc = reset_counters(h);
  if (rc) return rc;
  CUDA_TRY(h, reset_regulation_map(h));
  h->initialised = true;
  return VH_OK;
}

int vh_set_state(vh_handle* h, const double* q15, const double* e, const double* u4, const double* u4_prev, long long n_steps_done,
                 int mem_space) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (!q15 || !e || !u4 || !u4_prev || n_steps_done < 0) return fail(h, VH_ERR_ARG, "q15, e, u4, u4_prev are required; n_steps_done >= 0");
  if (mem_space != 0 && mem_space != 1) return fail(h, VH_ERR_ARG, "mem_space must be 0 (host) or 1 (device)");
  const DevParams& P = h->P;
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const unsigned nb = (unsigned)((np + 255) / 256);
  struct Item { const double* src; real* dst; int nc; };
  Item items[4] = {{q15, h->q[0], 15}, {e, h->e[0], 1}, {u4, h->u[0], 4}, {u4_prev, h->u[1], 4}};
  if (mem_space == 0) {
    int rc = ensure_stage(h, &h->stage_in, &h->stage_in_bytes, (size_t)16 * np * sizeof(double));
    if (rc) return rc;
  }
  for (int n = 0; n < 4; ++n) {
    const Item& it = items[n];
    const double* src = it.src;
    if (mem_space == 0) {
      CUDA_TRY(h, cudaMemcpyAsync(h->stage_in, it.src, (size_t)it.nc * np * sizeof(double), cudaMemcpyHostToDevice, h->stream));
      src = h->stage_in;
    }
    if (h->reduced && n != 1) {      // q15 / u4 / u4_prev: only the stored subset is kept (the dependent components are not state)
      import_reduced_kernel<<<nb, 256, 0, h->stream>>>(P, n == 0 ? src : nullptr, n == 0 ? nullptr : src, n == 0 ? it.dst : nullptr, n == 0 ? nullptr : it.dst);
    } else {
      pack_kernel<false><<<nb, 256, 0, h->stream>>>(P, it.dst, const_cast<double*>(src), it.nc);
    }
    h->launches++;
    CUDA_TRY(h, cudaGetLastError());
  }
  h->uprev_initial = false;      // u4_prev belongs to tau - dtau
  if (h->prm.eos == 2) pressure_kernel<2><<<nb, 256, 0, h->stream>>>(P, h->e[0], h->p[0]);
  else if (h->prm.eos == 1) pressure_kernel<1><<<nb, 256, 0, h->stream>>>(P, h->e[0], h->p[0]);
  else pressure_kernel<0><<<nb, 256, 0, h->stream>>>(P, h->e[0], h->p[0]);
  h->launches++;
  CUDA_TRY(h, cudaGetLastError());
  CUDA_TRY(h, launch_ghost(h, h->q[0], h->e[0], h->p[0], h->u[0]));
  h->n_steps = n_steps_done;
  h->next_part = 0;
  h->slab_nb[0] = h->slab_nb[1] = false;
  h->cur[0] = h->q[0]; h->cur[1] = h->e[0]; h->cur[2] = h->p[0]; h->cur[3] = h->u[0];
  int rc = reset_counters(h);
  if (rc) return rc;
  CUDA_TRY(h, reset_regulation_map(h));
  h->initialised = true;
  return VH_OK;
}

int vh_set_uprev(vh_handle* h, const double* u4_prev, int mem_space) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (!h->initialised) return fail(h, VH_ERR_STATE, "vh_set_uprev before vh_set_initial");
  if (!u4_prev || (mem_space != 0 && mem_space != 1)) return fail(h, VH_ERR_ARG, "bad argument");
  const DevParams& P = h->P;
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const double* src = u4_prev;
  if (mem_space == 0) {
    int rc = ensure_stage(h, &h->stage_in, &h->stage_in_bytes, (size_t)16 * np * sizeof(double));
    if (rc) return rc;
    CUDA_TRY(h, cudaMemcpyAsync(h->stage_in, u4_prev, 4 * np * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    src = h->stage_in;
  }
  if (h->reduced) import_reduced_kernel<<<(unsigned)((np + 255) / 256), 256, 0, h->stream>>>(P, nullptr, src, nullptr, h->u[1]);
  else pack_kernel<false><<<(unsigned)((np + 255) / 256), 256, 0, h->stream>>>(P, h->u[1], const_cast<double*>(src), 4);
  h->uprev_initial = false;
  h->launches++;
  CUDA_TRY(h, cudaGetLastError());
  if (mem_space == 0) CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  return VH_OK;
}

// reduced storage: (stage kernel, ghost kernel) per stage; same buffer rotation
static int one_step_reduced(vh_handle* h, cudaEvent_t* ev) {
  const double t = h->prm.tau0 + (double)h->n_steps * h->prm.dtau;
  const double t1 = t + h->prm.dtau;
  RedArgs A;
  A.q_in = h->q[0]; A.e_in = h->e[0]; A.p_in = h->p[0]; A.u_in = h->u[0]; A.u_prev = h->u[1]; A.q_n = nullptr;
  A.q_out = h->q[1]; A.e_out = h->e[1]; A.p_out = h->p[1]; A.u_out = h->u[2]; A.cnt = h->cnt;
  A.t = (real)t; A.t_post = (real)t1; A.t_prev = (real)(h->uprev_initial ? t : t - h->prm.dtau);
  if (ev) CUDA_TRY(h, cudaEventRecord(ev[0], h->stream));
  CUDA_TRY(h, vh_launch_stage_reduced(h, 1, A));
  if (ev) CUDA_TRY(h, cudaEventRecord(ev[1], h->stream));
  CUDA_TRY(h, launch_ghost(h, h->q[1], h->e[1], h->p[1], h->u[2]));
  if (ev) CUDA_TRY(h, cudaEventRecord(ev[2], h->stream));
  A.q_in = h->q[1]; A.e_in = h->e[1]; A.p_in = h->p[1]; A.u_in = h->u[2]; A.u_prev = h->u[0]; A.q_n = h->q[0];
  A.q_out = h->q[2]; A.e_out = h->e[0]; A.p_out = h->p[0]; A.u_out = h->u[1];
  A.t = (real)t1; A.t_post = (real)t1; A.t_prev = (real)t;
  CUDA_TRY(h, vh_launch_stage_reduced(h, 2, A));
  if (ev) CUDA_TRY(h, cudaEventRecord(ev[3], h->stream));
  CUDA_TRY(h, launch_ghost(h, h->q[2], h->e[0], h->p[0], h->u[1]));
  if (ev) CUDA_TRY(h, cudaEventRecord(ev[4], h->stream));
  real* un = h->u[1]; h->u[1] = h->u[0]; h->u[0] = un;
  real* qn = h->q[2]; h->q[2] = h->q[0]; h->q[0] = qn;
  h->n_steps++;
  h->uprev_initial = false;
  return VH_OK;
}

static int one_step(vh_handle* h, cudaEvent_t* ev) {
  if (h->reduced) return one_step_reduced(h, ev);
  const double t = h->prm.tau0 + (double)h->n_steps * h->prm.dtau;     // :493
  const double t1 = t + h->prm.dtau;
  StageArgs A;
  // steps 1-4: q* = E[q^n; e,p,u^n,u^{n-1}] at tau^n, then (e*,p*,u*) at tau^n + dtau, regulate, ghosts
  A.q_in = h->q[0]; A.e_in = h->e[0]; A.p_in = h->p[0]; A.u_in = h->u[0]; A.u_prev = h->u[1]; A.q_n = nullptr;
  A.q_out = h->q[1]; A.e_out = h->e[1]; A.p_out = h->p[1]; A.u_out = h->u[2]; A.cnt = h->cnt; A.t = t; A.t_post = t1;
  A.regfac = nullptr;      // the map is that of the step's last regularisation (stage 2)
  // variants 0, 2: (velocity kernel, stage kernel) per stage, ghost replicas written by the stage kernel;
  // variant 1: (cell kernel, ghost kernel) per stage.  ev[0..4] bracket the four launches of the step.
  const bool split = (h->variant != 1);
  if (ev) CUDA_TRY(h, cudaEventRecord(ev[0], h->stream));
  if (split) {
    CUDA_TRY(h, launch_stage_any(h, 1, A, ev ? ev[1] : nullptr));
  } else {
    CUDA_TRY(h, launch_stage_any(h, 1, A, nullptr));
    if (ev) CUDA_TRY(h, cudaEventRecord(ev[1], h->stream));
    CUDA_TRY(h, launch_ghost(h, h->q[1], h->e[1], h->p[1], h->u[2]));
  }
  if (ev) CUDA_TRY(h, cudaEventRecord(ev[2], h->stream));
  // steps 5-8: q** = E[q*; e*,p*,u*,u^n] at tau^n + dtau; q^{n+1} = (q^n + q**)/2; invert, regulate, ghosts.
  // u^{n+1} overwrites the buffer of u^{n-1}, e^{n+1}/p^{n+1} the buffers of e^n/p^n (neither is read by stage 2).
  A.q_in = h->q[1]; A.e_in = h->e[1]; A.p_in = h->p[1]; A.u_in = h->u[2]; A.u_prev = h->u[0]; A.q_n = h->q[0];
  A.q_out = h->q[2]; A.e_out = h->e[0]; A.p_out = h->p[0]; A.u_out = h->u[1]; A.t = t1; A.t_post = t1;
  A.regfac = h->regfac;
  if (split) {
    CUDA_TRY(h, launch_stage_any(h, 2, A, ev ? ev[3] : nullptr));
  } else {
    CUDA_TRY(h, launch_stage_any(h, 2, A, nullptr));
    if (ev) CUDA_TRY(h, cudaEventRecord(ev[3], h->stream));
    CUDA_TRY(h, launch_ghost(h, h->q[2], h->e[0], h->p[0], h->u[1]));
  }
  if (ev) CUDA_TRY(h, cudaEventRecord(ev[4], h->stream));
  // steps 7, 9: rotate.  u: (u^n, u^{n-1}, u*) <- (u^{n+1}, u^n, scratch); q: q^n <-> q^{n+1}
  real* un = h->u[1]; h->u[1] = h->u[0]; h->u[0] = un;
  real* qn = h->q[2]; h->q[2] = h->q[0]; h->q[0] = qn;
  h->n_steps++;
  h->cur[0] = h->q[0]; h->cur[1] = h->e[0]; h->cur[2] = h->p[0]; h->cur[3] = h->u[0];
  return VH_OK;
}

// ---- eta-slab decomposition: the step in four parts, boundary planes in between
static int slab_checks(vh_handle* h, const char* who) {
  if (!h->initialised) return fail(h, VH_ERR_STATE, std::string(who) + " before vh_set_initial");
  if (h->variant != 0 || h->reduced || h->two_d || h->P.n_batch != 1 || h->P.nz < 2)
    return fail(h, VH_ERR_STATE, std::string(who) + " needs the default pipeline (variant 0, storage 0), a 3+1d grid with nz >= 2 and n_batch = 1");
  return VH_OK;
}

int vh_step_part(vh_handle* h, int part) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (int rc = slab_checks(h, "vh_step_part")) return rc;
  if (part != h->next_part) return fail(h, VH_ERR_STATE, "vh_step_part: the parts of a step run in the order 0, 1, 2, 3 (next is " + std::to_string(h->next_part) + ")");
  const double t = h->prm.tau0 + (double)h->n_steps * h->prm.dtau, t1 = t + h->prm.dtau;
  StageArgs A;
  A.cnt = h->cnt;
  if (part < 2) {
    A.q_in = h->q[0]; A.e_in = h->e[0]; A.p_in = h->p[0]; A.u_in = h->u[0]; A.u_prev = h->u[1]; A.q_n = nullptr;
    A.q_out = h->q[1]; A.e_out = h->e[1]; A.p_out = h->p[1]; A.u_out = h->u[2]; A.t = t; A.t_post = t1; A.regfac = nullptr;
  } else {
    A.q_in = h->q[1]; A.e_in = h->e[1]; A.p_in = h->p[1]; A.u_in = h->u[2]; A.u_prev = h->u[0]; A.q_n = h->q[0];
    A.q_out = h->q[2]; A.e_out = h->e[0]; A.p_out = h->p[0]; A.u_out = h->u[1]; A.t = t1; A.t_post = t1; A.regfac = h->regfac;
  }
  CUDA_TRY(h, launch_stage_any(h, part < 2 ? 1 : 2, A, nullptr, (part % 2 == 0) ? 1 : 2));
  if (part == 1) { h->cur[0] = h->q[1]; h->cur[1] = h->e[1]; h->cur[2] = h->p[1]; h->cur[3] = h->u[2]; }
  if (part == 3) {
    real* un = h->u[1]; h->u[1] = h->u[0]; h->u[0] = un;
    real* qn = h->q[2]; h->q[2] = h->q[0]; h->q[0] = qn;
    h->n_steps++;
    h->cur[0] = h->q[0]; h->cur[1] = h->e[0]; h->cur[2] = h->p[0]; h->cur[3] = h->u[0];
  }
  h->next_part = (part + 1) % 4;
  return VH_OK;
}

int vh_halo_size(vh_handle* h, int what, long long* n_doubles) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  if ((what != 0 && what != 1) || !n_doubles) return fail(h, VH_ERR_ARG, "what must be 0 (state velocity) or 1 (state); n_doubles != NULL");
  *n_doubles = (what == 0 ? 1LL : 2LL * 21) * h->P.plane;
  return VH_OK;
}

static int halo_copy(vh_handle* h, int what, int side, double* buf, bool exporting) {
  if (int rc = slab_checks(h, exporting ? "vh_halo_export" : "vh_halo_import")) return rc;
  if ((what != 0 && what != 1) || (side != 0 && side != 1) || !buf) return fail(h, VH_ERR_ARG, "what in {0, 1}, side in {0, 1}, buf != NULL required");
  const DevParams& P = h->P;
  const long long fs = P.fstride;
  PlaneArgs G;
  if (what == 0) {
    // low face: the lower neighbour needs v of the state at the low face of my first plane (vL, eta direction) as its ghost plane nz, and gives me
    // v of the state at the high face of its last plane (vR) for my ghost plane -1; high face: the mirror image
    G.n_arr = 1; G.n_planes = 1;
    const bool lowface = (side == 0);
    G.arr[0] = (exporting == lowface) ? h->vL + 2 * fs : h->vR + 2 * fs;
    G.z0 = exporting ? (lowface ? 2 : P.nz + 1) : (lowface ? 1 : P.nz + 2);
  } else {
    G.n_arr = 21; G.n_planes = 2;
    for (int n = 0; n < 15; ++n) G.arr[n] = h->cur[0] + n * fs;
    G.arr[15] = h->cur[1]; G.arr[16] = h->cur[2];
    for (int n = 0; n < 4; ++n) G.arr[17 + n] = h->cur[3] + n * fs;
    G.z0 = exporting ? (side == 0 ? 2 : P.nz) : (side == 0 ? 0 : P.nz + 2);
  }
  dim3 grid((unsigned)((P.plane + 255) / 256), G.n_arr * G.n_planes);
  if (exporting) plane_kernel<true><<<grid, 256, 0, h->stream>>>(P, G, buf);
  else plane_kernel<false><<<grid, 256, 0, h->stream>>>(P, G, buf);
  if (!exporting) h->slab_nb[side] = true;      // from now on the interface states beyond this face are the neighbour's to count
  h->launches++;
  CUDA_TRY(h, cudaGetLastError());
  return VH_OK;
}
int vh_halo_export(vh_handle* h, int what, int side, double* buf_device) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  return halo_copy(h, what, side, buf_device, true);
}
int vh_halo_import(vh_handle* h, int what, int side, const double* buf_device) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  return halo_copy(h, what, side, const_cast<double*>(buf_device), false);
}

int vh_step(vh_handle* h, int n_steps) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (!h->initialised) return fail(h, VH_ERR_STATE, "vh_step before vh_set_initial");
  if (h->next_part != 0) return fail(h, VH_ERR_STATE, "vh_step in the middle of a step taken with vh_step_part");
  if (n_steps < 0) return fail(h, VH_ERR_ARG, "n_steps must be >= 0");
  for (int it = 0; it < n_steps; ++it) {
    int rc = one_step(h, nullptr);
    if (rc) return rc;
  }
  return VH_OK;
}

int vh_step_profile(vh_handle* h, int n_steps, double* ms4) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (!h->initialised) return fail(h, VH_ERR_STATE, "vh_step_profile before vh_set_initial");
  if (h->next_part != 0) return fail(h, VH_ERR_STATE, "vh_step_profile in the middle of a step taken with vh_step_part");
  if (n_steps < 1 || !ms4) return fail(h, VH_ERR_ARG, "n_steps >= 1 and ms4 != NULL required");
  cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  struct Guard { cudaEvent_t* e; ~Guard() { for (int i = 0; i < 5; ++i) if (e[i]) cudaEventDestroy(e[i]); } } guard{ev};      // also on every early return
  for (int i = 0; i < 5; ++i) CUDA_TRY(h, cudaEventCreate(&ev[i]));
  double acc[4] = {0, 0, 0, 0};
  for (int it = 0; it < n_steps; ++it) {
    int rc = one_step(h, ev);
    if (rc) return rc;
    CUDA_TRY(h, cudaEventSynchronize(ev[4]));
    for (int i = 0; i < 4; ++i) { float ms = 0; CUDA_TRY(h, cudaEventElapsedTime(&ms, ev[i], ev[i + 1])); acc[i] += ms; }
  }
  for (int i = 0; i < 4; ++i) ms4[i] = acc[i] / n_steps;
  return VH_OK;
}

int vh_get_fields(vh_handle* h, double* q15, double* e, double* p, double* u4, double* u4_prev, int mem_space) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (!h->initialised) return fail(h, VH_ERR_STATE, "vh_get_fields before vh_set_initial");
  if (mem_space != 0 && mem_space != 1) return fail(h, VH_ERR_ARG, "mem_space must be 0 (host) or 1 (device)");
  const DevParams& P = h->P;
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const unsigned nb = (unsigned)((np + 255) / 256);
  struct Item { double* dst; real* src; int nc; };
  Item items[5] = {{q15, h->q[0], 15}, {e, h->e[0], 1}, {p, h->p[0], 1}, {u4, h->u[0], 4}, {u4_prev, h->u[1], 4}};
  if (mem_space == 0) {
    int rc = ensure_stage(h, &h->stage_out, &h->stage_out_bytes, (size_t)15 * np * sizeof(double));
    if (rc) return rc;
  }
  const real tnow = (real)(h->prm.tau0 + (double)h->n_steps * h->prm.dtau);
  const real tprev = (real)(h->uprev_initial ? tnow : tnow - h->prm.dtau);
  for (int n = 0; n < 5; ++n) {
    const Item& it = items[n];
    if (!it.dst) continue;
    double* target = (mem_space == 1) ? it.dst : h->stage_out;
    if (h->reduced && (n == 0 || n >= 3)) {      // q15, u4, u4_prev: expanded from the stored subset (Eqs. 47-51, u.u = 1)
      const bool mil = (h->prm.geometry == 0);
      const real* qs = (n == 0) ? h->q[0] : nullptr;
      const real* us = (n == 4) ? h->u[1] : h->u[0];
      const real tt = (n == 4) ? tprev : tnow;
      if (mil) export_reduced_kernel<true><<<nb, 256, 0, h->stream>>>(P, qs, us, tt, n == 0 ? target : nullptr, n == 0 ? nullptr : target);
      else export_reduced_kernel<false><<<nb, 256, 0, h->stream>>>(P, qs, us, tt, n == 0 ? target : nullptr, n == 0 ? nullptr : target);
    } else
    pack_kernel<true><<<nb, 256, 0, h->stream>>>(P, it.src, target, it.nc);
    h->launches++;
    CUDA_TRY(h, cudaGetLastError());
    if (mem_space == 0) CUDA_TRY(h, cudaMemcpyAsync(it.dst, h->stage_out, (size_t)it.nc * np * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  }
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  return VH_OK;
}

int vh_get_status(vh_handle* h, double* tau, long long* n_steps_done, long long* n_inversion_failures, long long* n_nonfinite,
                  double* min_reg_factor) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  Counters c;
  CUDA_TRY(h, cudaMemcpyAsync(&c, h->cnt, sizeof(c), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  if (tau) *tau = h->prm.tau0 + (double)h->n_steps * h->prm.dtau;
  if (n_steps_done) *n_steps_done = h->n_steps;
  if (n_inversion_failures) *n_inversion_failures = (long long)c.n_fail;
  if (n_nonfinite) *n_nonfinite = (long long)c.n_nonfinite;
  if (min_reg_factor) std::memcpy(min_reg_factor, &c.min_reg_bits, sizeof(double));
  return VH_OK;
}

int vh_eos_table(double* nodes4, double* x0, double* h) {
  if (!nodes4) return fail(nullptr, VH_ERR_ARG, "nodes4 is NULL");
  static_assert(VH_EOS_TABLE_NODES == vh_eos::VH_EOS_N + 1, "header and builder disagree on the table size");
  const vh_eos::LatticeTable tab = vh_eos::Builder().build();
  std::memcpy(nodes4, tab.node.data(), tab.node.size() * sizeof(double));
  if (x0) *x0 = tab.x0;
  if (h) *h = tab.h;
  return VH_OK;
}

int vh_get_diagnostics(vh_handle* h, double* out10) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (h->reduced) return fail(h, VH_ERR_STATE, "vh_get_diagnostics is not available in reduced-storage mode (storage = 1): the diagnostics kernels read the full set of arrays");
  if (!h->initialised) return fail(h, VH_ERR_STATE, "vh_get_diagnostics before vh_set_initial");
  if (!out10) return fail(h, VH_ERR_ARG, "out10 is NULL");
  if (!h->diag && cudaMalloc((void**)&h->diag, 10 * sizeof(unsigned long long)) != cudaSuccess) { cudaGetLastError(); h->diag = nullptr; return fail(h, VH_ERR_ALLOC, "cudaMalloc(diagnostics) failed"); }
  CUDA_TRY(h, cudaMemsetAsync(h->diag, 0, 10 * sizeof(unsigned long long), h->stream));
  const double t = h->prm.tau0 + (double)h->n_steps * h->prm.dtau;
  if (h->prm.eos == 2) launch_diag<2>(h, t, nullptr); else if (h->prm.eos == 1) launch_diag<1>(h, t, nullptr); else launch_diag<0>(h, t, nullptr);
  CUDA_TRY(h, cudaGetLastError());
  unsigned long long bits[10];
  CUDA_TRY(h, cudaMemcpyAsync(bits, h->diag, sizeof(bits), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  std::memcpy(out10, bits, sizeof(bits));
  return VH_OK;
}

int vh_get_diagnostic_maps(vh_handle* h, double* maps10, int mem_space) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (h->reduced) return fail(h, VH_ERR_STATE, "vh_get_diagnostic_maps is not available in reduced-storage mode (storage = 1): the diagnostics kernels read the full set of arrays");
  if (!maps10) return fail(h, VH_ERR_ARG, "maps10 is NULL");
  if (mem_space != 0 && mem_space != 1) return fail(h, VH_ERR_ARG, "mem_space must be 0 (host) or 1 (device)");
  if (!h->initialised) return fail(h, VH_ERR_STATE, "vh_get_diagnostic_maps before vh_set_initial");
  if (!h->diag && cudaMalloc((void**)&h->diag, 10 * sizeof(unsigned long long)) != cudaSuccess) { cudaGetLastError(); h->diag = nullptr; return fail(h, VH_ERR_ALLOC, "cudaMalloc(diagnostics) failed"); }
  const size_t bytes = (size_t)10 * h->P.nx * h->P.ny * h->P.nz * h->P.n_batch * sizeof(double);
  double* dev = maps10;
  if (mem_space == 0) {      // host destination: through the staging buffer of vh_get_fields
    int rc = ensure_stage(h, &h->stage_out, &h->stage_out_bytes, bytes);
    if (rc) return rc;
    dev = h->stage_out;
  }
  CUDA_TRY(h, cudaMemsetAsync(h->diag, 0, 10 * sizeof(unsigned long long), h->stream));
  const double t = h->prm.tau0 + (double)h->n_steps * h->prm.dtau;
  if (h->prm.eos == 2) launch_diag<2>(h, t, dev); else if (h->prm.eos == 1) launch_diag<1>(h, t, dev); else launch_diag<0>(h, t, dev);
  CUDA_TRY(h, cudaGetLastError());
  if (mem_space == 0) CUDA_TRY(h, cudaMemcpyAsync(maps10, dev, bytes, cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  return VH_OK;
}

int vh_enable_regulation_map(vh_handle* h, int on) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (h->reduced) return fail(h, VH_ERR_STATE, "vh_enable_regulation_map is not available in reduced-storage mode (storage = 1): the diagnostics kernels read the full set of arrays");
  if (!on) {
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    cudaFree(h->regfac);
    h->regfac = nullptr;
    return VH_OK;
  }
  if (!h->regfac) {
    if (cudaMalloc((void**)&h->regfac, (size_t)h->P.fstride * sizeof(real)) != cudaSuccess) {
      cudaGetLastError();
      h->regfac = nullptr;
      return fail(h, VH_ERR_ALLOC, "cudaMalloc(regulation map) failed");
    }
    CUDA_TRY(h, reset_regulation_map(h));
  }
  return VH_OK;
}

int vh_get_regulation_map(vh_handle* h, double* map, int mem_space) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (h->reduced) return fail(h, VH_ERR_STATE, "vh_get_regulation_map is not available in reduced-storage mode (storage = 1): the diagnostics kernels read the full set of arrays");
  if (!map) return fail(h, VH_ERR_ARG, "map is NULL");
  if (mem_space != 0 && mem_space != 1) return fail(h, VH_ERR_ARG, "mem_space must be 0 (host) or 1 (device)");
  if (!h->regfac) return fail(h, VH_ERR_STATE, "vh_get_regulation_map without vh_enable_regulation_map(h, 1)");
  const DevParams& P = h->P;
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  double* target = map;
  if (mem_space == 0) {
    int rc = ensure_stage(h, &h->stage_out, &h->stage_out_bytes, (size_t)np * sizeof(double));
    if (rc) return rc;
    target = h->stage_out;
  }
  pack_kernel<true><<<(unsigned)((np + 255) / 256), 256, 0, h->stream>>>(P, h->regfac, target, 1);
  h->launches++;
  CUDA_TRY(h, cudaGetLastError());
  if (mem_space == 0) CUDA_TRY(h, cudaMemcpyAsync(map, h->stage_out, (size_t)np * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  return VH_OK;
}

int vh_run_until(vh_handle* h, double T_f, int max_steps, int check_every, long long* steps_done) {
  if (!h) return fail(nullptr, VH_ERR_ARG, "handle is NULL");
  VH_ENTER(h);
  if (h->reduced) return fail(h, VH_ERR_STATE, "vh_run_until is not available in reduced-storage mode (storage = 1): the diagnostics kernels read the full set of arrays");
  if (!h->initialised) return fail(h, VH_ERR_STATE, "vh_run_until before vh_set_initial");
  if (h->next_part != 0) return fail(h, VH_ERR_STATE, "vh_run_until in the middle of a step taken with vh_step_part");
  if (max_steps < 0 || check_every < 1 || !(T_f >= 0.0)) return fail(h, VH_ERR_ARG, "max_steps >= 0, check_every >= 1, T_f >= 0 required");
  long long done = 0;
  double d[10];
  while (done < max_steps) {
    int rc = vh_get_diagnostics(h, d);
    if (rc) return rc;
    if (d[0] < T_f) break;                                  // T < T_f everywhere (:494)
    const int n = (int)std::min<long long>(check_every, max_steps - done);
    rc = vh_step(h, n);
    if (rc) return rc;
    done += n;
  }
  if (steps_done) *steps_done = done;
  return VH_OK;
}

int vh_measure_peaks(void* cuda_stream, long long n_bytes, int repeats, double* copy_gbs, double* fp64_gflops) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (n_bytes < (1 << 20) || repeats < 1) return fail(nullptr, VH_ERR_ARG, "n_bytes >= 1 MiB and repeats >= 1 required");
  int dev = 0, nsm = 0;
  CUDA_TRY(nullptr, cudaGetDevice(&dev));
  CUDA_TRY(nullptr, cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
  cudaEvent_t e0, e1;
  CUDA_TRY(nullptr, cudaEventCreate(&e0));
  CUDA_TRY(nullptr, cudaEventCreate(&e1));
  if (copy_gbs) {
    double *a = nullptr, *b = nullptr;
    long long n2 = n_bytes / 16;
    if (cudaMalloc((void**)&a, n2 * 16) != cudaSuccess || cudaMalloc((void**)&b, n2 * 16) != cudaSuccess) {
      cudaFree(a); cudaFree(b);
      return fail(nullptr, VH_ERR_ALLOC, "cudaMalloc(copy buffers) failed");
    }
    cudaMemsetAsync(a, 0, n2 * 16, st);
    double best = 0;
    for (int r = 0; r < repeats + 1; ++r) {
      cudaEventRecord(e0, st);
      copy_kernel<<<nsm * 16, 256, 0, st>>>((const double2*)a, (double2*)b, n2);
      cudaEventRecord(e1, st);
      cudaEventSynchronize(e1);
      float ms = 0;
      cudaEventElapsedTime(&ms, e0, e1);
      double gbs = 2.0 * n2 * 16 / (ms * 1e-3) / 1e9;
      if (r > 0 && gbs > best) best = gbs;
    }
    cudaFree(a); cudaFree(b);
    *copy_gbs = best;
  }
  if (fp64_gflops) {
    double* o = nullptr;
    CUDA_TRY(nullptr, cudaMalloc((void**)&o, 8));
    const int iters = 4096, blocks = nsm * 8;
    double best = 0;
    for (int r = 0; r < repeats + 1; ++r) {
      cudaEventRecord(e0, st);
      fma_kernel<<<blocks, 256, 0, st>>>(o, iters, 0.999999, 1e-6);
      cudaEventRecord(e1, st);
      cudaEventSynchronize(e1);
      float ms = 0;
      cudaEventElapsedTime(&ms, e0, e1);
      double gf = 2.0 * 64.0 * iters * 256.0 * blocks / (ms * 1e-3) / 1e9;
      if (r > 0 && gf > best) best = gf;
    }
    cudaFree(o);
    *fp64_gflops = best;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  CUDA_TRY(nullptr, cudaGetLastError());
  return VH_OK;
}

int vh_measure_fp32_peak(void* cuda_stream, int repeats, double* fp32_gflops) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (repeats < 1 || !fp32_gflops) return fail(nullptr, VH_ERR_ARG, "repeats >= 1 and fp32_gflops != NULL required");
  int dev = 0, nsm = 0;
  CUDA_TRY(nullptr, cudaGetDevice(&dev));
  CUDA_TRY(nullptr, cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
  cudaEvent_t e0, e1;
  CUDA_TRY(nullptr, cudaEventCreate(&e0));
  if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return fail(nullptr, VH_ERR_CUDA, "cudaEventCreate failed"); }
  float* o = nullptr;
  if (cudaMalloc((void**)&o, 8) != cudaSuccess) { cudaGetLastError(); cudaEventDestroy(e0); cudaEventDestroy(e1); return fail(nullptr, VH_ERR_ALLOC, "cudaMalloc failed"); }
  const int iters = 8192, blocks = nsm * 8;
  double best = 0;
  for (int r = 0; r < repeats + 1; ++r) {
    cudaEventRecord(e0, st);
    fma32_kernel<<<blocks, 256, 0, st>>>(o, iters, 0.999999f, 1e-6f);
    cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    double gf = 2.0 * 64.0 * iters * 256.0 * blocks / (ms * 1e-3) / 1e9;
    if (r > 0 && gf > best) best = gf;
  }
  cudaFree(o);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *fp32_gflops = best;
  CUDA_TRY(nullptr, cudaGetLastError());
  return VH_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ diagnostics without allocation
// vh_diagnostics_noalloc (include/vh.h): the ten diagnostics for callers that may not allocate device memory - the host program gave the
// GPU's free memory to its own pool, or sits in a loop that cannot take the device-wide stall of cudaMalloc / cudaFree.  A variant of
// diagnostics_kernel (vh_kernels.cuh) that reads the caller's compact arrays and keeps everything it needs beyond them - per-block
// maxima, the last-block ticket, the EOS-2 table - in the two arrays below.  They are part of the library image: each GPU that loads the
// library carries them (about 390 KB) until the process exits, and every call on that GPU reuses them.
namespace vh {
constexpr int NA_THREADS = 256;                                        // one cell per thread, no grid-stride loop: block b owns cells [256 b, 256 b + 256)
constexpr int NA_MAX_BLOCKS = VH_NOALLOC_MAX_CELLS / NA_THREADS;        // 4096
constexpr int NA_RESULT = 10 * NA_MAX_BLOCKS;                          // [0, NA_RESULT): maximum s of block b at s * NA_MAX_BLOCKS + b
constexpr int NA_TICKET = NA_RESULT + 32;                              // [NA_RESULT, +10): the ten results when out10 is a host pointer
constexpr int NA_DOUBLES = NA_TICKET + 32;                             // [NA_TICKET]: the ticket (an unsigned int in a 256-byte line of its own)
static_assert(VH_NOALLOC_MAX_CELLS % NA_THREADS == 0, "the size limit is a whole number of blocks");
}  // namespace vh

// In HOST code these two names are only handles for cudaGetSymbolAddress; they are not device addresses and must never be passed to a
// kernel (noalloc_setup below does the lookup once per device).
static __device__ __align__(256) double vh_noalloc_scratch[vh::NA_DOUBLES];
static __device__ __align__(256) vh::real vh_noalloc_eos_table[4 * VH_EOS_TABLE_NODES];

namespace vh {

// max over the block of each of ten values; the result is valid in thread s < 10 (for value s)
__device__ __forceinline__ real block_max10(real (&m)[10], real (*sm)[NA_THREADS / 32]) {
#pragma unroll
  for (int s = 0; s < 10; ++s) {
    real v = m[s];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) sm[s][threadIdx.x >> 5] = v;
  }
  __syncthreads();
  real r = real(0.0);
  if (threadIdx.x < 10) {
#pragma unroll
    for (int w = 0; w < NA_THREADS / 32; ++w) r = fmax(r, sm[threadIdx.x][w]);
  }
  __syncthreads();      // sm may be reused by the caller
  return r;
}

// The per-cell arithmetic is that of diagnostics_kernel, statement by statement; what differs is where the data comes from (compact double
// arrays; a neighbour beyond the edge is the edge cell itself, which is what the ghost cells of Eqs. 75-76 hold; p = P0(e) computed here)
// and where the maxima go (no atomics on a zeroed array: per-block maxima into `scratch`, combined by whichever block draws the last ticket).
template <int EOS, bool MILNE>
__global__ void __launch_bounds__(NA_THREADS) diagnostics_noalloc_kernel(const __grid_constant__ DevParams P, const double* __restrict__ q, const double* __restrict__ e,
                                                                         const double* __restrict__ u, const double* __restrict__ u_prev, real t,
                                                                         double* scratch, double* result, double* __restrict__ maps) {
  __shared__ real sm[10][NA_THREADS / 32];
  __shared__ bool last_block;
  const long long np = (long long)P.nx * P.ny * P.nz * P.n_batch;
  const real t2 = MILNE ? t * t : real(1.0);
  real v[10] = {real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0), real(0.0)};
  const long long n = (long long)blockIdx.x * NA_THREADS + threadIdx.x;
  if (n < np) {
    const int i = (int)(n % P.nx);
    const int j = (int)((n / P.nx) % P.ny);
    const int k = (int)((n / ((long long)P.nx * P.ny)) % P.nz);
    const long long sy = P.nx, sz = (long long)P.nx * P.ny;
    const long long xm = n - (i > 0 ? 1 : 0), xp = n + (i < P.nx - 1 ? 1 : 0);
    const long long ym = n - (j > 0 ? sy : 0), yp = n + (j < P.ny - 1 ? sy : 0);
    const long long zm = n - (k > 0 ? sz : 0), zp = n + (k < P.nz - 1 ? sz : 0);
    const bool has_z = P.nz > 1;                      // nz = 1 is the 2+1d mode: no eta differences
    const real ee = (real)e[n], pp = eos_p<EOS>(P, ee);
    const real ut = (real)u[n], ux = (real)u[np + n], uy = (real)u[2 * np + n], un = (real)u[3 * np + n];
    real pi[10];
#pragma unroll
    for (int s = 0; s < 10; ++s) pi[s] = (real)q[(PTT + s) * np + n];
    const real Pi = (real)q[BPI * np + n];
    const real norm = ut * ut - ux * ux - uy * uy - t2 * un * un;
    const real tr = pi[0] - pi[4] - pi[7] - t2 * pi[9];
    const real pipi = pi[0] * pi[0] - real(2.0) * (pi[1] * pi[1] + pi[2] * pi[2] + t2 * pi[3] * pi[3]) + pi[4] * pi[4] + real(2.0) * pi[5] * pi[5] +
                        real(2.0) * t2 * pi[6] * pi[6] + pi[7] * pi[7] + real(2.0) * t2 * pi[8] * pi[8] + t2 * t2 * pi[9] * pi[9];
    const real c0 = pi[0] * ut - pi[1] * ux - pi[2] * uy - t2 * pi[3] * un;
    const real c1 = pi[1] * ut - pi[4] * ux - pi[5] * uy - t2 * pi[6] * un;
    const real c2 = pi[2] * ut - pi[5] * ux - pi[7] * uy - t2 * pi[8] * un;
    const real c3 = (pi[3] * ut - pi[6] * ux - pi[8] * uy - t2 * pi[9] * un) * (MILNE ? t : real(1.0));
    const real iw = real(1.0) / (ee + pp), ip = real(1.0) / pp;
    v[1] = fabs(norm - real(1.0));
    v[2] = fabs(tr) * iw;
    v[3] = fmax(fmax(fabs(c0), fabs(c1)), fmax(fabs(c2), fabs(c3))) * iw;
    v[4] = sqrt(fabs(pipi)) * ip;
    v[5] = fabs(Pi) * ip;
    real theta = (MILNE ? ut / t : real(0.0)) + (ut - (real)u_prev[n]) * P.inv_dtau;
    theta += ((real)u[np + xp] - (real)u[np + xm]) * (real(0.5) * P.inv_dx) + ((real)u[2 * np + yp] - (real)u[2 * np + ym]) * (real(0.5) * P.inv_dy);
    if (has_z) theta += ((real)u[3 * np + zp] - (real)u[3 * np + zm]) * (real(0.5) * P.inv_dz);
    if (P.shear || P.bulk) {
      const real uc[4] = {ut, ux, uy, un};
      real dt[4], dx[4], dy[4], dn[4];
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        const double* ua = u + a * np;
        dt[a] = ((real)ua[n] - (real)u_prev[a * np + n]) * P.inv_dtau;
        dx[a] = ((real)ua[xp] - (real)ua[xm]) * (real(0.5) * P.inv_dx);
        dy[a] = ((real)ua[yp] - (real)ua[ym]) * (real(0.5) * P.inv_dy);
        dn[a] = has_z ? ((real)ua[zp] - (real)ua[zm]) * (real(0.5) * P.inv_dz) : real(0.0);
      }
      Kin K;
      kinematics<MILNE>(uc, dt, dx, dy, dn, t, K);
      real r2s, r2b;
      second_order_reynolds<EOS, MILNE>(P, t, uc, K, pi, Pi, ee, r2s, r2b);
      v[8] = (P.shear && isfinite(r2s)) ? r2s : real(0.0);
      v[9] = (P.bulk && isfinite(r2b)) ? r2b : real(0.0);
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
    if (maps) {
#pragma unroll
      for (int s = 0; s < 10; ++s) maps[s * np + n] = (double)v[s];
    }
  }
  // this block's maxima (fmax drops a NaN, as the loop of diagnostics_kernel does)
  real m[10];
#pragma unroll
  for (int s = 0; s < 10; ++s) m[s] = fmax(real(0.0), v[s]);
  const real mine = block_max10(m, sm);
  if (threadIdx.x < 10) {
    __stcg(scratch + threadIdx.x * NA_MAX_BLOCKS + blockIdx.x, (double)mine);
    __threadfence();                                  // the maxima are visible device-wide before this block takes its ticket
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned int ticket = atomicAdd(reinterpret_cast<unsigned int*>(scratch + NA_TICKET), 1u);      // the host zeroed it before this launch
    last_block = (ticket == gridDim.x - 1);
  }
  __syncthreads();
  if (!last_block) return;
  __threadfence();
  // last block: combine the gridDim.x per-block maxima (only those - older, larger calls left more behind them in the array)
#pragma unroll
  for (int s = 0; s < 10; ++s) {
    real r = real(0.0);
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NA_THREADS) r = fmax(r, (real)__ldcg(scratch + s * NA_MAX_BLOCKS + b));
    m[s] = r;
  }
  const real all = block_max10(m, sm);
  if (threadIdx.x < 10) result[threadIdx.x] = (double)all;
}

}  // namespace vh

// Once per device and process, with that device current: the device addresses of the two arrays (checked), and the EOS-2 table
// uploaded into its array.  No allocation on the device; the table is built on the host as vh_create builds it.
namespace {
struct NoallocDevice {
  bool ready = false;
  double* scratch = nullptr;          // device address of vh_noalloc_scratch on this device
  vh::real* table = nullptr;          // device address of vh_noalloc_eos_table on this device
};
constexpr int kNoallocMaxDevices = 64;
NoallocDevice g_noalloc_dev[kNoallocMaxDevices];
vh_eos::LatticeTable g_noalloc_lattice;      // host copy (the scalars that go into DevParams), built with the first device
std::mutex g_noalloc_mutex;
}  // namespace

static int noalloc_setup(int dev, cudaStream_t st, const NoallocDevice** out) {
  if (dev < 0 || dev >= kNoallocMaxDevices) return fail(nullptr, VH_ERR_ARG, "vh_diagnostics_noalloc: device ordinal " + std::to_string(dev) + " is beyond the " + std::to_string(kNoallocMaxDevices) + " this entry point keeps books for");
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  NoallocDevice& d = g_noalloc_dev[dev];
  if (!d.ready) {
    double* scratch = nullptr;
    vh::real* table = nullptr;
    CUDA_TRY(nullptr, cudaGetSymbolAddress((void**)&scratch, vh_noalloc_scratch));
    CUDA_TRY(nullptr, cudaGetSymbolAddress((void**)&table, vh_noalloc_eos_table));
    if (!scratch || !table) return fail(nullptr, VH_ERR_CUDA, "vh_diagnostics_noalloc: cudaGetSymbolAddress returned a null address");
    if (g_noalloc_lattice.node.empty()) g_noalloc_lattice = vh_eos::Builder().build();
    const std::vector<real> nodes(g_noalloc_lattice.node.begin(), g_noalloc_lattice.node.end());      // the table in the library's precision
    if (nodes.size() != (size_t)4 * VH_EOS_TABLE_NODES) return fail(nullptr, VH_ERR_STATE, "vh_diagnostics_noalloc: EOS table size does not match its array");
    CUDA_TRY(nullptr, cudaMemcpyAsync(table, nodes.data(), nodes.size() * sizeof(real), cudaMemcpyHostToDevice, st));
    CUDA_TRY(nullptr, cudaStreamSynchronize(st));      // nodes lives on this stack frame
    d.scratch = scratch; d.table = table; d.ready = true;
  }
  *out = &d;
  return VH_OK;
}

extern "C" int vh_diagnostics_noalloc(const vh_params* p, double tau, const double* q15, const double* e, const double* u4, const double* u4_prev,
                                      double* out10, int out_mem_space, double* maps10, void* cuda_stream) {
  // argument checks first: none of them touches the device
  std::string why;
  if (check_params(p, why)) return fail(nullptr, VH_ERR_ARG, "vh_diagnostics_noalloc: " + why);
  if (!q15 || !e || !u4 || !u4_prev || !out10) return fail(nullptr, VH_ERR_ARG, "vh_diagnostics_noalloc: q15, e, u4, u4_prev and out10 are required");
  if (out_mem_space != 0 && out_mem_space != 1) return fail(nullptr, VH_ERR_ARG, "vh_diagnostics_noalloc: out_mem_space must be 0 (host) or 1 (device)");
  if (p->geometry == 0 && !(tau > 0)) return fail(nullptr, VH_ERR_ARG, "vh_diagnostics_noalloc: Milne geometry needs tau > 0");
  const long long np = (long long)p->nx * p->ny * p->nz * p->n_batch;
  if (np > VH_NOALLOC_MAX_CELLS)
    return fail(nullptr, VH_ERR_ARG, "vh_diagnostics_noalloc: the grid has " + std::to_string(np) + " cells, the fixed scratch array of this entry point serves at most " +
                                         std::to_string((long long)VH_NOALLOC_MAX_CELLS) + " (VH_NOALLOC_MAX_CELLS); use a handle and vh_get_diagnostics for larger grids");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = -1;
  CUDA_TRY(nullptr, cudaGetDevice(&dev));
  const NoallocDevice* d = nullptr;
  if (int rc = noalloc_setup(dev, st, &d)) return rc;
  DevParams P;
  fill_dev_params(*p, P);
  if (p->eos == 2) {      // as in vh_create, with the table in its fixed array
    const vh_eos::LatticeTable& tab = g_noalloc_lattice;
    const int n = vh_eos::VH_EOS_N;
    const double* nd = tab.node.data();
    const double e0 = std::pow(tab.x0, 4), eN = std::pow(tab.xN, 4);
    P.eos_tab = reinterpret_cast<const real2*>(d->table);
    P.eos_n = n; P.eos_x0 = tab.x0; P.eos_xN = tab.xN; P.eos_inv_h = 1.0 / tab.h;
    P.eos_lo_slope = nd[0] / e0; P.eos_pN = nd[4 * n]; P.eos_eN = eN;
    P.eos_T0_over_x0 = nd[2] / tab.x0; P.eos_TN_over_xN = nd[4 * n + 2] / tab.xN;
  }
  // the one word that has to start from zero; the per-block maxima are overwritten before they are read
  CUDA_TRY(nullptr, cudaMemsetAsync(d->scratch + NA_TICKET, 0, sizeof(unsigned int), st));
  double* result = (out_mem_space == 1) ? out10 : d->scratch + NA_RESULT;
  const unsigned nb = (unsigned)((np + NA_THREADS - 1) / NA_THREADS);
  const real t = (real)tau;
  const bool mil = (p->geometry == 0);
#define VH_NA_LAUNCH(E)                                                                                                               \
  do {                                                                                                                                \
    if (mil) diagnostics_noalloc_kernel<E, true><<<nb, NA_THREADS, 0, st>>>(P, q15, e, u4, u4_prev, t, d->scratch, result, maps10);    \
    else diagnostics_noalloc_kernel<E, false><<<nb, NA_THREADS, 0, st>>>(P, q15, e, u4, u4_prev, t, d->scratch, result, maps10);       \
  } while (0)
  if (p->eos == 2) VH_NA_LAUNCH(2); else if (p->eos == 1) VH_NA_LAUNCH(1); else VH_NA_LAUNCH(0);
#undef VH_NA_LAUNCH
  CUDA_TRY(nullptr, cudaGetLastError());
  if (out_mem_space == 0) {
    CUDA_TRY(nullptr, cudaMemcpyAsync(out10, result, 10 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(nullptr, cudaStreamSynchronize(st));
  }
  return VH_OK;
}
