/* vh.h -- C ABI of the B200-native Kurganov-Tadmor / Heun step for 3+1d relativistic viscous hydrodynamics
 * (arXiv 1608.06577, "GPU-VH").  Citations are PAPER.md line numbers / equation numbers.
 *
 * The library advances, entirely on one GPU, the 15 double-precision fields per cell
 *   q = (T^tt, T^tx, T^ty, T^tn,  pi^tt, pi^tx, pi^ty, pi^tn, pi^xx, pi^xy, pi^xn, pi^yy, pi^yn, pi^nn,  Pi)
 * (Eqs. 56-58, :357-363; pi^{y eta} restored, reading R2) by the program flow of PAPER.md :503-529:
 * two forward-Euler stages of the KT semi-discrete scheme (Eqs. 59-68) combined as Heun/RK2 (Eqs. 69-71), each stage
 * followed by the per-cell inversion to (e, p, u^mu) (Eqs. 52-54, 72), the regularisation of pi^{mu nu}, Pi
 * (Eqs. 73-74) and the ghost-cell boundary condition (Eqs. 75-76).
 *
 * Conventions for EVERY array argument:
 *   - physical cells only (no ghost cells), double precision,
 *   - index order x fastest, then y, then eta_s, then event (batch):  idx = i + nx*(j + ny*(k + nz*b)),
 *   - multi-component arrays are component-major SoA: u4 = 4 consecutive arrays (u^tau,u^x,u^y,u^eta: contravariant, :251),
 *     pi10 = 10 consecutive arrays in the order of q[4..13], q15 = 15 consecutive arrays,
 *   - mem_space 0: host pointer, 1: device pointer (e.g. the storage of a torch tensor) valid on the handle's stream,
 *   - the caller owns what it passes and may free it when the call returns; the library owns its padded internal buffers.
 * Units: natural units, e and pressures in fm^-4, T in fm^-1, lengths in fm (reading R13).
 *
 * Every function returns VH_OK (0) or a negative error code and never throws or aborts; vh_last_error() gives a
 * message for the most recent failure on that handle (or the global message when the handle is NULL).
 * All work of vh_set_initial / vh_step / vh_get_fields is enqueued on the CUDA stream given to vh_create;
 * vh_step is asynchronous; vh_get_fields and vh_get_status synchronise that stream before returning.
 * There is no CPU fallback: without a CUDA device vh_create fails with VH_ERR_CUDA.
 *
 * Two libraries export this ABI: libvh.so computes in double precision (the product; everything BASELINE.json measures) and libvh_f32.so
 * is the same source compiled with a float scalar (the paper's own runs are single precision).  Array arguments are double
 * in both; libvh_f32.so converts on the way in and out and refuses a Newton tolerance below 1e-6.
 */
#ifndef VH_H_
#define VH_H_

#ifdef __cplusplus
extern "C" {
#endif

#define VH_OK 0
#define VH_ERR_ARG (-1)      /* NULL pointer, non-positive size, unsupported combination */
#define VH_ERR_ALLOC (-2)    /* device allocation failed */
#define VH_ERR_CUDA (-3)     /* CUDA runtime error (message in vh_last_error) */
#define VH_ERR_STATE (-4)    /* call out of order (e.g. vh_step before vh_set_initial) */

typedef struct vh_handle vh_handle;

typedef struct {
  int nx, ny, nz, n_batch;          /* physical cells per event; nz == 1 -> 2+1d (:474); n_batch >= 1 independent events  */
  double dx, dy, dz;                /* fm, fm, rapidity units                                                           */
  double tau0, dtau;                /* fm                                                                               */
  int geometry;                     /* 0 Milne (Eqs. 27-29); 1 Cartesian: G terms and Christoffel symbols off, tau^2 -> 1 (:684) */
  int physics;                      /* bit0 shear pi^{mu nu}, bit1 bulk Pi; 0 = ideal (pi, Pi stay 0)                     */
  int eos;                          /* 0: p = e/3;  1: p = (e/3)(1 - alpha exp(-e/e0));  T = (e/a)^{1/4} for both;         */
                                    /* 2: lattice EOS of Eqs. 19-20 (:200-215) with T(e), c_s^2 from its table (DESIGN R19, R20) */
  double eos_a, eos_alpha, eos_e0;
  double eta_over_s;                /* constant                                                                         */
  int zeta_model;                   /* 0: zeta/s = 0; 1: amp*exp(-((T-T0)/width)^2) (BASELINE configs 3-5); 2: constant;  */
                                    /* 3: Eq. 17 (:174-186) times (zeta/s)_norm = zeta_amp with T_c = zeta_T0 (paper: 0.2 GeV) */
  double zeta_amp, zeta_T0, zeta_width;  /* T0, width in fm^-1                                                            */
  double c_tau_pi;                  /* tau_pi = c_tau_pi*eta/(e+p); Eq. 13 -> 5                                          */
  double c_tau_Pi;                  /* tau_Pi = c_tau_Pi*zeta/((e+p)(1/3-cs2)^2); configs 5, Eq. 10 -> 1/15              */
  double delta_pipi, tau_pipi, lambda_piPi;    /* delta_pipi/tau_pi, tau_pipi/tau_pi, lambda_piPi/tau_pi: 4/3, 10/7, 6/5 (Eqs. 14-16) */
  double delta_PiPi, lambda_Pipi_coef;         /* delta_PiPi/tau_Pi = 2/3, lambda_Pipi/tau_Pi = coef*(1/3-cs2), coef 8/5 (Eqs. 11-12) */
  double minmod_theta;              /* flux limiter theta in [1,2], Eq. 67                                              */
  double xi0, rho_max;              /* Eq. 74: 0.1, 1 (:445)                                                            */
  int newton_max_iter;              /* Newton-Raphson cap for Eq. 72 (reading R6: 50)                                   */
  double newton_rtol;               /* accuracy of the root: the last Newton correction satisfies |de| <= rtol*|e| (1e-13).  The kernels test
                                       |de| <= max(rtol, 0.1*sqrt(rtol))*|e| and then apply that correction: by quadratic convergence the
                                       next one is below rtol*|e| (R6), which saves the iteration that would only confirm it    */
  double tau_relax_floor_over_dtau; /* c: 1/tau_Pi, 1/tau_pi <= 1/(c*dtau) (reading R14); 0 disables                    */
  int storage;                      /* 0: all ten pi^{mu nu} and four u^mu are state (the paper's choice, :333); 1: reduced storage (:476,
                                       Eqs. 47-51, reading R22): pi^xx, pi^xy, pi^xeta, pi^yy, pi^yeta and u^x, u^y, u^eta only - 43 instead
                                       of 61 state arrays; a slower kernel of its own                                                    */
} vh_params;

/* Create a solver for the grid / physics in *p on the current CUDA device.  cuda_stream: a cudaStream_t (may be NULL =
 * default stream).  Allocates 67 padded SoA arrays (43 with storage = 1) (3 x 15 q, 3 x 4 u, 2 x e, 2 x p; :470-476 plus the ping-pong copy of
 * e, p needed because inversion is fused into the stage kernel; and the 6 state-velocity arrays the velocity kernel hands
 * to the stage kernel).  The handle belongs to that device: every later call switches to it.  *out is set only on success. */
int vh_create(const vh_params* p, void* cuda_stream, vh_handle** out);

/* Program-flow steps 3-5 (:489-491): build q^0 from (e, u^mu, pi^{mu nu}, Pi) by Eqs. 32-33 (:267-269), p = P0(e),
 * u^{-1} = u^0 (footnote 4, :519), fill ghost cells, reset tau = tau0 and all counters.  pi10 / Pi may be NULL (= 0).  */
int vh_set_initial(vh_handle* h, const double* e, const double* u4, const double* pi10, const double* Pi, int mem_space);

/* Optional, for a bit-exact restart: overwrite u^{n-1} (otherwise equal to u^n after vh_set_initial).                  */
int vh_set_uprev(vh_handle* h, const double* u4_prev, int mem_space);

/* Bit-exact restart from a state exported by vh_get_fields: installs q, e, u^n, u^{n-1} as they are (p = P0(e) is
 * recomputed, ghost cells refilled), sets the step counter so that tau = tau0 + n_steps_done*dtau, resets the status counters.
 * (vh_set_initial cannot do this: it rebuilds T^{tau mu} from the primitives, and pi^{mu nu} is regulated AFTER the
 * inversion - program-flow steps 2-3 - so (e, u, pi, Pi) no longer reproduce the stored T^{tau mu} exactly.)               */
int vh_set_state(vh_handle* h, const double* q15, const double* e, const double* u4, const double* u4_prev, long long n_steps_done,
                 int mem_space);

/* Advance n_steps full RK2 steps (program-flow steps 1-9, :503-529).  Asynchronous on the handle's stream.             */
int vh_step(vh_handle* h, int n_steps);

/* Slab decomposition along eta (8(f) NEXT-4; the paper's own multi-GPU outlook is independent events, :899).  A caller that owns
 * one eta-slab of a larger grid takes the RK2 step in four parts and exchanges boundary planes with the owners of the neighbouring slabs
 * in between (paper_1608_06577_b200/vh.py: SlabSolver does this with torch.distributed send / recv, NCCL over NVLink between GPUs):
 *   part 0: velocity kernel of stage 1     -> exchange what = 0 (the state velocity of the eta direction at the slab faces, one plane)
 *   part 1: stage kernel of stage 1        -> exchange what = 1 (the new state q*, e*, p*, u*: two planes x 21 arrays per face)
 *   part 2: velocity kernel of stage 2     -> exchange what = 0
 *   part 3: stage kernel of stage 2, buffer rotation, step counter -> exchange what = 1
 * (and one exchange of what = 1 after vh_set_initial / vh_set_state).  vh_halo_export copies the slab's outermost PHYSICAL planes at a face
 * (side 0: low eta, 1: high eta) into buf; vh_halo_import writes buf into the GHOST planes beyond that face, replacing the outflow copies
 * (Eqs. 75-76) the kernels put there - a face without a neighbour simply keeps them.  buf: DEVICE memory of vh_halo_size doubles (whole
 * padded planes, always double).  Asynchronous on the handle's stream.  Default pipeline, 3+1d, n_batch = 1 only (VH_ERR_STATE otherwise);
 * the result is bit-identical to a single handle over the whole grid, and the failure counters of the slabs add up to the single handle's: a
 * face that has received a vh_halo_import has a neighbour (until the next vh_set_initial / vh_set_state), which counts the interface states on
 * its side.  Between part 0 and part 3 of a step only vh_step_part, the halo calls and the read-only getters are allowed: vh_step,
 * vh_step_profile, vh_run_until and vh_set_kernel_variant return VH_ERR_STATE.                                                              */
int vh_step_part(vh_handle* h, int part);
int vh_halo_size(vh_handle* h, int what, long long* n_doubles);
int vh_halo_export(vh_handle* h, int what, int side, double* buf_device);
int vh_halo_import(vh_handle* h, int what, int side, const double* buf_device);

/* Same as vh_step, but brackets each of the four launches of a step (default pipeline: velocity kernel 1, stage kernel 1,
 * velocity kernel 2, stage kernel 2; kernel variant 1: stage 1, ghost 1, stage 2, ghost 2) with CUDA events
 * on the handle's stream and returns their mean durations in milliseconds in ms4[0..3] (for per-kernel roofline numbers;
 * synchronises once per step, so use vh_step for throughput).                                                            */
int vh_step_profile(vh_handle* h, int n_steps, double* ms4);

/* Copy the state at the current tau to caller arrays; any of q15, e, p, u4, u4_prev may be NULL.  p is P0(e).          */
int vh_get_fields(vh_handle* h, double* q15, double* e, double* p, double* u4, double* u4_prev, int mem_space);

/* tau, number of steps done, number of failed Newton inversions (interface states and cells, both stages), number of
 * cells whose inversion produced a non-finite e or u^tau, smallest regularisation factor tanh(rho)/rho applied.
 * Any pointer may be NULL.  Synchronises the stream.                                                                   */
int vh_get_status(vh_handle* h, double* tau, long long* n_steps_done, long long* n_inversion_failures,
                  long long* n_nonfinite, double* min_reg_factor);

/* On-device diagnostics of the current state, maxima over all physical cells and events, written to
 * out10[0..9]:  [0] max T in fm^-1 (freeze-out test "T < T_f everywhere", program-flow step 8, :494);  [1] max |u.u - 1| (:489);
 * [2] max |g_{mu nu} pi^{mu nu}|/(e+p) and [3] max over lambda of |pi^{lambda mu} u_mu|/(e+p) (the constraints of Eqs. 47-51,
 * :318-331, which are propagated, not enforced; the lambda = eta entry is multiplied by tau);  [4] max R_pi^-1 =
 * sqrt(pi^{mu nu} pi_{mu nu})/P0 and [5] max R_Pi^-1 = |Pi|/P0 (inverse Reynolds numbers, Eq. 89, :826);  [6] max Kn = tau_pi |theta|
 * and [7] max tau_Pi |theta| (Knudsen numbers, :830; theta of A.11 with the finite differences of the source terms, :424, and the
 * relaxation times the solver uses; cells with 1/tau = 0 do not count; 0 if the sector is off);  [8] max (R_pi^(2))^-1 =
 * sqrt(J^{mu nu} J_{mu nu})/(2 eta sqrt(sigma^{mu nu} sigma_{mu nu})) and [9] max (R_Pi^(2))^-1 = |J|/(zeta |theta|), the second-order
 * inverse Reynolds numbers of Eq. 90 (:831) with J^{mu nu}, J of Eq. 5 at n^mu = 0, built from the terms I2, I3, I4 of Eqs. 41-46
 * and the kinematics of App. A exactly as the source terms build them (cells with 0/0 do not count; 0 if the sector is off).
 * One reduction kernel; synchronises the stream.  out10 is a HOST pointer to VH_N_DIAGNOSTICS = 10 doubles.               */
#define VH_N_DIAGNOSTICS 10
int vh_get_diagnostics(vh_handle* h, double* out10);

/* The same ten quantities cell by cell (the maps of the paper's Figs. 15-16, :826-834, are slices of [4]..[9]):
 * maps10[m * np + c], m = 0..9 as in vh_get_diagnostics, np = n_batch*nz*ny*nx, c = ((b*nz + k)*ny + j)*nx + i (physical cells,
 * the layout of vh_get_fields).  maps10 holds 10*np doubles in mem_space (0 host, 1 device; a host destination goes
 * through the library's device staging buffer, grown to that size).  One kernel; synchronises the stream.            */
int vh_get_diagnostic_maps(vh_handle* h, double* maps10, int mem_space);

/* Map of the regularisation strength (the paper's Fig. 17, :820): when enabled, the last stage of every time step also stores, per
 * cell, the factor tanh(rho)/rho of Eqs. 73-74 it applied to pi^{mu nu} and Pi (one extra 8-byte store per cell and step; one
 * more padded array of device memory).  Off by default.  vh_enable_regulation_map(h, 1) allocates the array and sets it to 1
 * (as does every later vh_set_initial); (h, 0) frees it.  vh_get_regulation_map copies it out: map[c] of n_batch*nz*ny*nx
 * doubles in the layout of vh_get_fields, mem_space 0 host / 1 device; VH_ERR_STATE if the map is not enabled.  In ideal mode
 * nothing is regularised and the map stays 1.                                                                             */
int vh_enable_regulation_map(vh_handle* h, int on);
int vh_get_regulation_map(vh_handle* h, double* map, int mem_space);

/* The ten diagnostics above for a caller that must not allocate device memory - no handle, no cudaMalloc, no cudaFree, no library
 * routine that allocates.  Who needs this: a host program that has already handed the GPU's free memory to an allocator of its own (a
 * framework's caching pool, a fixed arena sized at start-up), where a cudaMalloc made behind its back fails or eats into what the pool
 * thinks it owns; and a time loop that cannot afford the device-wide synchronisation a cudaMalloc / cudaFree implies.  vh_create and the
 * lazily allocated reduction slots and staging buffers of vh_get_diagnostics / vh_get_diagnostic_maps are out of reach for such callers;
 * this entry point works directly on the caller's own arrays instead.
 *
 * Inputs (all DEVICE pointers on the current device, the layout of vh_get_fields: physical cells only, x fastest, component-major):
 *   p        grid and physics as for vh_create (same checks; `storage` is ignored - the arrays below are the full set),
 *   tau      the time of the state (Milne geometry: tau > 0),
 *   q15, e, u4, u4_prev   15 + 1 + 4 + 4 arrays of np = n_batch*nz*ny*nx doubles (u4_prev = u at tau - dtau; pass u4 twice for an
 *            initial state).  The pressure is P0(e).  Differences across the edge of the grid use the outflow ghost cells of
 *            Eqs. 75-76 (:459-464), i.e. the value of the outermost physical cell, exactly as the solver's padded arrays hold them.
 * Outputs:
 *   out10    the ten maxima (order of vh_get_diagnostics); out_mem_space 0: HOST pointer, the call copies them out and synchronises the
 *            stream before returning; 1: DEVICE pointer, the call only enqueues work on cuda_stream,
 *   maps10   NULL, or a DEVICE pointer to 10*np doubles that receives the ten quantities cell by cell (layout of vh_get_diagnostic_maps).
 * Results agree with vh_get_diagnostics / vh_get_diagnostic_maps of a handle holding this state (the same per-cell arithmetic; tested to 1e-9).
 *
 * Scratch: one kernel; its per-block maxima, the ticket that tells the last block to combine them, and the EOS-2 table live in arrays
 * compiled into the library (`static __device__`, about 390 KB in total), which every GPU that loads the library holds until the
 * process exits.  The price is a size limit: np <= VH_NOALLOC_MAX_CELLS (2^20, e.g. 128 x 128 x 64 or 100^3); a larger grid is refused
 * with VH_ERR_ARG and a message naming both numbers - use a handle and vh_get_diagnostics for it.
 * First call on a device: looks up the device addresses of those arrays and uploads the EOS-2 table (host work plus one stream
 * synchronisation, once per device and process).  Make that first call during start-up, and before any stream capture is begun.
 * Every call on a device shares the same scratch and finds in it what the previous call left; the call clears the ticket itself (an
 * asynchronous 4-byte memset on cuda_stream), nothing else has to start from zero.  Two calls whose kernels can overlap on one GPU
 * (different streams, or different host threads on different streams) race on the scratch and give wrong maxima: issue them on one
 * stream or order them with events.  Runs on the CURRENT device; cuda_stream (NULL = default stream) must belong to it.               */
#define VH_NOALLOC_MAX_CELLS 1048576
int vh_diagnostics_noalloc(const vh_params* p, double tau, const double* q15, const double* e, const double* u4, const double* u4_prev,
                           double* out10, int out_mem_space, double* maps10, void* cuda_stream);

/* Program-flow steps 6-8 (:492-494): advance until T < T_f (fm^-1) everywhere or max_steps steps have been taken, testing the
 * temperature every check_every steps (>= 1) with the reduction of vh_get_diagnostics.  *steps_done (may be NULL) receives the
 * number of steps taken by this call; returns VH_OK in both cases (compare vh_get_diagnostics()[0] with T_f to tell them apart). */
int vh_run_until(vh_handle* h, double T_f, int max_steps, int check_every, long long* steps_done);

/* The table of EOS 2 as the library builds it on the host (no CUDA call; for inspection and for the CPU-side test that compares it
 * with the independently built table of the test oracle): VH_EOS_TABLE_NODES = 2049 nodes uniform in x = e^{1/4}, node k at
 * x0 + k h holding (P, h dP/dx, T, h dT/dx) in nodes4[4k .. 4k+3] (fm^-4, fm^-1; R19, R20).  nodes4 must hold
 * 4 * 2049 doubles (host pointer); x0, h may be NULL.                                                                      */
#define VH_EOS_TABLE_NODES 2049
int vh_eos_table(double* nodes4, double* x0, double* h);

/* Number of kernels launched on the handle since vh_create (for bench.py's gpu_launches).                             */
long long vh_launch_count(vh_handle* h);

/* Select the stage-kernel implementation: 0 = default (best available), other values select alternatives for A/B
 * measurements.  Returns VH_ERR_ARG for an unknown variant.                                   */
int vh_set_kernel_variant(vh_handle* h, int variant);

/* Device peaks measured with this library's own microbenchmarks on the handle's device and stream:
 * FP64 stream copy (GB/s, read+write bytes) over n_bytes (>= 1 GiB recommended) and a dependent-free FP64 FMA kernel
 * (GFLOP/s, 2 flops per FMA) on all SMs; each the best of `repeats`.  Either output may be NULL.                       */
int vh_measure_peaks(void* cuda_stream, long long n_bytes, int repeats, double* copy_gbs, double* fp64_gflops);
/* The same dependent-free FMA kernel in single precision (GFLOP/s): the ALU roofline denominator of the single-precision build
 * (libvh_f32.so).                                                                                     */
int vh_measure_fp32_peak(void* cuda_stream, int repeats, double* fp32_gflops);

const char* vh_last_error(vh_handle* h);
void vh_destroy(vh_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* VH_H_ */
