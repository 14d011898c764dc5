"""Thin Python binding of the C ABI in include/vh.h (argument marshalling only; every step runs in the CUDA kernels).

torch is used for device memory (the arrays handed to / returned from the library) and for the CUDA stream.
There is no CPU fallback: if libvh.so is missing or no CUDA device is present, construction raises."""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(HERE, "libvh.so")
# the same sources compiled with real = float (the paper ran single precision): same C ABI, caller arrays stay double
LIBS = {"f64": SO, "f32": os.path.join(HERE, "libvh_f32.so")}

VH_OK = 0


class vh_params(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("n_batch", C.c_int),
        ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
        ("tau0", C.c_double), ("dtau", C.c_double),
        ("geometry", C.c_int), ("physics", C.c_int), ("eos", C.c_int),
        ("eos_a", C.c_double), ("eos_alpha", C.c_double), ("eos_e0", C.c_double),
        ("eta_over_s", C.c_double),
        ("zeta_model", C.c_int), ("zeta_amp", C.c_double), ("zeta_T0", C.c_double), ("zeta_width", C.c_double),
        ("c_tau_pi", C.c_double), ("c_tau_Pi", C.c_double),
        ("delta_pipi", C.c_double), ("tau_pipi", C.c_double), ("lambda_piPi", C.c_double),
        ("delta_PiPi", C.c_double), ("lambda_Pipi_coef", C.c_double),
        ("minmod_theta", C.c_double), ("xi0", C.c_double), ("rho_max", C.c_double),
        ("newton_max_iter", C.c_int), ("newton_rtol", C.c_double),
        ("tau_relax_floor_over_dtau", C.c_double),
        ("storage", C.c_int),
    ]


# every symbol include/vh.h declares
EXPORTS = ["vh_create", "vh_set_initial", "vh_set_state", "vh_set_uprev", "vh_step", "vh_step_part", "vh_halo_size", "vh_halo_export", "vh_halo_import", "vh_step_profile", "vh_get_fields", "vh_get_status", "vh_get_diagnostics", "vh_get_diagnostic_maps", "vh_diagnostics_noalloc", "vh_enable_regulation_map", "vh_get_regulation_map", "vh_run_until", "vh_eos_table", "vh_launch_count",
           "vh_set_kernel_variant", "vh_measure_peaks", "vh_measure_fp32_peak", "vh_last_error", "vh_destroy"]

_lib = None


def load_library(precision="f64"):
    """dlopen libvh.so (precision "f64") or libvh_f32.so ("f32") and declare the prototypes.  Works without a GPU (no CUDA call is made)."""
    global _lib
    if _lib is None:
        _lib = {}
    if precision in _lib:
        return _lib[precision]
    so = LIBS[precision]
    if not os.path.exists(so):
        raise RuntimeError("CUDA extension %s is missing: run `python -m paper_1608_06577_b200.build` (there is no CPU fallback)" % so)
    L = C.CDLL(so)
    vp = C.c_void_p
    for name in EXPORTS:
        getattr(L, name).restype = C.c_int
    L.vh_create.argtypes = [C.POINTER(vh_params), vp, C.POINTER(vp)]
    L.vh_set_initial.argtypes = [vp, vp, vp, vp, vp, C.c_int]
    L.vh_set_uprev.argtypes = [vp, vp, C.c_int]
    L.vh_set_state.argtypes = [vp, vp, vp, vp, vp, C.c_longlong, C.c_int]
    L.vh_step.argtypes = [vp, C.c_int]
    L.vh_step_part.argtypes = [vp, C.c_int]
    L.vh_halo_size.argtypes = [vp, C.c_int, C.POINTER(C.c_longlong)]
    L.vh_halo_export.argtypes = [vp, C.c_int, C.c_int, vp]
    L.vh_halo_import.argtypes = [vp, C.c_int, C.c_int, vp]
    L.vh_step_profile.argtypes = [vp, C.c_int, C.POINTER(C.c_double)]
    L.vh_get_fields.argtypes = [vp, vp, vp, vp, vp, vp, C.c_int]
    L.vh_get_status.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong), C.POINTER(C.c_longlong), C.POINTER(C.c_longlong), C.POINTER(C.c_double)]
    L.vh_get_diagnostics.argtypes = [vp, C.POINTER(C.c_double)]
    L.vh_get_diagnostic_maps.argtypes = [vp, vp, C.c_int]
    L.vh_diagnostics_noalloc.argtypes = [C.POINTER(vh_params), C.c_double, vp, vp, vp, vp, vp, C.c_int, vp, vp]
    L.vh_enable_regulation_map.argtypes = [vp, C.c_int]
    L.vh_get_regulation_map.argtypes = [vp, vp, C.c_int]
    L.vh_run_until.argtypes = [vp, C.c_double, C.c_int, C.c_int, C.POINTER(C.c_longlong)]
    L.vh_eos_table.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.vh_launch_count.argtypes = [vp]
    L.vh_launch_count.restype = C.c_longlong
    L.vh_set_kernel_variant.argtypes = [vp, C.c_int]
    L.vh_measure_peaks.argtypes = [vp, C.c_longlong, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.vh_measure_fp32_peak.argtypes = [vp, C.c_int, C.POINTER(C.c_double)]
    L.vh_last_error.argtypes = [vp]
    L.vh_last_error.restype = C.c_char_p
    L.vh_destroy.argtypes = [vp]
    L.vh_destroy.restype = None
    _lib[precision] = L
    return L


def make_params(d: dict) -> vh_params:
    p = vh_params()
    for name, _ in vh_params._fields_:
        if name not in d:
            raise KeyError("missing parameter %r" % name)
        setattr(p, name, d[name])
    return p


class VHError(RuntimeError):
    pass


def _ptr(t):
    if t is None:
        return None
    return C.c_void_p(t.data_ptr())


class Solver:
    """vh_create / vh_set_initial / vh_step / vh_get_fields on one GPU.

    Arrays are torch tensors (float64) of shape [..., n_batch, nz, ny, nx]: CUDA tensors are passed as device pointers
    (mem_space 1), CPU tensors as host pointers (mem_space 0; the library does the copies on its stream)."""

    def __init__(self, params: dict, device="cuda:0", stream=None, precision="f64"):
        import torch

        self.torch = torch
        self.precision = precision
        self.L = load_library(precision)
        if not torch.cuda.is_available():
            raise VHError("no CUDA device available (there is no CPU fallback)")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.d = dict(params)
        self.P = make_params(params)
        self.h = C.c_void_p()
        rc = self.L.vh_create(C.byref(self.P), C.c_void_p(self.stream.cuda_stream), C.byref(self.h))
        if rc != VH_OK:
            msg = self.L.vh_last_error(None)
            self.h = None
            raise VHError("vh_create failed (%d): %s" % (rc, msg.decode() if msg else "?"))
        self.shape = (self.P.n_batch, self.P.nz, self.P.ny, self.P.nx)
        self.variant = 0

    def close(self):
        if getattr(self, "h", None):
            self.L.vh_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        if rc != VH_OK:
            msg = self.L.vh_last_error(self.h)
            raise VHError("%s failed (%d): %s" % (what, rc, msg.decode() if msg else "?"))

    def _prep(self, a, lead):
        torch = self.torch
        if a is None:
            return None
        if not isinstance(a, torch.Tensor):
            a = torch.as_tensor(a, dtype=torch.float64)
        a = a.to(torch.float64).contiguous()
        want = 1
        for s in lead + self.shape:
            want *= s
        if a.numel() != want:
            raise ValueError("array has %d elements, expected %d" % (a.numel(), want))
        return a

    def _space(self, tensors):
        spaces = {t.is_cuda for t in tensors if t is not None}
        if len(spaces) != 1:
            raise ValueError("all arrays of one call must live in the same memory space")
        return 1 if spaces.pop() else 0

    def set_initial(self, e, u4, pi10=None, Pi=None):
        e = self._prep(e, ()); u4 = self._prep(u4, (4,)); pi10 = self._prep(pi10, (10,)); Pi = self._prep(Pi, ())
        ms = self._space([e, u4, pi10, Pi])
        self._check(self.L.vh_set_initial(self.h, _ptr(e), _ptr(u4), _ptr(pi10), _ptr(Pi), ms), "vh_set_initial")
        if ms == 1:
            self.stream.synchronize()      # the caller may free its tensors on return

    def set_state(self, q15, e, u4, u4_prev, n_steps_done=0):
        q15 = self._prep(q15, (15,)); e = self._prep(e, ()); u4 = self._prep(u4, (4,)); u4_prev = self._prep(u4_prev, (4,))
        ms = self._space([q15, e, u4, u4_prev])
        self._check(self.L.vh_set_state(self.h, _ptr(q15), _ptr(e), _ptr(u4), _ptr(u4_prev), int(n_steps_done), ms), "vh_set_state")
        self.stream.synchronize()

    def set_uprev(self, u4_prev):
        a = self._prep(u4_prev, (4,))
        ms = self._space([a])
        self._check(self.L.vh_set_uprev(self.h, _ptr(a), ms), "vh_set_uprev")
        if ms == 1:
            self.stream.synchronize()

    def step(self, n=1):
        self._check(self.L.vh_step(self.h, int(n)), "vh_step")

    def step_part(self, part):
        self._check(self.L.vh_step_part(self.h, int(part)), "vh_step_part")

    def halo_size(self, what):
        n = C.c_longlong()
        self._check(self.L.vh_halo_size(self.h, int(what), C.byref(n)), "vh_halo_size")
        return n.value

    def halo_export(self, what, side, buf):
        self._check(self.L.vh_halo_export(self.h, int(what), int(side), _ptr(buf)), "vh_halo_export")

    def halo_import(self, what, side, buf):
        self._check(self.L.vh_halo_import(self.h, int(what), int(side), _ptr(buf)), "vh_halo_import")

    def step_profile(self, n=1):
        """n steps with CUDA events around each of the four launches of a step; mean ms per launch, keyed by kernel:
        variants 0, 2: velocity1, stage1, velocity2, stage2; variant 1 and reduced storage: stage1, ghost1, stage2, ghost2."""
        ms = (C.c_double * 4)()
        self._check(self.L.vh_step_profile(self.h, int(n), ms), "vh_step_profile")
        names = ("stage1", "ghost1", "stage2", "ghost2") if (self.variant == 1 or self.d.get("storage", 0) == 1) else ("velocity1", "stage1", "velocity2", "stage2")
        return dict(zip(names, list(ms)))

    def get_fields(self, device=None, with_uprev=False, out=None):
        """Returns dict(q [15,...], e, p, u [4,...]) as tensors on `device` ('cpu' -> host buffers, mem_space 0)."""
        torch = self.torch
        dev = self.device if device is None else torch.device(device)
        if out is None:
            kw = dict(dtype=torch.float64, device=dev)
            if dev.type == "cpu":
                kw["pin_memory"] = True
            out = dict(q=torch.empty((15,) + self.shape, **kw), e=torch.empty(self.shape, **kw), p=torch.empty(self.shape, **kw),
                       u=torch.empty((4,) + self.shape, **kw))
            if with_uprev:
                out["up"] = torch.empty((4,) + self.shape, **kw)
        ms = self._space([v for v in out.values()])
        self._check(self.L.vh_get_fields(self.h, _ptr(out.get("q")), _ptr(out.get("e")), _ptr(out.get("p")), _ptr(out.get("u")),
                                         _ptr(out.get("up")), ms), "vh_get_fields")
        return out

    def status(self):
        tau, mr = C.c_double(), C.c_double()
        a, b, c = C.c_longlong(), C.c_longlong(), C.c_longlong()
        self._check(self.L.vh_get_status(self.h, C.byref(tau), C.byref(a), C.byref(b), C.byref(c), C.byref(mr)), "vh_get_status")
        return {"tau": tau.value, "n_steps": a.value, "n_inversion_failures": b.value, "n_nonfinite": c.value, "min_reg_factor": mr.value}

    DIAG_NAMES = ("max_T", "max_norm_violation", "max_trace_violation", "max_transversality_violation", "max_inv_reynolds_shear",
                  "max_inv_reynolds_bulk", "max_knudsen_shear", "max_knudsen_bulk", "max_inv_reynolds2_shear", "max_inv_reynolds2_bulk")

    def diagnostics(self):
        out = (C.c_double * 10)()
        self._check(self.L.vh_get_diagnostics(self.h, out), "vh_get_diagnostics")
        return dict(zip(self.DIAG_NAMES, list(out)))

    def diagnostic_maps(self, device=None):
        """The ten quantities of diagnostics() cell by cell: tensor [10, n_batch, nz, ny, nx] (order of DIAG_NAMES, without 'max_')."""
        torch = self.torch
        dev = self.device if device is None else torch.device(device)
        out = torch.empty((10,) + self.shape, dtype=torch.float64, device=dev)
        self._check(self.L.vh_get_diagnostic_maps(self.h, _ptr(out), self._space([out])), "vh_get_diagnostic_maps")
        return out

    def enable_regulation_map(self, on=True):
        self._check(self.L.vh_enable_regulation_map(self.h, 1 if on else 0), "vh_enable_regulation_map")

    def regulation_map(self, device=None):
        """tanh(rho)/rho applied by the last step's final regularisation, per cell (Fig. 17): tensor [n_batch, nz, ny, nx]."""
        torch = self.torch
        dev = self.device if device is None else torch.device(device)
        out = torch.empty(self.shape, dtype=torch.float64, device=dev)
        self._check(self.L.vh_get_regulation_map(self.h, _ptr(out), self._space([out])), "vh_get_regulation_map")
        return out

    def run_until(self, T_f, max_steps, check_every=10):
        """Advance until T < T_f everywhere or max_steps steps (PAPER.md :494); returns the number of steps taken."""
        done = C.c_longlong()
        self._check(self.L.vh_run_until(self.h, float(T_f), int(max_steps), int(check_every), C.byref(done)), "vh_run_until")
        return done.value

    def launch_count(self):
        return int(self.L.vh_launch_count(self.h))

    def set_kernel_variant(self, v):
        self._check(self.L.vh_set_kernel_variant(self.h, int(v)), "vh_set_kernel_variant")
        self.variant = int(v)


NOALLOC_MAX_CELLS = 1 << 20      # VH_NOALLOC_MAX_CELLS of include/vh.h


def diagnostics_noalloc(params: dict, tau, q15, e, u4, u4_prev, maps=None, stream=None, precision="f64"):
    """vh_diagnostics_noalloc: the ten diagnostics of Solver.diagnostics() computed straight from CUDA tensors the caller already holds,
    for programs that must not let the library allocate device memory (their own pool owns the GPU's memory, or a cudaMalloc stall is
    not acceptable where they call this).  No Solver is involved; the library's fixed scratch array limits the grid to NOALLOC_MAX_CELLS
    cells.  q15 [15, ...], e [...], u4 / u4_prev [4, ...]: contiguous float64 CUDA tensors on the current device, shape [..., n_batch, nz, ny, nx];
    maps: None or a float64 CUDA tensor of 10 * cells elements that receives the per-cell values.  Returns the dict of ten maxima
    (the call synchronises `stream`).  Marshalling only - this function itself creates no tensor.  Calls on different streams must not
    overlap (they share the scratch), and the first call on a device does a one-time set-up: make it before capturing a stream."""
    import torch

    L = load_library(precision)
    if not torch.cuda.is_available():
        raise VHError("no CUDA device available (there is no CPU fallback)")
    P = make_params(params)
    np_ = P.nx * P.ny * P.nz * P.n_batch
    for name, a, lead in (("q15", q15, 15), ("e", e, 1), ("u4", u4, 4), ("u4_prev", u4_prev, 4), ("maps", maps, 10)):
        if a is None and name == "maps":
            continue
        if not (isinstance(a, torch.Tensor) and a.is_cuda and a.dtype == torch.float64 and a.is_contiguous() and a.numel() == lead * np_):
            raise ValueError("%s must be a contiguous float64 CUDA tensor of %d elements" % (name, lead * np_))
    st = stream if stream is not None else torch.cuda.current_stream()
    out = (C.c_double * 10)()
    rc = L.vh_diagnostics_noalloc(C.byref(P), float(tau), _ptr(q15), _ptr(e), _ptr(u4), _ptr(u4_prev), C.cast(out, C.c_void_p), 0, _ptr(maps),
                                  C.c_void_p(st.cuda_stream))
    if rc != VH_OK:
        msg = L.vh_last_error(None)
        raise VHError("vh_diagnostics_noalloc failed (%d): %s" % (rc, msg.decode() if msg else "?"))
    return dict(zip(Solver.DIAG_NAMES, list(out)))


def eos_table():
    """(nodes [2049, 4] = (P, h dP/dx, T, h dT/dx), x0, h) of EOS 2 as the library builds it on the host (no GPU needed)."""
    import numpy as np

    L = load_library()
    nodes = np.empty((2049, 4))
    x0, h = C.c_double(), C.c_double()
    rc = L.vh_eos_table(nodes.ctypes.data_as(C.POINTER(C.c_double)), C.byref(x0), C.byref(h))
    if rc != VH_OK:
        raise VHError("vh_eos_table failed (%d)" % rc)
    return nodes, x0.value, h.value


def measure_peaks(n_bytes=1 << 30, repeats=10, stream=None):
    """(copy GB/s, FP64 FMA GFLOP/s) measured by the library's own microbenchmarks on the current device."""
    import torch

    L = load_library()
    if not torch.cuda.is_available():
        raise VHError("no CUDA device available")
    st = stream if stream is not None else torch.cuda.current_stream()
    a, b = C.c_double(), C.c_double()
    rc = L.vh_measure_peaks(C.c_void_p(st.cuda_stream), int(n_bytes), int(repeats), C.byref(a), C.byref(b))
    if rc != VH_OK:
        msg = L.vh_last_error(None)
        raise VHError("vh_measure_peaks failed (%d): %s" % (rc, msg.decode() if msg else "?"))
    return a.value, b.value


def measure_fp32_peak(repeats=10, stream=None):
    """FP32 FMA GFLOP/s of the current device (the ALU roofline denominator of the single-precision build)."""
    import torch

    L = load_library()
    if not torch.cuda.is_available():
        raise VHError("no CUDA device available")
    st = stream if stream is not None else torch.cuda.current_stream()
    a = C.c_double()
    rc = L.vh_measure_fp32_peak(C.c_void_p(st.cuda_stream), int(repeats), C.byref(a))
    if rc != VH_OK:
        msg = L.vh_last_error(None)
        raise VHError("vh_measure_fp32_peak failed (%d): %s" % (rc, msg.decode() if msg else "?"))
    return a.value


class SlabSolver:
    """One eta-slab of a larger 3+1d grid per rank of a torch.distributed group: rank r owns planes
    [r nz/W, (r+1) nz/W) and exchanges two boundary planes of the 21 state arrays (and one plane of state velocities) with its neighbours after
    every kernel of the step - neighbour send / recv.  With the NCCL backend the device buffers go to the backend as they are and the whole
    exchange is ordered on the solver's stream (export kernel -> send / recv -> import kernel; the host neither synchronises nor waits); with
    the gloo backend the planes are staged through host memory.  Argument marshalling and the exchange only: every step of the path runs in
    the library's kernels, and the result is bit-identical to a single Solver over the whole grid.
    Tested with gloo (two ranks sharing one GPU) and with several handles in one process; the NCCL path has NOT been run on more than one GPU
    (no multi-GPU box was available to this repository's tests).  device = None takes cuda:LOCAL_RANK."""

    def __init__(self, params: dict, group=None, device=None, precision="f64"):
        import torch
        import torch.distributed as dist

        self.torch, self.dist, self.group = torch, dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        nz = params["nz"]
        if nz % self.world or nz // self.world < 2:
            raise VHError("nz must be a multiple of the number of ranks with at least two planes per slab")
        self.nzl = nz // self.world
        self.z0 = self.rank * self.nzl
        local = dict(params, nz=self.nzl)
        if device is None:
            device = "cuda:%d" % int(os.environ.get("LOCAL_RANK", "0"))
        self.s = Solver(local, device=device, precision=precision)
        self.device = self.s.device
        self.host_staging = dist.get_backend(group) == "gloo"
        self.buf = {w: [[torch.empty(self.s.halo_size(w), dtype=torch.float64, device=self.device) for _ in range(2)] for _ in range(2)] for w in (0, 1)}
        self.lo = self.rank - 1 if self.rank > 0 else None
        self.hi = self.rank + 1 if self.rank + 1 < self.world else None

    def _slab(self, a):
        return None if a is None else a[..., self.z0:self.z0 + self.nzl, :, :].contiguous()

    def _exchange(self, what):
        """send my outermost physical planes at each face to the neighbour beyond it, receive its planes into my ghost planes.
        Everything is issued with the solver's stream as torch's current stream: NCCL orders its transfers after the work already on the
        current stream and `wait()` makes the current stream (not the host) wait for them, so export -> transfer -> import is a chain on
        the device; the host-staged copies of the gloo path are ordered by the same stream."""
        dist, torch = self.dist, self.torch
        with torch.cuda.stream(self.s.stream):
            ops, staged = [], []
            for side, nb in ((0, self.lo), (1, self.hi)):
                if nb is None:
                    continue
                out, inp = self.buf[what][side]
                self.s.halo_export(what, side, out)
                if self.host_staging:
                    out_h, inp_h = out.cpu(), torch.empty(inp.shape, dtype=inp.dtype)      # (.cpu() waits for the export on the current stream)
                    ops += [dist.P2POp(dist.isend, out_h, nb, self.group), dist.P2POp(dist.irecv, inp_h, nb, self.group)]
                    staged.append((side, inp, inp_h))
                else:
                    ops += [dist.P2POp(dist.isend, out, nb, self.group), dist.P2POp(dist.irecv, inp, nb, self.group)]
                    staged.append((side, inp, None))
            if ops:
                for r in dist.batch_isend_irecv(ops):
                    r.wait()      # gloo: the host waits for the planes; NCCL: the current stream does
            for side, inp, inp_h in staged:
                if inp_h is not None:
                    inp.copy_(inp_h)
                self.s.halo_import(what, side, inp)

    def set_initial(self, e, u4, pi10=None, Pi=None):
        """global arrays [..., nz, ny, nx]; every rank takes its own planes"""
        self.s.set_initial(self._slab(e), self._slab(u4), self._slab(pi10), self._slab(Pi))
        self._exchange(1)

    def set_uprev(self, u4_prev):
        self.s.set_uprev(self._slab(u4_prev))

    def step(self, n=1):
        for _ in range(int(n)):
            for part in range(4):
                self.s.step_part(part)
                self._exchange(part % 2)

    def get_fields(self, **kw):
        """this rank's slab"""
        return self.s.get_fields(**kw)

    def status(self):
        return self.s.status()

    def close(self):
        self.s.close()
