"""TEST INFRASTRUCTURE ONLY: ctypes binding of the serial CPU oracle (oracle/vh_oracle.hpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this
module.  It shares no code with the CUDA path (paper_1608_06577_b200/) and neither imports the other.
Parameters arrive as a plain dict (see paper_1608_06577_b200/inputs.py, which holds no arithmetic of the method).
"""
import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)
import build as _build  # noqa: E402  (oracle/build.py)


class Params(C.Structure):
    # mirrors vho::Params field by field
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


def make_params(d: dict) -> Params:
    p = Params()
    names = [f[0] for f in Params._fields_]
    for k in names:
        if k not in d:
            raise KeyError("missing parameter %r" % k)
        setattr(p, k, d[k])
    return p


_lib = None


def lib():
    global _lib
    if _lib is None:
        so = _build.build()
        L = C.CDLL(so)
        L.vho_create.restype = C.c_void_p
        L.vho_create.argtypes = [C.POINTER(Params)]
        L.vho_create_f32.restype = C.c_void_p
        L.vho_create_f32.argtypes = [C.POINTER(Params)]
        L.vho_destroy.argtypes = [C.c_void_p]
        dp = C.POINTER(C.c_double)
        L.vho_set_initial.argtypes = [C.c_void_p, dp, dp, dp, dp]
        L.vho_set_uprev.argtypes = [C.c_void_p, dp]
        L.vho_step.argtypes = [C.c_void_p, C.c_int]
        L.vho_get_fields.argtypes = [C.c_void_p, dp, dp, dp, dp, dp]
        L.vho_get_status.argtypes = [C.c_void_p, dp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong), C.POINTER(C.c_longlong), dp]
        L.vho_last_failure.argtypes = [C.c_void_p, C.c_int, dp]
        L.vho_diagnostics.argtypes = [C.c_void_p, dp]
        L.vho_diagnostic_maps.argtypes = [C.c_void_p, dp]
        L.vho_regulation_map.argtypes = [C.c_void_p, dp]
        L.vho_raw.restype = dp
        L.vho_raw.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.vho_set_tau.argtypes = [C.c_void_p, C.c_double]
        L.vho_sources_at.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, dp]
        L.vho_flux_at.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, dp]
        L.vho_post.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.vho_ghost.argtypes = [C.c_void_p, C.c_int]
        L.vho_minmod3.restype = C.c_double
        L.vho_minmod3.argtypes = [C.c_double] * 3
        L.vho_eos.argtypes = [C.POINTER(Params), C.c_double, dp]
        L.vho_transport.argtypes = [C.POINTER(Params), C.c_double, dp]
        L.vho_invert.restype = C.c_double
        L.vho_invert.argtypes = [C.POINTER(Params), C.c_double, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.vho_count_ops.argtypes = [C.POINTER(Params), dp, dp, dp, dp, C.c_int, C.c_int, C.POINTER(C.c_longlong)]
        L.vho_time_steps.restype = C.c_double
        L.vho_time_steps.argtypes = [C.c_void_p, C.c_int]
        assert L.vho_params_size() == C.sizeof(Params), "Params layout mismatch"
        _lib = L
    return _lib


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


WHICH = {"q": 0, "qS": 1, "Q": 2, "u": 3, "up": 4, "uS": 5, "e": 6, "p": 7}


class Oracle:
    """One oracle run.  Arrays: physical cells only, shape [..., n_batch, nz, ny, nx] (x fastest)."""

    def __init__(self, params: dict, precision="f64"):
        """precision "f32": the same algorithm with a float scalar (set_initial / set_uprev / step / get_fields / status only)."""
        self.L = lib()
        self.d = dict(params)
        self.P = make_params(params)
        self.precision = precision
        self.h = (self.L.vho_create_f32 if precision == "f32" else self.L.vho_create)(C.byref(self.P))
        if not self.h:
            raise ValueError("vho_create rejected the parameters")
        self.shape = (self.P.n_batch, self.P.nz, self.P.ny, self.P.nx)
        self.padded = (self.P.nz + 4, self.P.ny + 4, self.P.nx + 4)

    def __del__(self):
        if getattr(self, "h", None):
            self.L.vho_destroy(self.h)
            self.h = None

    def set_initial(self, e, u4, pi10=None, Pi=None):
        e = np.ascontiguousarray(e, dtype=np.float64).reshape(self.shape)
        u4 = np.ascontiguousarray(u4, dtype=np.float64).reshape((4,) + self.shape)
        pi10 = None if pi10 is None else np.ascontiguousarray(pi10, dtype=np.float64).reshape((10,) + self.shape)
        Pi = None if Pi is None else np.ascontiguousarray(Pi, dtype=np.float64).reshape(self.shape)
        self.L.vho_set_initial(self.h, _dp(e), _dp(u4), _dp(pi10), _dp(Pi))

    def set_uprev(self, up4):
        up4 = np.ascontiguousarray(up4, dtype=np.float64).reshape((4,) + self.shape)
        self.L.vho_set_uprev(self.h, _dp(up4))

    def step(self, n=1):
        self.L.vho_step(self.h, int(n))

    def time_steps(self, n):
        return self.L.vho_time_steps(self.h, int(n))

    def get_fields(self, with_uprev=False):
        q = np.empty((15,) + self.shape)
        e = np.empty(self.shape)
        p = np.empty(self.shape)
        u = np.empty((4,) + self.shape)
        up = np.empty((4,) + self.shape) if with_uprev else None
        self.L.vho_get_fields(self.h, _dp(q), _dp(e), _dp(p), _dp(u), _dp(up))
        out = {"q": q, "e": e, "p": p, "u": u}
        if with_uprev:
            out["up"] = up
        return out

    def status(self):
        tau = C.c_double()
        mr = C.c_double()
        a, b, c = C.c_longlong(), C.c_longlong(), C.c_longlong()
        self.L.vho_get_status(self.h, C.byref(tau), C.byref(a), C.byref(b), C.byref(c), C.byref(mr))
        return {"tau": tau.value, "n_steps": a.value, "n_inversion_failures": b.value, "n_nonfinite": c.value, "min_reg_factor": mr.value}

    def diagnostics(self):
        out = np.empty(10)
        self.L.vho_diagnostics(self.h, _dp(out))
        return dict(zip(DIAG_NAMES, out))

    def diagnostic_maps(self):
        out = np.empty((10,) + self.shape)
        self.L.vho_diagnostic_maps(self.h, _dp(out))
        return out

    def regulation_map(self):
        out = np.empty(self.shape)
        self.L.vho_regulation_map(self.h, _dp(out))
        return out

    def last_failure(self, ev=0):
        out = np.empty(4)
        self.L.vho_last_failure(self.h, ev, _dp(out))
        return dict(zip(['E', 'M2', 'Pi', 'guess'], out))

    # ---- unit-pin access
    def raw(self, which, comp=0, ev=0):
        """numpy view (padded, [NZ,NY,NX]) of an internal array."""
        ptr = self.L.vho_raw(self.h, ev, WHICH[which], comp)
        n = self.padded[0] * self.padded[1] * self.padded[2]
        return np.ctypeslib.as_array(ptr, shape=(n,)).reshape(self.padded)

    def set_tau(self, tau):
        self.L.vho_set_tau(self.h, float(tau))

    def sources_at(self, i, j, k, tau, ev=0):
        J = np.empty(15)
        self.L.vho_sources_at(self.h, ev, i, j, k, float(tau), _dp(J))
        return J

    def flux_at(self, i, j, k, r, upper, tau, ev=0):
        H = np.empty(15)
        self.L.vho_flux_at(self.h, ev, i, j, k, r, int(upper), float(tau), _dp(H))
        return H

    def post(self, tau, ev=0):
        self.L.vho_post(self.h, ev, float(tau))

    def ghost(self, ev=0):
        self.L.vho_ghost(self.h, ev)


def minmod3(x, y, z):
    return lib().vho_minmod3(x, y, z)


def eos(params: dict, e: float):
    out = np.empty(3)
    P = make_params(params)
    lib().vho_eos(C.byref(P), float(e), _dp(out))
    return {"p": out[0], "cs2": out[1], "T": out[2]}


def transport(params: dict, e: float):
    out = np.empty(5)
    P = make_params(params)
    lib().vho_transport(C.byref(P), float(e), _dp(out))
    return dict(zip(["inv_tau_pi", "eta_over_tau_pi", "inv_tau_Pi", "zeta_over_tau_Pi", "lambda_Pipi_over_tau_Pi"], out))


def invert(params: dict, E, M2, Pi, guess):
    P = make_params(params)
    it, fl = C.c_int(), C.c_int()
    e = lib().vho_invert(C.byref(P), float(E), float(M2), float(Pi), float(guess), C.byref(it), C.byref(fl))
    return e, it.value, fl.value


DIAG_NAMES = ("max_T", "max_norm_violation", "max_trace_violation", "max_transversality_violation", "max_inv_reynolds_shear", "max_inv_reynolds_bulk",
              "max_knudsen_shear", "max_knudsen_bulk", "max_inv_reynolds2_shear", "max_inv_reynolds2_bulk")
OP_CLASSES = ("add", "mul", "div", "cmp", "sqrt", "exp", "pow", "tanh")
# flop weights of SURVEY.md 8(d): add/mul 1, div 10, sqrt 15, exp 25, tanh 40; pow(x, 1/4) = two sqrt.  Compares carry NO flop weight
# (a select is not floating-point work; they are reported as their own class).
OP_WEIGHTS = dict(add=1, mul=1, div=10, cmp=0, sqrt=15, exp=25, pow=30, tanh=40)
SECTIONS = ("other", "flux", "invert", "slopes")
# how often the oracle evaluates the same thing: each interface from both adjacent cells (Alg. 2), each limited slope four times
# (as the slope of "this" cell and of "the next" cell, for the upper and the lower interface)
REPEATS = dict(other=1, flux=2, invert=2, slopes=4)


def count_ops(params: dict, e, u4, pi10=None, Pi=None, warm=1, n=1):
    """Operation counts of n RK2 steps with the counting scalar (after `warm` uncounted steps), summed over all cells, per section
    of the oracle: `slopes` = Eq. 67 inside flux(), `flux` = half-cell extrapolation and Eq. 61, `invert` = the interface-state
    inversions inside flux(), `other` = sources, stage update, cell inversion, regularisation."""
    P = make_params(params)
    shape = (P.n_batch, P.nz, P.ny, P.nx)
    e = np.ascontiguousarray(e, dtype=np.float64).reshape(shape)
    u4 = np.ascontiguousarray(u4, dtype=np.float64).reshape((4,) + shape)
    pi10 = None if pi10 is None else np.ascontiguousarray(pi10, dtype=np.float64).reshape((10,) + shape)
    Pi = None if Pi is None else np.ascontiguousarray(Pi, dtype=np.float64).reshape(shape)
    out = (C.c_longlong * 32)()
    rc = lib().vho_count_ops(C.byref(P), _dp(e), _dp(u4), _dp(pi10), _dp(Pi), int(warm), int(n), out)
    if rc < 0:
        raise ValueError("vho_count_ops needs n_batch == 1")
    vals = list(out)
    return {sec: dict(zip(OP_CLASSES, vals[8 * i:8 * i + 8])) for i, sec in enumerate(SECTIONS)}


def algorithmic_flops_per_cell_update(params: dict, e, u4, pi10=None, Pi=None):
    """MINIMAL algorithmic flops per cell per RK2 step: every section divided by the number of times the oracle repeats it
    (REPEATS), compares excluded, exact 0 / +-1 constants not counted.  Returns (flops, per-class counts incl. 'cmp',
    flops per section)."""
    c = count_ops(params, e, u4, pi10, Pi, warm=1, n=1)
    ncell = params["nx"] * params["ny"] * params["nz"]
    per = {k: sum(c[sec][k] / REPEATS[sec] for sec in SECTIONS) / ncell for k in OP_CLASSES}
    by_section = {sec: sum(OP_WEIGHTS[k] * c[sec][k] for k in OP_CLASSES) / REPEATS[sec] / ncell for sec in SECTIONS}
    flops = sum(by_section.values())
    return flops, per, by_section
