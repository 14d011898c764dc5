"""Single-precision build (libvh_f32.so, "all results in single precision").

Tolerance.  Both sides run the same algorithm with a 24-bit significand (eps = 6e-8): O(10^3) operations per cell-update whose flux
differences are divided by dr amplify rounding to ~1e-6 relative per step; the oracle's own float and double instantiations differ by
5e-6 after 10 steps of the generic state (measured on the CPU, test below).  The bar for GPU(f32) against either oracle instantiation is
therefore 1e-4 in the norm of DESIGN.md R18, written here; the FP64 build keeps 1e-9."""
import ctypes as C

import numpy as np
import pytest

from paper_1608_06577_b200 import inputs

TOL_F32 = 1e-4


def _generic(prm_over=None):
    prm = inputs.base_params(nx=36, ny=20, nz=10, dx=0.12, dy=0.1, dz=0.15, tau0=0.8, dtau=0.02, newton_rtol=2e-6, **(prm_over or {}))
    st = inputs.smooth_random_state(prm, seed=21)
    return prm, st


def test_f32_library_exports_the_same_abi():
    from paper_1608_06577_b200 import build, vh

    build.build()
    L = vh.load_library("f32")
    for n in vh.EXPORTS:
        assert hasattr(L, n), "libvh_f32.so does not export %s" % n
    # the stopping rule of Eq. 72 cannot be tighter than single precision: refused before any CUDA call
    p = vh.make_params(inputs.base_params(nx=4, ny=4, nz=4, newton_rtol=1e-13))
    h = C.c_void_p()
    assert L.vh_create(C.byref(p), None, C.byref(h)) == -1
    assert b"newton_rtol" in L.vh_last_error(None)


def test_oracle_float_instantiation_tracks_the_double_one(vo):
    prm, st = _generic()
    a, b = vo.Oracle(prm), vo.Oracle(prm, "f32")
    for o in (a, b):
        o.set_initial(st["e"], st["u"], st["pi"], st["Pi"])
        o.step(10)
    fa, fb = a.get_fields(), b.get_fields()
    S = np.max(np.abs(fa["q"][0]))
    worst = max(np.max(np.abs(fa["q"][n] - fb["q"][n])) / max(np.max(np.abs(fa["q"][n])), 1e-6 * S) for n in range(15))
    assert 1e-8 < worst < 3e-5                  # really single precision, and no worse than rounding explains
    assert b.status()["n_inversion_failures"] == 0


@pytest.mark.gpu
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_f32_gpu_parity_generic_state(vo, variant):
    import torch
    from paper_1608_06577_b200 import vh
    from test_gpu_parity import field_errors

    prm, st = _generic()
    t = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda:0")
    s = vh.Solver(prm, precision="f32")
    s.set_kernel_variant(variant)
    s.set_initial(t(st["e"]), t(st["u"]), t(st["pi"]), t(st["Pi"]))
    s.step(10)
    fg = {k: v.cpu().numpy() for k, v in s.get_fields(with_uprev=True).items()}
    sg = s.status()
    s.close()
    assert sg["n_inversion_failures"] == 0 and sg["n_nonfinite"] == 0
    for prec in ("f64", "f32"):
        o = vo.Oracle(prm, prec)
        o.set_initial(st["e"], st["u"], st["pi"], st["Pi"])
        o.step(10)
        errs = field_errors(o.get_fields(with_uprev=True), fg)
        bad = {k: v for k, v in errs.items() if not v <= TOL_F32}
        assert not bad, (prec, bad)
        assert max(errs.values()) > 1e-9        # the library really computes in single precision
        assert sg["min_reg_factor"] == pytest.approx(o.status()["min_reg_factor"], rel=1e-3)


@pytest.mark.gpu
def test_f32_gpu_config3_physics_2plus1d_and_lattice(vo):
    import torch
    from paper_1608_06577_b200 import vh
    from test_gpu_parity import field_errors

    t = lambda a: None if a is None else torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda:0")
    cases = []
    prm, init, _ = inputs.config_3d(40, 24, 12, n_hot=6, width=0.5, seed=inputs.BASE_SEED, radius=1.5, eta_half=0.5, newton_rtol=2e-6)
    cases.append((prm, init))
    prm2 = inputs.base_params(nx=40, ny=20, nz=1, n_batch=2, tau0=0.8, dtau=0.02, newton_rtol=2e-6, minmod_theta=1.5)
    cases.append((prm2, inputs.smooth_random_state(prm2, seed=29)))
    prm3 = inputs.base_params(nx=36, ny=12, nz=6, tau0=0.6, dtau=0.02, eos=2, zeta_model=3, zeta_amp=1.0, zeta_T0=0.2 / inputs.HBARC, newton_rtol=2e-6)
    cases.append((prm3, inputs.smooth_random_state(prm3, seed=31)))
    for prm, st in cases:
        s = vh.Solver(prm, precision="f32")
        s.set_initial(t(st["e"]), t(st["u"]), t(st.get("pi")), t(st.get("Pi")))
        s.step(10)
        fg = {k: v.cpu().numpy() for k, v in s.get_fields(with_uprev=True).items()}
        sg = s.status()
        s.close()
        o = vo.Oracle(prm)
        o.set_initial(st["e"], st["u"], st.get("pi"), st.get("Pi"))
        o.step(10)
        errs = field_errors(o.get_fields(with_uprev=True), fg)
        bad = {k: v for k, v in errs.items() if not v <= TOL_F32}
        assert not bad, (prm["eos"], prm["nz"], bad)
        assert sg["n_inversion_failures"] == 0 and sg["n_nonfinite"] == 0


@pytest.mark.gpu
@pytest.mark.parametrize("precision,workload", [("f64", "3d"), ("f32", "3d"), ("f64", "batched2d"), ("f32", "batched2d"), ("f32", "config5")])
def test_full_size_runs_are_bit_reproducible(precision, workload):
    """Regression test of the ring hand-back of the stage kernel: the 128^3 workload, whose 4096 tiles per
    launch keep every SM busy with as many CTAs as fit (two in single precision), must give bitwise the same fields on every run and no
    inversion failure.  Before the fix the two-CTA configuration corrupted about one tile per launch, differently each time; twenty runs of
    three steps are 120 stage launches = half a million tiles per case.  "config5" is the two-CTA build at the size of BASELINE.json
    configs[4] (512 x 512 x 128: 65 536 tiles per launch), five runs of two steps."""
    import torch
    from paper_1608_06577_b200 import vh

    rtol = 2e-6 if precision == "f32" else 1e-13
    n_runs, n_steps = 20, 3
    if workload == "3d":
        prm, init, _ = inputs.config_3d(newton_rtol=rtol)
    elif workload == "config5":
        prm, init, _ = inputs.config_3d(512, 512, 128, dx=0.05, dy=0.05, n_hot=200, newton_rtol=rtol)
        n_runs, n_steps = 5, 2
    else:       # the 2+1d instantiation of the same kernel: 64 events of 201 x 201 = 5824 tiles per launch
        prm, init, _ = inputs.config_batched2d(n_batch=64, newton_rtol=rtol)
    e0, u0 = torch.as_tensor(init["e"], device="cuda:0"), torch.as_tensor(init["u"], device="cuda:0")
    first = None
    for run in range(n_runs):
        s = vh.Solver(prm, precision=precision)
        s.set_initial(e0, u0)
        s.step(n_steps)
        f = s.get_fields()
        st = s.status()
        s.close()
        assert st["n_inversion_failures"] == 0 and st["n_nonfinite"] == 0
        got = torch.cat([f["q"].reshape(-1), f["e"].reshape(-1), f["u"].reshape(-1)])
        del f
        if first is None:
            first = got
        else:
            assert torch.equal(first, got), "run %d differs from run 0" % run
