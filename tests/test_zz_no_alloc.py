"""vh_diagnostics_noalloc (include/vh.h): the diagnostics entry point for callers that must not allocate device memory.

Who that is: a program whose own memory pool already owns the GPU's free memory (a raw cudaMalloc from inside this library would fail, or take
memory the pool counts as its own), or one that calls from a loop in which the device-wide stall of cudaMalloc / cudaFree is not acceptable.
The entry point therefore takes no handle (vh_create allocates), reads the caller's own device arrays and keeps its scratch in a fixed
array inside the library - which caps the grid at VH_NOALLOC_MAX_CELLS cells and makes overlapping calls on one GPU race.

What is checked: its ten maxima and its per-cell maps against the existing path (vh_get_diagnostics / vh_get_diagnostic_maps on a handle
holding the same state), at the 1e-9 of the other diagnostics tests, on consecutive calls whose states and grid sizes differ - so a result or
a scratch entry left over from the previous call cannot pass for the current one.  The file name sorts last on purpose: pytest -x stops at
the first failure, and nothing should hide behind this one.  Every test here passes on its own in a fresh process (the first call on a
device does the one-time set-up) and after the rest of the suite."""
import ctypes as C

import numpy as np
import pytest

from paper_1608_06577_b200 import inputs

TOL = 1e-9           # tests/test_gpu_parity.py: the bar of the diagnostics tests
TOL_F32 = 1e-4       # tests/test_f32.py: the bar of the single-precision build


def _call_raw(L, vh, prm, tau=1.0, ptrs=(1, 1, 1, 1, 1)):
    """The C entry point with made-up non-null pointers: only for calls that must be refused before the device is touched."""
    P = vh.make_params(prm)
    a = [C.c_void_p(x) if x else None for x in ptrs]
    return L.vh_diagnostics_noalloc(C.byref(P), float(tau), a[0], a[1], a[2], a[3], a[4], 1, None, None)


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_oversize_grid_and_bad_arguments_are_refused_before_any_cuda_call(precision):
    # runs without a GPU: the refusals come first in the entry point
    from paper_1608_06577_b200 import build, vh

    build.build()
    L = vh.load_library(precision)
    rtol = 1e-13 if precision == "f64" else 2e-6
    big = inputs.base_params(nx=128, ny=128, nz=65, newton_rtol=rtol)                     # 1 064 960 cells > 2^20
    assert 128 * 128 * 65 > vh.NOALLOC_MAX_CELLS == 1 << 20
    assert _call_raw(L, vh, big) == -1
    msg = L.vh_last_error(None).decode()
    assert "1064960" in msg and "1048576" in msg and "VH_NOALLOC_MAX_CELLS" in msg, msg
    ok = inputs.base_params(nx=8, ny=8, nz=8, newton_rtol=rtol)
    assert _call_raw(L, vh, ok, ptrs=(1, 1, 0, 1, 1)) == -1                               # u4 missing
    assert b"required" in L.vh_last_error(None)
    assert _call_raw(L, vh, ok, tau=0.0) == -1                                            # Milne needs tau > 0
    assert b"tau > 0" in L.vh_last_error(None)
    bad = dict(ok, nx=0)
    assert _call_raw(L, vh, bad) == -1                                                    # the parameter checks of vh_create


def _cases(precision):
    """(name, params, initial state as a dict for set_initial) of five differently sized problems, largest first."""
    rtol = {} if precision == "f64" else dict(newton_rtol=2e-6)
    prm_a, init_a, _ = inputs.config_3d(72, 40, 24, n_hot=6, width=0.5, seed=inputs.BASE_SEED + 11, radius=2.5, eta_half=0.8, **rtol)   # 69 120 cells = 270 blocks
    prm_b = inputs.base_params(nx=36, ny=20, nz=10, dx=0.12, dy=0.1, dz=0.15, tau0=0.8, dtau=0.02, **rtol)                              # 7 200 cells, ragged last block
    st_b = inputs.smooth_random_state(prm_b, seed=29)                                                                                  # every pi component, Pi, vorticity
    prm_c, init_c, _ = inputs.config_batched2d(n_batch=3, n=45, n_hot=5, seed=inputs.BASE_SEED + 6, radius=1.8, **rtol)                  # batched 2+1d: no eta differences
    lat = dict(eos=2, zeta_model=3, zeta_amp=1.0, zeta_T0=0.2 / inputs.HBARC)
    prm_d, init_d, _ = inputs.config_3d(40, 20, 8, n_hot=5, width=0.5, seed=inputs.BASE_SEED + 3, radius=1.5, eta_half=0.3, **dict(lat, **rtol))  # lattice EOS: the table in its fixed array
    prm_e, init_e, _ = inputs.config_3d(24, 20, 12, n_hot=4, width=0.5, seed=inputs.BASE_SEED + 12, radius=1.2, eta_half=0.5, geometry=1, **rtol)   # Cartesian: the other template instantiation
    return [("config3", prm_a, dict(e=init_a["e"], u=init_a["u"])), ("generic", prm_b, st_b), ("batched2d", prm_c, dict(e=init_c["e"], u=init_c["u"])),
            ("lattice", prm_d, dict(e=init_d["e"], u=init_d["u"])), ("cartesian", prm_e, dict(e=init_e["e"], u=init_e["u"]))]


@pytest.mark.gpu
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_noalloc_diagnostics_match_the_handle_path_on_consecutive_calls(precision):
    import torch

    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_1608_06577_b200 import vh

    tol = TOL if precision == "f64" else TOL_F32
    dev = "cuda:0"
    t = lambda a: None if a is None else torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
    calls = 0
    previous = None
    for name, prm, st in _cases(precision):
        s = vh.Solver(prm, device=dev, precision=precision)
        s.set_initial(t(st["e"]), t(st["u"]), t(st.get("pi")), t(st.get("Pi")))
        cells = prm["nx"] * prm["ny"] * prm["nz"] * prm["n_batch"]
        maps = torch.empty(10 * cells, dtype=torch.float64, device=dev)          # the caller's output array, made before the calls under test
        for n_steps in (3, 1):                                                   # two states per problem: call k + 1 follows call k directly
            s.step(n_steps)
            f = s.get_fields(with_uprev=True)                                    # CUDA tensors: the arrays such a caller already holds
            tau = s.status()["tau"]
            ref = s.diagnostics()                                                # existing path: vh_get_diagnostics
            ref_maps = s.diagnostic_maps().reshape(10, -1).cpu().numpy()         # existing path: vh_get_diagnostic_maps
            torch.cuda.synchronize()
            maps.fill_(-1.0)
            free0 = torch.cuda.mem_get_info()[0]
            got = vh.diagnostics_noalloc(prm, tau, f["q"], f["e"], f["u"], f["up"], maps=maps, precision=precision)
            free1 = torch.cuda.mem_get_info()[0]
            calls += 1
            if n_steps == 1:                                                     # (a problem's first call may load its kernel instantiation: code, not data)
                assert free1 >= free0, "device memory shrank by %d bytes across a call that must not allocate" % (free0 - free1)
            got_maps = maps.reshape(10, -1).cpu().numpy()
            assert list(got) == list(ref)
            for k, key in enumerate(ref):
                scale = max(ref[key], np.max(np.abs(ref_maps[k])))
                assert abs(got[key] - ref[key]) <= tol * scale, (name, n_steps, key, got[key], ref[key])
                assert np.all(np.abs(got_maps[k] - ref_maps[k]) <= tol * scale), (name, n_steps, key)
                assert got[key] == got_maps[k].max(), (name, n_steps, key)     # the combined per-block maxima are the maximum of the map
            assert ref["max_T"] > 0 and ref["max_inv_reynolds_shear"] > 0 and ref["max_knudsen_shear"] > 0      # not a comparison of zeros
            if previous is not None:                                             # and not a copy of what the previous call left in the scratch
                assert any(got[key] != previous[key] for key in got)
            previous = got
            # the same call once more with the maxima delivered to a DEVICE array (no synchronisation inside the entry point) and no maps
            out_dev = torch.full((10,), -1.0, dtype=torch.float64, device=dev)
            L = vh.load_library(precision)
            P = vh.make_params(prm)
            p = lambda x: C.c_void_p(x.data_ptr())
            rc = L.vh_diagnostics_noalloc(C.byref(P), float(tau), p(f["q"]), p(f["e"]), p(f["u"]), p(f["up"]), p(out_dev), 1, None,
                                          C.c_void_p(torch.cuda.current_stream().cuda_stream))
            assert rc == 0, L.vh_last_error(None)
            calls += 1
            assert out_dev.cpu().tolist() == list(got.values()), (name, n_steps)
        s.close()
    assert calls == 20
