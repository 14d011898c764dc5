"""GPU <-> oracle parity of the reduced-storage mode (vh_params.storage = 1; Eqs. 47-51; R22), through the C ABI.
Same norm and bar as tests/test_gpu_parity.py (1e-9 after 10 steps, counters equal)."""
import numpy as np
import pytest

from paper_1608_06577_b200 import inputs
from test_gpu_parity import assert_parity, vh  # noqa: F401

pytestmark = pytest.mark.gpu


def _t(a):
    import torch
    return None if a is None else torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda:0")


def _pair(vh, vo, prm, st, n_steps, uprev=None):
    o = vo.Oracle(prm)
    o.set_initial(st["e"], st["u"], st.get("pi"), st.get("Pi"))
    if uprev is not None:
        o.set_uprev(uprev)
    o.step(n_steps)
    s = vh.Solver(prm)
    s.set_initial(_t(st["e"]), _t(st["u"]), _t(st.get("pi")), _t(st.get("Pi")))
    if uprev is not None:
        s.set_uprev(_t(uprev))
    s.step(n_steps)
    fg = {k: v.cpu().numpy() for k, v in s.get_fields(with_uprev=True).items()}
    sg = s.status()
    s.close()
    return o.get_fields(with_uprev=True), o.status(), fg, sg


def test_reduced_generic_state_3d_and_constraints(vh, vo):
    prm = inputs.base_params(nx=36, ny=12, nz=6, dx=0.12, dy=0.1, dz=0.15, tau0=0.8, dtau=0.02, storage=1)
    st = inputs.smooth_random_state(prm, seed=21)
    up = st["u"] * 1.0
    up[1:] *= 0.97      # u^{n-1} != u^n: the time derivatives of the sources are exercised from the first step (u^tau of it is not state)
    fo, so, fg, sg = _pair(vh, vo, prm, st, 10, uprev=up)
    assert so["n_inversion_failures"] == 0
    assert_parity(fo, so, fg, sg)
    # the exported tensor satisfies Eqs. 47-51 to rounding (dense check as in tests/test_oracle_reduced.py)
    tau = sg["tau"]
    g = np.array([1.0, -1.0, -1.0, -tau * tau])
    slot = [[4, 5, 6, 7], [5, 8, 9, 10], [6, 9, 11, 12], [7, 10, 12, 13]]
    pi = np.array([[fg["q"][slot[m][n]] for n in range(4)] for m in range(4)])
    assert np.max(np.abs(np.einsum("lm...,m,m...->l...", pi, g, fg["u"]))) < 1e-13 * np.max(np.abs(pi)) * 10
    assert np.max(np.abs(np.einsum("m,mm...->...", g, pi))) < 1e-13 * np.max(np.abs(pi)) * 10


def test_reduced_config3_physics_2plus1d_cartesian_lattice(vh, vo):
    prm, init, _ = inputs.config_3d(40, 24, 12, n_hot=6, width=0.5, seed=inputs.BASE_SEED, radius=1.5, eta_half=0.5, storage=1)
    assert_parity(*_pair(vh, vo, prm, init, 10))
    prm2 = inputs.base_params(nx=40, ny=20, nz=1, n_batch=2, tau0=0.8, dtau=0.02, minmod_theta=1.5, storage=1)
    assert_parity(*_pair(vh, vo, prm2, inputs.smooth_random_state(prm2, seed=29), 10))
    prm3 = inputs.base_params(nx=36, ny=12, nz=6, tau0=0.8, dtau=0.02, geometry=1, physics=1, storage=1)
    assert_parity(*_pair(vh, vo, prm3, inputs.smooth_random_state(prm3, seed=23), 10))
    prm4 = inputs.base_params(nx=36, ny=12, nz=6, tau0=0.6, dtau=0.02, eos=2, zeta_model=3, zeta_amp=1.0, zeta_T0=0.2 / inputs.HBARC, storage=1)
    assert_parity(*_pair(vh, vo, prm4, inputs.smooth_random_state(prm4, seed=31), 10))


def test_reduced_storage_uses_less_memory_and_restarts(vh, vo):
    import torch
    prm = inputs.base_params(nx=64, ny=64, nz=32, storage=1)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    s1 = vh.Solver(prm)
    free1 = torch.cuda.mem_get_info()[0]
    s0 = vh.Solver(dict(prm, storage=0))
    free2 = torch.cuda.mem_get_info()[0]
    assert (free0 - free1) < 0.68 * (free1 - free2)          # 43 of 67 padded arrays
    s0.close()
    with pytest.raises(vh.VHError):
        s1.diagnostics()                                      # the diagnostics kernels need the full arrays
    s1.close()
    with pytest.raises(vh.VHError):
        vh.Solver(dict(prm, physics=2))                       # nothing to reduce without shear
    # restart through vh_set_state: bit-identical continuation
    prm = inputs.base_params(nx=20, ny=12, nz=6, tau0=0.6, dtau=0.02, storage=1)
    st = inputs.smooth_random_state(prm, seed=5)
    a = vh.Solver(prm)
    a.set_initial(_t(st["e"]), _t(st["u"]), _t(st["pi"]), _t(st["Pi"]))
    a.step(3)
    f = a.get_fields(with_uprev=True)
    b = vh.Solver(dict(prm, tau0=prm["tau0"]))
    b.set_state(f["q"], f["e"], f["u"], f["up"], n_steps_done=3)
    a.step(2); b.step(2)
    fa, fb = a.get_fields(), b.get_fields()
    for k in ("q", "e", "u"):
        assert torch.equal(fa[k], fb[k]), k
    a.close(); b.close()


@pytest.mark.parametrize("dims", [(1, 1, 1), (3, 2, 1), (2, 1, 3), (1, 5, 2), (33, 5, 5)])
@pytest.mark.parametrize("mode", ["reduced", "f32"])
def test_degenerate_grids_in_the_other_modes(vh, vo, dims, mode):
    # grids smaller than a tile, extents of 1 in any direction, ragged tiles: reduced storage (1e-9) and the single-precision build (1e-4)
    from test_gpu_parity import field_errors
    prm = inputs.base_params(nx=dims[0], ny=dims[1], nz=dims[2], tau0=0.7, dtau=0.01, newton_rtol=2e-6 if mode == "f32" else 1e-13,
                             storage=1 if mode == "reduced" else 0)
    st = inputs.smooth_random_state(prm, seed=3)
    o = vo.Oracle(prm)
    o.set_initial(st["e"], st["u"], st["pi"], st["Pi"])
    o.step(5)
    s = vh.Solver(prm, precision="f32" if mode == "f32" else "f64")
    s.set_initial(_t(st["e"]), _t(st["u"]), _t(st["pi"]), _t(st["Pi"]))
    s.step(5)
    fg = {k: v.cpu().numpy() for k, v in s.get_fields(with_uprev=True).items()}
    sg = s.status()
    s.close()
    assert max(field_errors(o.get_fields(with_uprev=True), fg).values()) <= (1e-4 if mode == "f32" else 1e-9)
    assert sg["n_inversion_failures"] == 0 and sg["n_nonfinite"] == 0
