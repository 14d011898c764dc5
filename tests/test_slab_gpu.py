"""eta-slab decomposition: the step in four parts with boundary planes exchanged between slabs.

(1) One process, two handles on the same GPU exchanging planes directly through vh_halo_export / vh_halo_import: bit-identical to one handle
    over the whole grid (the arithmetic of a cell does not depend on which slab it lives in).
(2) vh.SlabSolver with torch.distributed, world_size 2, gloo (planes staged through the host; with NCCL the same calls send device buffers
    over NVLink): both ranks on the one GPU this box has - each rank drives its own kernels and no kernel waits for another rank - again
    bit-identical to the single-handle run."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_1608_06577_b200 import inputs
from test_gpu_parity import vh  # noqa: F401

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _t(a):
    import torch
    return None if a is None else torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda:0")


def _case():
    prm = inputs.base_params(nx=36, ny=12, nz=16, dx=0.12, dy=0.1, dz=0.15, tau0=0.8, dtau=0.02)
    st = inputs.smooth_random_state(prm, seed=21)
    up = st["u"] * 1.0
    up[1:] *= 0.97
    up[0] = np.sqrt(1 + up[1] ** 2 + up[2] ** 2 + prm["tau0"] ** 2 * up[3] ** 2)
    return prm, st, up


def test_two_slabs_in_one_process_are_bit_identical_to_one_grid(vh):
    import torch
    prm, st, up = _case()
    ref = vh.Solver(prm)
    ref.set_initial(_t(st["e"]), _t(st["u"]), _t(st["pi"]), _t(st["Pi"]))
    ref.set_uprev(_t(up))
    ref.step(5)
    fr = ref.get_fields(with_uprev=True)
    ref.close()
    W = 4
    nzl = prm["nz"] // W
    sl = [vh.Solver(dict(prm, nz=nzl)) for _ in range(W)]
    cut = lambda a, r: None if a is None else _t(np.ascontiguousarray(a[..., r * nzl:(r + 1) * nzl, :, :]))
    bufs = {w: torch.empty(sl[0].halo_size(w), dtype=torch.float64, device="cuda:0") for w in (0, 1)}

    def exchange(what):
        for r in range(W - 1):      # face between slab r (its high side) and slab r + 1 (its low side)
            sl[r].halo_export(what, 1, bufs[what]); sl[r + 1].halo_import(what, 0, bufs[what])
            sl[r + 1].halo_export(what, 0, bufs[what]); sl[r].halo_import(what, 1, bufs[what])

    for r, s in enumerate(sl):
        s.set_initial(cut(st["e"], r), cut(st["u"], r), cut(st["pi"], r), cut(st["Pi"], r))
        s.set_uprev(cut(up, r))
    exchange(1)
    for _ in range(5):
        for part in range(4):
            for s in sl:
                s.step_part(part)
            exchange(part % 2)
    with pytest.raises(vh.VHError):
        sl[0].step_part(2)                       # parts run in order
    for r, s in enumerate(sl):
        f = s.get_fields(with_uprev=True)
        for k in ("q", "e", "p", "u", "up"):
            assert torch.equal(f[k], fr[k][..., r * nzl:(r + 1) * nzl, :, :]), (r, k)
        assert s.status()["n_inversion_failures"] == 0
        s.step(1)                                # a whole step on the same handle still works between part-wise steps
        s.close()
    s2 = vh.Solver(dict(prm, nz=1))
    s2.set_initial(_t(st["e"][:, :1]), _t(st["u"][:, :, :1]))
    with pytest.raises(vh.VHError):
        s2.step_part(0)                          # 2+1d: nothing to decompose
    s2.close()


WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["VH_ROOT"]); sys.path.insert(0, os.path.join(os.environ["VH_ROOT"], "tests"))
import numpy as np, torch
import torch.distributed as dist
from paper_1608_06577_b200 import inputs, vh
from test_slab_gpu import _case, _t
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
prm, st, up = _case()
s = vh.SlabSolver(prm, device="cuda:0")
s.set_initial(_t(st["e"]), _t(st["u"]), _t(st["pi"]), _t(st["Pi"]))
s.set_uprev(_t(up))
s.step(5)
f = s.get_fields()
np.save(os.path.join(os.environ["VH_OUT"], "slab%d.npy" % rank), torch.cat([f["q"].reshape(-1), f["e"].reshape(-1), f["u"].reshape(-1)]).cpu().numpy())
print(json.dumps(s.status()))
s.close()
dist.barrier()
dist.destroy_process_group()
"""


def test_slab_solver_two_ranks_gloo(vh, tmp_path):
    import torch
    prm, st, up = _case()
    ref = vh.Solver(prm)
    ref.set_initial(_t(st["e"]), _t(st["u"]), _t(st["pi"]), _t(st["Pi"]))
    ref.set_uprev(_t(up))
    ref.step(5)
    fr = ref.get_fields()
    ref.close()
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK="0", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), VH_ROOT=ROOT, VH_OUT=str(tmp_path))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    nzl = prm["nz"] // 2
    for r in range(2):
        got = np.load(tmp_path / ("slab%d.npy" % r))
        z = slice(r * nzl, (r + 1) * nzl)
        want = torch.cat([fr["q"][..., z, :, :].reshape(-1), fr["e"][..., z, :, :].reshape(-1), fr["u"][..., z, :, :].reshape(-1)]).cpu().numpy()
        assert np.array_equal(got, want), r
        assert json.loads(outs[r][0].strip().splitlines()[-1])["n_inversion_failures"] == 0


def test_slab_failure_counters_add_up_and_half_steps_are_guarded(vh):
    # a cell in the last plane of slab 0 whose inversion fails (E < 0, E + Pi > 0: reading R6) - the states extrapolated from it sit on the
    # interface between slab 0 and slab 1.  In one grid every interface state is counted once; with slabs each interior face has an owner on
    # either side, so the counters of the slabs must add up to the single grid's, and the fields stay bit-identical
    import torch
    prm, st, up = _case()
    W, nzl = 2, prm["nz"] // 2
    s0 = vh.Solver(prm)
    s0.set_initial(_t(st["e"]), _t(st["u"]), _t(st["pi"]), _t(st["Pi"]))
    s0.set_uprev(_t(up))
    f0 = s0.get_fields(with_uprev=True)
    for k, j, i in ((nzl - 1, 5, 20), (nzl, 7, 9), (0, 3, 3), (prm["nz"] - 1, 8, 30)):      # both sides of the cut, and the two physical boundaries
        e_c = float(f0["e"][0, k, j, i])
        f0["q"][0][0, k, j, i] = -0.05 * e_c + float(f0["q"][4][0, k, j, i])
        f0["q"][14][0, k, j, i] = 0.5 * e_c
    s0.set_state(f0["q"], f0["e"], f0["u"], f0["up"])
    s0.step(1)
    fr, n_ref = s0.get_fields(with_uprev=True), s0.status()["n_inversion_failures"]
    s0.close()
    assert n_ref >= 24
    sl = [vh.Solver(dict(prm, nz=nzl)) for _ in range(W)]
    cut = lambda a, r: a[..., r * nzl:(r + 1) * nzl, :, :].contiguous()
    bufs = {w: torch.empty(sl[0].halo_size(w), dtype=torch.float64, device="cuda:0") for w in (0, 1)}

    def exchange(what):
        sl[0].halo_export(what, 1, bufs[what]); sl[1].halo_import(what, 0, bufs[what])
        sl[1].halo_export(what, 0, bufs[what]); sl[0].halo_import(what, 1, bufs[what])

    for r, s in enumerate(sl):
        s.set_state(cut(f0["q"], r), cut(f0["e"], r), cut(f0["u"], r), cut(f0["up"], r))
    exchange(1)
    for part in range(4):
        for s in sl:
            s.step_part(part)
        if part == 1:      # in the middle of a step nothing that assumes a whole state may run
            for call in (lambda: sl[0].step(1), lambda: sl[0].step_profile(1), lambda: sl[0].run_until(0.1, 3), lambda: sl[0].set_kernel_variant(1)):
                with pytest.raises(vh.VHError):
                    call()
        exchange(part % 2)
    total = 0
    for r, s in enumerate(sl):
        f = s.get_fields(with_uprev=True)
        for k in ("q", "e", "p", "u", "up"):
            assert torch.equal(f[k], fr[k][..., r * nzl:(r + 1) * nzl, :, :]), (r, k)
        total += s.status()["n_inversion_failures"]
        s.close()
    assert total == n_ref, (total, n_ref)
