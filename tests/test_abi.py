"""CPU-side checks of the boundary: libvh.so loads without a GPU and exports every symbol include/vh.h declares;
the product path fails loudly (no CPU fallback) when no CUDA device is present; package hygiene."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1608_06577_b200 import build, vh

    build.build()
    return vh.load_library()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "vh.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(vh_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_1608_06577_b200 import vh

    names = declared_functions()
    assert len(names) >= 11
    for n in names:
        assert hasattr(lib, n), "libvh.so does not export %s" % n
    assert sorted(vh.EXPORTS) == names, "the Python binding and include/vh.h disagree on the entry points"


def test_params_struct_layout_matches_header():
    from paper_1608_06577_b200 import vh

    src = open(os.path.join(ROOT, "include", "vh.h")).read()
    body = src[src.index("typedef struct {") + len("typedef struct {") : src.index("} vh_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        m = re.match(r"\s*(int|double)\s+(.*)", decl.strip(), flags=re.S)
        if m:
            for name in m.group(2).split(","):
                fields.append((name.strip(), m.group(1)))
    got = [(n, "int" if t is C.c_int else "double") for n, t in vh.vh_params._fields_]
    assert got == fields


def test_no_gpu_means_loud_failure(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("this box has a GPU")
    from paper_1608_06577_b200 import inputs, vh

    with pytest.raises(vh.VHError):
        vh.Solver(inputs.base_params(nx=4, ny=4, nz=4))
    p = vh.make_params(inputs.base_params(nx=4, ny=4, nz=4))
    h = C.c_void_p()
    assert lib.vh_create(C.byref(p), None, C.byref(h)) == -3      # VH_ERR_CUDA
    assert h.value is None
    assert lib.vh_create(None, None, C.byref(h)) == -1            # VH_ERR_ARG before any CUDA call
    assert b"NULL" in lib.vh_last_error(None)


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1608_06577_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "vh_oracle" not in txt and "oracle/" not in txt.replace("shares nothing with oracle/", ""), os.path.join(dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".hpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libvh.so" not in txt and "import vh\n" not in txt and "vh_device" not in txt


def test_inputs_are_seeded_and_reproducible():
    import numpy as np

    from paper_1608_06577_b200 import inputs

    r = inputs.SplitMix64(inputs.BASE_SEED)
    first = [r.next_u64() for _ in range(3)]
    r2 = inputs.SplitMix64(inputs.BASE_SEED)
    assert first == [r2.next_u64() for _ in range(3)]
    # SplitMix64 reference value for seed 0 (first output of the published algorithm)
    assert inputs.SplitMix64(0).next_u64() == 0xE220A8397B1DCDAF
    _, a, _ = inputs.config_3d(16, 16, 8, n_hot=4)
    _, b, _ = inputs.config_3d(16, 16, 8, n_hot=4)
    np.testing.assert_array_equal(a["e"], b["e"])
    assert a["e"].min() >= 0.05 / inputs.HBARC * (1 - 1e-12)       # pedestal (reading R14)
    _, c, _ = inputs.config_batched2d(n_batch=2, n=12, n_hot=3)
    assert not np.array_equal(c["e"][0], c["e"][1])                 # event b uses seed + b


def test_lattice_eos_table_of_the_product_matches_the_oracle(vo):
    """EOS 2 (R19, R20): the CUDA library builds its table on the host with its own quadrature and root finder
    (csrc/vh_eos_lattice.hpp); the oracle builds its own (oracle/vh_oracle_lattice.hpp).  No code is shared, so agreement of the node
    values - here against the oracle's interpolant evaluated AT the nodes, where Hermite interpolation returns the node value -
    checks both builders against each other before any kernel runs."""
    import numpy as np
    from paper_1608_06577_b200 import inputs, vh

    nodes, x0, h = vh.eos_table()
    assert nodes.shape == (2049, 4) and np.all(np.isfinite(nodes)) and np.all(np.diff(nodes[:, 0]) > 0) and np.all(np.diff(nodes[:, 2]) > 0)
    prm = inputs.base_params(eos=2)
    for k in (0, 1, 7, 100, 511, 1024, 1777, 2047):
        xk = x0 + k * h
        xe = xk * (1 + 1e-13) if k == 0 else xk          # (stay inside the table at its first node)
        r = vo.eos(prm, xe**4)
        assert r["p"] == pytest.approx(nodes[k, 0], rel=1e-10)
        assert r["T"] == pytest.approx(nodes[k, 2], rel=1e-10)
        assert r["cs2"] == pytest.approx(nodes[k, 1] / h / (4 * xk**3), rel=1e-8)
    assert nodes[0, 2] * inputs.HBARC == pytest.approx(0.03, rel=1e-12) and nodes[-1, 2] * inputs.HBARC == pytest.approx(2.0, rel=1e-12)


def test_diagnostic_names_agree_with_the_header_and_the_oracle(vo):
    # the binding, the header and the test oracle describe the same ten diagnostics in the same order
    from paper_1608_06577_b200 import vh

    src = open(os.path.join(ROOT, "include", "vh.h")).read()
    n = int(re.search(r"#define\s+VH_N_DIAGNOSTICS\s+(\d+)", src).group(1))
    assert n == len(vh.Solver.DIAG_NAMES) == len(vo.DIAG_NAMES) == 10
    assert tuple(vh.Solver.DIAG_NAMES) == tuple(vo.DIAG_NAMES)


def test_committed_ncu_metrics_file_is_what_bench_reads():
    """bench.py takes roofline.traffic, executed_flops_per_cell and fp64_pipe_util from the committed raw ncu CSV: it must hold exactly one
    RK2 step of the default pipeline (velocity, stage, velocity, stage) with every metric bench.py uses, and plausible magnitudes."""
    sys.path.insert(0, ROOT)
    import bench

    pages = {"config3": 128 ** 3, "config4": 256 * 201 * 201, "config5": 512 * 512 * 128, "paper": 128 ** 3}
    for tag, ncell in pages.items():
        page = bench.metrics_page(workload=tag if tag.startswith("config") else "config3", physics="paper" if tag == "paper" else "config3")
        assert page and os.path.exists(page), tag
        m = bench.ncu_metrics(page)
        assert list(m) == list(bench.LAUNCH_KEYS), tag
        for key, row in m.items():
            assert ("velocity" in key) == ("velocity" in row["kernel"])
            flops = (2 * row["smsp__sass_thread_inst_executed_op_dfma_pred_on.sum"] + row["smsp__sass_thread_inst_executed_op_dadd_pred_on.sum"]
                     + row["smsp__sass_thread_inst_executed_op_dmul_pred_on.sum"]) / ncell
            assert 500 < flops < 5000, (tag, key, flops)
            assert 0.2 < row["sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"] / 100 < 1.0
            traffic = (row["dram__bytes_read.sum"] + row["dram__bytes_write.sum"]) / ncell
            assert 50 < traffic < 1500, (tag, key, traffic)
    # no page, no fraction: single precision, reduced storage and the A/B kernel variants have none
    assert bench.metrics_page(precision="f32") is None and bench.metrics_page(storage=1) is None and bench.metrics_page(variant=1) is None
