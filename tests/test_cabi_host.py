"""CPU-side checks of the boundary (no compute calls): the C-ABI library builds, loads and exports every symbol
include/dg.h declares; argument validation that needs no device; the roofline work model; the N>1 aggregation
of bench.py under gloo with world_size 2."""
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "dg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dg_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2208_11131_b200 import build, dg
    path = build.build()
    assert os.path.exists(path)
    lib = dg.load_library(build_if_missing=False)
    declared = _declared_symbols()
    assert len(declared) >= 18
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(dg.SYMBOLS) == declared      # the binding covers the header one to one


def test_library_is_sm100a_only():
    from paper_2208_11131_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_no_cpu_fallback_and_argument_validation():
    import torch
    from paper_2208_11131_b200 import dg
    lib = dg.load_library()
    o = dg.default_options()
    assert (o.f_cfl, o.rk_stages, o.av_enable, o.f_v, o.f_tau, o.f_w, o.s_onset0, o.alpha_max) == \
        (0.5, 3, 0, 2.5, 0.5, 0.2, 1e-4, 1.0)
    with pytest.raises(dg.DGError) as ei:                # bad order is rejected before any device work
        dg.Solver(2, (4, 4), 0.25, 0, 1.4, torch_workspace=False)
    assert ei.value.code == dg.DG_EINVAL
    with pytest.raises(dg.DGError) as ei:
        dg.Solver(4, (4, 4, 4), 0.25, 2, 1.4, torch_workspace=False)
    assert ei.value.code == dg.DG_EINVAL
    if not torch.cuda.is_available():                    # the product path fails loudly without a GPU
        with pytest.raises(dg.DGError) as ei:
            dg.Solver(2, (4, 4), 0.25, 2, 1.4, torch_workspace=False)
        assert ei.value.code == dg.DG_ECUDA
        with pytest.raises(dg.DGError):
            dg.Solver(2, (4, 4), 0.25, 2, 1.4)
    assert lib.dg_free(None) == 0


def test_workspace_size_matches_the_memory_model():
    """3 state buffers (u^n and two stage buffers) of V*M*Ncells doubles -- the paper's Eq. 59-62 book-keeping
     with f_t = 3 minus the dw/dt array the stage kernel never stores -- plus the projected
    face fluxes (d * Vc * m^(d-1) doubles per cell) and the two sensor scalars per cell."""
    import ctypes as C
    from paper_2208_11131_b200 import dg
    lib = dg.load_library()
    mesh = dg.dg_mesh()
    mesh.dim = 3
    for a in range(3):
        mesh.ncell[a], mesh.periodic[a] = 16, 1
    mesh.h = 1.0 / 16
    need = C.c_size_t()
    opt = dg.default_options(av_enable=1)
    assert lib.dg_workspace_bytes(C.byref(mesh), 4, C.byref(opt), C.byref(need)) == 0
    state = 6 * 64 * 16 ** 3 * 8
    flux = 3 * 5 * 16 * 16 ** 3 * 8
    assert 3 * state + flux <= need.value <= 3 * state + flux + 4 * 16 ** 3 * 8 + 4096


def test_roofline_model():
    from paper_2208_11131_b200 import roofline as rl
    assert rl.stage_bytes_per_cell(3, 4, True) == 8 * 6 * 64 * 8 / 3          # 8192 B
    f = [rl.stage_flops_per_cell(3, m, False, False) for m in range(1, 9)]
    assert all(b > a for a, b in zip(f, f[1:]))
    assert rl.stage_flops_per_cell(3, 4, True, True) > rl.stage_flops_per_cell(3, 4, True, False) > f[3]
    assert rl.stage_flops_per_cell(3, 4, True, True) == (rl.face_kernel_flops_per_cell(3, 4, True, True)
                                                         + rl.stage_kernel_flops_per_cell(3, 4, True, True))
    assert rl.kernel_bytes_per_cell(3, 4, True) == (3072 + 1920, 3072 * (1 + 2 / 3 + 1) + 1920)
    r = rl.roofline(3, 4, True, True, 128 ** 3, 10e-3, 6535.0, rl.NOMINAL_FP64_TFLOPS)
    assert r["bound"] == "alu" and 0 < r["alu_frac"] < 1 and abs(r["t_hbm_ms"] - 2.63) < 0.05


_GLOO = r"""
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group("gloo")
v, t = bench.aggregate(100.0 * (rank + 1), 2.0 + rank, 2, dist, None)
assert abs(t - 3.0) < 1e-12 and abs(v - 300.0 / 3.0) < 1e-9, (v, t)
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_bench_aggregate_world_size_2_gloo(tmp_path):
    script = tmp_path / "agg.py"
    script.write_text(_GLOO % ROOT)
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29541", str(script)],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    assert r.stdout.count("ok") == 2


def test_bench_reference_arm_is_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference"], env=env,
                       capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
