"""dg_totals_noalloc (include/dg.h): the conserved totals for callers that cannot allocate device memory.

Some users of this library reach it from a place where a cudaMalloc is off the table: a diagnostics hook that a
simulation calls on a GPU it has already filled, an operator inside a framework whose memory pool owns the whole
card, a process that was started under a fixed memory cap, a monitoring thread that must not cause the device-wide
stall an allocation brings.  For them the library carries one fixed scratch array (static __device__, about 128 KB,
good for meshes up to 4 194 304 cells and 8 variables) and an entry point that uses it and allocates nothing.

The test checks that entry point against the path every other test uses (a solver's dg_conserved_totals, which keeps
its per-variable results in the solver's allocated workspace), within the tolerance the existing totals tests use
(1e-12 of the largest total), on calls made back to back: all calls share the scratch array, which still holds the
previous call's block partials, so the second and third call would expose any read of a stale slot.  The file name
sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity tests.
It passes alone in a fresh process (the first call then performs the once-per-device symbol look-up) and after the
rest of the suite.
"""
import numpy as np
import pytest

from paper_2208_11131_b200 import workloads as wk

TOL = 1e-12      # as tests/test_gpu_parity.py: |difference| <= 1e-12 * max |total|


def _case(cfg, degree, ncell):
    """(device copy of the modal state, nvars, ncells, cell volume, totals from the solver path)"""
    import torch
    from paper_2208_11131_b200 import dg
    wl = wk.with_mesh(wk.config(cfg, degree=degree), ncell)
    w0 = wk.initial_modes(wl)
    g = dg.from_workload(wl)
    g.set_state(w0)
    ref = g.conserved_totals()
    g.free()
    return torch.from_numpy(np.ascontiguousarray(w0)).cuda(), wl.dim + 2, wl.ncells, wl.h ** wl.dim, ref


@pytest.mark.gpu
def test_noalloc_totals_match_the_solver_path_on_calls_in_a_row():
    import torch
    from paper_2208_11131_b200 import dg
    # A: 3D, 19 200 cells = 4 full blocks of 4096 cells + a ragged one; B: 2D, 63 cells = part of a single block
    wa, nva, nca, vola, refa = _case(4, 2, (40, 24, 20))
    wb, nvb, ncb, volb, refb = _case(1, None, (9, 7))
    out = torch.full((8,), -7.0, dtype=torch.float64, device="cuda")

    ta = dg.totals_noalloc(wa, nva, nca, vola)                 # first call (does the per-device set-up): host result
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]                 # what the driver itself reports as free
    tb = dg.totals_noalloc(wb, nvb, ncb, volb)                 # second call, smaller: scratch still holds A's partials
    dg.totals_noalloc(wa, nva, nca, vola, out=out)             # third call: device result, stream ordered
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before         # the calls took no device memory
    ta2 = out.cpu().numpy()

    assert np.max(np.abs(ta - refa)) <= TOL * np.max(np.abs(refa)), (ta, refa)
    assert np.max(np.abs(tb - refb)) <= TOL * np.max(np.abs(refb)), (tb, refb)
    assert np.array_equal(ta2[:nva], ta)                       # fixed-shape reduction: bitwise the same both times
    assert np.all(ta2[nva:] == -7.0)                           # nothing written beyond nvars
    assert np.max(np.abs(refa)) > 0 and np.max(np.abs(refb)) > 0


@pytest.mark.gpu
def test_noalloc_totals_refuse_what_the_fixed_scratch_cannot_hold():
    import torch
    from paper_2208_11131_b200 import dg
    w = torch.zeros(64, dtype=torch.float64, device="cuda")
    with pytest.raises(dg.DGError) as ei:                      # one cell too many: refused before any launch
        dg._check(dg.load_library().dg_totals_noalloc(w.data_ptr(), 1, dg.NOALLOC_MAX_CELLS + 1, 1.0,
                                                      w.data_ptr(), 0))
    assert ei.value.code == dg.DG_EINVAL and "DG_NOALLOC_MAX_CELLS" in str(ei.value)
    with pytest.raises(dg.DGError) as ei:
        dg.totals_noalloc(w, dg.NOALLOC_MAX_VARS + 1, 4, 1.0, out=np.empty(16))
    assert ei.value.code == dg.DG_EINVAL and "DG_NOALLOC_MAX_VARS" in str(ei.value)
    with pytest.raises(dg.DGError) as ei:                      # host memory is not a valid input
        host = np.zeros(64)
        dg._check(dg.load_library().dg_totals_noalloc(host.ctypes.data, 1, 64, 1.0, host.ctypes.data, 0))
    assert ei.value.code == dg.DG_EINVAL
    # the limit itself is accepted: one variable over 2^22 cells of ones (32 MB, allocated by the test, not the library)
    ones = torch.ones(dg.NOALLOC_MAX_CELLS, dtype=torch.float64, device="cuda")
    t = dg.totals_noalloc(ones, 1, dg.NOALLOC_MAX_CELLS, 0.5)
    assert t[0] == 0.5 * dg.NOALLOC_MAX_CELLS
