"""GPU parity tests (run on the B200 box with -m gpu): the CUDA path behind the C-ABI (include/dg.h) against
the CPU oracle (oracle/dg_oracle.py) on the same seeded inputs, element by element.

Tolerances (BASELINE.json north_star): max relative L-infinity difference per conserved variable
<= 1e-12 after one step and <= 1e-9 after 10 steps (norm: DESIGN.md reading A24).
"""
import numpy as np
import pytest

from paper_2208_11131_b200 import workloads as wk
from parity_util import make_gpu, make_oracle, parity_norm, rhs_scale

pytestmark = pytest.mark.gpu

TOL_1 = 1e-12
TOL_10 = 1e-9


def _wl(d, ncell, n, phys, f_cfl=0.3):
    return wk.Workload("rand", d, tuple(ncell), 1.0 / ncell[0], n, 1.4 if d == 2 else 5.0 / 3.0,
                       nu=0.01 if "ns" in phys else 0.0, chi=0.02 if "ns" in phys else 0.0,
                       av=("av" in phys), f_cfl=f_cfl)


def _random_pair(wl, seed=11, amp=0.04):
    w0, al = wk.random_smooth_modes(wl.dim, wl.ncell, wl.degree, wl.gamma, seed=seed, amp=amp,
                                    nvar_extra=1 if wl.av else 0)
    o = make_oracle(wl)
    g = make_gpu(wl)
    o.set_state(w0)
    g.set_state(w0)
    if wl.av:
        o.set_alpha(al)
        g.set_alpha(al)
    return o, g


# ---------------------------------------------------------------------------------------------------
# term-level: dw/dt = L(w) (Eq. 20) on random smooth states, every physics variant, ragged cell counts
# ---------------------------------------------------------------------------------------------------
RHS_CASES = [(2, (5, 3), n, ph) for n in (0, 1, 2, 3, 5, 7) for ph in ("euler", "ns", "av", "ns_av")] + \
            [(3, (3, 2, 2), n, ph) for n in (0, 1, 2, 3) for ph in ("euler", "ns", "av", "ns_av")] + \
            [(3, (2, 2, 3), 4, "ns_av"), (3, (2, 3, 2), 5, "euler"), (3, (2, 2, 2), 7, "euler"),
             (3, (2, 2, 2), 6, "ns_av"), (2, (37, 3), 3, "ns_av"), (3, (9, 4, 3), 3, "ns_av")]


@pytest.mark.parametrize("d,ncell,n,phys", RHS_CASES)
def test_rhs_parity(d, ncell, n, phys):
    wl = _wl(d, ncell, n, phys)
    o, g = _random_pair(wl)
    if wl.av:   # non-trivial lagged sensor state: take one step on both sides first (sensor set on stage 1)
        assert o.step(1) == 0
        g.step(1)
    L = o.rhs(o.w)
    Lg, Lal = g.eval_rhs(with_alpha=True)
    Vc = wl.dim + 2
    Lo = np.ascontiguousarray(L[:, :, :Vc].transpose(1, 2, 0)).ravel()
    err = np.max(np.abs(Lg - Lo).reshape(wl.modes, Vc, -1), axis=(0, 2)) / rhs_scale(Lo, wl)
    assert np.all(err < 5e-12), err
    if wl.av:
        La = np.ascontiguousarray(L[:, :, Vc].T).ravel()
        assert np.max(np.abs(Lal - La)) < 5e-12 * max(1.0, np.max(np.abs(La)))


# ---------------------------------------------------------------------------------------------------
# step-level parity on the five BASELINE configs at oracle-sized meshes (same ICs, same options)
# ---------------------------------------------------------------------------------------------------
def _scaled_config(i, degree=None):
    if i == 1:
        return wk.config(1)                                    # 16x16, full size
    if i == 2:
        return wk.with_mesh(wk.config(2), (24, 48))            # KH + NS, n = 3
    if i == 3:
        return wk.with_mesh(wk.config(3), (128, 2))            # Sod + AV, n = 5, jump on a cell boundary
    if i == 4:
        return wk.with_mesh(wk.config(4), (6, 6, 6))           # 3D NS + AV, n = 3
    return wk.with_mesh(wk.config(5, degree=degree), (6, 6, 6) if degree < 6 else (3, 3, 3))


STEP_CASES = [(1, None), (2, None), (3, None), (4, None)] + [(5, n) for n in range(1, 8)]


@pytest.mark.parametrize("cfg,degree", STEP_CASES)
def test_step_parity(cfg, degree):
    wl = _scaled_config(cfg, degree)
    w0 = wk.initial_modes(wl)
    o = make_oracle(wl)
    g = make_gpu(wl)
    o.set_state(w0)
    g.set_state(w0)
    assert o.step(1) == 0
    g.step(1)
    e1 = parity_norm(g.get_state(), o.get_state(), wl)
    assert np.all(e1 <= TOL_1), ("1 step", e1)
    to, dto = o.t, o.last_dt
    tg, dtg = g.get_time()
    assert abs(dtg - dto) <= 1e-14 * dto and abs(tg - to) <= 1e-14 * to
    assert o.step(9) == 0
    g.step(9)
    e10 = parity_norm(g.get_state(), o.get_state(), wl)
    assert np.all(e10 <= TOL_10), ("10 steps", e10)
    if wl.av:
        assert np.max(np.abs(g.get_alpha() - o.get_alpha())) <= TOL_10
    # conserved totals agree with the oracle's and with the initial ones
    tg = g.conserved_totals()
    assert np.max(np.abs(tg - o.conserved_totals())) <= 1e-12 * np.max(np.abs(tg))


def test_graph_and_plain_launch_bit_identical():
    wl = _scaled_config(4)
    w0 = wk.initial_modes(wl)
    res = []
    for use_graph in (1, 0, 1):
        g = make_gpu(wl, use_graph=use_graph)
        g.set_state(w0)
        g.step(3)
        res.append((g.get_state(), g.get_alpha(), g.get_time()))
    for r in res[1:]:
        assert np.array_equal(r[0], res[0][0]) and np.array_equal(r[1], res[0][1]) and r[2] == res[0][2]


@pytest.mark.parametrize("stages", [1, 2])
def test_lower_rk_parity(stages):
    wl = _scaled_config(2)
    w0 = wk.initial_modes(wl)
    o = make_oracle(wl, rk_stages=stages)
    g = make_gpu(wl, rk_stages=stages)
    o.set_state(w0)
    g.set_state(w0)
    assert o.step(3) == 0
    g.step(3)
    assert np.all(parity_norm(g.get_state(), o.get_state(), wl) <= 1e-11)


def test_fixed_dt_and_time():
    wl = _scaled_config(1)
    w0 = wk.initial_modes(wl)
    o = make_oracle(wl, fixed_dt=1e-3)
    g = make_gpu(wl, fixed_dt=1e-3)
    o.set_state(w0)
    g.set_state(w0)
    o.step(4)
    g.step(4)
    t, dt = g.get_time()
    assert dt == 1e-3 and abs(t - 4e-3) < 1e-15
    assert np.all(parity_norm(g.get_state(), o.get_state(), wl) <= 1e-12)


# ---------------------------------------------------------------------------------------------------
# invariants that hold at any size (used at the full BASELINE sizes by test_gpu_fullsize.py as well)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("d,n,phys", [(2, 3, "ns_av"), (3, 2, "ns_av"), (3, 3, "euler")])
def test_free_stream(d, n, phys):
    wl = _wl(d, (7, 5, 3)[:d], n, phys)
    Vc = d + 2
    w = np.zeros((wl.modes, Vc, wl.ncells))
    w[0] = np.array([1.3, 0.4, -0.7, 0.2, 3.1])[[0, 1, 2] + ([3] if d == 3 else []) + [4]][:, None]
    g = make_gpu(wl)
    g.set_state(w.ravel())
    L = g.eval_rhs().reshape(wl.modes, Vc, -1)
    assert np.max(np.abs(L)) < 1e-11


def test_conservation_and_totals():
    wl = _wl(3, (5, 4, 3), 2, "ns_av", f_cfl=0.1)
    o, g = _random_pair(wl, seed=5)
    t0 = g.conserved_totals()
    assert np.allclose(t0, o.conserved_totals(), rtol=1e-14, atol=1e-15)
    g.step(5)
    t1 = g.conserved_totals()
    assert np.max(np.abs(t1 - t0)) < 1e-13 * np.max(np.abs(t0))


def test_unphysical_state_is_reported():
    from paper_2208_11131_b200 import dg
    wl = _wl(2, (4, 4), 1, "euler")
    w = np.zeros((wl.modes, 4, wl.ncells))
    w[0, 0] = 1.0
    w[0, 3] = -1.0     # negative energy -> negative pressure
    g = make_gpu(wl)
    g.set_state(w.ravel())
    with pytest.raises(dg.DGError) as ei:
        g.step(1)
    assert ei.value.code == dg.DG_EUNPHYSICAL


def test_bad_arguments():
    from paper_2208_11131_b200 import dg
    with pytest.raises(dg.DGError) as ei:
        dg.Solver(2, (4, 4), 0.25, 9, 1.4)
    assert ei.value.code == dg.DG_EINVAL
    g = dg.Solver(2, (4, 4), 0.25, 2, 1.4)
    with pytest.raises(dg.DGError):
        g.set_state(np.zeros(7))
    with pytest.raises(dg.DGError):
        g.set_alpha(np.zeros(4 * 16))     # AV not enabled


def test_device_pointer_io():
    import torch
    wl = _scaled_config(1)
    w0 = wk.initial_modes(wl)
    g = make_gpu(wl)
    g.set_state(torch.from_numpy(w0).cuda())
    out = torch.empty(w0.size, dtype=torch.float64, device="cuda")
    g.get_state(out)
    assert np.array_equal(out.cpu().numpy(), w0)
