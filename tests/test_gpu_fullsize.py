"""Full-size GPU tests of the five BASELINE configs (run on the B200 box with -m gpu).

 * cfg2 (128x256, degree 3, NS) and cfg3 (1024x16, degree 5, AV) at FULL size against the numpy oracle:
   1 step <= 1e-12, 10 steps <= 1e-9 (north_star tolerances, norm A24), then the GPU alone to the full step count
   (100 / 200) under invariants: conserved totals, no unphysical state, bounded alpha (the
   maximum is reported).
 * cfg4 (128^3) 50 steps and cfg5 (64^3, degrees 1..7) 20 steps each under invariants; cfg5 and cfg1 against the
   exact advected solution (PAPER.md:434-442 style smooth wave; BASELINE configs 1 and 5).
 * cfg5 degrees 1..3 at 64^3: the STATE after one full RK3 step of sampled cells against a periodic 7^3 oracle patch
   (three stages reach three cells: the centre of a 7-cell-wide periodic patch sees no wrap-around), fixed dt.
"""
from dataclasses import replace

import numpy as np
import pytest

from paper_2208_11131_b200 import workloads as wk
from parity_util import make_gpu, make_oracle, parity_norm

pytestmark = pytest.mark.gpu

TOL_1 = 1e-12
TOL_10 = 1e-9


def _report(line):
    import os
    d = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    if os.path.isdir(d):
        with open(os.path.join(d, "parity_report.txt"), "a") as f:
            f.write(line + "\n")


def _drift(t1, t0, wl):
    """Relative drift of the conserved totals; the momentum components share the scale rho c_s |domain|."""
    d = wl.dim
    scale = np.abs(t0).copy()
    scale[1:1 + d] = max(np.max(np.abs(t0[1:1 + d])), abs(t0[0]))
    return np.max(np.abs(t1 - t0) / scale)


def _oracle_wave_speeds(o, wflat, wl, cells):
    """Eq. 23 inputs of the oracle, o.wave_speeds, over the cells `cells` (an index array or slice into
    the cell axis) of a full-size state in the C-ABI layout; `o` is any oracle of the same order and physics."""
    M, Vc = wl.modes, wl.dim + 2
    w = np.asarray(wflat).reshape(M, Vc, wl.ncells)[:, :, cells]
    return o.wave_speeds(np.ascontiguousarray(w.transpose(2, 0, 1)))


@pytest.mark.parametrize("cfg,steps", [(2, 100), (3, 200)])
def test_full_size_parity_then_full_length(cfg, steps):
    wl = wk.config(cfg)
    assert wl.ncell == ((128, 256) if cfg == 2 else (1024, 16))
    w0 = wk.initial_modes(wl)
    o = make_oracle(wl)
    g = make_gpu(wl)
    o.set_state(w0)
    g.set_state(w0)
    t0 = g.conserved_totals()
    assert o.step(1) == 0
    g.step(1)
    e1 = parity_norm(g.get_state(), o.get_state(), wl)
    assert np.all(e1 <= TOL_1), ("1 step", e1)
    assert abs(g.get_time()[1] - o.last_dt) <= 1e-14 * o.last_dt
    assert o.step(9) == 0
    g.step(9)
    e10 = parity_norm(g.get_state(), o.get_state(), wl)
    assert np.all(e10 <= TOL_10), ("10 steps", e10)
    if wl.av:
        assert np.max(np.abs(g.get_alpha() - o.get_alpha())) <= TOL_10
    g.step(steps - 10)                                     # raises on DG_EUNPHYSICAL
    d = g.diagnostics()
    assert d["steps"] == steps and d["unphysical"] == 0
    drift = _drift(g.conserved_totals(), t0, wl)
    assert drift <= 1e-13 * steps, drift
    if wl.av:
        # the switch acts at the shock; the raw field may exceed alpha_max = 1 there (only the point value entering
        # Eq. 46 is clamped, reading A17) but stays bounded
        assert 0.1 < d["alpha_max_seen"] < 4.0, d
    _report("%s FULL SIZE %s: 1 step %.3e, 10 steps %.3e; %d steps: totals drift %.2e, max alpha %.3f" % (
        wl.name, "x".join(map(str, wl.ncell)), np.max(e1), np.max(e10), steps, drift, d["alpha_max_seen"]))


def _exact_mean_density(wl, t):
    """Cell means of rho = 1 + 0.1 sin(2 pi (sum_a x_a - d t)) (advection with v = (1,..,1)): analytic average."""
    d, h = wl.dim, wl.h
    axes = [wl.origin[a] + (np.arange(wl.ncell[a]) + 0.5) * h for a in range(d)]
    grids = np.meshgrid(*axes[::-1], indexing="ij")          # z, y, x order: x fastest after ravel
    phase = 2.0 * np.pi * (sum(grids) - d * t)
    damp = (np.sin(np.pi * h) / (np.pi * h)) ** d
    return (1.0 + 0.1 * damp * np.sin(phase)).ravel()


def test_cfg1_exact_solution():
    wl = wk.config(1)
    g = make_gpu(wl)
    g.set_state(wk.initial_modes(wl))
    g.step(10)
    t, _ = g.get_time()
    rho = g.get_state().reshape(wl.modes, wl.dim + 2, -1)[0, 0]
    err = np.mean(np.abs(rho - _exact_mean_density(wl, t)))
    assert err < 2e-4, err                                    # degree 1 on 16x16: second order


def test_cfg4_full_size_50_steps():
    wl = wk.config(4)
    assert wl.ncell == (128, 128, 128)
    import torch
    host = torch.empty(wl.nvar_conserved * wl.modes * wl.ncells, dtype=torch.float64, pin_memory=True)
    wk.initial_modes_slabbed(wl, out=host.numpy())
    g = make_gpu(wl)
    g.set_state(host)
    t0 = g.conserved_totals()
    # one RK3 step at full size in the bench launch configuration, compared on sampled cells with the oracle run on the
    # periodic 7x7x7 patch around each cell (exact: three stages reach three cells)
    g.step(1)
    _, dt = g.get_time()
    d, Vc, M, N = wl.dim, wl.dim + 2, wl.modes, wl.ncells
    nx, ny, nz = wl.ncell
    sub = replace(wl, ncell=(7, 7, 7))
    # Eq. 23 at full size: the two global maxima behind the first dt (a reduction over 131 072 blocks on the GPU)
    # against the oracle's wave_speeds evaluated z-plane by z-plane over the whole initial state, and dt from them
    osp = make_oracle(sub)
    cmax = vmax = 0.0
    for iz in range(nz):
        c_, v_ = _oracle_wave_speeds(osp, host.numpy(), wl, slice(iz * nx * ny, (iz + 1) * nx * ny))
        cmax, vmax = max(cmax, c_), max(vmax, v_)
    dgn = g.diagnostics()
    assert abs(dgn["c_max"] - cmax) <= 1e-14 * cmax and abs(dgn["v_max"] - vmax) <= 1e-14 * vmax, (dgn, cmax, vmax)
    dt_oracle = wl.f_cfl * wl.h / (2.0 * wl.order * (cmax + vmax))
    assert abs(dt - dt_oracle) <= 1e-14 * dt_oracle
    _report("cfg4 FULL SIZE 128^3: Eq. 23 maxima vs oracle over all cells: c_max rel %.1e, v_max rel %.1e, dt rel %.1e" % (
        abs(dgn["c_max"] - cmax) / cmax, abs(dgn["v_max"] - vmax) / vmax, abs(dt - dt_oracle) / dt_oracle))
    dt = dt_oracle                                            # the oracle patches below run on the oracle's own dt
    w1 = g.get_state().reshape(M, Vc, N)
    a1 = g.get_alpha().reshape(M, N)
    wv = host.numpy().reshape(M, Vc, nz, ny, nx)
    worst = 0.0
    for (ix, iy, iz) in [(0, 0, 0), (127, 127, 127), (127, 0, 64), (5, 120, 1), (64, 64, 64)]:
        zi = [(iz + k) % nz for k in range(-3, 4)]
        yi = [(iy + k) % ny for k in range(-3, 4)]
        xi = [(ix + k) % nx for k in range(-3, 4)]
        o = make_oracle(sub, fixed_dt=dt)
        o.set_state(np.ascontiguousarray(wv[:, :, zi][:, :, :, yi][:, :, :, :, xi]).ravel())
        assert o.step(1) == 0
        centre = (3 * 7 + 3) * 7 + 3
        ref = o.get_state().reshape(M, Vc, 343)
        cell = (iz * ny + iy) * nx + ix
        scale = np.max(np.abs(ref[0]), axis=1)
        scale[1:1 + d] = np.max(scale[1:1 + d]) + np.max(np.abs(ref[0, 0]))
        err = np.max(np.abs(w1[:, :, cell] - ref[:, :, centre]) / scale[None, :])
        aerr = np.max(np.abs(a1[:, cell] - o.get_alpha().reshape(M, 343)[:, centre]))
        worst = max(worst, err)
        assert err <= TOL_1 and aerr <= 1e-9, ((ix, iy, iz), err, aerr)
    del w1, a1
    _report("cfg4 FULL SIZE 128^3: state after 1 step on sampled cells, worst %.3e" % worst)
    g.step(49)
    d = g.diagnostics()
    assert d["steps"] == 50 and d["unphysical"] == 0
    drift = _drift(g.conserved_totals(), t0, wl)
    assert drift <= 1e-13 * 50, drift
    assert 0.0 <= d["alpha_max_seen"] < 1.0, d
    _report("cfg4 FULL SIZE 128^3: 50 steps, totals drift %.2e, max alpha %.3e, t = %.4e" % (
        drift, d["alpha_max_seen"], d["t"]))


def test_cfg4_full_size_limiter_on_is_bitwise_inactive():
    """The paper's timing workload (NS + AV + positivity limiter) at full size: on this smooth flow the
    limiter must not change a single bit (fused form: every block takes the bound-based shortcut or finds F = 1), and
    Eq. 23 must give the same time steps."""
    wl = wk.config(4)
    import torch
    host = torch.empty(wl.nvar_conserved * wl.modes * wl.ncells, dtype=torch.float64, pin_memory=True)
    wk.initial_modes_slabbed(wl, out=host.numpy())
    out = []
    for lim in (0, 1):
        g = make_gpu(wl, limiter_enable=lim)
        g.set_state(host)
        g.step(3)
        dev = torch.empty(host.numel(), dtype=torch.float64, device="cuda")
        g.get_state(dev)
        out.append((dev, g.get_time(), g.diagnostics()["unphysical"]))
        g.free()
    assert out[0][1] == out[1][1] and out[0][2] == 0 and out[1][2] == 0
    assert torch.equal(out[0][0], out[1][0])
    _report("cfg4 FULL SIZE 128^3: 3 steps with the positivity limiter on are bit-identical to limiter off")


@pytest.mark.parametrize("degree", [1, 2, 3, 4, 5, 6, 7])
def test_cfg5_full_length_exact_solution(degree):
    wl = wk.config(5, degree=degree)
    assert wl.ncell == (64, 64, 64)
    import torch
    host = torch.empty(wl.nvar_conserved * wl.modes * wl.ncells, dtype=torch.float64, pin_memory=True)
    wk.initial_modes_slabbed(wl, out=host.numpy())
    g = make_gpu(wl)
    g.set_state(host)
    t0 = g.conserved_totals()
    g.step(20)
    d = g.diagnostics()
    assert d["steps"] == 20 and d["unphysical"] == 0
    drift = _drift(g.conserved_totals(), t0, wl)
    assert drift <= 1e-13 * 20, drift
    dev = torch.empty(wl.ncells, dtype=torch.float64, device="cuda")
    full = torch.empty(host.numel(), dtype=torch.float64, device="cuda")
    g.get_state(full)
    dev.copy_(full[:wl.ncells])                              # mode 0, variable rho
    rho = dev.cpu().numpy()
    err = float(np.mean(np.abs(rho - _exact_mean_density(wl, d["t"]))))
    # spatial error of the cell means ~ (2 pi h)^(n+1)-ish plus the O(dt^3) error of SSP-RK3 over 20 small steps
    bound = {1: 2e-5, 2: 1e-6, 3: 1e-8}.get(degree, 1e-9)
    assert err < bound, (degree, err)
    _report("cfg5 FULL SIZE 64^3 degree %d: 20 steps, L1 error of mean density %.3e, totals drift %.2e" % (
        degree, err, drift))


@pytest.mark.parametrize("degree", [1, 2, 3, 5, 7])     # 5, 7: the block layout (4 and 2 cells per block)
def test_cfg5_full_size_sampled_state_after_one_step(degree):
    wl = wk.config(5, degree=degree)
    d, Vc, M, N = wl.dim, wl.dim + 2, wl.modes, wl.ncells
    w0 = wk.initial_modes_slabbed(wl)
    g = make_gpu(wl)
    g.set_state(w0)
    g.step(1)
    _, dt = g.get_time()
    nx, ny, nz = wl.ncell
    sub = replace(wl, ncell=(7, 7, 7))                       # same h and physics
    # Eq. 23 at full size against the oracle.  The wave IC depends on x+y+z only, so the cells of the
    # plane iz = 0 with iy < 8 already hold every distinct cell state of the mesh ((ix + iy) mod 64 takes all values):
    # the oracle's maxima over those 512 cells are the global ones (up to the rounding of the IC projection).
    assert wl.ic == "wave" and nx == ny == nz
    cmax, vmax = _oracle_wave_speeds(make_oracle(sub), w0, wl, slice(0, 8 * nx))
    dgn = g.diagnostics()
    assert abs(dgn["c_max"] - cmax) <= 1e-14 * cmax and abs(dgn["v_max"] - vmax) <= 1e-14 * vmax, (dgn, cmax, vmax)
    dt_oracle = wl.f_cfl * wl.h / (2.0 * wl.order * (cmax + vmax))
    assert abs(dt - dt_oracle) <= 1e-14 * dt_oracle
    dt = dt_oracle                                            # the oracle patches below run on the oracle's own dt
    w1 = g.get_state().reshape(M, Vc, N)
    wv = w0.reshape(M, Vc, nz, ny, nx)
    worst = 0.0
    for (ix, iy, iz) in [(0, 0, 0), (63, 63, 63), (63, 0, 31), (2, 61, 1), (32, 32, 32), (17, 40, 5)]:
        zi = [(iz + k) % nz for k in range(-3, 4)]
        yi = [(iy + k) % ny for k in range(-3, 4)]
        xi = [(ix + k) % nx for k in range(-3, 4)]
        o = make_oracle(sub, fixed_dt=dt)
        o.set_state(np.ascontiguousarray(wv[:, :, zi][:, :, :, yi][:, :, :, :, xi]).ravel())
        assert o.step(1) == 0
        centre = (3 * 7 + 3) * 7 + 3
        ref = o.get_state().reshape(M, Vc, 343)
        cell = (iz * ny + iy) * nx + ix
        scale = np.max(np.abs(ref[0]), axis=1)
        scale[1:1 + d] = np.max(scale[1:1 + d])
        err = np.max(np.abs(w1[:, :, cell] - ref[:, :, centre]) / scale[None, :])
        worst = max(worst, err)
        assert err <= TOL_1, ((ix, iy, iz), err)
    _report("cfg5 FULL SIZE 64^3 degree %d: state after 1 step on sampled cells, worst %.3e" % (degree, worst))
