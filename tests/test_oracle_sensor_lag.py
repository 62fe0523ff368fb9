"""Pin of the sensor book-keeping inside DGOracle.step (reading A15).

PAPER.md:394-397: the wiggle source of Eq. 45 is "based on the time derivatives of the weights of the previous
timestep"; "two scalar quantities per cell".  Reading A15: per cell the pair (S^K, G^K = d ln S^K / dt) is
formed ONCE per step from (w^n, L(w^n)), i.e. from the first Runge-Kutta stage, is NOT used by the step that forms it
(all its stages still see the pair of the step before; zero during the very first step), and replaces the old pair
only after the last stage.

`sensor()` (Eq. 42 = Eq. 41, finite-difference d ln S/dt) and the use of a given (S, G) by `rhs()` are pinned
elsewhere (test_oracle_physics.py, test_oracle_bruteforce.py).  Here the bookkeeping in `step()` is pinned against
the sums of Eq. 42 / 45 written out as plain loops and against a hand-rolled Shu-Osher RK3 built from
`rhs()` alone, and the plausible slips (commit before stage 2; form the pair from the last stage; use the fresh pair
in the step that forms it) are shown to give measurably different results, so that any of them would fail.
"""
import numpy as np
import pytest

from oracle import dg_oracle as orc
from paper_2208_11131_b200 import workloads as wk


def _make(d, ncell, n, f_w=0.2, basis="tensor"):
    gamma = 1.4 if d == 2 else 5.0 / 3.0
    opt = orc.Options(f_cfl=0.3, av_enable=True, f_w=f_w, basis=basis)
    return orc.DGOracle(d, ncell, 1.0 / ncell[0], n + 1, gamma, 0.0, 0.0, opt), gamma


def _rough(d, ncell, n, gamma):
    seed = 5 if d == 2 else 7          # seeds for which the wiggle source is on in some cells and off in others
    w0, al = wk.random_smooth_modes(d, ncell, n, gamma, seed=seed, amp=0.08, nvar_extra=1)
    return w0, al


def _sensor_by_loops(o, w, L, d, n, total_degree=False):
    """Eq. 42: S = sum_{top} w_l^2 / sum_{all} w_l^2 on the density row; Eq. 45: G = d ln S / dt with the weights'
    time derivatives L: 2 sum_top w w' / sum_top w^2 - 2 sum_all w w' / sum_all w^2.  Top modes: highest degree n on
    at least one axis (tensor basis, reading A14) or l_x+l_y(+l_z) = n (total-degree basis)."""
    m = n + 1
    nc, M = w.shape[0], w.shape[1]
    S = np.zeros(nc)
    G = np.zeros(nc)
    for c in range(nc):
        A = B = dA = dB = 0.0
        for l in range(M):
            ls = [(l // m ** a) % m for a in range(d)]
            if total_degree and sum(ls) > n:
                continue
            top = (sum(ls) == n) if total_degree else (max(ls) == n)
            r, rd = w[c, l, 0], L[c, l, 0]
            B += r * r
            dB += 2.0 * r * rd
            if top:
                A += r * r
                dA += 2.0 * r * rd
        S[c] = A / B
        G[c] = dA / A - dB / B if A > 0.0 else 0.0
    return S, G


def _rk3_frozen(o, w, S, G, refresh_after_stage=None, refreshed=None):
    """Shu-Osher SSP-RK3 from o.rhs with the sensor pair held at (S, G); optionally (a deliberate slip)
    switch to `refreshed` after the given stage."""
    o.sensor_S, o.sensor_G = S.copy(), G.copy()
    dt = o.timestep(w)
    L0 = o.rhs(w)
    u1 = w + dt * L0
    if refresh_after_stage == 1:
        o.sensor_S, o.sensor_G = refreshed
    L1 = o.rhs(u1)
    u2 = 0.75 * w + 0.25 * (u1 + dt * L1)
    if refresh_after_stage == 2:
        o.sensor_S, o.sensor_G = refreshed
    L2 = o.rhs(u2)
    u3 = (1.0 / 3.0) * w + (2.0 / 3.0) * (u2 + dt * L2)
    return u3, L0, L2, u2, dt


CASES = [(2, (4, 3), 2, "tensor"), (2, (3, 3), 3, "total_degree"), (3, (3, 2, 2), 1, "tensor")]


@pytest.mark.parametrize("d,ncell,n,basis", CASES)
def test_first_step_ignores_the_wiggle_source_and_later_steps_do_not(d, ncell, n, basis):
    """Step 0 sees (S, G) = 0 <= S_onset, hence W = 0 whatever f_w is; from step 1 on f_w matters."""
    oa, gamma = _make(d, ncell, n, f_w=0.2, basis=basis)
    ob, _ = _make(d, ncell, n, f_w=7.0, basis=basis)
    w0, al = _rough(d, ncell, n, gamma)
    for o in (oa, ob):
        o.set_state(w0)
        o.set_alpha(0.3 * al)
        assert o.step(1) == 0
    assert np.array_equal(oa.w, ob.w)
    assert np.array_equal(oa.sensor_S, ob.sensor_S) and np.array_equal(oa.sensor_G, ob.sensor_G)
    for o in (oa, ob):
        assert o.step(1) == 0
    assert np.max(np.abs(oa.w[:, :, -1] - ob.w[:, :, -1])) > 1e-6      # the alpha rows now differ


@pytest.mark.parametrize("d,ncell,n,basis", CASES)
def test_step_forms_the_pair_from_stage_one_and_uses_it_one_step_later(d, ncell, n, basis):
    td = basis == "total_degree"
    o, gamma = _make(d, ncell, n, basis=basis)
    w0, al = _rough(d, ncell, n, gamma)
    o.set_state(w0)
    o.set_alpha(0.3 * al)
    wn = o.w.copy()
    assert np.all(o.sensor_S == 0.0) and np.all(o.sensor_G == 0.0)
    Ln = o.rhs(wn)                                   # stage 1 of step 0 (sensor pair still zero)
    S0, G0 = _sensor_by_loops(o, wn, Ln, d, n, td)
    assert o.step(1) == 0
    # (1) after step 0 the stored pair is Eq. 42 / 45 of (w^n, L(w^n))
    assert np.allclose(o.sensor_S, S0, rtol=1e-12, atol=0.0)
    assert np.allclose(o.sensor_G, G0, rtol=1e-10, atol=1e-12 * np.max(np.abs(G0)))
    # the case is not degenerate: the wiggle source is on in some cells and off in others
    s_onset = o.opt.s_onset0 / (n + 1) ** 2
    on = (S0 > s_onset) & (G0 > 0.0)
    assert 0 < np.count_nonzero(on) < on.size
    # step 0 itself used the zero pair
    twin, _ = _make(d, ncell, n, basis=basis)
    u_first, *_ = _rk3_frozen(twin, wn, np.zeros_like(S0), np.zeros_like(G0))
    assert np.max(np.abs(o.w - u_first)) <= 1e-13 * np.max(np.abs(u_first))

    # (2) step 1 = RK3 with the pair frozen at (S0, G0) through all three stages
    w1 = o.w.copy()
    u_ok, L0, L2, u2, dt = _rk3_frozen(twin, w1, S0, G0)
    S1, G1 = _sensor_by_loops(o, w1, L0, d, n, td)           # what step 1 must leave behind: from ITS stage 1
    assert o.step(1) == 0
    scale = np.max(np.abs(u_ok), axis=(0, 1))
    err = np.max(np.abs(o.w - u_ok), axis=(0, 1)) / scale
    assert np.all(err <= 1e-13), err
    assert o.last_dt == dt
    assert np.allclose(o.sensor_S, S1, rtol=1e-12, atol=0.0)
    assert np.allclose(o.sensor_G, G1, rtol=1e-10, atol=1e-12 * np.max(np.abs(G1)))

    # (3) the slips this pin is there to catch all land measurably elsewhere
    fresh = (S1.copy(), G1.copy())
    for stage in (1, 2):                                     # committing the new pair before stage 2 / stage 3
        u_bad, *_ = _rk3_frozen(twin, w1, S0, G0, refresh_after_stage=stage, refreshed=fresh)
        assert np.max(np.abs(u_bad[:, :, -1] - u_ok[:, :, -1])) > 1e-9 * scale[-1]
    u_bad, *_ = _rk3_frozen(twin, w1, S1, G1)                # using the fresh pair in the step that forms it
    assert np.max(np.abs(u_bad[:, :, -1] - u_ok[:, :, -1])) > 1e-9 * scale[-1]
    S_last, G_last = _sensor_by_loops(o, u2, L2, d, n, td)   # forming the pair from the last stage instead
    assert np.max(np.abs(S_last - S1)) > 1e-9 * np.max(S1)
    assert np.max(np.abs(G_last - G1)) > 1e-9 * np.max(np.abs(G1))
