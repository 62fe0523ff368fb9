"""GPU parity of the passive tracer row (Eq. 40) against the oracle, through
the C-ABI (dg_options.tracer_enable / eta, dg_tracer_total): dw/dt term level and RK steps, every physics variant, both
stage-kernel families (register tiles m = 2..5, pencil sweeps m = 1 and m >= 6 incl. the block layout), limiter on."""
import numpy as np
import pytest

from paper_2208_11131_b200 import workloads as wk
from parity_util import make_gpu, make_oracle

pytestmark = pytest.mark.gpu


def _wl(d, ncell, n, phys, f_cfl=0.3):
    return wk.Workload("rand", d, tuple(ncell), 1.0 / ncell[0], n, 1.4 if d == 2 else 5.0 / 3.0,
                       nu=0.01 if "ns" in phys else 0.0, chi=0.02 if "ns" in phys else 0.0,
                       av=("av" in phys), f_cfl=f_cfl)


def _state_with_tracer(wl, seed=13, amp=0.04):
    """random smooth hydrodynamic state + a tracer row c rho with c in (0.2, 0.8) varying from cell to cell and inside"""
    d, M = wl.dim, wl.modes
    w0, al = wk.random_smooth_modes(d, wl.ncell, wl.degree, wl.gamma, seed=seed, amp=amp, nvar_extra=1 if wl.av else 0)
    w = w0.reshape(M, d + 2, -1)
    rng = np.random.default_rng(seed + 1)
    out = np.zeros((M, d + 3, w.shape[2]))
    out[:, :d + 2] = w
    out[:, d + 2] = w[:, 0] * (0.5 + 0.3 * np.tanh(rng.standard_normal((1, w.shape[2]))))
    if M > 1:
        out[1:, d + 2] += 0.2 * amp * rng.standard_normal((M - 1, w.shape[2])) / np.arange(2, M + 1)[:, None]
    return out.ravel(), al


def _pair(wl, eta, **kw):
    w0, al = _state_with_tracer(wl)
    o = make_oracle(wl, tracer_enable=True, eta=eta, **kw)
    g = make_gpu(wl, tracer_enable=1, eta=eta, **{k: (1 if v is True else v) for k, v in kw.items()})
    o.set_state(w0)
    g.set_state(w0)
    if wl.av:
        o.set_alpha(al)
        g.set_alpha(al)
    return o, g


def _scales(L, wl):
    Vc = wl.dim + 3
    s = np.max(np.abs(L.reshape(wl.modes, Vc, -1)), axis=(0, 2))
    s[1:1 + wl.dim] = np.max(s[1:1 + wl.dim])
    return np.maximum(s, 1e-300)


CASES = [(2, (5, 3), n, ph, eta) for n in (0, 1, 3, 5) for ph, eta in (("euler", 0.0), ("euler", 0.02), ("ns_av", 0.02))] + \
        [(3, (3, 2, 2), n, ph, eta) for n in (1, 2, 3) for ph, eta in (("euler", 0.0), ("ns", 0.03), ("ns_av", 0.02))] + \
        [(3, (9, 4, 3), 3, "ns_av", 0.02), (3, (2, 2, 3), 4, "av", 0.01), (3, (3, 2, 3), 5, "euler", 0.02),
         (3, (2, 2, 2), 7, "ns", 0.02), (3, (2, 2, 2), 6, "ns_av", 0.02), (2, (37, 3), 3, "ns_av", 0.02)]


@pytest.mark.parametrize("d,ncell,n,phys,eta", CASES)
def test_tracer_rhs_parity(d, ncell, n, phys, eta):
    wl = _wl(d, ncell, n, phys)
    o, g = _pair(wl, eta)
    if wl.av:
        assert o.step(1) == 0
        g.step(1)
    L = o.rhs(o.w)
    Vc = d + 3
    Lo = np.ascontiguousarray(L[:, :, :Vc].transpose(1, 2, 0)).ravel()
    Lg, _ = g.eval_rhs(with_alpha=True)
    err = np.max(np.abs(Lg - Lo).reshape(wl.modes, Vc, -1), axis=(0, 2)) / _scales(Lo, wl)
    assert np.all(err < 5e-12), err


@pytest.mark.parametrize("d,ncell,n,phys,eta,lim", [
    (2, (6, 4), 2, "ns_av", 0.02, False), (3, (4, 3, 2), 3, "ns_av", 0.02, False), (3, (4, 3, 2), 3, "euler", 0.0, True),
    (3, (2, 2, 3), 6, "euler", 0.02, False), (2, (5, 4), 0, "euler", 0.0, False), (3, (3, 2, 2), 2, "ns_av", 0.01, True)])
def test_tracer_step_parity_and_conservation(d, ncell, n, phys, eta, lim):
    wl = _wl(d, ncell, n, phys)
    kw = {"limiter_enable": True} if lim else {}
    o, g = _pair(wl, eta, **kw)
    t0 = g.tracer_total()
    assert abs(t0 - o.conserved_totals()[d + 2]) < 1e-13 * abs(t0)
    for steps, tol in ((1, 1e-12), (9, 1e-9)):
        assert o.step(steps) == 0
        g.step(steps)
        a = g.get_state().reshape(wl.modes, d + 3, -1)
        b = o.get_state().reshape(wl.modes, d + 3, -1)
        scale = np.max(np.abs(b[0]), axis=1)
        scale[1:1 + d] = np.max(scale[1:1 + d]) + np.max(np.abs(b[0, 0]))
        err = np.max(np.abs(a - b), axis=(0, 2)) / scale
        assert np.all(err < tol), (steps, err)
    assert abs(g.tracer_total() - t0) < 1e-13 * 10 * abs(t0)
    tot = g.conserved_totals()
    assert tot.size == d + 2 and np.all(np.abs(tot - o.conserved_totals()[:d + 2]) < 1e-12 * np.max(np.abs(tot)))


def test_tracer_off_is_bitwise_the_plain_solver():
    """a uniform concentration changes nothing in the hydrodynamic rows (same kernels + one passive row)"""
    wl = _wl(3, (4, 3, 2), 3, "ns_av")
    w0, al = wk.random_smooth_modes(3, wl.ncell, 3, wl.gamma, seed=3, amp=0.04, nvar_extra=1)
    g0 = make_gpu(wl)
    g0.set_state(w0)
    g0.set_alpha(al)
    g0.step(3)
    w = w0.reshape(wl.modes, 5, -1)
    wt = np.zeros((wl.modes, 6, w.shape[2]))
    wt[:, :5] = w
    wt[:, 5] = 0.25 * w[:, 0]
    g1 = make_gpu(wl, tracer_enable=1, eta=0.0)
    g1.set_state(wt.ravel())
    g1.set_alpha(al)
    g1.step(3)
    a = g1.get_state().reshape(wl.modes, 6, -1)
    b = g0.get_state().reshape(wl.modes, 5, -1)
    np.testing.assert_array_equal(a[:, :5], b)
    assert np.max(np.abs(a[:, 5] - 0.25 * b[:, 0])) < 1e-14


def test_tracer_bad_arguments():
    from paper_2208_11131_b200 import dg
    wl = _wl(2, (4, 4), 1, "euler")
    with pytest.raises(dg.DGError):
        make_gpu(wl, tracer_enable=1, eta=-1.0)
    g = make_gpu(wl)
    with pytest.raises(dg.DGError):
        g.tracer_total()
    g1 = make_gpu(wl, tracer_enable=1)
    with pytest.raises(dg.DGError):
        g1.set_state(np.zeros(wl.modes * 4 * wl.ncells))     # count must include the tracer row
