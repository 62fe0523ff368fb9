"""Pins of the oracle's passive tracer (Eq. 40; readings T1-T3).

Eq. 40: d(c rho)/dt + div(c rho v) = div(eta rho grad c).  What the paper and the mathematics fix:
  * a uniform concentration is carried by the mass flux exactly: every term of the c rho row is c0 times the
    same term of the density row (advective, HLLC, AV), and grad c = 0 kills the diffusive flux;
  * the tracer is conserved on a periodic mesh;
  * pure advection in a uniform flow has the exact solution c(x - v t), error at order n + 1;
  * pure diffusion of c = c_bar + A sin(2 pi x) in a gas at rest decays as exp(-eta (2 pi)^2 t);
  * HLLC row: upwind limits and a stationary contact (no mass flux => no tracer flux).
"""
import math

import numpy as np
import pytest

from oracle import dg_oracle as orc
from paper_2208_11131_b200 import workloads as wk


def _with_tracer(w_flat, d, M, ncells, conc):
    """append the row c rho = conc * rho (conc: scalar or modal array [M, ncells] of c rho itself)"""
    w = w_flat.reshape(M, d + 2, ncells)
    out = np.zeros((M, d + 3, ncells))
    out[:, :d + 2] = w
    if np.isscalar(conc):
        out[:, d + 2] = conc * w[:, 0]
    else:
        out[:, d + 2] = conc
    return out.ravel()


@pytest.mark.parametrize("d,n,phys", [(2, 2, "euler"), (2, 3, "ns_av"), (3, 1, "ns_av"), (3, 2, "euler")])
def test_uniform_concentration_follows_the_mass_flux(d, n, phys):
    ncell = (4, 3) if d == 2 else (3, 2, 2)
    g = 1.4
    nu = chi = 0.01 if phys == "ns_av" else 0.0
    opt = orc.Options(av_enable=(phys == "ns_av"), tracer_enable=True, eta=0.02 if phys == "ns_av" else 0.0)
    o = orc.DGOracle(d, ncell, 0.25, n + 1, g, nu, chi, opt)
    w0, al = wk.random_smooth_modes(d, ncell, n, g, seed=7, amp=0.05, nvar_extra=1 if opt.av_enable else 0)
    c0 = 0.37
    o.set_state(_with_tracer(w0, d, o.M, o.ncells, c0))
    if opt.av_enable:
        o.set_alpha(al)
    L = o.rhs(o.w)
    scale = np.max(np.abs(L[:, :, 0]))
    assert scale > 0
    assert np.max(np.abs(L[:, :, d + 2] - c0 * L[:, :, 0])) < 2e-13 * scale
    # and the other rows do not know about the tracer
    o2 = orc.DGOracle(d, ncell, 0.25, n + 1, g, nu, chi, orc.Options(av_enable=opt.av_enable))
    o2.set_state(w0)
    if opt.av_enable:
        o2.set_alpha(al)
    L2 = o2.rhs(o2.w)
    keep = list(range(d + 2)) + ([d + 3] if opt.av_enable else [])
    np.testing.assert_array_equal(L[:, :, keep], L2)


@pytest.mark.parametrize("d", [2, 3])
def test_tracer_is_conserved(d):
    ncell = (5, 3) if d == 2 else (3, 2, 2)
    n, g = 2, 5.0 / 3.0
    opt = orc.Options(av_enable=True, tracer_enable=True, eta=0.03)
    o = orc.DGOracle(d, ncell, 0.2, n + 1, g, 0.01, 0.01, opt)
    w0, al = wk.random_smooth_modes(d, ncell, n, g, seed=11, amp=0.05, nvar_extra=1)
    rng = np.random.default_rng(5)
    conc = 0.3 * w0.reshape(o.M, d + 2, o.ncells)[:, 0] * (1.0 + 0.2 * rng.standard_normal((1, o.ncells)))
    conc[1:] += 0.01 * rng.standard_normal((o.M - 1, o.ncells))
    o.set_state(_with_tracer(w0, d, o.M, o.ncells, conc))
    o.set_alpha(al)
    L = o.rhs(o.w)
    assert abs(np.sum(L[:, 0, d + 2])) < 1e-12 * np.sum(np.abs(L[:, 0, d + 2]))
    t0 = o.conserved_totals()
    o.step(3)
    t1 = o.conserved_totals()
    assert t0.size == d + 3 and abs(t1[d + 2] - t0[d + 2]) < 1e-13 * abs(t0[d + 2])


def _project_1d_profile(o, N, n, fun):
    """modal coefficients [m*m, ncells] of a field f(x) (independent of y) on an N x 2 mesh"""
    xq, T = wk._proj_table(n, n + 3)
    m = n + 1
    out = np.zeros((m * m, o.ncells))
    for c in range(o.ncells):
        x = o.h * (c % N + 0.5 + 0.5 * xq)
        out[:m, c] = fun(x) @ T
    return out


def _tracer_amplitude(o, N):
    vals = o.evaluate(o.w, np.array([[0.0, 0.0]]))[:, 0, :]
    xc = (np.arange(o.ncells) % N + 0.5) * o.h
    c = vals[:, 4] / vals[:, 0]
    return 2.0 * np.mean(c * np.sin(2 * np.pi * xc)), 2.0 * np.mean(c * np.cos(2 * np.pi * xc))


@pytest.mark.parametrize("n", [1, 3])
def test_tracer_diffusion_decay_rate(n):
    """gas at rest, rho = P = 1, c = 0.5 + A sin(2 pi x): c_t = eta c_xx exactly => amplitude exp(-eta (2 pi)^2 t);
    pins the sign and size of eta rho grad c inside the cells and in the recovery face flux (f = 3/4 and f = 1)."""
    eta, A, g = 0.02, 0.1, 5.0 / 3.0
    N = 16 if n == 1 else 6
    o = orc.DGOracle(2, (N, 2), 1.0 / N, n + 1, g, 0.0, 0.0, orc.Options(f_cfl=0.2, tracer_enable=True, eta=eta))
    w = np.zeros((o.M, 5, o.ncells))
    w[0, 0] = 1.0
    w[0, 3] = 1.0 / (g - 1.0)
    w[:, 4] = _project_1d_profile(o, N, n, lambda x: 0.5 + A * np.sin(2 * np.pi * x))
    o.set_state(w.ravel())
    a0, _ = _tracer_amplitude(o, N)
    while o.t < 0.2:
        o.step(1)
    a1, _ = _tracer_amplitude(o, N)
    assert abs(a1 / a0 / math.exp(-eta * (2 * math.pi) ** 2 * o.t) - 1.0) < (5e-3 if n == 1 else 2e-4)
    # the gas itself stays at rest
    assert np.max(np.abs(o.w[:, :, 1:3])) < 1e-13


def test_tracer_advection_exact_solution_and_order():
    """uniform flow v = (1, 0), rho = P = 1: c(x, t) = 0.5 + 0.3 sin(2 pi (x - t)); the phase moves with the flow and
    the error falls at order n + 1 under mesh refinement (n = 2: factor ~8 per halving)."""
    g, n = 1.4, 2
    errs = []
    for N in (8, 16):
        o = orc.DGOracle(2, (N, 2), 1.0 / N, n + 1, g, 0.0, 0.0, orc.Options(f_cfl=0.1, tracer_enable=True))
        w = np.zeros((o.M, 5, o.ncells))
        w[0, 0] = 1.0
        w[0, 1] = 1.0
        w[0, 3] = 1.0 / (g - 1.0) + 0.5
        w[:, 4] = _project_1d_profile(o, N, n, lambda x: 0.5 + 0.3 * np.sin(2 * np.pi * x))
        o.set_state(w.ravel())
        while o.t < 0.1:
            o.step(1)
        xi = np.array([[-0.5, 0.0], [0.0, 0.0], [0.5, 0.0]])
        vals = o.evaluate(o.w, xi)                                   # [cell, point, var]
        xc = (np.arange(o.ncells) % N + 0.5)[:, None] * o.h + 0.5 * o.h * xi[None, :, 0]
        exact = 0.5 + 0.3 * np.sin(2 * np.pi * (xc - o.t))
        errs.append(np.max(np.abs(vals[:, :, 4] / vals[:, :, 0] - exact)))
    assert errs[0] < 5e-3 and errs[0] / errs[1] > 5.0


def test_hllc_tracer_row():
    g, d = 1.4, 2
    def cons(rho, v, p, c):
        return np.array([rho, rho * v[0], rho * v[1], p / (g - 1) + 0.5 * rho * (v[0] ** 2 + v[1] ** 2), c * rho])
    # consistency
    u = cons(1.3, (0.4, -0.2), 0.9, 0.6)
    np.testing.assert_allclose(orc.hllc_flux(u, u, 0, d, g), orc.euler_flux(u, 0, d, g), rtol=1e-14)
    # supersonic to the right / to the left: pure upwinding
    uL, uR = cons(1.0, (3.0, 0.1), 1.0, 0.2), cons(0.8, (2.8, 0.0), 0.9, 0.9)
    np.testing.assert_array_equal(orc.hllc_flux(uL, uR, 0, d, g), orc.euler_flux(uL, 0, d, g))
    uL, uR = cons(1.0, (-3.0, 0.1), 1.0, 0.2), cons(0.8, (-2.8, 0.0), 0.9, 0.9)
    np.testing.assert_array_equal(orc.hllc_flux(uL, uR, 0, d, g), orc.euler_flux(uR, 0, d, g))
    # stationary contact with a jump in density and concentration: no mass flux, no tracer flux
    uL, uR = cons(1.0, (0.0, 0.0), 1.0, 0.1), cons(0.25, (0.0, 0.0), 1.0, 0.8)
    F = orc.hllc_flux(uL, uR, 0, d, g)
    assert abs(F[0]) < 1e-15 and abs(F[4]) < 1e-15
    # subsonic: tracer flux = upwind concentration (by the sign of S*) times the HLLC mass flux
    uL, uR = cons(1.0, (0.3, 0.0), 1.0, 0.2), cons(0.9, (0.25, 0.0), 0.95, 0.7)
    F = orc.hllc_flux(uL, uR, 0, d, g)
    assert F[0] > 0 and abs(F[4] - 0.2 * F[0]) < 1e-15
    uL, uR = cons(1.0, (-0.3, 0.0), 1.0, 0.2), cons(0.9, (-0.25, 0.0), 0.95, 0.7)
    F = orc.hllc_flux(uL, uR, 0, d, g)
    assert F[0] < 0 and abs(F[4] - 0.7 * F[0]) < 1e-15


def test_limiter_scales_the_tracer_row_too():
    """Eq. 47 multiplies the higher modes of ALL fields ("to all fields and not just the density")."""
    d, n, g = 2, 2, 1.4
    o = orc.DGOracle(d, (2, 2), 0.5, n + 1, g, 0.0, 0.0, orc.Options(tracer_enable=True, limiter_enable=True))
    w = np.zeros((o.ncells, o.M, o.V))
    w[:, 0, 0] = 1.0
    w[:, 0, 3] = 2.5
    w[:, 0, 4] = 0.5
    w[0, 1, 0] = 0.9            # rho dips below zero at a face of cell 0
    w[0, 1, 4] = 0.05
    w[0, 2, 4] = 0.02
    out = o.positivity_limit(w)
    f = out[0, 1, 0] / w[0, 1, 0]
    assert 0.0 < f < 1.0
    np.testing.assert_allclose(out[0, 1:, 4], f * w[0, 1:, 4], rtol=1e-15)
    np.testing.assert_array_equal(out[1:], w[1:])
    np.testing.assert_array_equal(out[0, 0], w[0, 0])
