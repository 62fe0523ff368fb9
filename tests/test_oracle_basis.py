"""Pins P1, P2, P7, T1, T2, T3: basis, quadrature, mass matrix, recovery, memory model.
CPU only.  Each test pins oracle/dg_oracle.py against the paper or against a library routine it does not use."""
import math
import os

import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

from oracle import dg_oracle as orc
from paper_2208_11131_b200 import workloads as wk

GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.mark.parametrize("n", range(0, 8))
def test_p1_orthonormality_and_nodes(n):
    """PAPER.md:125 (Eq. 13): int P_l P_m = 2 delta; (n+1)-point Gauss exact to degree 2n+1 => V^T W V = 2I."""
    m = n + 1
    x, g = orc.gauss_legendre(m)
    xr, gr = npleg.leggauss(m)                       # library nodes, independent of the oracle's Newton
    assert np.allclose(x, xr, atol=1e-15) and np.allclose(g, gr, atol=1e-15)
    assert abs(g.sum() - 2.0) < 1e-14
    P, dP = orc.legendre_normalised(n, x)
    assert np.allclose(P @ np.diag(g) @ P.T, 2.0 * np.eye(m), atol=1e-13)
    Pp, _ = orc.legendre_normalised(n, np.array(1.0))
    Pm, _ = orc.legendre_normalised(n, np.array(-1.0))
    l = np.arange(m)
    assert np.allclose(Pp, np.sqrt(2 * l + 1)) and np.allclose(Pm, (-1.0) ** l * np.sqrt(2 * l + 1))
    # derivative against the library's closed form
    for ll in range(m):
        c = np.zeros(ll + 1)
        c[ll] = math.sqrt(2 * ll + 1)
        assert np.allclose(dP[ll], npleg.legval(x, npleg.legder(c)) if ll else 0.0, atol=1e-12)


def test_t6_p0_constant_p1_linear():
    """P_0 = 1, P_1 = sqrt(3) xi."""
    x = np.linspace(-1, 1, 7)
    P, _ = orc.legendre_normalised(1, x)
    assert np.allclose(P[0], 1.0) and np.allclose(P[1], math.sqrt(3.0) * x)


@pytest.mark.parametrize("d,n", [(2, 2), (2, 4), (3, 1), (3, 3)])
def test_p2_mass_matrix_projection_identity(d, n):
    """PAPER.md:100 (Eq. 9): int_K phi_l phi_m = delta |K|  =>  projecting (Eq. 11, done by the library-based
    workloads module) a degree-<=n polynomial and expanding it with the oracle (Eq. 6/21) is the identity.
    Also pins the mode ordering (x fastest) and the C-ABI layout conversion."""
    ncell = (3, 2, 2)[:d]
    h = 0.25
    m = n + 1
    o = orc.DGOracle(d, ncell, h, n + 1, 1.4)
    # mass matrix by the oracle's own volume rule
    Mm = o.Phi.T @ np.diag(o.gvol) @ o.Phi * (h / 2.0) ** d
    assert np.allclose(Mm, np.eye(m ** d) * h ** d, atol=1e-13)
    # polynomial with distinct per-axis powers: x^n + 2 y^(n-1) (+ 3 z^n) + x y
    def poly(X):
        r = X[0] ** n + 2.0 * X[1] ** max(n - 1, 0) + (X[0] * X[1] if n >= 1 else 0.0)
        if d == 3:
            r = r + 3.0 * X[2] ** n - (X[1] * X[2] if n >= 1 else 0.0)
        return r
    wl = wk.Workload("poly", d, ncell, h, n, 1.4, ic="uniform")
    nq = n + 3
    xq, T = wk._proj_table(n, nq)
    # project by hand through the library table, per cell
    w = np.zeros((m ** d, d + 2, o.ncells))
    rng = np.random.default_rng(1)
    xi = rng.uniform(-1, 1, size=(5, d))
    for c in range(o.ncells):
        idx = [c % ncell[0], (c // ncell[0]) % ncell[1]] + ([c // (ncell[0] * ncell[1])] if d == 3 else [])
        xc = [h * (i + 0.5) for i in idx]
        grids = np.meshgrid(*[xc[a] + 0.5 * h * xq for a in range(d)][::-1], indexing="ij")[::-1]
        A = poly(grids)
        if d == 2:
            W = np.einsum("qr,ql,rk->lk", A, T, T)          # [ly, lx]
        else:
            W = np.einsum("pqr,pl,qk,rj->lkj", A, T, T, T)  # [lz, ly, lx]
        w[:, 0, c] = W.ravel()
    o.set_state(np.where(np.arange(d + 2)[None, :, None] == 0, w, 1.0).ravel())
    vals = o.evaluate(o.w, xi)[:, :, 0]
    for c in range(o.ncells):
        idx = [c % ncell[0], (c // ncell[0]) % ncell[1]] + ([c // (ncell[0] * ncell[1])] if d == 3 else [])
        X = [h * (idx[a] + 0.5) + 0.5 * h * xi[:, a] for a in range(d)]
        assert np.allclose(vals[c], poly(X), atol=1e-12)
    # layout round trip
    assert np.array_equal(o.get_state().reshape(m ** d, d + 2, -1)[:, 0], w[:, 0])


def test_t1_table1_memory():
    """PAPER.md:744-757 Table 1 with Eq. 62: pins the p-vs-degree reading and the RK-stage rule f_t."""
    unit = {"MB": 2.0 ** 20, "GB": 2.0 ** 30, "TB": 2.0 ** 40}
    rows = [l.split() for l in open(os.path.join(GOLD, "table1_memory.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 10
    for Nc, p, val, u in rows:
        got = 8.0 * orc.min_memory_doubles(int(p), 3, int(Nc)) / unit[u]
        assert abs(got - float(val)) <= 0.006 * float(val) + 1e-9, (Nc, p, got, val)


def _gold(name):
    return {l.split()[0]: float(l.split()[1]) for l in open(os.path.join(GOLD, name)) if l.strip() and l[0] != "#"}


def test_t3_mode_count_ratios():
    """p^3 / N^3D(p) = 2 (p=2), 3.2 (p=4), > 4.5 (p=10), p the ORDER there (= n+1)."""
    g = _gold("recovery_eq36.txt")
    N3 = lambda n: (n + 1) * (n + 2) * (n + 3) // 6
    assert abs(2 ** 3 / N3(1) - g["ratio_p2"]) < 1e-12
    assert abs(4 ** 3 / N3(3) - g["ratio_p4"]) < 1e-12
    assert 10 ** 3 / N3(9) > g["ratio_p10_min"]


def test_t2_recovery_eq36_n0():
    """PAPER.md:301-303 (Eq. 36): n = 0, f = 3/4 => grad u~ = (u+ - u-)/h."""
    g = _gold("recovery_eq36.txt")
    Rm, Rp, Gm, Gp = orc.recovery_vectors(0, 0.75)
    assert abs(Gp[0] - g["grad_coeff_n0_f34"]) < 1e-13 and abs(Gm[0] + g["grad_coeff_n0_f34"]) < 1e-13
    assert abs(Rm[0] - 0.5) < 1e-13 and abs(Rp[0] - 0.5) < 1e-13
    assert orc.recovery_fraction(2) == 0.75 and orc.recovery_fraction(3) == 1.0


@pytest.mark.parametrize("n", range(0, 8))
@pytest.mark.parametrize("f", [0.75, 1.0])
def test_p7_recovery_reproduces_polynomials(n, f):
    """the recovered polynomial has degree n+1 over K*; a single global polynomial of
    degree <= n sampled in both cells must be reproduced exactly at the interface, value and slope.
    Symmetries: A+ = (-1)^(m+l) A-, R+_m = (-1)^m R-_m, G+_m = (-1)^(m+1) G-_m."""
    Am, Ap = orc.overlap_integrals(n, f)
    sgn = (-1.0) ** (np.arange(n + 1)[:, None] + np.arange(n + 2)[None, :])
    assert np.allclose(Ap, sgn * Am, atol=1e-13)
    Rm, Rp, Gm, Gp = orc.recovery_vectors(n, f)
    s = (-1.0) ** np.arange(n + 1)
    assert np.allclose(Rp, s * Rm, atol=1e-13) and np.allclose(Gp, -s * Gm, atol=1e-13)
    # global polynomial q(X) in physical coordinate X (interface at X = 0, cells of width h)
    h = 0.37
    rng = np.random.default_rng(n)
    coef = rng.standard_normal(n + 1)
    q = np.polynomial.Polynomial(coef)
    xg, gg = npleg.leggauss(n + 2)
    lnorm = np.sqrt(2.0 * np.arange(n + 1) + 1.0)
    def cell_modes(xc):
        vals = q(xc + 0.5 * h * xg)
        return 0.5 * (gg * vals) @ (npleg.legvander(xg, n) * lnorm)
    wL, wR = cell_modes(-0.5 * h), cell_modes(+0.5 * h)
    assert abs(Rm @ wL + Rp @ wR - q(0.0)) < 1e-11
    assert abs((Gm @ wL + Gp @ wR) / h - q.deriv()(0.0)) < 1e-10 / h
    # one degree higher is recovered too when f = 1 (2(n+1) data for n+2 unknowns: L2 projection onto
    # degree n+1 of a degree n+1 polynomial is exact only if both cells hold its exact L2 projections) --
    # not claimed by the paper, so not asserted.


def test_recovery_known_integrals_f1_n1():
    """Hand-evaluated overlap integrals for f = 1 (Eq. 33):
       A-_{0,0} = int_-1^0 1 dx = 1;  A-_{0,1} = int_-1^0 sqrt(3) x dx = -sqrt(3)/2;
       A-_{1,0} = int_-1^0 sqrt(3)(2x+1) dx = 0;  A-_{1,1} = int_-1^0 3 (2x+1) x dx = 1/2."""
    Am, Ap = orc.overlap_integrals(1, 1.0)
    assert abs(Am[0, 0] - 1.0) < 1e-14 and abs(Am[0, 1] + math.sqrt(3) / 2) < 1e-14
    assert abs(Am[1, 0]) < 1e-14 and abs(Am[1, 1] - 0.5) < 1e-14
    assert abs(Ap[0, 1] - math.sqrt(3) / 2) < 1e-14
