"""Pin P11: the matrix-based oracle RHS against a literal nested-loop evaluation of
Eq. 20 on 2x2 (2D) and 2x2x2 (3D) periodic meshes, where the left and the right
neighbour of a cell are the same cell (also a wrap-logic test).  The brute force below shares nothing with
oracle/dg_oracle.py: Legendre values come from numpy.polynomial.legendre, the recovery is done by directly
L2-projecting the two cell polynomials onto degree n+1 over K* (Eq. 27-32) with Gauss quadrature instead of
through the overlap matrices A+-, and all physics is retyped in scalar form from Eq. 1-5, 24, 37-39, 43-46.
CPU only; python loops, so tiny cases only."""
import itertools
import math

import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

from oracle import dg_oracle as orc
from paper_2208_11131_b200 import workloads as wk


def P(l, x, der=0):
    c = np.zeros(l + 1)
    c[l] = math.sqrt(2 * l + 1)
    for _ in range(der):
        c = npleg.legder(c)
    return float(npleg.legval(x, c))


class Brute:
    def __init__(self, d, n, h, gamma, nu, chi, av, opts, w, sensor=None, ncell=None):
        self.ncell = ncell if ncell is not None else (2,) * d
        self.d, self.n, self.m, self.h, self.g = d, n, n + 1, h, gamma
        self.nu, self.chi, self.av, self.o = nu, chi, av, opts
        self.w = w                       # [cell, mode, var]
        self.Vc = d + 2
        self.xg, self.gg = npleg.leggauss(self.m)
        self.f = 0.75 if n <= 2 else 1.0
        self.sensor = sensor
        self._ff = {}                    # face fluxes do not depend on the test mode: evaluate each once

    def nbr(self, c, a, s):              # periodic wrap, cell = (iz*Ny + iy)*Nx + ix
        idx = [c % self.ncell[0], (c // self.ncell[0]) % self.ncell[1]]
        if self.d == 3:
            idx.append(c // (self.ncell[0] * self.ncell[1]))
        idx[a] = (idx[a] + s) % self.ncell[a]
        c2 = idx[0] + self.ncell[0] * idx[1]
        return c2 + (self.ncell[0] * self.ncell[1] * idx[2] if self.d == 3 else 0)

    def ls(self, mode):
        return [(mode // self.m ** a) % self.m for a in range(self.d)]

    def phi(self, mode, xi, der_axis=None):
        r = 1.0
        for a, l in enumerate(self.ls(mode)):
            r *= P(l, xi[a], 1 if a == der_axis else 0)
        return r

    def u(self, c, xi, der_axis=None):
        """u^K(xi) (Eq. 21) or its PHYSICAL derivative d/dx_axis = (2/h) d/dxi_axis, all variables."""
        out = np.zeros(self.w.shape[2])
        for mode in range(self.m ** self.d):
            out += self.w[c, mode] * self.phi(mode, xi, der_axis)
        return out * ((2.0 / self.h) if der_axis is not None else 1.0)

    # ---- physics, scalar ----
    def prim(self, u):
        rho = u[0]
        v = u[1:1 + self.d] / rho
        p = (self.g - 1.0) * (u[1 + self.d] - 0.5 * rho * float(v @ v))
        return rho, v, p

    def feuler(self, u, a):
        rho, v, p = self.prim(u)
        F = np.zeros(self.Vc)
        F[0] = rho * v[a]
        for b in range(self.d):
            F[1 + b] = rho * v[a] * v[b] + (p if a == b else 0.0)
        F[1 + self.d] = (u[1 + self.d] + p) * v[a]
        return F

    def hllc(self, uL, uR, a):
        rl, vl, pl = self.prim(uL)
        rr, vr, pr = self.prim(uR)
        cl, cr = math.sqrt(self.g * pl / rl), math.sqrt(self.g * pr / rr)
        SL = min(vl[a] - cl, vr[a] - cr)
        SR = max(vl[a] + cl, vr[a] + cr)
        if SL >= 0:
            return self.feuler(uL, a)
        if SR <= 0:
            return self.feuler(uR, a)
        Ss = (pr - pl + rl * vl[a] * (SL - vl[a]) - rr * vr[a] * (SR - vr[a])) / (rl * (SL - vl[a]) - rr * (SR - vr[a]))
        def star(u, r, v, p, S):
            fac = r * (S - v[a]) / (S - Ss)
            Us = np.zeros(self.Vc)
            Us[0] = fac
            for b in range(self.d):
                Us[1 + b] = fac * (Ss if b == a else v[b])
            Us[1 + self.d] = fac * (u[1 + self.d] / r + (Ss - v[a]) * (Ss + p / (r * (S - v[a]))))
            return Us
        if Ss >= 0:
            return self.feuler(uL, a) + SL * (star(uL, rl, vl, pl, SL) - uL)
        return self.feuler(uR, a) + SR * (star(uR, rr, vr, pr, SR) - uR)

    def fns(self, u, grad, a):
        """F_NS column a (Eq. 38-39): grad[b] = d u / d x_b (conserved variables)."""
        d = self.d
        rho, v, p = self.prim(u)
        dv = np.array([[(grad[b][1 + c] - v[c] * grad[b][0]) / rho for c in range(d)] for b in range(d)])  # dv[b][c] = d_b v_c
        div = sum(dv[b][b] for b in range(d))
        F = np.zeros(self.Vc)
        for b in range(d):
            Pi = self.nu * rho * (dv[a][b] + dv[b][a] - (2.0 / 3.0 * div if a == b else 0.0))
            F[1 + b] = Pi
            F[1 + d] += v[b] * Pi
        e = u[1 + d]
        uth_a = grad[a][1 + d] / rho - e * grad[a][0] / rho ** 2 - sum(v[c] * dv[a][c] for c in range(d))
        F[1 + d] += self.chi * (self.g - 1.0) * rho * uth_a
        return F

    def eps(self, u, alpha):
        rho, v, p = self.prim(u)
        return min(max(alpha, 0.0), self.o.alpha_max) * math.sqrt(self.g * p / rho) * self.h / (self.n + 1)

    # ---- recovery by direct L2 projection over K* (Eq. 27-32) ----
    def recover(self, fL, fR):
        """fL(xi), fR(xi): the two cells' polynomials along the normal in their own local coordinate.
        Returns (value, d/dx) of the degree-(n+1) L2 projection over K* at the interface."""
        f, n = self.f, self.n
        xq, gq = npleg.leggauss(n + 3)
        val = der = 0.0
        for l in range(n + 2):
            q = 0.0
            for x, g in zip(xq, gq):
                xm, xp = 0.5 * (x - 1.0), 0.5 * (x + 1.0)          # [-1,0], [0,1]
                q += 0.5 * g * (fL(2 * f * xm + 1.0) * P(l, xm) + fR(2 * f * xp - 1.0) * P(l, xp))
            q *= 0.5                                                  # 1/2 int u~ P_l over [-1,1]
            val += q * P(l, 0.0)
            der += q * P(l, 0.0, 1) / (f * self.h)
        return val, der

    def face_flux(self, cL, cR, a, xit):
        """G^_a at transverse reference point xit (list of d-1 coords) between cL (left) and cR (right)."""
        key = (cL, cR, a, tuple(xit))
        if key in self._ff:
            return self._ff[key]
        d = self.d
        def full(x_a):
            xi = list(xit)
            xi.insert(a, x_a)
            return xi
        uL, uR = self.u(cL, full(+1.0)), self.u(cR, full(-1.0))
        F = self.hllc(uL[:self.Vc], uR[:self.Vc], a)
        if self.nu > 0 or self.chi > 0 or self.av:
            nv = self.w.shape[2]
            ut = np.zeros(nv)
            grad = [np.zeros(nv) for _ in range(d)]
            for var in range(nv):
                ut[var], grad[a][var] = self.recover(lambda x: self.u(cL, full(x))[var], lambda x: self.u(cR, full(x))[var])
                for t in range(d):
                    if t != a:
                        grad[t][var], _ = self.recover(lambda x: self.u(cL, full(x), t)[var],
                                                       lambda x: self.u(cR, full(x), t)[var])
            if self.nu > 0 or self.chi > 0:
                F = F - self.fns(ut[:self.Vc], [g[:self.Vc] for g in grad], a)
            if self.av:
                F = F - self.eps(ut[:self.Vc], ut[self.Vc]) * grad[a][:self.Vc]
        self._ff[key] = F
        return F

    def rhs(self):
        d, m, h = self.d, self.m, self.h
        pref = 2.0 ** (1 - d) / h
        ncell, M, nv = self.w.shape
        out = np.zeros_like(self.w)
        visc = self.nu > 0 or self.chi > 0
        for c in range(ncell):
            for mode in range(M):
                acc = np.zeros(self.Vc)
                acc_alpha = 0.0
                for jj in itertools.product(range(m), repeat=d):       # jj[a] = Gauss index along axis a
                    xi = [self.xg[j] for j in jj]
                    gw = np.prod([self.gg[j] for j in jj])
                    u = self.u(c, xi)
                    grad = [self.u(c, xi, b) for b in range(d)] if (visc or self.av) else None
                    for a in range(d):
                        G = self.feuler(u[:self.Vc], a)
                        if visc:
                            G = G - self.fns(u[:self.Vc], [g[:self.Vc] for g in grad], a)
                        if self.av:
                            G = G - self.eps(u[:self.Vc], u[self.Vc]) * grad[a][:self.Vc]
                        acc += gw * G * self.phi(mode, xi, a)
                    if self.av:
                        rho, v, p = self.prim(u[:self.Vc])
                        cs = math.sqrt(self.g * p / rho)
                        divv = sum((grad[b][1 + b] - v[b] * grad[b][0]) / rho for b in range(d))
                        S, Gs = self.sensor[0][c], self.sensor[1][c]
                        Wk = self.o.f_w * max(0.0, Gs) if S > self.o.s_onset0 / (self.n + 1) ** 2 else 0.0
                        tau = self.o.f_tau * h / ((self.n + 1) * cs)
                        acc_alpha += gw * self.phi(mode, xi) * (self.o.f_v * max(0.0, -divv) + Wk - u[self.Vc] / tau)
                for a in range(d):
                    for kk in itertools.product(range(m), repeat=d - 1):
                        xit = [self.xg[k] for k in kk]
                        gs = np.prod([self.gg[k] for k in kk])
                        xp = list(xit); xp.insert(a, +1.0)
                        xm = list(xit); xm.insert(a, -1.0)
                        acc -= gs * (self.phi(mode, xp) * self.face_flux(c, self.nbr(c, a, +1), a, xit)
                                     - self.phi(mode, xm) * self.face_flux(self.nbr(c, a, -1), c, a, xit))
                out[c, mode, :self.Vc] = pref * acc
                if self.av:
                    out[c, mode, self.Vc] = 2.0 ** (-d) * acc_alpha
        return out


CASES = [(2, 1, "ns_mesh43"), (2, 1, "euler"), (2, 2, "euler"), (2, 3, "euler"), (2, 1, "ns"), (2, 3, "ns"), (2, 2, "ns_av"),
         (2, 3, "av"), (3, 1, "euler"), (3, 1, "ns_av"), (3, 2, "euler")]


@pytest.mark.parametrize("d,n,phys", CASES)
def test_p11_bruteforce_rhs(d, n, phys):
    ncell = (4, 3) if "mesh43" in phys else (2,) * d     # 4x3: left and right neighbours differ
    h = 0.5
    gamma = 1.4
    nu, chi = (0.03, 0.05) if "ns" in phys else (0.0, 0.0)
    av = "av" in phys
    opts = orc.Options(av_enable=av)
    o = orc.DGOracle(d, ncell, h, n + 1, gamma, nu, chi, opts)
    w0, al = wk.random_smooth_modes(d, ncell, n, gamma, seed=11 + n, amp=0.08, nvar_extra=1 if av else 0)
    o.set_state(w0)
    if av:
        o.set_alpha(al)
        rng = np.random.default_rng(2)
        o.sensor_S = rng.uniform(0.0, 3e-4 / (n + 1) ** 2, o.ncells)     # straddles S_onset
        o.sensor_G = rng.uniform(-1.0, 2.0, o.ncells)
    L = o.rhs(o.w)
    b = Brute(d, n, h, gamma, nu, chi, av, opts, o.w.copy(), (o.sensor_S, o.sensor_G), ncell)
    Lb = b.rhs()
    scale = np.max(np.abs(Lb), axis=(0, 1)) + 1e-300
    assert np.max(np.abs(L - Lb) / scale) < 1e-11, np.max(np.abs(L - Lb) / scale, axis=(0, 1))
