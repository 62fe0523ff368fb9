"""CPU oracle for the modal DG hot path of arXiv:2208.11131 -- TEST INFRASTRUCTURE.

This file is test infrastructure, not product code.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline / `--impl reference` legs may import it.  It shares no code, table, constant
generator or helper with the CUDA path under `paper_2208_11131_b200/csrc/`; neither imports the other.

It is the plain, slow, literal algorithm: dense per-cell basis matrices (no sum factorisation), numpy fp64,
Legendre values by three-term recurrence, every step in the paper's order and notation:

  O1  basis            PAPER.md:121-139 (Eq. 13-16), tensor-product mode set (reading A1); option
                       basis="total_degree": the paper's truncated set, PAPER.md:141-148 (Eq. 17-18)
  O2  quadrature       PAPER.md:164-171 (Eq. 19), n_g = n+1
  O3  timestep         PAPER.md:202-206 (Eq. 23), p = n+1 (A2)
  O4  RHS (weak form)  PAPER.md:104 (Eq. 10), 175-190 (Eq. 20-21); prefactors per A3/A4
  O5  Euler flux       PAPER.md:49-66 (Eq. 1-5); energy row (e+p)v (A5)
  O6  HLLC             PAPER.md:106 (Toro's HLLC, Davis wave-speed bounds; A6: parity unpinned vs TENETGPU)
  O7  viscous interior PAPER.md:248, 311-323 (Eq. 37-39); traceless Pi (A7)
  O8  face recovery    PAPER.md:252-305 (Eq. 27-36), corrections A9/A10
  O9  artificial visc. PAPER.md:375-407 (Eq. 43-46), 218 (Eq. 24)
  O10 sensor           PAPER.md:347-365 (Eq. 41-42), 392-397 (Eq. 45); top set / lagging per A13/A15
  O11 SSP-RK           PAPER.md:200 (Shu-Osher forms; 3-stage default per BASELINE config 1)
  O12 totals           PAPER.md:127, 423 (mode 0 is the cell mean)
  O13 positivity lim.  PAPER.md:417-432 (Eq. 47), optional, after every RK stage (readings L1-L6 in DESIGN.md)
  O14 passive tracer   PAPER.md:325-329 (Eq. 40), optional extra row c rho: advective flux c rho v, HLLC row
                       c_K x (star mass flux), diffusive flux eta rho grad c (readings T1-T3 in DESIGN.md)

Parity pins (tests/test_oracle_*.py) cover every function here; the readings with no pin in the paper
(A6, A11, A12, A14, A15, A18, L2, L3, A19b, T1, T2 in DESIGN.md) are "parity unpinned" against the authors' code but pinned as
mathematics where a closed form exists (HLLC consistency/exact contact/Sod star state, etc.).

State array layout inside the oracle: w[cell, mode, var]; cell = (iz*Ny+iy)*Nx+ix, mode = (lz*m+ly)*m+lx,
var = rho, rho v_x, rho v_y, (rho v_z), e, [c rho], [alpha].  The C-ABI layout w[(mode*Vc+var)*Ncells+cell]
 is converted in set_state/get_state.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np


# ----------------------------------------------------------------------------------------------------
# O1 / O2: Legendre basis and Gauss quadrature
# ----------------------------------------------------------------------------------------------------
def legendre_normalised(lmax: int, x):
    """P_l(x) = sqrt(2l+1) Leg_l(x), l = 0..lmax, and dP_l/dx, so that int_-1^1 P_l P_m = 2 delta_lm
    (Eq. 13).  Three-term (Bonnet) recurrence; derivative from Leg'_{l+1} = Leg'_{l-1} + (2l+1) Leg_l."""
    x = np.asarray(x, dtype=np.float64)
    L = np.zeros((lmax + 1,) + x.shape)
    dL = np.zeros_like(L)
    L[0] = 1.0
    if lmax >= 1:
        L[1] = x
        dL[1] = 1.0
    for l in range(1, lmax):
        L[l + 1] = ((2 * l + 1) * x * L[l] - l * L[l - 1]) / (l + 1)
        dL[l + 1] = dL[l - 1] + (2 * l + 1) * L[l]
    s = np.sqrt(2.0 * np.arange(lmax + 1) + 1.0).reshape((-1,) + (1,) * x.ndim)
    return s * L, s * dL


def gauss_legendre(m: int):
    """m-point Gauss-Legendre nodes x_j (ascending) and weights g_j on [-1,1] (Eq. 19):
    roots of Leg_m by Newton iteration, g_j = 2 / ((1-x_j^2) Leg_m'(x_j)^2)."""
    i = np.arange(m)
    x = -np.cos(np.pi * (i + 0.75) / (m + 0.5))
    for _ in range(100):
        P, dP = legendre_normalised(m, x)
        s = math.sqrt(2 * m + 1)
        dx = (P[m] / s) / (dP[m] / s)
        x = x - dx
        if np.max(np.abs(dx)) < 1e-16:
            break
    P, dP = legendre_normalised(m, x)
    dLeg = dP[m] / math.sqrt(2 * m + 1)
    g = 2.0 / ((1.0 - x * x) * dLeg * dLeg)
    return x, g


def kron_axes(mats):
    """Tensor-product operator for per-axis matrices mats[a] (a = x, y[, z]); row/column flat index has the
    x index fastest: idx = (i_z*m + i_y)*m + i_x (Eq. 16)."""
    out = np.asarray(mats[0])
    for A in mats[1:]:
        out = np.kron(np.asarray(A), out)
    return out


def overlap_integrals(n: int, f: float):
    """Legendre overlap integrals of the face recovery (Eq. 33-34, with reading A9):
      A^-_{m,l} = int_{-1}^{0} P_m(2 f x + 1) P_l(x) dx,   A^+_{m,l} = int_{0}^{1} P_m(2 f x - 1) P_l(x) dx,
    m = 0..n (cell modes), l = 0..n+1 (recovered modes).  Integrands have degree <= 2n+1: an (n+2)-point
    Gauss rule mapped to each half interval is exact."""
    xg, gg = gauss_legendre(n + 2)
    Am = np.zeros((n + 1, n + 2))
    Ap = np.zeros((n + 1, n + 2))
    xm = 0.5 * (xg - 1.0)  # [-1, 0]
    xp = 0.5 * (xg + 1.0)  # [0, 1]
    Pm_cell, _ = legendre_normalised(n, 2.0 * f * xm + 1.0)
    Pm_star, _ = legendre_normalised(n + 1, xm)
    Pp_cell, _ = legendre_normalised(n, 2.0 * f * xp - 1.0)
    Pp_star, _ = legendre_normalised(n + 1, xp)
    for m in range(n + 1):
        for l in range(n + 2):
            Am[m, l] = 0.5 * np.sum(gg * Pm_cell[m] * Pm_star[l])
            Ap[m, l] = 0.5 * np.sum(gg * Pp_cell[m] * Pp_star[l])
    return Am, Ap


def recovery_fraction(n: int) -> float:
    """f = 3/4 for n <= 2, f = 1 for n > 2."""
    return 0.75 if n <= 2 else 1.0


def recovery_vectors(n: int, f: float):
    """Partial-sum vectors of the recovered interface value and normal derivative (Eq. 35
    with prefactor 1/2 and full sum over m, reading A10; evaluation at xi* = 0, Eq. 31):
      u~(face)     = sum_m R^-_m w^-_m + R^+_m w^+_m,            R^+-_m = 1/2 sum_l A^+-_{m,l} P_l(0)
      d u~/dx_n    = (1/h) [sum_m G^-_m w^-_m + G^+_m w^+_m],    G^+-_m = 1/2 sum_l A^+-_{m,l} P_l'(0) / f
    """
    Am, Ap = overlap_integrals(n, f)
    P0, dP0 = legendre_normalised(n + 1, np.array(0.0))
    Rm = 0.5 * Am @ P0
    Rp = 0.5 * Ap @ P0
    Gm = 0.5 * Am @ dP0 / f
    Gp = 0.5 * Ap @ dP0 / f
    return Rm, Rp, Gm, Gp


# ----------------------------------------------------------------------------------------------------
# O5-O7: point-wise physics
# ----------------------------------------------------------------------------------------------------
def primitives(u, d: int, gamma: float):
    """rho, v[..., d], p from conserved u = (rho, rho v, e); p = (gamma-1)(e - rho v^2/2)."""
    rho = u[..., 0]
    v = u[..., 1:1 + d] / rho[..., None]
    e = u[..., 1 + d]
    p = (gamma - 1.0) * (e - 0.5 * rho * np.sum(v * v, axis=-1))
    return rho, v, p


def euler_flux(u, a: int, d: int, gamma: float):
    """f_a(u), PAPER.md:62 (Eq. 4); energy row (e + p) v_a (reading A5)."""
    rho, v, p = primitives(u, d, gamma)
    f = np.empty_like(u)
    f[..., 0] = rho * v[..., a]
    for b in range(d):
        f[..., 1 + b] = rho * v[..., a] * v[..., b]
    f[..., 1 + a] += p
    f[..., 1 + d] = (u[..., 1 + d] + p) * v[..., a]
    for k in range(d + 2, u.shape[-1]):          # passive tracer rows c rho (Eq. 40): flux c rho v_a
        f[..., k] = u[..., k] * v[..., a]
    return f


def hllc_flux(uL, uR, a: int, d: int, gamma: float):
    """HLLC numerical flux along axis a for left state uL (cell on the -a side) and right state uR
    (textbook HLLC of the Toro reference with the direct Davis wave-speed bounds, reading A6):
      S_L = min(vL-cL, vR-cR), S_R = max(vL+cL, vR+cR),
      S*  = [pR - pL + rhoL vL (S_L - vL) - rhoR vR (S_R - vR)] / [rhoL (S_L - vL) - rhoR (S_R - vR)],
      F = F_L (S_L >= 0); F_R (S_R <= 0); else F_K + S_K (U*_K - U_K), K = L if S* >= 0 else R."""
    rhoL, vL, pL = primitives(uL, d, gamma)
    rhoR, vR, pR = primitives(uR, d, gamma)
    cL = np.sqrt(gamma * pL / rhoL)
    cR = np.sqrt(gamma * pR / rhoR)
    vnL = vL[..., a]
    vnR = vR[..., a]
    SL = np.minimum(vnL - cL, vnR - cR)
    SR = np.maximum(vnL + cL, vnR + cR)
    Sstar = (pR - pL + rhoL * vnL * (SL - vnL) - rhoR * vnR * (SR - vnR)) / (
        rhoL * (SL - vnL) - rhoR * (SR - vnR))
    FL = euler_flux(uL, a, d, gamma)
    FR = euler_flux(uR, a, d, gamma)

    def star_state(u, rho, v, p, vn, S):
        fac = rho * (S - vn) / (S - Sstar)
        us = np.empty_like(u)
        us[..., 0] = fac
        for b in range(d):
            us[..., 1 + b] = fac * (Sstar if b == a else v[..., b])
        us[..., 1 + d] = fac * (u[..., 1 + d] / rho + (Sstar - vn) * (Sstar + p / (rho * (S - vn))))
        for k in range(d + 2, u.shape[-1]):      # a passive scalar is carried like a transverse velocity (reading T1)
            us[..., k] = fac * (u[..., k] / rho)
        return us

    UsL = star_state(uL, rhoL, vL, pL, vnL, SL)
    UsR = star_state(uR, rhoR, vR, pR, vnR, SR)
    FsL = FL + SL[..., None] * (UsL - uL)
    FsR = FR + SR[..., None] * (UsR - uR)
    F = np.where((Sstar >= 0.0)[..., None], FsL, FsR)
    F = np.where((SL >= 0.0)[..., None], FL, F)
    F = np.where((SR <= 0.0)[..., None], FR, F)
    return F


def ns_flux(u, grad, a: int, d: int, gamma: float, nu: float, chi: float, eta: float = 0.0):
    """Navier-Stokes flux column a (Eq. 38-39), grad[b][..., var] = d u_var / d x_b:
      F_NS,a = (0, Pi_{a b}, sum_b v_b Pi_{a b} + chi (gamma-1) rho d_a u_th),
      Pi = nu rho (grad v + grad v^T - 2/3 (div v) I)   (traceless reading A7),
      grad v = [grad(rho v) - v grad rho] / rho, u_th = e/rho - v^2/2."""
    rho, v, p = primitives(u, d, gamma)
    e = u[..., 1 + d]
    dv = [[(grad[b][..., 1 + c] - v[..., c] * grad[b][..., 0]) / rho for c in range(d)] for b in range(d)]
    divv = sum(dv[b][b] for b in range(d))
    F = np.zeros_like(u)
    for b in range(d):
        Pi_ab = nu * rho * (dv[a][b] + dv[b][a] - ((2.0 / 3.0) * divv if a == b else 0.0))
        F[..., 1 + b] = Pi_ab
        F[..., 1 + d] += v[..., b] * Pi_ab
    duth = grad[a][..., 1 + d] / rho - e * grad[a][..., 0] / (rho * rho) - sum(
        v[..., c] * dv[a][c] for c in range(d))
    F[..., 1 + d] += chi * (gamma - 1.0) * rho * duth
    for k in range(d + 2, u.shape[-1]):
        # tracer diffusion eta rho d_a c (Eq. 40), grad c = [grad(c rho) - c grad rho] / rho
        c = u[..., k] / rho
        F[..., k] = eta * rho * (grad[a][..., k] - c * grad[a][..., 0]) / rho
    return F


# ----------------------------------------------------------------------------------------------------
# SSP-RK tables in Shu-Osher form: u^(i) = sum_k [ A[i][k] u^(k) + dt B[i][k] L(u^(k)) ],  u^(0) = u^n
# ----------------------------------------------------------------------------------------------------
def ssprk_tableau(stages: int):
    """SSP Runge-Kutta, stages by order.  1: forward Euler; 2: SSP-RK2 (Heun);
    3: SSP-RK3 (Shu-Osher; BASELINE config 1); 5: SSPRK(5,4) for order >= 4."""
    if stages == 1:
        return [[1.0]], [[1.0]]
    if stages == 2:
        return [[1.0], [0.5, 0.5]], [[1.0], [0.0, 0.5]]
    if stages == 3:
        return ([[1.0], [0.75, 0.25], [1.0 / 3.0, 0.0, 2.0 / 3.0]],
                [[1.0], [0.0, 0.25], [0.0, 0.0, 2.0 / 3.0]])
    if stages == 5:
        # 4th-order, five-stage SSP scheme in Shu-Osher form -- the scheme the paper selects for order >= 4
        # ("fourth-order five stage" after Schaal et al. 2015, App. D, which is not in the
        # container).  The coefficients are the optimal SSPRK(5,4) set of Spiteri & Ruuth (2002) as commonly
        # published; reading A19b: "parity unpinned" against the authors' table, pinned as mathematics
        # by the eight order-4 conditions, convexity (SSP) and the degree-4 Taylor polynomial on dw/dt = -w.
        return ([[1.0],
                 [0.444370493651235, 0.555629506348765],
                 [0.620101851488403, 0.0, 0.379898148511597],
                 [0.178079954393132, 0.0, 0.0, 0.821920045606868],
                 [0.0, 0.0, 0.517231671970585, 0.096059710526147, 0.386708617503269]],
                [[0.391752226571890],
                 [0.0, 0.368410593050371],
                 [0.0, 0.0, 0.251891774271694],
                 [0.0, 0.0, 0.0, 0.544974750228521],
                 [0.0, 0.0, 0.0, 0.063692468666290, 0.226007483236906]])
    raise ValueError("rk_stages must be 1, 2, 3 or 5")


@dataclass
class Options:
    """Runtime options; defaults PAPER.md:206, 413-415 (f_v=2.5, f_tau=0.5, f_w=0.2, S_onset=1e-4/(n+1)^2, alpha_max=1)."""
    f_cfl: float = 0.5
    rk_stages: int = 3
    av_enable: bool = False
    f_v: float = 2.5
    f_tau: float = 0.5
    f_w: float = 0.2
    s_onset0: float = 1.0e-4
    alpha_max: float = 1.0
    fixed_dt: float = 0.0  # > 0: use this dt instead of Eq. 23
    limiter_enable: bool = False  # positivity limiter after every RK stage (Eq. 47)
    # mode set: "tensor" = all (n+1)^d products (reading A1, BASELINE.json mode counts); "total_degree" = the paper's
    # own set, products whose total degree sum_a l_a exceeds n are discarded (Eq. 17-18)
    basis: str = "tensor"
    # passive tracer (Eq. 40): one more conserved row c rho behind the energy, diffusivity eta
    tracer_enable: bool = False
    eta: float = 0.0


class DGOracle:
    """Plain CPU DG solver on a uniform periodic Cartesian mesh (see module docstring)."""

    def __init__(self, dim, ncell, h, order, gamma, nu=0.0, chi=0.0, options: Options | None = None):
        assert dim in (2, 3)
        self.d = d = dim
        self.ncell = tuple(int(c) for c in ncell[:d])
        self.h = float(h)
        self.order = int(order)
        self.n = n = self.order - 1          # highest Legendre degree
        self.m = m = n + 1                   # Gauss points per axis
        self.gamma = float(gamma)
        self.nu = float(nu)
        self.chi = float(chi)
        self.opt = options if options is not None else Options()
        self.tracer = bool(self.opt.tracer_enable)
        self.eta = float(self.opt.eta) if self.tracer else 0.0
        self.Vc = d + 2 + (1 if self.tracer else 0)
        self.av = bool(self.opt.av_enable)
        self.V = self.Vc + (1 if self.av else 0)
        self.visc = (self.nu > 0.0) or (self.chi > 0.0) or (self.eta > 0.0)
        self.need_grad = self.visc or self.av
        self.M = m ** d
        self.Np = m ** d
        self.Nf = m ** (d - 1)
        self.ncells = int(np.prod(self.ncell))
        self._build_tables()
        self._build_neighbours()
        self.w = np.zeros((self.ncells, self.M, self.V))
        self.sensor_S = np.zeros(self.ncells)
        self.sensor_G = np.zeros(self.ncells)
        self.t = 0.0
        self.last_dt = 0.0
        self.unphysical = False
        self.max_alpha = 0.0

    # ---- tables (S0) -------------------------------------------------------------------------------
    def _build_tables(self):
        n, m, d = self.n, self.m, self.d
        self.x, self.g = gauss_legendre(m)
        P, dP = legendre_normalised(n, self.x)
        self.Vm = P.T.copy()      # Vm[j,l] = P_l(x_j)
        self.Dm = dP.T.copy()     # Dm[j,l] = P_l'(x_j)
        Pm1, _ = legendre_normalised(n, np.array(-1.0))
        Pp1, _ = legendre_normalised(n, np.array(+1.0))
        self.Pend = [Pm1.reshape(1, -1), Pp1.reshape(1, -1)]   # P_l(-1), P_l(+1)
        # volume: Phi[j,l] = phi_l(xi_j), dPhi[a][j,l] = d phi_l / d xi_a (xi_j)   (Eq. 16, 21)
        self.Phi = kron_axes([self.Vm] * d)
        self.dPhi = [kron_axes([self.Dm if b == a else self.Vm for b in range(d)]) for a in range(d)]
        self.gvol = kron_axes([self.g.reshape(-1, 1)] * d).ravel()
        self.gsur = kron_axes([self.g.reshape(-1, 1)] * (d - 1)).ravel()
        # faces: PhiF[a][s][k,l] = phi_l at face point k of the -a (s=0) / +a (s=1) face
        self.PhiF = [[kron_axes([self.Pend[s] if b == a else self.Vm for b in range(d)]) for s in (0, 1)]
                     for a in range(d)]
        # recovery (O8): index 0 = operator on the LEFT cell (uses R^-, G^-), 1 = on the RIGHT cell (R^+, G^+)
        self.f_rec = recovery_fraction(n)
        Rm, Rp, Gm, Gp = recovery_vectors(n, self.f_rec)
        self.Rvec = [Rm.reshape(1, -1), Rp.reshape(1, -1)]
        self.Gvec = [Gm.reshape(1, -1), Gp.reshape(1, -1)]
        self.RV = [[kron_axes([self.Rvec[s] if b == a else self.Vm for b in range(d)]) for s in (0, 1)]
                   for a in range(d)]
        self.RN = [[kron_axes([self.Gvec[s] if b == a else self.Vm for b in range(d)]) for s in (0, 1)]
                   for a in range(d)]
        # transverse derivative of the recovered face polynomial: cell basis kept transversally
        self.RT = [[[None if t == a else
                     kron_axes([self.Rvec[s] if b == a else (self.Dm if b == t else self.Vm) for b in range(d)])
                     for s in (0, 1)] for t in range(d)] for a in range(d)]
        # sensor "top" modes: max_a l_a = n (reading A13)
        l1 = np.arange(m)
        ls = np.meshgrid(*([l1] * d), indexing="ij")  # ls[0] varies slowest in C-order ravel -> reverse below
        lmax = np.zeros(self.M, dtype=int)
        for idx in range(self.M):
            rem, mx = idx, 0
            for _ in range(d):
                mx = max(mx, rem % m)
                rem //= m
            lmax[idx] = mx
        self.top = (lmax == n) if n >= 1 else np.zeros(self.M, dtype=bool)
        # total-degree truncation: keep[l] = (sum_a l_a <= n).  The basis is orthonormal, so the
        # Galerkin equations of the kept modes are those of Eq. 20 unchanged and the discarded weights stay zero;
        # the "highest-order" modes of the sensor (Eq. 42: l = N_{p-1}+1 .. N_p) are then those with sum_a l_a = n.
        assert self.opt.basis in ("tensor", "total_degree")
        lsum = np.zeros(self.M, dtype=int)
        for idx in range(self.M):
            rem = idx
            for _ in range(d):
                lsum[idx] += rem % m
                rem //= m
        self.keep = (lsum <= n) if self.opt.basis == "total_degree" else np.ones(self.M, dtype=bool)
        if self.opt.basis == "total_degree":
            self.top = (lsum == n) if n >= 1 else np.zeros(self.M, dtype=bool)

    def _build_neighbours(self):
        d = self.d
        shape = self.ncell[::-1]  # (Nz, Ny, Nx): x fastest
        idx = np.arange(self.ncells).reshape(shape)
        self.nbr = []
        for a in range(d):
            ax = d - 1 - a
            self.nbr.append([np.roll(idx, +1, axis=ax).ravel(), np.roll(idx, -1, axis=ax).ravel()])

    # ---- state I/O in the C-ABI layout -------------------------------------------------------------
    def set_state(self, w_flat):
        """w_flat[(mode*Vc + var)*Ncells + cell]; alpha := 0, sensor scalars := 0, t := 0."""
        w_flat = np.asarray(w_flat, dtype=np.float64)
        assert w_flat.size == self.M * self.Vc * self.ncells
        self.w[:] = 0.0
        self.w[:, :, :self.Vc] = w_flat.reshape(self.M, self.Vc, self.ncells).transpose(2, 0, 1)
        self.w[:, ~self.keep, :] = 0.0          # L2 projection onto the kept (orthonormal) modes
        self.sensor_S[:] = 0.0
        self.sensor_G[:] = 0.0
        self.t = 0.0
        self.last_dt = 0.0
        self.unphysical = False

    def get_state(self):
        return np.ascontiguousarray(self.w[:, :, :self.Vc].transpose(1, 2, 0)).ravel()

    def get_alpha(self):
        """alpha modal field, layout [mode*Ncells + cell]; zeros if AV is off."""
        if not self.av:
            return np.zeros(self.M * self.ncells)
        return np.ascontiguousarray(self.w[:, :, self.Vc].T).ravel()

    def set_alpha(self, a_flat):
        assert self.av
        self.w[:, :, self.Vc] = np.asarray(a_flat, dtype=np.float64).reshape(self.M, self.ncells).T
        self.w[:, ~self.keep, self.Vc] = 0.0

    def conserved_totals(self):
        """|K| sum_cells w_0 per conserved variable (O12), compensated summation."""
        vol = self.h ** self.d
        return np.array([vol * math.fsum(self.w[:, 0, v]) for v in range(self.Vc)])

    # ---- O3: timestep ------------------------------------------------------------------------------
    def wave_speeds(self, w):
        """Global max c_s and max |v| over all volume Gauss points (Eq. 23 inputs, reading A18)."""
        u = np.einsum("jl,clv->cjv", self.Phi, w[:, :, :self.Vc])
        rho, v, p = primitives(u, self.d, self.gamma)
        if np.any(rho <= 0.0) or np.any(p <= 0.0):
            self.unphysical = True
        cs = np.sqrt(self.gamma * p / rho)
        return float(np.max(cs)), float(np.max(np.sqrt(np.sum(v * v, axis=-1))))

    def timestep(self, w):
        """dt = f_CFL h / (2 (n+1) (c_s,max + v_max))  (Eq. 23 with p = n+1)."""
        if self.opt.fixed_dt > 0.0:
            return float(self.opt.fixed_dt)
        cmax, vmax = self.wave_speeds(w)
        return self.opt.f_cfl * self.h / (2.0 * (self.n + 1) * (cmax + vmax))

    # ---- O4: right-hand side ------------------------------------------------------------------------
    def rhs(self, w, terms=False):
        """dw/dt = L(w) per Eq. 20 with interior flux G_a = f_a - F_NS,a - eps d_a u and
        face flux G^_a = HLLC(traces) - F_NS,a(u~, grad u~) - eps~ d_a u~.  Returns dwdt (and optionally the
        volume and surface parts separately)."""
        d, Vc, h, n, gamma = self.d, self.Vc, self.h, self.n, self.gamma
        pref = 2.0 ** (1 - d) / h
        wc = w[:, :, :Vc]
        vol = np.zeros_like(w)
        sur = np.zeros_like(w)

        # --- volume term ---
        u = np.einsum("jl,clv->cjv", self.Phi, wc)                      # Eq. 21
        rho, v, p = primitives(u, d, gamma)
        if np.any(rho <= 0.0) or np.any(p <= 0.0):
            self.unphysical = True
        grad = None
        if self.need_grad:
            grad = [(2.0 / h) * np.einsum("jl,clv->cjv", self.dPhi[b], wc) for b in range(d)]
        if self.av:
            cs = np.sqrt(gamma * p / rho)
            alpha = np.einsum("jl,cl->cj", self.Phi, w[:, :, Vc])
            self.max_alpha = max(self.max_alpha, float(np.max(alpha)))
            eps = np.clip(alpha, 0.0, self.opt.alpha_max) * cs * h / (n + 1)      # Eq. 46, clamp A17
        for a in range(d):
            G = euler_flux(u, a, d, gamma)
            if self.visc:
                G = G - ns_flux(u, grad, a, d, gamma, self.nu, self.chi, self.eta)
            if self.av:
                G = G - eps[..., None] * grad[a]                                   # Eq. 24
            vol[:, :, :Vc] += pref * np.einsum("j,cjv,jl->clv", self.gvol, G, self.dPhi[a])
        if self.av:
            divv = sum((grad[b][..., 1 + b] - v[..., b] * grad[b][..., 0]) / rho for b in range(d))
            # Eq. 45 with lagged sensor (A15), onset threshold S_onset = s0/(n+1)^2 (A14)
            s_onset = self.opt.s_onset0 / (n + 1) ** 2
            W = np.where(self.sensor_S > s_onset, self.opt.f_w * np.maximum(0.0, self.sensor_G), 0.0)
            src = (self.opt.f_v * np.maximum(0.0, -divv) + W[:, None]
                   - alpha * ((n + 1) * cs / (self.opt.f_tau * h)))              # Eq. 43-44
            vol[:, :, Vc] = 2.0 ** (-d) * np.einsum("j,cj,jl->cl", self.gvol, src, self.Phi)

        # --- surface term: one flux per face, face between cell c (left) and nbr[a][1][c] (right) ---
        for a in range(d):
            R = self.nbr[a][1]
            uL = np.einsum("kl,clv->ckv", self.PhiF[a][1], wc)          # trace on the +a face of the left cell
            uR = np.einsum("kl,clv->ckv", self.PhiF[a][0], wc[R])       # trace on the -a face of the right cell
            for uu in (uL, uR):
                r_, _, p_ = primitives(uu, d, gamma)
                if np.any(r_ <= 0.0) or np.any(p_ <= 0.0):
                    self.unphysical = True
            Fh = hllc_flux(uL, uR, a, d, gamma)
            if self.need_grad:
                wl, wr = w, w[R]
                ut = (np.einsum("kl,clv->ckv", self.RV[a][0], wl) + np.einsum("kl,clv->ckv", self.RV[a][1], wr))
                gt = []
                for b in range(d):
                    if b == a:
                        gb = (np.einsum("kl,clv->ckv", self.RN[a][0], wl[:, :, :Vc])
                              + np.einsum("kl,clv->ckv", self.RN[a][1], wr[:, :, :Vc])) / h
                    else:
                        gb = (2.0 / h) * (np.einsum("kl,clv->ckv", self.RT[a][b][0], wl[:, :, :Vc])
                                          + np.einsum("kl,clv->ckv", self.RT[a][b][1], wr[:, :, :Vc]))
                    gt.append(gb)
                utc = ut[..., :Vc]
                rt, vt, pt = primitives(utc, d, gamma)
                if np.any(rt <= 0.0) or np.any(pt <= 0.0):
                    self.unphysical = True
                if self.visc:
                    Fh = Fh - ns_flux(utc, gt, a, d, gamma, self.nu, self.chi, self.eta)
                if self.av:
                    cst = np.sqrt(gamma * pt / rt)
                    epst = np.clip(ut[..., Vc], 0.0, self.opt.alpha_max) * cst * h / (n + 1)   # A12
                    Fh = Fh - epst[..., None] * gt[a]
            # lift (Eq. 20 surface lines): left cell sees the face as its +a face, right cell as its -a face
            sur[:, :, :Vc] -= pref * np.einsum("k,ckv,kl->clv", self.gsur, Fh, self.PhiF[a][1])
            contrib = pref * np.einsum("k,ckv,kl->clv", self.gsur, Fh, self.PhiF[a][0])
            sur[R, :, :Vc] += contrib          # R is a permutation of the cells: no duplicate indices
        # total-degree basis: only the kept modes are test functions of Eq. 20
        vol[:, ~self.keep, :] = 0.0
        sur[:, ~self.keep, :] = 0.0
        if terms:
            return vol + sur, vol, sur
        return vol + sur

    # ---- O10: sensor --------------------------------------------------------------------------------
    def sensor(self, w, dwdt):
        """S^K = sum_top w^2 / sum_all w^2 for the density row (Eq. 42) and d log S / dt from the weights'
        time derivatives, G = 2 sum_top w w' / A - 2 sum_all w w' / B (Eq. 45).  A = 0 => S = 0, G = 0."""
        r = w[:, :, 0]
        rd = dwdt[:, :, 0]
        A = np.sum(r[:, self.top] ** 2, axis=1)
        B = np.sum(r ** 2, axis=1)
        S = A / B
        dA = 2.0 * np.sum(r[:, self.top] * rd[:, self.top], axis=1)
        dB = 2.0 * np.sum(r * rd, axis=1)
        with np.errstate(divide="ignore", invalid="ignore"):
            G = np.where(A > 0.0, dA / np.where(A > 0.0, A, 1.0) - dB / B, 0.0)
        return S, G

    # ---- O11: one SSP-RK step -----------------------------------------------------------------------
    # ---- O13: positivity limiter (Eq. 47) ---------------------------------------------
    def positivity_limit(self, w):
        """Returns the limited copy of w[cell, mode, var].  Per cell, in the paper's order:
        mean density rho_bar = w_0 and mean pressure p_bar (pressure of the cell-mean state, reading L2); either
        <= 0: "a code crash is unavoidable" -> unphysical flag, cell left alone.  Evaluation points = union of the
        volume Gauss points and the Gauss points of the 2d faces.  Density: rho_bottom = 1e-6 rho_bar;
        if rho_min < rho_bottom, f = (rho_bar - rho_bottom)/(rho_bar - rho_min) and every mode but the mean of every
        conserved field is multiplied by f (Eq. 47; "l > 1" counts modes from 1, reading L1).  Pressure: p_bottom =
        1e-6 p_bar (reading L3); while p_min < p_bottom multiply the same modes by 0.5.  The
        artificial-viscosity field alpha is not a hydrodynamic field and is left untouched (reading L5)."""
        Vc = self.Vc
        w = w.copy()
        if self.M == 1:
            return w                                        # no higher modes to limit
        E = np.concatenate([self.Phi] + [self.PhiF[a][s] for a in range(self.d) for s in (0, 1)], axis=0)
        for c in range(self.ncells):
            mean = w[c, 0, :Vc].copy()
            rho_bar = mean[0]
            p_bar = (self.gamma - 1.0) * (mean[1 + self.d] - 0.5 * float(np.sum(mean[1:1 + self.d] ** 2)) / rho_bar) \
                if rho_bar > 0.0 else -1.0
            if not (rho_bar > 0.0) or not (p_bar > 0.0):
                self.unphysical = True
                continue
            u = E @ w[c, :, :Vc]                            # [point, var]
            rho_bottom = 1.0e-6 * rho_bar
            rho_min = float(np.min(u[:, 0]))
            if rho_min < rho_bottom:
                f = (rho_bar - rho_bottom) / (rho_bar - rho_min)
                w[c, 1:, :Vc] *= f
            p_bottom = 1.0e-6 * p_bar
            for _ in range(64):
                u = E @ w[c, :, :Vc]
                pr = (self.gamma - 1.0) * (u[:, 1 + self.d] - 0.5 * np.sum(u[:, 1:1 + self.d] ** 2, axis=1) / u[:, 0])
                if float(np.min(pr)) >= p_bottom:
                    break
                w[c, 1:, :Vc] *= 0.5
        return w

    def step(self, nsteps=1):
        A, B = ssprk_tableau(self.opt.rk_stages)
        for _ in range(nsteps):
            dt = self.timestep(self.w)
            us = [self.w]
            Ls = []
            for i in range(len(A)):
                Li = self.rhs(us[i])
                if i == 0 and self.av:
                    newS, newG = self.sensor(us[0], Li)   # refreshed once per step, used by the NEXT step (A15)
                Ls.append(Li)
                unew = np.zeros_like(self.w)
                for k in range(i + 1):
                    if A[i][k] != 0.0:
                        unew += A[i][k] * us[k]
                    if B[i][k] != 0.0:
                        unew += (B[i][k] * dt) * Ls[k]
                if self.opt.limiter_enable:
                    unew = self.positivity_limit(unew)
                us.append(unew)
            self.w = us[-1]
            if self.av:
                self.sensor_S, self.sensor_G = newS, newG
            self.t += dt
            self.last_dt = dt
        return 0 if not self.unphysical else -3

    # ---- helpers used by tests (evaluation, norms) --------------------------------------------------
    def evaluate(self, w, xi):
        """u^K(xi) for reference points xi (npts, d) in [-1,1]^d: Eq. 21 by direct evaluation."""
        cols = []
        for a in range(self.d):
            P, _ = legendre_normalised(self.n, xi[:, a])
            cols.append(P.T)  # (npts, m)
        phi = np.ones((xi.shape[0], 1))
        # x fastest mode index
        out = cols[0]
        for a in range(1, self.d):
            out = (cols[a][:, :, None] * out[:, None, :]).reshape(xi.shape[0], -1)
        return np.einsum("jl,clv->cjv", out, w)


def min_memory_doubles(n: int, d: int, Nc: int, total_degree: bool = True) -> int:
    """PAPER.md:765-786 (Eq. 59-62): N_w = [3 + d + f_t(p)] Nc^d N^dD, f_t(p) = p for p <= 3 else 5 (p = n+1),
    with the paper's total-degree mode count N^3D(n) = (n+1)(n+2)(n+3)/6 (Eq. 17) or N^2D (Eq. 18)."""
    p = n + 1
    ft = p if p <= 3 else 5
    if total_degree:
        N = (n + 1) * (n + 2) * (n + 3) // 6 if d == 3 else (n + 1) * (n + 2) // 2
    else:
        N = (n + 1) ** d
    return (3 + d + ft) * Nc ** d * N
