"""Seeded synthetic inputs for the DG hot path (BASELINE.json configs 1-5).

This module serves BOTH the CUDA path and the CPU oracle with identical inputs and holds none of the
solver's arithmetic: it evaluates the point-wise initial conditions the paper / BASELINE.json write down
and projects them onto the cell basis (Eq. 11) with library routines only
(`numpy.polynomial.legendre.leggauss` / `legvander`).  It imports neither `oracle/` nor the CUDA binding.

Output layout is the C-ABI state layout (include/dg.h): w[(mode*Vc + var)*Ncells + cell],
cell = (iz*Ny+iy)*Nx+ix, mode = (lz*m+ly)*m+lx, var = rho, rho v_x, rho v_y, (rho v_z), e.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np
from numpy.polynomial import legendre as npleg

SEED = 220811131  # harness seed


@dataclass(frozen=True)
class Workload:
    """One synthetic problem: mesh, physics switches, run length and the IC recipe name."""
    name: str
    dim: int
    ncell: tuple
    h: float
    degree: int                 # n; order p = n+1
    gamma: float
    nu: float = 0.0
    chi: float = 0.0
    av: bool = False
    f_cfl: float = 0.5
    steps: int = 10
    ic: str = "wave"
    origin: tuple = (0.0, 0.0, 0.0)
    params: dict = field(default_factory=dict)

    @property
    def order(self):
        return self.degree + 1

    @property
    def m(self):
        return self.degree + 1

    @property
    def modes(self):
        return self.m ** self.dim

    @property
    def ncells(self):
        return int(np.prod(self.ncell[:self.dim]))

    @property
    def nvar_conserved(self):
        return self.dim + 2

    @property
    def nvar(self):
        return self.dim + 2 + (1 if self.av else 0)


def config(i: int, degree: int | None = None, scale: float = 1.0) -> Workload:
    """BASELINE.json config i (1..5).  `scale` < 1 shrinks the cell counts (same domain, larger h) for
    oracle-sized parity runs; `degree` overrides the polynomial degree (config 5 sweeps 1..7)."""
    def sc(n):
        return max(2, int(round(n * scale)))
    if i == 1:   # 2D advected density wave, Euler (PAPER-style smooth test; exact solution known)
        n = 1 if degree is None else degree
        N = sc(16)
        return Workload("cfg1_wave2d", 2, (N, N), 1.0 / N, n, 5.0 / 3.0, f_cfl=0.3, steps=10, ic="wave")
    if i == 2:   # 2D smooth Kelvin-Helmholtz with physical viscosity (Eq. 53-54)
        n = 3 if degree is None else degree
        N = sc(128)
        return Workload("cfg2_kh2d", 2, (N, 2 * N), 1.0 / N, n, 5.0 / 3.0, nu=1e-5, chi=1e-5, f_cfl=0.5,
                        steps=100, ic="kh", params=dict(P=10.0, a=0.05, z1=0.5, z2=1.5, sigma2=0.04, A=0.01))
    if i == 3:   # 2D Sod shock tube with artificial viscosity (defaults)
        n = 5 if degree is None else degree
        N = sc(1024)
        Ny = max(2, N // 64)
        return Workload("cfg3_sod2d", 2, (N, Ny), 1.0 / N, n, 1.4, av=True, f_cfl=0.3, steps=200, ic="sod")
    if i == 4:   # 3D subsonic turbulence-shaped box, NS + AV (PAPER.md:800-802 timing workload shape)
        n = 3 if degree is None else degree
        N = sc(128)
        return Workload("cfg4_turb3d", 3, (N, N, N), 1.0 / N, n, 5.0 / 3.0, nu=1e-4, chi=1e-4, av=True,
                        f_cfl=0.5, steps=50, ic="turb", params=dict(mach=0.3, kmin=1.0, kmax=3.0))
    if i == 5:   # 3D advected density wave, Euler, order sweep
        n = 3 if degree is None else degree
        N = sc(64)
        return Workload("cfg5_wave3d", 3, (N, N, N), 1.0 / N, n, 5.0 / 3.0, f_cfl=0.3, steps=20, ic="wave")
    raise ValueError("config index must be 1..5")


def with_mesh(wl: Workload, ncell) -> Workload:
    """Same problem on a different cell count (domain kept: h rescaled by the x extent)."""
    L = wl.h * wl.ncell[0]
    return replace(wl, ncell=tuple(ncell), h=L / ncell[0])


# ----------------------------------------------------------------------------------------------------
# point-wise initial conditions: conserved state u(x) at arbitrary points
# ----------------------------------------------------------------------------------------------------
def _conserved(rho, v, P, gamma):
    e = P / (gamma - 1.0) + 0.5 * rho * sum(c * c for c in v)
    return [rho] + [rho * c for c in v] + [e]


def wave_exact(wl: Workload, X, t=0.0):
    """rho = 1 + 0.1 sin(2 pi (sum_a x_a - d t)), v = (1,..,1), P = 1: exact advected solution."""
    s = sum(X) - wl.dim * t
    rho = 1.0 + 0.1 * np.sin(2.0 * np.pi * s)
    one = np.ones_like(rho)
    return _conserved(rho, [one] * wl.dim, one, wl.gamma)


def _kh(wl, X):
    x, z = X
    p = wl.params
    a, z1, z2 = p["a"], p["z1"], p["z2"]
    th = np.tanh((z - z1) / a) - np.tanh((z - z2) / a)
    rho = 1.0 + 0.5 * th
    vx = th - 1.0
    vz = p["A"] * np.sin(2.0 * np.pi * x) * (np.exp(-(z - z1) ** 2 / p["sigma2"]) + np.exp(-(z - z2) ** 2 / p["sigma2"]))
    return _conserved(rho, [vx + 0.0 * x, vz], p["P"] + 0.0 * rho, wl.gamma)


def _sod(wl, X):
    x = X[0]
    left = (x < 0.5)
    rho = np.where(left, 1.0, 0.125)
    P = np.where(left, 1.0, 0.1)
    zero = np.zeros_like(rho)
    return _conserved(rho, [zero] * wl.dim, P, wl.gamma)


def vortex_exact(wl: Workload, X):
    """Isentropic vortex of Yee et al. (Eq. 48-51) on [-5,5]^2, gamma = 1.4, beta = 5: a steady
    solution of the Euler equations (the exact solution at any time is the initial state).  u = P/((gamma-1) rho) is
    the thermal energy per unit mass, so P = (gamma-1) rho u = rho^gamma (isentropic)."""
    x, y = X
    beta = wl.params.get("beta", 5.0)
    g = wl.gamma
    r2 = x * x + y * y
    f = (beta / (2.0 * np.pi)) * np.exp(0.5 * (1.0 - r2))
    u = 1.0 - (beta * beta / (8.0 * g * np.pi ** 2)) * np.exp(1.0 - r2)
    rho = ((g - 1.0) * u) ** (1.0 / (g - 1.0))
    return _conserved(rho, [-y * f, x * f], (g - 1.0) * rho * u, g)


def vortex(ncell=32, degree=3) -> Workload:
    """The isentropic-vortex workload: 2D Euler, periodic box [-5,5]^2."""
    return Workload("vortex2d", 2, (ncell, ncell), 10.0 / ncell, degree, 1.4, f_cfl=0.3, steps=10, ic="vortex",
                    origin=(-5.0, -5.0, 0.0), params=dict(beta=5.0))


def turbulence_modes(wl: Workload, seed=SEED):
    """Half-space integer wave vectors with kmin <= |k| <= kmax and their solenoidal complex amplitudes
    a_k -> (I - k k^T/k^2) a_k, a_k iid complex standard normal (flat spectrum), SURVEY.md 8(d) item 4."""
    rng = np.random.default_rng(seed)
    kmax = int(wl.params["kmax"])
    ks = []
    for kx in range(-kmax, kmax + 1):
        for ky in range(-kmax, kmax + 1):
            for kz in range(-kmax, kmax + 1):
                k2 = kx * kx + ky * ky + kz * kz
                if not (wl.params["kmin"] ** 2 <= k2 <= wl.params["kmax"] ** 2):
                    continue
                if (kz, ky, kx) > (0, 0, 0):   # one of each +-k pair
                    ks.append((kx, ky, kz))
    ks = np.array(ks, dtype=np.float64)
    amp = rng.standard_normal((len(ks), 3)) + 1j * rng.standard_normal((len(ks), 3))
    kk = np.sum(ks * ks, axis=1, keepdims=True)
    amp = amp - ks * (np.sum(ks * amp, axis=1, keepdims=True) / kk)
    return ks, amp


def _turb_velocity_1d_tables(wl, ks, xs):
    """e^{2 pi i k x} per distinct integer k for the 1D point sets xs[a]."""
    kmax = int(wl.params["kmax"])
    kk = np.arange(-kmax, kmax + 1)
    return kk, [np.exp(2j * np.pi * kk[:, None] * x[None, :]) for x in xs]


def turb_velocity_grid(wl, xs, seed=SEED):
    """v(x) = sum_k Re[a_k e^{2 pi i k.x}] on the tensor grid xs[0] x xs[1] x xs[2] (evaluated separably),
    returned as 3 arrays indexed [z, y, x]; NOT yet normalised."""
    ks, amp = turbulence_modes(wl, seed)
    kmax = int(wl.params["kmax"])
    nk = 2 * kmax + 1
    _, E = _turb_velocity_1d_tables(wl, ks, xs)
    out = []
    for c in range(3):
        T = np.zeros((nk, nk, nk), dtype=np.complex128)   # [kz, ky, kx]
        for (kx, ky, kz), a in zip(ks.astype(int), amp[:, c]):
            T[kz + kmax, ky + kmax, kx + kmax] = a
        t1 = np.tensordot(T, E[0], axes=([2], [0]))            # [kz, ky, x]
        t2 = np.tensordot(E[1].T, t1, axes=([1], [1]))         # [y, kz, x]
        v = np.tensordot(E[2].T, t2, axes=([1], [1]))          # [z, y, x]
        out.append(np.ascontiguousarray(v.real))
    return out


def turb_rms_scale(wl, seed=SEED):
    """Scale factor making sqrt(<|v|^2>) = mach * sqrt(gamma P / rho) (rho = P = 1): for a sum of
    Re[a_k e^{ikx}] over distinct half-space k the volume mean of |v|^2 is sum_k |a_k|^2 / 2 exactly."""
    _, amp = turbulence_modes(wl, seed)
    rms = np.sqrt(0.5 * np.sum(np.abs(amp) ** 2))
    return wl.params["mach"] * np.sqrt(wl.gamma) / rms


# ----------------------------------------------------------------------------------------------------
# projection onto the cell basis (Eq. 11) with an (n+3)-point Gauss rule per axis
# ----------------------------------------------------------------------------------------------------
def _proj_table(n, nq):
    """T[q, l] = 0.5 * g_q * sqrt(2l+1) Leg_l(x_q): 1D factor of (1/|K|) int u phi_l."""
    xq, gq = npleg.leggauss(nq)
    Vq = npleg.legvander(xq, n) * np.sqrt(2.0 * np.arange(n + 1) + 1.0)[None, :]
    return xq, 0.5 * gq[:, None] * Vq


def initial_modes(wl: Workload, seed=SEED, zslab=None):
    """Modal coefficients of the workload's IC in the C-ABI layout (flat float64 array).
    zslab = (iz0, iz1) restricts a 3D mesh to cell layers [iz0, iz1) (layout then uses that sub-mesh)."""
    d, n, m, h = wl.dim, wl.degree, wl.m, wl.h
    nq = n + 3
    xq, T = _proj_table(n, nq)
    N = list(wl.ncell[:d])
    i0 = [0] * d
    if zslab is not None:
        assert d == 3
        i0[2], N[2] = zslab[0], zslab[1] - zslab[0]
    # 1D physical coordinates of all quadrature points per axis: (cells*nq,)
    xs = [wl.origin[a] + h * (np.repeat(np.arange(i0[a], i0[a] + N[a]), nq) + 0.5 + 0.5 * np.tile(xq, N[a]))
          for a in range(d)]
    if wl.ic == "turb":
        v = turb_velocity_grid(wl, xs, seed)
        s = turb_rms_scale(wl, seed)
        rho = np.ones_like(v[0])
        U = _conserved(rho, [s * c for c in v], np.ones_like(rho), wl.gamma)
    else:
        grids = np.meshgrid(*xs[::-1], indexing="ij")[::-1]   # arrays indexed [z, y, x] (or [y, x])
        if wl.ic == "wave":
            U = wave_exact(wl, grids, 0.0)
        elif wl.ic == "kh":
            U = _kh(wl, grids)
        elif wl.ic == "sod":
            U = _sod(wl, grids)
        elif wl.ic == "vortex":
            U = vortex_exact(wl, grids)
        elif wl.ic == "uniform":
            one = np.ones_like(grids[0])
            U = _conserved(one, [0.0 * one] * d, one, wl.gamma)
        else:
            raise ValueError(wl.ic)
    Vc = d + 2
    ncells = int(np.prod(N))
    out = np.empty((m ** d, Vc, ncells))
    for var in range(Vc):
        A = np.asarray(U[var], dtype=np.float64)
        if d == 2:
            A = A.reshape(N[1], nq, N[0], nq)                    # [iy, qy, ix, qx]
            W = np.einsum("aqbr,ql,rk->lkab", A, T, T)           # [ly, lx, iy, ix]
        else:
            A = A.reshape(N[2], nq, N[1], nq, N[0], nq)          # [iz, qz, iy, qy, ix, qx]
            W = np.einsum("apbqcr,pl,qk,rj->lkjabc", A, T, T, T, optimize=True)   # [lz, ly, lx, iz, iy, ix]
        out[:, var, :] = W.reshape(m ** d, ncells)
    return out.ravel()


def random_smooth_modes(dim, ncell, degree, gamma, seed=SEED, amp=0.1, nvar_extra=0):
    """Seeded random positive state for parity / brute-force tests: mode 0 = a fixed physical base state,
    higher modes iid normal scaled by amp / (1 + sum l_a)^2 (smooth decay, rho and p stay > 0)."""
    rng = np.random.default_rng(seed)
    m = degree + 1
    M = m ** dim
    Vc = dim + 2
    ncells = int(np.prod(ncell[:dim]))
    base = np.array([1.0] + [0.3, -0.2, 0.1][:dim] + [2.5])
    w = np.zeros((M, Vc + nvar_extra, ncells))
    for mode in range(M):
        rem, deg = mode, 0
        for _ in range(dim):
            deg += rem % m
            rem //= m
        for var in range(Vc):
            if mode == 0:
                w[mode, var] = base[var] * (1.0 + 0.05 * rng.standard_normal(ncells))
            else:
                w[mode, var] = amp * base[0] * rng.standard_normal(ncells) / (1.0 + deg) ** 2
        for var in range(Vc, Vc + nvar_extra):   # e.g. an alpha field in [0, ~0.5]
            w[mode, var] = (0.3 if mode == 0 else 0.05 / (1.0 + deg) ** 2) * np.abs(rng.standard_normal(ncells))
    alpha = np.ascontiguousarray(w[:, Vc, :]).ravel() if nvar_extra else None   # layout [mode*Ncells + cell]
    return np.ascontiguousarray(w[:, :Vc, :]).ravel(), alpha


def initial_modes_slabbed(wl: Workload, seed=SEED, layers=8, out=None):
    """initial_modes() of a large 3D mesh built z-slab by z-slab (bounded host memory); same layout.
    `out` may be a preallocated flat float64 array (e.g. the numpy view of a pinned torch tensor)."""
    if wl.dim != 3 or wl.ncell[2] <= layers:
        w = initial_modes(wl, seed)
        if out is None:
            return w
        out[:] = w
        return out
    Vc, M, N = wl.dim + 2, wl.modes, wl.ncells
    if out is None:
        out = np.empty(M * Vc * N)
    full = out.reshape(M * Vc, N)
    plane = wl.ncell[0] * wl.ncell[1]
    for z0 in range(0, wl.ncell[2], layers):
        z1 = min(wl.ncell[2], z0 + layers)
        part = initial_modes(wl, seed, zslab=(z0, z1)).reshape(M * Vc, (z1 - z0) * plane)
        full[:, z0 * plane:z1 * plane] = part
    return out


def initial_modes_wave_by_shift(wl: Workload, seed=SEED, out=None):
    """initial_modes() of the 3D advected wave on a cubic mesh at the cost of ONE z-layer: the IC depends on x+y+z
    only, so cell (ix, iy, iz) carries the modes of cell ((ix + iz) mod N, iy, 0); the other layers are cyclic shifts
    of the projected layer iz = 0 (equal to the direct projection up to its rounding).  For bench.py's order sweep,
    where projecting 64^3 cells at degree 7 point by point takes longer than the timed run."""
    assert wl.ic == "wave" and wl.dim == 3 and wl.ncell[0] == wl.ncell[1] == wl.ncell[2]
    N = wl.ncell[0]
    R = wl.modes * (wl.dim + 2)
    layer = initial_modes(wl, seed, zslab=(0, 1)).reshape(R, N, N)          # [row, iy, ix]
    if out is None:
        out = np.empty(R * N ** 3)
    full = out.reshape(R, N, N, N)                                            # [row, iz, iy, ix]
    for iz in range(N):
        full[:, iz] = np.roll(layer, -iz, axis=2)
    return out


def supersonic_modes(dim, ncell, degree, gamma, axis, sign, mach=2.5, seed=SEED, amp=0.01):
    """Seeded smooth state whose mean flow is supersonic along +/- `axis` (Mach ~ `mach`), so that every face normal
    to that axis takes the fully upwinded branch of the Riemann solver (S_L >= 0 for sign = +1, S_R <= 0 for
    sign = -1).  Cell means from primitive variables rho = 1, P = 1, v = sign * mach * c_s along the axis and
    0.2 c_s on the other axes, each perturbed by 3 % per cell (so the mean pressure stays positive); higher modes iid
    normal scaled by amp / (1 + sum l_a)^2.  Holds no method arithmetic beyond the definition of e (Eq. 2-3)."""
    rng = np.random.default_rng(seed)
    m = degree + 1
    M = m ** dim
    Vc = dim + 2
    ncells = int(np.prod(ncell[:dim]))
    cs = np.sqrt(gamma)
    v0 = np.full(dim, 0.2 * cs)
    v0[axis] = sign * mach * cs
    rho = 1.0 + 0.03 * rng.standard_normal(ncells)
    vel = v0[:, None] * (1.0 + 0.03 * rng.standard_normal((dim, ncells)))
    prs = 1.0 + 0.03 * rng.standard_normal(ncells)
    w = np.zeros((M, Vc, ncells))
    w[0, 0] = rho
    w[0, 1:1 + dim] = rho * vel
    w[0, 1 + dim] = prs / (gamma - 1.0) + 0.5 * rho * np.sum(vel * vel, axis=0)
    for mode in range(1, M):
        rem, deg = mode, 0
        for _ in range(dim):
            deg += rem % m
            rem //= m
        w[mode] = amp * rng.standard_normal((Vc, ncells)) / (1.0 + deg) ** 2
    return w.ravel()


def alpha_field(dim, ncell, degree, lo=-0.2, hi=1.5, seed=SEED):
    """Seeded artificial-viscosity field whose cell means cover [lo, hi] evenly (in random order) (both ends of the clamp
    0 <= alpha <= alpha_max of Eq. 46 act), small higher modes; layout [mode*Ncells + cell]."""
    rng = np.random.default_rng(seed + 17)
    m = degree + 1
    M = m ** dim
    ncells = int(np.prod(ncell[:dim]))
    a = np.zeros((M, ncells))
    a[0] = rng.permutation(np.linspace(lo, hi, ncells))      # both ends are present on any mesh
    for mode in range(1, M):
        rem, deg = mode, 0
        for _ in range(dim):
            deg += rem % m
            rem //= m
        a[mode] = 0.03 * rng.standard_normal(ncells) / (1.0 + deg) ** 2
    return a.ravel()
