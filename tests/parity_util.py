"""Shared helpers of the GPU parity tests: oracle/GPU construction from one Workload and the parity norm."""
import numpy as np

from oracle import dg_oracle as orc
from paper_2208_11131_b200 import workloads as wk


def make_oracle(wl, **opt_kw):
    opt = orc.Options(f_cfl=wl.f_cfl, av_enable=wl.av, **opt_kw)
    return orc.DGOracle(wl.dim, wl.ncell, wl.h, wl.order, wl.gamma, wl.nu, wl.chi, opt)


def make_gpu(wl, **opt_kw):
    from paper_2208_11131_b200 import dg
    return dg.from_workload(wl, **opt_kw)


def parity_norm(w_gpu, w_orc, wl):
    """DESIGN.md reading A24: per conserved variable max_{cell,mode} |w_gpu - w_orc| / scale_var, where scale_var
    is the L-infinity norm of that variable's cell means; the momentum components share
    max(rho_mean * c_s_mean + |rho v|_mean) so that an identically-zero component is not divided by ~0."""
    d, Vc = wl.dim, wl.dim + 2
    M = wl.modes
    a = np.asarray(w_gpu).reshape(M, Vc, -1)
    b = np.asarray(w_orc).reshape(M, Vc, -1)
    mean = b[0]                                   # mode 0 = cell mean (P_0 = 1)
    rho = mean[0]
    mom = mean[1:1 + d]
    e = mean[1 + d]
    p = (wl.gamma - 1.0) * (e - 0.5 * np.sum(mom * mom, axis=0) / rho)
    cs = np.sqrt(np.abs(wl.gamma * p / rho))
    scale = np.empty(Vc)
    scale[0] = np.max(np.abs(rho))
    scale[1:1 + d] = np.max(rho * cs + np.sqrt(np.sum(mom * mom, axis=0)))
    scale[1 + d] = np.max(np.abs(e))
    diff = np.max(np.abs(a - b), axis=(0, 2))
    return diff / scale


def rhs_scale(L_orc, wl):
    """Scale for dw/dt comparisons: L-infinity norm of the oracle's dw/dt per variable (momentum shared)."""
    d, Vc = wl.dim, wl.dim + 2
    b = np.asarray(L_orc).reshape(wl.modes, Vc, -1)
    s = np.max(np.abs(b), axis=(0, 2))
    s[1:1 + d] = np.max(s[1:1 + d])
    return np.maximum(s, 1e-300)
