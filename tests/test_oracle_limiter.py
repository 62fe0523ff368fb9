"""Pins of the oracle's positivity limiter (Eq. 47) -- CPU only.

What the paper fixes: the cell mean is untouched; after the density step the minimum density over the union of volume
and face quadrature points is exactly rho_bottom = 1e-6 rho_bar ("this limits the minimum density ... to rho_bottom");
all fields get the same factor; the pressure step halves the higher modes until p_min >= p_bottom; smooth states are
not touched.  Point values are re-evaluated here by brute force (loops over modes with recurrence-evaluated Legendre
values at explicitly listed points), not with the oracle's evaluation matrices.
"""
import itertools

import numpy as np

from oracle import dg_oracle as orc


def _points(d, m):
    """Reference coordinates of the evaluation points: m^d volume Gauss points and the m^(d-1) Gauss points of each of
    the 2d faces."""
    x, _ = orc.gauss_legendre(m)
    pts = [p[::-1] for p in itertools.product(x, repeat=d)]            # x fastest
    for a in range(d):
        for side in (-1.0, 1.0):
            for t in itertools.product(x, repeat=d - 1):
                t = list(t[::-1])
                t.insert(a, side)
                pts.append(tuple(t))
    return np.array(pts)


def _evaluate(wc, d, m, gamma, pts):
    """Brute-force u(xi) = sum_l w_l prod_a P_{l_a}(xi_a) for one cell wc[mode, var]."""
    out = np.zeros((len(pts), wc.shape[1]))
    for ip, xi in enumerate(pts):
        P = [orc.legendre_normalised(m - 1, np.array(xi[a]))[0] for a in range(d)]
        for mode in range(m ** d):
            rem, phi = mode, 1.0
            for a in range(d):
                phi *= float(P[a][rem % m])
                rem //= m
            out[ip] += phi * wc[mode]
    return out


def _pressure(u, d, gamma):
    return (gamma - 1.0) * (u[:, 1 + d] - 0.5 * np.sum(u[:, 1:1 + d] ** 2, axis=1) / u[:, 0])


def _oracle(d, n, av=False):
    nc = (2, 2, 2)[:d]
    return orc.DGOracle(d, nc, 0.5, n + 1, 1.4, options=orc.Options(limiter_enable=True, av_enable=av))


def _base_state(o, rng, amp):
    w = np.zeros_like(o.w)
    w[:, 0, 0] = 1.0 + 0.1 * rng.random(o.ncells)
    w[:, 0, 1:1 + o.d] = 0.2 * rng.standard_normal((o.ncells, o.d))
    w[:, 0, 1 + o.d] = 2.5
    w[:, 1:, :o.Vc] = amp * rng.standard_normal((o.ncells, o.M - 1, o.Vc))
    return w


def test_smooth_state_is_untouched_bitwise():
    rng = np.random.default_rng(1)
    for d, n in [(2, 1), (2, 3), (3, 2)]:
        o = _oracle(d, n)
        w = _base_state(o, rng, 0.01)
        assert np.array_equal(o.positivity_limit(w), w)
        assert not o.unphysical


def test_density_limiter_closed_form():
    rng = np.random.default_rng(2)
    for d, n in [(2, 1), (2, 4), (3, 1), (3, 3)]:
        o = _oracle(d, n, av=True)
        m = n + 1
        pts = _points(d, m)
        w = _base_state(o, rng, 0.01)
        w[:, :, o.Vc:] = rng.random((o.ncells, o.M, w.shape[2] - o.Vc))      # alpha field
        w[:2, :, 1:1 + d] = 0.0   # gas at rest in the two test cells: the pressure step must not act (p = (gamma-1) e > 0)
        w[0, 1, 0] = 1.3          # P_1 along x: density far below zero on the lower x face, not at a volume point
        w[1, o.M - 1, 0] = -0.9   # highest mode
        before = _evaluate(w[0, :, :o.Vc], d, m, 1.4, pts)
        assert before[:m ** d, 0].min() > before[:, 0].min()                 # the minimum sits on a face point
        w2 = o.positivity_limit(w)
        for c in (0, 1):
            u = _evaluate(w2[c, :, :o.Vc], d, m, 1.4, pts)
            rho_bar = w[c, 0, 0]
            assert np.array_equal(w2[c, 0], w[c, 0])                         # cell means untouched
            assert abs(u[:, 0].min() - 1e-6 * rho_bar) < 1e-13 * rho_bar      # min density is exactly rho_bottom
            sel = w[c, 1:, :o.Vc] != 0.0
            ratio = w2[c, 1:, :o.Vc][sel] / w[c, 1:, :o.Vc][sel]
            assert np.ptp(ratio) < 1e-14 and 0.0 < ratio.flat[0] < 1.0       # one factor for all fields
            assert _pressure(u, d, 1.4).min() >= 1e-6 * _pressure(w[c:c + 1, 0, :o.Vc], d, 1.4)[0]
        assert np.array_equal(w2[2:], w[2:])                                 # other cells untouched
        assert np.array_equal(w2[:, :, o.Vc:], w[:, :, o.Vc:])               # alpha untouched (reading L5)


def test_pressure_limiter_halves_until_positive():
    rng = np.random.default_rng(3)
    for d, n in [(2, 2), (3, 2)]:
        o = _oracle(d, n)
        m = n + 1
        pts = _points(d, m)
        w = _base_state(o, rng, 0.005)
        w[0, 1, 1 + d] = 2.2      # energy oscillation: pressure negative near one x face, density stays positive
        u0 = _evaluate(w[0, :, :o.Vc], d, m, 1.4, pts)
        assert u0[:, 0].min() > 0.5 and _pressure(u0, d, 1.4).min() < 0.0
        w2 = o.positivity_limit(w)
        p_bar = _pressure(w[0:1, 0, :o.Vc], d, 1.4)[0]
        u = _evaluate(w2[0, :, :o.Vc], d, m, 1.4, pts)
        assert _pressure(u, d, 1.4).min() >= 1e-6 * p_bar
        ratio = w2[0, 1:, :o.Vc] / w[0, 1:, :o.Vc]
        k = np.log2(1.0 / ratio.flat[0])
        assert np.ptp(ratio) < 1e-15 and abs(k - round(k)) < 1e-12 and round(k) >= 1     # factor 0.5^k exactly
        wprev = w.copy()
        wprev[0, 1:, :o.Vc] *= 2.0 * ratio.flat[0]                                        # one halving less
        assert _pressure(_evaluate(wprev[0, :, :o.Vc], d, m, 1.4, pts), d, 1.4).min() < 1e-6 * p_bar
        assert np.array_equal(w2[1:], w[1:]) and np.array_equal(w2[0, 0], w[0, 0])


def test_negative_mean_is_flagged():
    o = _oracle(2, 2)
    w = _base_state(o, np.random.default_rng(4), 0.01)
    w[1, 0, 3] = 0.01            # mean pressure negative: (gamma-1)(e - |m|^2/2rho) < 0 with m != 0
    w[1, 0, 1] = 1.0
    w2 = o.positivity_limit(w)
    assert o.unphysical and np.array_equal(w2, w)


def test_limiter_is_inactive_on_smooth_steps():
    """"does not trigger for inherently smooth problems": steps with and without it are bit-identical."""
    res = []
    for lim in (False, True):
        o = orc.DGOracle(2, (4, 3), 0.25, 3, 1.4, options=orc.Options(limiter_enable=lim, f_cfl=0.3))
        w = _base_state(o, np.random.default_rng(5), 0.01)
        o.w = w
        assert o.step(2) == 0
        res.append(o.w.copy())
    assert np.array_equal(res[0], res[1])
