"""Exact Riemann solver for two (possibly different) stiffened gases, written for the tests only.

Textbook construction (two-rarefaction / two-shock branches of the pressure function, contact separating
the two materials); with p_inf = 0 it is the ideal-gas solver used for the Sod problem.  Works on the shifted
pressure P = p + p_inf on each side.  Shares nothing with oracle/ or the CUDA path.
"""
import numpy as np


def _f(P, rho, Pk, g):
    """pressure function of one side and its derivative; P, Pk are shifted pressures of that side."""
    if P > Pk:  # shock
        A = 2.0 / ((g + 1.0) * rho)
        B = (g - 1.0) / (g + 1.0) * Pk
        s = np.sqrt(A / (P + B))
        return (P - Pk) * s, s * (1.0 - 0.5 * (P - Pk) / (P + B))
    c = np.sqrt(g * Pk / rho)
    return 2.0 * c / (g - 1.0) * ((P / Pk) ** ((g - 1.0) / (2.0 * g)) - 1.0), 1.0 / (rho * c) * (P / Pk) ** (-(g + 1.0) / (2.0 * g))


def star(left, right):
    """left/right = (rho, u, p, gamma, p_inf). Returns p*, u*."""
    rl, ul, pl, gl, il = left
    rr, ur, pr, gr, ir = right
    lo = max(-il, -ir) + 1e-12 * max(abs(pl), abs(pr), 1.0)
    hi = max(pl, pr)

    def F(p):
        return _f(p + il, rl, pl + il, gl)[0] + _f(p + ir, rr, pr + ir, gr)[0] + (ur - ul)

    while F(hi) < 0.0:
        hi = 2.0 * hi + 1.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if F(mid) > 0.0:
            hi = mid
        else:
            lo = mid
    p = 0.5 * (lo + hi)
    u = 0.5 * (ul + ur) + 0.5 * (_f(p + ir, rr, pr + ir, gr)[0] - _f(p + il, rl, pl + il, gl)[0])
    return p, u


def sample(left, right, xi):
    """Solution (rho, u, p, is_left_material) at the similarity coordinates xi = x/t (numpy array)."""
    rl, ul, pl, gl, il = left
    rr, ur, pr, gr, ir = right
    ps, us = star(left, right)
    xi = np.asarray(xi, dtype=np.float64)
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    p = np.empty_like(xi)
    isl = xi < us
    for side, sgn in (("L", 1.0), ("R", -1.0)):
        if side == "L":
            r0, u0, p0, g, pinf, m = rl, ul, pl, gl, il, isl
        else:
            r0, u0, p0, g, pinf, m = rr, ur, pr, gr, ir, ~isl
        P0, Ps = p0 + pinf, ps + pinf
        c0 = np.sqrt(g * P0 / r0)
        x = xi[m]
        ro = np.empty_like(x)
        uo = np.empty_like(x)
        po = np.empty_like(x)
        if Ps > P0:  # shock on this side
            S = u0 - sgn * c0 * np.sqrt((g + 1.0) / (2.0 * g) * Ps / P0 + (g - 1.0) / (2.0 * g))
            rs = r0 * ((Ps / P0 + (g - 1.0) / (g + 1.0)) / ((g - 1.0) / (g + 1.0) * Ps / P0 + 1.0))
            pre = (x < S) if side == "L" else (x > S)
            ro[:] = np.where(pre, r0, rs)
            uo[:] = np.where(pre, u0, us)
            po[:] = np.where(pre, p0, ps)
        else:        # rarefaction
            cs = c0 * (Ps / P0) ** ((g - 1.0) / (2.0 * g))
            head, tail = u0 - sgn * c0, us - sgn * cs
            rs = r0 * (Ps / P0) ** (1.0 / g)
            pre = (x < head) if side == "L" else (x > head)
            post = (x > tail) if side == "L" else (x < tail)
            cf = 2.0 / (g + 1.0) * (c0 + sgn * (g - 1.0) / 2.0 * (u0 - x))
            uf = 2.0 / (g + 1.0) * (sgn * c0 + (g - 1.0) / 2.0 * u0 + x)
            rf = r0 * (np.abs(cf) / c0) ** (2.0 / (g - 1.0))
            Pf = P0 * (np.abs(cf) / c0) ** (2.0 * g / (g - 1.0))
            ro[:] = np.where(pre, r0, np.where(post, rs, rf))
            uo[:] = np.where(pre, u0, np.where(post, us, uf))
            po[:] = np.where(pre, p0, np.where(post, ps, Pf - pinf))
        rho[m], u[m], p[m] = ro, uo, po
    return rho, u, p, isl
