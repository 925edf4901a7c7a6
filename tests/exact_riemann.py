"""Exact solution of the 1-D Riemann problem for two stiffened gases separated by a contact
(each side a pure fluid with its own gamma, pi_inf).  Textbook construction (pressure function
solved by Newton iteration, ref. [31] of the paper) with p -> p + pi_inf per side.
Test-side code: it is NOT part of the oracle and shares nothing with it — it is what the
oracle's Sod / water-air runs are pinned against.
"""
import numpy as np


class Side:
    def __init__(self, rho, u, p, gamma, pinf):
        self.rho, self.u, self.p, self.g, self.pinf = rho, u, p, gamma, pinf
        self.ph = p + pinf
        self.c = np.sqrt(gamma * self.ph / rho)
        self.A = 2.0 / ((gamma + 1.0) * rho)
        self.B = (gamma - 1.0) / (gamma + 1.0) * self.ph

    def f(self, p):
        ph = p + self.pinf
        if ph > self.ph:  # shock
            s = np.sqrt(self.A / (ph + self.B))
            return (ph - self.ph) * s, s * (1.0 - 0.5 * (ph - self.ph) / (ph + self.B))
        e = (self.g - 1.0) / (2.0 * self.g)
        return 2.0 * self.c / (self.g - 1.0) * ((ph / self.ph) ** e - 1.0), (ph / self.ph) ** (-(self.g + 1.0) / (2.0 * self.g)) / (self.rho * self.c)

    def rho_star(self, p):
        r = (p + self.pinf) / self.ph
        if r > 1.0:
            m = (self.g - 1.0) / (self.g + 1.0)
            return self.rho * (r + m) / (m * r + 1.0)
        return self.rho * r ** (1.0 / self.g)


def solve_star(L, R):
    p = max(0.5 * (L.p + R.p), 1e-8)
    for _ in range(200):
        fl, dl = L.f(p)
        fr, dr = R.f(p)
        dp = (fl + fr + R.u - L.u) / (dl + dr)
        pn = p - dp
        lo = -min(L.pinf, R.pinf)
        if pn <= lo:
            pn = 0.5 * (p + lo) if lo > 0 or p > 0 else 1e-10
            pn = max(pn, 0.1 * p)
        conv = abs(pn - p) <= 1e-15 * max(abs(pn), abs(p))
        p = pn
        if conv:
            break
    fl, _ = L.f(p)
    fr, _ = R.f(p)
    return p, 0.5 * (L.u + R.u) + 0.5 * (fr - fl)


def sample(L, R, xi):
    """(rho, u, p, is_left_fluid) at similarity coordinate xi = (x - x0)/t (array)."""
    ps, us = solve_star(L, R)
    xi = np.asarray(xi, dtype=np.float64)
    rho = np.empty_like(xi); u = np.empty_like(xi); p = np.empty_like(xi)
    left = xi <= us
    for K, sgn, mask in ((L, -1.0, left), (R, +1.0, ~left)):
        rs = K.rho_star(ps)
        r = (ps + K.pinf) / K.ph
        x = xi[mask]
        rk = np.full_like(x, rs); uk = np.full_like(x, us); pk = np.full_like(x, ps)
        if r > 1.0:  # shock
            S = K.u + sgn * K.c * np.sqrt((K.g + 1.0) / (2.0 * K.g) * r + (K.g - 1.0) / (2.0 * K.g))
            out = (x < S) if sgn < 0 else (x > S)
            rk[out], uk[out], pk[out] = K.rho, K.u, K.p
        else:        # rarefaction
            cs = K.c * r ** ((K.g - 1.0) / (2.0 * K.g))
            head, tail = K.u + sgn * K.c, us + sgn * cs
            out = (x < head) if sgn < 0 else (x > head)
            fan = ((x >= head) & (x < tail)) if sgn < 0 else ((x <= head) & (x > tail))
            rk[out], uk[out], pk[out] = K.rho, K.u, K.p
            t = 2.0 / (K.g + 1.0) - sgn * (K.g - 1.0) / ((K.g + 1.0) * K.c) * (K.u - x[fan])
            rk[fan] = K.rho * t ** (2.0 / (K.g - 1.0))
            uk[fan] = 2.0 / (K.g + 1.0) * (-sgn * K.c + 0.5 * (K.g - 1.0) * K.u + x[fan])
            pk[fan] = K.ph * t ** (2.0 * K.g / (K.g - 1.0)) - K.pinf
        rho[mask], u[mask], p[mask] = rk, uk, pk
    return rho, u, p, left


def wave_speeds(L, R):
    """dict of characteristic positions xi: left head/tail or shock, contact, right shock or head/tail"""
    ps, us = solve_star(L, R)
    out = {"contact": us, "p_star": ps}
    for name, K, sgn in (("left", L, -1.0), ("right", R, 1.0)):
        r = (ps + K.pinf) / K.ph
        if r > 1.0:
            out[name + "_shock"] = K.u + sgn * K.c * np.sqrt((K.g + 1.0) / (2.0 * K.g) * r + (K.g - 1.0) / (2.0 * K.g))
        else:
            out[name + "_head"] = K.u + sgn * K.c
            out[name + "_tail"] = us + sgn * K.c * r ** ((K.g - 1.0) / (2.0 * K.g))
    return out
