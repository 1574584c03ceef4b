"""Exact Riemann solver for the 1-D Euler equations (Toro 2009, ch. 4) -- a test-side pin,
independent of oracle/ and of the CUDA path.  Used to sample the exact Sod solution and exact
Godunov fluxes."""
import math

import numpy as np


def _f(p, rho, pk, gamma):
    a = math.sqrt(gamma * pk / rho)
    if p > pk:   # shock
        A = 2.0 / ((gamma + 1.0) * rho)
        B = (gamma - 1.0) / (gamma + 1.0) * pk
        s = math.sqrt(A / (p + B))
        return (p - pk) * s, s * (1.0 - 0.5 * (p - pk) / (B + p))
    pr = p / pk  # rarefaction
    return (2.0 * a / (gamma - 1.0) * (pr ** ((gamma - 1.0) / (2.0 * gamma)) - 1.0),
            1.0 / (rho * a) * pr ** (-(gamma + 1.0) / (2.0 * gamma)))


def star_state(rl, ul, pl, rr, ur, pr, gamma):
    p = max(1e-12, 0.5 * (pl + pr))
    for _ in range(200):
        fl, dfl = _f(p, rl, pl, gamma)
        fr, dfr = _f(p, rr, pr, gamma)
        pn = p - (fl + fr + ur - ul) / (dfl + dfr)
        pn = max(pn, 1e-14)
        if abs(pn - p) <= 1e-15 * (pn + p):
            p = pn
            break
        p = pn
    fl, _ = _f(p, rl, pl, gamma)
    fr, _ = _f(p, rr, pr, gamma)
    return p, 0.5 * (ul + ur) + 0.5 * (fr - fl)


def sample(rl, ul, pl, rr, ur, pr, gamma, xi):
    """Exact (rho, u, p) at similarity coordinate xi = x/t (numpy array)."""
    xi = np.asarray(xi, dtype=np.float64)
    ps, us = star_state(rl, ul, pl, rr, ur, pr, gamma)
    g = gamma
    al, ar = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    p = np.empty_like(xi)
    for n, s in np.ndenumerate(xi):
        if s <= us:   # left of contact
            if ps > pl:
                sl = ul - al * math.sqrt((g + 1) / (2 * g) * ps / pl + (g - 1) / (2 * g))
                if s <= sl:
                    rho[n], u[n], p[n] = rl, ul, pl
                else:
                    rho[n] = rl * ((ps / pl + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pl + 1))
                    u[n], p[n] = us, ps
            else:
                shl = ul - al
                asl = al * (ps / pl) ** ((g - 1) / (2 * g))
                stl = us - asl
                if s <= shl:
                    rho[n], u[n], p[n] = rl, ul, pl
                elif s >= stl:
                    rho[n], u[n], p[n] = rl * (ps / pl) ** (1 / g), us, ps
                else:
                    c = 2 / (g + 1) + (g - 1) / ((g + 1) * al) * (ul - s)
                    rho[n] = rl * c ** (2 / (g - 1))
                    u[n] = 2 / (g + 1) * (al + (g - 1) / 2 * ul + s)
                    p[n] = pl * c ** (2 * g / (g - 1))
        else:
            if ps > pr:
                sr = ur + ar * math.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
                if s >= sr:
                    rho[n], u[n], p[n] = rr, ur, pr
                else:
                    rho[n] = rr * ((ps / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pr + 1))
                    u[n], p[n] = us, ps
            else:
                shr = ur + ar
                asr = ar * (ps / pr) ** ((g - 1) / (2 * g))
                strr = us + asr
                if s >= shr:
                    rho[n], u[n], p[n] = rr, ur, pr
                elif s <= strr:
                    rho[n], u[n], p[n] = rr * (ps / pr) ** (1 / g), us, ps
                else:
                    c = 2 / (g + 1) - (g - 1) / ((g + 1) * ar) * (ur - s)
                    rho[n] = rr * c ** (2 / (g - 1))
                    u[n] = 2 / (g + 1) * (-ar + (g - 1) / 2 * ur + s)
                    p[n] = pr * c ** (2 * g / (g - 1))
    return rho, u, p


def godunov_flux(rl, ul, vl, wl, pl, rr, ur, vr, wr, pr, gamma):
    """Exact flux (rho u, rho u^2 + p, rho u v, rho u w, u (E + p)) at x/t = 0."""
    rho, u, p = sample(rl, ul, pl, rr, ur, pr, gamma, np.array([0.0]))
    rho, u, p = float(rho[0]), float(u[0]), float(p[0])
    _, us = star_state(rl, ul, pl, rr, ur, pr, gamma)
    v, w = (vl, wl) if us >= 0.0 else (vr, wr)
    e = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)
    return np.array([rho * u, rho * u * u + p, rho * u * v, rho * u * w, u * (e + p)])
