"""Exact Riemann solver for a single stiffened gas (test helper; textbook, Toro ch. 4 with p -> p + pi_inf).

Used only to pin the oracle (Sod tube, config-0 star state).  Independent of oracle/ and of the CUDA path.
"""
from __future__ import annotations

import numpy as np


def _f(p, rho, pk, g, pinf):
    """Pressure function of one side and its derivative."""
    P, PK = p + pinf, pk + pinf
    if p > pk:  # shock
        A = 2.0 / ((g + 1.0) * rho)
        B = (g - 1.0) / (g + 1.0) * PK
        s = np.sqrt(A / (P + B))
        return (p - pk) * s, s * (1.0 - 0.5 * (p - pk) / (P + B))
    c = np.sqrt(g * PK / rho)  # rarefaction
    r = P / PK
    return 2.0 * c / (g - 1.0) * (r ** ((g - 1.0) / (2.0 * g)) - 1.0), (1.0 / (rho * c)) * r ** (-(g + 1.0) / (2.0 * g))


def star_state(rl, ul, pl, rr, ur, pr, gl, pil, gr=None, pir=None):
    """Returns p*, u*, rho*_L, rho*_R for left fluid (gl, pil) and right fluid (gr, pir)."""
    gr = gl if gr is None else gr
    pir = pil if pir is None else pir
    lo = max(-pil, -pir) * (1 - 1e-12) + 1e-300
    p = max(0.5 * (pl + pr), lo + 1.0)
    for _ in range(200):
        fl, dfl = _f(p, rl, pl, gl, pil)
        fr, dfr = _f(p, rr, pr, gr, pir)
        g = fl + fr + (ur - ul)
        pn = p - g / (dfl + dfr)
        if pn <= lo:
            pn = 0.5 * (p + lo)
        if abs(pn - p) <= 1e-15 * abs(pn):
            p = pn
            break
        p = pn
    fl, _ = _f(p, rl, pl, gl, pil)
    fr, _ = _f(p, rr, pr, gr, pir)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)

    def rho_star(rho, pk, g, pinf):
        r = (p + pinf) / (pk + pinf)
        if p > pk:
            m = (g - 1.0) / (g + 1.0)
            return rho * (r + m) / (m * r + 1.0)
        return rho * r ** (1.0 / g)

    return p, u, rho_star(rl, pl, gl, pil), rho_star(rr, pr, gr, pir)


def sample(xi, rl, ul, pl, rr, ur, pr, g, pinf=0.0):
    """Self-similar solution rho, u, p at xi = (x - x0)/t for one fluid (g, pinf) on both sides."""
    ps, us, rsl, rsr = star_state(rl, ul, pl, rr, ur, pr, g, pinf)
    xi = np.asarray(xi, dtype=np.float64)
    rho = np.empty_like(xi); u = np.empty_like(xi); p = np.empty_like(xi)
    cl = np.sqrt(g * (pl + pinf) / rl)
    cr = np.sqrt(g * (pr + pinf) / rr)
    for k, s in enumerate(xi.flat):
        if s <= us:  # left of contact
            if ps > pl:
                S = ul - cl * np.sqrt((g + 1) / (2 * g) * (ps + pinf) / (pl + pinf) + (g - 1) / (2 * g))
                out = (rl, ul, pl) if s <= S else (rsl, us, ps)
            else:
                csl = cl * ((ps + pinf) / (pl + pinf)) ** ((g - 1) / (2 * g))
                if s <= ul - cl:
                    out = (rl, ul, pl)
                elif s >= us - csl:
                    out = (rsl, us, ps)
                else:
                    c = 2 / (g + 1) * (cl + (g - 1) / 2 * (ul - s))
                    uu = 2 / (g + 1) * (cl + (g - 1) / 2 * ul + s)
                    out = (rl * (c / cl) ** (2 / (g - 1)), uu, (pl + pinf) * (c / cl) ** (2 * g / (g - 1)) - pinf)
        else:
            if ps > pr:
                S = ur + cr * np.sqrt((g + 1) / (2 * g) * (ps + pinf) / (pr + pinf) + (g - 1) / (2 * g))
                out = (rr, ur, pr) if s >= S else (rsr, us, ps)
            else:
                csr = cr * ((ps + pinf) / (pr + pinf)) ** ((g - 1) / (2 * g))
                if s >= ur + cr:
                    out = (rr, ur, pr)
                elif s <= us + csr:
                    out = (rsr, us, ps)
                else:
                    c = 2 / (g + 1) * (cr - (g - 1) / 2 * (ur - s))
                    uu = 2 / (g + 1) * (-cr + (g - 1) / 2 * ur + s)
                    out = (rr * (c / cr) ** (2 / (g - 1)), uu, (pr + pinf) * (c / cr) ** (2 * g / (g - 1)) - pinf)
        rho.flat[k], u.flat[k], p.flat[k] = out
    return rho, u, p
