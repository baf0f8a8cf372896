"""Exact solution of the 1D Riemann problem for the ideal-gas Euler equations (test helper).

Restates the classical exact solver (two-rarefaction / two-shock pressure functions, Newton
iteration on p*, then sampling of the self-similar solution) described in Toro's book
(PAPER.md ref. 39, L414).  Test infrastructure only; used to pin the oracle."""
import numpy as np


def _f(p, rho_k, p_k, g):
    a_k = np.sqrt(g * p_k / rho_k)
    if p > p_k:  # shock
        A, B = 2.0 / ((g + 1) * rho_k), (g - 1) / (g + 1) * p_k
        s = np.sqrt(A / (p + B))
        return (p - p_k) * s, s * (1.0 - 0.5 * (p - p_k) / (B + p))
    pr = p / p_k  # rarefaction
    return 2 * a_k / (g - 1) * (pr ** ((g - 1) / (2 * g)) - 1.0), (1.0 / (rho_k * a_k)) * pr ** (-(g + 1) / (2 * g))


def star_state(rl, ul, pl, rr, ur, pr, g=1.4):
    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dl = _f(p, rl, pl, g)
        fr, dr = _f(p, rr, pr, g)
        pn = max(1e-12, p - (fl + fr + ur - ul) / (dl + dr))
        if abs(pn - p) < 1e-15 * (pn + p):
            p = pn
            break
        p = pn
    fl, _ = _f(p, rl, pl, g)
    fr, _ = _f(p, rr, pr, g)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    gm = (g - 1) / (g + 1)
    rsl = rl * ((p / pl + gm) / (gm * p / pl + 1)) if p > pl else rl * (p / pl) ** (1 / g)
    rsr = rr * ((p / pr + gm) / (gm * p / pr + 1)) if p > pr else rr * (p / pr) ** (1 / g)
    return p, u, rsl, rsr


def sample(xi, rl, ul, pl, rr, ur, pr, g=1.4):
    """(rho, u, p) at similarity coordinates xi = (x - x0)/t (array)."""
    xi = np.asarray(xi, dtype=np.float64)
    ps, us, rsl, rsr = star_state(rl, ul, pl, rr, ur, pr, g)
    al, ar = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)
    rho, u, p = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    for n, s in enumerate(xi.ravel()):
        if s <= us:  # left of the contact
            if ps > pl:  # left shock
                sl = ul - al * np.sqrt((g + 1) / (2 * g) * ps / pl + (g - 1) / (2 * g))
                v = (rl, ul, pl) if s < sl else (rsl, us, ps)
            else:
                asl = al * (ps / pl) ** ((g - 1) / (2 * g))
                if s < ul - al:
                    v = (rl, ul, pl)
                elif s > us - asl:
                    v = (rsl, us, ps)
                else:
                    c = 2 / (g + 1) + (g - 1) / ((g + 1) * al) * (ul - s)
                    v = (rl * c ** (2 / (g - 1)), 2 / (g + 1) * (al + (g - 1) / 2 * ul + s),
                         pl * c ** (2 * g / (g - 1)))
        else:
            if ps > pr:  # right shock
                sr = ur + ar * np.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
                v = (rr, ur, pr) if s > sr else (rsr, us, ps)
            else:
                asr = ar * (ps / pr) ** ((g - 1) / (2 * g))
                if s > ur + ar:
                    v = (rr, ur, pr)
                elif s < us + asr:
                    v = (rsr, us, ps)
                else:
                    c = 2 / (g + 1) - (g - 1) / ((g + 1) * ar) * (ur - s)
                    v = (rr * c ** (2 / (g - 1)), 2 / (g + 1) * (-ar + (g - 1) / 2 * ur + s),
                         pr * c ** (2 * g / (g - 1)))
        rho.flat[n], u.flat[n], p.flat[n] = v
    return rho, u, p
