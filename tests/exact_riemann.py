"""Exact solution of the Riemann problem for the Euler equations (ideal gas).

Textbook construction (Toro 2009, ch. 4; cited by PAPER.md L313): the star pressure is
the root of f_L(p) + f_R(p) + u_R - u_L = 0 with f_K the shock (Rankine-Hugoniot) or
rarefaction (isentropic + Riemann invariant) branch; the solution is then sampled along
x/t.  Independent of oracle/ and of the CUDA path; pinned by tests/golden/sod_star.txt.
"""
import numpy as np


def _f(p, rho, pk, g):
    a = np.sqrt(g * pk / rho)
    if p > pk:   # shock
        A = 2.0 / ((g + 1) * rho)
        B = (g - 1) / (g + 1) * pk
        return (p - pk) * np.sqrt(A / (p + B))
    return 2 * a / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1.0)


def star(rl, ul, pl, rr, ur, pr, g):
    lo, hi = 1e-12, 10 * max(pl, pr)
    F = lambda p: _f(p, rl, pl, g) + _f(p, rr, pr, g) + ur - ul
    for _ in range(200):      # bisection: slow, obviously correct
        mid = 0.5 * (lo + hi)
        if F(mid) > 0:
            hi = mid
        else:
            lo = mid
    p = 0.5 * (lo + hi)
    u = 0.5 * (ul + ur) + 0.5 * (_f(p, rr, pr, g) - _f(p, rl, pl, g))
    return p, u


def sample(xi, rl, ul, pl, rr, ur, pr, g):
    """(rho, u, p) at similarity coordinate(s) xi = x/t."""
    ps, us = star(rl, ul, pl, rr, ur, pr, g)
    xi = np.atleast_1d(np.asarray(xi, dtype=float))
    out = np.empty((3, xi.size))
    al, ar = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)
    for n, s in enumerate(xi):
        if s <= us:   # left of the contact
            if ps > pl:
                sl = ul - al * np.sqrt((g + 1) / (2 * g) * ps / pl + (g - 1) / (2 * g))
                if s <= sl:
                    w = (rl, ul, pl)
                else:
                    w = (rl * ((ps / pl + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pl + 1)), us, ps)
            else:
                head = ul - al
                asl = al * (ps / pl) ** ((g - 1) / (2 * g))
                tail = us - asl
                if s <= head:
                    w = (rl, ul, pl)
                elif s >= tail:
                    w = (rl * (ps / pl) ** (1 / g), us, ps)
                else:
                    c = 2 / (g + 1) + (g - 1) / ((g + 1) * al) * (ul - s)
                    w = (rl * c ** (2 / (g - 1)), 2 / (g + 1) * (al + (g - 1) / 2 * ul + s), pl * c ** (2 * g / (g - 1)))
        else:
            if ps > pr:
                sr = ur + ar * np.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
                if s >= sr:
                    w = (rr, ur, pr)
                else:
                    w = (rr * ((ps / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pr + 1)), us, ps)
            else:
                head = ur + ar
                asr = ar * (ps / pr) ** ((g - 1) / (2 * g))
                tail = us + asr
                if s >= head:
                    w = (rr, ur, pr)
                elif s <= tail:
                    w = (rr * (ps / pr) ** (1 / g), us, ps)
                else:
                    c = 2 / (g + 1) - (g - 1) / ((g + 1) * ar) * (ur - s)
                    w = (rr * c ** (2 / (g - 1)), 2 / (g + 1) * (-ar + (g - 1) / 2 * ur + s), pr * c ** (2 * g / (g - 1)))
        out[:, n] = w
    return out
