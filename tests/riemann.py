"""Exact solution of the 1D Riemann problem for the Euler equations with an ideal gas.

The standard construction (pressure function with shock / rarefaction branches, Newton iteration for p*,
then sampling along x/t), as the paper does "following the procedure shown in [61]" (Toro's textbook;
PAPER.md:537).  Used ONLY by the tests as an independent pin for the oracle; not part of the product.
"""
import numpy as np


def _f_and_df(p, rho_k, p_k, c_k, g):
    if p > p_k:  # shock
        A = 2.0 / ((g + 1.0) * rho_k)
        B = (g - 1.0) / (g + 1.0) * p_k
        s = np.sqrt(A / (p + B))
        return (p - p_k) * s, s * (1.0 - 0.5 * (p - p_k) / (B + p))
    pr = p / p_k  # rarefaction
    return 2.0 * c_k / (g - 1.0) * (pr ** ((g - 1.0) / (2.0 * g)) - 1.0), (1.0 / (rho_k * c_k)) * pr ** (-(g + 1.0) / (2.0 * g))


def star_state(rhoL, uL, pL, rhoR, uR, pR, g=1.4, tol=1e-14):
    cL, cR = np.sqrt(g * pL / rhoL), np.sqrt(g * pR / rhoR)
    p = max(1e-12, 0.5 * (pL + pR))
    for _ in range(200):
        fL, dL = _f_and_df(p, rhoL, pL, cL, g)
        fR, dR = _f_and_df(p, rhoR, pR, cR, g)
        pn = p - (fL + fR + (uR - uL)) / (dL + dR)
        pn = max(pn, 1e-14)
        if abs(pn - p) <= tol * 0.5 * (pn + p):
            p = pn
            break
        p = pn
    fL, _ = _f_and_df(p, rhoL, pL, cL, g)
    fR, _ = _f_and_df(p, rhoR, pR, cR, g)
    u = 0.5 * (uL + uR) + 0.5 * (fR - fL)
    gm = (g - 1.0) / (g + 1.0)
    rho_sL = rhoL * ((p / pL + gm) / (gm * p / pL + 1.0)) if p > pL else rhoL * (p / pL) ** (1.0 / g)
    rho_sR = rhoR * ((p / pR + gm) / (gm * p / pR + 1.0)) if p > pR else rhoR * (p / pR) ** (1.0 / g)
    return p, u, rho_sL, rho_sR


def sample(xi, rhoL, uL, pL, rhoR, uR, pR, g=1.4):
    """(rho, u, p) at similarity coordinates xi = (x - x0)/t (array)."""
    xi = np.asarray(xi, dtype=np.float64)
    ps, us, rsL, rsR = star_state(rhoL, uL, pL, rhoR, uR, pR, g)
    cL, cR = np.sqrt(g * pL / rhoL), np.sqrt(g * pR / rhoR)
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    p = np.empty_like(xi)
    left = xi <= us
    # ---- left of the contact
    if ps > pL:
        SL = uL - cL * np.sqrt((g + 1.0) / (2.0 * g) * ps / pL + (g - 1.0) / (2.0 * g))
        a = left & (xi <= SL)
        b = left & (xi > SL)
        rho[a], u[a], p[a] = rhoL, uL, pL
        rho[b], u[b], p[b] = rsL, us, ps
    else:
        csL = cL * (ps / pL) ** ((g - 1.0) / (2.0 * g))
        head, tail = uL - cL, us - csL
        a = left & (xi <= head)
        b = left & (xi > head) & (xi < tail)
        c = left & (xi >= tail)
        rho[a], u[a], p[a] = rhoL, uL, pL
        fac = 2.0 / (g + 1.0) + (g - 1.0) / ((g + 1.0) * cL) * (uL - xi[b])
        rho[b] = rhoL * fac ** (2.0 / (g - 1.0))
        u[b] = 2.0 / (g + 1.0) * (cL + (g - 1.0) / 2.0 * uL + xi[b])
        p[b] = pL * fac ** (2.0 * g / (g - 1.0))
        rho[c], u[c], p[c] = rsL, us, ps
    # ---- right of the contact
    right = ~left
    if ps > pR:
        SR = uR + cR * np.sqrt((g + 1.0) / (2.0 * g) * ps / pR + (g - 1.0) / (2.0 * g))
        a = right & (xi >= SR)
        b = right & (xi < SR)
        rho[a], u[a], p[a] = rhoR, uR, pR
        rho[b], u[b], p[b] = rsR, us, ps
    else:
        csR = cR * (ps / pR) ** ((g - 1.0) / (2.0 * g))
        head, tail = uR + cR, us + csR
        a = right & (xi >= head)
        b = right & (xi < head) & (xi > tail)
        c = right & (xi <= tail)
        rho[a], u[a], p[a] = rhoR, uR, pR
        fac = 2.0 / (g + 1.0) - (g - 1.0) / ((g + 1.0) * cR) * (uR - xi[b])
        rho[b] = rhoR * fac ** (2.0 / (g - 1.0))
        u[b] = 2.0 / (g + 1.0) * (-cR + (g - 1.0) / 2.0 * uR + xi[b])
        p[b] = pR * fac ** (2.0 * g / (g - 1.0))
        rho[c], u[c], p[c] = rsR, us, ps
    return rho, u, p


def sod_wave_speeds(g=1.4):
    """shock speed, rarefaction head and tail for the Sod data (1,0,1 | 0.125,0,0.1)."""
    ps, us, rsL, rsR = star_state(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g)
    cL, cR = np.sqrt(g * 1.0 / 1.0), np.sqrt(g * 0.1 / 0.125)
    shock = cR * np.sqrt((g + 1.0) / (2.0 * g) * ps / 0.1 + (g - 1.0) / (2.0 * g))
    head = -cL
    tail = us - cL * (ps / 1.0) ** ((g - 1.0) / (2.0 * g))
    return shock, head, tail
