"""Independent evaluators used to PIN the oracle (tests only; pure numpy/Python).

Nothing here is copied from oracle/rts_oracle.c: the formal solution is evaluated by
numerical quadrature of its defining integral, the upwind point is found
geometrically (walk back along the ray until the first cell-face plane) and the
upwind values are obtained by a generic trilinear interpolation at that point, and
the dependency order is resolved by memoised recursion instead of a sweep.
"""
from __future__ import annotations

import math
from functools import lru_cache

import numpy as np

_GL_X, _GL_W = np.polynomial.legendre.leggauss(24)


def formal_integral(Iu: float, Su: float, Sp: float, dtau: float) -> float:
    """I_p = I_u e^{-dtau} + int_0^dtau S(t) e^{-(dtau - t)} dt, S linear in t from S_u to S_p.

    Transfer equation dI/dt = S - I along the ray, t = optical path from the upwind point
    (sec 5.1; linear source function: SURVEY 8(c) R6).  Evaluated by 24-point
    Gauss-Legendre quadrature (exact to rounding for dtau up to ~30; the integrand is a
    polynomial times an exponential), NOT by the closed-form psi weights.
    """
    if dtau == 0.0:
        return Iu
    # for large dtau only the last ~40 optical depths matter; integrate over that window
    lo = max(0.0, dtau - 40.0)
    t = 0.5 * (dtau - lo) * (_GL_X + 1.0) + lo
    w = 0.5 * (dtau - lo) * _GL_W
    S = Su + (Sp - Su) * t / dtau
    if dtau - lo > 8.0:
        # split the window so that the quadrature stays accurate
        total = 0.0
        edges = np.linspace(lo, dtau, int(math.ceil((dtau - lo) / 4.0)) + 1)
        for a, b in zip(edges[:-1], edges[1:]):
            tt = 0.5 * (b - a) * (_GL_X + 1.0) + a
            ww = 0.5 * (b - a) * _GL_W
            SS = Su + (Sp - Su) * tt / dtau
            total += float(np.sum(ww * SS * np.exp(-(dtau - tt))))
        return Iu * math.exp(-dtau) + total
    return Iu * math.exp(-dtau) + float(np.sum(w * S * np.exp(-(dtau - t))))


def upwind_point(node, mu, h):
    """Geometric upwind point of `node` (index coords) for direction `mu`.

    Walk back from the node along -mu until the first plane x_a = node_a -+ 1 is hit
    (short characteristics, nearest upwind cell-face intersection).
    Returns (point in index coordinates, path length in cm).
    """
    ts = []
    for a in range(3):
        ts.append(h[a] / abs(mu[a]) if mu[a] != 0.0 else math.inf)
    ds = min(ts)
    pt = [node[a] - ds * mu[a] / h[a] for a in range(3)]
    # snap the coordinate of the face that was hit to an exact integer
    for a in range(3):
        if ts[a] == ds:
            pt[a] = float(node[a] - (1 if mu[a] > 0 else -1))
    return pt, ds


def trilinear_nodes(pt):
    """Generic trilinear interpolation stencil at `pt`: list of ((i,j,k), weight), weight>0."""
    base = [math.floor(c) for c in pt]
    frac = [c - b for c, b in zip(pt, base)]
    out = []
    for ei in (0, 1):
        for ej in (0, 1):
            for ek in (0, 1):
                w = ((frac[0] if ei else 1 - frac[0]) * (frac[1] if ej else 1 - frac[1])
                     * (frac[2] if ek else 1 - frac[2]))
                if w > 0.0:
                    out.append(((base[0] + ei, base[1] + ej, base[2] + ek), w))
    return out


def recursive_solve(kaprho: np.ndarray, S: np.ndarray, mu, h, npasses: int) -> np.ndarray:
    """I^(P) for one band and one ray by memoised recursion (tiny grids only).

    value(node, p): boundary plane -> boundary value; p == 0 -> S; otherwise the formal
    integral from the geometric upwind point, whose stencil nodes are taken at pass p when
    their horizontal indices are inside the box and at pass p-1 (wrapped) when not
    (SURVEY 8(c) O-5).  No sweep order anywhere.
    """
    nz, ny, nx = S.shape
    up = mu[2] > 0
    kdir = 0 if up else nz - 1

    @lru_cache(maxsize=None)
    def value(i: int, j: int, k: int, p: int) -> float:
        if k == kdir:
            return float(S[k, j, i]) if up else 0.0
        if p == 0:
            return float(S[k, j, i])
        pt, ds = upwind_point((i, j, k), mu, h)
        Iu = ku = Su = 0.0
        for (a, b, c), w in trilinear_nodes(pt):
            wrapped = not (0 <= a < nx and 0 <= b < ny)
            aa, bb = a % nx, b % ny
            Iu += w * value(aa, bb, c, p - 1 if wrapped else p)
            ku += w * float(kaprho[c, bb, aa])
            Su += w * float(S[c, bb, aa])
        dtau = 0.5 * (ku + float(kaprho[k, j, i])) * ds
        return formal_integral(Iu, Su, float(S[k, j, i]), dtau)

    out = np.empty_like(S, dtype=np.float64)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                out[k, j, i] = value(i, j, k, npasses)
    return out


def oned_zface(kaprho_z: np.ndarray, S_z: np.ndarray, muz: float, dz: float) -> np.ndarray:
    """1-D plane-parallel recurrence for a ray that steps exactly one level per segment.

    Horizontally uniform medium, ray leaving each cell through its z face: the upwind point
    is on the previous level, where everything equals that level's value.  Uses the
    quadrature form of the formal integral.  Upward for muz > 0 (bottom I = S), downward
    for muz < 0 (top I = 0).
    """
    nz = S_z.shape[0]
    I = np.empty(nz, dtype=np.float64)
    ds = dz / abs(muz)
    if muz > 0:
        I[0] = S_z[0]
        for k in range(1, nz):
            dtau = 0.5 * (kaprho_z[k - 1] + kaprho_z[k]) * ds
            I[k] = formal_integral(I[k - 1], S_z[k - 1], S_z[k], dtau)
    else:
        I[nz - 1] = 0.0
        for k in range(nz - 2, -1, -1):
            dtau = 0.5 * (kaprho_z[k + 1] + kaprho_z[k]) * ds
            I[k] = formal_integral(I[k + 1], S_z[k + 1], S_z[k], dtau)
    return I
