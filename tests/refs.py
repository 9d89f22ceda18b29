"""Independent numpy references used ONLY to pin the oracle (tests/test_oracle_pins.py).

Nothing here is derived from oracle/rc_oracle.c: the ray/cell intersection is done by sorting
all grid-line crossing parameters (not by an incremental DDA), and the long-characteristics
solver integrates the transfer equation to the domain edge with a plain angular quadrature
("conventional long characteristics ray-casting").
"""
from __future__ import annotations

import numpy as np


def segments_by_sorting(nx, ny, px, py, theta, ta, tb):
    """Cells and lengths of {p + t w, ta<=t<=tb} within [0,nx]x[0,ny]: clip, collect every
    crossing with a vertical or horizontal grid line, sort, take the cell of each midpoint."""
    wx, wy = np.cos(theta), np.sin(theta)
    lo, hi = ta, tb
    for p, w, n in ((px, wx, nx), (py, wy, ny)):  # slab clip
        if w == 0.0:
            if not (0.0 <= p <= n):
                return np.zeros(0, int), np.zeros(0)
            continue
        t0, t1 = (0.0 - p) / w, (n - p) / w
        lo, hi = max(lo, min(t0, t1)), min(hi, max(t0, t1))
    if not hi > lo:
        return np.zeros(0, int), np.zeros(0)
    ts = [lo, hi]
    for p, w, n in ((px, wx, nx), (py, wy, ny)):
        if w != 0.0:
            g = np.arange(0, n + 1)
            t = (g - p) / w
            ts.extend(t[(t > lo) & (t < hi)])
    ts = np.unique(np.array(ts))
    mid = 0.5 * (ts[1:] + ts[:-1])
    ds = np.diff(ts)
    ix = np.floor(px + mid * wx).astype(int)
    iy = np.floor(py + mid * wy).astype(int)
    keep = (ds > 0) & (ix >= 0) & (ix < nx) & (iy >= 0) & (iy < ny)
    return (iy * nx + ix)[keep], ds[keep]


def integrate(chi, eta, cells, ds):
    """Transfer along given segments, first segment nearest the observer: returns I, T (scalars)
    from the formal solution of dI/ds = eta - chi I with piecewise-constant coefficients."""
    I, tau = 0.0, 0.0
    for c, d in zip(cells, ds):
        x = chi[c] * d
        src = eta[c] * d if x == 0.0 else eta[c] / chi[c] * (1.0 - np.exp(-x)) if x > 1e-3 else \
            eta[c] * d * (1.0 - x / 2 + x * x / 6 - x**3 / 24)
        I += np.exp(-tau) * src
        tau += x
    return I, np.exp(-tau)


def long_characteristics_J(chi2d, eta2d, cells_xy, ntheta, I_bc=0.0):
    """Brute-force long characteristics (vectorised over rays): from each listed cell centre,
    ntheta equally spaced directions theta_m = 2 pi (m + 1/2)/ntheta, piecewise-constant transfer
    to the domain edge, J = mean over directions.  chi2d/eta2d: [ny][nx] float64."""
    ny, nx = chi2d.shape
    cells_xy = np.asarray(cells_xy)
    th = 2.0 * np.pi * (np.arange(ntheta) + 0.5) / ntheta
    P = len(cells_xy)
    px = np.repeat(cells_xy[:, 0] + 0.5, ntheta)
    py = np.repeat(cells_xy[:, 1] + 0.5, ntheta)
    wx = np.tile(np.cos(th), P)
    wy = np.tile(np.sin(th), P)
    ix = np.floor(px).astype(int)
    iy = np.floor(py).astype(int)
    sx = np.where(wx > 0, 1, -1)
    sy = np.where(wy > 0, 1, -1)
    with np.errstate(divide="ignore"):
        tmx = np.where(wx != 0, ((ix + (sx > 0)) - px) / wx, np.inf)
        tmy = np.where(wy != 0, ((iy + (sy > 0)) - py) / wy, np.inf)
        tdx = np.where(wx != 0, 1.0 / np.abs(wx), np.inf)
        tdy = np.where(wy != 0, 1.0 / np.abs(wy), np.inf)
    t = np.zeros_like(px)
    I = np.zeros_like(px)
    tau = np.zeros_like(px)
    alive = np.ones(px.shape, bool)
    while alive.any():
        tn = np.minimum(tmx, tmy)
        ds = np.where(alive, tn - t, 0.0)
        cx = np.clip(ix, 0, nx - 1)
        cy = np.clip(iy, 0, ny - 1)
        ch = chi2d[cy, cx]
        et = eta2d[cy, cx]
        x = ch * ds
        with np.errstate(divide="ignore", invalid="ignore"):
            src = np.where(x > 1e-8, et / np.where(ch > 0, ch, 1.0) * -np.expm1(-x), et * ds)
        I += np.where(alive, np.exp(-tau) * src, 0.0)
        tau += x
        stepx = tmx <= tmy
        stepy = tmy <= tmx
        ix = np.where(alive & stepx, ix + sx, ix)
        iy = np.where(alive & stepy, iy + sy, iy)
        tmx = np.where(stepx, tmx + tdx, tmx)
        tmy = np.where(stepy, tmy + tdy, tmy)
        t = tn
        alive &= (ix >= 0) & (ix < nx) & (iy >= 0) & (iy < ny)
    I += np.exp(-tau) * I_bc
    return I.reshape(P, ntheta).mean(axis=1)
