"""Seeded synthetic atmospheres for the five BASELINE.json configurations.

This module holds NO arithmetic of the radiance-cascades method: it only draws the
input fields (`chi`, `eta`), the boundary intensities and the wavelength weights.
It is the one module shared by the CPU oracle's tests and the CUDA path's tests
and bench (numpy only; it never imports the CUDA binding nor `oracle/`).

The recipes are the ones SURVEY.md §8(d) states (restated in DESIGN.md §4); they
are synthetic stand-ins with the shapes and structure of the paper's workloads
(PAPER.md:52 and 241 test scenes; PAPER.md:429-460 prominence snapshot), not the
paper's data, which is not available here.

Layout of every field: C-contiguous float32 `[ny][nx][nlambda]`, wavelength
fastest, `y = 0` the bottom row (include/rc.h conventions).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SQRT_PI = float(np.sqrt(np.pi))


@dataclass
class Atmosphere:
    name: str
    nx: int
    ny: int
    nlambda: int
    ncascades: int
    chi: np.ndarray  # float32 [ny][nx][nlambda]
    eta: np.ndarray  # float32 [ny][nx][nlambda]
    I_below: np.ndarray  # float32 [nlambda], seen by rays heading down (omega_y < 0)
    I_above: np.ndarray  # float32 [nlambda], seen by rays heading up
    weights: np.ndarray  # float32 [nlambda] wavelength weights (for Jbar)
    accumulate: bool = False  # config 4: the checked output is Jbar = sum_l w_l J_l
    c0_interval: float = 1.0
    meta: dict = field(default_factory=dict)
    # 2.5D: direction cosines to the invariant axis and quadrature weights (sum 1) of the
    # inclined rays that replace every flatland ray; None = flatland
    mu: np.ndarray | None = None
    w_mu: np.ndarray | None = None
    # velocity-dependent line mode: per-cell line parameters instead of chi, eta (then None)
    line: np.ndarray | None = None  # float32 [ny][nx][6]: chi_c, S_c, chi_line, S_line, v_x, v_y (Doppler widths)
    xl: np.ndarray | None = None    # float64 [nlambda] offsets from line centre in Doppler widths
    bilinear_fix: bool = False      # solve with the bilinear fix
    # sparsity: uint8 [ny][nx], non-zero = cell of interest; None = every cell.  J is computed on the
    # flagged cells only (0 elsewhere) and the other cells are treated as transparent with no emission
    active: np.ndarray | None = None


# (nx, ny, nlambda, ncascades) of BASELINE.json's configs
FULL_SHAPES = {
    0: (64, 64, 1, 5),
    1: (512, 512, 16, 7),
    2: (1024, 1024, 64, 8),
    3: (2048, 2048, 32, 9),
    4: (4096, 1024, 64, 9),
}


def _smooth_normal(rng: np.random.Generator, ny: int, nx: int, sigma: float) -> np.ndarray:
    """Standard-normal field, periodic Gaussian filter via FFT, kernel exp(-2 pi^2 sigma^2 |k|^2)."""
    f = rng.standard_normal((ny, nx))
    ky = np.fft.fftfreq(ny)[:, None]
    kx = np.fft.rfftfreq(nx)[None, :]
    kern = np.exp(-2.0 * np.pi**2 * sigma**2 * (kx * kx + ky * ky))
    return np.fft.irfft2(np.fft.rfft2(f) * kern, s=(ny, nx))


def _unit01(f: np.ndarray) -> np.ndarray:
    return (f - f.min()) / (f.max() - f.min())


def _unitvar(f: np.ndarray) -> np.ndarray:
    return (f - f.mean()) / f.std()


def _phi(x):
    """Gaussian line profile in Doppler units."""
    return np.exp(-np.square(x)) / SQRT_PI


def _finish(name, nx, ny, L, ncasc, chi, eta, I_below=None, I_above=None, weights=None,
            accumulate=False, meta=None) -> Atmosphere:
    chi = np.ascontiguousarray(chi, dtype=np.float32)
    eta = np.ascontiguousarray(eta, dtype=np.float32)
    assert chi.shape == (ny, nx, L) and eta.shape == (ny, nx, L)
    z = np.zeros(L, np.float32)
    return Atmosphere(
        name=name, nx=nx, ny=ny, nlambda=L, ncascades=ncasc, chi=chi, eta=eta,
        I_below=z.copy() if I_below is None else np.asarray(I_below, np.float32),
        I_above=z.copy() if I_above is None else np.asarray(I_above, np.float32),
        weights=np.ones(L, np.float32) if weights is None else np.asarray(weights, np.float32),
        accumulate=accumulate, meta=meta or {})


def _dims(idx, nx, ny, nlambda, ncascades):
    fx, fy, fl, fc = FULL_SHAPES[idx]
    nx = fx if nx is None else nx
    ny = fy if ny is None else ny
    nlambda = fl if nlambda is None else nlambda
    ncascades = fc if ncascades is None else ncascades
    scale = nx / fx  # feature lengths (in cells) follow the grid
    return nx, ny, nlambda, ncascades, scale


def config0(nx=None, ny=None, nlambda=None, ncascades=None, seed=1000) -> Atmosphere:
    """64x64x1, 5 cascades: smooth chi in [0.01,10], S in [1,1.5], zero boundary."""
    nx, ny, L, nc, sc = _dims(0, nx, ny, nlambda, ncascades)
    rng = np.random.default_rng(seed)
    g = _unit01(_smooth_normal(rng, ny, nx, 4.0 * sc))
    h = _unit01(_smooth_normal(rng, ny, nx, 4.0 * sc))
    chi = 10.0 ** (3.0 * g - 2.0)
    S = 1.0 + 0.5 * h
    # extra wavelengths (only when a test asks for them): a plain geometric dimming of chi
    fac = 10.0 ** (-np.arange(L) / 4.0)
    chi3 = chi[:, :, None] * fac[None, None, :]
    return _finish("cfg0", nx, ny, L, nc, chi3, chi3 * S[:, :, None])


def config1(nx=None, ny=None, nlambda=None, ncascades=None, seed=1001) -> Atmosphere:
    """512x512x16, 7 cascades: 40 optically thick discs in a thin background."""
    nx, ny, L, nc, sc = _dims(1, nx, ny, nlambda, ncascades)
    rng = np.random.default_rng(seed)
    chi = np.full((ny, nx), 1e-3)
    S = np.zeros((ny, nx))
    yy, xx = np.mgrid[0:ny, 0:nx]
    xc, yc = xx + 0.5, yy + 0.5
    for _ in range(40):
        cx, cy = rng.uniform(0, nx), rng.uniform(0, ny)
        r = rng.uniform(5.0, 30.0) * sc
        chi_d = rng.uniform(1.0, 100.0)
        S_d = rng.uniform(0.5, 2.0)
        m = (xc - cx) ** 2 + (yc - cy) ** 2 <= r * r
        chi[m] = chi_d
        S[m] = S_d
    fac = 10.0 ** (-np.arange(L) / 5.0)
    chi3 = chi[:, :, None] * fac[None, None, :]
    return _finish("cfg1", nx, ny, L, nc, chi3, chi3 * S[:, :, None])


def _line_fields(rng, ny, nx, sc):
    g1 = _unitvar(_smooth_normal(rng, ny, nx, 8.0 * sc))
    g2 = _unitvar(_smooth_normal(rng, ny, nx, 8.0 * sc))
    u = _unit01(_smooth_normal(rng, ny, nx, 16.0 * sc))
    h = _unit01(_smooth_normal(rng, ny, nx, 8.0 * sc))
    return g1, g2, 3.0 * (2.0 * u - 1.0), 10.0 ** (2.0 * h - 1.0)


def _xgrid(L):
    return np.array([0.0]) if L == 1 else -5.0 + 10.0 * np.arange(L) / (L - 1)


def config2(nx=None, ny=None, nlambda=None, ncascades=None, seed=1002) -> Atmosphere:
    """1024x1024x64, 8 cascades: Doppler-shifted Gaussian line over a lognormal continuum."""
    nx, ny, L, nc, sc = _dims(2, nx, ny, nlambda, ncascades)
    rng = np.random.default_rng(seed)
    g1, g2, v, S = _line_fields(rng, ny, nx, sc)
    chi_c = (1e-3 * np.exp(g1)).astype(np.float32)
    chi_line = np.exp(g2).astype(np.float32)
    x = _xgrid(L).astype(np.float32)
    chi = np.empty((ny, nx, L), np.float32)
    for l in range(L):  # plane by plane: keeps the peak memory at one copy
        chi[:, :, l] = chi_c + chi_line * _phi(x[l] - v)
    eta = chi * S.astype(np.float32)[:, :, None]
    return _finish("cfg2", nx, ny, L, nc, chi, eta)


def line_config2(nx=None, ny=None, nlambda=None, ncascades=None, seed=1002) -> Atmosphere:
    """Config 2's recipe as a moving-line atmosphere: the same chi_c, chi_line, speed and
    S fields, but the velocity is a vector (speed x a smooth direction field) and the line is Doppler shifted
    per ray by the projected velocity; the line has its own source function field.  chi, eta are None."""
    nx, ny, L, nc, sc = _dims(2, nx, ny, nlambda, ncascades)
    rng = np.random.default_rng(seed)
    g1, g2, v, S = _line_fields(rng, ny, nx, sc)
    psi = 2.0 * np.pi * _unit01(_smooth_normal(rng, ny, nx, 16.0 * sc))
    h2 = _unit01(_smooth_normal(rng, ny, nx, 8.0 * sc))
    line = np.empty((ny, nx, 6), np.float32)
    line[..., 0] = 1e-3 * np.exp(g1)
    line[..., 1] = S
    line[..., 2] = np.exp(g2)
    line[..., 3] = 10.0 ** (2.0 * h2 - 1.0)
    line[..., 4] = v * np.cos(psi)
    line[..., 5] = v * np.sin(psi)
    z = np.zeros(L, np.float32)
    return Atmosphere(name="line2", nx=nx, ny=ny, nlambda=L, ncascades=nc, chi=None, eta=None, I_below=z.copy(),
                      I_above=z.copy(), weights=np.ones(L, np.float32), line=line, xl=_xgrid(L).astype(np.float64))


def config3(nx=None, ny=None, nlambda=None, ncascades=None, seed=1003) -> Atmosphere:
    """2048x2048x32, 9 cascades: dense sheet + strands in a 1e-6 corona, lit from below."""
    nx, ny, L, nc, sc = _dims(3, nx, ny, nlambda, ncascades)
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:ny, 0:nx]
    xc, yc = xx + 0.5, yy + 0.5
    chi_line = np.zeros((ny, nx))
    S = np.zeros((ny, nx))
    for _ in range(80):  # strands first; the sheet is painted over them
        x0, y0 = rng.uniform(0, nx), rng.uniform(0, ny)
        length = rng.uniform(150.0, 700.0) * sc
        ang = np.pi / 2 + np.deg2rad(rng.uniform(-30.0, 30.0))
        width = max(rng.uniform(2.0, 10.0) * sc, 1.0)
        amp = 10.0 ** rng.uniform(1.0, 4.0)
        S_s = rng.uniform(0.1, 0.5)
        ux, uy = np.cos(ang), np.sin(ang)
        along = (xc - x0) * ux + (yc - y0) * uy
        perp = np.abs(-(xc - x0) * uy + (yc - y0) * ux)
        m = (along >= 0) & (along <= length) & (perp <= 0.5 * width)
        chi_line[m] = amp
        S[m] = S_s
    g = _unit01(_smooth_normal(rng, ny, nx, 6.0 * sc))
    ycen = 0.55 * ny + 40.0 * sc * np.sin(2.0 * np.pi * xc / nx * 3.0)
    m = np.abs(yc - ycen) <= 24.0 * sc
    chi_line[m] = (1e4 * (0.3 + 0.7 * g))[m]
    S[m] = 0.2
    x = _xgrid(L).astype(np.float32)
    chi = np.empty((ny, nx, L), np.float32)
    cl = chi_line.astype(np.float32)
    for l in range(L):
        chi[:, :, l] = np.float32(1e-6) + cl * np.float32(_phi(x[l]))
    eta = chi * S.astype(np.float32)[:, :, None]
    return _finish("cfg3", nx, ny, L, nc, chi, eta, I_below=np.ones(L), I_above=np.zeros(L))


def config4(nx=None, ny=None, nlambda=None, ncascades=None, seed=1004) -> Atmosphere:
    """4096x1024x64, 9 cascades: >90% exactly-empty cells, truncated Gaussian blobs, Jbar output."""
    nx, ny, L, nc, sc = _dims(4, nx, ny, nlambda, ncascades)
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:ny, 0:nx]
    xc, yc = (xx + 0.5).astype(np.float32), (yy + 0.5).astype(np.float32)
    blobs = [(rng.uniform(0, nx), rng.uniform(0, ny), rng.uniform(4.0, 18.0) * sc,
              10.0 ** rng.uniform(-1.0, 2.0)) for _ in range(130)]
    nblob = len(blobs)
    while True:
        chi_line = np.zeros((ny, nx), np.float32)
        for (bx, by, sb, amp) in blobs[:nblob]:
            r = 2.5 * sb
            xa, xb = max(int(bx - r) - 1, 0), min(int(bx + r) + 2, nx)
            ya, yb = max(int(by - r) - 1, 0), min(int(by + r) + 2, ny)
            if xa >= xb or ya >= yb:
                continue
            d2 = (xc[ya:yb, xa:xb] - bx) ** 2 + (yc[ya:yb, xa:xb] - by) ** 2
            add = amp * np.exp(-d2 / (2.0 * sb * sb))
            add[d2 > r * r] = 0.0
            chi_line[ya:yb, xa:xb] += add.astype(np.float32)
        empty = float(np.mean(chi_line == 0.0))
        if empty > 0.90 or nblob <= 1:
            break
        nblob -= 5
    _, _, v, S = _line_fields(rng, ny, nx, sc)
    x = _xgrid(L).astype(np.float32)
    chi = np.empty((ny, nx, L), np.float32)
    for l in range(L):
        chi[:, :, l] = chi_line * _phi(x[l] - v).astype(np.float32)
    eta = chi * S.astype(np.float32)[:, :, None]
    w = _phi(_xgrid(L))
    w = w / w.sum()
    return _finish("cfg4", nx, ny, L, nc, chi, eta, weights=w, accumulate=True,
                   meta={"empty_fraction": empty, "nblobs": nblob})


def emitter_config(nx=128, ny=128, nlambda=4, ncascades=6, seed=2001, chi_emitter=0.0) -> Atmosphere:
    """Emission with next to no opacity (reading G11 of DESIGN.md: eq. 16 in the limit chi -> 0 adds eta ds): config 1's
    opaque discs in exact vacuum (chi = eta = 0), plus smooth patches of pure emitters with eta ~ 1e-3 and chi = `chi_emitter`
    (0, or e.g. 1e-12) - the one family of valid inputs that is not of the form eta = chi S with a moderate S.  Wavelength l
    scales the discs' opacity by 10^(-l) (from opaque to translucent) and leaves the emitters alone."""
    rng = np.random.default_rng(seed)
    sc = nx / 512.0
    chi = np.zeros((ny, nx))
    S = np.zeros((ny, nx))
    yy, xx = np.mgrid[0:ny, 0:nx]
    xc, yc = xx + 0.5, yy + 0.5
    for _ in range(12):
        cx, cy = rng.uniform(0, nx), rng.uniform(0, ny)
        r = max(rng.uniform(5.0, 30.0) * sc, 1.5)
        m = (xc - cx) ** 2 + (yc - cy) ** 2 <= r * r
        chi[m] = rng.uniform(1.0, 100.0)
        S[m] = rng.uniform(0.5, 2.0)
    g = _unit01(_smooth_normal(rng, ny, nx, max(16.0 * sc, 2.0)))
    h = _unit01(_smooth_normal(rng, ny, nx, max(8.0 * sc, 2.0)))
    emit = (g > 0.6) & (chi == 0.0)
    fac = 10.0 ** (-np.arange(nlambda, dtype=np.float64))
    chi3 = chi[:, :, None] * fac[None, None, :]
    eta3 = chi3 * S[:, :, None]
    chi3[emit] = chi_emitter
    eta3[emit] = (1e-3 * (0.5 + h))[emit][:, None]
    return _finish("emit", nx, ny, nlambda, ncascades, chi3, eta3, meta={"emitter_fraction": float(emit.mean())})


def wild_config(nx=96, ny=96, nlambda=8, ncascades=5, seed=3001) -> Atmosphere:
    """Neighbouring wavelengths whose opacities differ by many orders of magnitude in the same cell (nothing a spectral
    line does, but valid input): smooth fields chi0, S0 times a per-wavelength factor that jumps between 1e-9 and 1e2,
    plus a faint wavelength-independent emissivity everywhere - so that in one cell a wavelength emits from the optically
    thin limit (eta ds) right beside one that is opaque.  For the march's per-channel form of the cell update."""
    rng = np.random.default_rng(seed)
    sc = max(nx / 64.0, 1.0)
    g = _unit01(_smooth_normal(rng, ny, nx, 4.0 * sc))
    h = _unit01(_smooth_normal(rng, ny, nx, 3.0 * sc))
    e = _unit01(_smooth_normal(rng, ny, nx, 5.0 * sc))
    chi0 = 10.0 ** (2.0 * g - 1.0)                       # 0.1 .. 10 per cell
    S0 = 0.5 + h
    fac = np.array([1.0, 1e-9, 1e2, 1e-5, 3e-2, 1e-12, 1.0, 1e-3])[np.arange(nlambda) % 8]
    chi3 = chi0[:, :, None] * fac[None, None, :]
    eta3 = chi3 * S0[:, :, None] + (1e-4 * (0.2 + e))[:, :, None]
    return _finish("wild", nx, ny, nlambda, ncascades, chi3, eta3, meta={"factors": fac.tolist()})


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}


def gauss_radau(n: int):
    """n-point Gauss-Radau rule on mu in [0, 1] with the fixed node at mu = 0 (the in-plane ray), weights
    summing to 1 - the inclination quadrature of PAPER.md:281 ("a Gauss-Radau quadrature with eight rays for
    inclination", integrating one hemisphere).  The paper does not say which end is fixed; mu = 1 would be a
    ray along the invariant axis with an infinite path (reading G20).  Textbook rule: on [-1, 1]
    the free nodes are the roots of (P_{n-1} + P_n)/(1 + x), w_1 = 2/n^2, w_i = (1 - x_i)/(n P_{n-1}(x_i))^2.
    Inputs only: the method's arithmetic never sees how mu, w were made."""
    from numpy.polynomial import legendre as Lg
    if n == 1:
        return np.zeros(1), np.ones(1)
    c = np.zeros(n + 1)
    c[n - 1] = c[n] = 1.0
    x = np.sort(np.real(Lg.legroots(c)))
    x[0] = -1.0
    pnm1 = Lg.legval(x, np.eye(n)[n - 1])
    w = (1.0 - x) / (n * pnm1) ** 2
    w[0] = 2.0 / n ** 2
    return (x + 1.0) / 2.0, w / 2.0


def with_inclinations(atm: Atmosphere, n: int) -> Atmosphere:
    """The same atmosphere solved in 2.5D with an n-point Gauss-Radau inclination quadrature."""
    import dataclasses
    mu, w = gauss_radau(n)
    return dataclasses.replace(atm, name=f"{atm.name}_incl{n}", mu=mu, w_mu=w)


def with_active_cells(atm: Atmosphere, mode="occupied", fraction=None, dilate=0) -> Atmosphere:
    """The same atmosphere with a cells-of-interest flag ("in the current implementation this is simply a
    temperature flag"; here, with no temperature, the stand-in is where the opacity is).  mode "occupied": cells whose
    opacity (any wavelength; line mode: chi_c + chi_line) exceeds the smallest positive value by a factor 10, dilated by
    `dilate` cells; "fraction": the `fraction` of cells with the largest wavelength-summed opacity (e.g. 0.25, the paper's
    production run)."""
    import dataclasses
    op = (atm.line[..., 0] + atm.line[..., 2]).astype(np.float64) if atm.line is not None else atm.chi.astype(np.float64).sum(axis=2)
    if mode == "fraction":
        k = int(round(fraction * op.size))
        order = np.argsort(-op.ravel(), kind="stable")       # ties (e.g. a uniform corona) go by cell index: exactly k cells
        act = np.zeros(op.size, bool)
        act[order[:k]] = True
        act = act.reshape(op.shape)
    else:
        pos = op[op > 0]
        act = op > (10.0 * pos.min() if pos.size else 0.0)
    for _ in range(dilate):
        a = act.copy()
        a[1:, :] |= act[:-1, :]; a[:-1, :] |= act[1:, :]; a[:, 1:] |= act[:, :-1]; a[:, :-1] |= act[:, 1:]
        act = a
    return dataclasses.replace(atm, name=f"{atm.name}_active", active=act.astype(np.uint8),
                               meta=dict(atm.meta, active_fraction=float(act.mean())))


def make_config(idx: int, **kw) -> Atmosphere:
    """Config `idx` of BASELINE.json; keyword overrides (nx, ny, nlambda, ncascades, seed)
    give the reduced-size variants the parity tests use (feature sizes scale with nx)."""
    return CONFIGS[idx](**kw)


def random_field(nx: int, ny: int, nlambda: int, seed: int, chi_lo=1e-3, chi_hi=10.0,
                 zero_fraction=0.0):
    """Unstructured log-uniform chi and uniform S in [0.1, 2]; for unit tests."""
    rng = np.random.default_rng(seed)
    chi = np.exp(rng.uniform(np.log(chi_lo), np.log(chi_hi), (ny, nx, nlambda)))
    if zero_fraction > 0:
        chi[rng.uniform(size=(ny, nx)) < zero_fraction] = 0.0
    S = rng.uniform(0.1, 2.0, (ny, nx, nlambda))
    return chi.astype(np.float32), (chi * S).astype(np.float32)
