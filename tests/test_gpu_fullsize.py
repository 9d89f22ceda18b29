"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

  config 1, config 2   EVERY cell against the oracle (config 2: 1.7e11 segment-wavelengths, a few minutes of the GPU
                       box's host cores, 16 wavelengths at a time; marked `slow`, still part of `-m gpu`)
  config 3, config 4   the oracle cannot finish them in test time (6.6e11, 1.2e12 segment-wavelengths), but J in a cell
                       depends only on the few probes per cascade its bilinear lookups reach, so the oracle computes
                       windows of 4 x 4 cells (oracle.solve(window=...), bit-identical to its full solve:
                       tests/test_oracle_pins.py::test_window_solve_is_the_full_solve_restricted): >= 16 windows placed
                       inside the structure, in its shadow, at its edges, at the four box edges and corners and across
                       every seam of the L2 bands; the mask scale comes from the oracle
  + at those sizes, on EVERY cell and without oracle time: J = S, the x-flip symmetry, and bit-identity of the
    banded against the unbanded march and of the hit-list and distance-field marches against the lock-step march.
  + the widened modes at the sizes profiles/bench_*.md quotes times for: the bilinear fix on config 3 (its unbanded launches
    gather from HBM), 8 inclinations and the moving line x 8 inclinations x 25 % of the cells flagged on the config-2 grid.
"""
import dataclasses

import numpy as np
import pytest

from paper_2408_14425_b200 import atmospheres as A

pytestmark = pytest.mark.gpu
TOL = 2e-4


def gpu(atm, **kw):
    from paper_2408_14425_b200 import binding
    J, rc = binding.solve_atmosphere(atm, **kw)
    st = rc.get_stats()
    out = J.cpu().numpy()
    rc.close()
    return out, st


def plane_errors(Jg, Jo, scale=None):
    """max relative error per wavelength plane over cells with Jo > 1e-6 scale (default: the oracle's own maximum)"""
    worst = 0.0
    Jg = np.asarray(Jg, np.float64)
    if Jo.ndim == 2:
        Jg, Jo = Jg[..., None], Jo[..., None]
    for l in range(Jo.shape[-1]):
        o, g = Jo[..., l], Jg[..., l]
        m = o > 1e-6 * (o.max() if scale is None else scale[l])
        if m.any():
            worst = max(worst, float(np.max(np.abs(g[m] - o[m]) / o[m])))
    return worst


def feature_windows(atm, size=4, nrand=4, seed=0):
    """Windows of size x size cells: the four corners and edge mid-points of the box, the seams of the L2 bands the plan
    uses, and - from the wavelength-summed opacity - the most opaque cell (inside the sheet / a blob), the steepest opacity
    gradients (edges of blobs and strands), a spot in the shadow above the structure, the emptiest region, plus random ones."""
    from paper_2408_14425_b200 import binding
    nx, ny = atm.nx, atm.ny
    c = size // 2
    pts = [(c, c), (nx - c, c), (c, ny - c), (nx - c, ny - c), (nx // 2, c), (nx // 2, ny - c), (c, ny // 2), (nx - c, ny // 2)]
    plan = binding.plan_query(atm.ncascades, nx, ny, atm.nlambda)
    if plan.nbands > 1:
        n_axis = nx if plan.band_axis else ny
        ext = -(-n_axis // plan.nbands)
        for k in range(1, plan.nbands):          # straddling every seam, at two places along it
            for frac in (0.3, 0.8):
                pts.append((k * ext, int(frac * ny)) if plan.band_axis else (int(frac * nx), k * ext))
    op = atm.chi.astype(np.float64).sum(axis=2)
    y, x = np.unravel_index(int(np.argmax(op)), op.shape)
    pts.append((x, y))
    gx, gy = np.abs(np.diff(op, axis=1)), np.abs(np.diff(op, axis=0))
    for g in (gx, gy):
        yy, xx = np.unravel_index(int(np.argmax(g)), g.shape)
        pts.append((xx + 1, yy + 1))
    col = int(np.argmax(op.max(axis=0)))                       # the column of the most opaque cell: above it lies the shadow
    top = int(np.max(np.nonzero(op[:, col] > 0.5 * op[:, col].max())[0]))
    pts.append((col, min(top + 40, ny - c)))
    yy, xx = np.unravel_index(int(np.argmin(op)), op.shape)
    pts.append((xx, yy))
    rng = np.random.default_rng(seed)
    pts += [(int(rng.integers(c, nx - c)), int(rng.integers(c, ny - c))) for _ in range(nrand)]
    out = []
    for (px, py) in pts:
        x0 = int(min(max(px - c, 0), nx - size))
        y0 = int(min(max(py - c, 0), ny - size))
        w = (x0, x0 + size, y0, y0 + size)
        if w not in out:
            out.append(w)
    return out


def run_windows(atm, oracle, size=4, nrand=4, min_windows=16, max_windows=None, **kw):
    Jg, st = gpu(atm, **kw)
    wins = feature_windows(atm, size, nrand, seed=atm.nx)
    if max_windows is not None and len(wins) > max_windows:      # an even pick over box edges, seams and features
        wins = [wins[i] for i in np.unique(np.linspace(0, len(wins) - 1, max_windows).round().astype(int))]
    assert len(wins) >= min_windows
    ref = []
    for w in wins:
        o = oracle.solve_atmosphere(atm, window=w)
        ref.append(o["Jbar"][..., None] if atm.accumulate else o["J"])
    scale = np.max([r.reshape(-1, r.shape[-1]).max(axis=0) for r in ref], axis=0)   # the oracle's own brightest sampled cell
    worst = 0.0
    for (x0, x1, y0, y1), Jo in zip(wins, ref):
        g = Jg[y0:y1, x0:x1]
        worst = max(worst, plane_errors(g[..., None] if atm.accumulate else g, Jo, scale))
    print(f"{atm.name} full size: max rel err over {len(wins)} windows of {size}x{size} cells = {worst:.3e}")
    assert worst <= TOL, worst
    return Jg, st


def test_config1_full_grid_every_cell(oracle):
    atm = A.make_config(1)
    Jg, _ = gpu(atm)
    assert plane_errors(Jg, oracle.solve_atmosphere(atm)["J"]) <= TOL


@pytest.mark.slow
def test_config2_full_grid_every_cell(oracle):
    """The configuration the metric is quoted on, every one of its 1024 x 1024 x 64 values against the oracle (the march of
    cascades 4-5 runs the 128-register ring-of-3 variant on rays of up to 1365 cells here, and nowhere smaller)."""
    from paper_2408_14425_b200 import sharding
    atm = A.make_config(2)
    Jg, _ = gpu(atm)
    worst = 0.0
    for r in range(4):                       # 16 wavelengths at a time: 2 x 0.5 GB of oracle cascade storage
        l0, l1 = sharding.wavelength_block(atm.nlambda, r, 4)
        Jo = oracle.solve_atmosphere(sharding.shard_atmosphere(atm, r, 4))["J"]
        worst = max(worst, plane_errors(Jg[..., l0:l1], Jo))
    print(f"cfg2 full grid, every cell and wavelength: max rel err {worst:.3e}")
    assert worst <= TOL, worst


def test_config3_windows_and_invariants(oracle):
    atm = A.make_config(3)
    Jg, st = run_windows(atm, oracle)
    # the banded launches at production extents against the unbanded march of the same inputs: every cell, every bit
    from paper_2408_14425_b200 import binding
    assert binding.plan_query(atm.ncascades, atm.nx, atm.ny, atm.nlambda).nbands > 1
    Ju, _ = gpu(atm, tuning=dict(bands=1))
    assert np.array_equal(Jg, Ju)
    # x-flip: the direction set and the lattices are mirror symmetric, so J of the mirrored atmosphere is the mirrored J
    flip = dataclasses.replace(atm, chi=np.ascontiguousarray(atm.chi[:, ::-1]), eta=np.ascontiguousarray(atm.eta[:, ::-1]))
    Jf, _ = gpu(flip)
    m = Jg > 1e-6 * Jg.max()
    assert np.max(np.abs(Jf[:, ::-1][m] / Jg[m] - 1)) < 2e-5
    # J = S: eta = chi S0 and boundary S0 on every side give J = S0 in every cell (north_star), here with config 3's opacities
    S0 = np.float32(0.75)
    const = dataclasses.replace(atm, eta=atm.chi * S0, I_below=np.full(atm.nlambda, S0), I_above=np.full(atm.nlambda, S0))
    Jc, _ = gpu(const)
    assert np.max(np.abs(Jc / S0 - 1)) < 2e-5


def test_config4_windows_and_invariants(oracle):
    atm = A.make_config(4)
    Jg, st = run_windows(atm, oracle, analyse=True)               # as bench.py runs it: the march over hit lists, Jbar
    assert st.sparse_march == 1 and st.sparse_lists >= 1 and st.empty_cells > 0.9 * atm.nx * atm.ny
    Jd, st = gpu(atm)                                             # the lock-step march (banded at this size): every cell, every bit
    assert st.sparse_march == 0 and np.array_equal(Jg, Jd)
    # what a caller gets who lends no second buffer (rc_set_sparse_workspace): the distance-field fan march, at this size
    Jfan, st = gpu(atm, analyse=True, tuning=dict(lists=0))
    assert st.sparse_march == 1 and st.sparse_lists == 0 and np.array_equal(Jg, Jfan)
    flip = dataclasses.replace(atm, chi=np.ascontiguousarray(atm.chi[:, ::-1]), eta=np.ascontiguousarray(atm.eta[:, ::-1]))
    Jf, _ = gpu(flip, analyse=True)
    m = Jg > 1e-6 * Jg.max()
    assert np.max(np.abs(Jf[:, ::-1][m] / Jg[m] - 1)) < 2e-5
    S0 = np.float32(1.5)
    w = np.full(atm.nlambda, 1.0 / atm.nlambda, np.float32)
    const = dataclasses.replace(atm, eta=atm.chi * S0, I_below=np.full(atm.nlambda, S0), I_above=np.full(atm.nlambda, S0), weights=w)
    Jc, _ = gpu(const, analyse=True)
    assert np.max(np.abs(Jc / S0 - 1)) < 2e-5


def test_config3_quarter_of_the_cells_active(oracle):
    """The paper's regime (~25 % of the cells active): config 3 with its densest quarter flagged."""
    atm = A.with_active_cells(A.make_config(3), mode="fraction", fraction=0.25)
    Jg, st = run_windows(atm, oracle, nrand=2, min_windows=12)
    assert st.active_cells == int((atm.active != 0).sum())
    assert np.all(Jg[atm.active == 0] == 0.0)


# ------------------------------------------------------------------ the widened modes at size (512 x 512 x 16, 7 cascades)
def test_config1_size_bilinear_fix(oracle):
    run_windows(dataclasses.replace(A.make_config(1), name="cfg1_fix", bilinear_fix=True), oracle, size=3, nrand=2, min_windows=8)


def test_config1_size_inclinations(oracle):
    run_windows(A.with_inclinations(A.make_config(1), 8), oracle, size=3, nrand=2, min_windows=8)


def test_config1_size_moving_line_with_inclinations(oracle):
    atm = A.with_inclinations(A.line_config2(nx=512, ny=512, nlambda=16, ncascades=7), 4)
    from paper_2408_14425_b200 import binding
    Jg, _ = gpu(atm)
    rng = np.random.default_rng(3)
    wins = [(0, 3, 0, 3), (509, 512, 255, 258)] + [(int(x), int(x) + 3, int(y), int(y) + 3) for x, y in rng.integers(0, 509, (4, 2))]
    worst = 0.0
    for (x0, x1, y0, y1) in wins:
        Jo = oracle.solve_atmosphere(atm, window=(x0, x1, y0, y1))["J"]
        worst = max(worst, plane_errors(Jg[y0:y1, x0:x1], Jo, scale=Jg.reshape(-1, atm.nlambda).max(axis=0)))
    assert worst <= TOL, worst


# ------------------------------------------------------------------ the widened modes at the sizes their timings are quoted for
def _windows_at(points, nx, ny, size):
    out = []
    for (px, py) in points:
        x0, y0 = int(min(max(px - size // 2, 0), nx - size)), int(min(max(py - size // 2, 0), ny - size))
        if (x0, x0 + size, y0, y0 + size) not in out:
            out.append((x0, x0 + size, y0, y0 + size))
    return out


@pytest.mark.slow
def test_config3_size_bilinear_fix(oracle):
    """PAPER.md:243-249 on config 3's 2048 x 2048 grid: with the fix no cascade is banded, so cascades 5-6 gather from HBM -
    launches that no smaller grid reaches."""
    atm = dataclasses.replace(A.make_config(3), name="cfg3_fix", bilinear_fix=True)
    run_windows(atm, oracle, size=3, nrand=0, min_windows=12, max_windows=12)


@pytest.mark.slow
def test_config2_size_eight_inclinations(oracle):
    """PAPER.md:281, 571 (every result of the paper uses 8 inclinations) on config 2's 1024 x 1024 grid: 8 channels per lane,
    one wavelength per batch (the shape profiles/bench_r2.md quotes 510 ms for)."""
    atm = A.with_inclinations(A.make_config(2), 8)
    run_windows(atm, oracle, size=2, nrand=0, min_windows=8, max_windows=8)


@pytest.mark.slow
def test_config2_size_moving_line_eight_inclinations_quarter_active(oracle):
    """The paper's production regime: moving line x 8 inclinations x the densest 25 % of the cells
    flagged, on config 2's 1024 x 1024 x 64 grid, marched over hit lists.  Windows sit on flagged
    cells: deep inside, on the rim of the flagged set and next to the box edges."""
    atm = A.with_active_cells(A.with_inclinations(A.line_config2(), 8), mode="fraction", fraction=0.25)
    Jg, st = gpu(atm, analyse=True)
    act = atm.active != 0
    assert st.active_cells == int(act.sum()) and np.all(Jg[~act] == 0.0)
    op = (atm.line[..., 0] + atm.line[..., 2]).astype(np.float64)
    ys, xs = np.nonzero(act)
    rim = act & ~(np.roll(act, 1, 0) & np.roll(act, -1, 0) & np.roll(act, 1, 1) & np.roll(act, -1, 1))
    ry, rx = np.nonzero(rim)
    rng = np.random.default_rng(8)
    pts = [np.unravel_index(int(np.argmax(op)), op.shape)[::-1]]
    pts += [(int(rx[i]), int(ry[i])) for i in rng.integers(0, rx.size, 3)]
    pts += [(int(xs[i]), int(ys[i])) for i in (int(np.argmin(xs)), int(np.argmax(xs)), int(np.argmin(ys)), int(np.argmax(ys)))]
    pts += [(int(xs[i]), int(ys[i])) for i in rng.integers(0, xs.size, 2)]
    wins = _windows_at(pts, atm.nx, atm.ny, 2)
    assert len(wins) >= 8
    ref = [oracle.solve_atmosphere(atm, window=w)["J"] for w in wins]
    scale = np.nanmax([np.nanmax(r.reshape(-1, r.shape[-1]), axis=0) for r in ref], axis=0)
    worst, checked = 0.0, 0
    for (x0, x1, y0, y1), Jo in zip(wins, ref):
        a = act[y0:y1, x0:x1]
        assert np.all(np.isfinite(Jo[a]))
        worst = max(worst, plane_errors(np.where(a[..., None], Jg[y0:y1, x0:x1], 0.0), np.where(a[..., None], Jo, 0.0), scale))
        checked += int(a.sum())
    print(f"{atm.name}: max rel err over {checked} flagged cells in {len(wins)} windows = {worst:.3e}")
    assert checked >= 16 and worst <= TOL, worst
