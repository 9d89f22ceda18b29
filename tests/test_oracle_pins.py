"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

Each test names the pin of SURVEY.md §8(c) / DESIGN.md §5 it implements and the passage of
/root/reference/PAPER.md it rests on.  None of the expected values comes from the oracle itself
or from the CUDA path: they are closed forms, invariants or the independent numpy references in
tests/refs.py.
"""
import numpy as np
import pytest

from paper_2408_14425_b200 import atmospheres as A
from tests import refs

R2 = np.sqrt(2.0)


def t_of(i, c0=1.0):
    return c0 * (4.0**i - 1.0) / 3.0


# ----------------------------------------------------------------------------- P1: DDA + eq. 16
def test_P1_segments_match_sorting_reference(oracle):
    """DDA vs crossing-sort reference on random rays; sum(ds) = in-box length."""
    rng = np.random.default_rng(1)
    nx, ny = 37, 23
    for _ in range(300):
        px, py = rng.uniform(0, nx), rng.uniform(0, ny)
        if rng.uniform() < 0.5:  # probes of cascades i>=1 sit on integer vertices
            px, py = float(rng.integers(1, nx)), float(rng.integers(1, ny))
        th = rng.uniform(0, 2 * np.pi)
        ta = rng.uniform(0, 20)
        tb = ta + rng.uniform(0.1, 40) if rng.uniform() < 0.7 else np.inf
        c, d = oracle.ray_segments(nx, ny, px, py, theta=th, ta=ta, tb=tb)
        cr, dr = refs.segments_by_sorting(nx, ny, px, py, th, ta, tb if np.isfinite(tb) else 1e9)
        x0, y0 = px + ta * np.cos(th), py + ta * np.sin(th)
        if not (0 <= x0 <= nx and 0 <= y0 <= ny):
            assert len(c) == 0
            continue
        keep, keepr = d > 1e-9, dr > 1e-9  # slivers at near-ties may differ; their length may not
        assert np.array_equal(c[keep], cr[keepr])
        assert np.allclose(d[keep], dr[keepr], rtol=0, atol=1e-11)
        assert abs(d.sum() - dr.sum()) < 1e-11


def test_P1_uniform_medium_closed_form(oracle):
    """Uniform chi, S: T = exp(-chi l), I = S (1 - exp(-chi l)) for any split into cells (eq. 16)."""
    rng = np.random.default_rng(2)
    nx, ny, L = 32, 20, 3
    chi0 = np.array([0.03, 0.7, 5.0])
    S0 = np.array([2.0, 0.5, 1.25])
    chi = np.broadcast_to(chi0, (ny, nx, L)).astype(np.float32)
    eta = (chi.astype(np.float64) * S0).astype(np.float32)
    chi64, eta64 = chi[0, 0].astype(np.float64), eta[0, 0].astype(np.float64)
    for _ in range(100):
        px, py = float(rng.integers(1, nx)), float(rng.integers(1, ny))
        th = rng.uniform(0, 2 * np.pi)
        ta, tb = 0.3, rng.uniform(1, 60)
        _, d = oracle.ray_segments(nx, ny, px, py, theta=th, ta=ta, tb=tb)
        ell = refs.segments_by_sorting(nx, ny, px, py, th, ta, tb)[1].sum()
        assert abs(d.sum() - ell) < 1e-11
        for order in (0, 1):
            I, T = oracle.interval(chi, eta, px, py, theta=th, ta=ta, tb=tb, order=order)
            assert np.allclose(T, np.exp(-chi64 * ell), rtol=1e-12, atol=0)
            assert np.allclose(I, eta64 / chi64 * -np.expm1(-chi64 * ell), rtol=1e-12, atol=1e-300)


def test_P1_random_field_vs_independent_integration(oracle):
    """Random chi/eta: oracle interval = independent segment list + independent integration."""
    rng = np.random.default_rng(3)
    nx, ny = 24, 24
    chi, eta = A.random_field(nx, ny, 2, seed=5, zero_fraction=0.2)
    for _ in range(60):
        px, py = float(rng.integers(1, nx)), float(rng.integers(1, ny))
        th = rng.uniform(0, 2 * np.pi)
        ta, tb = rng.uniform(0, 5), rng.uniform(6, 50)
        I, T = oracle.interval(chi, eta, px, py, theta=th, ta=ta, tb=tb)
        c, d = refs.segments_by_sorting(nx, ny, px, py, th, ta, tb)
        for l in range(2):
            Ir, Tr = refs.integrate(chi.reshape(-1, 2)[:, l].astype(float),
                                    eta.reshape(-1, 2)[:, l].astype(float), c, d)
            assert np.isclose(I[l], Ir, rtol=1e-9, atol=1e-14)
            assert np.isclose(T[l], Tr, rtol=1e-9, atol=1e-300)


# ----------------------------------------------------------------------------- P2 / G1 / G13
def test_P2_split_and_merge_equals_whole(oracle):
    """March [a,c] = M(march [a,b], march [b,c]): fixes the garbled eq. 11 to
    'near attenuates far' (reading G1); the swapped reading fails this."""
    rng = np.random.default_rng(4)
    nx = ny = 40
    chi, eta = A.random_field(nx, ny, 1, seed=6, chi_lo=1e-2, chi_hi=2.0)
    worst_swapped = 0.0
    for _ in range(100):
        px, py = float(rng.integers(4, nx - 4)), float(rng.integers(4, ny - 4))
        th = rng.uniform(0, 2 * np.pi)
        a, c = rng.uniform(0, 3), rng.uniform(8, 30)
        b = rng.uniform(a, c)
        Iw, Tw = oracle.interval(chi, eta, px, py, theta=th, ta=a, tb=c)
        In, Tn = oracle.interval(chi, eta, px, py, theta=th, ta=a, tb=b)
        If, Tf = oracle.interval(chi, eta, px, py, theta=th, ta=b, tb=c)
        Im, taum = oracle.merge(In[0], -np.log(Tn[0]), If[0], -np.log(Tf[0]))
        assert np.isclose(Im, Iw[0], rtol=1e-12)
        assert np.isclose(np.exp(-taum), Tw[0], rtol=1e-12)
        assert np.isclose(Im, In[0] + Tn[0] * If[0], rtol=1e-14)  # eq. 11, physical reading
        worst_swapped = max(worst_swapped, abs((If[0] + Tf[0] * In[0]) - Iw[0]) / Iw[0])
    assert worst_swapped > 1e-2  # the printed subscripts, read literally, are not a merge


def test_G13_back_to_front_equals_front_to_back(oracle):
    """integrating towards the probe or away from it gives the same interval."""
    a = A.make_config(0, nx=32, ny=32, ncascades=4)
    J0 = oracle.solve_atmosphere(a, order=0)["J"]
    J1 = oracle.solve_atmosphere(a, order=1)["J"]
    assert np.max(np.abs(J0 - J1) / J0) < 1e-13


# ----------------------------------------------------------------------------- P13: cascade 0
def test_P13_cascade0_closed_form(oracle):
    """Cascade-0 interval [0,1] along the diagonals from a cell centre: sqrt2/2 in
    the own cell, 1 - sqrt2/2 in the diagonal neighbour (vacuum outside the box)."""
    nx, ny = 8, 8
    chi, eta = A.random_field(nx, ny, 1, seed=7)
    out = oracle.solve(chi, eta, 2, dump_cascade=0)
    c64, e64 = chi[..., 0].astype(float), eta[..., 0].astype(float)
    a, b = R2 / 2, 1 - R2 / 2
    quad = [(1, 1), (-1, 1), (-1, -1), (1, -1)]  # theta = pi/4 + q pi/2
    for y in range(ny):
        for x in range(nx):
            for q, (sx, sy) in enumerate(quad):
                xo, yo = x + sx, y + sy
                inside = 0 <= xo < nx and 0 <= yo < ny
                cd, ed = (c64[yo, xo], e64[yo, xo]) if inside else (0.0, 0.0)
                To = np.exp(-c64[y, x] * a)
                I = e64[y, x] / c64[y, x] * (1 - To) + To * (ed / cd * (1 - np.exp(-cd * b)) if inside else 0.0)
                T = To * np.exp(-cd * b)
                assert np.isclose(out["dump_I"][y, x, q, 0], I, rtol=1e-12)
                assert np.isclose(out["dump_T"][y, x, q, 0], T, rtol=1e-12)


def test_hand_derived_2x2_two_cascades(oracle):
    """2x2 cells, 2 cascades, written out by hand.  Cascade 1 has one probe at the grid centre
    (1,1) with 16 directions theta_k = 2 pi (k+1/2)/16 and interval [1, inf): the ray stays in the
    quadrant cell of its direction and leaves the box at t = 1/max(|cos|,|sin|).  Cascade 0:
    P13 geometry; every cell has that single (clamped) parent, so the bilinear weights collapse
    and U_k is the mean of children 4k..4k+3.  J = mean_k (I0_k + T0_k U_k)."""
    chi = np.array([[[0.7], [1.3]], [[0.2], [2.1]]], np.float32)  # [y][x][l]
    S = np.array([[[1.0], [0.5]], [[2.0], [0.25]]], np.float32)
    eta = chi * S
    Ib, Ia = 0.3, 0.9
    c, e = chi[..., 0].astype(float), eta[..., 0].astype(float)
    M1 = np.zeros(16)
    for k in range(16):
        th = 2 * np.pi * (k + 0.5) / 16
        cx, sy = np.cos(th), np.sin(th)
        ell = 1.0 / max(abs(cx), abs(sy)) - 1.0
        x, y = (1 if cx > 0 else 0), (1 if sy > 0 else 0)
        T = np.exp(-c[y, x] * ell)
        M1[k] = e[y, x] / c[y, x] * (1 - T) + T * (Ib if sy < 0 else Ia)
    U = M1.reshape(4, 4).mean(axis=1)
    a, b = R2 / 2, 1 - R2 / 2
    quad = [(1, 1), (-1, 1), (-1, -1), (1, -1)]
    J = np.zeros((2, 2))
    for y in range(2):
        for x in range(2):
            for q, (sx, sy) in enumerate(quad):
                xo, yo = x + sx, y + sy
                To = np.exp(-c[y, x] * a)
                I = e[y, x] / c[y, x] * (1 - To)
                T = To
                if 0 <= xo < 2 and 0 <= yo < 2:
                    Td = np.exp(-c[yo, xo] * b)
                    I += To * e[yo, xo] / c[yo, xo] * (1 - Td)
                    T *= Td
                J[y, x] += 0.25 * (I + T * U[q])
    out = oracle.solve(chi, eta, 2, I_below=[Ib], I_above=[Ia])
    assert np.allclose(out["J"][..., 0], J, rtol=1e-13)


# ----------------------------------------------------------------------------- P3 / P4
@pytest.mark.parametrize("ncasc", [1, 2, 3, 5])
def test_P3_constant_source_gives_J_equal_S(oracle, ncasc):
    """eta = chi S0 everywhere and boundary intensity S0 => J = S0 (north_star; pins the BC
    placement G9/G10, the bilinear weights G5/G6, child averaging and the J normalisation)."""
    a = A.make_config(0, nx=48, ny=32, nlambda=2, ncascades=ncasc)
    S0 = 2.0  # exact in fp32 so that eta/chi == S0 exactly
    chi = a.chi.copy()
    chi[5:9, 7:20] = 0.0  # holes of exact vacuum (G11)
    out = oracle.solve(chi, chi * np.float32(S0), ncasc, I_below=[S0] * 2, I_above=[S0] * 2)
    assert np.max(np.abs(out["J"] - S0)) < 1e-13


@pytest.mark.parametrize("ncasc", [1, 3, 5])
def test_P4_empty_domain_passes_boundary_through(oracle, ncasc):
    """chi = eta = 0: isotropic B => J = B; lit from below only => J = B/2 exactly (half of every
    direction set points down) — 'an empty domain passes boundary intensity through unchanged'."""
    z = np.zeros((32, 64, 1), np.float32)
    B = 0.8125
    assert np.max(np.abs(oracle.solve(z, z, ncasc, I_below=[B], I_above=[B])["J"] - B)) < 1e-15
    assert np.max(np.abs(oracle.solve(z, z, ncasc, I_below=[B], I_above=[0])["J"] - B / 2)) < 1e-15
    assert np.max(np.abs(oracle.solve(z, z, ncasc)["J"])) == 0.0


def test_G11_vacuum_limit_is_continuous(oracle):
    a = A.make_config(0, nx=32, ny=32, ncascades=3)
    chi, eta = a.chi.copy(), a.eta.copy()
    chi[10:20, 10:20] = 0.0
    eta[10:20, 10:20] = 0.0
    J0 = oracle.solve(chi, eta, 3)["J"]
    chi[10:20, 10:20] = 1e-30
    J1 = oracle.solve(chi, eta, 3)["J"]
    assert np.max(np.abs(J0 - J1)) < 1e-14


# ----------------------------------------------------------------------------- P5
def test_P5_single_cascade_is_four_ray_long_characteristics(oracle):
    """ncasc = 1: 4 diagonal rays to the edge.  Uniform chi, S, isotropic B:
    J = S - (S - B) 1/4 sum_k exp(-chi sqrt2 min(dx_k, dy_k)), d = centre-to-face distances
    (the 'uniform slab follows the closed-form exp(-tau) attenuation' check of north_star)."""
    nx, ny, chi0, S0, B = 24, 16, 0.11, 1.5, 0.25
    chi = np.full((ny, nx, 1), chi0, np.float32)
    eta = np.full((ny, nx, 1), np.float32(chi0) * np.float32(S0), np.float32)
    c = float(chi[0, 0, 0])
    S = float(eta[0, 0, 0]) / c
    J = oracle.solve(chi, eta, 1, I_below=[B], I_above=[B])["J"][..., 0]
    y, x = np.mgrid[0:ny, 0:nx]
    dxp, dxm, dyp, dym = nx - (x + 0.5), x + 0.5, ny - (y + 0.5), y + 0.5
    att = sum(np.exp(-c * R2 * np.minimum(dx, dy))
              for dx, dy in ((dxp, dyp), (dxm, dyp), (dxm, dym), (dxp, dym)))
    assert np.allclose(J, S - (S - B) * att / 4, rtol=1e-13)


# ----------------------------------------------------------------------------- P6 / P7 / P8
def test_P6_linearity_in_eta_and_boundary(oracle):
    a = A.make_config(0, nx=32, ny=32, ncascades=4)
    rng = np.random.default_rng(8)
    e1 = a.eta
    e2 = (a.chi * rng.uniform(0, 1, a.chi.shape)).astype(np.float32)
    J1 = oracle.solve(a.chi, e1, 4, I_below=[0.5], I_above=[0.0])["J"]
    J2 = oracle.solve(a.chi, e2, 4, I_below=[0.0], I_above=[0.25])["J"]
    esum = e1.astype(np.float64) + 4.0 * e2  # 4*e2 exact; keep the sum exactly representable
    esum32 = esum.astype(np.float32)
    ok = esum32.astype(np.float64) == esum
    e1b = np.where(ok, e1, 0).astype(np.float32)  # drop the few cells where the sum rounds
    e2b = np.where(ok, e2, 0).astype(np.float32)
    J1 = oracle.solve(a.chi, e1b, 4, I_below=[0.5], I_above=[0.0])["J"]
    J2 = oracle.solve(a.chi, e2b, 4, I_below=[0.0], I_above=[0.25])["J"]
    J12 = oracle.solve(a.chi, (e1b.astype(np.float64) + 4.0 * e2b).astype(np.float32), 4,
                       I_below=[0.5], I_above=[1.0])["J"]
    assert np.allclose(J12, J1 + 4.0 * J2, rtol=1e-12)


def _d4(f, op):
    """Apply an element of D4 to a [ny][nx][L] field (square grids)."""
    return {"id": lambda g: g, "fx": lambda g: g[:, ::-1], "fy": lambda g: g[::-1],
            "r180": lambda g: g[::-1, ::-1], "t": lambda g: g.transpose(1, 0, 2),
            "r90": lambda g: g.transpose(1, 0, 2)[::-1], "r270": lambda g: g.transpose(1, 0, 2)[:, ::-1],
            "at": lambda g: g.transpose(1, 0, 2)[::-1, ::-1]}[op](f)


@pytest.mark.parametrize("op", ["fx", "fy", "r180", "t", "r90", "r270", "at"])
def test_P7_d4_symmetry(oracle, op):
    """Direction set theta_k = 2 pi (k+1/2)/N and the probe lattices are D4-symmetric (G4, G5):
    transforming the inputs transforms J.  Catches wrong child mapping 4k+j / parent indexing."""
    a = A.make_config(0, nx=32, ny=32, ncascades=4, seed=11)
    J = oracle.solve(a.chi, a.eta, 4)["J"]
    chi2 = np.ascontiguousarray(_d4(a.chi, op))
    eta2 = np.ascontiguousarray(_d4(a.eta, op))
    J2 = oracle.solve(chi2, eta2, 4)["J"]
    assert np.allclose(J2, _d4(J, op), rtol=1e-11)


def test_P7_axis_flips_with_anisotropic_boundary(oracle):
    a = A.make_config(4, nx=128, ny=32, nlambda=2, ncascades=5)
    Jf = oracle.solve(a.chi, a.eta, 5, I_below=[1, 2], I_above=[0, 0.5])["J"]
    chi2, eta2 = np.ascontiguousarray(a.chi[::-1]), np.ascontiguousarray(a.eta[::-1])
    J2 = oracle.solve(chi2, eta2, 5, I_below=[0, 0.5], I_above=[1, 2])["J"]  # flip y: swap BC
    assert np.allclose(J2, Jf[::-1], rtol=1e-11, atol=1e-15)
    chi3, eta3 = np.ascontiguousarray(a.chi[:, ::-1]), np.ascontiguousarray(a.eta[:, ::-1])
    J3 = oracle.solve(chi3, eta3, 5, I_below=[1, 2], I_above=[0, 0.5])["J"]
    assert np.allclose(J3, Jf[:, ::-1], rtol=1e-11, atol=1e-15)


def test_P8_wavelengths_are_independent(oracle):
    a = A.make_config(2, nx=32, ny=32, nlambda=5, ncascades=4)
    full = oracle.solve_atmosphere(a)
    perm = [3, 0, 4, 1, 2]
    Jp = oracle.solve(np.ascontiguousarray(a.chi[..., perm]), np.ascontiguousarray(a.eta[..., perm]), 4)["J"]
    assert np.array_equal(Jp, full["J"][..., perm])
    for l in (0, 3):
        Jl = oracle.solve(np.ascontiguousarray(a.chi[..., l:l + 1]), np.ascontiguousarray(a.eta[..., l:l + 1]), 4)["J"]
        assert np.array_equal(Jl[..., 0], full["J"][..., l])
    w = np.array([0.1, 0.2, 0.3, 0.25, 0.15], np.float32)
    out = oracle.solve(a.chi, a.eta, 4, weights=w)
    assert np.allclose(out["Jbar"], (out["J"] * w.astype(np.float64)).sum(-1), rtol=1e-15)


# ----------------------------------------------------------------------------- P9
def test_P9_ray_counts(oracle):
    """alpha = 2: every cascade has 4 nx ny intervals; cascade 0 walks exactly
    2 cells per interior ray; wholly-outside cascades walk none (cfg 0)."""
    a = A.make_config(0)
    out = oracle.solve_atmosphere(a, want_counts=True)
    assert list(out["intervals"]) == [4 * 64 * 64] * 5
    assert out["segments"][0] == 2 * 4 * 64 * 64 - 4 * (2 * 64 - 1)  # edge cells lose the neighbour
    assert out["segments"][4] == 0  # t_4 = 85 from a probe at most 64 sqrt2 = 90.5 from a corner...
    assert 6.5e5 < out["segments"].sum() < 7.0e5  # 6.93e5 in SURVEY.md (cascade 0 over-counted there)


def test_window_solve_is_the_full_solve_restricted(oracle):
    """The sampled-cell path used at full size computes bit-identical numbers."""
    a = A.make_config(1, nx=64, ny=64, nlambda=2, ncascades=5)
    full = oracle.solve_atmosphere(a)["J"]
    for (x0, x1, y0, y1) in [(0, 1, 0, 1), (63, 64, 63, 64), (17, 22, 40, 41), (30, 34, 30, 34), (0, 64, 5, 6)]:
        w = oracle.solve_atmosphere(a, window=(x0, x1, y0, y1))["J"]
        assert np.array_equal(w, full[y0:y1, x0:x1])


# ----------------------------------------------------------------------------- P10 / P12
def test_P10_against_brute_force_long_characteristics(oracle):
    """The oracle computes radiative transfer, not just something self-consistent: compare with
    brute-force long characteristics (2048 directions to the edge) on config 0.  The method is an
    approximation ('less than a few per cent' in resolved models; worse within a few
    cells of the edge where the lookup is clamped): interior max < 5 %, mean < 1 %."""
    a = A.make_config(0)
    J = oracle.solve_atmosphere(a)["J"][..., 0]
    rng = np.random.default_rng(9)
    cells = np.stack([rng.integers(8, 56, 120), rng.integers(8, 56, 120)], axis=1)
    Jlc = refs.long_characteristics_J(a.chi[..., 0].astype(float), a.eta[..., 0].astype(float), cells, 2048)
    rel = np.abs(J[cells[:, 1], cells[:, 0]] - Jlc) / Jlc
    assert rel.max() < 0.05 and rel.mean() < 0.01, (rel.max(), rel.mean())


def test_P10_lc_reference_is_converged():
    a = A.make_config(0)
    cells = np.array([[10, 10], [32, 32], [50, 20]])
    c, e = a.chi[..., 0].astype(float), a.eta[..., 0].astype(float)
    J1 = refs.long_characteristics_J(c, e, cells, 1024)
    J2 = refs.long_characteristics_J(c, e, cells, 4096)
    assert np.max(np.abs(J1 - J2) / J2) < 1e-3


def test_P12_opaque_disc_falloff(oracle):
    """Fig. 6: one opaque disc in vacuum, zero boundary.  Flatland theory: the
    disc subtends 2 asin(R/r) of 2 pi, J(r) = S asin(R/r)/pi.  The paper: the cascades solution
    lies above theory (pixelised disc), error high in the first pixels, ringing of order 10 %,
    rising again near the edge.  Asserted: sign, and a loose bound on the size."""
    n, R, S0 = 128, 6.0, 1.0
    y, x = np.mgrid[0:n, 0:n]
    r = np.hypot(x + 0.5 - n / 2, y + 0.5 - n / 2)
    chi = np.where(r <= R, 100.0, 0.0).astype(np.float32)[..., None]
    eta = chi * np.float32(S0)
    J = oracle.solve(chi, eta, 6)["J"][..., 0]
    sel = (r > R + 3) & (r < n / 2 - 14)
    theory = S0 * np.arcsin(R / r[sel]) / np.pi
    err = (J[sel] - theory) / theory
    assert err.min() > -0.02, err.min()      # 'always lies above the theoretically predicted solution'
    assert 0.02 < err.mean() < 0.20, err.mean()
    assert err.max() < 0.45, err.max()


# ----------------------------------------------------------------------------- 2.5D inclinations (f2)
def test_gauss_radau_rule_is_exact_for_polynomials():
    """The inclination quadrature handed to both sides (Gauss-Radau, 8 rays, one hemisphere):
    n nodes with one fixed at mu = 0 integrate mu^p over [0, 1] exactly for p <= 2n - 2; weights sum to 1."""
    for n in (1, 2, 3, 4, 8):
        mu, w = A.gauss_radau(n)
        assert mu[0] == 0.0 and np.all(np.diff(mu) > 0) and mu[-1] < 1.0 and np.all(w > 0)
        for p in range(2 * n - 1):
            assert abs(np.sum(w * mu ** p) - 1.0 / (p + 1)) < 1e-12
    assert abs(np.sum(A.gauss_radau(8)[1] * A.gauss_radau(8)[0] ** 15) - 1.0 / 16) > 1e-9  # and not beyond


def test_I1_inclined_uniform_slab_closed_form(oracle):
    """ncasc = 1, uniform chi and S, isotropic boundary B, inclined rays: the ray with direction cosine mu
    to the invariant axis has path length l / sqrt(1 - mu^2) for projected length l, so
    J = S - (S - B) sum_m w_m 1/4 sum_k exp(-chi sqrt2 min(dx_k, dy_k) / sqrt(1 - mu_m^2))."""
    nx, ny, chi0, S0, B = 24, 16, 0.11, 1.5, 0.25
    chi = np.full((ny, nx, 1), chi0, np.float32)
    eta = np.full((ny, nx, 1), np.float32(chi0) * np.float32(S0), np.float32)
    c = float(chi[0, 0, 0])
    S = float(eta[0, 0, 0]) / c
    mu, w = A.gauss_radau(4)
    J = oracle.solve_inclined(chi, eta, 1, mu, w, I_below=[B], I_above=[B])["J"][..., 0]
    y, x = np.mgrid[0:ny, 0:nx]
    dxp, dxm, dyp, dym = nx - (x + 0.5), x + 0.5, ny - (y + 0.5), y + 0.5
    att = 0.0
    for m in range(4):
        f = 1.0 / np.sqrt(1.0 - mu[m] ** 2)
        att = att + w[m] * sum(np.exp(-c * f * R2 * np.minimum(dx, dy))
                               for dx, dy in ((dxp, dyp), (dxm, dyp), (dxm, dym), (dxp, dym))) / 4
    assert np.allclose(J, S - (S - B) * att, rtol=1e-13)


def test_I2_inclined_invariants(oracle):
    """(a) one in-plane ray (mu = 0, w = 1) is the flatland solve, bit for bit; (b) constant S with boundary
    S gives J = S for any inclination set; (c) an empty domain passes the boundary through: J = B sum w;
    (d) a path scale f is the flatland solve of the atmosphere (f chi, f eta) when f is a power of two
    (the scaled inputs are then exact in fp32)."""
    a = A.make_config(0, nx=32, ny=32, nlambda=2, ncascades=4, seed=21)
    flat = oracle.solve(a.chi, a.eta, 4, I_below=[0.3, 0.1], I_above=[0.0, 0.2])["J"]
    one = oracle.solve_inclined(a.chi, a.eta, 4, [0.0], [1.0], I_below=[0.3, 0.1], I_above=[0.0, 0.2])["J"]
    assert np.array_equal(flat, one)
    mu, w = A.gauss_radau(8)
    S0 = 0.75
    eta = (a.chi * np.float32(S0)).astype(np.float32)
    ok = eta.astype(np.float64) == a.chi.astype(np.float64) * S0   # 0.75 chi is exact unless it rounds
    chi = np.where(ok, a.chi, 0).astype(np.float32)
    eta = np.where(ok, eta, 0).astype(np.float32)
    J = oracle.solve_inclined(chi, eta, 4, mu, w, I_below=[S0, S0], I_above=[S0, S0])["J"]
    assert np.allclose(J, S0, rtol=1e-13)
    z = np.zeros_like(a.chi)
    J = oracle.solve_inclined(z, z, 4, mu, w, I_below=[0.5, 1.0], I_above=[0.0, 1.0])["J"]
    assert np.allclose(J[..., 0], 0.25, rtol=1e-14) and np.allclose(J[..., 1], 1.0, rtol=1e-14)
    scaled = oracle.solve(a.chi, a.eta, 4, path_scale=4.0)["J"]
    direct = oracle.solve((4 * a.chi).astype(np.float32), (4 * a.eta).astype(np.float32), 4)["J"]
    assert np.allclose(scaled, direct, rtol=1e-13)


def test_I3_inclined_rays_see_more_optical_depth(oracle):
    """Sanity of the sign of the effect: an absorbing, non-emitting slab lit from below transmits less along
    inclined rays (longer paths), so J with the 8-ray quadrature lies strictly below the in-plane J and
    above the J of the most inclined ray alone."""
    a = A.make_config(0, nx=32, ny=32, ncascades=4, seed=3)
    z = np.zeros_like(a.eta)
    mu, w = A.gauss_radau(8)
    flat = oracle.solve(a.chi, z, 4, I_below=[1.0])["J"]
    incl = oracle.solve_inclined(a.chi, z, 4, mu, w, I_below=[1.0])["J"]
    steep = oracle.solve_inclined(a.chi, z, 4, mu[-1:], [1.0], I_below=[1.0])["J"]
    m = flat > 1e-6
    assert np.all(incl[m] < flat[m]) and np.all(steep[m] < incl[m])


# ----------------------------------------------------------------------------- moving line (f1)
def _static_fields(line, xl, wx=0.0, wy=0.0):
    """chi, eta [ny][nx][L] in fp64 of a line atmosphere as seen along one direction (test-side restatement)."""
    f = line.astype(np.float64)
    a = xl[None, None, :] + (f[..., 4] * wx + f[..., 5] * wy)[..., None]
    phi = np.exp(-a * a) / np.sqrt(np.pi)
    chi = f[..., 0:1] + f[..., 2:3] * phi
    eta = f[..., 0:1] * f[..., 1:2] + f[..., 2:3] * f[..., 3:4] * phi
    return chi, eta


def test_V1_static_line_equals_precomputed_opacities(oracle):
    """v = 0: the on-the-fly line mode is the GivenFs solve of chi_l = chi_c + chi_line phi(x_l),
    eta_l = chi_c S_c + chi_line S_line phi(x_l); equal up to the fp32 rounding of the precomputed inputs."""
    a = A.line_config2(nx=32, ny=32, nlambda=5, ncascades=4)
    a.line[..., 4:6] = 0.0
    chi, eta = _static_fields(a.line, a.xl)
    J1 = oracle.solve_line(a.line, a.xl, 4, I_below=[0.2] * 5)["J"]
    J0 = oracle.solve(chi.astype(np.float32), eta.astype(np.float32), 4, I_below=[0.2] * 5)["J"]
    assert np.allclose(J1, J0, rtol=5e-7)


def test_V2_uniform_flow_single_cascade_closed_form(oracle):
    """ncasc = 1 (4 diagonal rays to the edge), uniform medium with a uniform flow v: the ray traced along
    w_k carries photons moving along -w_k, which see the line at x = -v.w_k:
    J_l = 1/4 sum_k [S_kl (1 - e^{-chi_kl d_k}) + B e^{-chi_kl d_k}], chi_kl = chi_c + chi_line phi(x_l + v.w_k)."""
    nx, ny, L = 12, 20, 7
    xl = np.linspace(-3, 3, L)
    cell = np.array([0.01, 0.7, 0.4, 2.0, 1.3, -0.6], np.float32)
    line = np.broadcast_to(cell, (ny, nx, 6)).copy()
    B = 0.35
    J = oracle.solve_line(line, xl, 1, I_below=[B] * L, I_above=[B] * L)["J"]
    c = cell.astype(np.float64)
    y, x = np.mgrid[0:ny, 0:nx]
    dxp, dxm, dyp, dym = nx - (x + 0.5), x + 0.5, ny - (y + 0.5), y + 0.5
    want = np.zeros((ny, nx, L))
    for (sx, sy), (dx, dy) in zip(((1, 1), (-1, 1), (-1, -1), (1, -1)), ((dxp, dyp), (dxm, dyp), (dxm, dym), (dxp, dym))):
        wx, wy = sx / R2, sy / R2
        d = R2 * np.minimum(dx, dy)
        for l in range(L):
            a_ = xl[l] + (c[4] * wx + c[5] * wy)
            phi = np.exp(-a_ * a_) / np.sqrt(np.pi)
            chi = c[0] + c[2] * phi
            S = (c[0] * c[1] + c[2] * c[3] * phi) / chi
            att = np.exp(-chi * d)
            want[..., l] += (S * (1 - att) + B * att) / 4
    assert np.allclose(J, want, rtol=1e-12)


def test_V3_moving_line_symmetries(oracle):
    """(a) reversing every velocity and mirroring the wavelength grid leaves J_l -> J_{L-1-l} (phi is even);
    (b) rotating the atmosphere by 90 degrees, velocities included, rotates J; (c) a velocity field changes J
    (the mode is not ignoring it)."""
    a = A.line_config2(nx=32, ny=32, nlambda=6, ncascades=4, seed=4)
    J = oracle.solve_line(a.line, a.xl, 4)["J"]
    rev = a.line.copy()
    rev[..., 4:6] *= -1
    Jr = oracle.solve_line(rev, -a.xl[::-1], 4)["J"]
    assert np.allclose(Jr, J[..., ::-1], rtol=1e-12)
    # np.rot90(f, 1, axes=(0, 1)): r[y'][x'] = f[x'][n-1-y'], i.e. the point (x, y) goes to (y, -x): a clockwise
    # quarter turn, under which a vector (v_x, v_y) becomes (v_y, -v_x)
    rot = np.rot90(a.line, 1, axes=(0, 1)).copy()
    vx, vy = rot[..., 4].copy(), rot[..., 5].copy()
    rot[..., 4], rot[..., 5] = vy, -vx
    J90 = oracle.solve_line(rot, a.xl, 4)["J"]
    assert np.allclose(J90, np.rot90(J, 1, axes=(0, 1)), rtol=1e-11)
    rot[..., 4], rot[..., 5] = -vy, vx                     # the vector turned the wrong way must NOT match
    assert not np.allclose(oracle.solve_line(rot, a.xl, 4)["J"], np.rot90(J, 1, axes=(0, 1)), rtol=1e-4)
    still = a.line.copy()
    still[..., 4:6] = 0
    assert np.max(np.abs(oracle.solve_line(still, a.xl, 4)["J"] / J - 1)) > 1e-2


def test_V4_inclined_moving_line(oracle):
    """f1 x f2: (a) v = 0 is the inclined GivenFs solve of the precomputed opacities; (b) uniform flow, one
    cascade, one inclined ray set: per-ray closed form with path d / sin(i) and projected velocity v.w sin(i)."""
    a = A.line_config2(nx=32, ny=32, nlambda=4, ncascades=4)
    mu, w = A.gauss_radau(4)
    still = a.line.copy()
    still[..., 4:6] = 0.0
    chi, eta = _static_fields(still, a.xl)
    J1 = oracle.solve_line(still, a.xl, 4, mu=mu, w_mu=w)["J"]
    J0 = oracle.solve_inclined(chi.astype(np.float32), eta.astype(np.float32), 4, mu, w)["J"]
    assert np.allclose(J1, J0, rtol=5e-7)
    nx, ny, L = 10, 14, 5
    xl = np.linspace(-2, 2, L)
    cell = np.array([0.02, 0.5, 0.3, 1.7, -0.9, 1.1], np.float32)
    line = np.broadcast_to(cell, (ny, nx, 6)).copy()
    B, m0 = 0.2, 0.6
    J = oracle.solve_line(line, xl, 1, I_below=[B] * L, I_above=[B] * L, mu=[m0], w_mu=[1.0])["J"]
    c = cell.astype(np.float64)
    si = np.sqrt(1 - m0 * m0)
    y, x = np.mgrid[0:ny, 0:nx]
    dxp, dxm, dyp, dym = nx - (x + 0.5), x + 0.5, ny - (y + 0.5), y + 0.5
    want = np.zeros((ny, nx, L))
    for (sx, sy), (dx, dy) in zip(((1, 1), (-1, 1), (-1, -1), (1, -1)), ((dxp, dyp), (dxm, dyp), (dxm, dym), (dxp, dym))):
        d = R2 * np.minimum(dx, dy) / si
        for l in range(L):
            a_ = xl[l] + si * (c[4] * sx + c[5] * sy) / R2
            phi = np.exp(-a_ * a_) / np.sqrt(np.pi)
            chi_ = c[0] + c[2] * phi
            S = (c[0] * c[1] + c[2] * c[3] * phi) / chi_
            att = np.exp(-chi_ * d)
            want[..., l] += (S * (1 - att) + B * att) / 4
    assert np.allclose(J, want, rtol=1e-12)


# ----------------------------------------------------------------------------- bilinear fix (f3)
def test_F1_bilinear_fix_invariants(oracle):
    """With the bilinear fix: J = S for a constant source function with boundary S; an empty
    domain passes the boundary through; with a single cascade (no parents) the fix changes nothing; D4 symmetry
    still holds (transpose)."""
    a = A.make_config(0, nx=32, ny=32, ncascades=4, seed=2)
    S0 = 0.75
    eta = (a.chi * np.float32(S0)).astype(np.float32)
    ok = eta.astype(np.float64) == a.chi.astype(np.float64) * S0
    chi = np.where(ok, a.chi, 0).astype(np.float32)
    eta = np.where(ok, eta, 0).astype(np.float32)
    for nc in (2, 3, 4):
        J = oracle.solve(chi, eta, nc, I_below=[S0], I_above=[S0], bilinear_fix=True)["J"]
        assert np.allclose(J, S0, rtol=1e-13)
    z = np.zeros_like(chi)
    assert np.allclose(oracle.solve(z, z, 4, I_below=[1.0], bilinear_fix=True)["J"], 0.5, rtol=1e-14)
    one = oracle.solve(a.chi, a.eta, 1, I_below=[0.3])["J"]
    assert np.array_equal(one, oracle.solve(a.chi, a.eta, 1, I_below=[0.3], bilinear_fix=True)["J"])
    J = oracle.solve(a.chi, a.eta, 4, bilinear_fix=True)["J"]
    Jt = oracle.solve(np.ascontiguousarray(a.chi.transpose(1, 0, 2)), np.ascontiguousarray(a.eta.transpose(1, 0, 2)), 4,
                      bilinear_fix=True)["J"]
    assert np.allclose(Jt.transpose(1, 0, 2), J, rtol=1e-11)
    assert np.max(np.abs(J / oracle.solve(a.chi, a.eta, 4)["J"] - 1)) > 1e-3   # and it is not a no-op


def test_F2_bilinear_fix_against_independent_two_cascade_reference(oracle):
    """Brute-force restatement with the sorting-based ray/cell intersection of tests/refs.py, 2 cascades on a
    small grid: cascade 1 (top) marches to the edge; every cascade-0 ray is traced four times, from its start
    p + t_0 w to q + t_1 w for each of the four parents q, merged with the mean of q's four children of that
    direction and combined with the bilinear weights 3/4, 1/4 (clamped at the lattice edge)."""
    nx, ny = 8, 6
    rng = np.random.default_rng(12)
    chi = rng.uniform(0.05, 1.5, (ny, nx, 1)).astype(np.float32)
    eta = (chi * rng.uniform(0.2, 2.0, (ny, nx, 1))).astype(np.float32)
    Ib, Ia = 0.4, 0.1
    J = oracle.solve(chi, eta, 2, I_below=[Ib], I_above=[Ia], bilinear_fix=True)["J"][..., 0]
    c, e = chi[..., 0].astype(np.float64).ravel(), eta[..., 0].astype(np.float64).ravel()
    t1 = 1.0
    M1 = np.zeros((ny // 2, nx // 2, 16))
    for b in range(ny // 2):
        for a_ in range(nx // 2):
            for k in range(16):
                th = 2 * np.pi * (k + 0.5) / 16
                cells, ds = refs.segments_by_sorting(nx, ny, (a_ + 0.5) * 2, (b + 0.5) * 2, th, t1, 1e9)
                I, T = refs.integrate(c, e, cells, ds)
                M1[b, a_, k] = I + T * (Ib if np.sin(th) < 0 else Ia)

    def parents(a_, n):
        base, f = ((a_ - 1) // 2, 0.25) if a_ % 2 else (a_ // 2 - 1, 0.75)
        return (min(max(base, 0), n - 1), 1 - f), (min(max(base + 1, 0), n - 1), f)

    want = np.zeros((ny, nx))
    for y in range(ny):
        for x in range(nx):
            for k in range(4):
                th = 2 * np.pi * (k + 0.5) / 4
                w = np.array([np.cos(th), np.sin(th)])
                A0 = np.array([x + 0.5, y + 0.5])           # t_0 = 0
                for (bq, wb) in parents(y, ny // 2):
                    for (aq, wa) in parents(x, nx // 2):
                        B = np.array([(aq + 0.5) * 2, (bq + 0.5) * 2]) + t1 * w
                        d = B - A0
                        ln = np.hypot(*d)
                        cells, ds = refs.segments_by_sorting(nx, ny, A0[0], A0[1], np.arctan2(d[1], d[0]), 0.0, ln)
                        I, T = refs.integrate(c, e, cells, ds)
                        want[y, x] += 0.25 * wa * wb * (I + T * M1[bq, aq, 4 * k:4 * k + 4].mean())
    assert np.allclose(J, want, rtol=1e-10)


def test_F3_bilinear_fix_reduces_the_ringing(oracle):
    """Fig. 6: around a small opaque disc in vacuum the basic method rings where the
    cascades hand over; the fix removes most of it.  Against flatland theory J = S asin(R/r)/pi: rms and
    maximum error drop by more than a third (the rest is the pixelised disc being larger than the circle:
    still always above theory)."""
    n, R = 128, 6
    y, x = np.mgrid[0:n, 0:n]
    r = np.hypot(x + 0.5 - n / 2, y + 0.5 - n / 2)
    chi = np.where(r <= R, 100.0, 0.0).astype(np.float32)[..., None]
    m = (r > R + 3) & (r < 50)
    theory = np.arcsin(R / r[m]) / np.pi
    err = {}
    for fix in (False, True):
        J = oracle.solve(chi, chi.copy(), 6, bilinear_fix=fix)["J"][..., 0]
        err[fix] = J[m] / theory - 1
    assert np.all(err[True] > 0)
    assert np.sqrt(np.mean(err[True] ** 2)) < 0.65 * np.sqrt(np.mean(err[False] ** 2))
    assert err[True].max() < 0.65 * err[False].max()


# ----------------------------------------------------------------------------- diagonal ALO (f4)
def test_A1_alo_is_the_own_cell_transmittance_of_cascade_0(oracle):
    """eq. 17: Lambda* = exp(-chi ds), ds from the cell centre to its edge along the ray.  Cascade
    0's interval [0, 1] covers the own cell over sqrt2/2 and the diagonal neighbour over 1 - sqrt2/2 (P13): in an
    atmosphere whose occupied cells have vacuum diagonal neighbours, the oracle's own cascade-0 transmittances
    (dump_T, all four directions) ARE the ALO.  Also: vacuum gives 1; weights of the inclinations sum to 1."""
    rng = np.random.default_rng(3)
    ny = nx = 16
    y, x = np.mgrid[0:ny, 0:nx]
    occ = (x % 2 == 0) & (y % 2 == 0)           # diagonal neighbours of an occupied cell are (odd, odd): empty
    chi = np.where(occ, rng.uniform(0.1, 3.0, (ny, nx)), 0.0).astype(np.float32)[..., None]
    d = oracle.solve(chi, chi.copy(), 2, dump_cascade=0)
    lam = oracle.alo(chi=chi)
    for k in range(4):
        assert np.allclose(d["dump_T"][:, :, k, :][occ], lam[occ], rtol=1e-14)
    assert np.all(lam[~occ] == 1.0)
    mu, w = A.gauss_radau(4)
    big = oracle.alo(chi=np.full((2, 2, 1), 1e-9, np.float32), mu=mu, w_mu=w)
    assert np.allclose(big, 1.0, atol=1e-8)
    li = oracle.alo(chi=chi, mu=mu, w_mu=w)
    assert np.all(li[occ] < lam[occ]) and np.all(li[occ] > 0)        # inclined rays see more optical depth
    # line mode with v = 0 is the GivenFs value of the static opacities
    a = A.line_config2(nx=8, ny=8, nlambda=3, ncascades=2)
    a.line[..., 4:6] = 0
    c, _ = _static_fields(a.line, a.xl)
    assert np.allclose(oracle.alo(line=a.line, xl=a.xl), np.exp(-c * np.sqrt(0.5)), rtol=1e-12)


def _checkerboard(rng, n=16):
    y, x = np.mgrid[0:n, 0:n]
    occ = (x % 2 == 0) & (y % 2 == 0)           # diagonal neighbours of an occupied cell are (odd, odd): empty
    return occ


def test_A2_inclined_alo_is_the_inclined_cascade_0_transmittance(oracle):
    """eq. 17 with the 2.5D rays of PAPER.md:281: for EVERY inclination separately, the ALO of that inclination alone
    (mu = [mu_m], weight 1) equals the cascade-0 transmittances of the oracle's own inclined march (path_scale =
    1/sin(inclination), dump_T, all four directions) on the checkerboard atmosphere, where the diagonal neighbour of
    an occupied cell is vacuum; and the quadrature is the weighted sum of those.  Fails if the path from the cell
    centre to its edge is scaled by anything but 1/sin(inclination)."""
    rng = np.random.default_rng(31)
    occ = _checkerboard(rng)
    chi = np.where(occ[..., None], rng.uniform(0.1, 3.0, occ.shape + (3,)), 0.0).astype(np.float32)
    mu, w = A.gauss_radau(8)
    total = 0.0
    for m in range(1, 8):                        # mu[0] = 0 is the flatland ray of A1
        ps = 1.0 / np.sqrt(1.0 - mu[m] ** 2)
        d = oracle.solve(chi, chi.copy(), 2, dump_cascade=0, path_scale=ps)
        lam = oracle.alo(chi=chi, mu=[mu[m]], w_mu=[1.0])
        for k in range(4):
            assert np.allclose(d["dump_T"][:, :, k, :][occ], lam[occ], rtol=1e-13), (m, k)
        assert np.max(np.abs(lam[occ] / oracle.alo(chi=chi)[occ] - 1)) > 1e-3 * m   # and it is not the flatland value
        total = total + w[m] * d["dump_T"][:, :, 0, :]
    total = total + w[0] * oracle.solve(chi, chi.copy(), 2, dump_cascade=0)["dump_T"][:, :, 0, :]
    assert np.allclose(oracle.alo(chi=chi, mu=mu, w_mu=w)[occ], total[occ], rtol=1e-13)


@pytest.mark.parametrize("mu_m", [0.0, 0.6, 0.95])
def test_A3_moving_line_alo_is_the_directional_cascade_0_transmittance(oracle, mu_m):
    """eq. 17 in the line mode with v != 0 ("the monochromatic, directional ALO"): the opacity a
    cascade-0 ray sees depends on its direction through the projected velocity, and for an inclined ray on
    sin(inclination) too (path / sin, in-plane velocity x sin).  On the checkerboard atmosphere the mean over the four
    directions of the oracle's own line-mode cascade-0 transmittances (dump_T of the march, rc_oracle.c) is the ALO.
    Fails if the velocity projection or the path scale of the restated formula is wrong."""
    rng = np.random.default_rng(32)
    occ = _checkerboard(rng)
    n = occ.shape[0]
    line = np.zeros((n, n, 6), np.float32)
    line[..., 0] = np.where(occ, rng.uniform(0.01, 0.3, occ.shape), 0.0)
    line[..., 1] = 1.0
    line[..., 2] = np.where(occ, rng.uniform(0.5, 5.0, occ.shape), 0.0)
    line[..., 3] = 2.0
    line[..., 4] = rng.uniform(-2.0, 2.0, occ.shape)        # v_x, v_y != 0: the four diagonals see four different opacities
    line[..., 5] = rng.uniform(-2.0, 2.0, occ.shape)
    xl = np.array([-1.5, -0.3, 0.0, 0.8, 2.0])
    ps = 1.0 / np.sqrt(1.0 - mu_m ** 2)
    d = oracle.line_intervals(line, xl, 2, 0, path_scale=ps)
    T = d["dump_T"]                                          # [ny][nx][4][L]
    lam = oracle.alo(line=line, xl=xl, mu=[mu_m], w_mu=[1.0])
    assert np.allclose(T.mean(axis=2)[occ], lam[occ], rtol=1e-13)
    spread = T[occ].max(axis=1) / T[occ].min(axis=1)
    assert np.median(spread) > 1.05                          # the direction dependence is really there
    if mu_m > 0:                                             # and so is the dependence on the inclination beyond the path scale
        flat = oracle.alo(line=line, xl=xl)
        assert np.max(np.abs(np.log(lam[occ]) / (np.log(flat[occ]) * ps) - 1)) > 1e-2


def test_A4_plain_bilinear_weights_against_independent_two_cascade_reference(oracle):
    """The non-fix twin of F2 ("the sample for each interval is bilinearly interpolated from the four
    closest probes of cascade i+1", 241 clamp): an independent two-cascade brute force on 8 x 6 cells with the
    sorting-based ray/cell intersection of tests/refs.py, the interpolation weights written from the GEOMETRIC position
    of the cascade-0 probe among the cascade-1 probes - child centre x + 1/2, parents at 2 (q + 1/2): u = x/2 - 1/4 in
    parent index units, lower parent floor(u), weight of the upper parent u - floor(u) - and the indices clamped to the
    lattice.  Swapping 3/4 and 1/4 in the oracle fails this exactly."""
    nx, ny = 8, 6
    rng = np.random.default_rng(14)
    chi = rng.uniform(0.05, 1.5, (ny, nx, 1)).astype(np.float32)
    eta = (chi * rng.uniform(0.2, 2.0, (ny, nx, 1))).astype(np.float32)
    Ib, Ia = 0.4, 0.1
    J = oracle.solve(chi, eta, 2, I_below=[Ib], I_above=[Ia])["J"][..., 0]
    c, e = chi[..., 0].astype(np.float64).ravel(), eta[..., 0].astype(np.float64).ravel()
    t1 = 1.0
    M1 = np.zeros((ny // 2, nx // 2, 16))
    for b in range(ny // 2):
        for a_ in range(nx // 2):
            for k in range(16):
                th = 2 * np.pi * (k + 0.5) / 16
                cells, ds = refs.segments_by_sorting(nx, ny, (a_ + 0.5) * 2, (b + 0.5) * 2, th, t1, 1e9)
                I, T = refs.integrate(c, e, cells, ds)
                M1[b, a_, k] = I + T * (Ib if np.sin(th) < 0 else Ia)

    def interp(a_, n):
        u = (a_ + 0.5) / 2.0 - 0.5                          # position among the parents, in parent index units
        lo = int(np.floor(u))
        f = u - lo
        cl = lambda q: min(max(q, 0), n - 1)
        return (cl(lo), 1.0 - f), (cl(lo + 1), f)

    want = np.zeros((ny, nx))
    for y in range(ny):
        for x in range(nx):
            for k in range(4):
                th = 2 * np.pi * (k + 0.5) / 4
                cells, ds = refs.segments_by_sorting(nx, ny, x + 0.5, y + 0.5, th, 0.0, t1)
                I, T = refs.integrate(c, e, cells, ds)
                U = 0.0
                for (bq, wb) in interp(y, ny // 2):
                    for (aq, wa) in interp(x, nx // 2):
                        U += wa * wb * M1[bq, aq, 4 * k:4 * k + 4].mean()
                want[y, x] += 0.25 * (I + T * U)
    assert np.allclose(J, want, rtol=1e-10)
    # the weights matter at this precision: the swapped pair (1/4 to the nearer parent) is off by far more
    def swapped(a_, n):
        (q0, w0), (q1, w1) = interp(a_, n)
        return (q0, w1), (q1, w0)
    wrong = np.zeros((ny, nx))
    for y in range(ny):
        for x in range(nx):
            for k in range(4):
                th = 2 * np.pi * (k + 0.5) / 4
                cells, ds = refs.segments_by_sorting(nx, ny, x + 0.5, y + 0.5, th, 0.0, t1)
                I, T = refs.integrate(c, e, cells, ds)
                U = sum(wa * wb * M1[bq, aq, 4 * k:4 * k + 4].mean() for (bq, wb) in swapped(y, ny // 2) for (aq, wa) in swapped(x, nx // 2))
                wrong[y, x] += 0.25 * (I + T * U)
    assert np.max(np.abs(wrong / J - 1)) > 1e-3


def test_I4_boundary_per_inclination(oracle):
    """A boundary intensity table over inclination: in an empty domain every constructed ray returns
    its own boundary value, so J_l = sum_m w_m (I_below[m][l] + I_above[m][l]) / 2; a table with equal rows is the
    plain per-wavelength boundary."""
    mu, w = A.gauss_radau(4)
    z = np.zeros((16, 16, 2), np.float32)
    Ib = np.array([[1.0, 0.5], [0.8, 0.4], [0.6, 0.3], [0.2, 0.1]])
    Ia = 0.25 * Ib[::-1]
    J = oracle.solve_inclined(z, z, 3, mu, w, I_below=Ib, I_above=Ia)["J"]
    want = (w[:, None] * (Ib + Ia) / 2).sum(0)
    assert np.allclose(J, want[None, None, :], rtol=1e-14)
    a = A.make_config(0, nx=16, ny=16, nlambda=2, ncascades=3)
    J1 = oracle.solve_inclined(a.chi, a.eta, 3, mu, w, I_below=[0.7, 0.2])["J"]
    J2 = oracle.solve_inclined(a.chi, a.eta, 3, mu, w, I_below=np.tile([0.7, 0.2], (4, 1)))["J"]
    assert np.array_equal(J1, J2)


# ----------------------------------------------------------------------------- sparsity (f4)
def _flagged_counts_geometric(active, ncasc):
    """Flagged probes per cascade from the GEOMETRY alone (no parity rule): the bilinear parents of a probe at
    position p (cell units, per axis) among the cascade-(i+1) probes at (q + 1/2) 2^(i+1) are the two nearest ones,
    q = floor(p / 2^(i+1) - 1/2) and q + 1, clamped to the lattice."""
    ny, nx = active.shape
    flag = active.astype(bool)
    counts = [int(flag.sum())]
    for i in range(ncasc - 1):
        S = 2 ** (i + 1)
        up = np.zeros((ny // S, nx // S), bool)
        bs, as_ = np.nonzero(flag)
        py, px = (bs + 0.5) * 2 ** i, (as_ + 0.5) * 2 ** i
        for dy in (0, 1):
            for dx in (0, 1):
                qy = np.clip(np.floor(py / S - 0.5).astype(int) + dy, 0, ny // S - 1)
                qx = np.clip(np.floor(px / S - 0.5).astype(int) + dx, 0, nx // S - 1)
                up[qy, qx] = True
        flag = up
        counts.append(int(flag.sum()))
    return counts


def test_S1_all_cells_flagged_is_the_dense_solve_bit_for_bit(oracle):
    a = A.make_config(3, nx=64, ny=32, nlambda=3, ncascades=5)
    dense = oracle.solve_atmosphere(a, want_counts=True)
    ones = oracle.solve_atmosphere(a, active=np.ones((32, 64), np.uint8), want_counts=True)
    assert np.array_equal(dense["J"], ones["J"]) and np.array_equal(dense["Jbar"], ones["Jbar"])
    assert np.array_equal(dense["intervals"], ones["intervals"]) and np.array_equal(dense["segments"], ones["segments"])
    line = A.line_config2(nx=32, ny=32, nlambda=3, ncascades=4)
    assert np.array_equal(oracle.solve_atmosphere(line)["J"], oracle.solve_atmosphere(line, active=np.ones((32, 32)))["J"])


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_S2_flagged_probes_are_the_recursive_bilinear_parents(oracle, seed):
    """"This flag then defines the probes of cascade 0 that may be involved ... Their bilinear "parents"
    are recursively flagged up to the maximum cascade, and the radiance intervals are only computed for these flagged
    probes": the number of intervals the oracle computes per cascade = 4^(i+1) x the flagged probes, counted here from
    the geometry (nearest two parents per axis).  A single flagged cell away from the edges flags 2 x 2 parents."""
    rng = np.random.default_rng(seed)
    nx, ny, nc = 64, 48, 5
    act = np.zeros((ny, nx), np.uint8)
    for _ in range(3 + seed):                                  # a few blobs and single cells, some on the edges
        cx, cy, r = rng.integers(0, nx), rng.integers(0, ny), rng.integers(0, 6)
        yy, xx = np.mgrid[0:ny, 0:nx]
        act[(xx - cx) ** 2 + (yy - cy) ** 2 <= r * r] = 1
    act[0, 0] = 1
    chi, eta = A.random_field(nx, ny, 1, seed=seed)
    out = oracle.solve(chi, eta, nc, active=act, want_counts=True)
    want = _flagged_counts_geometric(act, nc)
    assert [int(n) // 4 ** (i + 1) for i, n in enumerate(out["intervals"])] == want
    single = np.zeros((ny, nx), np.uint8)
    single[20, 30] = 1
    out = oracle.solve(chi, eta, 3, active=single, want_counts=True)
    # by hand: cell x = 30 sits at 30.5, between the cascade-1 probes 14 (at 29) and 15 (at 31); those sit between the
    # cascade-2 probes {6, 7} (at 26, 30) and {7, 8}: 3 columns.  y = 20 -> {9, 10} (at 19, 21) -> {4, 5} both: 2 rows.
    assert list(out["intervals"]) == [4 * 1, 16 * (2 * 2), 64 * (3 * 2)]


def test_S3_flagged_cells_keep_their_J_when_the_rest_is_vacuum_anyway(oracle):
    """If the cells that are not flagged hold nothing, the sparse solve must give, on the flagged cells, exactly the dense
    solve (every interval it computes is the same interval) - and 0 on the others; it never reads an interval it did
    not compute (those are NaN inside the oracle)."""
    a = A.make_config(4, nx=128, ny=64, nlambda=3, ncascades=5)
    act = (a.chi.sum(axis=2) > 0).astype(np.uint8)
    assert 0.02 < act.mean() < 0.5
    dense = oracle.solve_atmosphere(a, want_counts=True)
    sparse = oracle.solve_atmosphere(a, active=act, want_counts=True)
    on = act > 0
    assert np.array_equal(sparse["J"][on], dense["J"][on]) and np.array_equal(sparse["Jbar"][on], dense["Jbar"][on])
    assert np.all(sparse["J"][~on] == 0.0) and np.all(np.isfinite(sparse["J"]))
    assert sparse["intervals"][0] == 4 * on.sum() and np.all(sparse["intervals"] <= dense["intervals"])
    assert sparse["segments"].sum() < dense["segments"].sum()
    # with the bilinear fix and inclinations too
    fx = oracle.solve_atmosphere(a, active=act, bilinear_fix=True)["J"]
    assert np.array_equal(fx[on], oracle.solve_atmosphere(a, bilinear_fix=True)["J"][on])
    mu, w = A.gauss_radau(2)
    inc = oracle.solve_inclined(a.chi, a.eta, 5, mu, w, active=act)["J"]
    assert np.array_equal(inc[on], oracle.solve_inclined(a.chi, a.eta, 5, mu, w)["J"][on])


def test_S4_cells_that_are_not_flagged_are_transparent_and_dark(oracle):
    """"non-flagged cells are treated as transparent with no emission": whatever chi, eta hold there."""
    a = A.make_config(0, nx=64, ny=64, nlambda=2, ncascades=5)
    yy, xx = np.mgrid[0:64, 0:64]
    act = (((xx - 20) ** 2 + (yy - 30) ** 2 < 15 ** 2) | ((xx > 50) & (yy < 10))).astype(np.uint8)
    on = act > 0
    zeroed_chi, zeroed_eta = a.chi.copy(), a.eta.copy()
    zeroed_chi[~on] = 0
    zeroed_eta[~on] = 0
    got = oracle.solve(a.chi, a.eta, 5, active=act, I_below=[0.3, 0.1])["J"]
    ref = oracle.solve(zeroed_chi, zeroed_eta, 5, I_below=[0.3, 0.1])["J"]
    assert np.array_equal(got[on], ref[on])
    assert np.max(np.abs(got[on] / oracle.solve(a.chi, a.eta, 5, I_below=[0.3, 0.1])["J"][on] - 1)) > 0.05   # the flag matters
    line = A.line_config2(nx=32, ny=32, nlambda=2, ncascades=4)
    lact = act[:32, :32]
    lz = line.line.copy()
    lz[lact == 0] = 0
    assert np.array_equal(oracle.solve_line(line.line, line.xl, 4, active=lact)["J"][lact > 0],
                          oracle.solve_line(lz, line.xl, 4)["J"][lact > 0])


def test_S5_sparse_window_solve_is_the_sparse_full_solve_restricted(oracle):
    a = A.make_config(4, nx=128, ny=64, nlambda=2, ncascades=5)
    act = (a.chi.sum(axis=2) > 0).astype(np.uint8)
    full = oracle.solve_atmosphere(a, active=act)
    for win in ((0, 8, 0, 8), (60, 75, 20, 41), (120, 128, 56, 64)):
        x0, x1, y0, y1 = win
        w = oracle.solve_atmosphere(a, active=act, window=win)
        assert np.array_equal(w["J"], full["J"][y0:y1, x0:x1]) and np.array_equal(w["Jbar"], full["Jbar"][y0:y1, x0:x1])


# ----------------------------------------------------------------------------- cascade-0 interval length != 1 (eq. 12-13)
# PAPER.md:171-176 (eq. 12-13 with alpha = 2): t_i = c0 (4^i - 1)/3 for ANY cascade-0 interval length c0; PAPER.md:571 runs
# the paper's models with c0 = 1.5 voxels.  Every pin above has c0 = 1, where c0, c0^2, 1/c0 ... are the same number.
C0 = 1.5


def test_C1_cascade0_closed_form_with_interval_one_and_a_half(oracle):
    """P13 with the interval [0, 1.5]: sqrt2/2 in the own cell, 1.5 - sqrt2/2 in the diagonal neighbour (whose far
    corner lies at 3 sqrt2/2 > 1.5), vacuum outside the box."""
    nx, ny = 8, 8
    chi, eta = A.random_field(nx, ny, 1, seed=17)
    out = oracle.solve(chi, eta, 2, c0=C0, dump_cascade=0)
    c64, e64 = chi[..., 0].astype(float), eta[..., 0].astype(float)
    a, b = R2 / 2, C0 - R2 / 2
    for y in range(ny):
        for x in range(nx):
            for q, (sx, sy) in enumerate([(1, 1), (-1, 1), (-1, -1), (1, -1)]):
                xo, yo = x + sx, y + sy
                inside = 0 <= xo < nx and 0 <= yo < ny
                cd, ed = (c64[yo, xo], e64[yo, xo]) if inside else (0.0, 0.0)
                To = np.exp(-c64[y, x] * a)
                I = e64[y, x] / c64[y, x] * (1 - To) + To * (ed / cd * (1 - np.exp(-cd * b)) if inside else 0.0)
                assert np.isclose(out["dump_I"][y, x, q, 0], I, rtol=1e-12)
                assert np.isclose(out["dump_T"][y, x, q, 0], To * np.exp(-cd * b), rtol=1e-12)


def test_C2_hand_derived_2x2_with_cascade_1_starting_outside_the_box(oracle):
    """2 x 2 cells, 2 cascades, c0 = 1.5.  Cascade 1's single probe sits at the grid centre and its rays start at
    t_1 = 1.5 > sqrt2 >= the distance to the box edge in any direction: every cascade-1 interval starts outside, is
    empty, and carries the boundary intensity alone (reading G10).  Cascade 0 covers [0, 1.5]: own cell
    sqrt2/2, then 1.5 - sqrt2/2 of the diagonal neighbour where there is one.  With t_1 = 1 (the c0 = 1 value) or 2.25
    (c0^2) either cascade 1 or cascade 0 would integrate different lengths."""
    chi = np.array([[[0.7], [1.3]], [[0.2], [2.1]]], np.float32)
    eta = chi * np.array([[[1.0], [0.5]], [[2.0], [0.25]]], np.float32)
    Ib, Ia = 0.3, 0.9
    c, e = chi[..., 0].astype(float), eta[..., 0].astype(float)
    a, b = R2 / 2, C0 - R2 / 2
    J = np.zeros((2, 2))
    for y in range(2):
        for x in range(2):
            for q, (sx, sy) in enumerate([(1, 1), (-1, 1), (-1, -1), (1, -1)]):
                xo, yo = x + sx, y + sy
                To = np.exp(-c[y, x] * a)
                I, T = e[y, x] / c[y, x] * (1 - To), To
                if 0 <= xo < 2 and 0 <= yo < 2:
                    Td = np.exp(-c[yo, xo] * b)
                    I, T = I + To * e[yo, xo] / c[yo, xo] * (1 - Td), T * Td
                J[y, x] += 0.25 * (I + T * (Ia if sy > 0 else Ib))   # the 4 children of quadrant q all head the same way in y
    out = oracle.solve(chi, eta, 2, c0=C0, I_below=[Ib], I_above=[Ia])
    assert np.allclose(out["J"][..., 0], J, rtol=1e-13)


def _independent_cascades(chi, eta, ncasc, c0, Ib, Ia):
    """J by an independent brute force over `ncasc` cascades: ray/cell intersections by sorting (tests/refs.py), interval
    ends t_i = c0 (4^i - 1)/3 typed out here, parents from the geometric position of the child among them (A4)."""
    ny, nx = chi.shape[:2]
    c, e = chi[..., 0].astype(np.float64).ravel(), eta[..., 0].astype(np.float64).ravel()
    ends = [c0 * (4.0 ** i - 1.0) / 3.0 for i in range(ncasc)] + [1e9]

    def interp(a_, n):
        u = (a_ + 0.5) / 2.0 - 0.5
        lo = int(np.floor(u))
        cl = lambda q: min(max(q, 0), n - 1)
        return (cl(lo), 1.0 - (u - lo)), (cl(lo + 1), u - lo)

    M_up = None
    for i in range(ncasc - 1, -1, -1):
        s, nd = 2 ** i, 4 ** (i + 1)
        M = np.zeros((ny // s, nx // s, nd))
        for b in range(ny // s):
            for a_ in range(nx // s):
                for k in range(nd):
                    th = 2 * np.pi * (k + 0.5) / nd
                    cells, ds = refs.segments_by_sorting(nx, ny, (a_ + 0.5) * s, (b + 0.5) * s, th, ends[i], ends[i + 1])
                    I, T = refs.integrate(c, e, cells, ds)
                    if M_up is None:
                        U = Ib if np.sin(th) < 0 else Ia
                    else:
                        U = sum(wa * wb * M_up[bq, aq, 4 * k:4 * k + 4].mean()
                                for (bq, wb) in interp(b, ny // (2 * s)) for (aq, wa) in interp(a_, nx // (2 * s)))
                    M[b, a_, k] = I + T * U
        M_up = M
    return M_up.mean(axis=2)


def test_C3_three_cascades_with_interval_one_and_a_half_against_independent_reference(oracle):
    """The twin of A4 with three cascades and c0 = 1.5: intervals [0, 1.5], [1.5, 7.5], [7.5, inf) on 12 x 8 cells, so
    that t_1 and t_2 both lie inside the box and both scale with c0.  The same reference at c0 = 1
    reproduces the oracle too, and the two differ by far more than the tolerance."""
    nx, ny = 12, 8
    rng = np.random.default_rng(31)
    chi = rng.uniform(0.05, 0.6, (ny, nx, 1)).astype(np.float32)
    eta = (chi * rng.uniform(0.2, 2.0, (ny, nx, 1))).astype(np.float32)
    Ib, Ia = 0.4, 0.1
    got = {c0: oracle.solve(chi, eta, 3, c0=c0, I_below=[Ib], I_above=[Ia])["J"][..., 0] for c0 in (1.0, C0)}
    for c0 in (1.0, C0):
        assert np.allclose(got[c0], _independent_cascades(chi, eta, 3, c0, Ib, Ia), rtol=1e-10)
    assert np.max(np.abs(got[C0] / got[1.0] - 1)) > 1e-3
