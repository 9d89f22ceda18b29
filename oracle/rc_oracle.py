"""ctypes wrapper around oracle/rc_oracle.c (the fp64 CPU oracle).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "rc_oracle.c"
_SO = _HERE / "librc_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """gcc -O2 -fopenmp; no -ffast-math (the oracle's arithmetic is exactly what the source says)."""
    if force or not _SO.exists() or _SO.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _SO.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared",
                               "-o", str(tmp), str(_SRC), "-lm"])
        os.replace(tmp, _SO)
    return _SO


class Counts(C.Structure):
    _fields_ = [("intervals", C.c_int64 * 16), ("segments", C.c_int64 * 16)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.rc_oracle_ray_segments.restype = C.c_int
        _lib.rc_oracle_ray_segments.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                                C.c_int, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        _lib.rc_oracle_interval.restype = C.c_int
        _lib.rc_oracle_interval.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int,
                                            C.c_double, C.c_double, C.c_double, C.c_int, C.c_double,
                                            C.c_double, C.c_int, C.c_void_p, C.c_void_p]
        _lib.rc_oracle_merge.restype = None
        _lib.rc_oracle_merge.argtypes = [C.c_double] * 4 + [C.c_void_p, C.c_void_p]
        _lib.rc_oracle_solve.restype = C.c_int
        _lib.rc_oracle_solve.argtypes = ([C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int,
                                          C.c_double, C.c_void_p, C.c_void_p, C.c_void_p] +
                                         [C.c_int] * 4 + [C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                                          C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                                          C.c_void_p, C.c_void_p])
        _lib.rc_oracle_solve_scaled.restype = C.c_int
        _lib.rc_oracle_solve_scaled.argtypes = _lib.rc_oracle_solve.argtypes + [C.c_double]
        _lib.rc_oracle_solve_line.restype = C.c_int
        _lib.rc_oracle_solve_line.argtypes = ([C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double,
                                               C.c_void_p, C.c_void_p, C.c_void_p] + [C.c_int] * 4 +
                                              [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_double])
        _lib.rc_oracle_solve_active.restype = C.c_int
        _lib.rc_oracle_solve_active.argtypes = ([C.c_void_p] * 4 + [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double,
                                                 C.c_void_p, C.c_void_p, C.c_void_p] + [C.c_int] * 4 +
                                                [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_double, C.c_void_p])
        _lib.rc_oracle_solve_line_dump.restype = C.c_int
        _lib.rc_oracle_solve_line_dump.argtypes = ([C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double,
                                                    C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int,
                                                    C.c_int, C.c_int] + [C.c_void_p] * 4 + [C.c_double])
        _lib.rc_oracle_num_threads.restype = C.c_int
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().rc_oracle_num_threads())


def ray_segments(nx, ny, px, py, theta=0.0, diag_q=-1, ta=0.0, tb=np.inf):
    cells = np.empty(nx + ny + 4, np.int32)
    ds = np.empty(nx + ny + 4, np.float64)
    n = lib().rc_oracle_ray_segments(nx, ny, px, py, theta, diag_q, ta, tb, _ptr(cells), _ptr(ds))
    return cells[:n].copy(), ds[:n].copy()


def interval(chi, eta, px, py, theta=0.0, diag_q=-1, ta=0.0, tb=np.inf, order=0):
    chi, eta = _f32(chi), _f32(eta)
    ny, nx, L = chi.shape
    I = np.empty(L)
    T = np.empty(L)
    lib().rc_oracle_interval(_ptr(chi), _ptr(eta), nx, ny, L, px, py, theta, diag_q, ta, tb, order,
                             _ptr(I), _ptr(T))
    return I, T


def merge(I_near, tau_near, I_far, tau_far):
    a = C.c_double()
    b = C.c_double()
    lib().rc_oracle_merge(I_near, tau_near, I_far, tau_far, C.byref(a), C.byref(b))
    return a.value, b.value


def _active_u8(active, ny, nx):
    a = np.ascontiguousarray(np.asarray(active) != 0, dtype=np.uint8)
    assert a.shape == (ny, nx), f"active mask must be [ny][nx] = {(ny, nx)}, got {a.shape}"
    return a


def solve(chi, eta, ncascades, c0=1.0, I_below=None, I_above=None, weights=None, window=None,
          nthreads=0, order=0, dump_cascade=-1, want_counts=False, path_scale=1.0, bilinear_fix=False, active=None):
    """J [wy][wx][L] (float64) for the cascade-0 cell window (x0, x1, y0, y1) (default: whole grid).

    Returns a dict: J, Jbar, and if asked counts / dump_{I,T,M,win} of one cascade."""
    chi, eta = _f32(chi), _f32(eta)
    ny, nx, L = chi.shape
    assert eta.shape == chi.shape
    x0, x1, y0, y1 = (0, nx, 0, ny) if window is None else window
    J = np.empty((y1 - y0, x1 - x0, L))
    Jbar = np.empty((y1 - y0, x1 - x0))
    Ib = None if I_below is None else _f32(I_below)
    Ia = None if I_above is None else _f32(I_above)
    w = None if weights is None else _f32(weights)
    cnt = Counts()
    dI = dT = dM = None
    win = np.zeros(4, np.int32)
    if dump_cascade >= 0:
        # upper bound on the window of that cascade: the whole lattice
        s = 1 << dump_cascade
        N = 4 ** (dump_cascade + 1)
        shape = (ny // s, nx // s, N, L)
        dI, dT, dM = np.zeros(shape), np.zeros(shape), np.zeros(shape)
        assert window is None, "dump only with the full window (dense layout)"
    order = int(order) | (2 if bilinear_fix else 0)  # bit 1: the bilinear fix
    if active is not None:
        # sparse solve: intervals only for the flagged probes, non-flagged cells transparent
        assert dump_cascade < 0
        act = _active_u8(active, ny, nx)
        rc = lib().rc_oracle_solve_active(_ptr(chi), _ptr(eta), None, None, nx, ny, L, ncascades, c0, _ptr(Ib), _ptr(Ia),
                                          _ptr(w), x0, x1, y0, y1, _ptr(J), _ptr(Jbar), nthreads, order, C.byref(cnt),
                                          float(path_scale), _ptr(act))
        if rc != 0:
            raise ValueError(f"rc_oracle_solve_active failed: {rc}")
        out = {"J": J, "Jbar": Jbar}
        if want_counts:
            out["intervals"] = np.array(cnt.intervals[:ncascades])
            out["segments"] = np.array(cnt.segments[:ncascades])
        return out
    rc = lib().rc_oracle_solve_scaled(_ptr(chi), _ptr(eta), nx, ny, L, ncascades, c0, _ptr(Ib), _ptr(Ia),
                                      _ptr(w), x0, x1, y0, y1, _ptr(J), _ptr(Jbar), nthreads, order,
                                      dump_cascade, _ptr(dI), _ptr(dT), _ptr(dM), _ptr(win), C.byref(cnt),
                                      float(path_scale))
    if rc != 0:
        raise ValueError(f"rc_oracle_solve failed: {rc}")
    out = {"J": J, "Jbar": Jbar}
    if want_counts:
        out["intervals"] = np.array(cnt.intervals[:ncascades])
        out["segments"] = np.array(cnt.segments[:ncascades])
    if dump_cascade >= 0:
        out.update(dump_I=dI, dump_T=dT, dump_M=dM, dump_win=win)
    return out


def solve_inclined(chi, eta, ncascades, mu, w_mu, **kw):
    """2.5D solve: the model is homogeneous along the axis perpendicular
    to the grid; every flatland ray is replaced by len(mu) rays with the same projection and direction
    cosine mu[m] to that axis.  Such a ray crosses the same cells with path lengths ds / sqrt(1 - mu^2), so
    each inclination is the flatland solve with that path scale, and J = sum_m w_mu[m] J_m (the quadrature
    over one hemisphere, weights summing to 1; the other hemisphere is its mirror image).  Written out as
    exactly that: one plain solve per inclination, summed in order."""
    mu = np.asarray(mu, np.float64)
    w_mu = np.asarray(w_mu, np.float64)
    assert mu.shape == w_mu.shape and mu.ndim == 1 and np.all(mu >= 0.0) and np.all(mu < 1.0)
    out = None
    # boundary intensities may be given per inclination, [len(mu)][L] (a table over inclination
    # and wavelength): inclination m then sees row m
    Ib, Ia = kw.pop("I_below", None), kw.pop("I_above", None)
    for m in range(len(mu)):
        bm = None if Ib is None else (np.asarray(Ib)[m] if np.ndim(Ib) == 2 else Ib)
        am = None if Ia is None else (np.asarray(Ia)[m] if np.ndim(Ia) == 2 else Ia)
        o = solve(chi, eta, ncascades, path_scale=1.0 / np.sqrt(1.0 - mu[m] * mu[m]), I_below=bm, I_above=am, **kw)
        if out is None:
            out = {"J": w_mu[m] * o["J"], "Jbar": w_mu[m] * o["Jbar"]}
            for key in ("intervals", "segments"):
                if key in o:
                    out[key] = o[key]
        else:
            out["J"] += w_mu[m] * o["J"]
            out["Jbar"] += w_mu[m] * o["Jbar"]
    return out


def solve_line(line, xl, ncascades, c0=1.0, I_below=None, I_above=None, weights=None, window=None,
               nthreads=0, order=0, want_counts=False, mu=None, w_mu=None, path_scale=1.0, bilinear_fix=False, active=None):
    """Velocity-dependent line mode: per cell chi_c, S_c, chi_line, S_line,
    v_x, v_y; opacity and emissivity are evaluated per ray from the projected velocity (rc_oracle.c,
    cell_chi_eta).  line: float32 [ny][nx][6]; xl: [L] Doppler-width offsets.  Returns J, Jbar like solve()."""
    if mu is not None:
        # 2.5D: one plain solve per inclination (path 1/sqrt(1-mu^2), in-plane velocity projection sqrt(1-mu^2)),
        # summed with the quadrature weights, exactly as solve_inclined does for the GivenFs mode
        out = None
        for m in range(len(mu)):
            bm = None if I_below is None else (np.asarray(I_below)[m] if np.ndim(I_below) == 2 else I_below)
            am = None if I_above is None else (np.asarray(I_above)[m] if np.ndim(I_above) == 2 else I_above)
            o = solve_line(line, xl, ncascades, c0, bm, am, weights, window, nthreads, order, want_counts,
                           path_scale=1.0 / np.sqrt(1.0 - float(mu[m]) ** 2), bilinear_fix=bilinear_fix, active=active)
            if out is None:
                out = dict(o)
                out["J"] = w_mu[m] * o["J"]
                out["Jbar"] = w_mu[m] * o["Jbar"]
            else:
                out["J"] += w_mu[m] * o["J"]
                out["Jbar"] += w_mu[m] * o["Jbar"]
        return out
    line = _f32(line)
    xl = np.ascontiguousarray(xl, dtype=np.float64)
    ny, nx, six = line.shape
    assert six == 6
    L = xl.size
    x0, x1, y0, y1 = (0, nx, 0, ny) if window is None else window
    J = np.empty((y1 - y0, x1 - x0, L))
    Jbar = np.empty((y1 - y0, x1 - x0))
    Ib = None if I_below is None else _f32(I_below)
    Ia = None if I_above is None else _f32(I_above)
    w = None if weights is None else _f32(weights)
    cnt = Counts()
    order = int(order) | (2 if bilinear_fix else 0)
    if active is not None:
        act = _active_u8(active, ny, nx)
        rc = lib().rc_oracle_solve_active(None, None, _ptr(line), _ptr(xl), nx, ny, L, ncascades, c0, _ptr(Ib), _ptr(Ia),
                                          _ptr(w), x0, x1, y0, y1, _ptr(J), _ptr(Jbar), nthreads, order, C.byref(cnt),
                                          float(path_scale), _ptr(act))
    else:
        rc = lib().rc_oracle_solve_line(_ptr(line), _ptr(xl), nx, ny, L, ncascades, c0, _ptr(Ib), _ptr(Ia), _ptr(w),
                                        x0, x1, y0, y1, _ptr(J), _ptr(Jbar), nthreads, order, C.byref(cnt),
                                        float(path_scale))
    if rc != 0:
        raise ValueError(f"rc_oracle_solve_line failed: {rc}")
    out = {"J": J, "Jbar": Jbar}
    if want_counts:
        out["intervals"] = np.array(cnt.intervals[:ncascades])
        out["segments"] = np.array(cnt.segments[:ncascades])
    return out


def line_intervals(line, xl, ncascades, cascade, c0=1.0, path_scale=1.0):
    """Line mode: the intervals [I, T] of one cascade before merging (dump_I, dump_T: [npy][npx][N][L]) and after
    (dump_M), through exactly the code of solve_line (rc_oracle_solve_line_dump): for the pins."""
    line = _f32(line)
    xl = np.ascontiguousarray(xl, dtype=np.float64)
    ny, nx, _ = line.shape
    L = xl.size
    s = 1 << cascade
    shape = (ny // s, nx // s, 4 ** (cascade + 1), L)
    dI, dT, dM = np.zeros(shape), np.zeros(shape), np.zeros(shape)
    win = np.zeros(4, np.int32)
    J = np.empty((ny, nx, L))
    rc = lib().rc_oracle_solve_line_dump(_ptr(line), _ptr(xl), nx, ny, L, ncascades, c0, None, None, None, _ptr(J), None,
                                         0, 0, cascade, _ptr(dI), _ptr(dT), _ptr(dM), _ptr(win), float(path_scale))
    if rc != 0:
        raise ValueError(f"rc_oracle_solve_line_dump failed: {rc}")
    return {"J": J, "dump_I": dI, "dump_T": dT, "dump_M": dM}


def alo(chi=None, line=None, xl=None, mu=None, w_mu=None):
    """Diagonal approximate lambda operator of cascade 0 (eq. 17): Lambda*(k) = exp(-tau),
    tau = chi ds "from the centre to the edge of cell k along direction w".  Cascade 0's directions are the four
    diagonals: ds = sqrt(2)/2 in the plane, divided by sin(inclination) for an inclined ray.  Returned: the mean
    over the 4 directions, summed over the inclinations with their weights, [ny][nx][L] float64.  GivenFs mode:
    chi [ny][nx][L]; line mode: the opacity seen along each diagonal (cell_chi_eta's formula, written out)."""
    mu = np.zeros(1) if mu is None else np.asarray(mu, np.float64)
    w_mu = np.ones(1) if w_mu is None else np.asarray(w_mu, np.float64)
    out = 0.0
    for m in range(len(mu)):
        si = np.sqrt(1.0 - mu[m] ** 2)
        ds = np.sqrt(2.0) / 2.0 / si
        if line is None:
            out = out + w_mu[m] * np.exp(-np.asarray(chi, np.float32).astype(np.float64) * ds)
        else:
            f = np.asarray(line, np.float32).astype(np.float64)
            x = np.asarray(xl, np.float64)
            acc = 0.0
            for k in range(4):
                th = 2.0 * np.pi * (k + 0.5) / 4.0
                a = x[None, None, :] + si * (f[..., 4] * np.cos(th) + f[..., 5] * np.sin(th))[..., None]
                c = f[..., 0:1] + f[..., 2:3] * np.exp(-a * a) / np.sqrt(np.pi)
                acc = acc + np.exp(-c * ds) / 4.0
            out = out + w_mu[m] * acc
    return out


def solve_atmosphere(atm, **kw):
    """Convenience: oracle solve of a paper_2408_14425_b200.atmospheres.Atmosphere-like object."""
    if getattr(atm, "bilinear_fix", False):
        kw.setdefault("bilinear_fix", True)
    if getattr(atm, "active", None) is not None:
        kw.setdefault("active", atm.active)
    if getattr(atm, "line", None) is not None:
        return solve_line(atm.line, atm.xl, atm.ncascades, c0=atm.c0_interval, I_below=atm.I_below,
                          I_above=atm.I_above, weights=atm.weights, mu=getattr(atm, "mu", None),
                          w_mu=getattr(atm, "w_mu", None), **kw)
    if getattr(atm, "mu", None) is not None:
        return solve_inclined(atm.chi, atm.eta, atm.ncascades, atm.mu, atm.w_mu, c0=atm.c0_interval,
                              I_below=atm.I_below, I_above=atm.I_above, weights=atm.weights, **kw)
    return solve(atm.chi, atm.eta, atm.ncascades, c0=atm.c0_interval, I_below=atm.I_below,
                 I_above=atm.I_above, weights=atm.weights, **kw)
