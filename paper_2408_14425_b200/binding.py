"""Thin ctypes binding over librc.so — same names as include/rc.h, argument marshalling only.

Every step of the path (ray march, boundary, interpolate + merge, J) runs in the CUDA kernels
behind the C ABI; PyTorch is used for device memory and streams.  There is no CPU fallback:
`load()` raises if the library cannot be loaded.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from . import build as _build

RC_OK = 0
RC_ACCUM_J, RC_VALIDATE, RC_NO_EARLY_EXIT, RC_BILINEAR_FIX = 1, 2, 4, 8
RC_MAX_CASCADES = 12
ERRORS = {-1: "RC_ERR_NULL_ARG", -2: "RC_ERR_BAD_SHAPE", -3: "RC_ERR_NO_DEVICE", -4: "RC_ERR_NO_WORKSPACE",
          -5: "RC_ERR_BAD_VALUE", -6: "RC_ERR_CUDA", -7: "RC_ERR_NO_ATMOSPHERE"}


class rc_config(C.Structure):
    _fields_ = [("ncascades", C.c_int), ("c0_interval", C.c_float), ("device", C.c_int),
                ("lambda_batch", C.c_int), ("flags", C.c_int)]


class rc_stats(C.Structure):
    _fields_ = [("ncascades", C.c_int), ("lambda_batch", C.c_int), ("kernel_launches", C.c_int),
                ("solves_timed", C.c_int), ("ms_pack", C.c_float * RC_MAX_CASCADES),
                ("ms_march", C.c_float * RC_MAX_CASCADES), ("ms_total", C.c_float),
                ("rays", C.c_int64 * RC_MAX_CASCADES), ("table_steps", C.c_int64 * RC_MAX_CASCADES),
                ("workspace_bytes", C.c_size_t), ("empty_cells", C.c_int64), ("sparse_march", C.c_int),
                ("active_cells", C.c_int64), ("probes_flagged", C.c_int64 * RC_MAX_CASCADES),
                ("sparse_lists", C.c_int), ("sparse_list_bytes", C.c_int64)]


class rc_plan_info(C.Structure):
    _fields_ = [("workspace_bytes", C.c_size_t), ("lambda_batch", C.c_int), ("channels", C.c_int), ("nbatches", C.c_int),
                ("nbands", C.c_int), ("band_axis", C.c_int), ("cascade_empty", C.c_int * RC_MAX_CASCADES),
                ("cascade_banded", C.c_int * RC_MAX_CASCADES), ("patch_w", C.c_int * RC_MAX_CASCADES),
                ("cascade_sorted", C.c_int * RC_MAX_CASCADES), ("lane_utilisation", C.c_float * RC_MAX_CASCADES),
                ("table_steps", C.c_int64 * RC_MAX_CASCADES)]


def plan_query(ncascades, nx, ny, nlambda, ninclinations=1, line_mode=False, c0_interval=1.0, lambda_batch=0, flags=0):
    """Host-only: the launch plan for a problem (no device needed)."""
    cfg = rc_config(int(ncascades), float(c0_interval), 0, int(lambda_batch), int(flags))
    info = rc_plan_info()
    rc = load().rc_plan_query(C.byref(cfg), int(ninclinations), int(bool(line_mode)), int(nx), int(ny), int(nlambda), C.byref(info))
    if rc != RC_OK:
        raise RcError(rc, "rc_plan_query failed")
    return info


# every symbol include/rc.h declares: name -> (restype, argtypes)
SYMBOLS = {
    "rc_plan_query": (C.c_int, [C.POINTER(rc_config), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(rc_plan_info)]),
    "rc_create": (C.c_int, [C.POINTER(C.c_void_p), C.POINTER(rc_config)]),
    "rc_workspace_bytes": (C.c_size_t, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]),
    "rc_set_workspace": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "rc_set_stream": (C.c_int, [C.c_void_p, C.c_void_p]),
    "rc_set_tuning": (C.c_int, [C.c_void_p, C.c_char_p, C.c_double]),
    "rc_set_atmosphere": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int]),
    "rc_set_line_atmosphere": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int]),
    "rc_set_active_cells": (C.c_int, [C.c_void_p, C.c_void_p]),
    "rc_analyse_atmosphere": (C.c_int, [C.c_void_p]),
    "rc_set_sparse_workspace": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "rc_set_boundary": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "rc_set_boundary_inclined": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "rc_set_lambda_weights": (C.c_int, [C.c_void_p, C.c_void_p]),
    "rc_set_inclinations": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]),
    "rc_solve_J": (C.c_int, [C.c_void_p, C.c_void_p]),
    "rc_compute_alo": (C.c_int, [C.c_void_p, C.c_void_p]),
    "rc_solve_J_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]),
    "rc_solve_J_line_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_void_p]),
    "rc_count_walked": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "rc_set_timing": (C.c_int, [C.c_void_p, C.c_int]),
    "rc_get_stats": (C.c_int, [C.c_void_p, C.POINTER(rc_stats)]),
    "rc_count_segments": (C.c_int, [C.c_void_p, C.c_void_p]),
    "rc_probe_gather_bandwidth": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_double)]),
    "rc_probe_bulk_copy_bandwidth": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_double)]),
    "rc_count_empty_cells_static": (C.c_int, [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p,
                                              C.c_void_p, C.c_char_p, C.c_size_t]),
    "rc_last_error": (C.c_char_p, [C.c_void_p]),
    "rc_version": (C.c_char_p, []),
    "rc_destroy": (C.c_int, [C.c_void_p]),
}

_lib = None


def library_path() -> Path:
    return _build.LIB


def load(build_if_missing: bool = True):
    """dlopen librc.so (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is None:
        if build_if_missing:
            try:
                _build.build()
            except Exception:
                if not _build.LIB.exists() or _build.stale():
                    raise  # never run a library older than its sources
        if not _build.LIB.exists():
            raise RuntimeError(f"{_build.LIB} is missing: build it with paper_2408_14425_b200.build.build(); "
                               "there is no CPU fallback")
        lib = C.CDLL(str(_build.LIB))
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


class RcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


def _host_f32(a, n):
    if a is None:
        return None, None
    arr = np.ascontiguousarray(a, dtype=np.float32)
    assert arr.size == n, f"expected {n} values, got {arr.size}"
    return arr, arr.ctypes.data_as(C.c_void_p)


class RadianceCascades:
    """One rc_ctx plus the torch-owned workspace it borrows.  Methods mirror the C entry points."""

    def __init__(self, ncascades, c0_interval=1.0, device=0, lambda_batch=0, flags=0):
        self.lib = load()
        self.cfg = rc_config(int(ncascades), float(c0_interval), int(device), int(lambda_batch), int(flags))
        self.handle = C.c_void_p()
        rc = self.lib.rc_create(C.byref(self.handle), C.byref(self.cfg))
        if rc != RC_OK:
            self.handle = C.c_void_p()
            raise RcError(rc, "rc_create failed")
        self.device = int(device)
        self.flags = int(flags)
        self._ws = None
        self._sws = None
        self._keep = ()
        self.shape = None

    def _check(self, rc):
        if rc != RC_OK:
            raise RcError(rc, self.lib.rc_last_error(self.handle).decode())

    def workspace_bytes(self, nx, ny, nlambda, host_io=False) -> int:
        return int(self.lib.rc_workspace_bytes(self.handle, nx, ny, nlambda, int(host_io)))

    def set_workspace(self, tensor):
        self._ws = tensor
        self._check(self.lib.rc_set_workspace(self.handle, C.c_void_p(tensor.data_ptr()), tensor.numel() * tensor.element_size()))

    def ensure_workspace(self, nx, ny, nlambda, host_io=False):
        import torch
        need = self.workspace_bytes(nx, ny, nlambda, host_io)
        if need == 0:
            raise RcError(-2, f"bad shape {nx}x{ny}x{nlambda} for {self.cfg.ncascades} cascades")
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self.set_workspace(torch.empty(need, dtype=torch.uint8, device=f"cuda:{self.device}"))

    def set_stream(self, stream=None):
        import torch
        s = torch.cuda.current_stream(self.device) if stream is None else stream
        self._check(self.lib.rc_set_stream(self.handle, C.c_void_p(s.cuda_stream)))

    def set_tuning(self, **knobs):
        """Launch knobs (rc_set_tuning): e.g. set_tuning(march_variant=0, bands=3).  Before set_atmosphere."""
        for k, v in knobs.items():
            self._check(self.lib.rc_set_tuning(self.handle, k.encode(), float(v)))

    def set_atmosphere(self, chi, eta):
        """chi, eta: CUDA float32 tensors [ny][nx][nlambda] (borrowed until replaced)."""
        assert chi.is_cuda and eta.is_cuda and chi.dtype == eta.dtype and chi.shape == eta.shape
        assert chi.is_contiguous() and eta.is_contiguous() and chi.dim() == 3
        ny, nx, L = chi.shape
        self.ensure_workspace(nx, ny, L)
        self.set_stream()
        self._check(self.lib.rc_set_atmosphere(self.handle, C.c_void_p(chi.data_ptr()), C.c_void_p(eta.data_ptr()), nx, ny, L))
        self._keep = (chi, eta)
        self.shape = (ny, nx, L)

    def set_line_atmosphere(self, line, xl):
        """line: CUDA float32 tensor [ny][nx][6] (borrowed); xl: host array [nlambda] in Doppler widths."""
        import numpy as np
        assert line.is_cuda and line.is_contiguous() and line.dim() == 3 and line.shape[2] == 6
        ny, nx, _ = line.shape
        x = np.ascontiguousarray(xl, dtype=np.float32)
        self.ensure_workspace(nx, ny, int(x.size))
        self.set_stream()
        self._check(self.lib.rc_set_line_atmosphere(self.handle, C.c_void_p(line.data_ptr()), nx, ny,
                                                    x.ctypes.data_as(C.c_void_p), int(x.size)))
        self._keep = (line,)
        self.shape = (ny, nx, int(x.size))

    def set_active_cells(self, active=None):
        """active: CUDA uint8 tensor [ny][nx] (non-zero = cell of interest; copied by the library) or None = every cell."""
        if active is None:
            self._check(self.lib.rc_set_active_cells(self.handle, None))
            return
        ny, nx, _ = self.shape
        assert active.is_cuda and active.is_contiguous() and active.element_size() == 1 and tuple(active.shape) == (ny, nx)
        self.set_stream()
        self._check(self.lib.rc_set_active_cells(self.handle, C.c_void_p(active.data_ptr())))

    def analyse_atmosphere(self, lists=True):
        """Empty-cell scan + distance field of the current atmosphere (synchronises); see rc_analyse_atmosphere.
        lists: when the atmosphere is sparse, lend the library a second buffer of the size it reports for its hit
        lists (rc_set_sparse_workspace) and analyse again."""
        import torch
        self.set_stream()
        self._check(self.lib.rc_analyse_atmosphere(self.handle))
        st = self.get_stats()
        if lists and not st.sparse_lists and st.sparse_list_bytes > 0:   # (> 0: the atmosphere is sparse)
            if self._sws is None or self._sws.numel() < st.sparse_list_bytes:
                self._sws = None
                self._sws = torch.empty(int(st.sparse_list_bytes * 1.02) + 4096, dtype=torch.uint8, device=f"cuda:{self.device}")
                self._check(self.lib.rc_set_sparse_workspace(self.handle, C.c_void_p(self._sws.data_ptr()), self._sws.numel()))
            self._check(self.lib.rc_analyse_atmosphere(self.handle))
            st = self.get_stats()
        return st

    def set_boundary(self, I_below=None, I_above=None):
        """[nlambda] arrays, or [ninclinations][nlambda] (one value per inclined ray set)."""
        L = self.shape[2]
        two_d = any(x is not None and np.ndim(x) == 2 for x in (I_below, I_above))
        if two_d:
            n = next(np.shape(x)[0] for x in (I_below, I_above) if x is not None and np.ndim(x) == 2)
            a, pa = _host_f32(None if I_below is None else np.broadcast_to(I_below, (n, L)), n * L)
            b, pb = _host_f32(None if I_above is None else np.broadcast_to(I_above, (n, L)), n * L)
            self._check(self.lib.rc_set_boundary_inclined(self.handle, pa, pb))
            return
        a, pa = _host_f32(I_below, L)
        b, pb = _host_f32(I_above, L)
        self._check(self.lib.rc_set_boundary(self.handle, pa, pb))

    def set_lambda_weights(self, w=None):
        a, pa = _host_f32(w, self.shape[2])
        self._check(self.lib.rc_set_lambda_weights(self.handle, pa))

    def set_inclinations(self, mu=None, w=None):
        """2.5D inclination quadrature (before set_atmosphere); mu = None restores flatland."""
        import numpy as np
        if mu is None:
            self._check(self.lib.rc_set_inclinations(self.handle, 1, None, None))
        else:
            m = np.ascontiguousarray(mu, dtype=np.float32)
            ww = np.ascontiguousarray(w, dtype=np.float32)
            assert m.shape == ww.shape and m.ndim == 1
            self._check(self.lib.rc_set_inclinations(self.handle, int(m.size), m.ctypes.data_as(C.c_void_p),
                                                     ww.ctypes.data_as(C.c_void_p)))
        self._ws = None  # the workspace size depends on the number of inclinations

    def solve_J(self, out=None):
        """Enqueue one solve on torch's current stream; returns the output tensor (not synchronised)."""
        import torch
        ny, nx, L = self.shape
        shape = (ny, nx) if self.flags & RC_ACCUM_J else (ny, nx, L)
        if out is None:
            out = torch.empty(shape, dtype=torch.float32, device=f"cuda:{self.device}")
        assert out.is_cuda and out.is_contiguous() and tuple(out.shape) == shape
        self.set_stream()
        self._check(self.lib.rc_solve_J(self.handle, C.c_void_p(out.data_ptr())))
        return out

    def solve_J_host(self, chi_host, eta_host, out_host=None):
        """Host tensors (ideally pinned) in, host tensor out; H2D + solve + D2H, synchronised."""
        import torch
        ny, nx, L = chi_host.shape
        self.ensure_workspace(nx, ny, L, host_io=True)
        self.set_stream()
        shape = (ny, nx) if self.flags & RC_ACCUM_J else (ny, nx, L)
        if out_host is None:
            out_host = torch.empty(shape, dtype=torch.float32, pin_memory=True)
        self._check(self.lib.rc_solve_J_host(self.handle, C.c_void_p(chi_host.data_ptr()), C.c_void_p(eta_host.data_ptr()),
                                             nx, ny, L, C.c_void_p(out_host.data_ptr())))
        self.shape = (ny, nx, L)
        return out_host

    def solve_J_line_host(self, line_host, xl, out_host=None):
        """Line mode, host tensors (ideally pinned) in and out: H2D + solve + D2H through rc_solve_J_line_host."""
        import torch
        ny, nx, _ = line_host.shape
        x = np.ascontiguousarray(xl, dtype=np.float32)
        L = int(x.size)
        self.ensure_workspace(nx, ny, L, host_io=True)
        self.set_stream()
        shape = (ny, nx) if self.flags & RC_ACCUM_J else (ny, nx, L)
        if out_host is None:
            out_host = torch.empty(shape, dtype=torch.float32, pin_memory=True)
        self._check(self.lib.rc_solve_J_line_host(self.handle, C.c_void_p(line_host.data_ptr()), nx, ny,
                                                  x.ctypes.data_as(C.c_void_p), L, C.c_void_p(out_host.data_ptr())))
        self.shape = (ny, nx, L)
        return out_host

    def count_walked(self, out=None):
        """One solve with counters: cell segments actually integrated per cascade and wavelength (rc_count_walked)."""
        import torch
        ny, nx, L = self.shape
        shape = (ny, nx) if self.flags & RC_ACCUM_J else (ny, nx, L)
        if out is None:
            out = torch.empty(shape, dtype=torch.float32, device=f"cuda:{self.device}")
        self.set_stream()
        res = (C.c_int64 * RC_MAX_CASCADES)()
        self._check(self.lib.rc_count_walked(self.handle, C.c_void_p(out.data_ptr()), res))
        return [int(res[i]) for i in range(self.cfg.ncascades)]

    def compute_alo(self):
        """Diagonal ALO of cascade 0 (eq. 17) of the current atmosphere: CUDA tensor [ny][nx][nlambda]."""
        import torch
        out = torch.empty(self.shape, dtype=torch.float32, device=f"cuda:{self.device}")
        self.set_stream()
        self._check(self.lib.rc_compute_alo(self.handle, C.c_void_p(out.data_ptr())))
        return out

    def set_timing(self, nsets=1):
        self._check(self.lib.rc_set_timing(self.handle, int(nsets)))

    def count_segments(self):
        """Per-cascade geometric segment counts (per wavelength) of the current atmosphere's grid."""
        out = (C.c_int64 * RC_MAX_CASCADES)()
        self._check(self.lib.rc_count_segments(self.handle, out))
        return [int(out[i]) for i in range(self.cfg.ncascades)]

    def probe_gather_bandwidth(self, mbytes=64):
        """GB/s of the march's gather pattern alone over the first `mbytes` MB of the workspace."""
        gbs = C.c_double(0.0)
        self._check(self.lib.rc_probe_gather_bandwidth(self.handle, int(mbytes), C.byref(gbs)))
        return float(gbs.value)

    def probe_bulk_copy_bandwidth(self, mbytes=64):
        """GB/s of the same pattern staged through shared memory with TMA bulk copies (the design not taken)."""
        gbs = C.c_double(0.0)
        self._check(self.lib.rc_probe_bulk_copy_bandwidth(self.handle, int(mbytes), C.byref(gbs)))
        return float(gbs.value)

    def get_stats(self) -> rc_stats:
        st = rc_stats()
        self._check(self.lib.rc_get_stats(self.handle, C.byref(st)))
        return st

    def close(self):
        if self.handle:
            self.lib.rc_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


RC_STATIC_MAX_CELLS = 1 << 20


def count_empty_cells_static(chi, eta, active=None, out=None):
    """rc_count_empty_cells_static: the empty-cell count of an atmosphere for callers that cannot allocate device memory
    (a host application's pool owns the GPU, or cudaMalloc is banned in their loop): no context, no workspace, the
    scratch is an array inside librc.so (grids up to RC_STATIC_MAX_CELLS cells; calls must not overlap on the GPU).
    chi, eta: CUDA float32 [ny][nx][nlambda]; active: CUDA uint8 [ny][nx] or None; out: CUDA int64 tensor of one
    element that receives the count (enqueued on torch's current stream, not synchronised).  Only when `out` is left
    out does this wrapper allocate one itself - a convenience for tests, not something the C call does."""
    import torch
    assert chi.is_cuda and eta.is_cuda and chi.dtype == torch.float32 and eta.dtype == torch.float32
    assert chi.is_contiguous() and eta.is_contiguous() and chi.dim() == 3 and chi.shape == eta.shape
    ny, nx, L = chi.shape
    dev = chi.device.index
    if active is not None:
        assert active.is_cuda and active.is_contiguous() and active.element_size() == 1 and tuple(active.shape) == (ny, nx)
    if out is None:
        out = torch.empty(1, dtype=torch.int64, device=chi.device)
    assert out.is_cuda and out.dtype == torch.int64 and out.numel() == 1
    err = C.create_string_buffer(512)
    rc = load().rc_count_empty_cells_static(dev, C.c_void_p(chi.data_ptr()), C.c_void_p(eta.data_ptr()),
                                            None if active is None else C.c_void_p(active.data_ptr()), nx, ny, L,
                                            C.c_void_p(out.data_ptr()), C.c_void_p(torch.cuda.current_stream(dev).cuda_stream),
                                            err, len(err))
    if rc != RC_OK:
        raise RcError(rc, err.value.decode())
    return out


def solve_atmosphere(atm, device=0, lambda_batch=0, flags=0, rc=None, analyse=False, tuning=None):
    """Convenience for tests/bench: upload an `atmospheres.Atmosphere`, solve, return (J tensor, ctx)."""
    import torch
    dev = f"cuda:{device}"
    fl = flags | (RC_ACCUM_J if atm.accumulate else 0) | (RC_BILINEAR_FIX if getattr(atm, "bilinear_fix", False) else 0)
    if rc is None:
        rc = RadianceCascades(atm.ncascades, atm.c0_interval, device, lambda_batch, fl)
    if tuning:
        rc.set_tuning(**tuning)
    if getattr(atm, "line", None) is not None:
        if getattr(atm, "mu", None) is not None:
            rc.set_inclinations(atm.mu, atm.w_mu)
        rc.set_line_atmosphere(torch.from_numpy(atm.line).to(dev), atm.xl)
    else:
        chi = torch.from_numpy(atm.chi).to(dev)
        eta = torch.from_numpy(atm.eta).to(dev)
        if getattr(atm, "mu", None) is not None:
            rc.set_inclinations(atm.mu, atm.w_mu)
        rc.set_atmosphere(chi, eta)
    rc.set_boundary(atm.I_below, atm.I_above)
    rc.set_lambda_weights(atm.weights)
    if getattr(atm, "active", None) is not None:
        rc.set_active_cells(torch.from_numpy(np.ascontiguousarray(atm.active, dtype=np.uint8)).to(dev))
    if analyse:
        rc.analyse_atmosphere()
    J = rc.solve_J()
    torch.cuda.synchronize(device)
    return J, rc
