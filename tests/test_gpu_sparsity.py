"""GPU parity of the sparsity row through the C ABI:

  rc_set_active_cells     cells of interest -> flagged cascade-0 probes -> bilinear parents flagged recursively,
                          intervals only for flagged probes, other cells transparent and dark, J = 0 there
  rc_analyse_atmosphere   free-space acceleration: every lane walks its own ray over the distance field of the
                          occupied cells (bit-identical to the lock-step march)
"""
import dataclasses

import numpy as np
import pytest

from paper_2408_14425_b200 import atmospheres as A

pytestmark = pytest.mark.gpu
TOL = 2e-4


def rel_err(Jg, Jo):
    Jg = np.asarray(Jg, np.float64)
    Jo = np.asarray(Jo, np.float64)
    if Jo.ndim == 2:
        Jg, Jo = Jg[..., None], Jo[..., None]
    worst = 0.0
    for l in range(Jo.shape[-1]):
        o, g = Jo[..., l], Jg[..., l]
        m = o > 1e-6 * o.max()
        if m.any():
            worst = max(worst, float(np.max(np.abs(g[m] - o[m]) / o[m])))
        assert np.all(np.abs(g[~m]) <= 1e-5 * max(o.max(), 1e-300) + 1e-30)
    return worst


def gpu(atm, **kw):
    from paper_2408_14425_b200 import binding
    J, rc = binding.solve_atmosphere(atm, **kw)
    st = rc.get_stats()
    out = J.cpu().numpy()
    rc.close()
    return out, st


def check(atm, oracle, **kw):
    o = oracle.solve_atmosphere(atm)
    Jo = o["Jbar"] if atm.accumulate else o["J"]
    Jg, st = gpu(atm, **kw)
    e = rel_err(Jg, Jo)
    assert e <= TOL, f"{atm.name}: max rel err {e:.3e}"
    if atm.active is not None:
        off = atm.active == 0
        assert np.all(Jg[off] == 0.0)            # J is not computed outside the cells of interest
    return st


# ------------------------------------------------------------------ active cells
@pytest.mark.parametrize("idx,kw,mode", [
    (4, dict(nx=256, ny=128, nlambda=11, ncascades=6), "occupied"),
    (3, dict(nx=128, ny=128, nlambda=8, ncascades=6), "occupied"),
    (3, dict(nx=192, ny=128, nlambda=5, ncascades=6), 0.25),
    (2, dict(nx=128, ny=64, nlambda=9, ncascades=5), 0.25),
    (1, dict(nx=128, ny=128, nlambda=16, ncascades=6), 0.5),
    (0, dict(nx=64, ny=64, nlambda=1, ncascades=5), 0.05),
    (0, dict(nx=32, ny=16, nlambda=3, ncascades=1), 0.3),
])
def test_active_cells_match_the_oracle(oracle, idx, kw, mode):
    """The five recipes with a cells-of-interest flag (where the opacity is; or the densest 5-50 % of the cells, 25 % being
    the paper's production run): J on the flagged cells against the oracle's sparse solve, 0 elsewhere."""
    atm = A.make_config(idx, **kw)
    atm = A.with_active_cells(atm) if mode == "occupied" else A.with_active_cells(atm, mode="fraction", fraction=mode)
    st = check(atm, oracle)
    assert st.active_cells == int((atm.active != 0).sum())
    # flagged probes per cascade = the oracle's interval counts / directions
    ref = oracle.solve_atmosphere(atm, want_counts=True)["intervals"]
    assert [int(st.probes_flagged[i]) for i in range(atm.ncascades)] == [int(n) // 4 ** (i + 1) for i, n in enumerate(ref)]


def test_active_cells_in_every_mode(oracle):
    """With the bilinear fix (lanes are parity classes: 4 patch lists), inclinations, the moving line, Jbar, banded launches,
    child-per-warp and every lane patch shape."""
    base = A.with_active_cells(A.make_config(3, nx=128, ny=128, nlambda=6, ncascades=6), mode="fraction", fraction=0.2)
    check(dataclasses.replace(base, bilinear_fix=True), oracle)
    check(A.with_inclinations(base, 4), oracle)
    line = A.with_active_cells(A.line_config2(nx=96, ny=64, nlambda=5, ncascades=5), mode="fraction", fraction=0.3)
    check(line, oracle)
    check(A.with_inclinations(dataclasses.replace(line, bilinear_fix=True), 2), oracle)
    c4 = A.with_active_cells(A.make_config(4, nx=256, ny=64, nlambda=9, ncascades=5))
    assert c4.accumulate
    check(c4, oracle)
    ref, _ = gpu(base)
    for knobs in (dict(bands=3), dict(cpw_from=0), dict(patch_log2=2), dict(patch_log2=5, march_variant=0), dict(cpw_from=-1, bands=2)):
        got, _ = gpu(base, tuning=knobs)
        assert np.array_equal(ref, got), knobs


def test_all_cells_active_is_the_dense_solve_bit_for_bit():
    atm = A.make_config(2, nx=128, ny=64, nlambda=11, ncascades=5)
    dense, st0 = gpu(atm)
    ones, st1 = gpu(dataclasses.replace(atm, active=np.ones((64, 128), np.uint8)))
    assert np.array_equal(dense, ones)
    assert st0.active_cells == -1 and st1.active_cells == 64 * 128


def test_unflagged_cells_are_transparent_and_the_flag_can_be_dropped(oracle):
    import torch
    from paper_2408_14425_b200 import binding
    atm = A.make_config(0, nx=64, ny=64, nlambda=2, ncascades=5)
    yy, xx = np.mgrid[0:64, 0:64]
    act = (((xx - 20) ** 2 + (yy - 30) ** 2 < 15 ** 2) | ((xx > 50) & (yy < 10))).astype(np.uint8)
    flagged = dataclasses.replace(atm, active=act)
    check(flagged, oracle)
    J, rc = binding.solve_atmosphere(flagged)
    dense_ref, _ = gpu(atm)
    rc.set_active_cells(None)                       # back to every cell
    J2 = rc.solve_J()
    torch.cuda.synchronize()
    assert np.array_equal(J2.cpu().numpy(), dense_ref)
    assert not np.array_equal(J.cpu().numpy()[act > 0], dense_ref[act > 0])
    # a new atmosphere of the same shape keeps the flags
    rc.set_active_cells(torch.from_numpy(act).cuda())
    other = A.make_config(0, nx=64, ny=64, nlambda=2, ncascades=5, seed=5)
    chi, eta = torch.from_numpy(other.chi).cuda(), torch.from_numpy(other.eta).cuda()
    rc.set_atmosphere(chi, eta)
    J3 = rc.solve_J().cpu().numpy()
    Jo = oracle.solve_atmosphere(dataclasses.replace(other, active=act))["J"]
    assert rel_err(J3, Jo) <= TOL
    rc.close()


# ------------------------------------------------------------------ free-space acceleration
@pytest.mark.parametrize("kw", [
    dict(nx=256, ny=128, nlambda=11, ncascades=6),
    dict(nx=512, ny=128, nlambda=8, ncascades=7),
    dict(nx=96, ny=160, nlambda=3, ncascades=5),
    dict(nx=64, ny=64, nlambda=1, ncascades=1),
])
def test_distance_field_march_is_bit_identical(oracle, kw):
    """Config 4's recipe (> 90 % of the cells exactly empty): after rc_analyse_atmosphere every lane walks its own ray
    and jumps over empty space on the distance field.  Empty cells change no bit of (tau, T, I), so J must equal the
    lock-step march bit for bit - any occupied cell a jump missed would show - and match the oracle."""
    atm = A.make_config(4, **kw)
    dense, st0 = gpu(atm)
    walk, st1 = gpu(atm, analyse=True)
    assert st0.sparse_march == 0 and st1.sparse_march == 1
    assert st1.empty_cells > 0.8 * atm.nx * atm.ny
    assert np.array_equal(dense, walk)
    for mode in (0, 1, 2, 3):                    # launch variants of the walk (rc_set_tuning "sparse_mode")
        got, st = gpu(atm, analyse=True, tuning=dict(sparse_mode=mode, lists=0))
        assert st.sparse_march == 1 and st.sparse_lists == 0 and np.array_equal(dense, got), mode
    check(atm, oracle, analyse=True)
    # per-wavelength J too (config 4 accumulates Jbar), with a boundary intensity so that the top cascade matters
    pl = dataclasses.replace(atm, accumulate=False)
    pl.I_below[:] = 0.7
    a, _ = gpu(pl)
    b, _ = gpu(pl, analyse=True)
    assert np.array_equal(a, b)


@pytest.mark.parametrize("nlambda", [3, 16, 40, 43])
def test_march_over_hit_lists_is_bit_identical(oracle, nlambda):
    """rc_set_sparse_workspace: the occupied steps of every ray are found once per analysed atmosphere (they depend on
    the geometry and the occupancy alone) and the march only gathers and integrates them - the same cells in the same order
    as the distance-field walk and the lock-step march, so J agrees bit for bit; 8 wavelength batches per warp (cell-major
    packed arrays) from 5 batches on, one otherwise; ragged last batch; without the second buffer the walk stays in use."""
    import torch
    from paper_2408_14425_b200 import binding
    atm = dataclasses.replace(A.make_config(4, nx=256, ny=128, nlambda=nlambda, ncascades=6), accumulate=nlambda == 40)
    dense, _ = gpu(atm)
    walk, st0 = gpu(atm, analyse=True, tuning=dict(lists=0))
    lists, st1 = gpu(atm, analyse=True)
    assert st0.sparse_march == 1 and st0.sparse_lists == 0
    assert st1.sparse_march == 1 and st1.sparse_lists == 1 and st1.sparse_list_bytes > 0
    assert np.array_equal(dense, walk) and np.array_equal(dense, lists)
    flagged = A.with_active_cells(atm)
    a, _ = gpu(flagged)
    b, st = gpu(flagged, analyse=True)
    assert st.sparse_lists == 1 and np.array_equal(a, b)
    # through the raw ABI without a second buffer: the size is reported, the walk is used
    J, rc = binding.solve_atmosphere(atm)
    assert rc.lib.rc_analyse_atmosphere(rc.handle) == 0
    st = rc.get_stats()
    assert st.sparse_march == 1 and st.sparse_lists == 0 and st.sparse_list_bytes == st1.sparse_list_bytes
    assert np.array_equal(rc.solve_J().cpu().numpy(), dense)
    small = torch.empty(1 << 16, dtype=torch.uint8, device="cuda")       # too small: still the walk
    assert rc.lib.rc_set_sparse_workspace(rc.handle, small.data_ptr(), small.numel()) == 0
    assert rc.lib.rc_analyse_atmosphere(rc.handle) == 0 and rc.get_stats().sparse_lists == 0
    assert np.array_equal(rc.solve_J().cpu().numpy(), dense)
    rc.close()
    if nlambda == 3:
        check(atm, oracle, analyse=True)


def test_distance_field_march_on_dense_and_flagged_atmospheres(oracle):
    """Forced (tuning sparse = 1) where nothing is empty - the distance field is 0 everywhere and every step is walked -
    and combined with active cells (cells that are not flagged count as empty); one wavelength per lane up to eight."""
    dense = A.make_config(2, nx=128, ny=64, nlambda=5, ncascades=5)
    ref, _ = gpu(dense)
    got, st = gpu(dense, analyse=True, tuning=dict(sparse=1))
    assert st.sparse_march == 1 and st.empty_cells == 0 and np.array_equal(ref, got)
    _, st = gpu(dense, analyse=True)
    assert st.sparse_march == 0                       # automatic: a dense atmosphere keeps the lock-step march
    flagged = A.with_active_cells(A.make_config(3, nx=128, ny=128, nlambda=8, ncascades=6), mode="fraction", fraction=0.15)
    ref, _ = gpu(flagged)
    for lb in (0, 1, 2, 4):
        got, st = gpu(flagged, analyse=True, lambda_batch=lb)
        assert st.sparse_march == 1 and np.array_equal(ref, got), lb
    check(flagged, oracle, analyse=True)
    emit = A.emitter_config(nx=128, ny=96, nlambda=3, ncascades=5)      # discs + pure emitters in exact vacuum
    ref, _ = gpu(emit)
    got, st = gpu(emit, analyse=True, tuning=dict(sparse=1))
    assert np.array_equal(ref, got)
    check(emit, oracle, analyse=True, tuning=dict(sparse=1))


@pytest.mark.parametrize("n,nlambda", [(2, 5), (4, 16), (8, 9), (8, 1)])
def test_march_over_hit_lists_with_inclinations(oracle, n, nlambda):
    """2.5D inclinations over hit lists (the distance-field walk has no inclined version: without the second buffer the
    solve stays lock-step): bit-identical to the lock-step march, with flagged probes too, and against the oracle."""
    from paper_2408_14425_b200 import binding
    atm = A.with_inclinations(dataclasses.replace(A.make_config(4, nx=256, ny=64, nlambda=nlambda, ncascades=5), accumulate=nlambda == 9), n)
    ref, st0 = gpu(atm)
    got, st1 = gpu(atm, analyse=True)
    assert st0.sparse_march == 0 and st1.sparse_march == 1 and st1.sparse_lists == 1
    assert np.array_equal(ref, got)
    flagged = A.with_active_cells(atm)
    a, _ = gpu(flagged)
    b, st = gpu(flagged, analyse=True)
    assert st.sparse_lists == 1 and np.array_equal(a, b)
    J, rc = binding.solve_atmosphere(atm)                 # raw analysis without a buffer: stays lock-step
    assert rc.lib.rc_analyse_atmosphere(rc.handle) == 0
    st = rc.get_stats()
    assert st.sparse_march == 0 and st.sparse_list_bytes > 0
    assert np.array_equal(rc.solve_J().cpu().numpy(), ref)
    rc.close()
    if n == 4:
        check(atm, oracle, analyse=True)


@pytest.mark.parametrize("n,nlambda", [(1, 6), (1, 1), (2, 9), (8, 3)])
def test_march_over_hit_lists_with_the_moving_line(oracle, n, nlambda):
    """The paper's production set-up - velocity-dependent line, inclinations, a quarter of the cells flagged
     - over hit lists: bit-identical to the lock-step march of the same flagged atmosphere."""
    line = A.with_active_cells(A.line_config2(nx=128, ny=96, nlambda=nlambda, ncascades=5), mode="fraction", fraction=0.25)
    if n > 1:
        line = A.with_inclinations(line, n)
    ref, st0 = gpu(line)
    got, st1 = gpu(line, analyse=True)
    assert st0.sparse_march == 0 and st1.sparse_march == 1 and st1.sparse_lists == 1
    assert np.array_equal(ref, got)
    if n <= 2:
        check(line, oracle, analyse=True)


def test_hit_lists_are_kept_while_the_occupancy_stands():
    """A new atmosphere with the same occupancy map (other values in the same cells) keeps the hit lists (sparse_lists = 2);
    another map rebuilds them (1); both give the lock-step result bit for bit."""
    import torch
    from paper_2408_14425_b200 import binding
    atm = dataclasses.replace(A.make_config(4, nx=256, ny=128, nlambda=8, ncascades=6), accumulate=False)
    J, rc = binding.solve_atmosphere(atm, analyse=True)
    assert rc.get_stats().sparse_lists == 1
    for scale, seed, want in ((3.0, None, 2), (1.0, 99, 1), (0.5, 99, 2)):
        other = atm if seed is None else dataclasses.replace(A.make_config(4, nx=256, ny=128, nlambda=8, ncascades=6, seed=seed), accumulate=False)
        other = dataclasses.replace(other, chi=(other.chi * scale).astype(np.float32), eta=(other.eta * scale * 0.7).astype(np.float32))
        chi, eta = torch.from_numpy(other.chi).cuda(), torch.from_numpy(other.eta).cuda()
        rc.set_atmosphere(chi, eta)
        st = rc.analyse_atmosphere()
        assert st.sparse_march == 1 and st.sparse_lists == want, (scale, seed, st.sparse_lists)
        got = rc.solve_J().cpu().numpy()
        ref, _ = gpu(other)
        assert np.array_equal(ref, got)
    rc.close()


def test_analysis_belongs_to_one_atmosphere():
    """A new atmosphere switches the distance-field march off until it is analysed again; rc_solve_J_host repeats the
    analysis by itself once the context has used it."""
    import torch
    from paper_2408_14425_b200 import binding
    atm = A.make_config(4, nx=256, ny=64, nlambda=4, ncascades=5)
    rc = binding.RadianceCascades(atm.ncascades, flags=binding.RC_ACCUM_J)
    rc.ensure_workspace(atm.nx, atm.ny, atm.nlambda, host_io=True)   # room for the host path from the start (a new workspace resets weights)
    J, rc = binding.solve_atmosphere(atm, rc=rc, analyse=True)
    assert rc.get_stats().sparse_march == 1
    other = A.make_config(4, nx=256, ny=64, nlambda=4, ncascades=5, seed=99)
    chi, eta = torch.from_numpy(other.chi).cuda(), torch.from_numpy(other.eta).cuda()
    rc.set_atmosphere(chi, eta)
    assert rc.get_stats().sparse_march == 0
    J1 = rc.solve_J().cpu().numpy()
    rc.analyse_atmosphere()
    assert rc.get_stats().sparse_march == 1
    assert np.array_equal(J1, rc.solve_J().cpu().numpy())
    Jh = rc.solve_J_host(torch.from_numpy(other.chi).pin_memory(), torch.from_numpy(other.eta).pin_memory())
    assert rc.get_stats().sparse_march == 1 and np.array_equal(Jh.numpy(), J1)
    rc.close()
