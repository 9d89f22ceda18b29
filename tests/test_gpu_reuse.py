"""One context used again and again (the iteration of PAPER.md:316-342 keeps its context for hundreds of formal
solutions): whatever the library caches between calls - the uploaded wavelengths of the line mode, the captured launch
graph of small grids, the staging layout of the host paths - has to follow every change of shape, mode, workspace and
tuning.  Each case compares the reused context with a fresh one, bit for bit.
"""
import numpy as np
import pytest

from paper_2408_14425_b200 import atmospheres as A

pytestmark = pytest.mark.gpu


def fresh(atm, **kw):
    import torch
    from paper_2408_14425_b200 import binding
    J, rc = binding.solve_atmosphere(atm, **kw)
    out = J.clone()
    rc.close()
    torch.cuda.synchronize()
    return out


def test_line_wavelengths_follow_the_plan_across_shapes_modes_and_workspaces():
    """Same x_lambda, but the place it lives in the workspace moves: a second grid size, a GivenFs atmosphere in
    between (its packed arrays cover those bytes), a larger workspace."""
    import torch
    from paper_2408_14425_b200 import binding
    small = A.line_config2(nx=64, ny=64, nlambda=8, ncascades=5)
    large = A.line_config2(nx=128, ny=96, nlambda=8, ncascades=5, seed=5)
    given = A.make_config(2, nx=64, ny=64, nlambda=8, ncascades=5)
    assert np.array_equal(small.xl, large.xl)
    ref_small, ref_large, ref_given = fresh(small), fresh(large), fresh(given)

    rc = binding.RadianceCascades(5)
    # one workspace large enough for everything below, so that only the plan moves
    need = max(rc.workspace_bytes(128, 96, 8), rc.workspace_bytes(64, 64, 8))
    rc.set_workspace(torch.full((need,), 0xFF, dtype=torch.uint8, device="cuda"))     # NaN-poisoned
    ls, ll = torch.from_numpy(small.line).cuda(), torch.from_numpy(large.line).cuda()
    chi, eta = torch.from_numpy(given.chi).cuda(), torch.from_numpy(given.eta).cuda()
    rc.set_line_atmosphere(ls, small.xl)
    assert torch.equal(rc.solve_J(), ref_small)
    rc.set_line_atmosphere(ll, large.xl)                   # new shape, same wavelengths
    assert torch.equal(rc.solve_J(), ref_large)
    rc.set_line_atmosphere(ls, small.xl)
    assert torch.equal(rc.solve_J(), ref_small)
    rc.set_atmosphere(chi, eta)                            # same shape, other mode
    assert torch.equal(rc.solve_J(), ref_given)
    rc.set_line_atmosphere(ls, small.xl)
    assert torch.equal(rc.solve_J(), ref_small)
    assert torch.equal(rc.compute_alo(), _alo(small))
    rc.set_workspace(torch.full((need + 4096,), 0xFF, dtype=torch.uint8, device="cuda"))   # the caller moves the workspace
    rc.set_line_atmosphere(ls, small.xl)
    assert torch.equal(rc.solve_J(), ref_small)
    rc.close()


def _alo(atm):
    import torch
    from paper_2408_14425_b200 import binding
    rc = binding.RadianceCascades(atm.ncascades)
    rc.set_line_atmosphere(torch.from_numpy(atm.line).cuda(), atm.xl)
    out = rc.compute_alo().clone()
    rc.close()
    return out


def test_a_knob_changed_on_a_live_small_grid_context_is_not_answered_from_the_old_graph():
    """Config 0 replays a captured graph.  tau_cut = 2 visibly changes J (transmittances below 1/4 are dropped), so a
    solve that still replays the graph captured before the knob changed shows up as the old J."""
    import torch
    from paper_2408_14425_b200 import binding
    atm = A.make_config(0)
    ref_default, ref_cut = fresh(atm), fresh(atm, tuning=dict(tau_cut=2.0))
    assert not torch.equal(ref_default, ref_cut)
    ref_nosort = fresh(atm, tuning=dict(sorted=0, cpw_from=-1))
    rc = binding.RadianceCascades(atm.ncascades)
    chi, eta = torch.from_numpy(atm.chi).cuda(), torch.from_numpy(atm.eta).cuda()
    out = torch.empty_like(ref_default)
    rc.set_atmosphere(chi, eta)
    for _ in range(2):
        assert torch.equal(rc.solve_J(out), ref_default)
    rc.set_tuning(tau_cut=2.0)
    rc.set_atmosphere(chi, eta)                            # same pointers, same shape, same output
    assert torch.equal(rc.solve_J(out), ref_cut)
    rc.set_tuning(tau_cut=126.0, sorted=0, cpw_from=-1)    # knobs that move the layout and the launch variants
    rc.set_atmosphere(chi, eta)
    assert torch.equal(rc.solve_J(out), ref_nosort)
    rc.close()


def test_host_path_validates_this_calls_data_at_pipelined_size():
    """RC_VALIDATE through rc_solve_J_host on a grid large enough for the two-half pipeline: the check has to see the
    arrays of THIS call - a bad value is refused on the first call (the staging buffers then hold nothing yet) and on a
    later one (they then hold the previous, valid, arrays)."""
    import torch
    from paper_2408_14425_b200 import binding
    atm = A.make_config(2, nx=512, ny=512, nlambda=64, ncascades=7)
    chi_h, eta_h = torch.from_numpy(atm.chi).pin_memory(), torch.from_numpy(atm.eta).pin_memory()
    bad = chi_h.clone().pin_memory()
    bad[300, 17, 40] = -1.0

    rc = binding.RadianceCascades(atm.ncascades, flags=binding.RC_VALIDATE)
    with pytest.raises(binding.RcError) as e:
        rc.solve_J_host(bad, eta_h)
    assert e.value.code == -5
    ref = rc.solve_J_host(chi_h, eta_h).clone()
    with pytest.raises(binding.RcError) as e:
        rc.solve_J_host(bad, eta_h)
    assert e.value.code == -5
    rc.close()

    plain = binding.RadianceCascades(atm.ncascades)        # the pipelined path, no validation: same J
    assert torch.equal(plain.solve_J_host(chi_h, eta_h), ref)
    plain.close()


@pytest.mark.parametrize("L", [1, 2, 8])
def test_line_host_path_stages_behind_the_line_plan(L):
    """rc_solve_J_line_host stages its input and J in the host_io part of the workspace; with few wavelengths the line
    plan reaches further than the GivenFs plan that region was laid out for."""
    import torch
    from paper_2408_14425_b200 import binding
    atm = A.line_config2(nx=64, ny=64, nlambda=L, ncascades=5)
    ref = fresh(atm)
    rc = binding.RadianceCascades(atm.ncascades)
    out = rc.solve_J_line_host(torch.from_numpy(atm.line).pin_memory(), atm.xl)
    assert torch.equal(out.cuda(), ref)
    out = rc.solve_J_line_host(torch.from_numpy(atm.line).pin_memory(), atm.xl)
    assert torch.equal(out.cuda(), ref)
    rc.close()
