"""CPU tests of the host logic behind the launches: rc_plan_query computes, without a device, the plan
rc_set_atmosphere would use (workspace layout, wavelengths per thread, lane patches, L2 banding, table sizes)."""
import pytest

from paper_2408_14425_b200 import atmospheres as A
from paper_2408_14425_b200 import binding

FIX = binding.RC_BILINEAR_FIX


def plan(cfg, **kw):
    nx, ny, L, nc = A.FULL_SHAPES[cfg]
    return binding.plan_query(nc, nx, ny, L, **kw)


def test_lane_patches_follow_the_clipping_of_the_cascades():
    """Short rays: 32x1 patches (longest contiguous gathers).  Cascades clipped by the box: 8x4 (config 2,
    cascade 5: lock-step utilisation 0.51 -> 0.75).  Never wider than the probe lattice."""
    p = plan(2)
    assert [p.patch_w[i] for i in range(4)] == [32, 32, 32, 32]
    assert p.patch_w[5] == 8 and p.patch_w[4] in (8, 16)
    assert p.patch_w[7] <= 8                      # 8 x 8 probes on the top cascade
    assert p.cascade_empty[7] == 1 and p.cascade_empty[6] == 0   # t_7 = 5461 > the diagonal; t_6 = 1365 < 1448
    p0 = plan(0)
    assert p0.patch_w[4] <= 4 and p0.cascade_empty[4] == 0   # 4 x 4 probes; t_4 = 85 < 90.5
    p4 = plan(4)                                   # 4096 x 1024: wide patches stay good along x
    assert p4.patch_w[5] >= 16 and p4.patch_w[4] == 32


def test_sorted_quads_where_the_box_clips_the_rays():
    """Lanes from quads sorted by ray length replace the rectangular patch where that raises the estimated lock-step
    utilisation (config 2: cascade 5 0.75 -> 0.88, cascade 4 0.92 -> 0.97); never on the short cascades and never on banded
    cascades (config 3, cascade 5)."""
    p = plan(2)
    assert [p.cascade_sorted[i] for i in range(8)] == [0, 0, 0, 1, 1, 1, 0, 0]
    assert 0.86 < p.lane_utilisation[5] < 0.90 and 0.96 < p.lane_utilisation[4] < 0.98
    assert all(p.lane_utilisation[i] > 0.99 for i in range(3))
    pf = plan(2, flags=FIX)                        # with the fix: the lattice of one parity class, same lists for the 4 classes
    assert [pf.cascade_sorted[i] for i in range(8)] == [0, 0, 0, 0, 1, 1, 0, 0]
    p3 = plan(3)
    assert p3.cascade_banded[5] == 1 and p3.cascade_sorted[5] == 0
    assert p3.cascade_banded[4] == 0 and p3.cascade_sorted[4] == 1    # rays short against the banded axis: no bands needed
    assert p3.cascade_sorted[6] == 1


def test_wavelength_batches_and_channels():
    assert (plan(2).lambda_batch, plan(2).nbatches, plan(2).channels) == (8, 8, 8)
    assert (plan(0).lambda_batch, plan(0).nbatches) == (1, 1)
    p = plan(2, ninclinations=8)
    assert (p.lambda_batch, p.channels, p.nbatches) == (1, 8, 64)
    p = plan(2, ninclinations=4)
    assert (p.lambda_batch, p.channels, p.nbatches) == (2, 8, 32)
    nx, ny, L, nc = A.FULL_SHAPES[1]
    p = binding.plan_query(nc, nx, ny, 11, lambda_batch=4)
    assert (p.lambda_batch, p.nbatches) == (4, 3)            # ragged last batch


def test_l2_banding_only_where_a_batch_exceeds_l2():
    """Config 2: one batch of packed chi, S is 64 MB: no bands.  Configs 3 and 4: 256 MB: 4 bands along the
    longer axis, for the cascades whose rays are long against that axis (> 0.3 of it) and whose patches are small against
    a band: cascade 5 of config 3; never cascades 0-4."""
    assert plan(2).nbands == 1 and not any(plan(2).cascade_banded[i] for i in range(8))
    p3, p4 = plan(3), plan(4)
    assert (p3.nbands, p3.band_axis) == (4, 0) and (p4.nbands, p4.band_axis) == (4, 1)
    assert [p3.cascade_banded[i] for i in range(9)] == [0, 0, 0, 0, 0, 1, 0, 0, 0]
    assert not any(p4.cascade_banded[i] for i in range(4))
    # the moving-line mode gathers 24 bytes per cell for all wavelengths: always L2-resident
    assert plan(3, line_mode=True).nbands == 1 or not any(plan(3, line_mode=True).cascade_banded[i] for i in range(9))
    # the bilinear fix is not banded
    nx, ny, L, nc = A.FULL_SHAPES[3]
    pf = binding.plan_query(nc, nx, ny, L, flags=FIX)
    assert not any(pf.cascade_banded[i] for i in range(9))


def test_workspace_and_tables_scale_as_documented():
    p2 = plan(2)
    assert 1.0e9 < p2.workspace_bytes < 1.3e9                 # 4 fields of 268 MB + tables (1.6 GB with host_io)
    # every cascade below the clipped ones has ~ 4^(i+1) directions x 4^i (sqrt2-ish) steps
    assert p2.table_steps[0] == 12                            # 4 diagonals x (own cell, diagonal neighbour, 1 spare)
    assert p2.table_steps[7] == 0 and p2.table_steps[5] > p2.table_steps[4] > p2.table_steps[3]
    nx, ny, L, nc = A.FULL_SHAPES[2]
    pf = binding.plan_query(nc, nx, ny, L, flags=FIX)
    assert pf.table_steps[7] == 0 and pf.table_steps[3] > 10 * p2.table_steps[3]   # 16 tables per direction
    assert pf.workspace_bytes > p2.workspace_bytes
    pi = plan(2, ninclinations=8)
    assert pi.workspace_bytes > p2.workspace_bytes + 2 * 7 * 268e6     # merged cascades hold 8x the channels
    assert plan(2, line_mode=True).workspace_bytes < p2.workspace_bytes   # 24 B per cell instead of 512


def test_bad_arguments():
    with pytest.raises(binding.RcError) as e:
        binding.plan_query(8, 1000, 1024, 4)       # 1000 is not a multiple of 2^7
    assert e.value.code == -2
    with pytest.raises(binding.RcError):
        binding.plan_query(8, 1024, 1024, 4, ninclinations=3)
    with pytest.raises(binding.RcError):
        binding.plan_query(0, 64, 64, 1)
