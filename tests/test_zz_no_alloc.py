"""rc_count_empty_cells_static - the entry point for callers that cannot allocate device memory.

Who that is: code running inside an application whose memory pool took the whole GPU at start-up (cudaMalloc fails
there), or inside a real-time / serving loop where cudaMalloc and cudaFree are forbidden because they stall the device.
Such a caller cannot lend the workspace every other call of librc.so works out of, so this one call keeps its scratch in
an array built into the library (RC_STATIC_MAX_CELLS cells at most; shared by all calls, which therefore must not overlap
on the GPU).

Checked here: its count equals what the ordinary path reports (rc_analyse_atmosphere -> rc_stats.empty_cells, which works
out of a lent workspace) - exactly, it is an integer - on calls made back to back over the SAME built-in array, so a
call that trusted the array to be clean, or left something behind that the next one trips over, fails.  The file name
sorts last on purpose: pytest -x stops at the first failure, and a failure here should hide no other test.  It does not
depend on the other tests having run (or not): everything it needs it sets up itself.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2408_14425_b200 import atmospheres as A


def _cases():
    """(atmosphere, use an active-cell mask) - mostly-empty blobs (config 4's recipe) at sizes that take both load widths
    of the kernel (nlambda a multiple of 4, and not), a dense one, and shapes that shrink and grow between calls."""
    big = A.make_config(4, nx=512, ny=256, nlambda=12, ncascades=6)
    odd = A.make_config(4, nx=256, ny=128, nlambda=11, ncascades=6, seed=77)
    dense = A.make_config(1, nx=128, ny=128, nlambda=4, ncascades=5)
    return [(big, False), (A.with_active_cells(odd, "fraction", fraction=0.02), True), (odd, False), (dense, False),
            (A.with_active_cells(big, "occupied"), True), (big, False)]


def _existing_path(atm, use_active):
    """The count as the context-based path gives it: lent workspace, rc_analyse_atmosphere, rc_stats.empty_cells."""
    import torch
    from paper_2408_14425_b200 import binding
    rc = binding.RadianceCascades(atm.ncascades, atm.c0_interval, 0, 0, 0)
    chi, eta = torch.from_numpy(atm.chi).cuda(), torch.from_numpy(atm.eta).cuda()
    rc.set_atmosphere(chi, eta)
    if use_active:
        rc.set_active_cells(torch.from_numpy(np.ascontiguousarray(atm.active, dtype=np.uint8)).cuda())
    n = int(rc.analyse_atmosphere(lists=False).empty_cells)
    rc.close()
    return n


@pytest.mark.gpu
def test_static_scratch_count_matches_the_workspace_path_on_consecutive_calls():
    import torch
    from paper_2408_14425_b200 import binding
    cases = _cases()
    want = [_existing_path(atm, ua) for atm, ua in cases]
    assert 0 < want[0] < cases[0][0].nx * cases[0][0].ny and want[3] == 0      # the cases are not degenerate
    assert want[1] > want[2]                                                    # the mask makes more cells empty

    dev = [(torch.from_numpy(atm.chi).cuda(), torch.from_numpy(atm.eta).cuda(),
            torch.from_numpy(np.ascontiguousarray(atm.active, dtype=np.uint8)).cuda() if ua else None) for atm, ua in cases]
    outs = torch.full((2, len(cases)), -1, dtype=torch.int64, device="cuda")   # the caller's outputs, made up front
    torch.cuda.synchronize()
    # two rounds, every call right behind the previous one on one stream, nothing synchronised in between: each call
    # finds the array as the call before left it (another grid size, another mask)
    for r in range(2):
        if r == 1:
            free_before = torch.cuda.mem_get_info()[0]     # round 0 has loaded both kernel variants
        for i, (chi, eta, act) in enumerate(dev):
            binding.count_empty_cells_static(chi, eta, act, out=outs[r, i:i + 1])
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    got = outs.cpu().numpy()
    for r in range(2):
        assert got[r].tolist() == want, f"round {r}: static-scratch counts {got[r].tolist()} != workspace path {want}"
    # independent of both paths: the definition, counted by numpy
    for (atm, ua), w in zip(cases, want):
        occ = (atm.chi != 0).any(axis=2) | (atm.eta != 0).any(axis=2)
        if ua:
            occ &= atm.active != 0
        assert int((~occ).sum()) == w
    assert free_after >= free_before, "the calls of round 1 took device memory from somewhere"


@pytest.mark.gpu
def test_static_scratch_accepts_the_largest_grid_and_unaligned_arrays():
    """RC_STATIC_MAX_CELLS cells exactly (one wavelength), and arrays that start 4 bytes off a 16-byte boundary."""
    import torch
    from paper_2408_14425_b200 import binding
    g = torch.Generator(device="cuda").manual_seed(5)
    ny, nx = 1024, binding.RC_STATIC_MAX_CELLS // 1024
    chi = (torch.rand((ny, nx, 1), generator=g, device="cuda") < 0.3).float()
    eta = torch.zeros_like(chi)
    eta[7, 9, 0] = 2.0                                                  # emission without opacity is occupied too
    want = int(((chi == 0) & (eta == 0)).all(dim=2).sum())
    assert int(binding.count_empty_cells_static(chi, eta)) == want
    buf = torch.zeros(2 * 64 * 32 * 4 + 2, device="cuda")
    c4 = buf[1:1 + 64 * 32 * 4].view(64, 32, 4)                         # contiguous, 4 bytes off alignment
    c4[3, 5, 2] = 1.0
    e4 = buf[1 + 64 * 32 * 4:1 + 2 * 64 * 32 * 4].view(64, 32, 4)
    e4[60, 31, 3] = 1.0
    assert int(binding.count_empty_cells_static(c4, e4)) == 64 * 32 - 2


def test_static_scratch_rejects_what_does_not_fit_before_touching_the_device():
    """No GPU needed: shapes beyond the built-in array and null arguments come back as error codes with a message."""
    from paper_2408_14425_b200 import binding
    lib = binding.load()
    err = C.create_string_buffer(512)
    fake = C.c_void_p(256)                                              # never dereferenced: the checks come first
    rc = lib.rc_count_empty_cells_static(0, fake, fake, None, 2048, 1024, 4, fake, None, err, len(err))
    assert rc == -2 and b"RC_STATIC_MAX_CELLS" in err.value and b"2097152" in err.value
    rc = lib.rc_count_empty_cells_static(0, fake, fake, None, 1024, 1025, 1, fake, None, None, 0)   # errbuf is optional
    assert rc == -2
    assert lib.rc_count_empty_cells_static(0, None, fake, None, 8, 8, 1, fake, None, err, len(err)) == -1 and err.value
    assert lib.rc_count_empty_cells_static(0, fake, fake, None, 0, 8, 1, fake, None, err, len(err)) == -2
