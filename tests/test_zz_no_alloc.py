"""GPU test of chaoticus_ld_neighbour_diffs_noalloc, the one entry point for callers that cannot
allocate device memory (a host application that owns all of the HBM, or a loop that cannot take the
device-wide stall of cudaMalloc).  Its intermediate values (the members' Lagrangian descriptors) live
in a fixed 8 MiB array inside the library that every call shares and that keeps the last call's
contents, so the check is made on TWO calls in a row with different inputs and sizes: the second call
must not see anything of the first.  The reference is the existing path, chaoticus_ld_neighbours with
caller-owned arrays (itself checked against the oracle in test_gpu_more_kernels.py::test_ld_neighbours);
both run the same arithmetic, so the differences must agree bit for bit -- which is inside the 1e-9 M
absolute tolerance that the oracle comparison of these differences uses.

The file is named so that pytest collects it last: a failure here cannot hide another test under -x.
It needs no state from the other tests (run alone: the first call does the library's one-time look-up
of the array's address; run after the others: the array may hold anything)."""
import numpy as np
import pytest

from paper_2507_00622_b200 import workloads as W

pytestmark = pytest.mark.gpu
HH, C3 = W.SYS_HENON_HEILES, W.SYS_COUPLED3


@pytest.fixture(scope="module")
def chs():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2507_00622_b200 import binding
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _both_paths(chs, sysid, prm, y0, sigma, h, n_steps, forward=True, backward=True):
    """(existing path, no-alloc path) differences for the same input; the outputs of the no-alloc call are
    pre-filled with a canary so that an element it failed to write shows."""
    import torch
    n, n_ic = y0.shape
    ref = chs.ld_neighbours(sysid, prm, dev(y0), sigma, 0.0, h, n_steps, forward=forward, backward=backward)
    df = torch.full((2 * n, n_ic), -7.0, dtype=torch.float64, device="cuda") if forward else None
    db = torch.full((2 * n, n_ic), -7.0, dtype=torch.float64, device="cuda") if backward else None
    chs.ld_neighbour_diffs_noalloc(sysid, prm, dev(y0), sigma, 0.0, h, n_steps, df, db)
    torch.cuda.synchronize()
    return ref, df, db


def _same(got, want, scale):
    g, w = got.cpu().numpy(), want.cpu().numpy()
    assert g.shape == w.shape and np.isfinite(w).all() and w.max() > 0.0
    assert np.abs(g - w).max() <= 1e-9 * scale       # the tolerance of test_ld_neighbours
    assert (g == w).all()                            # and in fact the same bits: same kernels, same order


def test_no_alloc_diffs_match_the_existing_path_on_two_calls_in_a_row(chs):
    # call 1: Henon-Heiles, 133 ICs (ragged against the 128-thread blocks), both directions
    y1 = W.hh_grid(0.125, 19, 7)
    ref, df, db = _both_paths(chs, HH, None, y1, 1e-3, 0.01, 600)
    _same(df, ref["diff_fwd"], ref["fwd"][0].max().item())
    _same(db, ref["diff_bwd"], ref["bwd"][0].max().item())
    # call 2, straight after: another system (n = 6: 13 members), another size, so every offset in the
    # shared array now means something else and holds call 1's leftovers
    prm = W.coupled3_params(0.1)
    y2 = W.coupled3_ics(70, seed=1)
    ref, df, db = _both_paths(chs, C3, prm, y2, 1e-2, 0.01, 500)
    _same(df, ref["diff_fwd"], ref["fwd"][0].max().item())
    _same(db, ref["diff_bwd"], ref["bwd"][0].max().item())
    # call 3: call 1's input again, one direction only (the backward block then sits at offset 0)
    ref, df, db = _both_paths(chs, HH, None, y1, 1e-3, 0.01, 600, forward=False)
    assert df is None
    _same(db, ref["diff_bwd"], ref["bwd"][0].max().item())


def test_no_alloc_rejects_what_does_not_fit(chs):
    import torch
    cap = chs.NOALLOC_MAX_DOUBLES
    # Henon-Heiles: 9 members per IC and direction, each direction's block rounded up to 32 doubles
    fits_two = (cap // 2) // 9          # 58 254
    fits_one = cap // 9                 # 116 508
    y = dev(np.ascontiguousarray(np.tile(W.hh_grid(0.125, 4, 4)[:, :1], (1, fits_one + 1))))
    out_f = torch.zeros((8, fits_one + 1), dtype=torch.float64, device="cuda")
    out_b = torch.zeros((8, fits_one + 1), dtype=torch.float64, device="cuda")
    for n_ic, two, ok in ((fits_two, True, True), (fits_two + 1, True, False), (fits_one, False, True),
                          (fits_one + 1, False, False)):
        yy = y[:, :n_ic].contiguous() if n_ic != y.shape[1] else y
        f = out_f[:, :n_ic].contiguous() if n_ic != out_f.shape[1] else out_f
        b = (out_b[:, :n_ic].contiguous() if n_ic != out_b.shape[1] else out_b) if two else None
        if ok:
            chs.ld_neighbour_diffs_noalloc(HH, None, yy, 1e-3, 0.0, 0.01, 3, f, b)
            torch.cuda.synchronize()
            # all ICs are the same point: every column of a row carries the same value, up to the last one
            assert torch.isfinite(f).all().item() and (f == f[:, :1]).all().item()
        else:
            with pytest.raises(chs.ChaoticusError) as ei:
                chs.ld_neighbour_diffs_noalloc(HH, None, yy, 1e-3, 0.0, 0.01, 3, f, b)
            assert "scratch" in str(ei.value) and str(cap) in str(ei.value)
    # bad arguments are refused as on the existing path; nothing requested / empty ensemble: no-ops
    with pytest.raises(chs.ChaoticusError):
        chs.ld_neighbour_diffs_noalloc(HH, None, y[:, :8].contiguous(), -1.0, 0.0, 0.01, 3, out_f[:, :8].contiguous())
    chs.ld_neighbour_diffs_noalloc(HH, None, y[:, :8].contiguous(), 1e-3, 0.0, 0.01, 3, None, None)
    e = torch.empty((4, 0), dtype=torch.float64, device="cuda")
    chs.ld_neighbour_diffs_noalloc(HH, None, e, 1e-3, 0.0, 0.01, 3, torch.empty((8, 0), dtype=torch.float64, device="cuda"))


def test_no_alloc_call_leaves_free_device_memory_unchanged(chs):
    """The driver's free-memory figure before and after a run of calls: the library call itself takes nothing
    (the tensors are made beforehand; torch's caching allocator is not asked for anything in between)."""
    import torch
    y = dev(W.hh_grid(0.125, 32, 32))
    df = torch.empty((8, y.shape[1]), dtype=torch.float64, device="cuda")
    db = torch.empty_like(df)
    chs.ld_neighbour_diffs_noalloc(HH, None, y, 1e-3, 0.0, 0.01, 5, df, db)     # set-up call (module load)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(5):
        chs.ld_neighbour_diffs_noalloc(HH, None, y, 1e-3, 0.0, 0.01, 5, df, db)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
