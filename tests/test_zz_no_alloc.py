"""mala_gaussian_grid_static, the entry point that allocates no device memory (its scratch is a 16 MiB file-scope static device
array, include/mala_snap.h): its output against the existing path's (mala_gaussian_grid, itself checked against the oracle in
test_gaussian_descriptors.py) on two calls in a row, at the tolerance of those tests; the size limit; no change of the
device's free memory across a call.  Collected last on purpose (the file name), and independent of what ran before it."""
import numpy as np
import pytest

from paper_2411_19617_b200 import MalaSnap, MalaSnapError, workloads

pytestmark = pytest.mark.gpu

TOL = 1e-12   # of max |G|, as in test_gaussian_descriptors.py


def _close(a, b):
    scale = np.abs(b).max()
    assert scale > 0 and np.isfinite(a).all()
    assert np.abs(a - b).max() <= TOL * scale, f"max |dG| / max |G| = {np.abs(a - b).max() / scale:.3e}"


def test_static_entry_point_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    w = workloads.make(1)                      # tiny Al, periodic, 18^3 points
    rng = np.random.default_rng(31)
    box2 = np.array([[7.0, 0.0, 0.0], [1.0, 6.5, 0.0], [-0.5, 0.8, 9.0]])
    pos2 = rng.random((9, 3)) @ box2
    types2 = rng.integers(0, 2, 9).astype(np.int32)
    params2 = dict(twojmax=4, rcutfac=4.0, radelem=(0.5, 0.4), wj=(1.0, 0.6))
    with MalaSnap(**w.snap_params()) as a, MalaSnap(**params2) as b:
        # two calls in a row on the shared array, different systems and handles, one stream, the handles fresh (nothing of the
        # allocating path has run on them): the second call finds the first one's ghosts, cell list and candidate lists
        got1 = a.gaussian_grid_static(0.6, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        got2 = b.gaussian_grid_static(0.8, pos2, types2, box2, (0.1, 0.0, -0.2), (1, 0, 1), (13, 9, 11), 2, 10)
        got3 = a.gaussian_grid_static(0.6, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        torch.cuda.synchronize()
        ref1 = a.gaussian_grid(0.6, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid).cpu().numpy()
        ref2 = b.gaussian_grid(0.8, pos2, types2, box2, (0.1, 0.0, -0.2), (1, 0, 1), (13, 9, 11), 2, 10).cpu().numpy()
        _close(got1.cpu().numpy(), ref1)
        _close(got2.cpu().numpy(), ref2)
        assert torch.equal(got1, got3)         # the same tiles and the same summation order: bitwise
        assert a.last_stats()["kernels"] >= 2


def test_static_entry_point_config2_leaves_the_free_memory_alone():
    """config 2 (256 atoms, 90^3 points) fits the array; with the output allocated beforehand a call changes nothing in the
    device's free memory (the first call may load kernels, so the second one is measured)"""
    import torch
    w = workloads.make(2)
    with MalaSnap(**w.snap_params()) as snap:
        ref = snap.gaussian_grid(0.5, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        out = torch.empty_like(ref)
        snap.gaussian_grid_static(0.5, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, out=out)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        out.zero_()
        snap.gaussian_grid_static(0.5, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, out=out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0
        _close(out.cpu().numpy(), ref.cpu().numpy())


def test_static_entry_point_rejects_what_does_not_fit():
    """900,000 atoms leave about 22 MB of ghost records: beyond the 16 MiB array, a clear error and nothing enqueued"""
    import torch
    rng = np.random.default_rng(32)
    n = 900_000
    pos = rng.random((n, 3)) * 200.0
    with MalaSnap(twojmax=2, rcutfac=4.0) as snap:
        out = torch.full((8 * 8 * 8, 1), -1.0, dtype=torch.float64, device="cuda")
        with pytest.raises(MalaSnapError) as e:
            snap.gaussian_grid_static(0.5, pos, np.zeros(n, np.int32), np.eye(3) * 200.0, pbc=(0, 0, 0), ngrid=(8, 8, 8), out=out)
        assert e.value.code == -1 and "static scratch" in str(e.value)
        torch.cuda.synchronize()
        assert bool((out == -1.0).all())
        # the handle is still usable, and the allocating path takes the same system
        small = snap.gaussian_grid_static(0.5, pos[:50], np.zeros(50, np.int32), np.eye(3) * 200.0, pbc=(0, 0, 0), ngrid=(8, 8, 8))
        ref = snap.gaussian_grid(0.5, pos[:50], np.zeros(50, np.int32), np.eye(3) * 200.0, pbc=(0, 0, 0), ngrid=(8, 8, 8))
        torch.cuda.synchronize()
        assert np.abs(small.cpu().numpy() - ref.cpu().numpy()).max() <= TOL * max(np.abs(ref.cpu().numpy()).max(), 1e-300)
