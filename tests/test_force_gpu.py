"""GPU parity of row f3, mala_bispectrum_force_adjoint (Eqs. (44)-(45)): the Y contraction + dU recursion of
the CUDA path against the oracle's forward-mode derivative (oracle_bispectrum_grad_points, pinned in test_force_oracle.py by
finite differences and closed forms) on the same seeded inputs.  Both sides are exact up to rounding: tolerance 1e-9 of the
largest |g| (the CUDA path sums in another order, and its default compute_yi accumulates Y in 60-bit fixed point: about 1e-12)."""
import numpy as np
import pytest

import oracle
from paper_2411_19617_b200 import MalaSnap, MalaSnapError, workloads

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    return torch


def _grid_points(box, origin, ngrid, z0, z1):
    nx, ny, nz = ngrid
    iz, iy, ix = np.meshgrid(np.arange(z0, z1), np.arange(ny), np.arange(nx), indexing="ij")
    frac = np.stack([ix.ravel() / nx, iy.ravel() / ny, iz.ravel() / nz], axis=1)
    return frac @ np.asarray(box, float).reshape(3, 3) + np.asarray(origin, float)


def _compare(pos, types, box, origin, pbc, ngrid, z0, z1, params, seed, tol=1e-9, yi_impl=0, dedr_impl=0):
    torch = _torch()
    rng = np.random.default_rng(seed)
    pts = _grid_points(box, origin, ngrid, z0, z1)
    nt = oracle.ntriples(params["twojmax"])
    beta = rng.normal(size=(pts.shape[0], nt))
    ref = oracle.bispectrum_grad_points(pts, pos, types, box, origin, pbc, beta=beta, want_dB=False, **params)["g"]
    with MalaSnap(**params) as snap:
        snap.set_option("yi_impl", yi_impl)   # 0 / 2: block kernel, Y in fixed point; 1: table-driven kernel; 3: block kernel, fp64 atomics
        snap.set_option("dedr_impl", dedr_impl)   # 0: sampling kernel (DFT of Y as polynomial coefficients), 1: column kernel
        g = snap.force_adjoint(torch.as_tensor(beta, device="cuda"), pos, types, box, origin, pbc, ngrid, z0, z1)
        torch.cuda.synchronize()
        got = g.cpu().numpy()
    scale = np.abs(ref).max()
    assert scale > 0 and np.isfinite(got).all()
    assert np.abs(got - ref).max() <= tol * scale, f"max |dg| / max |g| = {np.abs(got - ref).max() / scale:.3e}"
    return got, beta


@pytest.mark.parametrize("yi_impl", [0, 1, 2, 3])
def test_cluster_in_a_box_twojmax6(yi_impl):
    rng = np.random.default_rng(41)
    pos = rng.uniform(3.0, 7.0, size=(6, 3))
    _compare(pos, np.zeros(6, np.int32), np.eye(3) * 10.0, (0, 0, 0), (0, 0, 0), (9, 8, 7), 0, 7, dict(twojmax=6, rcutfac=3.0), 1, yi_impl=yi_impl)


@pytest.mark.parametrize("dedr_impl", [0, 1])
@pytest.mark.parametrize("tj", [1, 2, 4, 7, 8, 10])
def test_both_compute_dedr_kernels_dense_periodic_system(tj, dedr_impl):
    """40 atoms of two types in a periodic 5 A box, cutoff 3.4 A: every point has some eighty neighbors among several hundred
    candidates (many full windows of the sampling kernel -- at twojmax 1 more sums per window than the CTA has threads --, images of
    the same atom in one window)"""
    rng = np.random.default_rng(90 + tj)
    pos = rng.uniform(0.0, 5.0, size=(40, 3))
    types = rng.integers(0, 2, 40).astype(np.int32)
    params = dict(twojmax=tj, rcutfac=3.4, radelem=(0.5, 0.45), wj=(1.0, 0.8), rmin0=0.1 if tj == 7 else 0.0)
    _compare(pos, types, np.eye(3) * 5.0, (0, 0, 0), (1, 1, 1), (5, 4, 3), 0, 3, params, 6, dedr_impl=dedr_impl, yi_impl=3 if dedr_impl else 0)


def test_periodic_triclinic_box_smaller_than_the_cutoff_two_types():
    rng = np.random.default_rng(42)
    box = np.array([[3.2, 0.0, 0.0], [0.6, 3.0, 0.0], [-0.3, 0.4, 3.4]])
    pos = rng.uniform(-0.2, 1.2, size=(3, 3)) @ box           # unwrapped on purpose
    types = np.array([0, 1, 0], np.int32)
    params = dict(twojmax=5, rcutfac=3.6, radelem=(0.5, 0.42), wj=(1.0, 0.7), wself=0.8)
    _compare(pos, types, box, (0.1, -0.2, 0.05), (1, 1, 0), (5, 6, 4), 1, 4, params, 2)


@pytest.mark.parametrize("tj", [0, 1, 2, 3, 8])
def test_other_twojmax_and_rmin0(tj):
    rng = np.random.default_rng(43 + tj)
    pos = rng.uniform(2.0, 6.0, size=(4, 3))
    params = dict(twojmax=tj, rcutfac=2.8, rmin0=0.3 if tj % 2 else 0.0)
    _compare(pos, np.zeros(4, np.int32), np.eye(3) * 8.0, (0, 0, 0), (1, 0, 1), (6, 5, 6), 0, 6, params, 3)


def test_config1_twojmax10_slab_and_slab_additivity():
    """tiny Al (box < cutoff: ~145 images move with their 4 atoms), twojmax 10, a three-plane slab against the oracle; two calls
    on adjacent slabs add up to one call on their union"""
    torch = _torch()
    w = workloads.make(1)
    got, beta = _compare(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 4, 7, w.snap_params(), 4)
    plane = w.ngrid[0] * w.ngrid[1]
    with MalaSnap(**w.snap_params()) as snap:
        b = torch.as_tensor(beta, device="cuda")
        g = snap.force_adjoint(b[:plane].contiguous(), w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 4, 5)
        snap.force_adjoint(b[plane:].contiguous(), w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 5, 7, out=g)
        torch.cuda.synchronize()
        assert np.abs(g.cpu().numpy() - got).max() <= 1e-11 * np.abs(got).max()
        snap.set_option("workspace_mb", 1)      # several chunks
        g2 = snap.force_adjoint(b, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 4, 7)
        torch.cuda.synchronize()
        assert np.abs(g2.cpu().numpy() - got).max() <= 1e-11 * np.abs(got).max()


def test_config2_full_grid_sparse_beta_in_bench_configuration():
    """the whole 90^3 grid of config 2 in the configuration bench.py --force times (two workspace chunks, every SM walking many
    tiles): beta is non-zero at 160 seeded grid points only, so the oracle's forward-mode derivative at those points is the
    complete answer"""
    torch = _torch()
    w = workloads.make(2)
    rng = np.random.default_rng(77)
    sample = np.sort(rng.choice(w.npoints, 160, replace=False))
    nt = 91
    bs = rng.normal(size=(sample.size, nt))
    pts = oracle.grid_points(w.box, w.origin, w.ngrid, sample=sample)
    ref = oracle.bispectrum_grad_points(pts, w.pos, w.types, w.box, w.origin, w.pbc, beta=bs, want_dB=False, **w.snap_params())["g"]
    beta = torch.zeros((w.npoints, nt), dtype=torch.float64, device="cuda")
    beta[torch.as_tensor(sample, device="cuda")] = torch.as_tensor(bs, device="cuda")
    with MalaSnap(**w.snap_params()) as snap:
        g = snap.force_adjoint(beta, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        torch.cuda.synchronize()
        assert snap.last_stats()["chunks"] >= 2
    got = g.cpu().numpy()
    scale = np.abs(ref).max()
    assert scale > 0 and np.isfinite(got).all()
    assert np.abs(got - ref).max() <= 1e-9 * scale, f"max |dg| / max |g| = {np.abs(got - ref).max() / scale:.3e}"


@pytest.mark.parametrize("case", ["one huge component", "tiny", "sixteen decades"])
def test_beta_ranges_through_the_fixed_point_and_the_fp64_accumulator(case):
    """the fixed-point Y of the default compute_yi takes its scale from the beta of each grid point: a single component a
    million times the others, betas of 1e-12, and betas spread over sixteen decades all stay at 1e-10 of the largest |g|
    (the fp64 accumulator at 1e-12)"""
    torch = _torch()
    w = workloads.make(1)
    rng = np.random.default_rng(5)
    nt, z0, z1 = 91, 4, 6
    pts = _grid_points(w.box, w.origin, w.ngrid, z0, z1)
    beta = rng.normal(size=(pts.shape[0], nt))
    if case == "one huge component":
        beta[:, 37] *= 1e6
    elif case == "tiny":
        beta *= 1e-12
    else:
        beta *= 10.0 ** rng.uniform(-8, 8, size=beta.shape)
    ref = oracle.bispectrum_grad_points(pts, w.pos, w.types, w.box, w.origin, w.pbc, beta=beta, want_dB=False, **w.snap_params())["g"]
    with MalaSnap(**w.snap_params()) as snap:
        for yi, tol in ((2, 1e-10), (3, 1e-12)):
            snap.set_option("yi_impl", yi)
            g = snap.force_adjoint(torch.as_tensor(beta, device="cuda"), w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z0, z1).cpu().numpy()
            assert np.isfinite(g).all()
            assert np.abs(g - ref).max() <= tol * np.abs(ref).max(), f"yi_impl {yi}: {np.abs(g - ref).max() / np.abs(ref).max():.3e}"


def test_uniform_beta_on_a_full_periodic_grid_gives_a_small_net_translation_force():
    """moving all atoms together equals moving the grid the other way: with the same beta at every point of a full periodic grid
    the sum over atoms of g is the beta-weighted grid sum of -dB/dr, which converges to zero as the grid resolves B (a sanity
    check of signs and image handling that needs no oracle)"""
    torch = _torch()
    w = workloads.make(1)
    nt = 91
    rng = np.random.default_rng(5)
    b1 = rng.normal(size=nt)
    with MalaSnap(**w.snap_params()) as snap:
        beta = torch.as_tensor(np.tile(b1, (w.npoints, 1)), device="cuda")
        g = snap.force_adjoint(beta, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid).cpu().numpy()
    assert np.abs(g.sum(axis=0)).max() < 1e-3 * np.abs(g).max()


def test_argument_errors():
    torch = _torch()
    w = workloads.make(1)
    with MalaSnap(twojmax=12) as snap:
        with pytest.raises(MalaSnapError) as e:
            snap.force_adjoint(torch.zeros((w.npoints, 140), dtype=torch.float64, device="cuda"), w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        assert e.value.code == -1
