"""Gaussian descriptors (Eqs. (40)-(43) PAPER.md:396-412; reading G1).

CPU part pins the oracle to closed forms it does not contain: the value of one Gaussian, the unit integral of each
Gaussian (a Riemann sum over a fine grid must return the number of atoms times the weight), the Jacobi-theta lattice
sum of a periodic crystal, and invariances.  GPU part: element-wise parity of mala_gaussian_grid with the oracle."""
import math
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402

BIG = np.eye(3) * 60.0


def test_single_gaussian_value_weight_and_cutoff():
    s = 0.7
    d = np.array([0.3, -0.5, 1.1])
    want = math.exp(-d @ d / (2 * s * s)) / ((2 * math.pi) ** 1.5 * s ** 3)
    g = oracle.gaussian_points([[5, 5, 5]], [d + 5], [0], BIG, pbc=(0, 0, 0), sigma=s, wj=(2.5,))
    assert g.shape == (1, 1) and abs(g[0, 0] - 2.5 * want) < 1e-15
    # two types, two channels, different cutoffs: the far atom of type 1 is outside its own (short) cutoff
    g2 = oracle.gaussian_points([[5, 5, 5]], [d + 5, [5, 5, 8.0]], [0, 1], BIG, pbc=(0, 0, 0), sigma=s, rcutfac=4.0,
                                radelem=(0.5, 0.25), wj=(1.0, 3.0))
    assert abs(g2[0, 0] - want) < 1e-15 and g2[0, 1] == 0.0
    g3 = oracle.gaussian_points([[5, 5, 5]], [d + 5, [5, 5, 6.9]], [0, 1], BIG, pbc=(0, 0, 0), sigma=s, rcutfac=4.0,
                                radelem=(0.5, 0.25), wj=(1.0, 3.0))
    assert abs(g3[0, 1] - 3.0 * math.exp(-1.9 ** 2 / (2 * s * s)) / ((2 * math.pi) ** 1.5 * s ** 3)) < 1e-15


def test_unit_integral_riemann_sum():
    # cutoff 8 sigma: the truncated tail is < 1e-13; a 0.1-sigma grid integrates a Gaussian to ~1e-15
    s, n = 0.5, 80
    L = 8.0
    pos = np.array([[3.1, 4.2, 3.7], [4.9, 3.3, 4.4], [4.0, 4.0, 4.05]])
    pts = oracle.grid_points(np.eye(3) * L, (0, 0, 0), (n, n, n))
    g = oracle.gaussian_points(pts, pos, [0, 0, 0], np.eye(3) * L, pbc=(0, 0, 0), sigma=s, rcutfac=4.0, wj=(1.5,))
    assert abs(g.sum() * (L / n) ** 3 - 3 * 1.5) < 1e-9


def test_periodic_lattice_sum_is_a_theta_function():
    # simple cubic lattice, grid point at the origin, cutoff far out: the 3-D sum factorises into (sum_n exp(-(n a)^2/2s^2))^3
    a, s = 1.3, 0.6
    g = oracle.gaussian_points([[0, 0, 0]], [[0, 0, 0]], [0], np.eye(3) * a, pbc=(1, 1, 1), sigma=s, rcutfac=9.0)
    theta = sum(math.exp(-(n * a) ** 2 / (2 * s * s)) for n in range(-12, 13))
    full = theta ** 3 / ((2 * math.pi) ** 1.5 * s ** 3)
    # the sphere of radius 9 cuts terms below exp(-81/0.72) ~ 1e-49 only
    assert abs(g[0, 0] - full) < 1e-13 * full


def test_invariances():
    rng = np.random.default_rng(8)
    box = np.array([[5.0, 0, 0], [1.0, 4.5, 0], [0.5, -0.7, 5.5]])
    pos = rng.random((7, 3)) @ box
    types = [0, 1, 0, 1, 1, 0, 0]
    kw = dict(sigma=0.8, rcutfac=3.5, radelem=(0.5, 0.45), wj=(1.0, 0.7))
    pts = rng.random((5, 3)) @ box
    g = oracle.gaussian_points(pts, pos, types, box, pbc=(1, 1, 0), **kw)
    perm = rng.permutation(7)
    np.testing.assert_allclose(oracle.gaussian_points(pts, pos[perm], np.array(types)[perm], box, pbc=(1, 1, 0), **kw), g, rtol=1e-13)
    shifted = pos + np.outer(rng.integers(-2, 3, 7), box[0]) + np.outer(rng.integers(-2, 3, 7), box[1])
    np.testing.assert_allclose(oracle.gaussian_points(pts, shifted, types, box, pbc=(1, 1, 0), **kw), g, rtol=1e-12)


# ----------------------------------------------------------------------------------------------------------------
def _gpu(w_or_sys, sigma, **kw):
    import torch
    from paper_2411_19617_b200 import MalaSnap
    pos, types, box, origin, pbc, ngrid, params = w_or_sys
    with MalaSnap(**params) as snap:
        out = snap.gaussian_grid(sigma, pos, types, box, origin, pbc, ngrid, **kw)
        torch.cuda.synchronize()
        return out.cpu().numpy(), snap.last_stats()


@pytest.mark.gpu
def test_gpu_parity_tiny_al_full_grid_and_slabs():
    from paper_2411_19617_b200 import workloads
    w = workloads.make(1)
    sysd = (w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, w.snap_params())
    sigma = 0.6
    got, stats = _gpu(sysd, sigma)
    ref = oracle.gaussian_points(oracle.grid_points(w.box, w.origin, w.ngrid), w.pos, w.types, w.box, w.origin, w.pbc,
                                 sigma=sigma, rcutfac=w.rcutfac, radelem=w.radelem, wj=w.wj)
    assert got.shape == ref.shape == (w.npoints, 1)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    part, _ = _gpu(sysd, sigma, z_begin=5, z_end=12)
    # another slab means other tiles and another summation order of the candidates: equal to rounding, not bitwise
    assert np.abs(part - got[5 * 18 * 18:12 * 18 * 18]).max() <= 1e-14 * np.abs(ref).max()
    assert stats["kernels"] >= 2


@pytest.mark.gpu
def test_gpu_parity_two_types_triclinic_mixed_pbc_and_vacuum():
    rng = np.random.default_rng(21)
    box = np.array([[6.0, 0, 0], [1.5, 5.0, 0], [0.4, -0.8, 7.0]])
    pos = rng.random((9, 3)) @ box + np.array([0.3, -0.2, 9.0])   # unwrapped along the periodic axes
    types = rng.integers(0, 2, 9).astype(np.int32)
    params = dict(twojmax=2, rcutfac=3.0, rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5, 0.4), wj=(1.0, 0.6))
    ngrid = (13, 9, 21)
    origin = (0.1, 0.2, -0.3)
    got, _ = _gpu((pos, types, box, origin, (1, 1, 0), ngrid, params), 0.9)
    ref = oracle.gaussian_points(oracle.grid_points(box, origin, ngrid), pos, types, box, origin, (1, 1, 0), sigma=0.9,
                                 rcutfac=3.0, radelem=(0.5, 0.4), wj=(1.0, 0.6))
    assert got.shape == (13 * 9 * 21, 2)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    assert (ref == 0).any() and np.array_equal(got == 0, ref == 0)      # points in vacuum are exactly zero on both sides


@pytest.mark.gpu
def test_gpu_parity_boron_cluster_full_size_sampled():
    from paper_2411_19617_b200 import workloads
    w = workloads.make(4)
    got, _ = _gpu((w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, w.snap_params()), 0.5)
    rng = np.random.default_rng(4)
    samp = rng.integers(0, w.npoints, 4000)
    ref = oracle.gaussian_points(oracle.grid_points(w.box, w.origin, w.ngrid, sample=samp), w.pos, w.types, w.box, w.origin,
                                 w.pbc, sigma=0.5, rcutfac=w.rcutfac, radelem=w.radelem, wj=w.wj)
    assert np.abs(got[samp] - ref).max() <= 1e-12 * np.abs(ref).max()
    assert (got == 0).mean() > 0.7                                      # most of the box is vacuum


@pytest.mark.gpu
def test_gpu_invalid_arguments():
    from paper_2411_19617_b200 import MalaSnap, MalaSnapError
    with MalaSnap(twojmax=2, rcutfac=3.0, rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5,) * 5, wj=(1.0,) * 5) as snap:
        with pytest.raises(MalaSnapError):
            snap.gaussian_grid(0.5, np.zeros((1, 3)), [0], np.eye(3) * 4, ngrid=(4, 4, 4))     # more than 4 types
    with MalaSnap(twojmax=2, rcutfac=3.0, rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5,), wj=(1.0,)) as snap:
        with pytest.raises(MalaSnapError):
            snap.gaussian_grid(0.0, np.zeros((1, 3)), [0], np.eye(3) * 4, ngrid=(4, 4, 4))     # sigma must be positive
