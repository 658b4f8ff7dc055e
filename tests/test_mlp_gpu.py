"""GPU parity of the descriptor -> LDOS network: the tcgen05 kernel behind mala_mlp_forward and the
fused mala_bispectrum_ldos_grid against the fp64 oracles (oracle/mlp_oracle.py on top of oracle/snap_oracle.c).

Tolerance: TF32 operands carry 11 significant bits, rounded to nearest on both sides, so a product is
off by at most 2^-10 relative; accumulation, bias and activation are fp32 (negligible beside that).  For a pre-activation
z_k = sum_j w_kj h_j of a layer with K inputs this gives |dz_k| <= 2^-10 sum_j |w_kj h_j| in the worst case -- about
2^-10 * 0.8 sqrt(K) = 1.2e-2 of the rms of z for K = 256 inputs of random sign -- and about 2^-11.5 rms|z| = 3e-4 typically
(random walk).  The activations are 1-Lipschitz and the He-scaled synthetic weights keep |h| ~ |z| from layer to layer, so the
errors of the layers add: typically ~1e-3 of the output scale after three layers, with a tail that reaches a few times that
over the ~1e6 values a test compares (5.4e-3 observed on the full config-1 grid).  The tests allow 1e-2 of the largest |y| of
each output channel, floored at a tenth of the largest channel -- the worst-case bound of a single 256-wide layer.
"""
import numpy as np
import pytest

import oracle
from oracle import mlp_oracle
from paper_2411_19617_b200 import MalaMlp, MalaSnap, MalaSnapError, bispectrum_ldos_grid, workloads

pytestmark = pytest.mark.gpu
TOL = 1e-2


def _torch():
    import torch
    return torch


def assert_close(got, ref, tol=TOL):
    assert got.shape == ref.shape and np.isfinite(got).all()
    # per output channel, relative to the channel's largest value -- but not below a tenth of the largest channel: the rounding
    # error of a pre-activation scales with |w_k| |h|, not with what the activation lets through (a ReLU channel that is
    # almost always off has a tiny maximum and the same absolute error as its neighbours)
    scale = np.abs(ref).max(axis=0)
    scale = np.maximum(scale, 0.1 * scale.max())
    err = np.abs(got - ref).max(axis=0) / scale
    assert err.max() <= tol, f"max err/scale {err.max():.3e} at channel {int(err.argmax())}"
    return float(err.max())


def _net(rng, sizes):
    ws = [rng.normal(size=(b, a)) * np.sqrt(2.0 / a) for a, b in zip(sizes[:-1], sizes[1:])]
    bs = [0.1 * rng.normal(size=b) for b in sizes[1:]]
    return ws, bs


@pytest.mark.parametrize("sizes,act,last,npts", [((91, 256, 256, 241), "leaky_relu", True, 1000), ((8, 16), "identity", True, 128),
                                                  ((91, 64, 241), "sigmoid", False, 129), ((91, 100, 37, 241), "relu", True, 127),
                                                  ((30, 256, 256, 256, 256, 250), "leaky_relu", False, 777), ((5, 1), "identity", False, 1)])
def test_mlp_forward_matches_the_fp64_oracle(sizes, act, last, npts):
    torch = _torch()
    rng = np.random.default_rng(sum(sizes) + npts)
    ws, bs = _net(rng, sizes)
    x = rng.normal(size=(npts, sizes[0])) * 3.0 + 1.0
    shift, scale = rng.normal(size=sizes[0]), rng.uniform(0.2, 0.6, size=sizes[0])
    ref = mlp_oracle.mlp_forward(x, ws, bs, act, last, shift, scale)
    with MalaMlp(ws, bs, act, last, shift, scale) as net:
        assert (net.w_in, net.w_out) == (sizes[0], sizes[-1])
        y = net.forward(torch.as_tensor(x, device="cuda"))
        y2 = net.forward(torch.as_tensor(x, device="cuda"))
        torch.cuda.synchronize()
        assert torch.equal(y, y2)                       # deterministic
    assert_close(y.cpu().numpy().astype(np.float64), ref)


def test_mlp_exact_on_tf32_representable_data():
    """integers and small dyadic weights are exact in TF32 and their sums exact in fp32: the tensor-core path must then
    reproduce the oracle bit for bit up to the final fp32 rounding -- pins operand layout, K order, bias and padding"""
    torch = _torch()
    rng = np.random.default_rng(5)
    sizes = (91, 48, 241)
    ws = [rng.integers(-4, 5, size=(b, a)).astype(np.float64) / 8.0 for a, b in zip(sizes[:-1], sizes[1:])]
    bs = [rng.integers(-8, 9, size=b).astype(np.float64) / 4.0 for b in sizes[1:]]
    x = rng.integers(-8, 9, size=(300, 91)).astype(np.float64)
    ref = mlp_oracle.mlp_forward(x, ws, bs, "relu", True)
    with MalaMlp(ws, bs, "relu", True) as net:
        y = net.forward(torch.as_tensor(x, device="cuda"))
        torch.cuda.synchronize()
    assert np.array_equal(y.cpu().numpy().astype(np.float64), ref)


def test_mlp_argument_errors():
    with pytest.raises(MalaSnapError) as e:
        MalaMlp([np.zeros((300, 91))], [np.zeros(300)])
    assert e.value.code == -1
    with pytest.raises(MalaSnapError):
        MalaMlp([np.full((4, 4), np.nan)], [np.zeros(4)])
    w = workloads.make(1)
    with MalaSnap(**w.snap_params()) as snap, MalaMlp([np.zeros((5, 30))], [np.zeros(5)]) as net:
        with pytest.raises(MalaSnapError) as e:       # 30 inputs, 91 descriptor components
            bispectrum_ldos_grid(snap, net, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        assert e.value.code == -1


def test_fused_descriptor_network_config1_full_grid():
    """config 1 (ragged 18^3 grid, several tiles per region) through mala_bispectrum_ldos_grid: LDOS of every grid point
    against oracle MLP(oracle descriptors); also z-slabs and a tiny workspace (many chunks)"""
    torch = _torch()
    w = workloads.make(1)
    ws, bs, shift, scale = workloads.ldos_network()
    B = oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, **w.snap_params())
    ref = mlp_oracle.mlp_forward(B, ws, bs, "leaky_relu", True, shift, scale)
    with MalaSnap(**w.snap_params()) as snap, MalaMlp(ws, bs, "leaky_relu", True, shift, scale) as net:
        ldos = bispectrum_ldos_grid(snap, net, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        torch.cuda.synchronize()
        full = ldos.cpu().numpy().astype(np.float64)
        assert_close(full, ref)
        part = bispectrum_ldos_grid(snap, net, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 5, 11)
        torch.cuda.synchronize()
        n = 18 * 18
        assert_close(part.cpu().numpy().astype(np.float64), ref[5 * n:11 * n])
        snap.set_option("workspace_mb", 1)          # 183 tiles in chunks of 148: same tiles, same bits
        chunked = bispectrum_ldos_grid(snap, net, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        torch.cuda.synchronize()
        assert snap.last_stats()["chunks"] > 1
        assert torch.equal(chunked, ldos)
        # the network alone on the library's own descriptors gives the same bits as the fused call
        snap.set_option("workspace_mb", 4096)
        Bg = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        alone = net.forward(Bg)
        torch.cuda.synchronize()
        assert torch.equal(alone, ldos)


def test_fused_descriptor_network_empty_tiles_and_other_twojmax():
    """a cluster in vacuum (empty tiles take the constant descriptor) at twojmax 6, and a half-tile case at twojmax 12"""
    torch = _torch()
    rng = np.random.default_rng(9)
    box = np.eye(3) * 12.0
    pos = rng.uniform(4.0, 8.0, size=(5, 3))
    types = np.zeros(5, np.int32)
    for tj, ngrid in ((6, (20, 18, 16)), (12, (9, 7, 8))):
        params = dict(twojmax=tj, rcutfac=2.5)
        nc = (tj + 2) * (tj + 3) * (tj + 4) // 24
        ws, bs = _net(rng, (nc, 64, 50))
        scale = np.full(nc, 0.05)
        B = oracle.bispectrum_grid(pos, types, box, (0, 0, 0), (0, 0, 0), ngrid, **params)
        ref = mlp_oracle.mlp_forward(B, ws, bs, "leaky_relu", True, None, scale)
        with MalaSnap(**params) as snap, MalaMlp(ws, bs, "leaky_relu", True, None, scale) as net:
            ldos = bispectrum_ldos_grid(snap, net, pos, types, box, (0, 0, 0), (0, 0, 0), ngrid)
            torch.cuda.synchronize()
        assert_close(ldos.cpu().numpy().astype(np.float64), ref)
