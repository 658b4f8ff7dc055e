"""GPU parity: the CUDA path behind the C ABI against the CPU oracle, element by element, on the same seeded inputs.

Bar (BASELINE.json north_star): for each component k, max_p |B_gpu[p,k] - B_oracle[p,k]| <= 1e-9 * max_p |B_oracle[p,k]|.
Small cases compare whole grids; the full-size configs compare seeded samples of points (the oracle computes any
point on its own) plus properties that hold at any size (constant vector on empty points, slab-split identity).
"""
import numpy as np
import pytest

import oracle
from paper_2411_19617_b200 import MalaSnap, MalaSnapError, workloads

pytestmark = pytest.mark.gpu
TOL = 1e-9


def _torch():
    import torch
    return torch


def assert_parity(got, ref, tol=TOL):
    assert got.shape == ref.shape
    assert np.isfinite(got).all()
    scale = np.abs(ref).max(axis=0)
    err = np.abs(got - ref).max(axis=0)
    bad = err > tol * scale
    assert not bad.any(), f"components {np.nonzero(bad)[0][:8]}: err/scale = {(err / scale)[bad][:8]}"
    return float((err / scale).max())


def gpu_grid(w, z0=0, z1=None, **opts):
    torch = _torch()
    with MalaSnap(**w.snap_params()) as snap:
        for k, v in opts.items():
            snap.set_option(k, v)
        out = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z0, z1)
        torch.cuda.synchronize()
        return out.cpu().numpy()


def oracle_grid(w, z0=0, z1=None, sample=None):
    return oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z0, z1, sample=sample, **w.snap_params())


# ---------------------------------------------------------------------------------------------------------------
# config 1 in full, both contraction kernels, whole grid = many tiles + ragged tails (18 is not a multiple of 4)
# ---------------------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def tiny_ref():
    w = workloads.make(1)
    return w, oracle_grid(w)


@pytest.mark.parametrize("zi_impl", [1, 2, 3, 4])
def test_config1_tiny_al_full_grid(tiny_ref, zi_impl):
    w, ref = tiny_ref
    got = gpu_grid(w, zi_impl=zi_impl)
    assert_parity(got, ref)


@pytest.mark.parametrize("ui_impl", [1, 2, 3])
def test_config1_both_compute_ui_kernels(tiny_ref, ui_impl):
    """the column kernel (polynomial recursion), the sampling kernel (roots of unity + inverse DFT) and its producer / consumer
    form against the oracle"""
    w, ref = tiny_ref
    got = gpu_grid(w, ui_impl=ui_impl)
    assert_parity(got, ref)


@pytest.mark.parametrize("twojmax", [1, 3, 6, 8, 9])
def test_compute_ui_kernels_other_twojmax(twojmax):
    torch = _torch()
    pos, types, box, origin, pbc, ngrid, params = _small_case(7000 + twojmax, twojmax, 5, (1, 0, 1), True, True)
    ref = oracle.bispectrum_grid(pos, types, box, origin, pbc, ngrid, **params)
    for ui in ((1, 2, 3) if twojmax >= 8 else (1, 2)):
        with MalaSnap(**params) as snap:
            snap.set_option("ui_impl", ui)
            got = snap.bispectrum_grid(pos, types, box, origin, pbc, ngrid)
            torch.cuda.synchronize()
        assert_parity(got.cpu().numpy(), ref)
    with MalaSnap(twojmax=12) as snap, pytest.raises(MalaSnapError):
        snap.set_option("ui_impl", 2)


@pytest.mark.parametrize("twojmax", [8, 10, 12, 14])
def test_dense_system_several_candidate_windows(twojmax):
    """70 atoms in a 6 A box: every grid point has far more neighbors than one window of candidates holds (48 in the sampling
    kernel, 32..40 entries per point in the pipelined one, where several windows are sent once per accumulation pass)"""
    torch = _torch()
    rng = np.random.default_rng(909 + twojmax)
    box = np.eye(3) * 6.0
    pos = rng.uniform(0.0, 6.0, size=(70, 3))
    types = rng.integers(0, 2, 70).astype(np.int32)
    params = dict(twojmax=twojmax, rcutfac=4.2, rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5, 0.45), wj=(1.0, 0.8))
    ngrid = (5, 6, 3)
    ref = oracle.bispectrum_grid(pos, types, box, (0, 0, 0), (1, 1, 1), ngrid, **params)
    for ui in ((0, 1, 2, 3) if twojmax <= 10 else (0, 1, 3)):   # 0: automatic
        with MalaSnap(**params) as snap:
            snap.set_option("ui_impl", ui)
            got = snap.bispectrum_grid(pos, types, box, (0, 0, 0), (1, 1, 1), ngrid)
            torch.cuda.synchronize()
        assert_parity(got.cpu().numpy(), ref)


def test_very_dense_system_more_windows_than_the_spill_keeps():
    """260 atoms in a 6 A box: about a thousand candidates per tile, i.e. more windows than the 16 whose pair geometry the
    pipelined compute_ui keeps for its later passes -- the rest is prepared again in every pass"""
    torch = _torch()
    rng = np.random.default_rng(4242)
    box = np.eye(3) * 6.0
    pos = rng.uniform(0.0, 6.0, size=(260, 3))
    types = np.zeros(260, np.int32)
    params = dict(twojmax=8, rcutfac=4.2, rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5,), wj=(1.0,))
    ngrid = (4, 4, 2)
    ref = oracle.bispectrum_grid(pos, types, box, (0, 0, 0), (1, 1, 1), ngrid, **params)
    for ui in (2, 3):
        with MalaSnap(**params) as snap:
            snap.set_option("ui_impl", ui)
            got = snap.bispectrum_grid(pos, types, box, (0, 0, 0), (1, 1, 1), ngrid)
            torch.cuda.synchronize()
            assert snap.last_stats()["cand_cap"] > 16 * 40
        assert_parity(got.cpu().numpy(), ref)


def test_triples_match_oracle_order():
    with MalaSnap(twojmax=10) as s:
        assert s.ncomp == 91
        assert np.array_equal(s.triples(), oracle.triples(10))


def test_slab_split_and_small_workspace_are_identical(tiny_ref):
    """grid points are independent: any z split / internal chunking reproduces the full result"""
    w, ref = tiny_ref
    full = gpu_grid(w)
    # a slab may get another tile shape, hence another neighbor summation order: equal to rounding
    parts = np.concatenate([gpu_grid(w, a, b) for a, b in ((0, 5), (5, 6), (6, 18))])
    assert np.abs(parts - full).max() <= 1e-13 * np.abs(full).max()
    assert_parity(parts, ref)
    # internal chunking keeps the tiles, so it is bit-identical
    chunked = gpu_grid(w, workspace_mb=1)
    assert np.array_equal(chunked, full)
    assert gpu_grid(w, 7, 7).shape[0] == 0


def test_repeat_calls_are_bitwise_deterministic(tiny_ref):
    w, _ = tiny_ref
    torch = _torch()
    with MalaSnap(**w.snap_params()) as snap:
        a = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid).clone()
        b = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        torch.cuda.synchronize()
        assert torch.equal(a, b)


def test_host_output_entry_point(tiny_ref):
    w, ref = tiny_ref
    torch = _torch()
    with MalaSnap(**w.snap_params()) as snap:
        snap.set_option("host_chunk_mb", 1)
        out = snap.bispectrum_grid_host(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        dev = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        torch.cuda.synchronize()
    assert np.array_equal(out.numpy(), dev.cpu().numpy())
    assert_parity(out.numpy(), ref)


# ---------------------------------------------------------------------------------------------------------------
# U_tot itself (rows a3 + a4) against the oracle's explicit Wigner-D sum
# ---------------------------------------------------------------------------------------------------------------
def test_utot_matches_explicit_wigner_D(tiny_ref):
    w, _ = tiny_ref
    torch = _torch()
    with MalaSnap(**w.snap_params()) as snap:
        u = snap.debug_utot(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 2, 3).cpu().numpy()
    nx, ny, nz = w.ngrid
    ix, iy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    frac = np.stack([ix.ravel() / nx, iy.ravel() / ny, np.full(nx * ny, 2 / nz)], axis=1)
    pts = frac @ w.box + np.asarray(w.origin)
    res = oracle.bispectrum_points(pts, w.pos, w.types, w.box, w.origin, w.pbc, want_U=True, **w.snap_params())
    U = res["U"]
    # B is the same for D, D^T, conj(D) and D^dagger (reading #16); the library may store any ONE of them, everywhere
    worst = np.zeros(4)
    e = 0
    for J in range(w.twojmax + 1):
        D = U[:, oracle.uoff(J):oracle.uoff(J) + (J + 1) ** 2].reshape(-1, J + 1, J + 1)
        for mb in range(J // 2 + 1):
            for ma in range(J + 1):
                g = u[:, e, 0] + 1j * u[:, e, 1]
                cands = (D[:, ma, mb], D[:, mb, ma], np.conj(D[:, ma, mb]), np.conj(D[:, mb, ma]))
                for c, v in enumerate(cands):
                    worst[c] = max(worst[c], np.abs(g - v).max())
                e += 1
    assert e == u.shape[1]
    assert worst.min() < 1e-11 * np.abs(U).max(), worst


# ---------------------------------------------------------------------------------------------------------------
# brute force on tiny inputs: every twojmax, triclinic box, mixed pbc, two types, box smaller than rcut
# ---------------------------------------------------------------------------------------------------------------
def _small_case(seed, twojmax, natoms, pbc, triclinic, two_types, ngrid=(7, 5, 6)):
    rng = np.random.default_rng(seed)
    box = np.diag([3.1, 3.7, 4.3])
    if triclinic:
        box = box + np.array([[0.0, 0.0, 0.0], [0.9, 0.0, 0.0], [-0.6, 0.8, 0.0]])
        if seed % 2:
            box = box[[1, 0, 2]]  # left-handed
    pos = rng.random((natoms, 3)) @ box * 1.6 - 0.9  # unwrapped, partly outside the cell
    ntypes = 2 if two_types else 1
    types = rng.integers(0, ntypes, natoms).astype(np.int32)
    params = dict(twojmax=twojmax, rcutfac=2.4, rfac0=0.99363, rmin0=0.0 if seed % 3 else 0.3, wself=1.0 if seed % 2 else 0.7,
                  radelem=(0.5, 0.37)[:ntypes], wj=(1.0, 0.6)[:ntypes])
    origin = (0.1, -0.2, 0.05)
    return pos, types, box, origin, pbc, ngrid, params


@pytest.mark.parametrize("twojmax", [0, 1, 2, 3, 4, 5, 7, 8, 9, 10, 11, 12, 13, 14])
def test_small_cases_every_twojmax(twojmax):
    """twojmax 11..14 run on half tiles (16 points per CTA, two items per warp): SURVEY.md 8(f) row f4"""
    torch = _torch()
    for seed, (natoms, pbc, tri, two) in enumerate([(0, (1, 1, 1), False, False), (1, (0, 0, 0), False, False),
                                                    (3, (1, 1, 1), True, True), (5, (1, 0, 1), True, True),
                                                    (2, (0, 1, 0), False, True)]):
        pos, types, box, origin, pbc, ngrid, params = _small_case(100 * twojmax + seed, twojmax, natoms, pbc, tri, two)
        ref = oracle.bispectrum_grid(pos, types, box, origin, pbc, ngrid, **params)
        with MalaSnap(**params) as snap:
            for zi in ([3, 4] if twojmax > 10 else [0]):   # half tiles: the anti-diagonal and the block kernel
                snap.set_option("zi_impl", zi)
                got = snap.bispectrum_grid(pos, types, box, origin, pbc, ngrid)
                torch.cuda.synchronize()
                assert snap.ncomp == ref.shape[1]
                assert_parity(got.cpu().numpy(), ref)


@pytest.mark.parametrize("ngrid,zr", [((1, 1, 1), (0, 1)), ((2, 3, 1), (0, 1)), ((9, 1, 5), (1, 4)), ((5, 13, 7), (0, 7)),
                                      ((33, 2, 3), (0, 3)), ((6, 10, 9), (2, 9)), ((17, 17, 2), (0, 2))])
def test_ragged_grid_shapes_cover_every_point_once(ngrid, zr):
    """the region tiling (main bricks, x strip, y strip, corner) on extents that are not multiples of any brick, with z-slabs"""
    torch = _torch()
    pos, types, box, origin, pbc, _, params = _small_case(77, 3, 4, (1, 1, 0), True, True)
    ref = oracle.bispectrum_grid(pos, types, box, origin, pbc, ngrid, zr[0], zr[1], **params)
    with MalaSnap(**params) as snap:
        out = torch.full((ref.shape[0] + 3, ref.shape[1]), float("nan"), dtype=torch.float64, device="cuda")
        snap.bispectrum_grid(pos, types, box, origin, pbc, ngrid, zr[0], zr[1], out=out)
        torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.isnan(got[ref.shape[0]:]).all()          # nothing written past the slab
    assert_parity(got[:ref.shape[0]], ref)


def test_random_small_systems_all_kernels():
    """60 seeded random systems (twojmax 0..10, 0..6 atoms, one or two types, triclinic / left-handed boxes, any periodicity,
    grids 1..13 per axis, random z-slabs, sometimes a 1 MB workspace) through every zi kernel"""
    torch = _torch()
    rng = np.random.default_rng(2024)
    n = 0
    for it in range(60):
        tj = int(rng.integers(0, 15 if it % 5 == 0 else 11))
        box = np.diag(rng.uniform(2.5, 6.0, 3))
        if rng.random() < 0.5:
            box = box + np.tril(rng.uniform(-1, 1, (3, 3)), -1)
        if rng.random() < 0.3:
            box = box[[1, 0, 2]]
        natoms = int(rng.integers(0, 7))
        pos = rng.random((natoms, 3)) @ box * 1.5 - 0.5
        ntypes = int(rng.integers(1, 3))
        types = rng.integers(0, ntypes, natoms).astype(np.int32)
        pbc = tuple(int(x) for x in rng.integers(0, 2, 3))
        ngrid = tuple(int(x) for x in rng.integers(1, 14, 3))
        z0 = int(rng.integers(0, ngrid[2]))
        z1 = int(rng.integers(z0 + 1, ngrid[2] + 1))
        params = dict(twojmax=tj, rcutfac=float(rng.uniform(1.5, 3.2)), rfac0=0.99363, rmin0=float(rng.choice([0.0, 0.2])),
                      wself=float(rng.choice([1.0, 0.5])), radelem=(0.5, 0.4)[:ntypes], wj=(1.0, 0.7)[:ntypes])
        origin = tuple(rng.uniform(-0.3, 0.3, 3))
        ref = oracle.bispectrum_grid(pos, types, box, origin, pbc, ngrid, z0, z1, **params)
        with MalaSnap(**params) as snap:
            for zi in ([3, 4, 0] if tj > 10 else ([1, 3, 4] if tj != 10 else [1, 2, 3, 4])):
                snap.set_option("zi_impl", zi)
                if rng.random() < 0.3:
                    snap.set_option("workspace_mb", 1)
                got = snap.bispectrum_grid(pos, types, box, origin, pbc, ngrid, z0, z1)
                torch.cuda.synchronize()
                assert_parity(got.cpu().numpy(), ref)
                n += 1
    assert n >= 160


def test_zero_atoms_gives_self_term_everywhere():
    """closed form: B_{j1 j2 j} = wself^3 (j+1) for every triple (north_star: zero neighbors -> self term only)"""
    torch = _torch()
    with MalaSnap(twojmax=10, wself=1.3) as snap:
        out = snap.bispectrum_grid(np.zeros((0, 3)), np.zeros(0, np.int32), np.eye(3) * 5.0, ngrid=(9, 6, 5))
        torch.cuda.synchronize()
        expect = 1.3 ** 3 * (snap.triples()[:, 2] + 1.0)
    got = out.cpu().numpy()
    assert got.shape == (270, 91)
    assert np.abs(got - expect[None, :]).max() < 1e-12 * expect.max()


def test_atom_exactly_on_a_grid_point_and_at_the_cutoff():
    """reading #11 (continuous limit at r = 0) and #12 (strict < at rcut; f_c(rcut) = 0)"""
    torch = _torch()
    box = np.eye(3) * 8.0
    ngrid = (8, 8, 8)
    pos = np.array([[2.0, 3.0, 4.0],      # on grid point (2,3,4)
                    [5.0, 3.0, 4.0 + 1e-13]])  # 3.0 = rcut away from (2,3,4) up to rounding
    types = np.zeros(2, np.int32)
    params = dict(twojmax=6, rcutfac=3.0)
    ref = oracle.bispectrum_grid(pos, types, box, (0, 0, 0), (1, 1, 1), ngrid, **params)
    with MalaSnap(**params) as snap:
        got = snap.bispectrum_grid(pos, types, box, ngrid=ngrid)
        torch.cuda.synchronize()
    assert_parity(got.cpu().numpy(), ref)


def test_neighbor_inside_rmin0_reading22():
    """reading #22: f_c saturates at 1 and theta0 turns negative for r < rmin0 (pinned on the oracle side by closed forms)"""
    torch = _torch()
    box = np.eye(3) * 6.0
    ngrid = (6, 6, 6)
    pos = np.array([[1.0 + 0.12, 2.0 - 0.1, 3.0 + 0.12],   # 0.197 from grid point (1,2,3): inside rmin0 = 0.3
                    [4.0, 4.0 + 0.31, 1.0],                # just outside rmin0 of grid point (4,4,1)
                    [2.5, 2.6, 0.4], [5.1, 0.3, 3.3]])
    types = np.array([0, 1, 0, 1], np.int32)
    params = dict(twojmax=8, rcutfac=2.6, rmin0=0.3, wself=0.9, radelem=(0.5, 0.45), wj=(1.0, 0.7))
    ref = oracle.bispectrum_grid(pos, types, box, (0, 0, 0), (1, 1, 1), ngrid, **params)
    with MalaSnap(**params) as snap:
        got = snap.bispectrum_grid(pos, types, box, ngrid=ngrid)
        torch.cuda.synchronize()
    assert_parity(got.cpu().numpy(), ref)


def test_candidate_overflow_is_reported_not_silent():
    """the per-tile candidate capacity is an exact host bound; if it is ever violated (forced here through the test hook) the
    truncation must surface as an error code, both from the status query and from the next call on the handle"""
    torch = _torch()
    w = workloads.make(1)
    with MalaSnap(**w.snap_params()) as snap:
        ok = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        assert snap.last_stats()["status"] == 0 and snap.last_stats()["cand_cap"] > 32
        snap.set_option("cand_cap_limit", 32)
        snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, out=ok)   # enqueued; overflows on the device
        with pytest.raises(MalaSnapError) as e:
            snap.last_stats()
        assert e.value.code == -2 and "overflow" in str(e.value)
        snap.set_option("cand_cap_limit", 0)
        with pytest.raises(MalaSnapError) as e:      # sticky: the handle refuses further work
            snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, out=ok)
        assert e.value.code == -2
        with pytest.raises(MalaSnapError):
            snap.bispectrum_grid_host(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
    torch.cuda.synchronize()
    with MalaSnap(**w.snap_params()) as snap:       # a fresh handle is healthy; the host entry point reports it on return
        snap.set_option("cand_cap_limit", 32)
        with pytest.raises(MalaSnapError) as e:
            snap.bispectrum_grid_host(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        assert e.value.code == -2


def test_calls_on_two_streams_and_two_handles_do_not_interfere(tiny_ref):
    """one handle used from two streams back to back (serialised on the device by the library), interleaved with a second
    handle of another twojmax on a third stream: every result equals its stand-alone value bit for bit"""
    torch = _torch()
    w, ref = tiny_ref
    pos, types, box, origin, pbc, ngrid, params = _small_case(5, 6, 5, (1, 1, 1), True, True, ngrid=(11, 9, 10))
    s1, s2, s3 = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    with MalaSnap(**w.snap_params()) as a, MalaSnap(**params) as b, MalaSnap(**{**params, "twojmax": 8}) as c:
        alone_a = a.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid).clone()
        alone_b = b.bispectrum_grid(pos, types, box, origin, pbc, ngrid).clone()
        alone_c = c.bispectrum_grid(pos, types, box, origin, pbc, ngrid).clone()
        torch.cuda.synchronize()
        outs = []
        for it in range(3):
            oa1 = torch.empty_like(alone_a); oa2 = torch.empty_like(alone_a)
            ob = torch.empty_like(alone_b); oc = torch.empty_like(alone_c)
            a.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, out=oa1, stream=s1)
            b.bispectrum_grid(pos, types, box, origin, pbc, ngrid, out=ob, stream=s3)
            a.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 0, 9, out=oa2, stream=s2)
            c.bispectrum_grid(pos, types, box, origin, pbc, ngrid, out=oc, stream=s1)
            outs.append((oa1, oa2, ob, oc))
        torch.cuda.synchronize()
        n9 = 9 * w.ngrid[0] * w.ngrid[1]
        part = a.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 0, 9)
        torch.cuda.synchronize()
        for oa1, oa2, ob, oc in outs:
            assert torch.equal(oa1, alone_a) and torch.equal(ob, alone_b) and torch.equal(oc, alone_c)
            assert torch.equal(oa2[:n9], part)
    assert_parity(alone_a.cpu().numpy(), ref)


def test_invalid_arguments_are_rejected_without_enqueueing():
    torch = _torch()
    w = workloads.make(1)
    with MalaSnap(**w.snap_params()) as snap:
        out = torch.zeros((20 * 18 * 18, 91), dtype=torch.float64, device="cuda")
        for kw in (dict(ngrid=(18, 18, 0)), dict(z_begin=3, z_end=2), dict(z_end=19), dict(types=np.array([0, 0, 1, 0])),
                   dict(box=np.zeros((3, 3))), dict(pos=np.full((4, 3), np.nan))):
            a = dict(pos=w.pos, types=w.types, box=w.box, origin=w.origin, pbc=w.pbc, ngrid=w.ngrid, z_begin=0, z_end=1)
            a.update(kw)
            with pytest.raises(MalaSnapError) as e:
                snap.bispectrum_grid(out=out, **a)
            assert e.value.code == -1
        torch.cuda.synchronize()
        assert float(out.abs().max()) == 0.0
        with pytest.raises(MalaSnapError):
            snap.set_option("no_such_option", 1)


# ---------------------------------------------------------------------------------------------------------------
# full-size configs in the launch configuration bench.py times: sampled points + any-size properties
# ---------------------------------------------------------------------------------------------------------------
def _sampled_parity(w, got, nsample, seed):
    rng = np.random.default_rng(seed)
    npts = w.npoints
    sample = np.unique(np.concatenate([rng.integers(0, npts, nsample), [0, npts - 1, w.ngrid[0] - 1, npts - w.ngrid[0]]]))
    ref = oracle_grid(w, sample=sample)
    return assert_parity(got[sample], ref), sample, ref


def _bj0j_full_grid(w, got, z_begin=0, z_end=None):
    """every grid point of the slab: the 11 components B_{j,0,j} against the Chebyshev closed form (second oracle: no
    Wigner-D, no CG; SURVEY 8(c) pins) -- a wrong tile, lane or region anywhere on the grid shows up here"""
    tr = oracle.triples(10)
    idx = [int(np.where((tr[:, 0] == j) & (tr[:, 1] == 0) & (tr[:, 2] == j))[0][0]) for j in range(11)]
    ref = oracle.bj0j_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z_begin, z_end, **w.snap_params())
    sub = got[:, idx]
    assert sub.shape == ref.shape
    scale = np.abs(ref).max(axis=0)
    assert (np.abs(sub - ref).max(axis=0) <= TOL * scale).all()


def test_config2_solid_al_full_size_sampled():
    """headline workload: 256-atom Al, 90^3 grid; 3,000 seeded sample points + two complete z-planes"""
    torch = _torch()
    w = workloads.make(2)
    with MalaSnap(**w.snap_params()) as snap:
        out = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert snap.last_stats()["points"] == 729000
        # the same slab computed alone agrees to rounding
        part = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 44, 46).cpu().numpy()
    _sampled_parity(w, got, 3000, 22)
    _bj0j_full_grid(w, got)
    plane = 90 * 90
    assert np.abs(part - got[44 * plane:46 * plane]).max() <= 1e-13 * np.abs(part).max()
    assert_parity(part[:plane], oracle_grid(w, 44, 45))
    # lattice translation of one atom / permutation of atoms: invariances (north_star) hold to rounding on the GPU too
    pos2 = w.pos[::-1].copy()
    pos2[3] += w.box[0] - 2 * w.box[2]
    part2 = gpu_grid(workloads.Workload(**{**w.__dict__, "pos": pos2}), 44, 45)
    assert np.abs(part2 - part[:plane]).max() <= 1e-11 * np.abs(part).max()


def test_config2_multi_chunk_workspace_is_bit_identical():
    """the workspace-capped chunk loop at real size: 1 GiB cap -> >= 3 chunks of the 90^3 grid, same tiles, same bits"""
    torch = _torch()
    w = workloads.make(2)
    with MalaSnap(**w.snap_params()) as snap:
        one = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        assert snap.last_stats()["chunks"] == 1
        snap.set_option("workspace_mb", 1024)
        many = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        st = snap.last_stats()
        assert st["chunks"] >= 3 and st["workspace_bytes"] <= 1024 << 20
        assert torch.equal(one, many)
        snap.set_option("workspace_mb", 300)
        many = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid)
        assert snap.last_stats()["chunks"] >= 10
        assert torch.equal(one, many)


def test_config3_liquid_al_full_size_sampled():
    w = workloads.make(3)
    got = gpu_grid(w)
    _sampled_parity(w, got, 2000, 33)
    _bj0j_full_grid(w, got)


def test_config4_boron_cluster_full_size_sampled_and_empty_points():
    """79 % of the points have no neighbor and must hold exactly the constant self-only vector"""
    w = workloads.make(4)
    got = gpu_grid(w)
    nx, ny, nz = w.ngrid
    rng = np.random.default_rng(44)
    # sample biased towards the cluster (uniform sampling would mostly hit empty points)
    near = []
    while len(near) < 1500:
        i = rng.integers(0, nx, 3)
        p = i / np.array(w.ngrid) * 20.0
        if np.linalg.norm(p - 10.0) < 8.5:
            near.append((i[2] * ny + i[1]) * nx + i[0])
    sample = np.unique(np.concatenate([near, rng.integers(0, w.npoints, 500)]))
    ref = oracle_grid(w, sample=sample)
    assert_parity(got[sample], ref)
    # every point farther than rcut from all atoms: self term only, closed form wself^3 (j+1)
    ix, iy, iz = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    idx = ((iz * ny + iy) * nx + ix).ravel()
    pts = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1) / np.array(w.ngrid) * 20.0
    d2min = np.full(pts.shape[0], np.inf)
    for a in w.pos:
        d2min = np.minimum(d2min, ((pts - a) ** 2).sum(1))
    empty = idx[d2min > (w.rcutfac * (1 + 1e-12)) ** 2]
    assert 0.75 < empty.size / w.npoints < 0.83
    expect = oracle.triples(10)[:, 2] + 1.0
    assert np.abs(got[empty] - expect[None, :]).max() < 1e-12 * expect.max()
    _bj0j_full_grid(w, got)


def test_config5_be_slab_z_slabs_sampled():
    """16,384-atom Be slab with the stacking fault; output streamed in z-slabs (here: the slab through the fault, one
    at the periodic boundary and a ragged last slab), sampled against the oracle"""
    torch = _torch()
    w = workloads.make(5)
    nx, ny, nz = w.ngrid
    assert (nx, ny, nz) == (183, 317, 287)
    rng = np.random.default_rng(55)
    with MalaSnap(**w.snap_params()) as snap:
        for z0, z1 in ((140, 148), (0, 3), (280, 287)):
            out = snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z0, z1)
            torch.cuda.synchronize()
            got = out.cpu().numpy()
            n = (z1 - z0) * ny * nx
            sample = np.unique(np.concatenate([rng.integers(0, n, 250), [0, n - 1]]))
            ref = oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z0, z1, sample=sample, **w.snap_params())
            assert_parity(got[sample], ref)
            if z0 == 140:  # one complete plane through the stacking fault against the Chebyshev closed form
                _bj0j_full_grid(w, got[3 * ny * nx:4 * ny * nx], 143, 144)
            del out


def test_config5_whole_grid_streamed_to_host():
    """north_star: "fp64 output streamed in z-slabs" -- the WHOLE 183 x 317 x 287 grid (16.6 M points, 12.1 GB) through
    mala_bispectrum_grid_host into one host buffer.  Checked with the stratified sample of SURVEY.md 8(d): the closed-form
    second oracle (11 components B_{j,0,j}) on every 8th z-plane plus the planes at both fault interfaces, and 2,000 seeded
    random points on all 91 components against the full oracle."""
    torch = _torch()
    w = workloads.make(5)
    nx, ny, nz = w.ngrid
    plane = nx * ny
    try:
        host = torch.empty((w.npoints, 91), dtype=torch.float64, pin_memory=True)
    except RuntimeError:
        host = torch.empty((w.npoints, 91), dtype=torch.float64)
    host[::plane].fill_(float("nan"))
    with MalaSnap(**w.snap_params()) as snap:
        snap.bispectrum_grid_host(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, out=host)
        st = snap.last_stats()
    assert st["status"] == 0
    got = host.numpy()
    assert np.isfinite(got[::plane]).all() and np.isfinite(got[-1]).all()
    # the two fault interfaces: basal layers 15|16 (middle of the cell) and 31|0 (periodic boundary), c/2 = 1.792 A per layer.
    # The oracle visits all 16,384 atoms x 125 images per point (~20 ms of one core), so complete planes are checked at the two
    # interfaces and 500 seeded points in every 8th plane and in the planes next to the interfaces.
    zf = int(round(16 * 1.792 / 57.344 * nz))
    for z in (zf, 0):
        _bj0j_full_grid(w, got[z * plane:(z + 1) * plane], z, z + 1)
    rng = np.random.default_rng(555)
    tr = oracle.triples(10)
    idx = [int(np.where((tr[:, 0] == j) & (tr[:, 1] == 0) & (tr[:, 2] == j))[0][0]) for j in range(11)]
    for z in sorted(set(range(0, nz, 8)) | {zf - 1, zf + 1, nz - 1}):
        smp = np.unique(np.concatenate([rng.integers(0, plane, 500), [0, nx - 1, plane - nx, plane - 1]]))
        ref = oracle.bj0j_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z, z + 1, sample=smp, **w.snap_params())
        sub = got[z * plane + smp][:, idx]
        assert (np.abs(sub - ref).max(axis=0) <= TOL * np.abs(ref).max(axis=0)).all(), z
    sample = np.unique(np.concatenate([rng.integers(0, w.npoints, 2000), [0, w.npoints - 1]]))
    ref = oracle_grid(w, sample=sample)
    assert_parity(got[sample], ref)
