"""Pins for the derivative oracle of row f3 (oracle_bispectrum_grad_points; Eqs. (44)-(45)) against
things other than itself: central finite differences of the already pinned descriptor oracle, closed forms, the
point-versus-atoms translation identity and rotation covariance."""
import numpy as np
import pytest

import oracle

RFAC0 = 0.99363
BIG = np.eye(3) * 50.0


def fc_and_slope(r, rcut, rmin0=0.0):
    x = (r - rmin0) / (rcut - rmin0)
    if x <= 0.0:
        return 1.0, 0.0
    return 0.5 * (np.cos(np.pi * x) + 1.0), -0.5 * np.pi * np.sin(np.pi * x) / (rcut - rmin0)


def _cluster(rng, n, rmax):
    p = rng.normal(size=(n, 3))
    p *= (rng.uniform(0.35, 1.0, size=(n, 1)) * rmax) / np.linalg.norm(p, axis=1, keepdims=True)
    return p


@pytest.mark.parametrize("case", ["cluster_tj6", "periodic_small_box_two_types", "rmin0"])
def test_gradient_equals_central_finite_differences(case):
    rng = np.random.default_rng(31)
    if case == "cluster_tj6":
        box, pbc, kw = BIG, (0, 0, 0), dict(twojmax=6, rcutfac=3.5)
        pos = _cluster(rng, 5, 3.0) + 25.0
        types = [0] * 5
        pts = 25.0 + 0.4 * rng.normal(size=(2, 3))
    elif case == "periodic_small_box_two_types":   # box smaller than the cutoff: every atom moves together with its images
        box = np.array([[3.2, 0.0, 0.0], [0.6, 3.0, 0.0], [-0.3, 0.4, 3.4]])
        pbc, kw = (1, 1, 0), dict(twojmax=4, rcutfac=3.6, radelem=(0.5, 0.42), wj=(1.0, 0.7), wself=0.8)
        pos = rng.uniform(0, 1, size=(3, 3)) @ box
        types = [0, 1, 0]
        pts = rng.uniform(0, 1, size=(2, 3)) @ box
    else:
        box, pbc, kw = BIG, (0, 0, 0), dict(twojmax=5, rcutfac=3.0, rmin0=0.3)
        pts = np.array([[25.0, 25.0, 25.0]])
        pos = np.concatenate([pts[0] + np.array([[0.12, -0.1, 0.12]]), pts[0] + _cluster(rng, 3, 2.5)])   # one neighbor inside rmin0
        types = [0] * 4
    res = oracle.bispectrum_grad_points(pts, pos, types, box, pbc=pbc, **kw)
    dB = res["dB"]
    h = 1e-5
    for a in range(len(pos)):
        for k in range(3):
            pp, pm = np.array(pos, float), np.array(pos, float)
            pp[a, k] += h
            pm[a, k] -= h
            Bp = oracle.bispectrum_points(pts, pp, types, box, pbc=pbc, **kw)["B"]
            Bm = oracle.bispectrum_points(pts, pm, types, box, pbc=pbc, **kw)["B"]
            fd = (Bp - Bm) / (2 * h)
            scale = np.abs(dB).max() + 1e-30
            assert np.abs(dB[:, a, k, :] - fd).max() <= 2e-8 * scale, (case, a, k)


def test_single_neighbor_closed_form_gradient():
    """B_t = (w f_c(r))^3 (j + 1) for one neighbor and wself = 0, any direction => dB_t/dR = 3 w^3 f_c^2 f_c'(r) (j + 1) d/r"""
    rng = np.random.default_rng(32)
    for tj in (3, 10):
        d = _cluster(rng, 1, 3.8)[0]
        w, rc = 0.8, 4.676
        res = oracle.bispectrum_grad_points([[0, 0, 0]], [d], [0], BIG, pbc=(0, 0, 0), wself=0.0, wj=(w,), rcutfac=rc, twojmax=tj)
        r = np.linalg.norm(d)
        fc, fcp = fc_and_slope(r, rc)
        jp1 = oracle.triples(tj)[:, 2] + 1.0
        expect = 3 * w ** 3 * fc ** 2 * fcp * jp1[None, :] * (d / r)[:, None]
        np.testing.assert_allclose(res["dB"][0, 0], expect, rtol=1e-9, atol=1e-12 * np.abs(expect).max())


def test_B000_gradient_closed_form_periodic_two_types():
    """B_000 = (wself + sum w f_c)^3 => dB_000/dR_alpha = 3 S^2 sum_{images of alpha} w f_c'(r) d/r (independent numpy images)"""
    rng = np.random.default_rng(33)
    box = np.array([[3.1, 0.0, 0.0], [0.7, 2.9, 0.0], [-0.4, 0.5, 3.3]])
    pos = rng.uniform(0, 1, size=(3, 3)) @ box
    types = [0, 1, 0]
    radelem, wj, rcutfac, wself = (0.5, 0.4), (1.0, 0.6), 3.9, 1.3
    pts = rng.uniform(0, 1, size=(3, 3)) @ box
    res = oracle.bispectrum_grad_points(pts, pos, types, box, pbc=(1, 1, 1), twojmax=2, rcutfac=rcutfac, wself=wself, radelem=radelem, wj=wj)
    rng_img = range(-4, 5)
    for ip, p in enumerate(pts):
        S = wself
        grads = np.zeros((3, 3))
        for a in range(3):
            rc = 2 * rcutfac * radelem[types[a]]
            for n1 in rng_img:
                for n2 in rng_img:
                    for n3 in rng_img:
                        d = pos[a] + n1 * box[0] + n2 * box[1] + n3 * box[2] - p
                        r = np.linalg.norm(d)
                        if r < rc:
                            fc, fcp = fc_and_slope(r, rc)
                            S += wj[types[a]] * fc
                            grads[a] += wj[types[a]] * fcp * d / r
        np.testing.assert_allclose(res["dB"][ip, :, :, 0], 3 * S ** 2 * grads, rtol=1e-10, atol=1e-12)


def test_moving_all_atoms_equals_moving_the_point_back_and_rotation_covariance():
    rng = np.random.default_rng(34)
    pos = _cluster(rng, 6, 3.2) + 25.0
    types = [0, 1, 0, 1, 1, 0]
    kw = dict(twojmax=6, rcutfac=3.6, radelem=(0.5, 0.45), wj=(1.0, 0.8))
    p = np.array([[25.1, 24.9, 25.2]])
    dB = oracle.bispectrum_grad_points(p, pos, types, BIG, pbc=(0, 0, 0), **kw)["dB"][0]      # [atom, k, t]
    h = 1e-5
    for k in range(3):
        e = np.zeros(3)
        e[k] = h
        Bp = oracle.bispectrum_points(p + e, pos, types, BIG, pbc=(0, 0, 0), **kw)["B"][0]
        Bm = oracle.bispectrum_points(p - e, pos, types, BIG, pbc=(0, 0, 0), **kw)["B"][0]
        np.testing.assert_allclose(dB[:, k, :].sum(axis=0), -(Bp - Bm) / (2 * h), rtol=0, atol=2e-8 * np.abs(dB).max())
    # rotate the atoms about the point: B is invariant, its gradient turns with the rotation
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    Rm = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                   [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                   [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])
    pos_r = p[0] + (pos - p[0]) @ Rm.T
    dBr = oracle.bispectrum_grad_points(p, pos_r, types, BIG, pbc=(0, 0, 0), **kw)["dB"][0]
    np.testing.assert_allclose(dBr, np.einsum("ij,ajt->ait", Rm, dB), rtol=0, atol=1e-10 * np.abs(dB).max())


def test_adjoint_is_the_beta_weighted_sum():
    rng = np.random.default_rng(35)
    pos = _cluster(rng, 4, 3.0) + 25.0
    pts = 25.0 + 0.5 * rng.normal(size=(5, 3))
    kw = dict(twojmax=4, rcutfac=3.4)
    beta = rng.normal(size=(5, oracle.ntriples(4)))
    res = oracle.bispectrum_grad_points(pts, pos, [0] * 4, BIG, pbc=(0, 0, 0), beta=beta, **kw)
    np.testing.assert_allclose(res["g"], np.einsum("pt,pakt->ak", beta, res["dB"]), rtol=1e-12, atol=1e-13)
