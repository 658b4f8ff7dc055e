"""Pins for the CPU oracle (oracle/snap_oracle.c) against things other than itself:
paper-printed counts, closed forms, group-theory identities, sympy, invariances.
SURVEY.md 8(c) "What pins each part"; BASELINE.json north_star invariants."""
import os

import numpy as np
import pytest
from scipy.special import eval_chebyu

import oracle

RFAC0 = 0.99363
HERE = os.path.dirname(os.path.abspath(__file__))


# ----------------------------------------------------------------------------------------------
# helpers written independently of the oracle's code: brute-force neighbor enumeration in numpy
# ----------------------------------------------------------------------------------------------
def brute_neighbors(point, pos, types, box, origin, pbc, rcut_t, nimg=4):
    """All (atom, image) displacement vectors d = R + n.A - point with |d| < rcut_type.  Atoms are first
    wrapped into the cell along periodic axes."""
    box = np.asarray(box, float).reshape(3, 3)
    inv = np.linalg.inv(box)
    f = (np.asarray(pos, float).reshape(-1, 3) - origin) @ inv
    for i in range(3):
        if pbc[i]:
            f[:, i] -= np.floor(f[:, i])
    w = origin + f @ box
    rng = [range(-nimg, nimg + 1) if pbc[i] else range(0, 1) for i in range(3)]
    out = []
    for n in range(w.shape[0]):
        for n1 in rng[0]:
            for n2 in rng[1]:
                for n3 in rng[2]:
                    d = w[n] + n1 * box[0] + n2 * box[1] + n3 * box[2] - point
                    if np.linalg.norm(d) < rcut_t[types[n]]:
                        out.append((d, types[n]))
    return out


def fc_theta(r, rcut, rmin0=0.0):
    """(f_c, theta0), written from DESIGN.md readings #3, #4 and #22: the switching function saturates at 1 for
    r <= rmin0, the theta0 map is linear in r throughout (negative below rmin0)."""
    x = (r - rmin0) / (rcut - rmin0)
    fc = 1.0 if x <= 0.0 else 0.5 * (np.cos(np.pi * x) + 1.0)
    return fc, RFAC0 * np.pi * x


def rand_unit_quat(rng):
    q = rng.normal(size=4)
    return q / np.linalg.norm(q)


def ab_of(q):
    return complex(q[0], -q[3]), complex(q[2], -q[1])


def rot_matrix(rng):
    q = rand_unit_quat(rng)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def cluster(rng, n, rmax):
    p = rng.normal(size=(n, 3))
    p *= (rng.uniform(0.3, 1.0, size=(n, 1)) * rmax) / np.linalg.norm(p, axis=1, keepdims=True)
    return p


BIG = np.eye(3) * 50.0


# ----------------------------------------------------------------------------------------------
# Eq. (26): component count
# ----------------------------------------------------------------------------------------------
def test_component_count_matches_paper_eq26():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "eq26_component_counts.txt")) if l[0] != "#"]
    for tj, cnt in rows:
        tj, cnt = int(tj), int(cnt)
        assert (tj + 2) * (tj + 3) * (tj + 4) // 24 == cnt          # the fixture is the paper's formula
        assert oracle.ntriples(tj) == cnt
        tr = oracle.triples(tj)
        assert len({tuple(t) for t in tr}) == cnt
        for j1, j2, j in tr:
            assert j2 <= j1 <= j <= tj and (j1 + j2 + j) % 2 == 0 and j1 - j2 <= j <= j1 + j2
    assert oracle.ntriples(10) == 91


# ----------------------------------------------------------------------------------------------
# Wigner-D
# ----------------------------------------------------------------------------------------------
def test_D1_is_g_itself():
    rng = np.random.default_rng(1)
    a, b = ab_of(rand_unit_quat(rng))
    g = np.array([[a, -np.conj(b)], [b, np.conj(a)]])
    D = oracle.wigner_D(1, a, b)
    # basis e_0 = eta, e_1 = xi and (xi, eta) -> (g00 xi + g01 eta, g10 xi + g11 eta):
    # D^1[m'][m] = g[1-m][1-m']  (g itself up to basis order / transposition)
    np.testing.assert_allclose(D, np.array([[g[1, 1], g[0, 1]], [g[1, 0], g[0, 0]]]), atol=1e-15)


@pytest.mark.parametrize("J", range(0, 15))
def test_D_unitary_and_trace_is_chebyshev(J):
    rng = np.random.default_rng(100 + J)
    for _ in range(5):
        q = rand_unit_quat(rng)
        a, b = ab_of(q)
        D = oracle.wigner_D(J, a, b)
        np.testing.assert_allclose(D @ D.conj().T, np.eye(J + 1), atol=2e-14)
        th0 = np.arccos(q[0])
        np.testing.assert_allclose(np.trace(D), np.sin((J + 1) * th0) / np.sin(th0), atol=4e-13)
        assert abs(np.trace(D).imag) < 1e-13


@pytest.mark.parametrize("J", [1, 2, 3, 6, 10])
def test_D_is_a_representation(J):
    rng = np.random.default_rng(200 + J)
    a1, b1 = ab_of(rand_unit_quat(rng))
    a2, b2 = ab_of(rand_unit_quat(rng))
    g1 = np.array([[a1, -np.conj(b1)], [b1, np.conj(a1)]])
    g2 = np.array([[a2, -np.conj(b2)], [b2, np.conj(a2)]])
    D1, D2 = oracle.wigner_D(J, a1, b1), oracle.wigner_D(J, a2, b2)
    g12, g21 = g1 @ g2, g2 @ g1
    D12 = oracle.wigner_D(J, g12[0, 0], g12[1, 0])
    D21 = oracle.wigner_D(J, g21[0, 0], g21[1, 0])
    e_h = np.abs(D1 @ D2 - D12).max()
    e_a = np.abs(D1 @ D2 - D21).max()
    assert min(e_h, e_a) < 5e-14            # homomorphism or anti-homomorphism, either is a valid convention
    assert max(e_h, e_a) > 1e-3 or J == 0   # and the test can tell them apart


# ----------------------------------------------------------------------------------------------
# Clebsch-Gordan
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("J1,J2", [(1, 1), (2, 1), (3, 2), (4, 4), (5, 3), (10, 10), (9, 4), (10, 7), (14, 14), (13, 9), (12, 5)])
def test_cg_orthogonality(J1, J2):
    js = list(range(abs(J1 - J2), J1 + J2 + 1, 2))
    cols = [(J, M) for J in js for M in range(-J, J + 1, 2)]
    rows = [(M1, M2) for M1 in range(-J1, J1 + 1, 2) for M2 in range(-J2, J2 + 1, 2)]
    C = np.array([[oracle.cg(J1, M1, J2, M2, J, M) for (J, M) in cols] for (M1, M2) in rows])
    assert C.shape[0] == C.shape[1]
    np.testing.assert_allclose(C.T @ C, np.eye(len(cols)), atol=5e-13)
    np.testing.assert_allclose(C @ C.T, np.eye(len(rows)), atol=5e-13)


def test_cg_against_sympy():
    from sympy import Rational
    from sympy.physics.quantum.cg import CG
    rng = np.random.default_rng(7)
    n = 0
    while n < 120:
        J1, J2 = rng.integers(0, 11, size=2)
        J = rng.choice(range(abs(J1 - J2), J1 + J2 + 1, 2))
        M1 = rng.choice(range(-J1, J1 + 1, 2))
        M2 = rng.choice(range(-J2, J2 + 1, 2))
        M = M1 + M2
        if abs(M) > J:
            continue
        ref = float(CG(Rational(int(J1), 2), Rational(int(M1), 2), Rational(int(J2), 2), Rational(int(M2), 2),
                       Rational(int(J), 2), Rational(int(M), 2)).doit())
        assert abs(oracle.cg(J1, M1, J2, M2, J, M) - ref) < 1e-13
        n += 1
    # textbook values
    assert abs(oracle.cg(1, 1, 1, -1, 0, 0) - 1 / np.sqrt(2)) < 1e-15
    assert abs(oracle.cg(1, -1, 1, 1, 0, 0) + 1 / np.sqrt(2)) < 1e-15
    assert abs(oracle.cg(2, 0, 2, 0, 4, 0) - np.sqrt(2 / 3)) < 1e-15
    assert oracle.cg(2, 0, 2, 0, 2, 0) == 0.0


# ----------------------------------------------------------------------------------------------
# closed forms for the whole pipeline
# ----------------------------------------------------------------------------------------------
def test_zero_neighbors_gives_self_term_only():
    for wself in (1.0, 0.7):
        r = oracle.bispectrum_points([[1.0, 2.0, 3.0]], np.zeros((0, 3)), [], BIG, pbc=(0, 0, 0), wself=wself)
        tr = r["triples"]
        np.testing.assert_allclose(r["B"][0], wself ** 3 * (tr[:, 2] + 1), rtol=1e-14)
    # atoms present but all beyond the cutoff
    r = oracle.bispectrum_points([[0, 0, 0]], [[4.7, 0, 0], [0, -5, 1]], [0, 0], BIG, pbc=(0, 0, 0), rcutfac=4.676)
    np.testing.assert_allclose(r["B"][0], r["triples"][:, 2] + 1, rtol=1e-14)
    assert r["nnbr"][0] == 0


def test_single_neighbor_closed_form():
    rng = np.random.default_rng(3)
    for it in range(6):
        d = cluster(rng, 1, 4.0)[0]
        w = 0.8
        tj = (10, 10, 10, 10, 12, 14)[it]     # twojmax above 10: SURVEY.md 8(f) row f4
        r = oracle.bispectrum_points([[0, 0, 0]], [d], [0], BIG, pbc=(0, 0, 0), wself=0.0, wj=(w,), rcutfac=4.676, twojmax=tj)
        fc, _ = fc_theta(np.linalg.norm(d), 4.676)
        assert r["B"].shape[1] == (tj + 2) * (tj + 3) * (tj + 4) // 24
        np.testing.assert_allclose(r["B"][0], (w * fc) ** 3 * (r["triples"][:, 2] + 1), rtol=4e-12)


def test_B000_closed_form_twojmax0_periodic_two_types():
    # tiny periodic triclinic box smaller than rcut, two species with different radii and weights
    rng = np.random.default_rng(4)
    box = np.array([[3.1, 0.0, 0.0], [0.7, 2.9, 0.0], [-0.4, 0.5, 3.3]])
    pos = rng.uniform(0, 1, size=(3, 3)) @ box
    types = [0, 1, 0]
    radelem, wj, rcutfac, wself = (0.5, 0.4), (1.0, 0.6), 3.9, 1.3
    rcut_t = [2 * rcutfac * x for x in radelem]
    pts = rng.uniform(0, 1, size=(4, 3)) @ box
    r = oracle.bispectrum_points(pts, pos, types, box, pbc=(1, 1, 1), twojmax=0, rcutfac=rcutfac, wself=wself,
                                 radelem=radelem, wj=wj)
    for p, B in zip(pts, r["B"]):
        nb = brute_neighbors(p, pos, types, box, np.zeros(3), (1, 1, 1), rcut_t)
        s = wself + sum(wj[t] * fc_theta(np.linalg.norm(d), rcut_t[t])[0] for d, t in nb)
        assert len(nb) > 10
        np.testing.assert_allclose(B[0], s ** 3, rtol=1e-13)


def chebyshev_bj0j(point, pos, types, box, origin, pbc, rcut_t, wj, wself, twojmax, rmin0=0.0):
    """B_{j,0,j} = (sum_k c_k) * sum_{k,l} c_k c_l U_j(<q_k,q_l>), k,l over the self term and all neighbors
    (SURVEY.md 8(c)); needs neither Wigner-D nor CG."""
    nb = brute_neighbors(point, pos, types, box, origin, pbc, rcut_t)
    cs, qs = [wself], [np.array([1.0, 0, 0, 0])]
    for d, t in nb:
        r = np.linalg.norm(d)
        fc, th0 = fc_theta(r, rcut_t[t], rmin0)
        cs.append(wj[t] * fc)
        qs.append(np.concatenate([[np.cos(th0)], np.sin(th0) * d / r]))
    cs, qs = np.array(cs), np.array(qs)
    G = np.clip(qs @ qs.T, -1, 1)
    return np.array([cs.sum() * (cs @ eval_chebyu(j, G) @ cs) for j in range(twojmax + 1)]), len(nb)


@pytest.mark.parametrize("case", ["cubic_small", "triclinic_mixed_pbc", "cluster"])
def test_chebyshev_closed_form_for_Bj0j(case):
    rng = np.random.default_rng(11)
    if case == "cubic_small":
        box, pbc = np.eye(3) * 4.05, (1, 1, 1)
        pos = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]]) * 4.05 + 0.05 * rng.normal(size=(4, 3))
        types, radelem, wj, rcutfac = [0] * 4, (0.5,), (1.0,), 4.676
    elif case == "triclinic_mixed_pbc":
        box, pbc = np.array([[5.0, 0.3, 0.0], [1.0, 4.5, 0.2], [0.0, -0.6, 6.0]]), (1, 0, 1)
        pos = rng.uniform(-0.3, 1.3, size=(6, 3)) @ box       # unwrapped on purpose
        types, radelem, wj, rcutfac = [0, 1, 1, 0, 1, 0], (0.5, 0.45), (1.0, 0.8), 4.2
    else:
        box, pbc = BIG, (0, 0, 0)
        pos = cluster(rng, 12, 3.5) + 25.0
        types, radelem, wj, rcutfac = [0] * 12, (0.5,), (1.0,), 4.0
    rcut_t = [2 * rcutfac * x for x in radelem]
    origin = np.array([0.1, -0.2, 0.05]) if case == "triclinic_mixed_pbc" else np.zeros(3)
    pts = origin + rng.uniform(0, 1, size=(5, 3)) @ box if case != "cluster" else 25.0 + rng.normal(size=(5, 3))
    r = oracle.bispectrum_points(pts, pos, types, box, origin=origin, pbc=pbc, rcutfac=rcutfac, radelem=radelem, wj=wj)
    tr = r["triples"]
    idx = [int(np.where((tr[:, 0] == j) & (tr[:, 1] == 0) & (tr[:, 2] == j))[0][0]) for j in range(11)]
    for p, B, nn in zip(pts, r["B"], r["nnbr"]):
        ref, n_ref = chebyshev_bj0j(p, pos, types, box, origin, pbc, rcut_t, wj, 1.0, 10)
        assert nn == n_ref and nn > 0
        np.testing.assert_allclose(B[idx], ref, rtol=1e-11)


def test_rmin0_branch_B000_and_Bj0j_closed_forms():
    """reading #22 (rmin0 != 0): f_c = 1 and theta0 < 0 for a neighbor inside rmin0.  Pinned by the two closed forms with an
    independent numpy neighbor list: B_000 = (wself + sum w f_c)^3 sees the saturation of f_c, the Chebyshev form of
    B_{j,0,j} sees the sign of theta0 through the quaternion dot products with the other neighbors."""
    rng = np.random.default_rng(21)
    rmin0, rcutfac, wself = 0.3, 3.9, 1.3
    radelem, wj = (0.5, 0.4), (1.0, 0.6)
    rcut_t = [2 * rcutfac * x for x in radelem]
    pts = np.array([[25.0, 25.0, 25.0], [25.4, 24.8, 25.1]])
    # neighbors of the first point: one inside rmin0 (r = 0.2), one just outside (0.31), the rest spread up to the cutoff
    near = np.array([[0.12, -0.1, 0.12], [0.2, 0.2, -0.126]])
    assert abs(np.linalg.norm(near[0]) - 0.197) < 1e-3 and 0.3 < np.linalg.norm(near[1]) < 0.32
    pos = np.concatenate([pts[0] + near, pts[0] + cluster(rng, 9, 3.0)])
    types = [0, 1] + [int(t) for t in rng.integers(0, 2, 9)]
    r = oracle.bispectrum_points(pts, pos, types, BIG, pbc=(0, 0, 0), rcutfac=rcutfac, wself=wself, radelem=radelem, wj=wj,
                                 rmin0=rmin0)
    tr = r["triples"]
    idx = [int(np.where((tr[:, 0] == j) & (tr[:, 1] == 0) & (tr[:, 2] == j))[0][0]) for j in range(11)]
    for p, B, nn in zip(pts, r["B"], r["nnbr"]):
        nb = brute_neighbors(p, pos, types, BIG, np.zeros(3), (0, 0, 0), rcut_t)
        assert nn == len(nb) >= 6
        s = wself + sum(wj[t] * fc_theta(np.linalg.norm(d), rcut_t[t], rmin0)[0] for d, t in nb)
        np.testing.assert_allclose(B[0], s ** 3, rtol=1e-13)
        ref, _ = chebyshev_bj0j(p, pos, types, BIG, np.zeros(3), (0, 0, 0), rcut_t, wj, wself, 10, rmin0)
        np.testing.assert_allclose(B[idx], ref, rtol=1e-11)
    # the test can tell the readings apart: clamping theta0 at 0 inside rmin0 changes B_{j,0,j} of the first point
    nb = brute_neighbors(pts[0], pos, types, BIG, np.zeros(3), (0, 0, 0), rcut_t)
    cs, qs = [wself], [np.array([1.0, 0, 0, 0])]
    for d, t in nb:
        rr = np.linalg.norm(d)
        fc, th0 = fc_theta(rr, rcut_t[t], rmin0)
        th0 = max(th0, 0.0)
        cs.append(wj[t] * fc)
        qs.append(np.concatenate([[np.cos(th0)], np.sin(th0) * d / rr]))
    cs, qs = np.array(cs), np.array(qs)
    clamped = np.array([cs.sum() * (cs @ eval_chebyu(j, np.clip(qs @ qs.T, -1, 1)) @ cs) for j in range(11)])
    assert np.abs(clamped - r["B"][0][idx]).max() > 1e-3 * np.abs(clamped).max()
    # a neighbor at r < rmin0 with wself = 0 and nothing else: (w * 1)^3 (j + 1), any direction (single-neighbor closed form)
    one = oracle.bispectrum_points([[0, 0, 0]], [[0.1, 0.05, -0.12]], [0], BIG, pbc=(0, 0, 0), wself=0.0, wj=(0.8,), rmin0=rmin0)
    np.testing.assert_allclose(one["B"][0], 0.8 ** 3 * (one["triples"][:, 2] + 1), rtol=2e-12)


def test_chebyshev_grid_oracle_agrees_with_the_wigner_cg_path():
    """oracle.bj0j_grid (closed form, C) is the second oracle of the full-size GPU tests: here it is tied to the main path
    (explicit Wigner-D + Racah CG) on a whole tiny-Al grid and on a two-type triclinic mixed-pbc slab"""
    from paper_2411_19617_b200 import workloads
    w = workloads.make(1)
    tr = oracle.triples(10)
    idx = [int(np.where((tr[:, 0] == j) & (tr[:, 1] == 0) & (tr[:, 2] == j))[0][0]) for j in range(11)]
    ref = oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 0, 6, **w.snap_params())
    ch = oracle.bj0j_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, 0, 6, **w.snap_params())
    np.testing.assert_allclose(ch, ref[:, idx], rtol=1e-11)
    rng = np.random.default_rng(12)
    box = np.array([[5.0, 0.3, 0.0], [1.0, 4.5, 0.2], [0.0, -0.6, 6.0]])
    pos = rng.uniform(-0.3, 1.3, size=(6, 3)) @ box
    kw = dict(twojmax=6, rcutfac=4.2, radelem=(0.5, 0.45), wj=(1.0, 0.8), wself=0.7, rmin0=0.2)
    tr6 = oracle.triples(6)
    idx6 = [int(np.where((tr6[:, 0] == j) & (tr6[:, 1] == 0) & (tr6[:, 2] == j))[0][0]) for j in range(7)]
    ref = oracle.bispectrum_grid(pos, [0, 1, 1, 0, 1, 0], box, (0.1, -0.2, 0.05), (1, 0, 1), (5, 4, 6), 1, 5, **kw)
    ch = oracle.bj0j_grid(pos, [0, 1, 1, 0, 1, 0], box, (0.1, -0.2, 0.05), (1, 0, 1), (5, 4, 6), 1, 5, **kw)
    np.testing.assert_allclose(ch, ref[:, idx6], rtol=1e-11)


def test_atom_exactly_on_grid_point_uses_continuous_limit():
    # reading #11: r -> 0 contributes w * I
    r = oracle.bispectrum_points([[2.0, 2.0, 2.0]], [[2.0, 2.0, 2.0]], [0], BIG, pbc=(0, 0, 0), wj=(0.5,))
    np.testing.assert_allclose(r["B"][0], 1.5 ** 3 * (r["triples"][:, 2] + 1), rtol=1e-14)
    r2 = oracle.bispectrum_points([[2.0, 2.0, 2.0]], [[2.0, 2.0, 2.0 + 1e-7]], [0], BIG, pbc=(0, 0, 0), wj=(0.5,))
    np.testing.assert_allclose(r2["B"][0], r["B"][0], rtol=1e-9)


def test_continuity_across_cutoff():
    rc = 4.676
    others = [[1.0, 1.5, -2.0], [-2.0, 0.5, 1.0]]
    inside = oracle.bispectrum_points([[0, 0, 0]], others + [[0, 0, rc * (1 - 1e-7)]], [0] * 3, BIG, pbc=(0, 0, 0),
                                      rcutfac=rc)
    outside = oracle.bispectrum_points([[0, 0, 0]], others + [[0, 0, rc * (1 + 1e-7)]], [0] * 3, BIG, pbc=(0, 0, 0),
                                       rcutfac=rc)
    assert inside["nnbr"][0] == 3 and outside["nnbr"][0] == 2
    np.testing.assert_allclose(inside["B"][0], outside["B"][0], rtol=1e-10)


# ----------------------------------------------------------------------------------------------
# symmetries of B
# ----------------------------------------------------------------------------------------------
def test_index_permutation_symmetries():
    rng = np.random.default_rng(5)
    pos = cluster(rng, 9, 4.0) + 25
    tj = 6
    tl = [(j1, j2, j) for j1 in range(tj + 1) for j2 in range(tj + 1) for j in range(abs(j1 - j2), min(tj, j1 + j2) + 1, 2)]
    r = oracle.bispectrum_points([[25, 25, 25]], pos, [0] * 9, BIG, pbc=(0, 0, 0), twojmax=tj, triple_list=tl,
                                 want_imag=True)
    B = {t: v for t, v in zip(tl, r["B"][0])}
    scale = np.abs(r["B"][0]).max()
    assert np.abs(r["imag"][0]).max() < 1e-13 * scale           # "real-valued" PAPER.md:261
    n = 0
    for (j1, j2, j) in tl:
        assert abs(B[(j1, j2, j)] - B[(j2, j1, j)]) < 1e-12 * scale
        assert abs(B[(j1, j2, j)] / (j + 1) - B[(j, j2, j1)] / (j1 + 1)) < 1e-12 * scale
        n += 1
    assert n > 100


def _B(pts, pos, **kw):
    return oracle.bispectrum_points(pts, pos, [0] * len(pos), kw.pop("box", BIG), pbc=kw.pop("pbc", (0, 0, 0)), **kw)["B"]


def test_rotation_reflection_permutation_invariance():
    rng = np.random.default_rng(6)
    c = np.array([25.0, 24.0, 26.0])
    rel = cluster(rng, 14, 4.3)
    B0 = _B([c], c + rel)[0]
    scale = np.abs(B0).max()
    assert np.ptp(B0) > 1.0
    R = rot_matrix(rng)
    np.testing.assert_allclose(_B([c], c + rel @ R.T)[0], B0, atol=1e-12 * scale)      # "rotationally invariant"
    np.testing.assert_allclose(_B([c], c + rel * [1, 1, -1])[0], B0, atol=1e-12 * scale)
    np.testing.assert_allclose(_B([c], c - rel)[0], B0, atol=1e-12 * scale)
    np.testing.assert_allclose(_B([c], c + rel[rng.permutation(14)])[0], B0, atol=1e-12 * scale)
    # and B does change when the environment really changes
    rel2 = rel.copy()
    rel2[0] *= 0.8
    assert np.abs(_B([c], c + rel2)[0] - B0).max() > 1e-3 * scale


def test_translation_invariances_periodic():
    rng = np.random.default_rng(8)
    box = np.array([[4.4, 0, 0], [0.5, 4.0, 0], [0.2, -0.3, 4.8]])
    pos = rng.uniform(0, 1, size=(5, 3)) @ box
    pts = rng.uniform(0, 1, size=(3, 3)) @ box
    kw = dict(box=box, pbc=(1, 1, 1), rcutfac=4.2)
    B0 = _B(pts, pos, **kw)
    scale = np.abs(B0).max()
    pos2 = pos.copy()
    pos2[1] += 2 * box[0] - box[2]
    pos2[3] -= 3 * box[1]
    np.testing.assert_allclose(_B(pts, pos2, **kw), B0, atol=1e-12 * scale)          # lattice translation of atoms
    t = np.array([0.37, -1.2, 0.81])
    Bt = oracle.bispectrum_points(pts + t, pos + t, [0] * 5, box, origin=t, pbc=(1, 1, 1), rcutfac=4.2)["B"]
    np.testing.assert_allclose(Bt, B0, atol=1e-12 * scale)                            # atoms + origin together
    np.testing.assert_allclose(_B(pts + box[1], pos, **kw), B0, atol=1e-12 * scale)   # grid point by a lattice vector


def test_grid_layout_and_slab_split():
    rng = np.random.default_rng(9)
    box = np.array([[4.0, 0, 0], [0.3, 4.2, 0], [0, 0.1, 3.9]])
    pos = rng.uniform(0, 1, size=(3, 3)) @ box
    origin = np.array([0.2, 0.0, -0.1])
    ng = (3, 4, 5)
    kw = dict(twojmax=4, rcutfac=3.5)
    full = oracle.bispectrum_grid(pos, [0] * 3, box, origin, (1, 1, 0), ng, **kw)
    assert full.shape == (60, 14)
    a = oracle.bispectrum_grid(pos, [0] * 3, box, origin, (1, 1, 0), ng, 0, 2, **kw)
    b = oracle.bispectrum_grid(pos, [0] * 3, box, origin, (1, 1, 0), ng, 2, 5, **kw)
    np.testing.assert_array_equal(np.vstack([a, b]), full)
    # point (ix,iy,iz) sits at origin + ix/nx a1 + iy/ny a2 + iz/nz a3, ix fastest
    ix, iy, iz = 2, 3, 4
    p = origin + ix / 3 * box[0] + iy / 4 * box[1] + iz / 5 * box[2]
    one = oracle.bispectrum_points([p], pos, [0] * 3, box, origin=origin, pbc=(1, 1, 0), **kw)["B"][0]
    np.testing.assert_allclose(full[(iz * 4 + iy) * 3 + ix], one, rtol=1e-13)
    smp = oracle.bispectrum_grid(pos, [0] * 3, box, origin, (1, 1, 0), ng, 1, 5, sample=[0, 7, 47], **kw)
    np.testing.assert_array_equal(smp, full[12:][[0, 7, 47]])


def test_U_reflection_symmetry_and_self_term():
    rng = np.random.default_rng(10)
    pos = cluster(rng, 7, 4.0) + 25
    r = oracle.bispectrum_points([[25, 25, 25]], pos, [0] * 7, BIG, pbc=(0, 0, 0), want_U=True, wself=1.0)
    U = r["U"][0]
    for J in range(11):
        UJ = U[oracle.uoff(J):oracle.uoff(J + 1)].reshape(J + 1, J + 1)
        sgn = (-1.0) ** (np.arange(J + 1)[:, None] - np.arange(J + 1)[None, :])
        np.testing.assert_allclose(UJ[::-1, ::-1], sgn * UJ.conj(), atol=1e-13)
