"""The exact symmetries the CUDA contraction kernels use to skip work, checked here with the
oracle's Wigner-D and Clebsch-Gordan values only (no CUDA): the contribution of an "item" (output column mb, factor
columns mb1 and mb2 = mb + sh - mb1) to B_{j1 j2 j},

    b(mb, mb1) = Re sum_ma conj(U^j[ma][mb]) * CG(mb1, mb2) * sum_{ma1 + ma2 - sh = ma} CG(ma1, ma2) U^{j1}[ma1][mb1] U^{j2}[ma2][mb2],

satisfies  (F) b(mb, mb1) = b(J - mb, J1 - mb1)   column flip (half-column storage),
           (S) j1 == j2:  b(mb, mb1) = b(mb, mb2)  the two factors swapped,
           (H) j == j1:   b(mb, mb1) = b(mb1, mb)  output and first factor swapped,
           (S3) j1 == j2 == j: b depends only on the class of (mu1, mu2, mu3) = (mb1 - J/2, mb2 - J/2, J/2 - mb) under
                permutations and a common sign change; the class sizes are the weights of the anti-diagonal kernel.
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402


@pytest.fixture(scope="module")
def utot():
    rng = np.random.default_rng(3)
    tj = 8
    U = {J: np.eye(J + 1, dtype=complex) for J in range(tj + 1)}
    for d in rng.normal(size=(12, 3)) * 1.5:
        ok, a, b, c = oracle.pair(d, 4.676)
        if ok:
            for J in range(tj + 1):
                U[J] = U[J] + c * oracle.wigner_D(J, a, b)
    return U


def item_b(U, J1, J2, J, mb, mb1):
    sh = (J1 + J2 - J) // 2
    mb2 = mb + sh - mb1
    if not (0 <= mb2 <= J2):
        return None

    def cg(m1, m2):
        m = m1 + m2 - sh
        return oracle.cg(J1, 2 * m1 - J1, J2, 2 * m2 - J2, J, 2 * m - J) if 0 <= m <= J else 0.0

    z = np.zeros(J + 1, dtype=complex)
    for ma1 in range(J1 + 1):
        for ma2 in range(J2 + 1):
            ma = ma1 + ma2 - sh
            if 0 <= ma <= J:
                z[ma] += cg(ma1, ma2) * U[J1][ma1, mb1] * U[J2][ma2, mb2]
    return float((cg(mb1, mb2) * np.conj(U[J][:, mb]) @ z).real)


@pytest.mark.parametrize("triple", [(8, 4, 8), (7, 2, 7), (5, 4, 5), (6, 6, 8), (4, 4, 4), (7, 5, 8), (8, 3, 7)])
def test_item_symmetries(utot, triple):
    J1, J2, J = triple
    sh = (J1 + J2 - J) // 2
    scale = max(abs(item_b(utot, J1, J2, J, mb, mb1) or 0.0) for mb in range(J + 1) for mb1 in range(J1 + 1))
    checked = 0
    for mb in range(J + 1):
        for mb1 in range(J1 + 1):
            x = item_b(utot, J1, J2, J, mb, mb1)
            if x is None:
                continue
            assert abs(x - item_b(utot, J1, J2, J, J - mb, J1 - mb1)) < 1e-12 * scale          # (F)
            if J1 == J2:
                assert abs(x - item_b(utot, J1, J2, J, mb, mb + sh - mb1)) < 1e-12 * scale      # (S)
            if J == J1:
                assert abs(x - item_b(utot, J1, J2, J, mb1, mb)) < 1e-12 * scale                # (H)
            checked += 1
    assert checked > 10


@pytest.mark.parametrize("J", [2, 4, 6])
def test_fully_symmetric_triples_have_s3_classes(utot, J):
    sh = J // 2
    classes = {}
    for mb in range(J + 1):
        for mb1 in range(J + 1):
            x = item_b(utot, J, J, J, mb, mb1)
            if x is None:
                continue
            mu = (mb1 - J // 2, mb + sh - mb1 - J // 2, J // 2 - mb)
            key = min(tuple(sorted(mu)), tuple(sorted(-m for m in mu)))
            classes.setdefault(key, []).append(x)
    scale = max(abs(v) for vals in classes.values() for v in vals)
    for key, vals in classes.items():
        assert max(vals) - min(vals) < 1e-12 * scale
        m1, m2, m3 = key
        perms = 1 if m1 == m2 == m3 else (3 if (m1 == m2 or m2 == m3) else 6)
        both = 1 if sorted(key)[1] == 0 else 2
        assert perms * both == len(vals)          # the weight the kernel gives the class representative
    # the representative the kernel computes: mu1 <= mu2 <= mu3, mu2 <= 0  <=>  mb <= mb1 <= (mb + J/2) / 2, mb <= J/2
    kept = set()
    for mb in range(J // 2 + 1):
        for mb1 in range(mb, (mb + sh) // 2 + 1):
            mu = (mb1 - J // 2, mb + sh - mb1 - J // 2, J // 2 - mb)
            assert mu[0] <= mu[1] <= mu[2] and mu[1] <= 0
            kept.add(min(tuple(sorted(mu)), tuple(sorted(-m for m in mu))))
    assert kept == set(classes)
