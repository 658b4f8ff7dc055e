"""Seeded synthetic workloads (input generators only -- none of the method's arithmetic).

These stand in for the paper's Al / B / Be DFT snapshots (Tabs. 3-6), which
are not available; shapes follow BASELINE.json `configs` and SURVEY.md 8(d).  The arrays produced here are
handed unchanged to both the CUDA path and the CPU oracle (which never imports this module itself).

Every workload: twojmax=10, rfac0=0.99363, rmin0=0, wself=1, one atom type, radelem=0.5 (so rcut=rcutfac),
wj=1, origin=(0,0,0).  Gaussian displacements are per Cartesian component (reading #18 in DESIGN.md).
"""
from dataclasses import dataclass, field

import numpy as np


@dataclass
class Workload:
    name: str
    pos: np.ndarray            # [natoms,3] fp64, Angstrom
    types: np.ndarray          # [natoms] int32
    box: np.ndarray            # [3,3] rows a1,a2,a3
    pbc: tuple
    ngrid: tuple               # (nx,ny,nz)
    rcutfac: float
    origin: tuple = (0.0, 0.0, 0.0)
    twojmax: int = 10
    rfac0: float = 0.99363
    rmin0: float = 0.0
    wself: float = 1.0
    radelem: tuple = (0.5,)
    wj: tuple = (1.0,)
    seed: int = 0
    notes: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def npoints(self):
        return int(self.ngrid[0]) * int(self.ngrid[1]) * int(self.ngrid[2])

    def snap_params(self):
        return dict(twojmax=self.twojmax, rcutfac=self.rcutfac, rfac0=self.rfac0, rmin0=self.rmin0,
                    wself=self.wself, radelem=self.radelem, wj=self.wj)


class _Rng:
    """Uniform doubles from numpy's PCG64 stream + a hand-written Box-Muller, so the numbers do not depend
    on any library's normal-distribution algorithm."""

    def __init__(self, seed):
        self.g = np.random.Generator(np.random.PCG64(seed))

    def uniform(self, n=None):
        return self.g.random(n)

    def normal(self, shape):
        n = int(np.prod(shape))
        m = (n + 1) // 2
        u1 = 1.0 - self.g.random(m)      # (0,1]
        u2 = self.g.random(m)
        r = np.sqrt(-2.0 * np.log(u1))
        z = np.concatenate([r * np.cos(2 * np.pi * u2), r * np.sin(2 * np.pi * u2)])[:n]
        return z.reshape(shape)


_FCC = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]], dtype=np.float64)


def _fcc(ncell, a):
    cells = np.array([[i, j, k] for i in range(ncell) for j in range(ncell) for k in range(ncell)], dtype=np.float64)
    return ((cells[:, None, :] + _FCC[None, :, :]) * a).reshape(-1, 3)


def tiny_al(seed=1001):
    a = 4.05
    rng = _Rng(seed)
    pos = _fcc(1, a) + 0.05 * rng.normal((4, 3))
    return Workload("tiny_al", pos, np.zeros(4, np.int32), np.eye(3) * a, (1, 1, 1), (18, 18, 18), 4.676, seed=seed,
                    notes="4-atom fcc cell a=4.05, sigma=0.05, 18^3 grid; box < rcut so every atom has many images")


def solid_al(seed=1002, ngrid=(90, 90, 90)):
    a = 4.05
    rng = _Rng(seed)
    pos = _fcc(4, a) + 0.1 * rng.normal((256, 3))
    return Workload("solid_al", pos, np.zeros(256, np.int32), np.eye(3) * 4 * a, (1, 1, 1), tuple(ngrid), 4.676,
                    seed=seed, notes="256-atom 4x4x4 fcc Al, sigma=0.1, 90^3 grid (headline workload)")


def liquid_al(seed=1003, ngrid=(100, 100, 100)):
    n, rho, dmin = 256, 0.0530, 2.3
    L = (n / rho) ** (1.0 / 3.0)
    rng = _Rng(seed)
    pts = np.zeros((0, 3))
    while pts.shape[0] < n:
        p = rng.uniform(3) * L
        if pts.shape[0]:
            d = pts - p
            d -= L * np.round(d / L)
            if np.min(np.einsum("ij,ij->i", d, d)) < dmin * dmin:
                continue
        pts = np.vstack([pts, p])
    return Workload("liquid_al", pts, np.zeros(n, np.int32), np.eye(3) * L, (1, 1, 1), tuple(ngrid), 4.676, seed=seed,
                    notes="256 atoms by random sequential addition (min image distance 2.3), 0.0530 atoms/A^3, 100^3 grid")


def boron_cluster(seed=1004, ngrid=(160, 160, 160)):
    n, R, dmin, L = 40, 4.0, 1.6, 20.0
    rng = _Rng(seed)
    c = np.array([L / 2] * 3)
    pts = np.zeros((0, 3))
    while pts.shape[0] < n:
        p = (2 * rng.uniform(3) - 1) * R
        if p @ p > R * R:
            continue
        if pts.shape[0] and np.min(np.einsum("ij,ij->i", pts - (p + c), pts - (p + c))) < dmin * dmin:
            continue
        pts = np.vstack([pts, p + c])
    return Workload("boron_cluster", pts, np.zeros(n, np.int32), np.eye(3) * L, (0, 0, 0), tuple(ngrid), 4.0, seed=seed,
                    notes="40 atoms in a sphere R=4 (min distance 1.6) in a 20 A non-periodic box, 160^3 grid, ~79% empty points")


def be_slab(seed=1005, ncell=(16, 16, 16), spacing=0.2):
    a, c = 2.286, 3.584
    cell = np.array([a, np.sqrt(3.0) * a, c])
    basis = np.array([[0, 0, 0], [.5, .5, 0], [.5, 1 / 6, .5], [0, 2 / 3, .5]], dtype=np.float64)
    nxc, nyc, nzc = ncell
    pos = []
    half = nzc  # layer index 2*cz + (0|1); fault: layers >= nzc (the middle basal plane) shifted by +1/3 along y
    for cx in range(nxc):
        for cy in range(nyc):
            for cz in range(nzc):
                for b in basis:
                    f = np.array([cx, cy, cz], dtype=np.float64) + b
                    layer = 2 * cz + (1 if b[2] > 0.25 else 0)
                    if layer >= half:
                        f[1] += 1.0 / 3.0
                    pos.append(f * cell)
    pos = np.array(pos)
    rng = _Rng(seed)
    pos = pos + 0.05 * rng.normal(pos.shape)
    Ls = cell * np.array(ncell, dtype=np.float64)
    ngrid = tuple(int(round(x / spacing)) for x in Ls)
    return Workload("be_slab", pos, np.zeros(pos.shape[0], np.int32), np.diag(Ls), (1, 1, 1), ngrid, 4.5, seed=seed,
                    notes="hcp Be 16x16x16 orthorhombic cells (16,384 atoms), ...ABAB|CACA... fault at the middle basal "
                          "plane (reading #19), sigma=0.05, grid spacing ~0.2 A")


def solid_al_200(seed=1002):
    """paper-scale grid for the same 256-atom cell: 200^3 = 8.0e6 points (Tab. 5)"""
    w = solid_al(seed, ngrid=(200, 200, 200))
    w.name = "solid_al_200cube"
    w.notes = "256-atom 4x4x4 fcc Al, sigma=0.1, 200^3 grid (8.0e6 points: the grid of the paper's 256-atom Al runs, Tab. 5)"
    return w


def binary_alloy(seed=1006, ngrid=(90, 90, 90)):
    """two species with distinct radii and weights (PAPER.md:252 per-species cutoff R^eta, weights w_eta of Eq. (24)):
    the 256-site fcc cell of config 2 with every site assigned type 0 or 1 by a seeded coin; rcut = 4.676 / 3.74 A."""
    a = 4.05
    rng = _Rng(seed)
    pos = _fcc(4, a) + 0.1 * rng.normal((256, 3))
    types = (rng.uniform(256) < 0.5).astype(np.int32)
    return Workload("binary_alloy", pos, types, np.eye(3) * 4 * a, (1, 1, 1), tuple(ngrid), 4.676, radelem=(0.5, 0.4), wj=(1.0, 0.6),
                    seed=seed, notes="256-site fcc cell, two species by a seeded coin: radelem (0.5, 0.4), wj (1.0, 0.6), 90^3 grid")


def ldos_network(seed=2001, sizes=(91, 256, 256, 241), in_scale=0.02):
    """Seeded synthetic weights of a descriptor -> LDOS network: the paper's trained models are not
    available, so every W_l is N(0, 2 / w_l) and every b_l is N(0, 0.1^2) (hand-written Box-Muller); 241 outputs as in
    PAPER.md:542.  The input scaling is the same constant for every feature: x_0 = in_scale * B, which puts the
    descriptors of the Al configs into the range [0, 5].  Returns (weights, biases, in_shift, in_scale) as fp64 arrays."""
    rng = _Rng(seed)
    ws, bs = [], []
    for wk, wn in zip(sizes[:-1], sizes[1:]):
        ws.append(rng.normal((wn, wk)) * np.sqrt(2.0 / wk))
        bs.append(0.1 * rng.normal((wn,)))
    return ws, bs, np.zeros(sizes[0]), np.full(sizes[0], float(in_scale))


CONFIGS = {
    1: tiny_al, 2: solid_al, 3: liquid_al, 4: boron_cluster, 5: be_slab,
    "tiny_al": tiny_al, "solid_al": solid_al, "liquid_al": liquid_al, "boron_cluster": boron_cluster, "be_slab": be_slab,
    "200cube": solid_al_200, "binary": binary_alloy,
}


def make(config, twojmax=None, **kw):
    """config: 1..5 (BASELINE.json `configs`), "200cube" or "binary"; twojmax overrides the default 10."""
    w = CONFIGS[config](**kw)
    if twojmax is not None:
        w.twojmax = int(twojmax)
    return w
