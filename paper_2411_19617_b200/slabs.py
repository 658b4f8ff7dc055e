"""z-slab partition of a grid over independent workers.

Grid points are independent given the atom list, so several GPUs share one grid by calling
`mala_bispectrum_grid` on disjoint `[z_begin, z_end)` ranges with the atoms replicated; nothing is exchanged.
Host-side index arithmetic only.
"""


def z_slabs(nz, nparts):
    """Contiguous, disjoint, near-equal slabs [(z_begin, z_end), ...] covering [0, nz); empty slabs when nparts > nz."""
    if nz < 0 or nparts < 1:
        raise ValueError("nz must be >= 0 and nparts >= 1")
    base, extra = divmod(nz, nparts)
    out, z = [], 0
    for r in range(nparts):
        n = base + (1 if r < extra else 0)
        out.append((z, z + n))
        z += n
    return out


def weighted_z_slabs(plane_cost, nparts):
    """Slabs balanced by a per-plane cost (e.g. the number of non-empty points of each z-plane of a cluster in
    vacuum): boundaries at the planes where the running cost crosses k/nparts of the total."""
    nz = len(plane_cost)
    total = float(sum(plane_cost))
    if total <= 0.0:
        return z_slabs(nz, nparts)
    out, z, run = [], 0, 0.0
    for r in range(nparts):
        target = total * (r + 1) / nparts
        z0 = z
        while z < nz and (r == nparts - 1 or run + 0.5 * plane_cost[z] <= target):
            run += plane_cost[z]
            z += 1
        out.append((z0, z))
    return out
