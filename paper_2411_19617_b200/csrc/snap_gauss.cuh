// snap_gauss.cuh -- Gaussian descriptors on the grid (Eqs. (40)-(43) PAPER.md:396-412).
//
// Reading: one channel per atom type,
//     G_t(r) = w_t (2 pi sigma^2)^(-3/2) sum exp(-|R - r|^2 / (2 sigma^2))
// over the atoms of type t and their periodic images with |R - r| < rcut_t.  Same ghost list, cell list and per-tile
// candidate lists as the bispectrum path (tile_bin_kernel); lane = grid point, one warp per 32-point tile.
// HBM-bound on the output (8 ntypes bytes per point); the pair work is ~45 FP64 instructions.
#pragma once
#include "snap_common.cuh"
#include "snap_ui.cuh"

namespace mala {

constexpr int kGaussMaxTypes = 4;

__global__ void __launch_bounds__(256) gaussian_grid_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb,
                                                            double inv2s2, double pref, double *out) {
    const int lane = threadIdx.x & 31;
    const int wt = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    if (wt >= cb.ntiles) return;
    const int tile = cb.tile_begin + wt;
    int ix, iy, iz;
    bool valid;
    lane_point(g, tile, lane, ix, iy, iz, valid);
    const int cx = min(ix, g.nx - 1), cy = min(iy, g.ny - 1), cz = min(iz, g.z1 - 1);
    double px, py, pz;
    point_position(g, cx, cy, cz, px, py, pz);
    double acc[kGaussMaxTypes];
#pragma unroll
    for (int t = 0; t < kGaussMaxTypes; t++) acc[t] = 0.0;
    const int nc = cb.ncand[wt];
    const int *mycand = cb.cand + (size_t)wt * cb.cand_cap;
    for (int base = 0; base < nc; base += 32) {
        // one candidate per lane, broadcast to the warp
        Ghost mine = {0.0, 0.0, 0.0, 0, 0};
        if (base + lane < nc) mine = cb.ghosts[mycand[base + lane]];
        const int nb = min(32, nc - base);
        for (int k = 0; k < nb; k++) {
            const double gx = __shfl_sync(0xffffffffu, mine.x, k), gy = __shfl_sync(0xffffffffu, mine.y, k);
            const double gz = __shfl_sync(0xffffffffu, mine.z, k);
            const int ty = __shfl_sync(0xffffffffu, mine.type, k);
            const double dx = gx - px, dy = gy - py, dz = gz - pz;
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (sqrt(r2) < tb.type_rcut[ty]) {
                const double v = tb.type_w[ty] * pref * exp(-r2 * inv2s2);
#pragma unroll
                for (int t = 0; t < kGaussMaxTypes; t++) acc[t] += (t == ty) ? v : 0.0;
            }
        }
    }
    if (!valid) return;
    double *dst = out + ((size_t)((size_t)(iz - g.z0) * g.ny + iy) * g.nx + ix) * sc.ntypes;
#pragma unroll
    for (int t = 0; t < kGaussMaxTypes; t++)
        if (t < sc.ntypes) __stcs(dst + t, acc[t]);
}

}  // namespace mala
