// snap_common.cuh -- structures shared by the host planner and the kernels.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "snap_tables.h"

namespace mala {

constexpr int kTilePoints = 32;  // grid points per tile = lanes of a warp ("lanes as points")
constexpr int kMaxTwoJ = 14;      // largest supported twojmax
constexpr int kFullTileTwoJ = 10;  // up to here U_tot of a whole 32-point tile fits one SM's shared memory; above it the
                                   // contraction works on half tiles (16 points) and U_tot is stored half tile by half tile

// Geometry of one slab call, passed by value to every kernel.
struct GridGeom {
    double a1[3], a2[3], a3[3], origin[3];  // cell rows and the position of grid point (0,0,0)
    int nx, ny, nz;                          // grid
    int z0, z1;                              // slab [z0, z1) handled by this launch sequence
    // The slab is covered by up to four regions in (x, y), each tiled by its own 32-point brick: the part the main brick
    // covers exactly, the strips left over along x and along y, and their corner.  A grid whose extents are not
    // multiples of the brick (90 = 22 * 4 + 2) then wastes lanes only where the strips are ragged themselves.
    int nreg;
    struct Region {
        int x0, y0, nxr, nyr;                // first point and extent of the region
        int tx, ty, tz;                      // tile shape in points, tx*ty*tz == 32
        int ntx, nty, ntz;                   // tiles per axis (ntz counts from z0)
        int tile_begin;                      // id of the region's first tile
        int pad;
        double tile_radius;                  // bounding-sphere radius of one tile around its centre
    } reg[4];
    double tile_radius;                      // largest of the regions' radii (host-side candidate bound)
    int total_tiles;
    // Cartesian cell list over the ghost atoms
    double cell_lo[3], cell_inv[3];
    int ncx, ncy, ncz;
    double rcutmax;
};

struct SnapConst {
    int twojmax, ntriples, nelem, ntypes;
    double rfac0, rmin0, wself;
};

// one ghost atom (an atom or one of its periodic images): position and type, 32 bytes
struct __align__(16) Ghost {
    double x, y, z;
    int type;
    int pad;   // index of the atom this ghost is an image of (row f3 scatters the adjoint back to atoms)
};

// device pointers of one handle
struct DeviceTables {
    const int *triples;      // [ntriples*4] j1, j2, j, cg offset
    const double *cg;        // dense CG blocks
    const double *unorm;     // [nelem]
    const int *udiag;        // [nelem]
    const int *order;        // [ntriples] cost-sorted work order
    const double *type_rcut; // [ntypes]
    const double *type_w;    // [ntypes]
    const double *bconst;    // [ntriples] zero-neighbor descriptor
};

// per-chunk work buffers
struct ChunkBuffers {
    const Ghost *ghosts;     // sorted by cell
    const int *cell_start;   // [ncells+1]
    int *cand;               // [chunk_tiles * cand_cap] ghost indices per tile
    int *ncand;              // [chunk_tiles]
    int *active;             // [chunk_tiles] compacted list of non-empty tiles (local tile ids)
    int *counters;           // [0] number of active tiles, [1] ui work counter, [2] zi / yi work counter, [3] dedr work counter
                             // (zeroed per chunk)
    int *status;             // handle-wide status word, never cleared by a chunk: kStatus* bits
    double2 *utot;           // [chunk_tiles][nelem][32], or [chunk_tiles][2][nelem][16] when utot_half is set
    int utot_half;           // 1: half-tile layout (twojmax > kFullTileTwoJ)
    int compact_out;         // 1: descriptors go to out[(local tile) * 32 + lane][ncomp] (staging for the fused network)
                             //    instead of out[grid point][ncomp]
    int cand_cap;
    double *ui_spill;        // compute_ui_pipe_kernel: per CTA, the pair geometry of the first ui_spill_windows windows of a tile that
    int ui_spill_windows;    // comes in several (kept for the later accumulation passes); nullptr / 0: every pass prepares them again
    int tile_begin;          // first global tile id of the chunk
    int ntiles;              // tiles in the chunk
};

constexpr int kStatusCandOverflow = 1;  // tile_bin_kernel had to truncate a candidate list (host bound violated)

// one tile: its first grid point, its shape, and the end of its region (points beyond it do not belong to the tile)
struct TileInfo {
    int ix0, iy0, iz0, tx, ty, tz, xend, yend;
    double radius;
};

__host__ __device__ inline TileInfo tile_info(const GridGeom &g, int tile) {
    int r = 0;
    while (r + 1 < g.nreg && tile >= g.reg[r + 1].tile_begin) r++;
    const GridGeom::Region &R = g.reg[r];
    int t = tile - R.tile_begin;
    const int txi = t % R.ntx;
    t /= R.ntx;
    const int tyi = t % R.nty, tzi = t / R.nty;
    TileInfo ti;
    ti.ix0 = R.x0 + txi * R.tx; ti.iy0 = R.y0 + tyi * R.ty; ti.iz0 = g.z0 + tzi * R.tz;
    ti.tx = R.tx; ti.ty = R.ty; ti.tz = R.tz;
    ti.xend = R.x0 + R.nxr; ti.yend = R.y0 + R.nyr;
    ti.radius = R.tile_radius;
    return ti;
}

// grid point of lane `lane` of tile `tile` (bricks are filled x fastest); valid = the point exists (ragged tiles, slab end)
__host__ __device__ inline void lane_point(const GridGeom &g, int tile, int lane, int &ix, int &iy, int &iz, bool &valid) {
    const TileInfo ti = tile_info(g, tile);
    const int lx = lane % ti.tx, ly = (lane / ti.tx) % ti.ty, lz = lane / (ti.tx * ti.ty);
    ix = ti.ix0 + lx;
    iy = ti.iy0 + ly;
    iz = ti.iz0 + lz;
    valid = (ix < ti.xend) && (iy < ti.yend) && (iz < g.z1);
}


}  // namespace mala
