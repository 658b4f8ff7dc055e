// snap_internal.h -- declarations shared by the translation units of libmala_snap.so (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>

#include <string>

#include "snap_common.cuh"

struct mala_mlp;

namespace mala {

// records the thread-local message behind mala_last_error() and returns `code`
int set_error(int code, const std::string &msg);

// Where the rows of one mlp_forward launch come from and go to.
//   plain:   row r reads x[r][w_in] and writes y[r][w_out]                                   (mala_mlp_forward)
//   compact: row r = (local tile) * 32 + lane of a chunk of grid tiles; reads x[r][w_in] (the compact descriptor
//            staging written by compute_zi_bi) and writes y[point][w_out] at the grid point the lane stands for;
//            lanes beyond a ragged tile are skipped                                           (mala_bispectrum_ldos_grid)
struct MlpRows {
    long long nrows;
    const double *x;
    float *y;
    int compact;
    int tile_begin;
    GridGeom geom;
};

// enqueue the network on `st`; returns 0 or a MALA_SNAP_* code (message recorded)
int mlp_launch(const mala_mlp *net, const MlpRows &rows, cudaStream_t st);
int mlp_in_width(const mala_mlp *net);
int mlp_out_width(const mala_mlp *net);

}  // namespace mala
