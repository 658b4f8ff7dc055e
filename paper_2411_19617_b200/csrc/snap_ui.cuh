// snap_ui.cuh -- tile binning (row a2) and the compute_ui kernel (rows a3 + a4 of SURVEY.md 8(a)).
//
// compute_ui accumulates, for the 32 grid points of a tile, U_tot^J = wself*I + sum_neighbors c * U^J(neighbor)
// (Eq. (24)-(25)) in the half-column storage of snap_tables.h.
//
// Formulation used here (differs from the textbook root-weighted recursion):
// with u^J[ma][mb] = sqrt(C(J,mb)/C(J,ma)) * q^J[ma][mb], column mb of level J is the coefficient list of the
// polynomial  Q_{J,mb}(x) = (b + a x)^mb * (conj(a) - conj(b) x)^(J-mb),  a, b the Cayley-Klein parameters of the
// neighbor.  So one column is advanced from level to level by multiplying with a linear factor -- no square
// roots, no coupling between columns -- and the binomial weights are applied once per tile at the end.
// Thread = (grid point, column): warp m owns column m of every level for the 32 points, so accumulation into
// shared memory needs no atomics and is deterministic.  Two neighbors are advanced together to halve the
// shared-memory read-modify-write traffic.
#pragma once
#include "snap_common.cuh"

namespace mala {

constexpr int kGeoCap = 48;     // neighbor entries per grid point buffered between two accumulate passes
constexpr int kUiPoints = 16;   // grid points per compute_ui CTA: half a tile; lane = (point, half), the halves split the neighbors

__device__ __forceinline__ void point_position(const GridGeom &g, int ix, int iy, int iz, double &x, double &y, double &z) {
    const double fx = (double)ix / (double)g.nx, fy = (double)iy / (double)g.ny, fz = (double)iz / (double)g.nz;
    x = g.origin[0] + fx * g.a1[0] + fy * g.a2[0] + fz * g.a3[0];
    y = g.origin[1] + fx * g.a1[1] + fy * g.a2[1] + fz * g.a3[1];
    z = g.origin[2] + fx * g.a1[2] + fy * g.a2[2] + fz * g.a3[2];
}

// ---------------------------------------------------------------------------------------------------------
// tile_bin_kernel: one warp per tile.  Collects the ghost atoms that can reach any point of the tile
// (|R - centre| < tile_radius + rcut_type) from the Cartesian cell list, in a deterministic order.
// Tiles with no candidate are filled with the constant zero-neighbor descriptor right here; the others are
// appended to the active list consumed by compute_ui / compute_zi_bi.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) tile_bin_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb, double *out) {
    const int lane = threadIdx.x & 31;
    const int wt = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    if (wt >= cb.ntiles) return;
    const int tile = cb.tile_begin + wt;
    const TileInfo ti = tile_info(g, tile);
    // tile centre (fractional mid-point of the full tile, also for ragged tiles: conservative)
    const double fx = (ti.ix0 + 0.5 * (ti.tx - 1)) / (double)g.nx;
    const double fy = (ti.iy0 + 0.5 * (ti.ty - 1)) / (double)g.ny;
    const double fz = (ti.iz0 + 0.5 * (ti.tz - 1)) / (double)g.nz;
    const double cx = g.origin[0] + fx * g.a1[0] + fy * g.a2[0] + fz * g.a3[0];
    const double cy = g.origin[1] + fx * g.a1[1] + fy * g.a2[1] + fz * g.a3[1];
    const double cz = g.origin[2] + fx * g.a1[2] + fy * g.a2[2] + fz * g.a3[2];
    const double reach = ti.radius + g.rcutmax;
    int lo[3], hi[3];
    const double c3[3] = {cx, cy, cz};
    const int nc3[3] = {g.ncx, g.ncy, g.ncz};
    bool any = true;
    for (int d = 0; d < 3; d++) {
        const double l = floor((c3[d] - reach - g.cell_lo[d]) * g.cell_inv[d]);
        const double h = floor((c3[d] + reach - g.cell_lo[d]) * g.cell_inv[d]);
        if (h < 0.0 || l >= (double)nc3[d]) any = false;
        lo[d] = (int)fmax(l, 0.0);
        hi[d] = (int)fmin(h, (double)(nc3[d] - 1));
    }
    int n = 0;
    int *mycand = cb.cand + (size_t)wt * cb.cand_cap;
    if (any) {
        for (int kz = lo[2]; kz <= hi[2]; kz++)
            for (int ky = lo[1]; ky <= hi[1]; ky++) {
                const int row = (kz * g.ncy + ky) * g.ncx;
                const int g0 = cb.cell_start[row + lo[0]];
                const int g1 = cb.cell_start[row + hi[0] + 1];
                for (int base = g0; base < g1; base += 32) {
                    const int gi = base + lane;
                    bool ok = false;
                    if (gi < g1) {
                        const Ghost gh = cb.ghosts[gi];
                        const double dx = gh.x - cx, dy = gh.y - cy, dz = gh.z - cz;
                        const double rr = ti.radius + tb.type_rcut[gh.type];
                        ok = (dx * dx + dy * dy + dz * dz) < rr * rr;
                    }
                    const unsigned bal = __ballot_sync(0xffffffffu, ok);
                    const int p = n + __popc(bal & ((1u << lane) - 1u));
                    if (ok && p < cb.cand_cap) mycand[p] = gi;
                    n += __popc(bal);
                }
            }
    }
    if (n > cb.cand_cap) {  // cannot happen when the host bound is right: raise the handle's status word (read back by the host)
        if (lane == 0) atomicOr(cb.status, kStatusCandOverflow);
        n = cb.cand_cap;
    }
    if (lane == 0) cb.ncand[wt] = n;
    if (n > 0) {
        if (lane == 0) {
            const int slot = atomicAdd(&cb.counters[0], 1);
            cb.active[slot] = wt;
        }
        return;
    }
    if (out == nullptr) return;
    // empty tile: constant descriptor, written as contiguous rows of tx points
    const int nt = sc.ntriples;
    // a run of n doubles repeating the nt constants: 16-byte streaming stores where the run is 16-byte aligned
    auto fill_run = [&](double *dst, const int n) {
        if ((((uintptr_t)dst) & 15) == 0) {
            double2 *d2 = reinterpret_cast<double2 *>(dst);
            for (int i = lane; i < (n >> 1); i += 32) {
                const int k = (2 * i) % nt;
                __stcs(d2 + i, make_double2(__ldg(tb.bconst + k), __ldg(tb.bconst + (k + 1 == nt ? 0 : k + 1))));
            }
            if ((n & 1) && lane == 0) __stcs(dst + n - 1, __ldg(tb.bconst + (n - 1) % nt));
        } else {
            for (int i = lane; i < n; i += 32) __stcs(dst + i, __ldg(tb.bconst + i % nt));
        }
    };
    if (cb.compact_out) {
        fill_run(out + (size_t)wt * 32 * nt, 32 * nt);
        return;
    }
    const int ix0 = ti.ix0;
    const int npx = min(ti.tx, ti.xend - ix0);
    for (int r = 0; r < ti.ty * ti.tz; r++) {
        const int iy = ti.iy0 + (r % ti.ty);
        const int iz = ti.iz0 + (r / ti.ty);
        if (iy >= ti.yend || iz >= g.z1) continue;
        fill_run(out + ((size_t)((size_t)(iz - g.z0) * g.ny + iy) * g.nx + ix0) * nt, npx * nt);
    }
}

// ---------------------------------------------------------------------------------------------------------
// one column (M) of all levels for two neighbors at once; accumulates levels J >= 2M into shared memory.
// Ul points at element 0 of this lane (stride 32 double2 between elements).
// ---------------------------------------------------------------------------------------------------------
// M is a run-time argument on purpose: all column-warps then run the SAME instructions, so the SM fetches one
// instruction stream instead of one per column (the per-column template instances stalled on instruction fetch).
template <int TJMAX, bool EXACT>
__device__ __noinline__ void ui_column_pair(double2 *Ul, const int tj, const int M, const bool upper,
                                               const double c0, const double a0r, const double a0i, const double b0r, const double b0i,
                                               const double c1, const double a1r, const double a1i, const double b1r, const double b1i) {
    double pr[2][TJMAX + 1], pi[2][TJMAX + 1];
    const double ar[2] = {a0r, a1r}, ai[2] = {a0i, a1i}, br[2] = {b0r, b1r}, bi[2] = {b0i, b1i};
    pr[0][0] = c0; pi[0][0] = 0.0;
    pr[1][0] = c1; pi[1][0] = 0.0;
    // The two half-warps hold different neighbors of the same 16 points: they add into shared memory one after the
    // other (lower half first), so the summation order is fixed and the result bit-reproducible.
    if (M == 0) {
        const double s = c0 + c1;
        double2 v = Ul[0];
        v.x += s;
        if (!upper) Ul[0] = v;
        __syncwarp();
        v = Ul[0];
        v.x += s;
        if (upper) Ul[0] = v;
        __syncwarp();
    }
#pragma unroll
    for (int r = 1; r <= TJMAX; r++) {
        if (EXACT || r <= tj) {
#pragma unroll
            for (int n = 0; n < 2; n++) {
                // linear factor f0 + f1 x :  (b + a x) for the first M rounds, (conj(a) - conj(b) x) afterwards
                const double f0r = (r <= M) ? br[n] : ar[n];
                const double f0i = (r <= M) ? bi[n] : -ai[n];
                const double f1r = (r <= M) ? ar[n] : -br[n];
                const double f1i = (r <= M) ? ai[n] : bi[n];
                // in place, highest coefficient first; explicit fma chains: 4 FP64 instructions per component
                pr[n][r] = fma(-f1i, pi[n][r - 1], f1r * pr[n][r - 1]);
                pi[n][r] = fma(f1i, pr[n][r - 1], f1r * pi[n][r - 1]);
#pragma unroll
                for (int k = r - 1; k >= 1; k--) {
                    double tr = f0r * pr[n][k];
                    double ti = f0r * pi[n][k];
                    tr = fma(-f0i, pi[n][k], tr);
                    ti = fma(f0i, pr[n][k], ti);
                    tr = fma(f1r, pr[n][k - 1], tr);
                    ti = fma(f1r, pi[n][k - 1], ti);
                    tr = fma(-f1i, pi[n][k - 1], tr);
                    ti = fma(f1i, pr[n][k - 1], ti);
                    pr[n][k] = tr;
                    pi[n][k] = ti;
                }
                const double t0r = fma(-f0i, pi[n][0], f0r * pr[n][0]);
                const double t0i = fma(f0i, pr[n][0], f0r * pi[n][0]);
                pr[n][0] = t0r;
                pi[n][0] = t0i;
            }
            if (r >= 2 * M) {
                double2 *Ue = Ul + (size_t)(uhalf_off(r) + M * (r + 1)) * kUiPoints;
#pragma unroll
                for (int k = 0; k <= r; k++) {
                    double2 v = Ue[k * kUiPoints];
                    v.x += pr[0][k] + pr[1][k];
                    v.y += pi[0][k] + pi[1][k];
                    if (!upper) Ue[k * kUiPoints] = v;
                }
                __syncwarp();
#pragma unroll
                for (int k = 0; k <= r; k++) {
                    double2 v = Ue[k * kUiPoints];
                    v.x += pr[0][k] + pr[1][k];
                    v.y += pi[0][k] + pi[1][k];
                    if (upper) Ue[k * kUiPoints] = v;
                }
                __syncwarp();
            }
        }
    }
}

// Cayley-Klein parameters and weight of one (grid point, neighbor) pair -- row a3.
// d = R_neighbor - r_point, r2 = |d|^2 < rcut^2.
__device__ __forceinline__ void pair_geometry(const double dx, const double dy, const double dz, const double r2, const double rcut,
                                              const double w, const double rfac0, const double rmin0, double &c, double &ar, double &ai,
                                              double &br, double &bi) {
    const double r = sqrt(r2);
    if (r < 1e-10 * rcut) {  // reading #11: continuous limit for an atom on the grid point
        c = w; ar = 1.0; ai = 0.0; br = 0.0; bi = 0.0;
        return;
    }
    // reading #22: inside rmin0 the switching function saturates at 1; the theta0 map stays linear in r (theta0 < 0 there)
    const double x = (r - rmin0) / (rcut - rmin0);
    c = (x <= 0.0) ? w : w * 0.5 * (cospi(x) + 1.0);
    double s, co;
    sincospi(rfac0 * x, &s, &co);
    const double sr = s / r;
    ar = co;
    ai = -sr * dz;
    br = sr * dy;
    bi = -sr * dx;
}

// Work item = half a tile (16 grid points).  Lane = (point p = lane & 15, half h = lane >> 4): both halves see the same
// points and split each point's neighbors (entries of even / odd index), so a CTA needs shared-memory accumulators for
// 16 points only (69 KB) and two CTAs share an SM -- twice the warps to hide the FP64 latency with.
// Instances: <10, true> (twojmax = 10, the configs of the paper), <10, false> (twojmax < 10, run-time guards on the levels),
// both with 6 column warps and two CTAs per SM; <14, false> (twojmax 11..14): 8 column warps, one CTA per SM (the accumulators
// of 16 points take 167 KB at twojmax = 14).
template <int TJMAX, bool EXACT>
__global__ void __launch_bounds__((TJMAX / 2 + 1) * 32, (TJMAX <= kFullTileTwoJ ? 2 : 1))
compute_ui_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb) {
    constexpr int NW = TJMAX / 2 + 1;
    constexpr int NP = kUiPoints;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nelem = sc.nelem;
    double2 *uacc = reinterpret_cast<double2 *>(smem_raw);                       // [nelem][NP]
    double *geo = reinterpret_cast<double *>(uacc + (size_t)uhalf_size(TJMAX) * NP);  // [kGeoCap][5][NP]
    double *crec = geo + kGeoCap * 5 * NP;                                          // [kGeoCap][6]
    unsigned char *hitk = reinterpret_cast<unsigned char *>(crec + kGeoCap * 6);    // [NP][kGeoCap]
    __shared__ int s_item;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int p = lane & (NP - 1);
    const bool upper = lane >= NP;
    const int tj = sc.twojmax;

    for (;;) {
        __syncthreads();  // everybody is done with the previous item (uacc reads, s_item)
        if (threadIdx.x == 0) s_item = atomicAdd(&cb.counters[1], 1);
        __syncthreads();
        const int item = s_item;
        const int slot = item >> 1, hh = item & 1;
        if (slot >= cb.counters[0]) break;
        const int wt = cb.active[slot];
        const int tile = cb.tile_begin + wt;
        int ix, iy, iz;
        bool valid;
        lane_point(g, tile, hh * NP + p, ix, iy, iz, valid);
        // ragged tiles: clamp onto a valid point (its result is never written)
        ix = min(ix, g.nx - 1); iy = min(iy, g.ny - 1); iz = min(iz, g.z1 - 1);
        double px, py, pz;
        point_position(g, ix, iy, iz, px, py, pz);

        for (int e = threadIdx.x; e < nelem * NP; e += NW * 32) uacc[e] = make_double2(0.0, 0.0);

        // this lane takes the entries of its point with index = half (mod 2), two at a time
        auto accumulate = [&](const int cnt) {
            if (warp > tj / 2) return;
            const int nmax = __reduce_max_sync(0xffffffffu, cnt);
            double2 *Ul = uacc + p;
            for (int i0 = 0; i0 < nmax; i0 += 4) {  // uniform trip count: ui_column_pair synchronises the warp
                const int i = i0 + (upper ? 1 : 0);
                double c0 = 0.0, a0r = 1.0, a0i = 0.0, b0r = 0.0, b0i = 0.0;
                double c1 = 0.0, a1r = 1.0, a1i = 0.0, b1r = 0.0, b1i = 0.0;
                if (i < cnt) {
                    const double *q = geo + (size_t)i * 5 * NP + p;
                    c0 = q[0]; a0r = q[NP]; a0i = q[2 * NP]; b0r = q[3 * NP]; b0i = q[4 * NP];
                }
                if (i + 2 < cnt) {
                    const double *q = geo + (size_t)(i + 2) * 5 * NP + p;
                    c1 = q[0]; a1r = q[NP]; a1i = q[2 * NP]; b1r = q[3 * NP]; b1i = q[4 * NP];
                }
                ui_column_pair<TJMAX, EXACT>(Ul, tj, warp, upper, c0, a0r, a0i, b0r, b0i, c1, a1r, a1i, b1r, b1i);
            }
        };

        // Candidates are taken in windows of kGeoCap.  Per window: (A) every lane runs the distance tests of its point
        // (the count must be known everywhere) and one half-warp records which candidates hit; (B) the hits of a point are
        // dealt to the twelve (warp, half) lanes of that point, which compute the pair geometry with all lanes busy
        // instead of whichever lanes happen to hit a given candidate; (C) the column warps accumulate.
        const int nc = cb.ncand[wt];
        const int *mycand = cb.cand + (size_t)wt * cb.cand_cap;
        for (int wbase = 0; wbase < nc || wbase == 0; wbase += kGeoCap) {
            const int nw = min(kGeoCap, nc - wbase);
            __syncthreads();  // crec, hitk and geo free again; first time: uacc zeroed
            if ((int)threadIdx.x < nw) {
                const Ghost gh = cb.ghosts[mycand[wbase + threadIdx.x]];
                const double rc = tb.type_rcut[gh.type];
                double *q = crec + threadIdx.x * 6;
                q[0] = gh.x; q[1] = gh.y; q[2] = gh.z; q[3] = rc; q[4] = tb.type_w[gh.type]; q[5] = rc * rc;
            }
            __syncthreads();
            int cnt = 0;  // neighbors of this lane's point in the window (identical in both halves and every warp)
            for (int k = 0; k < nw; k++) {
                const double *q = crec + k * 6;
                const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                if (dx * dx + dy * dy + dz * dz < q[5]) {
                    if (warp == 0 && !upper) hitk[p * kGeoCap + cnt] = (unsigned char)k;
                    cnt++;
                }
            }
            __syncthreads();
            for (int e = warp * 2 + (upper ? 1 : 0); e < cnt; e += NW * 2) {
                const double *q = crec + (int)hitk[p * kGeoCap + e] * 6;
                const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                const double r2 = dx * dx + dy * dy + dz * dz;
                double c, ar, ai, br, bi;
                pair_geometry(dx, dy, dz, r2, q[3], q[4], sc.rfac0, sc.rmin0, c, ar, ai, br, bi);
                double *o = geo + (size_t)e * 5 * NP + p;
                o[0] = c; o[NP] = ar; o[2 * NP] = ai; o[3 * NP] = br; o[4 * NP] = bi;
            }
            __syncthreads();
            accumulate(cnt);
            if (nc == 0) break;
        }
        __syncthreads();
        // binomial normalisation, self term (delta(0) of Eq. (24)), store of the half tile: lanes hh*16 .. hh*16+15 of
        // every element; each half-warp takes an element of its own
        double2 *dst = cb.utot_half ? cb.utot + (size_t)item * nelem * NP : cb.utot + (size_t)slot * nelem * 32 + hh * NP;
        const int estride = cb.utot_half ? NP : 32;
        for (int e = warp * 2 + (upper ? 1 : 0); e < nelem; e += NW * 2) {
            double2 v = uacc[e * NP + p];
            const double sN = tb.unorm[e];
            v.x = v.x * sN + (tb.udiag[e] ? sc.wself : 0.0);
            v.y = v.y * sN;
            dst[e * estride + p] = v;
        }
    }
}

inline size_t compute_ui_smem_bytes(int tjmax) {
    return (size_t)uhalf_size(tjmax) * kUiPoints * sizeof(double2) + (size_t)kGeoCap * 5 * kUiPoints * sizeof(double) +
           (size_t)kGeoCap * 6 * sizeof(double) + (size_t)kUiPoints * kGeoCap;
}

// debug: scatter U_tot tiles into [point][nelem] order; points of empty tiles get wself on the diagonal
__global__ void utot_scatter_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb, double2 *u_out) {
    const int lane = threadIdx.x & 31;
    const int wt = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    if (wt >= cb.ntiles) return;
    const int tile = cb.tile_begin + wt;
    int ix, iy, iz;
    bool valid;
    lane_point(g, tile, lane, ix, iy, iz, valid);
    if (!valid) return;
    // find the slot of this tile (linear search is fine for a test hook)
    int slot = -1;
    const int na = cb.counters[0];
    for (int s = 0; s < na; s++)
        if (cb.active[s] == wt) { slot = s; break; }
    double2 *dst = u_out + ((size_t)((size_t)(iz - g.z0) * g.ny + iy) * g.nx + ix) * sc.nelem;
    for (int e = 0; e < sc.nelem; e++) {
        double2 v;
        if (slot >= 0)
            v = cb.utot_half ? cb.utot[((size_t)(2 * slot + (lane >> 4)) * sc.nelem + e) * 16 + (lane & 15)]
                             : cb.utot[((size_t)slot * sc.nelem + e) * 32 + lane];
        else v = make_double2(tb.udiag[e] ? sc.wself : 0.0, 0.0);
        dst[e] = v;
    }
}

}  // namespace mala
