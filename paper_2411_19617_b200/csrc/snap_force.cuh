// snap_force.cuh -- row f3: the adjoint of the descriptor map, "apply dB(r, j)/dR_alpha to an array" (Eq. (45),
// PAPER.md:424-428):   g[alpha][k] += sum_{points r of the slab} sum_t beta[r][t] * dB_t(r)/dR_{alpha,k}.
//
// The energy-like scalar of one grid point, E_r = sum_t beta_t B_t(U_tot), is trilinear in U_tot.  Its derivative with
// respect to U_tot is one more Z-type contraction (compute_yi):
//     dE_r = Re sum_J sum_{ma,mb} conj(dU^J[ma][mb]) Y^J[ma][mb],
//     Y^J  = sum_t beta_t ( [J = j] Z^j_{j1 j2} + [J = j1] (j+1)/(j1+1) Z^{j1}_{j j2} + [J = j2] (j+1)/(j2+1) Z^{j2}_{j j1} ),
// where the second and third term are the derivatives with respect to the first two factors of the triple product, turned
// into the shape of the first by the index symmetry B_{j1 j2 j}/(j+1) = B_{j j2 j1}/(j1+1) of the Clebsch-Gordan coupling
// (checked numerically against the oracle's forward derivative before use).  Y has the same
// column symmetry as U, so half columns suffice here too.
// Then, per (grid point, neighbor), dU_tot/dR is contracted with Y (compute_dedr).  In the polynomial column form of
// snap_ui.cuh the derivative needs no recursion of its own: with Q_{J,mb}(x) = (b + a x)^mb (conj(a) - conj(b) x)^(J-mb),
//     dQ_{J,mb}/db = mb Q_{J-1,mb-1},   dQ/da = mb x Q_{J-1,mb-1},   dQ/dconj(a) = (J-mb) Q_{J-1,mb},   dQ/dconj(b) = -(J-mb) x Q_{J-1,mb},
// i.e. the derivatives of level J are the polynomials of level J-1 that the U recursion produces anyway.  Warp m, holding
// Q_{r,m} at round r, therefore adds its coefficients -- dotted with columns m and m+1 of Y^{r+1} -- to five complex sums
// (G_0 for the weight, G_a, G_b, G_conj(a), G_conj(b)), and
//     dE_r/dR_k = dc_k Re G_0 + c Re( conj(da_k) G_a + conj(db_k) G_b + da_k G_conj(a) + db_k G_conj(b) ).
// The three components are summed per (tile, candidate atom) in shared memory and added to g with one atomic per candidate.
#pragma once
#include "snap_common.cuh"
#include "snap_ui.cuh"
#include "snap_zi.cuh"

namespace mala {

struct YTerm {          // one contribution  Y^C += coef * beta[index] * Z^C_{AB}
    short A, B, C, index;
    int cgoff;          // dense CG block [m2 (B+1)][m1 (A+1)] for the coupling (A, B) -> C
    double coef;        // 1, (j+1)/(j1+1) or (j+1)/(j2+1)
};

struct ForceTables {
    const YTerm *terms;       // sorted by target level C
    const int *level_begin;   // [twojmax + 2]: terms of level C are [level_begin[C], level_begin[C+1])
    const double *cg;         // CG blocks of the terms
    const int *eorder;        // [nelem] Y elements by decreasing cost
    const double *yweight;    // [nelem] unorm[e] * (2 for columns below the middle, 1 in the middle column)
};

// ---------------------------------------------------------------------------------------------------------
// compute_yi: Y of one 32-point tile, element by element (warp = one Y element for the 32 lanes = points)
// ---------------------------------------------------------------------------------------------------------
constexpr int kYiWarps = 8;

__device__ __forceinline__ double2 u_at(const double2 *Ul, const int *uoff, int J, int ma, int mb) {  // U^J[ma][mb], any column
    if (mb <= J / 2) return Ul[(size_t)(uoff[J] + mb * (J + 1) + ma) * 32];
    const double2 v = Ul[(size_t)(uoff[J] + (J - mb) * (J + 1) + (J - ma)) * 32];
    const double s = ((ma - mb) & 1) ? -1.0 : 1.0;
    return make_double2(s * v.x, -s * v.y);
}

__global__ void __launch_bounds__(kYiWarps * 32, 1)
compute_yi_kernel(GridGeom g, SnapConst sc, ForceTables ft, ChunkBuffers cb, const double *beta, double2 *ytot) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nelem = sc.nelem, nt = sc.ntriples;
    double2 *U = reinterpret_cast<double2 *>(smem_raw);                 // [nelem][32]
    double *Bt = reinterpret_cast<double *>(U + (size_t)nelem * 32);    // [nt][32] beta of the tile, lane fastest
    __shared__ uint64_t bar;
    __shared__ int s_slot, s_next;
    __shared__ int s_uoff[kMaxTwoJ + 2];
    const int lane = threadIdx.x & 31;
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    if (threadIdx.x <= kMaxTwoJ + 1) s_uoff[threadIdx.x] = uhalf_off(threadIdx.x);
    uint32_t parity = 0;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) {
            s_slot = atomicAdd(&cb.counters[2], 1);
            s_next = 0;
        }
        __syncthreads();
        const int slot = s_slot;
        if (slot >= cb.counters[0]) break;
        const int wt = cb.active[slot];
        if (threadIdx.x == 0) tma_load_tile(U, cb.utot + (size_t)slot * nelem * 32, nelem, &bar);
        // beta rows of the tile's points (zero for lanes outside a ragged tile)
        for (int idx = threadIdx.x; idx < 32 * nt; idx += kYiWarps * 32) {
            const int l = idx / nt, t = idx - l * nt;
            int ix, iy, iz;
            bool valid;
            lane_point(g, cb.tile_begin + wt, l, ix, iy, iz, valid);
            Bt[t * 32 + l] = valid ? beta[((size_t)((size_t)(iz - g.z0) * g.ny + iy) * g.nx + ix) * nt + t] : 0.0;
        }
        mbar_wait(&bar, parity);
        parity ^= 1u;
        __syncthreads();
        const double2 *Ul = U + lane;
        double2 *Yt = ytot + (size_t)slot * nelem * 32 + lane;
        for (;;) {
            int pos = 0;
            if (lane == 0) pos = atomicAdd(&s_next, 1);
            pos = __shfl_sync(0xffffffffu, pos, 0);
            if (pos >= nelem) break;
            const int e = ft.eorder[pos];
            // element e -> (C, mb, ma)
            int C = 0;
            while (s_uoff[C + 1] <= e) C++;
            const int mb = (e - s_uoff[C]) / (C + 1), ma = (e - s_uoff[C]) - mb * (C + 1);
            double yr = 0.0, yi = 0.0;
            for (int k = ft.level_begin[C]; k < ft.level_begin[C + 1]; k++) {
                const YTerm T = ft.terms[k];
                const int A = T.A, B = T.B;
                const int sh = (A + B - C) / 2;
                const double *cg = ft.cg + T.cgoff;
                double zr = 0.0, zi = 0.0;
                const int mb1lo = max(0, mb + sh - B), mb1hi = min(A, mb + sh);
                const int ma1lo = max(0, ma + sh - B), ma1hi = min(A, ma + sh);
                for (int mb1 = mb1lo; mb1 <= mb1hi; mb1++) {
                    const int mb2 = mb + sh - mb1;
                    const double cgb = cg[mb2 * (A + 1) + mb1];
                    double sr = 0.0, si = 0.0;
                    for (int ma1 = ma1lo; ma1 <= ma1hi; ma1++) {
                        const int ma2 = ma + sh - ma1;
                        const double cga = cg[ma2 * (A + 1) + ma1];
                        const double2 x = u_at(Ul, s_uoff, A, ma1, mb1), y = u_at(Ul, s_uoff, B, ma2, mb2);
                        sr += cga * (x.x * y.x - x.y * y.y);
                        si += cga * (x.x * y.y + x.y * y.x);
                    }
                    zr += cgb * sr;
                    zi += cgb * si;
                }
                const double w = T.coef * Bt[T.index * 32 + lane];
                yr += w * zr;
                yi += w * zi;
            }
            const double yw = ft.yweight[e];   // normalisation of the polynomial form and the half-column doubling
            Yt[(size_t)e * 32] = make_double2(yw * yr, yw * yi);
        }
    }
}

inline size_t compute_yi_smem_bytes(int nelem, int nt) {
    return (size_t)nelem * 32 * sizeof(double2) + (size_t)32 * nt * sizeof(double) + 16;
}

// ---------------------------------------------------------------------------------------------------------
// compute_dedr: per (grid point, neighbor) contract dU_tot/dR with Y.  Work item = half a tile (16 points), warp m =
// column m of every level, lane = (point, half), the halves take the neighbors of a point alternately -- the layout of
// compute_ui_kernel, with its accumulation replaced by dot products against the weighted Y of the tile.
// ---------------------------------------------------------------------------------------------------------
constexpr int kFrcPoints = 16;
constexpr int kFrcCap = 48;   // candidates per window

template <int TJMAX>
__global__ void __launch_bounds__((TJMAX / 2 + 1) * 32, 2)
compute_dedr_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb, const double2 *ytot, double *gout) {
    constexpr int NW = TJMAX / 2 + 1;
    constexpr int NP = kFrcPoints;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nelem = sc.nelem;
    double2 *Y = reinterpret_cast<double2 *>(smem_raw);                       // [nelem + pad][NP], weighted
    double *crec = reinterpret_cast<double *>(Y + (size_t)(uhalf_size(TJMAX) + TJMAX + 2) * NP);  // [kFrcCap][6]
    double *fsum = crec + kFrcCap * 6;                                        // [kFrcCap][3]
    int *catom = reinterpret_cast<int *>(fsum + kFrcCap * 3);                 // [kFrcCap] atom index of the candidate
    unsigned char *hitk = reinterpret_cast<unsigned char *>(catom + kFrcCap); // [NP][kFrcCap]
    __shared__ int s_item;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int p = lane & (NP - 1);
    const bool upper = lane >= NP;
    const int tj = sc.twojmax;
    const int M = warp;

    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(&cb.counters[3], 1);   // counters[1] and [2] belong to compute_ui / compute_yi
        __syncthreads();
        const int item = s_item;
        const int slot = item >> 1, hh = item & 1;
        if (slot >= cb.counters[0]) break;
        const int wt = cb.active[slot];
        const int tile = cb.tile_begin + wt;
        int ix, iy, iz;
        bool valid;
        lane_point(g, tile, hh * NP + p, ix, iy, iz, valid);
        ix = min(ix, g.nx - 1); iy = min(iy, g.ny - 1); iz = min(iz, g.z1 - 1);  // ragged tiles: beta (hence Y) is zero there
        double px, py, pz;
        point_position(g, ix, iy, iz, px, py, pz);
        // Y of this half tile; one zero row behind the last element so that "row ma + 1" of the last column is readable
        const double2 *src = ytot + (size_t)slot * nelem * 32 + hh * NP;
        for (int e = threadIdx.x; e < (nelem + TJMAX + 2) * NP; e += NW * 32) {
            const int el = e / NP, pp = e - el * NP;
            Y[e] = (el < nelem) ? src[(size_t)el * 32 + pp] : make_double2(0.0, 0.0);
        }
        const int nc = cb.ncand[wt];
        const int *mycand = cb.cand + (size_t)wt * cb.cand_cap;
        for (int wbase = 0; wbase < nc; wbase += kFrcCap) {
            const int nw = min(kFrcCap, nc - wbase);
            __syncthreads();  // previous window flushed; first time: Y loaded
            if ((int)threadIdx.x < nw) {
                const Ghost gh = cb.ghosts[mycand[wbase + threadIdx.x]];
                const double rc = tb.type_rcut[gh.type];
                double *q = crec + threadIdx.x * 6;
                q[0] = gh.x; q[1] = gh.y; q[2] = gh.z; q[3] = rc; q[4] = tb.type_w[gh.type]; q[5] = rc * rc;
                catom[threadIdx.x] = gh.pad;
                fsum[threadIdx.x * 3] = 0.0; fsum[threadIdx.x * 3 + 1] = 0.0; fsum[threadIdx.x * 3 + 2] = 0.0;
            }
            __syncthreads();
            int cnt = 0;
            for (int k = 0; k < nw; k++) {
                const double *q = crec + k * 6;
                const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                if (dx * dx + dy * dy + dz * dz < q[5]) {
                    if (warp == 0 && !upper) hitk[p * kFrcCap + cnt] = (unsigned char)k;
                    cnt++;
                }
            }
            __syncthreads();
            if (M <= tj / 2) {
                const int nmax = __reduce_max_sync(0xffffffffu, cnt);
                const double2 *Yl = Y + p;
                for (int i0 = 0; i0 < nmax; i0 += 2) {
                    const int i = i0 + (upper ? 1 : 0);
                    const bool live = i < cnt;
                    const int kc = live ? (int)hitk[p * kFrcCap + i] : 0;
                    const double *q = crec + kc * 6;
                    const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    // pair geometry and its gradient with respect to the atom position (row a3 and its derivative)
                    const double rcut = q[3], w = q[4];
                    const double r = sqrt(r2);
                    double c = 0.0, ar = 1.0, ai = 0.0, br = 0.0, bi = 0.0;
                    double dc[3] = {0.0, 0.0, 0.0}, dar[3] = {0.0, 0.0, 0.0}, dai[3] = {0.0, 0.0, 0.0}, dbr[3] = {0.0, 0.0, 0.0},
                           dbi[3] = {0.0, 0.0, 0.0};
                    if (live && r >= 1e-10 * rcut) {
                        const double inv = 1.0 / (rcut - sc.rmin0);
                        const double x = (r - sc.rmin0) * inv;
                        double fcp = 0.0;
                        if (x <= 0.0) c = w;
                        else {
                            double sp, cp;
                            sincospi(x, &sp, &cp);
                            c = w * 0.5 * (cp + 1.0);
                            fcp = -0.5 * 3.14159265358979323846 * sp * inv * w;
                        }
                        double s0, c0;
                        sincospi(sc.rfac0 * x, &s0, &c0);
                        const double th0p = sc.rfac0 * 3.14159265358979323846 * inv;
                        const double ir = 1.0 / r;
                        const double u[3] = {dx * ir, dy * ir, dz * ir};
                        ar = c0; ai = -s0 * u[2]; br = s0 * u[1]; bi = -s0 * u[0];
#pragma unroll
                        for (int k = 0; k < 3; k++) {
                            const double dr = u[k];
                            dc[k] = fcp * dr;
                            const double dq0 = -s0 * th0p * dr;
                            double dq[3];
#pragma unroll
                            for (int ii = 0; ii < 3; ii++) dq[ii] = c0 * th0p * dr * u[ii] + s0 * (((ii == k) ? 1.0 : 0.0) - u[ii] * u[k]) * ir;
                            dar[k] = dq0; dai[k] = -dq[2]; dbr[k] = dq[1]; dbi[k] = -dq[0];
                        }
                    }
                    // column M of every level by the polynomial recursion (unit weight); dot products against Y on the way
                    double pr[TJMAX + 1], pi[TJMAX + 1];
                    pr[0] = 1.0; pi[0] = 0.0;
                    double g0r = 0.0, gar = 0.0, gai = 0.0, gbr = 0.0, gbi = 0.0, gcar = 0.0, gcai = 0.0, gcbr = 0.0, gcbi = 0.0;
#pragma unroll
                    for (int rr = 0; rr <= TJMAX; rr++) {
                        if (rr <= tj) {
                            if (rr >= 1) {
                                const double f0r = (rr <= M) ? br : ar;
                                const double f0i = (rr <= M) ? bi : -ai;
                                const double f1r = (rr <= M) ? ar : -br;
                                const double f1i = (rr <= M) ? ai : bi;
                                pr[rr] = fma(-f1i, pi[rr - 1], f1r * pr[rr - 1]);
                                pi[rr] = fma(f1i, pr[rr - 1], f1r * pi[rr - 1]);
#pragma unroll
                                for (int k = rr - 1; k >= 1; k--) {
                                    double tr = f0r * pr[k];
                                    double ti = f0r * pi[k];
                                    tr = fma(-f0i, pi[k], tr);
                                    ti = fma(f0i, pr[k], ti);
                                    tr = fma(f1r, pr[k - 1], tr);
                                    ti = fma(f1r, pi[k - 1], ti);
                                    tr = fma(-f1i, pi[k - 1], tr);
                                    ti = fma(f1i, pr[k - 1], ti);
                                    pr[k] = tr;
                                    pi[k] = ti;
                                }
                                const double t0r = fma(-f0i, pi[0], f0r * pr[0]);
                                const double t0i = fma(f0i, pr[0], f0r * pi[0]);
                                pr[0] = t0r;
                                pi[0] = t0i;
                            }
                            // the polynomial is Q_{rr,M} once rr >= M
                            if (rr >= 2 * M) {  // stored element (rr, M, k): weight term
                                const double2 *Yc = Yl + (size_t)(uhalf_off(rr) + M * (rr + 1)) * NP;
#pragma unroll
                                for (int k = 0; k <= rr; k++) {
                                    const double2 y = Yc[k * NP];
                                    g0r = fma(pr[k], y.x, g0r);
                                    g0r = fma(pi[k], y.y, g0r);
                                }
                            }
                            if (rr + 1 <= tj && rr >= M) {
                                if (2 * (M + 1) <= rr + 1) {  // target (rr + 1, M + 1): d/db and d/da, factor M + 1
                                    const double2 *Yc = Yl + (size_t)(uhalf_off(rr + 1) + (M + 1) * (rr + 2)) * NP;
                                    const double f = (double)(M + 1);
#pragma unroll
                                    for (int k = 0; k <= rr; k++) {
                                        const double2 y0 = Yc[k * NP], y1 = Yc[(k + 1) * NP];
                                        const double qr = f * pr[k], qi = f * pi[k];   // conj(q) * y = (qr y.x + qi y.y) + i (qr y.y - qi y.x)
                                        gbr = fma(qr, y0.x, gbr); gbr = fma(qi, y0.y, gbr);
                                        gbi = fma(qr, y0.y, gbi); gbi = fma(-qi, y0.x, gbi);
                                        gar = fma(qr, y1.x, gar); gar = fma(qi, y1.y, gar);
                                        gai = fma(qr, y1.y, gai); gai = fma(-qi, y1.x, gai);
                                    }
                                }
                                if (2 * M <= rr + 1) {        // target (rr + 1, M): d/dconj(a) and d/dconj(b), factor rr + 1 - M
                                    const double2 *Yc = Yl + (size_t)(uhalf_off(rr + 1) + M * (rr + 2)) * NP;
                                    const double f = (double)(rr + 1 - M);
#pragma unroll
                                    for (int k = 0; k <= rr; k++) {
                                        const double2 y0 = Yc[k * NP], y1 = Yc[(k + 1) * NP];
                                        const double qr = f * pr[k], qi = f * pi[k];
                                        gcar = fma(qr, y0.x, gcar); gcar = fma(qi, y0.y, gcar);
                                        gcai = fma(qr, y0.y, gcai); gcai = fma(-qi, y0.x, gcai);
                                        gcbr = fma(-qr, y1.x, gcbr); gcbr = fma(-qi, y1.y, gcbr);
                                        gcbi = fma(-qr, y1.y, gcbi); gcbi = fma(qi, y1.x, gcbi);
                                    }
                                }
                            }
                        }
                    }
                    if (live) {
#pragma unroll
                        for (int k = 0; k < 3; k++) {
                            // dc Re G0 + c Re( conj(da) Ga + conj(db) Gb + da Gca + db Gcb )
                            double s = dc[k] * g0r;
                            double t = dar[k] * gar + dai[k] * gai + dbr[k] * gbr + dbi[k] * gbi;
                            t += dar[k] * gcar - dai[k] * gcai + dbr[k] * gcbr - dbi[k] * gcbi;
                            s = fma(c, t, s);
                            atomicAdd(&fsum[kc * 3 + k], s);
                        }
                    }
                }
            }
            __syncthreads();
            if ((int)threadIdx.x < nw * 3) {
                const int k = threadIdx.x / 3, d = threadIdx.x - 3 * k;
                const double v = fsum[k * 3 + d];
                if (v != 0.0) atomicAdd(gout + (size_t)catom[k] * 3 + d, v);
            }
        }
    }
}

inline size_t compute_dedr_smem_bytes(int tjmax) {
    return (size_t)(uhalf_size(tjmax) + tjmax + 2) * kFrcPoints * sizeof(double2) + (size_t)kFrcCap * 9 * sizeof(double) +
           (size_t)kFrcCap * sizeof(int) + (size_t)kFrcPoints * kFrcCap;
}

}  // namespace mala
