// snap_dedr_dft.cuh -- compute_dedr of row f3 in the sampling form of snap_ui_dft.cuh (twojmax 1..10).
//
// compute_dedr contracts dU_tot/dR of every (grid point, neighbor) pair with the weighted Y of the point (snap_force.cuh):
//     E_pair = c Re sum_{J,mb,k} q_{J,mb,k} conj(Y_{J,mb,k}),   q_{J,mb,k} = coefficient k of Q_{J,mb}(x) = (b + a x)^mb (conj(a) - conj(b) x)^(J-mb)
// and g[atom] += dE_pair/dR.  With the N = twojmax + 1 roots of unity x_s, q_k = (1/N) sum_s Q(x_s) x_s^(-k), so by Parseval
//     sum_k q_k conj(Y_k) = (1/N) sum_s Q_{J,mb}(x_s) conj(Yhat_{J,mb}(x_s)),      Yhat_{J,mb}(x_s) = sum_k Y_{J,mb,k} x_s^k,
// and Q_{J,mb}(x_s) = u_s^mb v_s^(J-mb) with u_s = b + a x_s, v_s = conj(a) - conj(b) x_s.  Per sample point the pair energy is
// therefore a bivariate polynomial with coefficients that belong to the grid point only,
//     E_pair = c Re sum_s F_s(u_s, v_s),   F_s(u, v) = sum_{mb <= n} W_{s,mb,n} u^mb v^n,   W_{s,mb,n} = conj(Yhat_{mb+n,mb}(x_s)) / N,
// and its gradient follows from F_s, dF_s/du and dF_s/dv by du_s = db + da x_s, dv_s = conj(da) - conj(db) x_s.
//   * warp s owns sample point x_s, lane = grid point (a whole 32-point tile); once per tile the warp takes the DFT of the Y
//     columns of its lanes (Y of the tile in shared memory) and keeps the 36 complex W in REGISTERS for all neighbors;
//   * per (sample, neighbor): F, dF/dw (w = u v) and the v-derivative by Horner in v inside Horner in w -- about 300 FP64
//     instructions -- then dE/dR_k = alpha u_k + beta h_k from five real numbers (the chain rule through c, theta0 and the unit
//     vector is linear in them), added per (neighbor entry, point) in shared memory (atomics between the warps: the order of the
//     eleven samples is not fixed, results are reproducible to rounding as before) and per candidate atom at the end of a window;
//   * no recursion of U, no second pass over Y per neighbor: 3,900 instead of ~10,000 FP64 instructions per pair.
// Candidate windows, distance tests (bit masks) and the dealing of the hits to the warps are those of compute_ui_dft_kernel;
// a queue entry holds what the chain rule needs: c, dc/dr, sin and cos of theta0, dtheta0/dr, 1/r and the unit vector.
#pragma once
#include "snap_ui_dft.cuh"
#include "snap_zi.cuh"

namespace mala {

constexpr int kDdCap = 24;      // candidates per window = queue entries per grid point (a window never overflows its queue)
constexpr int kDdEntry = 9;     // doubles per queue entry: c, dc/dr, s0, c0, dtheta0/dr, 1/r, ux, uy, uz

template <int TJ>
__global__ void __launch_bounds__((TJ + 1) * 32, 1)
compute_dedr_dft_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb, const double2 *ytot, double *gout) {
    constexpr int NW = TJ + 1;          // warps = sample points
    constexpr int NJM = dft_njm(TJ);
    constexpr int nelem = uhalf_size(TJ);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *Y = reinterpret_cast<double2 *>(smem_raw);                                   // [nelem][32], weighted (compute_yi)
    double *geo = reinterpret_cast<double *>(Y + (size_t)nelem * 32);                     // [kDdCap][kDdEntry][32]
    double *crec = geo + (size_t)kDdCap * kDdEntry * 32;                                  // [kDdCap][6]
    double *facc = crec + kDdCap * 6;                                                     // [kDdCap][3][32] force of entry e on lane's pair
    unsigned long long *hmask = reinterpret_cast<unsigned long long *>(facc + kDdCap * 3 * 32); // [NW + 1][32], the last row: all warps
    int *catom = reinterpret_cast<int *>(hmask + (NW + 1) * 32);                          // [kDdCap] atom of the candidate
    __shared__ uint64_t bar;
    __shared__ int s_item;
    __shared__ double2 s_root[NW];      // e^{2 pi i m / NW}
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x < NW) {
        double sn, cs;
        sincospi(2.0 * (double)threadIdx.x / (double)NW, &sn, &cs);
        s_root[threadIdx.x] = make_double2(cs, sn);
    }
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    double xsr, xsi;                    // this warp's sample point x_s
    {
        double sn, cs;
        sincospi(2.0 * (double)warp / (double)NW, &sn, &cs);
        xsr = cs; xsi = sn;
    }
    uint32_t parity = 0;

    for (;;) {
        __syncthreads();  // everybody is done with the previous tile (Y, s_item)
        if (threadIdx.x == 0) s_item = atomicAdd(&cb.counters[3], 1);   // counters[1] and [2] belong to compute_ui / compute_yi
        __syncthreads();
        const int slot = s_item;
        if (slot >= cb.counters[0]) break;
        const int wt = cb.active[slot];
        if (threadIdx.x == 0) tma_load_tile(Y, ytot + (size_t)slot * nelem * 32, nelem, &bar);
        int ix, iy, iz;
        bool valid;
        lane_point(g, cb.tile_begin + wt, lane, ix, iy, iz, valid);
        ix = min(ix, g.nx - 1); iy = min(iy, g.ny - 1); iz = min(iz, g.z1 - 1);  // ragged tiles: beta (hence Y) is zero there
        double px, py, pz;
        point_position(g, ix, iy, iz, px, py, pz);
        mbar_wait(&bar, parity);
        parity ^= 1u;

        // W_{mb,n} = conj(Yhat_{mb+n,mb}(x_s)) / NW for this lane's grid point.  36 complex W are 144 registers, more than a thread has
        // at twelve warps: from twojmax 8 up the W of the longest chain (mb = 0) live in shared memory -- in the bytes of Y, which
        // is dead once every warp has its W; until then they wait in the (still unused) queue and force buffers
        constexpr bool W0_SHARED = TJ >= 8;
        static_assert(!W0_SHARED || (size_t)NW * NW * 32 * sizeof(double2) <= (size_t)kDdCap * (kDdEntry + 3) * 32 * sizeof(double), "staging of W0");
        double2 *W0 = reinterpret_cast<double2 *>(smem_raw) + (size_t)warp * NW * 32 + lane;      // [warp][n][lane]
        double2 *W0stage = reinterpret_cast<double2 *>(geo) + (size_t)warp * NW * 32 + lane;
        double wr[NJM], wi[NJM];
#pragma unroll
        for (int mb = 0; mb <= TJ / 2; mb++) {
#pragma unroll
            for (int n = mb; n <= TJ - mb; n++) {
                const int J = mb + n;
                const double2 *Yc = Y + (size_t)(uhalf_off(J) + mb * (J + 1)) * 32 + lane;
                double sr = 0.0, si = 0.0;
                int m = 0;   // (warp * k) mod NW
                for (int k = 0; k <= J; k++) {
                    const double2 y = Yc[(size_t)k * 32], t = s_root[m];
                    sr = fma(y.x, t.x, sr); sr = fma(-y.y, t.y, sr);
                    si = fma(y.x, t.y, si); si = fma(y.y, t.x, si);
                    m += warp;
                    if (m >= NW) m -= NW;
                }
                if (W0_SHARED && mb == 0) W0stage[n * 32] = make_double2(sr * (1.0 / (double)NW), -si * (1.0 / (double)NW));
                else {
                    wr[dft_index(TJ, mb, n)] = sr * (1.0 / (double)NW);
                    wi[dft_index(TJ, mb, n)] = -si * (1.0 / (double)NW);
                }
            }
        }
        if constexpr (W0_SHARED) {
            __syncthreads();   // Y is dead
#pragma unroll
            for (int n = 0; n <= TJ; n++) W0[n * 32] = W0stage[n * 32];
        }

        const int nc = cb.ncand[wt];
        const int *mycand = cb.cand + (size_t)wt * cb.cand_cap;
        for (int wbase = 0; wbase < nc; wbase += kDdCap) {
            const int nw = min(kDdCap, nc - wbase);
            __syncthreads();  // the previous window is flushed: crec, geo and facc are free (first time: W is taken from Y)
            if ((int)threadIdx.x < nw) {
                const Ghost gh = cb.ghosts[mycand[wbase + threadIdx.x]];
                const double rc = tb.type_rcut[gh.type];
                double *q = crec + threadIdx.x * 6;
                q[0] = gh.x; q[1] = gh.y; q[2] = gh.z; q[3] = rc; q[4] = tb.type_w[gh.type]; q[5] = rc * rc;
                catom[threadIdx.x] = gh.pad;
            }
            for (int i = threadIdx.x; i < kDdCap * 3 * 32; i += NW * 32) facc[i] = 0.0;
            __syncthreads();
            // distance tests: warp w takes candidates w, w + NW, ... for the 32 points and publishes its hits as a bit mask
            unsigned long long mine = 0ull;
            for (int k = warp; k < nw; k += NW) {
                const double *q = crec + k * 6;
                const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                if (dx * dx + dy * dy + dz * dz < q[5]) mine |= 1ull << k;
            }
            hmask[warp * 32 + lane] = mine;
            __syncthreads();
            unsigned long long hits = 0ull;   // neighbors of this lane's point in the window, identical in every warp
#pragma unroll
            for (int w2 = 0; w2 < NW; w2++) hits |= hmask[w2 * 32 + lane];
            const int cnt = __popcll(hits);
            if (warp == 0) hmask[NW * 32 + lane] = hits;
            // the hits of a point (in candidate order) are dealt to the NW lanes of that point: pair geometry once per pair
            {
                int e = 0, turn = 0;   // turn = e mod NW
                for (unsigned long long r = hits; r != 0ull; r &= r - 1ull, e++) {
                    if (turn == warp) {
                        const int k = __ffsll((long long)r) - 1;
                        const double *q = crec + k * 6;
                        const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                        const double rcut = q[3], w = q[4];
                        const double rr = sqrt(dx * dx + dy * dy + dz * dz);
                        // row a3 and what its gradient needs; an atom on the grid point (reading #11) has a = 1, b = 0 and no force
                        double c = w, fcp = 0.0, s0 = 0.0, c0 = 1.0, th0p = 0.0, ir = 0.0;
                        if (rr >= 1e-10 * rcut) {
                            const double inv = 1.0 / (rcut - sc.rmin0);
                            const double x = (rr - sc.rmin0) * inv;
                            if (x > 0.0) {   // reading #22: inside rmin0 the switching function stays at 1
                                double sp, cp;
                                sincospi(x, &sp, &cp);
                                c = w * 0.5 * (cp + 1.0);
                                fcp = -0.5 * 3.14159265358979323846 * sp * inv * w;
                            }
                            sincospi(sc.rfac0 * x, &s0, &c0);
                            th0p = sc.rfac0 * 3.14159265358979323846 * inv;
                            ir = 1.0 / rr;
                        }
                        double *o = geo + (size_t)e * kDdEntry * 32 + lane;
                        o[0] = c; o[32] = fcp; o[64] = s0; o[96] = c0; o[128] = th0p; o[160] = ir;
                        o[192] = dx * ir; o[224] = dy * ir; o[256] = dz * ir;
                    }
                    turn = (turn + 1 == NW) ? 0 : turn + 1;
                }
            }
            __syncthreads();
            const int nmax = __reduce_max_sync(0xffffffffu, cnt);
            // the warps add to the same (entry, lane) sums: each starts at another entry so that they seldom meet
            const int rot = (warp * 3) % max(nmax, 1);
#pragma unroll 1
            for (int i0 = 0; i0 < nmax; i0++) {
                const int i = (i0 + rot >= nmax) ? i0 + rot - nmax : i0 + rot;
                const bool live = i < cnt;
                double c = 0.0, fcp = 0.0, s0 = 0.0, c0 = 1.0, th0p = 0.0, ir = 0.0, ux = 0.0, uy = 0.0, uz = 0.0;
                if (live) {
                    const double *q = geo + (size_t)i * kDdEntry * 32 + lane;
                    c = q[0]; fcp = q[32]; s0 = q[64]; c0 = q[96]; th0p = q[128]; ir = q[160]; ux = q[192]; uy = q[224]; uz = q[256];
                }
                const double ar = c0, ai = -s0 * uz, br = s0 * uy, bi = -s0 * ux;
                // u = b + a x_s,  v = conj(a) - conj(b) x_s,  w = u v
                const double ur = fma(-ai, xsi, fma(ar, xsr, br)), ui = fma(ai, xsr, fma(ar, xsi, bi));
                const double vr = ar - fma(bi, xsi, br * xsr), vi = -ai - fma(-bi, xsr, br * xsi);
                const double pwr = fma(-ui, vi, ur * vr), pwi = fma(ui, vr, ur * vi);
                // F = sum_mb w^mb P_mb(v), P_mb(v) = sum_n W_{mb,n} v^(n-mb): Horner in v inside Horner in w, with dF/dw (A_w) and
                // the sum of the v-derivatives (B_v) on the way
                double Ar = 0.0, Ai = 0.0, Awr = 0.0, Awi = 0.0, Bvr = 0.0, Bvi = 0.0;
#pragma unroll
                for (int mb = TJ / 2; mb >= 0; mb--) {
                    double Pr, Pi, Dr = 0.0, Di = 0.0;
                    if (W0_SHARED && mb == 0) { const double2 t = W0[TJ * 32]; Pr = t.x; Pi = t.y; }
                    else { Pr = wr[dft_index(TJ, mb, TJ - mb)]; Pi = wi[dft_index(TJ, mb, TJ - mb)]; }
#pragma unroll
                    for (int n = TJ - mb - 1; n >= mb; n--) {
                        double cr, ci;
                        if (W0_SHARED && mb == 0) { const double2 t = W0[n * 32]; cr = t.x; ci = t.y; }
                        else { cr = wr[dft_index(TJ, mb, n)]; ci = wi[dft_index(TJ, mb, n)]; }
                        const double dr2 = fma(-Di, vi, fma(Dr, vr, Pr)), di2 = fma(Di, vr, fma(Dr, vi, Pi));
                        const double pr2 = fma(-Pi, vi, fma(Pr, vr, cr)), pi2 = fma(Pi, vr, fma(Pr, vi, ci));
                        Dr = dr2; Di = di2; Pr = pr2; Pi = pi2;
                    }
                    const double awr = fma(-Awi, pwi, fma(Awr, pwr, Ar)), awi = fma(Awi, pwr, fma(Awr, pwi, Ai));
                    const double a2r = fma(-Ai, pwi, fma(Ar, pwr, Pr)), a2i = fma(Ai, pwr, fma(Ar, pwi, Pi));
                    const double b2r = fma(-Bvi, pwi, fma(Bvr, pwr, Dr)), b2i = fma(Bvi, pwr, fma(Bvr, pwi, Di));
                    Awr = awr; Awi = awi; Ar = a2r; Ai = a2i; Bvr = b2r; Bvi = b2i;
                }
                // dF/du = v A_w,  dF/dv = u A_w + B_v, and both times x_s
                const double fur = fma(-vi, Awi, vr * Awr), fui = fma(vi, Awr, vr * Awi);
                const double fvr = fma(-ui, Awi, fma(ur, Awr, Bvr)), fvi = fma(ui, Awr, fma(ur, Awi, Bvi));
                const double fuxr = fma(-fui, xsi, fur * xsr), fuxi = fma(fui, xsr, fur * xsi);
                const double fvxr = fma(-fvi, xsi, fvr * xsr), fvxi = fma(fvi, xsr, fvr * xsi);
                // dE/dR_k = dc_k Re F + c Re(db_k F_u + da_k F_u x + conj(da_k) F_v - conj(db_k) F_v x); with a = c0 - i s0 u_z,
                // b = s0 u_y - i s0 u_x the chain rule through r, theta0 and the unit vector collapses to alpha u_k + beta h_k
                const double Ha = fuxr + fvr, h0 = fui + fvxi, h1 = fur - fvxr, h2 = fuxi - fvi;
                const double uh = fma(ux, h0, fma(uy, h1, uz * h2));
                const double alpha = fma(fcp, Ar, c * fma(-s0 * th0p, Ha, (c0 * th0p - s0 * ir) * uh));
                const double beta = c * s0 * ir;
                if (live) {
                    double *f = facc + (size_t)i * 96 + lane;
                    atomicAdd(f, fma(alpha, ux, beta * h0));
                    atomicAdd(f + 32, fma(alpha, uy, beta * h1));
                    atomicAdd(f + 64, fma(alpha, uz, beta * h2));
                }
            }
            __syncthreads();
            // per candidate: the sum over the points that have it as a neighbor (entry = its rank among the hits of the point)
            for (int t = threadIdx.x; t < nw * 3; t += NW * 32) {   // (twojmax 1 has 64 threads for up to 72 sums)
                const int k = t / 3, d = t - 3 * k;
                double v = 0.0;
                for (int l = 0; l < 32; l++) {
                    const unsigned long long hl = hmask[NW * 32 + l];
                    if (hl >> k & 1ull) v += facc[(size_t)__popcll(hl & ((1ull << k) - 1ull)) * 96 + d * 32 + l];
                }
                if (v != 0.0) atomicAdd(gout + (size_t)catom[k] * 3 + d, v);
            }
        }
    }
}

template <int TJ>
inline size_t compute_dedr_dft_smem_bytes() {
    return (size_t)uhalf_size(TJ) * 32 * sizeof(double2) + (size_t)kDdCap * kDdEntry * 32 * sizeof(double) + (size_t)kDdCap * 6 * sizeof(double) +
           (size_t)kDdCap * 3 * 32 * sizeof(double) + (size_t)(TJ + 2) * 32 * sizeof(unsigned long long) + (size_t)kDdCap * sizeof(int) + 16;
}

}  // namespace mala
