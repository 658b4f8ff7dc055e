// snap_ui_dft.cuh -- compute_ui by sampling the column polynomials (rows a3 + a4 of SURVEY.md 8(a)), twojmax 1..10.
//
// Same quantity and the same storage as snap_ui.cuh: U_tot^J = wself*I + sum_neighbors c * U^J(neighbor) in half columns,
// where column mb of level J is the coefficient list of the polynomial Q_{J,mb}(x) = (b + a x)^mb (conj(a) - conj(b) x)^(J-mb),
// a and b the Cayley-Klein parameters of the neighbor (Eq. (24)-(25)).
//
// (Written for twojmax = 10; the kernel is a template on twojmax with twojmax + 1 sample points and warps.)
// A polynomial of degree <= 10 is fixed by its values at the 11th roots of unity x_s, and there its value is a product of
// powers:  Q_{J,mb}(x_s) = u_s^mb v_s^(J-mb),  u_s = b + a x_s,  v_s = conj(a) - conj(b) x_s.  So instead of carrying
// coefficient lists through a recursion and adding them to accumulators in shared memory neighbor by neighbor (snap_ui.cuh:
// 4,300 FP64 instructions per pair, half of the issue slots lost to barriers, shared-memory round trips and bookkeeping),
//   * warp s owns sample point x_s, lane = grid point (a whole 32-point tile), and keeps the 36 sums
//     S_{J,mb}(x_s) = sum_neighbors c u_s^mb v_s^(J-mb) in REGISTERS over all neighbors of the point: per neighbor one complex
//     multiplication and one complex addition per (J, mb) -- 224 FP64 instructions, nothing else but five loads;
//   * once per tile the coefficients come back by the inverse DFT of length 11, q_k = (1/11) sum_s S(x_s) x_s^(-k)
//     (unitary, hence well conditioned: 1.6e-14 absolute on sums of 30 neighbors), followed by the binomial normalisation
//     and the self term as before.  Sample points come in conjugate pairs, which halves the multiply-adds of the DFT.
// 2,460 + 250 (DFT, amortised over ~26 neighbors) FP64 instructions per pair, one instruction stream for all eleven warps,
// no atomics, fixed summation order (bit-reproducible).  From twojmax 9 up the sums are taken in two passes over the
// neighbors of the tile (dft_split) so that the accumulators leave registers for the compiler to overlap the chains.
// Everything in front of the accumulation (candidate windows, distance tests, dealing the hits to all warps for the pair
// geometry) is that of compute_ui_kernel, on whole tiles.
#pragma once
#include "snap_ui.cuh"

namespace mala {

#ifndef MALA_DFT_UNROLL
#define MALA_DFT_UNROLL 1
#endif
constexpr int kDftUnroll = MALA_DFT_UNROLL;   // neighbors per trip of the accumulation loop
constexpr int kDftCap = 48;   // neighbor entries per grid point buffered between two accumulate passes (<= 64: hit masks)

constexpr int dft_njm(int tj) {   // number of (J, mb <= J/2) columns
    int n = 0;
    for (int J = 0; J <= tj; J++) n += J / 2 + 1;
    return n;
}
// accumulator index of column (mb, n = J - mb), n >= mb: mb-major, the order in which the kernel produces them
constexpr int dft_index(int tj, int mb, int n) {
    int idx = 0;
    for (int m = 0; m < mb; m++) idx += tj - 2 * m + 1;
    return idx + (n - mb);
}

// resident CTAs per SM: the 4 * dft_njm accumulator registers per thread decide
constexpr int dft_ctas(int tj) { return tj >= 8 ? 1 : (tj >= 6 ? 2 : 3); }
// From twojmax 8 up the sums of a sample would take 100..144 of the 168 registers and leave the compiler no room to run two
// multiplication chains side by side; there the columns are accumulated in two passes over the neighbors of the tile, chains
// mb < dft_split first, the others second (u, v and w are computed twice: +20 of 224 FP64 instructions per neighbor).
#ifndef MALA_DFT_SPLIT
#define MALA_DFT_SPLIT 1
#endif
#ifndef MALA_DFT_TWO_MIN
#define MALA_DFT_TWO_MIN 9
#endif
constexpr int dft_split(int tj) { return tj >= MALA_DFT_TWO_MIN ? MALA_DFT_SPLIT : tj / 2 + 1; }
// byte offset of the phase-1 buffers (pair geometry, candidate records, hit masks) inside the sample array S: behind the
// columns of the first pass when there are two (S of the first pass is written while the geometry is still needed)
constexpr size_t dft_phase1_offset(int tj) {
    return dft_split(tj) > tj / 2 ? 0 : (size_t)dft_index(tj, dft_split(tj), dft_split(tj)) * (tj + 1) * 32 * sizeof(double2);
}

// sums of the columns of chains MB0 <= mb < MB1 over the queued neighbors of this lane's point, added to acc
template <int TJ, int MB0, int MB1>
__device__ __forceinline__ void dft_accumulate(const double *geo, const int lane, const int cnt, const double xsr, const double xsi,
                                               double (&accr)[dft_njm(TJ)], double (&acci)[dft_njm(TJ)]) {
    constexpr int K0 = dft_index(TJ, MB0, MB0);
    const int nmax = __reduce_max_sync(0xffffffffu, cnt);
#pragma unroll kDftUnroll
    for (int i = 0; i < nmax; i++) {
        double c = 0.0, ar = 1.0, ai = 0.0, br = 0.0, bi = 0.0;   // lanes past their count add zeros
        if (i < cnt) {
            const double *q = geo + (size_t)i * 5 * 32 + lane;
            c = q[0]; ar = q[32]; ai = q[64]; br = q[96]; bi = q[128];
        }
        // u = b + a x_s,  v = conj(a) - conj(b) x_s,  w = u v
        const double ur = fma(-ai, xsi, fma(ar, xsr, br)), ui = fma(ai, xsr, fma(ar, xsi, bi));
        const double vr = ar - fma(bi, xsi, br * xsr), vi = -ai - fma(-bi, xsr, br * xsi);
        const double wr = fma(-ui, vi, ur * vr), wi = fma(ui, vr, ur * vi);
        double pr = c, pi = 0.0;   // c w^mb
#pragma unroll
        for (int mb = 0; mb < MB0; mb++) {
            const double tr = fma(-pi, wi, pr * wr), ti = fma(pi, wr, pr * wi);
            pr = tr; pi = ti;
        }
#pragma unroll
        for (int mb = MB0; mb < MB1; mb++) {
            double zr = pr, zi = pi;   // c u^mb v^n, n = mb .. TJ - mb
            accr[dft_index(TJ, mb, mb) - K0] += zr;
            acci[dft_index(TJ, mb, mb) - K0] += zi;
#pragma unroll
            for (int n = mb + 1; n <= TJ - mb; n++) {
                const double tr = fma(-zi, vi, zr * vr), ti = fma(zi, vr, zr * vi);
                zr = tr; zi = ti;
                accr[dft_index(TJ, mb, n) - K0] += zr;
                acci[dft_index(TJ, mb, n) - K0] += zi;
            }
            if (mb + 1 < MB1) {
                const double tr = fma(-pi, wi, pr * wr), ti = fma(pi, wr, pr * wi);
                pr = tr; pi = ti;
            }
        }
    }
}

template <int TJ>
__global__ void __launch_bounds__((TJ + 1) * 32, dft_ctas(TJ))
compute_ui_dft_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb) {
    constexpr int NW = TJ + 1;          // warps = sample points
    constexpr int NJM = dft_njm(TJ);
    constexpr int nelem = uhalf_size(TJ);
    constexpr int SPLIT = dft_split(TJ);
    constexpr bool TWO = SPLIT <= TJ / 2;   // two accumulation passes
    constexpr int KA = TWO ? dft_index(TJ, SPLIT, SPLIT) : NJM;   // columns of the first pass
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // S [NJM][NW][32] double2, the samples of every column; phase 1 (bytes of S that are not yet in use): geo [kDftCap][5][32],
    // crec [kDftCap][6], hmask [NW][32]
    double2 *S = reinterpret_cast<double2 *>(smem_raw);
    double *geo = reinterpret_cast<double *>(smem_raw + dft_phase1_offset(TJ));
    double *crec = geo + kDftCap * 5 * 32;
    unsigned long long *hmask = reinterpret_cast<unsigned long long *>(crec + kDftCap * 6);   // [NW][32] hit masks of the warps
    __shared__ int s_item;
    __shared__ double2 s_tw[NW * NW];   // [k][s] = x_s^(-k) = e^{-2 pi i s k / NW}
    __shared__ unsigned short s_col[NJM];      // work order of the inverse DFT: column (J << 4 | mb), longest columns first
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x < NW * NW) {
        double sn, cs;
        sincospi(2.0 * (double)(((threadIdx.x / NW) * (threadIdx.x % NW)) % NW) / (double)NW, &sn, &cs);
        s_tw[threadIdx.x] = make_double2(cs, -sn);
    }
    if (threadIdx.x == 0) {   // columns by decreasing length, dealt to the warps round-robin
        int n = 0;
        for (int J = TJ; J >= 0; J--)
            for (int mb = 0; mb <= J / 2; mb++) s_col[n++] = (unsigned short)((J << 4) | mb);
    }
    double xsr, xsi;                    // this warp's sample point x_s = e^{2 pi i s / NW}
    {
        double sn, cs;
        sincospi(2.0 * (double)warp / (double)NW, &sn, &cs);
        xsr = cs; xsi = sn;
    }

    for (;;) {
        __syncthreads();  // everybody is done with the previous tile (S reads, s_item)
        if (threadIdx.x == 0) s_item = atomicAdd(&cb.counters[1], 1);
        __syncthreads();
        const int slot = s_item;
        if (slot >= cb.counters[0]) break;
        const int wt = cb.active[slot];
        const int tile = cb.tile_begin + wt;
        int ix, iy, iz;
        bool valid;
        lane_point(g, tile, lane, ix, iy, iz, valid);
        ix = min(ix, g.nx - 1); iy = min(iy, g.ny - 1); iz = min(iz, g.z1 - 1);  // ragged tiles: a valid point whose result is never used
        double px, py, pz;
        point_position(g, ix, iy, iz, px, py, pz);
        const int nc = cb.ncand[wt];
        const int *mycand = cb.cand + (size_t)wt * cb.cand_cap;

        // one window of candidates: distance tests, then the pair geometry of the hits queued per point in geo; returns the
        // number of neighbors of this lane's point in the window
        auto window = [&](const int wbase) {
            const int nw = min(kDftCap, nc - wbase);
            __syncthreads();  // crec, hmask and geo free again
            if ((int)threadIdx.x < nw) {
                const Ghost gh = cb.ghosts[mycand[wbase + threadIdx.x]];
                const double rc = tb.type_rcut[gh.type];
                double *q = crec + threadIdx.x * 6;
                q[0] = gh.x; q[1] = gh.y; q[2] = gh.z; q[3] = rc; q[4] = tb.type_w[gh.type]; q[5] = rc * rc;
            }
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
            // the hits of a point (in candidate order) are dealt to the NW lanes of that point: pair geometry once per pair
            int e = 0, turn = 0;   // turn = e mod NW
            for (unsigned long long r = hits; r != 0ull; r &= r - 1ull, e++) {
                if (turn == warp) {
                    const double *q = crec + (__ffsll((long long)r) - 1) * 6;
                    const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    double c, ar, ai, br, bi;
                    pair_geometry(dx, dy, dz, r2, q[3], q[4], sc.rfac0, sc.rmin0, c, ar, ai, br, bi);
                    double *o = geo + (size_t)e * 5 * 32 + lane;
                    o[0] = c; o[32] = ar; o[64] = ai; o[96] = br; o[128] = bi;
                }
                turn = (turn + 1 == NW) ? 0 : turn + 1;
            }
            __syncthreads();
            return __popcll(hits);
        };

        int cnt = 0;
        {   // first pass (the only one below twojmax 8)
            double accr[NJM], acci[NJM];   // KA of them in use
#pragma unroll
            for (int k = 0; k < KA; k++) { accr[k] = 0.0; acci[k] = 0.0; }
            for (int wbase = 0; wbase < nc; wbase += kDftCap) {
                cnt = window(wbase);
                dft_accumulate<TJ, 0, TWO ? SPLIT : TJ / 2 + 1>(geo, lane, cnt, xsr, xsi, accr, acci);
            }
            if (!TWO) __syncthreads();  // geo is dead: its bytes become S
#pragma unroll
            for (int k = 0; k < KA; k++) S[((size_t)k * NW + warp) * 32 + lane] = make_double2(accr[k], acci[k]);
        }
        if constexpr (TWO) {   // second pass: the geometry of a single window is still there, several windows are walked again
            double accr[NJM], acci[NJM];   // NJM - KA of them in use
#pragma unroll
            for (int k = 0; k < NJM - KA; k++) { accr[k] = 0.0; acci[k] = 0.0; }
            if (nc <= kDftCap) dft_accumulate<TJ, SPLIT, TJ / 2 + 1>(geo, lane, cnt, xsr, xsi, accr, acci);
            else
                for (int wbase = 0; wbase < nc; wbase += kDftCap) {
                    cnt = window(wbase);
                    dft_accumulate<TJ, SPLIT, TJ / 2 + 1>(geo, lane, cnt, xsr, xsi, accr, acci);
                }
            __syncthreads();  // geo is dead: its bytes become S
#pragma unroll
            for (int k = 0; k < NJM - KA; k++) S[((size_t)(KA + k) * NW + warp) * 32 + lane] = make_double2(accr[k], acci[k]);
        }
        __syncthreads();
        // inverse DFT per column: q_k = (1/NW) sum_s S_s x_s^(-k); then the binomial normalisation and the self term
        double2 *dst = cb.utot + (size_t)slot * nelem * 32;
        for (int c = warp; c < NJM; c += NW) {   // one column per trip: its NW samples in registers, all of its J + 1 coefficients
            const int J = s_col[c] >> 4, mb = s_col[c] & 15;
            const double2 *Sp = S + (size_t)dft_index(TJ, mb, J - mb) * NW * 32 + lane;
            // x_{NW-s} = conj(x_s): with P = S_s + S_{NW-s}, M = S_s - S_{NW-s} a pair of samples costs four multiply-adds, not eight:
            // S_s t + S_{NW-s} conj(t) = (Pr c - Mi d) + i (Pi c + Mr d),  t = x_s^(-k) = c + i d
            constexpr int NP = (NW - 1) / 2;
            double pr_[NP > 0 ? NP : 1], pi_[NP > 0 ? NP : 1], mr_[NP > 0 ? NP : 1], mi_[NP > 0 ? NP : 1];
            const double2 v0 = Sp[0];
            double2 vh = make_double2(0.0, 0.0);   // the sample at x = -1 (even NW only)
            if constexpr (NW % 2 == 0) vh = Sp[(size_t)(NW / 2) * 32];
#pragma unroll
            for (int sI = 1; sI <= NP; sI++) {
                const double2 va = Sp[(size_t)sI * 32], vb = Sp[(size_t)(NW - sI) * 32];
                pr_[sI - 1] = va.x + vb.x; pi_[sI - 1] = va.y + vb.y;
                mr_[sI - 1] = va.x - vb.x; mi_[sI - 1] = va.y - vb.y;
            }
            const int e0 = uhalf_off(J) + mb * (J + 1);
#pragma unroll 2
            for (int k = 0; k <= J; k++) {
                const double2 *tw = s_tw + k * NW;
                const double sg = (k & 1) ? -1.0 : 1.0;
                double sr = fma(sg, vh.x, v0.x), si = fma(sg, vh.y, v0.y);
#pragma unroll
                for (int sI = 1; sI <= NP; sI++) {
                    const double2 t = tw[sI];
                    sr = fma(pr_[sI - 1], t.x, sr); sr = fma(-mi_[sI - 1], t.y, sr);
                    si = fma(pi_[sI - 1], t.x, si); si = fma(mr_[sI - 1], t.y, si);
                }
                const int e = e0 + k;
                const double sN = tb.unorm[e] * (1.0 / (double)NW);
                dst[(size_t)e * 32 + lane] = make_double2(sr * sN + (tb.udiag[e] ? sc.wself : 0.0), si * sN);
            }
        }
    }
}

template <int TJ>
inline size_t compute_ui_dft_smem_bytes() {
    const size_t phase1 = dft_phase1_offset(TJ) + (size_t)kDftCap * 5 * 32 * sizeof(double) + (size_t)kDftCap * 6 * sizeof(double) +
                          (size_t)(TJ + 1) * 32 * sizeof(unsigned long long);
    const size_t phase2 = (size_t)(TJ + 1) * dft_njm(TJ) * 32 * sizeof(double2);
    return (phase1 > phase2 ? phase1 : phase2) + 16;
}

}  // namespace mala
