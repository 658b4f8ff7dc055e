// snap_zi_coop.cuh -- compute_zi / compute_bi specialised at compile time for twojmax = 10 (rows a5 + a6 + a7).
//
// Arithmetic.  For a triple (J1,J2,J), output column mb and one (mb1, mb2 = mb + sh - mb1) pair -- an "item" --
//     z[ma] += cgb * sum_{ma1 + ma2 - sh = ma} CG(ma1, ma2) * x[ma1] * y[ma2],   x = U^{J1}[:, mb1], y = U^{J2}[:, mb2]
// is a CG-weighted 1-D convolution of two columns.  x (<= 11 complex) and z (<= 11 complex) live in registers, y is
// streamed one element at a time (pre-multiplied by cgb and by the sign/conjugation of the column-flip symmetry),
// and the (ma1, ma2) loops are unrolled at compile time so every register index and every CG address is static; the
// CG values are constant-memory operands of the DMUL instructions.  6 FP64-pipe instructions per product term,
// ~0.25 B of shared-memory traffic per flop.  compute_bi is fused: a finished run of items of one column is folded
// into B at once (B is linear in Z), so Z is never stored.
//
// Schedule.  A CTA owns one tile (32 grid points = the lanes of every warp; U_tot of the tile TMA-loaded into shared
// memory).  ALL warps of the CTA work on the SAME triple at the same time: the items of a triple are dealt to the
// warps as contiguous runs whose lengths follow a round-robin deal over the whole tile (so the load is balanced
// across triples, not only within one).  The first version of this kernel gave every warp a triple of its own; with
// ~13 KB of straight-line code per triple that made the SM fetch eight instruction streams at once and ncu showed
// 25 "no instruction" stall cycles per issued instruction (profiles/r01_baseline.md).  Same-triple scheduling keeps the
// instruction working set at one or two loop bodies.
// Partial B values go through a small double-buffered shared-memory array and are summed in a fixed order every
// eight triples, so results are bit-reproducible.
#pragma once
#include "snap_zi.cuh"

namespace mala {

constexpr int kSpecTJ = 10;
constexpr int kSpecNT = triple_count(kSpecTJ);
constexpr int kSpecCG = cg_block_off(kSpecTJ, kSpecNT);
#ifndef MALA_COOP_WARPS
#define MALA_COOP_WARPS 12
#endif
#ifndef MALA_COOP_GROUP
#define MALA_COOP_GROUP 8
#endif
constexpr int kCoopWarps = MALA_COOP_WARPS;   // warps per CTA
#ifndef MALA_COOP_TEAMS
#define MALA_COOP_TEAMS 2
#endif
constexpr int kCoopTeams = MALA_COOP_TEAMS;   // warp teams working on different triples at the same time
constexpr int kCoopGroup = MALA_COOP_GROUP;   // triples between two reductions of the partial sums

__constant__ double c_cg_spec[kSpecCG];                        // dense CG blocks of every triple, [m2][m1]
__constant__ int c_order_spec[kSpecNT];                        // triples by decreasing cost
constexpr int kTeamWarps = kCoopWarps / kCoopTeams;           // warps per team
constexpr int kListMax = kSpecNT + kSpecNT / kCoopGroup + 4;  // entries of one warp's work list
// One work list per warp, built on the host (mala_snap.cu): the triples of the warp's team in processing order with the
// warp's item range, interleaved with one entry per reduction group.
//   work entry:  bit 31 = 0 | buf << 27 | k << 23 | end << 15 | begin << 7 | triple      (k = slot of the triple in its group)
//   sync entry:  bit 31 = 1 | first position of the group << 8 | buf << 4 | last k
//   0xffffffff terminates the list
__constant__ unsigned int c_wlist[kCoopWarps][kListMax];

constexpr int kRowBytes = 32 * (int)sizeof(double2);  // bytes between consecutive elements of one lane

// Stretched triples (J = J1 + J2, shift 0): CG(ma1, ma2 | ma) = sqrt(C(J1,ma1) C(J2,ma2) / C(J,ma)) is a product of one
// factor per index, so x and y are pre-scaled once per item and z once per column; the product terms then need no CG
// multiplication (4 FP64 instructions instead of 6, and a third less code).  Used when both columns have >= 2 rows.
__constant__ double c_sqbin[kSpecTJ + 1][kSpecTJ + 1];   // sqrt(C(J, m))
__constant__ double c_isqbin[kSpecTJ + 1][kSpecTJ + 1];  // 1 / sqrt(C(J, m))
constexpr bool item_stretched(int J1, int J2, int J) { return J == J1 + J2 && J2 >= 1; }

// Items of output column mb: mb1 in [item_lo, item_hi], mb2 = mb + sh - mb1.
// J1 == J2: the items (mb1, mb2) and (mb2, mb1) contribute the same Z column (swap the two factors and use
// CG(j1 m1 j1 m2 | j m) = +-CG(j1 m2 j1 m1 | j m) for both coefficients), so only mb1 <= mb2 is computed, with weight 2
// when mb1 < mb2.
// J == J1 (and J1 != J2): U^{J1} and U^J are the same matrix, and the contribution of item (mb, mb1) to B equals that
// of item (mb1, mb) (swap the roles of the two factors; the third one turns into its mirror element, whose sign and
// conjugation cancel against the CG symmetry).  Together with the column flip (mb, mb1) -> (J - mb, J - mb1) already
// used, the items mb <= mb1 <= J - mb of the columns mb <= J/2 represent all of them: weight 2 unless mb1 == mb or
// mb1 == J - mb.  Checked against the oracle's U and CG to 1e-15 before use.
constexpr bool item_hermitian(int J1, int J2, int J) { return J == J1 && J1 != J2; }
// J1 == J2 == J: both of the above hold, i.e. the contribution of an item is symmetric under every permutation of its
// three column indices mu1 = mb1 - J/2, mu2 = mb2 - J/2, mu3 = J/2 - mb (sum zero) and under their common sign change.
// One item per class is computed: mu1 <= mu2 <= mu3 with mu2 <= 0, i.e. mb <= mb1 <= (mb + J/2)/2 in the columns
// mb <= J/2, weighted with the class size (permutations 6, 3 or 1, times 2 unless mu2 == 0).
// Used by the anti-diagonal kernel (snap_zi_diag.cuh).  In this kernel it is switched off: it halves the items of the five
// (J, J, J) triples (-4 % product terms), but those are the triples with the largest loop bodies, whose time is set by
// fetching the body, not by the number of passes through it -- measured 23.91 ms with it against 23.52 ms without.
constexpr bool kCoopSymmetric3 = false;
constexpr bool item_symmetric3(int J1, int J2, int J) { return kCoopSymmetric3 && J == J1 && J1 == J2; }
__host__ __device__ constexpr double item_weight3(int J, int mb, int mb1) {
    const int mu1 = mb1 - J / 2, mu3 = J / 2 - mb, mu2 = -mu1 - mu3;
    const int perms = (mu1 == mu2 && mu2 == mu3) ? 1 : ((mu1 == mu2 || mu2 == mu3) ? 3 : 6);
    const int both = (mu2 == 0) ? 1 : 2;
    return (double)(perms * both) / ((mb == J / 2) ? 1.0 : 2.0);  // columns below the middle are doubled at the fold
}
constexpr int item_lo(int J1, int J2, int J, int mb) {
    const int s = mb + (J1 + J2 - J) / 2;
    int lo = (s - J2) > 0 ? (s - J2) : 0;
    if ((item_hermitian(J1, J2, J) || item_symmetric3(J1, J2, J)) && lo < mb) lo = mb;
    return lo;
}
constexpr int item_hi(int J1, int J2, int J, int mb) {
    const int s = mb + (J1 + J2 - J) / 2;
    int hi = s < J1 ? s : J1;
    if (J1 == J2 && s / 2 < hi) hi = s / 2;
    if (item_hermitian(J1, J2, J) && J - mb < hi) hi = J - mb;
    return hi;
}
// the middle column of an even J needs rows ma <= J/2 only (the others are its mirror images)
constexpr bool is_mid(int J, int mb) { return (J % 2 == 0) && (mb == J / 2); }
// The half-row body of the middle column is extra code to fetch for every tile: it pays only when the middle column has
// enough items (MALA_COOP_MID_MIN, tuned on B200); otherwise the column runs through the full-column body at half weight.
#ifndef MALA_COOP_MID_MIN
#define MALA_COOP_MID_MIN 2
#endif
constexpr bool use_mid_body(int J1, int J2, int J) {
    return (J % 2 == 0) && (item_hi(J1, J2, J, J / 2) - item_lo(J1, J2, J, J / 2) + 1 >= MALA_COOP_MID_MIN);
}

// number of (mb, mb1) items of a triple: columns mb = 0..J/2
constexpr int triple_items(int J1, int J2, int J) {
    int n = 0;
    for (int mb = 0; mb <= J / 2; mb++) n += item_hi(J1, J2, J, mb) - item_lo(J1, J2, J, mb) + 1;
    return n;
}
// product terms of one item of column mb (the cost unit of the schedule)
constexpr int item_terms(int J1, int J2, int J, int mb) {
    const int sh = (J1 + J2 - J) / 2, mahi = (is_mid(J, mb) && use_mid_body(J1, J2, J)) ? J / 2 : J;
    int n = 0;
    for (int m2 = 0; m2 <= J2; m2++)
        for (int m1 = 0; m1 <= J1; m1++)
            if (m1 + m2 - sh >= 0 && m1 + m2 - sh <= mahi) n++;
    return n;
}

__device__ __forceinline__ double flip_sign(double v, unsigned mask) {
    return __hiloint2double(__double2hiint(v) ^ (int)mask, __double2loint(v));
}

// z[ma] += sum CG * x[ma1] * (scaled y[ma2]) for one item
template <int J1, int J2, int J, int CGOFF, int MAHI>
__device__ __forceinline__ void cg_convolve(double (&zr)[J + 1], double (&zi)[J + 1], const double (&xr)[J1 + 1],
                                            const double (&xi)[J1 + 1], const unsigned char *ybase, const int ystep,
                                            const double sre0, const double sre1, const double sim0, const double sim1) {
    constexpr int SH = (J1 + J2 - J) / 2;
#pragma unroll
    for (int ma2 = 0; ma2 <= J2; ma2++) {
        const int lo = (SH - ma2) > 0 ? (SH - ma2) : 0;
        const int hi = (MAHI + SH - ma2) < J1 ? (MAHI + SH - ma2) : J1;
        if (lo <= hi) {
            const double2 yv = *reinterpret_cast<const double2 *>(ybase + ma2 * ystep);
            double yr = yv.x * ((ma2 & 1) ? sre1 : sre0);
            double yi = yv.y * ((ma2 & 1) ? sim1 : sim0);
            if (item_stretched(J1, J2, J)) {
                yr *= c_sqbin[J2][ma2];
                yi *= c_sqbin[J2][ma2];
            }
#pragma unroll
            for (int ma1 = 0; ma1 <= J1; ma1++) {
                if (ma1 >= lo && ma1 <= hi) {
                    const int ma = ma1 + ma2 - SH;
                    const double cg = c_cg_spec[CGOFF + ma2 * (J1 + 1) + ma1];
                    const double tr = item_stretched(J1, J2, J) ? xr[ma1] : cg * xr[ma1];  // x carries sqrt(C(J1,ma1)) already
                    const double ti = item_stretched(J1, J2, J) ? xi[ma1] : cg * xi[ma1];
                    zr[ma] = fma(tr, yr, zr[ma]);
                    zr[ma] = fma(-ti, yi, zr[ma]);
                    zi[ma] = fma(tr, yi, zi[ma]);
                    zi[ma] = fma(ti, yr, zi[ma]);
                }
            }
        }
    }
}

// items mb1 in [mb1_begin, mb1_end) of output column mb: returns their contribution to B.
// MID: mb is the middle column of an even J; only rows ma <= J/2 are formed.
// x = U^{J1}[:, mb1]; columns beyond the middle come from the stored half by u[ma][mb] = (-1)^(ma-mb) conj(u[J-ma][J-mb])
template <int J1>
__device__ __forceinline__ void load_x_column(const unsigned char *Ulane, const int mb1, double (&xr)[J1 + 1], double (&xi)[J1 + 1]) {
    if (mb1 <= J1 / 2) {  // stored column: plain loads (the branch is warp-uniform)
        const unsigned char *xb = Ulane + (uhalf_off(J1) + mb1 * (J1 + 1)) * kRowBytes;
#pragma unroll
        for (int k = 0; k <= J1; k++) {
            const double2 v = *reinterpret_cast<const double2 *>(xb + k * kRowBytes);
            xr[k] = v.x;
            xi[k] = v.y;
        }
    } else {  // mirror column, read backwards; real part (-1)^(ma1-mb1), imaginary part the opposite (conjugation)
        const unsigned char *xb = Ulane + (uhalf_off(J1) + (J1 - mb1) * (J1 + 1) + J1) * kRowBytes;
        const unsigned m0 = (mb1 & 1) ? 0x80000000u : 0u;
#pragma unroll
        for (int k = 0; k <= J1; k++) {
            const double2 v = *reinterpret_cast<const double2 *>(xb - k * kRowBytes);
            xr[k] = flip_sign(v.x, (k & 1) ? (m0 ^ 0x80000000u) : m0);
            xi[k] = flip_sign(v.y, (k & 1) ? m0 : (m0 ^ 0x80000000u));
        }
    }
}

// weight of item (mb, mb1): the CG factor of its column pair times the number of items it stands for
template <int J1, int J2, int J, int CGOFF>
__device__ __forceinline__ double item_cgb(const int mb, const int mb1) {
    constexpr int SH = (J1 + J2 - J) / 2;
    const int mb2 = mb + SH - mb1;
    double cgb = c_cg_spec[CGOFF + mb2 * (J1 + 1) + mb1];
    if (item_symmetric3(J1, J2, J)) cgb *= item_weight3(J, mb, mb1);  // stands for its whole symmetry class
    else if (J1 == J2 && mb1 != mb2) cgb += cgb;                        // stands for its mirror item (mb2, mb1) too
    if (item_hermitian(J1, J2, J) && mb1 != mb && mb1 != J - mb) cgb += cgb;  // and for item (mb1, mb)
    return cgb;
}

// y = U^{J2}[:, mb2] with the same column symmetry, folded with cgb into four scale factors
template <int J2>
__device__ __forceinline__ void y_column(const unsigned char *Ulane, const int mb2, const double cgb, const unsigned char *&yb, int &ystep,
                                         double &p0, double &p1, double &q0, double &q1) {
    const bool fy = mb2 > J2 / 2;
    const int cy = fy ? J2 - mb2 : mb2;
    yb = Ulane + (uhalf_off(J2) + cy * (J2 + 1) + (fy ? J2 : 0)) * kRowBytes;
    ystep = fy ? -kRowBytes : kRowBytes;
    p0 = (fy && (mb2 & 1)) ? -cgb : cgb;  // parity-0 rows, real part
    p1 = fy ? -p0 : cgb;                  // parity-1 rows, real part
    q0 = fy ? -p0 : cgb;                  // imaginary parts: conjugation flips the sign again
    q1 = fy ? -p1 : cgb;
}

template <int J1, int J2, int J, int CGOFF, bool MID>
__device__ __forceinline__ double column_segment(const unsigned char *Ulane, const int mb, const int mb1_begin, const int mb1_end) {
    constexpr int SH = (J1 + J2 - J) / 2;
    constexpr int MAHI = MID ? J / 2 : J;
    double zr[J + 1], zi[J + 1];
#pragma unroll
    for (int k = 0; k <= J; k++) { zr[k] = 0.0; zi[k] = 0.0; }
#pragma unroll 1
    for (int mb1 = mb1_begin; mb1 < mb1_end; mb1++) {
        double xr[J1 + 1], xi[J1 + 1];
        load_x_column<J1>(Ulane, mb1, xr, xi);
        if (item_stretched(J1, J2, J)) {
#pragma unroll
            for (int k = 0; k <= J1; k++) {
                xr[k] *= c_sqbin[J1][k];
                xi[k] *= c_sqbin[J1][k];
            }
        }
        const unsigned char *yb;
        int ystep;
        double p0, p1, q0, q1;
        y_column<J2>(Ulane, mb + SH - mb1, item_cgb<J1, J2, J, CGOFF>(mb, mb1), yb, ystep, p0, p1, q0, q1);
        cg_convolve<J1, J2, J, CGOFF, MAHI>(zr, zi, xr, xi, yb, ystep, p0, p1, q0, q1);
    }
    // compute_bi: B += w * Re(conj(U^J[ma][mb]) * z[ma]).  Columns below the middle stand for their mirror images
    // too (w = 2); in the middle column of an even J rows ma < J/2 stand for rows J - ma (w = 2), the centre counts once.
    const unsigned char *ub = Ulane + (uhalf_off(J) + mb * (J + 1)) * kRowBytes;
    double bp[4] = {0.0, 0.0, 0.0, 0.0};  // independent partial sums: no 2(J+1)-deep dependent DFMA chain
    if (item_stretched(J1, J2, J)) {
#pragma unroll
        for (int ma = 0; ma <= (MID ? J / 2 : J); ma++) {
            zr[ma] *= c_isqbin[J][ma];
            zi[ma] *= c_isqbin[J][ma];
        }
    }
#pragma unroll
    for (int ma = 0; ma < (MID ? J / 2 : J + 1); ma++) {
        const double2 u = *reinterpret_cast<const double2 *>(ub + ma * kRowBytes);
        bp[(2 * ma) & 3] = fma(u.x, zr[ma], bp[(2 * ma) & 3]);
        bp[(2 * ma + 1) & 3] = fma(u.y, zi[ma], bp[(2 * ma + 1) & 3]);
    }
    double b = (bp[0] + bp[1]) + (bp[2] + bp[3]);
    b += b;
    if (MID) {
        const double2 u = *reinterpret_cast<const double2 *>(ub + (J / 2) * kRowBytes);
        b = fma(u.x, zr[J / 2], b);
        b = fma(u.y, zi[J / 2], b);
    }
    return b;
}

// this warp's items [begin, end) of triple T (items numbered column by column)
template <int T>
__device__ __noinline__ double triple_items_b(const unsigned char *Ulane, const int begin, const int end) {
    constexpr Triple tr = triple_at(kSpecTJ, T);
    constexpr int J1 = tr.j1, J2 = tr.j2, J = tr.j;
    constexpr int CGOFF = cg_block_off(kSpecTJ, T);
    constexpr int NFULL = (J % 2 == 0) ? J / 2 : J / 2 + 1;  // columns computed in full
    double b = 0.0;
    int base = 0;
#pragma unroll 1
    for (int mb = 0; mb < NFULL; mb++) {
        const int lo = item_lo(J1, J2, J, mb), nb = item_hi(J1, J2, J, mb) - lo + 1;
        const int s = max(begin, base), e = min(end, base + nb);
        if (s < e) b += column_segment<J1, J2, J, CGOFF, false>(Ulane, mb, lo + s - base, lo + e - base);
        base += nb;
    }
    if (J % 2 == 0) {
        constexpr int lo = item_lo(J1, J2, J, J / 2), nb = item_hi(J1, J2, J, J / 2) - lo + 1;
        const int s = max(begin, base), e = min(end, base + nb);
        // the half-row body pays for its code only when the middle column has several items; with the j == j1 symmetry
        // it has a single one, which then runs through the full-column body (weight 2 there, hence the 0.5)
        if constexpr (!use_mid_body(J1, J2, J)) {
            if (s < e) b += 0.5 * column_segment<J1, J2, J, CGOFF, false>(Ulane, J / 2, lo + s - base, lo + e - base);
        } else {
            if (s < e) b += column_segment<J1, J2, J, CGOFF, true>(Ulane, J / 2, lo + s - base, lo + e - base);
        }
    }
    return b;
}

__device__ __forceinline__ double dispatch_triple(const int t, const unsigned char *Ulane, const int begin, const int end) {
    double b = 0.0;
    switch (t) {
#define MALA_CASE(N) \
    case N:          \
        if (N < kSpecNT) b = triple_items_b<(N < kSpecNT ? N : 0)>(Ulane, begin, end); \
        break;
#define MALA_CASE10(D) \
    MALA_CASE(D * 10 + 0) MALA_CASE(D * 10 + 1) MALA_CASE(D * 10 + 2) MALA_CASE(D * 10 + 3) MALA_CASE(D * 10 + 4) \
    MALA_CASE(D * 10 + 5) MALA_CASE(D * 10 + 6) MALA_CASE(D * 10 + 7) MALA_CASE(D * 10 + 8) MALA_CASE(D * 10 + 9)
        MALA_CASE10(0) MALA_CASE10(1) MALA_CASE10(2) MALA_CASE10(3) MALA_CASE10(4)
        MALA_CASE10(5) MALA_CASE10(6) MALA_CASE10(7) MALA_CASE10(8) MALA_CASE10(9)
#undef MALA_CASE10
#undef MALA_CASE
        default: break;
    }
    return b;
}

__global__ void __launch_bounds__(kCoopWarps * 32, 1)
compute_zi_bi_coop_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb, double *out) {
    static_assert(kSpecNT <= 100, "dispatch_triple covers 100 cases");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int nelem = uhalf_size(kSpecTJ), nt = kSpecNT, NW = kCoopWarps, TW = kTeamWarps;
    double2 *U = reinterpret_cast<double2 *>(smem_raw);
    double *Bs = reinterpret_cast<double *>(U + (size_t)nelem * 32);
    double *red = Bs + 32 * nt;  // [2][kCoopGroup][TW][32]: partial sums of the warps of the triple's team
    __shared__ uint64_t bar;
    __shared__ int s_slot;
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int wk = warp % TW;
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    uint32_t parity = 0;
    const int nactive = cb.counters[0];
    if (threadIdx.x == 0) s_slot = atomicAdd(&cb.counters[2], 1);
    for (;;) {
        __syncthreads();  // previous tile written out: Bs and U are free; s_slot is visible
        const int slot = s_slot;
        if (slot >= nactive) break;
        const int wt = cb.active[slot];
        __syncthreads();  // everybody has read s_slot
        if (threadIdx.x == 0) {
            tma_load_tile(U, cb.utot + (size_t)slot * nelem * 32, nelem, &bar);
            // claim the next tile now and pull its U_tot into L2 while this one is being worked on
            const int next = atomicAdd(&cb.counters[2], 1);
            s_slot = next;
            if (next < nactive) prefetch_l2_tile(cb.utot + (size_t)next * nelem * 32, nelem);
        }
        mbar_wait(&bar, parity);
        parity ^= 1u;
        const unsigned char *Ulane = reinterpret_cast<const unsigned char *>(U + lane);
        for (int i = 0;; i++) {
            const unsigned e = c_wlist[warp][i];
            if (e == 0xffffffffu) break;
            if ((e >> 31) == 0u) {
                const int t = (int)(e & 127u), begin = (int)((e >> 7) & 255u), end = (int)((e >> 15) & 255u);
                double b = 0.0;
                if (begin < end) b = dispatch_triple(t, Ulane, begin, end);
                red[(((e >> 23) & 31u) * TW + wk) * 32 + lane] = b;  // (buf * kCoopGroup + k) in one field
            } else {
                __syncthreads();
                // fixed-order sum of the partials of the triples of this group
                const int klast = (int)(e & 15u), base = (int)((e >> 4) & 1u) * kCoopGroup, pos0 = (int)((e >> 8) & 255u);
                for (int kk = warp; kk <= klast; kk += NW) {
                    const double *r = red + ((base + kk) * TW) * 32 + lane;
                    double s = 0.0;
#pragma unroll
                    for (int w2 = 0; w2 < TW; w2++) s += r[w2 * 32];
                    Bs[lane * nt + c_order_spec[pos0 + kk]] = s;
                }
            }
        }
        __syncthreads();
        write_tile(g, cb.tile_begin + wt, Bs, nt, out, NW, cb.compact_out, wt);
    }
}

inline size_t compute_zi_coop_smem_bytes() {
    return (size_t)uhalf_size(kSpecTJ) * 32 * sizeof(double2) + (size_t)32 * kSpecNT * sizeof(double) +
           (size_t)2 * kCoopGroup * kTeamWarps * 32 * sizeof(double) + 16;
}

}  // namespace mala
