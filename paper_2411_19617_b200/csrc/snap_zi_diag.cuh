// snap_zi_diag.cuh -- compute_zi / compute_bi with anti-diagonal accumulators (rows a5 + a6 + a7), any twojmax <= 14.
//
// Same arithmetic as snap_zi_coop.cuh (an *item* = triple (J1,J2,J), output column mb, one (mb1, mb2) pair; its Z column
// is a CG-weighted 1-D convolution of x = U^{J1}[:, mb1] and y = U^{J2}[:, mb2]), organised so that the code depends on
// J1 only:
//   * the accumulators are indexed by the anti-diagonal d = ma1 + k of the (ma1, row) rectangle, r[0 .. 2 J1], with
//     the rows k = ma2 + (J1 - J2) right-aligned.  Row k touches r[k .. k + J1]: all register indices are static for a
//     body unrolled over the J1 + 1 possible rows, and a triple with fewer rows enters the body at row J1 - J2
//     (a switch with fall-through), so the rows run without any branch between them;
//   * J2, J, the shift sh = (J1 + J2 - J)/2 and the CG block are run-time values: z[ma] = r[ma + sh + J1 - J2] is
//     resolved when the column is folded into B (compute_bi), where only the *address* of conj(U^J[ma][mb]) depends on
//     it.  Products outside the band 0 <= ma <= J are computed with the zero entries of the dense CG table (+24 % FP64
//     work at twojmax = 10) -- the price for an instruction footprint of one body per J1 (mostly resident in the
//     instruction caches) instead of one body per triple (~750 KB streamed from L2 for every tile; profiles/).
// Scheduling, the fixed-order reduction of the partial sums and the writer are those of the coop kernel.
//
// Tables (CG blocks, processing order, per-warp item ranges) are per-handle arrays in global memory, read through the
// read-only path with warp-uniform addresses: handles of different twojmax can run side by side, and twojmax is not capped
// by the 64 KB constant bank.
//
// Two kernels:
//   compute_zi_bi_diag_kernel       twojmax <= 10: a 32-point tile of U_tot in shared memory, lane = grid point;
//   compute_zi_bi_diag_half_kernel  twojmax 11..14: U_tot of 32 points no longer fits one SM's shared memory, so the work
//                                   item is half a tile (16 points) and the two half-warps work on two different items of
//                                   the same triple at the same time: lane = (point, item slot).  Everything that depends
//                                   on the item (columns, flips, signs, the weight) is per-lane data; everything the code
//                                   depends on (J1, the entry row, the CG rectangle) is per-triple, hence warp-uniform.
#pragma once
#include "snap_ui.cuh"
#include "snap_zi.cuh"

namespace mala {

#ifndef MALA_DIAG_WARPS
#define MALA_DIAG_WARPS 12
#endif
#ifndef MALA_DIAG_GROUP
#define MALA_DIAG_GROUP 8
#endif
constexpr int kDiagWarps = MALA_DIAG_WARPS;  // warps per CTA, 32-point kernel
constexpr int kDiagHalfWarps = 8;            // warps per CTA, 16-point kernel (J1 up to 14 needs ~250 registers per thread)
constexpr int kDiagGroup = MALA_DIAG_GROUP;  // triples between two reductions of the partial sums
constexpr int diag_stride(int J1) { return (J1 + 2) & ~1; }  // CG row stride: J1 + 1 rounded up to even (16-byte rows)
constexpr int kDiagTeams = 2;        // warp teams working on different triples at the same time
constexpr int kDiagPadBytes = 5120;  // zeros in front of U in shared memory (see the fold in diag_segment)
constexpr int kDiagRowBytes = 32 * (int)sizeof(double2);      // 32-point tile: bytes between consecutive elements of a lane
constexpr int kDiagHalfRowBytes = 16 * (int)sizeof(double2);  // 16-point tile
// the fold reads up to d0 = sh + J1 - J2 <= J1 rows in front of a column: they must fall into the zero pad
static_assert(kDiagPadBytes >= 10 * kDiagRowBytes, "zero pad too small for the 32-point kernel (J1 <= 10)");
static_assert(kDiagPadBytes >= kMaxTwoJ * kDiagHalfRowBytes, "zero pad too small for the 16-point kernel (J1 <= kMaxTwoJ)");

struct DiagTriple {  // one entry per position of the processing order
    short J1, J2, J, index;  // index = component number in output order
    int cgoff;               // offset (in doubles, even) of the dense CG block [m2][diag_stride(J1)] in DiagTables::cg2
    int itemoff;             // offset of the triple's item descriptors in DiagTables::items
};

struct DiagTables {               // per-handle, global memory
    const double2 *cg2;           // dense CG blocks, zero where m is out of range
    const DiagTriple *triple;     // [nt] processing order: J1 descending, then cost
    const unsigned short *sched;  // [nt][warps][2] = item range [begin, end) of every warp
    const unsigned short *items;  // per triple, item -> bit 15: last item of its column | mb << 8 | mb1
};

// item range of output column mb (run-time version of item_lo / item_hi of snap_zi_coop.cuh)
__host__ __device__ inline void diag_item_range(int J1, int J2, int J, int mb, int &lo, int &hi) {
    const int s = mb + (J1 + J2 - J) / 2;
    lo = (s - J2) > 0 ? (s - J2) : 0;
    hi = s < J1 ? s : J1;
    if (J1 == J2 && s / 2 < hi) hi = s / 2;  // mirror items (mb2, mb1) are folded into weight 2
    if (J == J1 && J1 != J2) {               // item (mb, mb1) == item (mb1, mb): see item_hermitian in snap_zi_coop.cuh
        if (lo < mb) lo = mb;
        if (J - mb < hi) hi = J - mb;
    }
    if (J == J1 && J1 == J2 && lo < mb) lo = mb;  // one item per S3 x Z2 class: item_symmetric3 in snap_zi_coop.cuh
}

// class size of an item of a (J, J, J) triple over the column doubling of the fold (item_weight3 of snap_zi_coop.cuh)
__device__ __forceinline__ double diag_weight3(int J, int mb, int mb1) {
    const int mu1 = mb1 - J / 2, mu3 = J / 2 - mb, mu2 = -mu1 - mu3;
    const int perms = (mu1 == mu2 && mu2 == mu3) ? 1 : ((mu1 == mu2 || mu2 == mu3) ? 3 : 6);
    const int both = (mu2 == 0) ? 1 : 2;
    return (double)(perms * both) / ((mb == J / 2) ? 1.0 : 2.0);
}

// weight of one item: the CG factor of its column pair times the size of the symmetry class it stands for
__device__ __forceinline__ double diag_item_weight(const double *cgs, int cgoff, int S, int J1, int J2, int J, int sh, int mb, int mb1) {
    const int mb2 = mb + sh - mb1;
    double cgb = __ldg(cgs + cgoff + mb2 * S + mb1);
    if (J == J1 && J1 == J2) cgb *= diag_weight3(J, mb, mb1);
    else if (J1 == J2 && mb1 != mb2) cgb += cgb;
    if (J == J1 && J1 != J2 && mb1 != mb && mb1 != J - mb) cgb += cgb;
    return cgb;
}

__device__ __forceinline__ double diag_flip(double v, unsigned mask) {
    return __hiloint2double(__double2hiint(v) ^ (int)mask, __double2loint(v));
}

// one row of the rectangle: r[ma1 + K] += CG[row][ma1] * x[ma1] * y,  y pre-scaled.  yp walks down the y column.
template <int J1, int K>
__device__ __forceinline__ void diag_row(double (&rr)[2 * J1 + 1], double (&ri)[2 * J1 + 1], const double (&xr)[J1 + 1],
                                         const double (&xi)[J1 + 1], const unsigned char *&yp, const int ystep, const double2 *cgrow,
                                         const double se, const double so, const double te, const double to) {
    constexpr int S = diag_stride(J1);
    const double2 yv = *reinterpret_cast<const double2 *>(yp);
    yp += ystep;
    const double yr = yv.x * ((K & 1) ? so : se);
    const double yi = yv.y * ((K & 1) ? to : te);
#pragma unroll
    for (int p = 0; p <= J1 / 2; p++) {
        const double2 c2 = __ldg(cgrow + (K * S) / 2 + p);  // 16-byte load, warp-uniform address: CG of ma1 = 2p and 2p + 1
#pragma unroll
        for (int q = 0; q < 2; q++) {
            const int ma1 = 2 * p + q;
            if (ma1 <= J1) {
                const double cg = q ? c2.y : c2.x;
                const double tr = cg * xr[ma1];
                const double ti = cg * xi[ma1];
                rr[ma1 + K] = fma(tr, yr, rr[ma1 + K]);
                rr[ma1 + K] = fma(-ti, yi, rr[ma1 + K]);
                ri[ma1 + K] = fma(tr, yi, ri[ma1 + K]);
                ri[ma1 + K] = fma(ti, yr, ri[ma1 + K]);
            }
        }
    }
}

// all rows of one item, entered at row `off` = J1 - J2
template <int J1>
__device__ __forceinline__ void diag_rows(double (&rr)[2 * J1 + 1], double (&ri)[2 * J1 + 1], const double (&xr)[J1 + 1],
                                          const double (&xi)[J1 + 1], const unsigned char *yp, const int ystep, const double2 *cgrow,
                                          const int off, const double se, const double so, const double te, const double to) {
    switch (off) {
#define MALA_DIAG_ROW(K)                                                                                      \
    case K:                                                                                                   \
        if constexpr (K <= J1) diag_row<J1, (K <= J1 ? K : 0)>(rr, ri, xr, xi, yp, ystep, cgrow, se, so, te, to); \
        [[fallthrough]];
        MALA_DIAG_ROW(0) MALA_DIAG_ROW(1) MALA_DIAG_ROW(2) MALA_DIAG_ROW(3) MALA_DIAG_ROW(4) MALA_DIAG_ROW(5)
        MALA_DIAG_ROW(6) MALA_DIAG_ROW(7) MALA_DIAG_ROW(8) MALA_DIAG_ROW(9) MALA_DIAG_ROW(10) MALA_DIAG_ROW(11)
        MALA_DIAG_ROW(12) MALA_DIAG_ROW(13) MALA_DIAG_ROW(14)
#undef MALA_DIAG_ROW
        default: break;
    }
}

// compute_bi for one column: B += w * Re(conj(U^J[ma][mb]) * z[ma]), z[ma] = r[ma + d0], d0 = sh + off.  Columns below the
// middle stand for their mirror images too (w = 2).  r[d] is exactly zero wherever ma = d - d0 falls outside [0, J] (those
// products used the zero entries of the CG table), so the fold runs over all d with plain loads: addresses outside the
// column read other finite shared-memory words (the zero pad in front of U, other elements of U, or Bs) and multiply them
// by zero.  In the middle column of an even J rows ma < J/2 stand for rows J - ma, the centre counts once and rows above it
// are dropped: r is masked first.
template <int J1, int ROWB>
__device__ __forceinline__ double diag_fold(double (&rr)[2 * J1 + 1], double (&ri)[2 * J1 + 1], const unsigned char *Ulane, const int uoffJ,
                                            const int J, const int mb, const int d0) {
    constexpr int ND = 2 * J1 + 1;
    const bool mid = ((J & 1) == 0) && (mb == J / 2);
    if (mid) {
#pragma unroll
        for (int d = 0; d < ND; d++) {
            const int ma = d - d0;
            const double w = (ma < J / 2) ? 1.0 : ((ma == J / 2) ? 0.5 : 0.0);
            rr[d] *= w;
            ri[d] *= w;
        }
    }
    const unsigned char *ub = Ulane + (uoffJ + mb * (J + 1) - d0) * ROWB;
    double bp[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int d = 0; d < ND; d++) {
        const double2 u = *reinterpret_cast<const double2 *>(ub + d * ROWB);
        bp[(2 * d) & 3] = fma(u.x, rr[d], bp[(2 * d) & 3]);
        bp[(2 * d + 1) & 3] = fma(u.y, ri[d], bp[(2 * d + 1) & 3]);
    }
    const double b = (bp[0] + bp[1]) + (bp[2] + bp[3]);
    return b + b;
}

// ---------------------------------------------------------------------------------------------------------------------
// 32-point kernel: items mb1 in [mb1_begin, mb1_end) of output column mb of one triple: their contribution to B
// ---------------------------------------------------------------------------------------------------------------------
template <int J1>
__device__ __forceinline__ double diag_segment(const unsigned char *Ulane, const DiagTables &T, const int *uoff, const int J2, const int J,
                                               const int sh, const int cgoff, const int mb, const int mb1_begin, const int mb1_end) {
    constexpr int ND = 2 * J1 + 1;
    constexpr int S = diag_stride(J1);
    constexpr int ROWB = kDiagRowBytes;
    double rr[ND], ri[ND];
#pragma unroll
    for (int d = 0; d < ND; d++) { rr[d] = 0.0; ri[d] = 0.0; }
    const int off = J1 - J2;  // first row of the unrolled body
    const int uoff2 = uoff[J2];
    const double2 *cgrow = T.cg2 + (cgoff - off * S) / 2;  // rows are numbered k = ma2 + off
    const double *cgs = reinterpret_cast<const double *>(T.cg2);
#pragma unroll 1
    for (int mb1 = mb1_begin; mb1 < mb1_end; mb1++) {
        const int mb2 = mb + sh - mb1;
        const double cgb = diag_item_weight(cgs, cgoff, S, J1, J2, J, sh, mb, mb1);
        // x = U^{J1}[:, mb1]; columns beyond the middle come from the stored half by
        // u[ma][mb] = (-1)^(ma-mb) conj(u[J-ma][J-mb])
        double xr[J1 + 1], xi[J1 + 1];
        if (mb1 <= J1 / 2) {
            const unsigned char *xb = Ulane + (uhalf_off(J1) + mb1 * (J1 + 1)) * ROWB;
#pragma unroll
            for (int k = 0; k <= J1; k++) {
                const double2 v = *reinterpret_cast<const double2 *>(xb + k * ROWB);
                xr[k] = v.x;
                xi[k] = v.y;
            }
        } else {
            const unsigned char *xb = Ulane + (uhalf_off(J1) + (J1 - mb1) * (J1 + 1) + J1) * ROWB;
            const unsigned m0 = (mb1 & 1) ? 0x80000000u : 0u;  // sign of the real part on even rows
#pragma unroll
            for (int k = 0; k <= J1; k++) {
                const double2 v = *reinterpret_cast<const double2 *>(xb - k * ROWB);
                xr[k] = diag_flip(v.x, (k & 1) ? (m0 ^ 0x80000000u) : m0);
                xi[k] = diag_flip(v.y, (k & 1) ? m0 : (m0 ^ 0x80000000u));
            }
        }
        // y = U^{J2}[:, mb2], same symmetry, folded with cgb into scale factors by the parity of ma2
        const bool fy = mb2 > J2 / 2;
        const int cy = fy ? J2 - mb2 : mb2;
        int ystep = fy ? -ROWB : ROWB;
        const unsigned char *yp = Ulane + (uoff2 + cy * (J2 + 1) + (fy ? J2 : 0)) * ROWB;
        asm volatile("" : "+r"(ystep));  // keep the step in a register: one add per row, nothing recomputed
        const double p0 = (fy && (mb2 & 1)) ? -cgb : cgb;  // even ma2, real part
        const double p1 = fy ? -p0 : cgb;                  // odd ma2, real part
        const double q0 = fy ? -p0 : cgb;                  // imaginary parts: conjugation flips the sign again
        const double q1 = fy ? -p1 : cgb;
        const bool odd = off & 1;  // parities re-based from ma2 to the row number k
        const double se = odd ? p1 : p0, so = odd ? p0 : p1, te = odd ? q1 : q0, to = odd ? q0 : q1;
        diag_rows<J1>(rr, ri, xr, xi, yp, ystep, cgrow, off, se, so, te, to);
    }
    return diag_fold<J1, ROWB>(rr, ri, Ulane, uoff[J], J, mb, sh + off);
}

// this warp's items [begin, end) of one triple (items numbered column by column)
template <int J1>
__device__ __noinline__ double diag_items(const unsigned char *Ulane, const DiagTables T, const int *uoff, const int J2_, const int J_,
                                          const int cgoff_, const int begin_, const int end_) {
    // every argument but Ulane is warp-uniform; a broadcast from lane 0 tells the compiler so (uniform registers,
    // uniform branches, warp-uniform table addresses)
    const int J2 = __shfl_sync(0xffffffffu, J2_, 0), J = __shfl_sync(0xffffffffu, J_, 0);
    const int cgoff = __shfl_sync(0xffffffffu, cgoff_, 0);
    const int begin = __shfl_sync(0xffffffffu, begin_, 0), end = __shfl_sync(0xffffffffu, end_, 0);
    const int sh = (J1 + J2 - J) / 2;
    double b = 0.0;
    int base = 0;
#pragma unroll 1
    for (int mb = 0; mb <= J / 2 && base < end; mb++) {
        int lo, hi;
        diag_item_range(J1, J2, J, mb, lo, hi);
        const int nb = hi - lo + 1;
        const int s = max(begin, base), e = min(end, base + nb);
        if (s < e) b += diag_segment<J1>(Ulane, T, uoff, J2, J, sh, cgoff, mb, lo + s - base, lo + e - base);
        base += nb;
    }
    return b;
}

__device__ __forceinline__ double diag_dispatch(const int J1, const unsigned char *Ulane, const DiagTables &T, const int *uoff, const int J2,
                                                const int J, const int cgoff, const int begin, const int end) {
    switch (J1) {
        case 0: return diag_items<0>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 1: return diag_items<1>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 2: return diag_items<2>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 3: return diag_items<3>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 4: return diag_items<4>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 5: return diag_items<5>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 6: return diag_items<6>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 7: return diag_items<7>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 8: return diag_items<8>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 9: return diag_items<9>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        case 10: return diag_items<10>(Ulane, T, uoff, J2, J, cgoff, begin, end);
        default: return 0.0;
    }
}

__global__ void __launch_bounds__(kDiagWarps * 32, 1)
compute_zi_bi_diag_kernel(GridGeom g, SnapConst sc, DeviceTables tb, DiagTables T, ChunkBuffers cb, double *out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NW = kDiagWarps;
    const int nelem = sc.nelem, nt = sc.ntriples;
    double2 *U = reinterpret_cast<double2 *>(smem_raw + kDiagPadBytes);
    double *Bs = reinterpret_cast<double *>(U + (size_t)nelem * 32);
    double *red = Bs + 32 * nt;  // [2][kDiagGroup][NW][32]
    __shared__ uint64_t bar;
    __shared__ int s_slot;
    __shared__ int s_uoff[kMaxTwoJ + 2];
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    if (threadIdx.x <= kMaxTwoJ + 1) s_uoff[threadIdx.x] = uhalf_off(threadIdx.x);
    // the fold of diag_segment may read (and multiply by zero) words of the pad and of Bs: make them finite
    for (int i = threadIdx.x; i < kDiagPadBytes / 8; i += NW * 32) reinterpret_cast<double *>(smem_raw)[i] = 0.0;
    for (int i = threadIdx.x; i < 32 * nt + 2 * kDiagGroup * NW * 32; i += NW * 32) Bs[i] = 0.0;  // Bs and red
    uint32_t parity = 0;
    for (;;) {
        __syncthreads();  // previous tile written out: Bs, U and s_slot are free
        if (threadIdx.x == 0) s_slot = atomicAdd(&cb.counters[2], 1);
        __syncthreads();
        const int slot = s_slot;
        if (slot >= cb.counters[0]) break;
        const int wt = cb.active[slot];
        if (threadIdx.x == 0) tma_load_tile(U, cb.utot + (size_t)slot * nelem * 32, nelem, &bar);
        mbar_wait(&bar, parity);
        parity ^= 1u;
        const unsigned char *Ulane = reinterpret_cast<const unsigned char *>(U + lane);
        for (int pos = 0; pos < nt; pos++) {
            const int begin = __ldg(T.sched + (pos * NW + warp) * 2), end = __ldg(T.sched + (pos * NW + warp) * 2 + 1);
            double b = 0.0;
            if (begin < end) {
                const DiagTriple t = T.triple[pos];
                b = diag_dispatch(t.J1, Ulane, T, s_uoff, t.J2, t.J, t.cgoff, begin, end);
            }
            const int buf = (pos / kDiagGroup) & 1, k = pos % kDiagGroup;
            red[((buf * kDiagGroup + k) * NW + warp) * 32 + lane] = b;
            if (k == kDiagGroup - 1 || pos == nt - 1) {
                __syncthreads();
                // fixed-order sum of the partials of the triples of this group
                for (int kk = warp; kk <= k; kk += NW) {
                    const double *r = red + ((buf * kDiagGroup + kk) * NW) * 32 + lane;
                    double s = 0.0;
#pragma unroll
                    for (int w2 = 0; w2 < NW; w2++) s += r[w2 * 32];
                    Bs[lane * nt + T.triple[pos - k + kk].index] = s;
                }
            }
        }
        __syncthreads();
        write_tile(g, cb.tile_begin + wt, Bs, nt, out, NW, cb.compact_out, wt);
    }
}

inline size_t compute_zi_diag_smem_bytes(int nelem, int nt) {
    return (size_t)kDiagPadBytes + (size_t)nelem * 32 * sizeof(double2) + (size_t)32 * nt * sizeof(double) +
           (size_t)2 * kDiagGroup * kDiagWarps * 32 * sizeof(double) + 16;
}

// ---------------------------------------------------------------------------------------------------------------------
// 16-point kernel (twojmax 11..14).  Lane = (point p = lane & 15, item slot hs = lane >> 4).  A warp's items [begin, end) of
// a triple are split into two contiguous runs, one per half-warp; both halves walk their runs in lock step (the shorter one
// pads with a weight-zero item), load their own columns with per-lane addresses and sign masks, share the CG rectangle, and
// fold a column into B whenever their own run leaves it (a divergent branch around the fold only).
// ---------------------------------------------------------------------------------------------------------------------
template <int J1>
__device__ __noinline__ double diag_items_half(const unsigned char *Upt, const int hs, const DiagTables T, const int *uoff, const int J2_,
                                               const int J_, const int cgoff_, const int itemoff_, const int begin_, const int end_) {
    constexpr int ND = 2 * J1 + 1;
    constexpr int S = diag_stride(J1);
    constexpr int ROWB = kDiagHalfRowBytes;
    const int J2 = __shfl_sync(0xffffffffu, J2_, 0), J = __shfl_sync(0xffffffffu, J_, 0);
    const int cgoff = __shfl_sync(0xffffffffu, cgoff_, 0), itemoff = __shfl_sync(0xffffffffu, itemoff_, 0);
    const int begin = __shfl_sync(0xffffffffu, begin_, 0), end = __shfl_sync(0xffffffffu, end_, 0);
    const int sh = (J1 + J2 - J) / 2, off = J1 - J2;
    const int nh = (end - begin + 1) >> 1;  // items per half-warp
    const int my_begin = begin + hs * nh, my_end = min(end, my_begin + nh);
    const int uoff2 = uoff[J2], uoffJ = uoff[J];
    const double2 *cgrow = T.cg2 + (cgoff - off * S) / 2;
    const double *cgs = reinterpret_cast<const double *>(T.cg2);
    const bool odd = off & 1;
    double rr[ND], ri[ND];
#pragma unroll
    for (int d = 0; d < ND; d++) { rr[d] = 0.0; ri[d] = 0.0; }
    double b = 0.0;
#pragma unroll 1
    for (int i = 0; i < nh; i++) {
        const int it = my_begin + i;
        const bool live = it < my_end;
        const unsigned desc = live ? (unsigned)__ldg(T.items + itemoff + it) : 0u;
        const int mb = (int)((desc >> 8) & 0x7fu), mb1 = (int)(desc & 0xffu);
        const int mb2 = mb + sh - mb1;
        const double cgb = live ? diag_item_weight(cgs, cgoff, S, J1, J2, J, sh, mb, mb1) : 0.0;
        // x = U^{J1}[:, mb1], mirrored through u[ma][mb] = (-1)^(ma-mb) conj(u[J-ma][J-mb]) when mb1 > J1/2: per-lane start,
        // direction and sign masks instead of a branch
        double xr[J1 + 1], xi[J1 + 1];
        {
            const bool fx = mb1 > J1 / 2;
            const int cx = fx ? J1 - mb1 : mb1;
            const unsigned char *xp = Upt + (uhalf_off(J1) + cx * (J1 + 1) + (fx ? J1 : 0)) * ROWB;
            const int xstep = fx ? -ROWB : ROWB;
            const unsigned m0 = (fx && (mb1 & 1)) ? 0x80000000u : 0u;  // real part, even rows
            const unsigned m1 = fx ? (m0 ^ 0x80000000u) : 0u;           // real part, odd rows = imaginary part, even rows
#pragma unroll
            for (int k = 0; k <= J1; k++) {
                const double2 v = *reinterpret_cast<const double2 *>(xp + k * xstep);
                xr[k] = diag_flip(v.x, (k & 1) ? m1 : m0);
                xi[k] = diag_flip(v.y, (k & 1) ? m0 : m1);
            }
        }
        const bool fy = mb2 > J2 / 2;
        const int cy = fy ? J2 - mb2 : mb2;
        const int ystep = fy ? -ROWB : ROWB;
        const unsigned char *yp = Upt + (uoff2 + cy * (J2 + 1) + (fy ? J2 : 0)) * ROWB;
        const double p0 = (fy && (mb2 & 1)) ? -cgb : cgb;
        const double p1 = fy ? -p0 : cgb;
        const double q0 = fy ? -p0 : cgb;
        const double q1 = fy ? -p1 : cgb;
        const double se = odd ? p1 : p0, so = odd ? p0 : p1, te = odd ? q1 : q0, to = odd ? q0 : q1;
        diag_rows<J1>(rr, ri, xr, xi, yp, ystep, cgrow, off, se, so, te, to);
        // leave the column: the item is the last of its column, or the last of this half-warp's run
        if (live && ((desc >> 15) != 0u || it == my_end - 1)) {
            b += diag_fold<J1, ROWB>(rr, ri, Upt, uoffJ, J, mb, sh + off);
#pragma unroll
            for (int d = 0; d < ND; d++) { rr[d] = 0.0; ri[d] = 0.0; }
        }
    }
    return b + __shfl_xor_sync(0xffffffffu, b, 16);  // both item slots of a point
}

__device__ __forceinline__ double diag_dispatch_half(const int J1, const unsigned char *Upt, const int hs, const DiagTables &T,
                                                     const int *uoff, const DiagTriple &t, const int begin, const int end) {
    switch (J1) {
#define MALA_DIAG_HALF(N) \
    case N: return diag_items_half<N>(Upt, hs, T, uoff, t.J2, t.J, t.cgoff, t.itemoff, begin, end);
        MALA_DIAG_HALF(0) MALA_DIAG_HALF(1) MALA_DIAG_HALF(2) MALA_DIAG_HALF(3) MALA_DIAG_HALF(4) MALA_DIAG_HALF(5) MALA_DIAG_HALF(6)
        MALA_DIAG_HALF(7) MALA_DIAG_HALF(8) MALA_DIAG_HALF(9) MALA_DIAG_HALF(10) MALA_DIAG_HALF(11) MALA_DIAG_HALF(12)
        MALA_DIAG_HALF(13) MALA_DIAG_HALF(14)
#undef MALA_DIAG_HALF
        default: return 0.0;
    }
}

// B of 16 points, staged as Bs[point][nt], to out[point][nt]: one warp per point row of nt doubles
__device__ __forceinline__ void write_half_tile(const GridGeom &g, int tile, int half, const double *Bs, int nt, double *out, int nwarps,
                                                int compact, int wt) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (compact) {
        double *dst = out + ((size_t)wt * 32 + half * 16) * nt;
        for (int i = threadIdx.x; i < 16 * nt; i += nwarps * 32) __stcs(dst + i, Bs[i]);
        return;
    }
    for (int p = warp; p < 16; p += nwarps) {
        int ix, iy, iz;
        bool valid;
        lane_point(g, tile, half * 16 + p, ix, iy, iz, valid);
        if (!valid) continue;
        double *dst = out + ((size_t)((size_t)(iz - g.z0) * g.ny + iy) * g.nx + ix) * nt;
        for (int i = lane; i < nt; i += 32) __stcs(dst + i, Bs[p * nt + i]);
    }
}

__global__ void __launch_bounds__(kDiagHalfWarps * 32, 1)
compute_zi_bi_diag_half_kernel(GridGeom g, SnapConst sc, DeviceTables tb, DiagTables T, ChunkBuffers cb, double *out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NW = kDiagHalfWarps;
    const int nelem = sc.nelem, nt = sc.ntriples;
    double2 *U = reinterpret_cast<double2 *>(smem_raw + kDiagPadBytes);  // [nelem][16]
    double *Bs = reinterpret_cast<double *>(U + (size_t)nelem * 16);      // [16][nt]
    double *red = Bs + 16 * nt;                                           // [2][kDiagGroup][NW][16]
    __shared__ uint64_t bar;
    __shared__ int s_item;
    __shared__ int s_uoff[kMaxTwoJ + 2];
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    const int p = lane & 15, hs = lane >> 4;
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    if (threadIdx.x <= kMaxTwoJ + 1) s_uoff[threadIdx.x] = uhalf_off(threadIdx.x);
    for (int i = threadIdx.x; i < kDiagPadBytes / 8; i += NW * 32) reinterpret_cast<double *>(smem_raw)[i] = 0.0;
    for (int i = threadIdx.x; i < 16 * nt + 2 * kDiagGroup * NW * 16; i += NW * 32) Bs[i] = 0.0;  // Bs and red
    uint32_t parity = 0;
    const size_t half_elems = (size_t)nelem * 16;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(&cb.counters[2], 1);
        __syncthreads();
        const int item = s_item;
        const int slot = item >> 1, half = item & 1;
        if (slot >= cb.counters[0]) break;
        const int wt = cb.active[slot];
        // compute_ui wrote this half tile as one contiguous [nelem][16] block (ChunkBuffers::utot_half_layout)
        if (threadIdx.x == 0) tma_load_bytes(U, cb.utot + (size_t)item * half_elems, (uint32_t)(half_elems * sizeof(double2)), &bar);
        mbar_wait(&bar, parity);
        parity ^= 1u;
        const unsigned char *Upt = reinterpret_cast<const unsigned char *>(U + p);
        for (int pos = 0; pos < nt; pos++) {
            const int begin = __ldg(T.sched + (pos * NW + warp) * 2), end = __ldg(T.sched + (pos * NW + warp) * 2 + 1);
            double b = 0.0;
            if (begin < end) {
                const DiagTriple t = T.triple[pos];
                b = diag_dispatch_half(t.J1, Upt, hs, T, s_uoff, t, begin, end);
            }
            const int buf = (pos / kDiagGroup) & 1, k = pos % kDiagGroup;
            if (hs == 0) red[((buf * kDiagGroup + k) * NW + warp) * 16 + p] = b;
            if (k == kDiagGroup - 1 || pos == nt - 1) {
                __syncthreads();
                // fixed-order sum of the partials: half-warp hs of warp w takes triples 2 w + hs, 2 w + hs + 2 NW, ...
                for (int kk = 2 * warp + hs; kk <= k; kk += 2 * NW) {
                    const double *r = red + ((buf * kDiagGroup + kk) * NW) * 16 + p;
                    double s = 0.0;
#pragma unroll
                    for (int w2 = 0; w2 < NW; w2++) s += r[w2 * 16];
                    Bs[p * nt + T.triple[pos - k + kk].index] = s;
                }
            }
        }
        __syncthreads();
        write_half_tile(g, cb.tile_begin + wt, half, Bs, nt, out, NW, cb.compact_out, wt);
    }
}

inline size_t compute_zi_diag_half_smem_bytes(int nelem, int nt) {
    return (size_t)kDiagPadBytes + (size_t)nelem * 16 * sizeof(double2) + (size_t)16 * nt * sizeof(double) +
           (size_t)2 * kDiagGroup * kDiagHalfWarps * 16 * sizeof(double) + 16;
}

}  // namespace mala
