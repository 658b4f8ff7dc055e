// snap_yi_block.cuh -- compute_yi of row f3 on the machinery of snap_zi_block.cuh:
//     Y^C[ma][mb] = yweight * sum_terms coef * beta[index] * Z^C_{AB}[ma][mb]          (snap_force.cuh; Eq. (45))
// Every term (A, B -> C) is the same contraction as compute_zi's -- a column of Z is the CG-weighted anti-diagonal sum of
// T = sum_items w x (x) y -- so it runs through the same register-tiled item loops and record streams.  What differs is
// where a finished block goes: its anti-diagonal sums z are not dotted with U (compute_bi) but added, times the lane's
// coef * beta, to the rows of column (C, mb) of Y.  Y is as large as U_tot (139 KB for 32 points) and does not fit beside it
// in shared memory, so a tile is processed in passes over groups of target levels (10 | 9 | 8 | 7,6 | 5..0 at twojmax 10): the
// accumulator holds the levels of one group (<= 34 KB), is flushed to global memory (with the weights of snap_force.cuh) and
// cleared between passes.  Units of different warps may hit the same Y element at the same time: the additions are
// shared-memory atomics (a compare-and-swap loop on sm_100a), so Y -- like the forces that follow -- is reproducible to
// rounding, not bit for bit.  The middle column of an even level is computed up to its centre row only; the flush fills the
// rows above it by Y[C - ma][C/2] = (-1)^(ma - C/2) conj(Y[ma][C/2]).
#pragma once
#include "snap_zi_block.cuh"

namespace mala {

constexpr int kYBlkMaxPasses = 8;

// Unit records of the Y streams (16-byte words):
//   header 0   int4    { nitems, byte offset of row ma0 of column (C, mb) in the pass's accumulator (may be negative),
//                        beta index, words to skip behind the unit }
//   header 1   int2 + double { first and last anti-diagonal whose row lies inside the column, coef }
//   items, coefficients as in snap_zi_block.cuh (coefficients = plain CG, zero outside 0 <= ma <= C)
struct YBlkTables {
    const int4 *stream;
    const int *wrange;      // [warps][passes][kBlkShapes] units per shape, then per warp {first word, word count}: see yblk_wrange_*
    const int *pass_elem;   // [npasses][2] first and one-past-last element (uhalf order) of the levels of every pass
    const double *yweight;  // [nelem]
    const int *mirror;      // [nelem] -1, or (element to mirror << 1 | odd sign) for the rows above the centre of a middle column
    int npasses, yacc_elems;
};
__host__ __device__ inline int yblk_wrange_count(int warp, int pass, int shape, int npasses) {
    return (warp * npasses + pass) * kBlkShapes + shape;
}
__host__ __device__ inline int yblk_wrange_first(int warp, int npasses) { return kBlkWarps * npasses * kBlkShapes + 2 * warp; }

__device__ __forceinline__ void yblk_atomic_add(double *addr, double v) { atomicAdd(addr, v); }

template <int BX, int BY>
__device__ __forceinline__ void yblk_unit(const unsigned char *Ulane, BlkReader &rd, unsigned char *Yl, const double *Btl) {
    constexpr int RB = 32 * (int)sizeof(double2);
    constexpr int NCW = (BX * BY + 1) / 2;
    double tr[BX][BY], ti[BX][BY];
    rd.ensure(rd.wpos + 2);
    uint32_t base = rd.ring + (uint32_t)((rd.wpos & (kBlkRingWords - 1)) * 16);
    const int4 hd = blk_lds4(base);
    const int4 h1 = blk_lds4(base + 16);
    const int nitems = hd.x, yoff = hd.y;
    const int dlo = h1.x, dhi = h1.y;
    const double wl = __hiloint2double(h1.w, h1.z) * Btl[hd.z * 32];   // coef * beta of this lane's grid point
    const int wend = rd.wpos + 2 + 3 * nitems + NCW;
    rd.ensure(wend);
    rd.wpos = wend + hd.w;
    base += 32;
    blk_item<BX, BY, true>(Ulane, base, tr, ti);
    base += 48;
#pragma unroll 1
    for (int i = 1; i < nitems; i++) {
        blk_item<BX, BY, false>(Ulane, base, tr, ti);
        base += 48;
    }
    unsigned char *yb = Yl + yoff;
    double2 cpair = make_double2(0.0, 0.0);
#pragma unroll
    for (int d = 0; d < BX + BY - 1; d++) {
        double zr = 0.0, zi = 0.0;
#pragma unroll
        for (int a = 0; a < BX; a++) {
            const int b = d - a;
            if (b >= 0 && b < BY) {
                const int k = blk_coef_index(BX, BY, d, a);   // a compile-time constant once the loops are unrolled
                if ((k & 1) == 0) cpair = blk_lds2(base + 8 * k);   // two coefficients per 16-byte load, in consumption order
                const double c = (k & 1) ? cpair.y : cpair.x;
                zr = fma(c, tr[a][b], zr);
                zi = fma(c, ti[a][b], zi);
            }
        }
        if (d >= dlo && d <= dhi) {   // rows outside the column carry exact zeros: skipped (warp-uniform)
            double *y = reinterpret_cast<double *>(yb + d * RB);   // real parts of the 32 lanes, then the imaginary parts: conflict-free
            yblk_atomic_add(y, wl * zr);
            yblk_atomic_add(y + 32, wl * zi);
        }
    }
    rd.fill();
}

template <int BX, int BY>
__device__ __forceinline__ void yblk_run_all(const unsigned char *Ulane, const YBlkTables &T, const int warp, const int pass, BlkReader &rd,
                                             unsigned char *Yl, const double *Btl) {
    if constexpr (BX >= kBlkBXMin && BY >= kBlkBYMin) {
        const int n = __ldg(T.wrange + yblk_wrange_count(warp, pass, (BX - 1) * kBlkBY + (BY - 1), T.npasses));
#pragma unroll 1
        for (int k = 0; k < n; k++) yblk_unit<BX, BY>(Ulane, rd, Yl, Btl);
    }
    if constexpr (BY > 1) yblk_run_all<BX, BY - 1>(Ulane, T, warp, pass, rd, Yl, Btl);
    else if constexpr (BX > 1) yblk_run_all<BX - 1, kBlkBY>(Ulane, T, warp, pass, rd, Yl, Btl);
}

__global__ void __launch_bounds__(kBlkWarps * 32, 1)
compute_yi_block_kernel(GridGeom g, SnapConst sc, YBlkTables T, ChunkBuffers cb, const double *beta, double2 *ytot) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NW = kBlkWarps;
    const int nelem = sc.nelem, nt = sc.ntriples;
    double2 *U = reinterpret_cast<double2 *>(smem_raw + kBlkPadBytes);
    double *Bt = reinterpret_cast<double *>(U + (size_t)nelem * 32);                 // [nt][32] beta of the tile, lane fastest
    double *Yacc = Bt + (size_t)32 * nt;                                             // [yacc_elems][re | im][32]
    int4 *rings = reinterpret_cast<int4 *>(Yacc + (size_t)T.yacc_elems * 64);        // [NW][kBlkRingWords]
    __shared__ uint64_t bar;
    __shared__ int s_slot;
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    for (int i = threadIdx.x; i < kBlkPadBytes / 8; i += NW * 32) reinterpret_cast<double *>(smem_raw)[i] = 0.0;
    uint32_t parity = 0;
    const int nactive = cb.counters[0];
    if (threadIdx.x == 0) s_slot = atomicAdd(&cb.counters[2], 1);
    for (;;) {
        __syncthreads();  // previous tile flushed: U, Bt and Yacc are free; s_slot is visible
        const int slot = s_slot;
        if (slot >= nactive) break;
        const int wt = cb.active[slot];
        __syncthreads();  // everybody has read s_slot
        if (threadIdx.x == 0) {
            tma_load_tile(U, cb.utot + (size_t)slot * nelem * 32, nelem, &bar);
            const int next = atomicAdd(&cb.counters[2], 1);
            s_slot = next;
            if (next < nactive) prefetch_l2_tile(cb.utot + (size_t)next * nelem * 32, nelem);
        }
        // beta rows of the tile's points (zero for lanes outside a ragged tile)
        for (int idx = threadIdx.x; idx < 32 * nt; idx += NW * 32) {
            const int l = idx / nt, t = idx - l * nt;
            int ix, iy, iz;
            bool valid;
            lane_point(g, cb.tile_begin + wt, l, ix, iy, iz, valid);
            Bt[t * 32 + l] = valid ? beta[((size_t)((size_t)(iz - g.z0) * g.ny + iy) * g.nx + ix) * nt + t] : 0.0;
        }
        for (int i = threadIdx.x; i < T.yacc_elems * 64; i += NW * 32) Yacc[i] = 0.0;
        BlkReader rd;
        rd.src = T.stream + __ldg(T.wrange + yblk_wrange_first(warp, T.npasses));
        rd.wtotal = __ldg(T.wrange + yblk_wrange_first(warp, T.npasses) + 1);
        rd.ring = smem_u32(rings + warp * kBlkRingWords);
        rd.lane = lane; rd.wpos = 0; rd.wreq = 0; rd.wready = 0;
        rd.fill();
        mbar_wait(&bar, parity);
        parity ^= 1u;
        __syncthreads();  // Bt and Yacc ready
        const unsigned char *Ulane = reinterpret_cast<const unsigned char *>(U + lane);
        unsigned char *Yl = reinterpret_cast<unsigned char *>(Yacc + lane);
        double2 *Yt = ytot + (size_t)slot * nelem * 32;
        for (int pass = 0; pass < T.npasses; pass++) {
            yblk_run_all<kBlkBX, kBlkBY>(Ulane, T, warp, pass, rd, Yl, Bt + lane);
            __syncthreads();
            // flush the levels of this pass with the weights of the polynomial form and the half-column doubling; clear
            const int e0 = __ldg(T.pass_elem + 2 * pass), e1 = __ldg(T.pass_elem + 2 * pass + 1);
            for (int i = threadIdx.x; i < (e1 - e0) * 32; i += NW * 32) {
                const int e = e0 + (i >> 5);
                const double yw = __ldg(T.yweight + e);
                const int mm = __ldg(T.mirror + e);
                if (mm < 0) {
                    const int at = (i >> 5) * 64 + (i & 31);
                    Yt[(size_t)e * 32 + (i & 31)] = make_double2(yw * Yacc[at], yw * Yacc[at + 32]);
                } else {   // a row above the centre of a middle column: the conjugate of its mirror row, with the sign of the symmetry
                    const int at = ((mm >> 1) - e0) * 64 + (i & 31);
                    const double sg = (mm & 1) ? -yw : yw;
                    Yt[(size_t)e * 32 + (i & 31)] = make_double2(sg * Yacc[at], -sg * Yacc[at + 32]);
                }
            }
            __syncthreads();   // the mirror rows have read their sources
            for (int i = threadIdx.x; i < (e1 - e0) * 64; i += NW * 32) Yacc[i] = 0.0;
            __syncthreads();
        }
    }
}

inline size_t compute_yi_block_smem_bytes(int nelem, int nt, int yacc_elems) {
    return (size_t)kBlkPadBytes + (size_t)nelem * 32 * sizeof(double2) + (size_t)32 * nt * sizeof(double) +
           (size_t)yacc_elems * 32 * sizeof(double2) + (size_t)kBlkWarps * kBlkRingWords * 16 + 16;
}

}  // namespace mala
