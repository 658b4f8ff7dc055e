// snap_yi_fix.cuh -- compute_yi of row f3 as in snap_yi_block.cuh, with Y accumulated in FIXED POINT by native atomics.
//
// On sm_100a every 64-bit shared-memory atomic -- fp64 or integer -- is an ATOMS.CAST.SPIN.64 loop: a load, the add, a
// compare-and-swap and a branch, two dependent shared-memory round trips per element and twenty elements per unit, a quarter
// of compute_yi_block_kernel.  Only the 32-bit ATOMS.ADD is native, and it needs no answer.  Here a component of Y is a
// 60-bit fixed-point number kept as three 20-bit digits in three 32-bit words:
//   * every grid point (lane) gets a power-of-two scale per tile, 2^59 over a bound of its |Y| (max |U component|^2 x sum |beta|
//     x a constant of the tables), so that no sum leaves 60 bits;
//   * an addend v is rounded to q = rint(v * scale) and split into q = d2 2^40 + d1 2^20 + d0 with 0 <= d0, d1 < 2^20; each digit
//     goes to its own word with one ATOMS.ADD.  A word takes up to 2^11 addends before it could wrap (a Y element receives a
//     few hundred);
//   * the flush puts the words together in 64-bit integer arithmetic and scales back.
// Rounding: 2^-59 of the bound per addend; the bound is loose by a few thousand, which leaves about 1e-14 of the largest |Y| of
// the grid point -- the level of the fp64 sums it replaces.  Integer addition is associative: Y no longer depends on the order
// in which the warps add.
// The accumulator is 768 bytes per element instead of 512; the shared memory for it comes from the beta tile, which this
// kernel reads from global memory (L2) instead: one value per lane and unit, requested when the unit starts.
#pragma once
#include "snap_yi_block.cuh"

namespace mala {

constexpr int kYFixRowBytes = 768;   // one Y element: {re d0, re d1, re d2, im d0, im d1, im d2} x 32 lanes x 4 bytes
constexpr int kYFixDigit = 20;

__device__ __forceinline__ void yfix_add(int *y, const double v) {
    const long long q = __double2ll_rn(v);
    constexpr int M = (1 << kYFixDigit) - 1;
    atomicAdd(y, (int)(q & M));
    atomicAdd(y + 32, (int)((q >> kYFixDigit) & M));
    atomicAdd(y + 64, (int)(q >> (2 * kYFixDigit)));
}
__device__ __forceinline__ double yfix_value(const int *y) {
    const long long q = ((long long)y[64] << (2 * kYFixDigit)) + ((long long)(unsigned)y[32] << kYFixDigit) + (long long)(unsigned)y[0];
    return (double)q;
}

template <int BX, int BY>
__device__ __forceinline__ void yfix_unit(const unsigned char *Ulane, BlkReader &rd, unsigned char *Yl, const double *betal, const double scale) {
    constexpr int NCW = (BX * BY + 1) / 2;
    double tr[BX][BY], ti[BX][BY];
    rd.ensure(rd.wpos + 2);
    uint32_t base = rd.ring + (uint32_t)((rd.wpos & (kBlkRingWords - 1)) * 16);
    const int4 hd = blk_lds4(base);
    const int4 h1 = blk_lds4(base + 16);
    const int nitems = hd.x;
    const int yoff = hd.y + (hd.y >> 1);   // the stream counts rows of 512 bytes
    const int dlo = h1.x, dhi = h1.y;
    const double bl = betal ? __ldg(betal + hd.z) : 0.0;   // beta of this lane's grid point: in flight during the items
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
    const double wl = __hiloint2double(h1.w, h1.z) * bl * scale;   // coef * beta, in units of the lane's fixed point
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
            int *y = reinterpret_cast<int *>(yb + d * kYFixRowBytes);
            yfix_add(y, wl * zr);
            yfix_add(y + 96, wl * zi);
        }
    }
    rd.fill();
}

template <int BX, int BY>
__device__ __forceinline__ void yfix_run_all(const unsigned char *Ulane, const YBlkTables &T, const int warp, const int pass, BlkReader &rd,
                                             unsigned char *Yl, const double *betal, const double scale) {
    if constexpr (BX >= kBlkBXMin && BY >= kBlkBYMin) {
        const int n = __ldg(T.wrange + yblk_wrange_count(warp, pass, (BX - 1) * kBlkBY + (BY - 1), T.npasses));
#pragma unroll 1
        for (int k = 0; k < n; k++) yfix_unit<BX, BY>(Ulane, rd, Yl, betal, scale);
    }
    if constexpr (BY > 1) yfix_run_all<BX, BY - 1>(Ulane, T, warp, pass, rd, Yl, betal, scale);
    else if constexpr (BX > 1) yfix_run_all<BX - 1, kBlkBY>(Ulane, T, warp, pass, rd, Yl, betal, scale);
}

__global__ void __launch_bounds__(kBlkWarps * 32, 1)
compute_yi_fix_kernel(GridGeom g, SnapConst sc, YBlkTables T, ChunkBuffers cb, const double *beta, double2 *ytot, const double bound_factor) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NW = kBlkWarps;
    const int nelem = sc.nelem, nt = sc.ntriples;
    double2 *U = reinterpret_cast<double2 *>(smem_raw + kBlkPadBytes);
    int *Yacc = reinterpret_cast<int *>(U + (size_t)nelem * 32);                                  // [yacc_elems][6][32]
    int4 *rings = reinterpret_cast<int4 *>(Yacc + (size_t)T.yacc_elems * (kYFixRowBytes / 4));   // [NW][kBlkRingWords]
    __shared__ uint64_t bar;
    __shared__ int s_slot;
    __shared__ double s_umax[NW][32], s_bsum[NW][32], s_scale[32], s_unscale[32];
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    for (int i = threadIdx.x; i < kBlkPadBytes / 8; i += NW * 32) reinterpret_cast<double *>(smem_raw)[i] = 0.0;
    uint32_t parity = 0;
    const int nactive = cb.counters[0];
    if (threadIdx.x == 0) s_slot = atomicAdd(&cb.counters[2], 1);
    for (;;) {
        __syncthreads();  // previous tile flushed: U and Yacc are free; s_slot is visible
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
        // the beta row of this lane's grid point (none for lanes outside a ragged tile)
        const double *betal = nullptr;
        {
            int ix, iy, iz;
            bool valid;
            lane_point(g, cb.tile_begin + wt, lane, ix, iy, iz, valid);
            if (valid) betal = beta + ((size_t)((size_t)(iz - g.z0) * g.ny + iy) * g.nx + ix) * nt;
        }
        for (int i = threadIdx.x; i < T.yacc_elems * (kYFixRowBytes / 4); i += NW * 32) Yacc[i] = 0;
        BlkReader rd;
        rd.src = T.stream + __ldg(T.wrange + yblk_wrange_first(warp, T.npasses));
        rd.wtotal = __ldg(T.wrange + yblk_wrange_first(warp, T.npasses) + 1);
        rd.ring = smem_u32(rings + warp * kBlkRingWords);
        rd.lane = lane; rd.wpos = 0; rd.wreq = 0; rd.wready = 0;
        rd.fill();
        // fixed-point scale of every grid point: 2^59 over a bound of its |Y|; an input that is not finite makes it NaN, and Y with it
        double bs = 0.0, chk = 0.0;
        if (betal)
            for (int t = warp; t < nt; t += NW) {
                const double b = __ldg(betal + t);
                bs += fabs(b);
                chk = fma(b, 0.0, chk);
            }
        mbar_wait(&bar, parity);
        parity ^= 1u;
        double um = 0.0;
        for (int e = warp; e < nelem; e += NW) {
            const double2 u = U[(size_t)e * 32 + lane];
            um = fmax(um, fmax(fabs(u.x), fabs(u.y)));
            chk = fma(u.x, 0.0, fma(u.y, 0.0, chk));
        }
        s_umax[warp][lane] = (chk == 0.0) ? um : chk;
        s_bsum[warp][lane] = bs;
        __syncthreads();  // Yacc zeroed too
        if (warp == 0) {
            um = 0.0; bs = 0.0; chk = 0.0;
            for (int w2 = 0; w2 < NW; w2++) {
                const double a = s_umax[w2][lane];
                if (a != a) chk = a;
                um = fmax(um, a);
                bs += s_bsum[w2][lane];
            }
            const double bound = bound_factor * um * um * bs;
            double scale = 1.0;
            if (chk != chk || !(bound < 1e300)) scale = chk * 0.0 + (bound - bound);   // NaN
            else if (bound > 0.0) {
                int ex;
                frexp(bound, &ex);   // bound < 2^ex
                scale = ldexp(1.0, 59 - ex);
            }
            s_scale[lane] = scale;
            s_unscale[lane] = 1.0 / scale;
        }
        __syncthreads();
        const double scale = s_scale[lane];
        const unsigned char *Ulane = reinterpret_cast<const unsigned char *>(U + lane);
        unsigned char *Yl = reinterpret_cast<unsigned char *>(Yacc + lane);
        double2 *Yt = ytot + (size_t)slot * nelem * 32;
        for (int pass = 0; pass < T.npasses; pass++) {
            yfix_run_all<kBlkBX, kBlkBY>(Ulane, T, warp, pass, rd, Yl, betal, scale);
            __syncthreads();
            // flush the levels of this pass with the weights of the polynomial form and the half-column doubling; clear
            const int e0 = __ldg(T.pass_elem + 2 * pass), e1 = __ldg(T.pass_elem + 2 * pass + 1);
            for (int i = threadIdx.x; i < (e1 - e0) * 32; i += NW * 32) {
                const int e = e0 + (i >> 5);
                const double yw = __ldg(T.yweight + e) * s_unscale[i & 31];   // back from fixed point
                const int mm = __ldg(T.mirror + e);
                if (mm < 0) {
                    const int *y = Yacc + (i >> 5) * (kYFixRowBytes / 4) + (i & 31);
                    Yt[(size_t)e * 32 + (i & 31)] = make_double2(yw * yfix_value(y), yw * yfix_value(y + 96));
                } else {   // a row above the centre of a middle column: the conjugate of its mirror row, with the sign of the symmetry
                    const int *y = Yacc + ((mm >> 1) - e0) * (kYFixRowBytes / 4) + (i & 31);
                    const double sg = (mm & 1) ? -yw : yw;
                    Yt[(size_t)e * 32 + (i & 31)] = make_double2(sg * yfix_value(y), -sg * yfix_value(y + 96));
                }
            }
            __syncthreads();   // the mirror rows have read their sources
            for (int i = threadIdx.x; i < (e1 - e0) * (kYFixRowBytes / 4); i += NW * 32) Yacc[i] = 0;
            __syncthreads();
        }
    }
}

inline size_t compute_yi_fix_smem_bytes(int nelem, int yacc_elems) {
    return (size_t)kBlkPadBytes + (size_t)nelem * 32 * sizeof(double2) + (size_t)yacc_elems * kYFixRowBytes + (size_t)kBlkWarps * kBlkRingWords * 16 + 16;
}

}  // namespace mala
