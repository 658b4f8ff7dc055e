// snap_zi_block.cuh -- compute_zi / compute_bi as register-tiled outer products (rows a5 + a6 + a7), any twojmax (half tiles above 10).
//
// For a triple (J1,J2,J) and an output column mb, the Z column is
//     z[ma] = sum_{ma1 + ma2 - sh = ma} CG(ma1, ma2) * T[ma1][ma2],     T[ma1][ma2] = sum_items w_i x_i[ma1] y_i[ma2],
// where the items i are the (mb1, mb2 = mb + sh - mb1) column pairs, x_i = U^{J1}[:, mb1], y_i = U^{J2}[:, mb2] and w_i the
// Clebsch-Gordan factor of the column pair times the size of the symmetry class the item stands for (snap_zi_coop.cuh).
// The per-triple and the anti-diagonal kernel apply CG(ma1, ma2) inside the item loop (6 FP64 instructions per product
// term) and unroll the whole (ma1, ma2) rectangle, which makes their code long and walked once per item.  Here the item
// loop is the INNER loop: a BX x BY block of T lives in registers, an item adds the outer product of BX elements of x and
// BY elements of y (4 FP64 instructions per term), and the CG coefficients -- with the weights of the compute_bi fold
// already multiplied in -- are applied once per block and column afterwards.  The body depends on the block shape only:
// every triple, column and block runs through the same 30 small loops, which stay in the instruction caches.
//
// Work unit = (triple, column, block); the host cuts every rectangle into blocks of at most 6 x 5, trims each block to the
// bounding box of its non-zero coefficients (the band 0 <= ma <= J, or ma <= J/2 in the middle column of an even J), packs
// the coefficients per unit and deals the units of whole triples to the warps (the heaviest triples are split).  A unit adds
// its share of B to a partial-sum slot owned by one warp; the slots of a triple are summed in a fixed order at the end of
// the tile: bit-reproducible, no atomics, one CTA-wide barrier per tile.
#pragma once
#include "snap_zi.cuh"

namespace mala {

#ifndef MALA_BLK_WARPS
#define MALA_BLK_WARPS 12
#endif
#ifndef MALA_BLK_BX
#define MALA_BLK_BX 6
#endif
#ifndef MALA_BLK_BY
#define MALA_BLK_BY 5
#endif
constexpr int kBlkWarps = MALA_BLK_WARPS;   // 12 warps = 168 registers per thread: a 6 x 5 complex block takes 120 of them
constexpr int kBlkBX = MALA_BLK_BX, kBlkBY = MALA_BLK_BY;
#ifndef MALA_BLK_BXMIN
#define MALA_BLK_BXMIN 3
#endif
#ifndef MALA_BLK_BYMIN
#define MALA_BLK_BYMIN 3
#endif
// smaller blocks are padded to the minimum shape with zero coefficients (2-3 % more FP64 work): 12 loop bodies instead of 30,
// which is what the instruction caches reward (twojmax 6: 3.0 ms with all 30 shapes and the first item peeled, 1.8 ms with 12 and none)
constexpr int kBlkBXMin = MALA_BLK_BXMIN, kBlkBYMin = MALA_BLK_BYMIN;
constexpr int kBlkShapes = kBlkBX * kBlkBY;
constexpr int kBlkPadBytes = 3072;   // zeros in front of U: the fold may read up to 5 rows before a column (times an exact zero)
constexpr int kBlkMaxSlots = 120;    // partial-sum slots (one per (warp, triple) pair that has work)

// Every warp reads ONE contiguous stream of 16-byte words, in the order it consumes them (units sorted by shape):
//   unit header   int4   { nitems, byte offset of U^J[ma0][mb] (row of the block's first anti-diagonal; may be negative), slot,
//                          words to skip behind the unit (the host keeps a unit from straddling the end of the ring) }
//   nitems x      int4   { x offset, x step, y offset, y step }                (bytes; a step is +-512)
//                 int4   { sign mask of even x rows, of odd x rows, x reversed, 0 }
//                 double2{ scale of even y rows, scale of odd y rows }
//   coefficients  double2 x ceil(BX BY / 2)      CG x fold weight, [a][b]
// Offsets are bytes from the first element of the tile's U_tot to the element the block reads first, for lane 0; a column
// beyond the middle is read backwards from its mirror image (u[ma][mb] = (-1)^(ma-mb) conj(u[J-ma][J-mb])): x gets its signs
// by flipping sign bits (real part: mask of the row parity; imaginary part: the mask of the other parity), y has them folded
// into its two scale factors (real part of an even row and imaginary part of an odd row take the first, the others the second).
struct BlkTables {
    const int4 *stream;              // all warps, one after the other
    const int *wrange;               // [warps][kBlkShapes + 2]: number of units per shape, then the warp's first word and word count
    const int *tslot;                // [nt + 1] slots of triple t are tslot[t] .. tslot[t+1]-1
    int nslots;
};

__device__ __forceinline__ double blk_flip(double v, unsigned mask) {
    return __hiloint2double(__double2hiint(v) ^ (int)mask, __double2loint(v));
}
// The warp's record stream comes through a private ring in shared memory, filled 512 bytes at a time by one cp.async per lane:
// requests run up to four chunks ahead of the word being consumed, so the records are on chip long before they are needed
// (read straight from L2 they cost a quarter of the kernel's time in long-scoreboard stalls).
constexpr int kBlkRingWords = 128;   // 16-byte words per warp (2 KB)
__device__ __forceinline__ int4 blk_lds4(const uint32_t addr) {
    int4 v;
    asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ double blk_lds1(const uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ double2 blk_lds2(const uint32_t addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
struct BlkReader {
    const int4 *src;     // the warp's stream
    uint32_t ring;       // shared-memory address of the warp's ring
    int lane;
    int wpos, wreq, wready, wtotal;   // words consumed / requested / known to have arrived (multiples of 32) / in the stream
    __device__ __forceinline__ void fill() {
        // chunk [wreq, wreq + 32) takes the place of [wreq - 128, wreq - 96): free once wpos has passed it
        while (wreq - (kBlkRingWords - 32) <= wpos && wreq < wtotal) {
            const uint32_t dst = ring + (uint32_t)(((wreq + lane) & (kBlkRingWords - 1)) * 16);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src + wreq + lane) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
            wreq += 32;
        }
    }
    __device__ __forceinline__ void ensure(const int wend) {   // words below wend must be readable
        if (wend > wready) {
            asm volatile("cp.async.wait_all;" ::: "memory");
            __syncwarp();
            wready = wreq;
        }
    }
    __device__ __forceinline__ int4 word(const int w) const {
        int4 v;
        asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(ring + (uint32_t)((w & (kBlkRingWords - 1)) * 16)));
        return v;
    }
    __device__ __forceinline__ double2 dword(const int w) const {
        double2 v;
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(ring + (uint32_t)((w & (kBlkRingWords - 1)) * 16)));
        return v;
    }
};

// position of coefficient (a, b = d - a) in the order the projection consumes them: anti-diagonal by anti-diagonal, a ascending
__host__ __device__ constexpr int blk_coef_index(int BX, int BY, int d, int a) {
    int k = 0;
    for (int dd = 0; dd <= d; dd++)
        for (int aa = 0; aa < BX; aa++) {
            const int bb = dd - aa;
            if (bb < 0 || bb >= BY) continue;
            if (dd == d && aa == a) return k;
            k++;
        }
    return k;
}

// one item of a unit: T (+)= x (x) y.  FIRST: the block starts from this item's products (no zeroing pass)
template <int BX, int BY, bool FIRST>
__device__ __forceinline__ void blk_item(const unsigned char *Ulane, const uint32_t base, double (&tr)[BX][BY], double (&ti)[BX][BY]) {
    const int4 r = blk_lds4(base);
    const int4 m = blk_lds4(base + 16);
    const double2 sc = blk_lds2(base + 32);
    const unsigned char *xp = Ulane + r.x, *yp = Ulane + r.z;
    const int xstep = r.y, ystep = r.w;
    double yr[BY], yi[BY];
#pragma unroll
    for (int b = 0; b < BY; b++) {
        const double2 v = *reinterpret_cast<const double2 *>(yp + b * ystep);
        yr[b] = v.x * ((b & 1) ? sc.y : sc.x);
        yi[b] = v.y * ((b & 1) ? sc.x : sc.y);
    }
    const unsigned me = (unsigned)m.x, mo = (unsigned)m.y;   // mirrored x column: (-1)^(ma1 - mb1) conj (zero masks otherwise)
#pragma unroll
    for (int a = 0; a < BX; a++) {
        const double2 v = *reinterpret_cast<const double2 *>(xp + a * xstep);
        const double xr = blk_flip(v.x, (a & 1) ? mo : me);
        const double xi = blk_flip(v.y, (a & 1) ? me : mo);
#pragma unroll
        for (int b = 0; b < BY; b++) {
            if (FIRST) {
                tr[a][b] = fma(-xi, yi[b], xr * yr[b]);
                ti[a][b] = fma(xi, yr[b], xr * yi[b]);
            } else {
                tr[a][b] = fma(xr, yr[b], tr[a][b]);
                tr[a][b] = fma(-xi, yi[b], tr[a][b]);
                ti[a][b] = fma(xr, yi[b], ti[a][b]);
                ti[a][b] = fma(xi, yr[b], ti[a][b]);
            }
        }
    }
}

// one unit: consumes its records from the reader and returns its contribution to B of its triple, per lane
// HALF (twojmax 11..14: U_tot of 32 points does not fit shared memory): the tile is 16 points, lane = (point, half), and the
// two half-warps take the items of the unit alternately (the host pads the item list to an even length with a zero-weight
// item); T, z and the dot product are linear in the items, so each half finishes its own share and the two scalars are added.
template <int BX, int BY, bool PEEL, bool HALF>
__device__ __forceinline__ double blk_unit(const unsigned char *Ulane, BlkReader &rd, int &slot, const int h) {
    constexpr int RB = (HALF ? 16 : 32) * (int)sizeof(double2);
    constexpr int NCW = (BX * BY + 1) / 2;
    double tr[BX][BY], ti[BX][BY];
    rd.ensure(rd.wpos + 1);
    // a unit never wraps around the ring: its words are read at fixed offsets from `base`
    uint32_t base = rd.ring + (uint32_t)((rd.wpos & (kBlkRingWords - 1)) * 16);
    const int4 hd = blk_lds4(base);
    const int nitems = hd.x, uboff = hd.y;   // nitems >= 1
    slot = hd.z;
    const int wend = rd.wpos + 1 + 3 * nitems + NCW;
    rd.ensure(wend);
    rd.wpos = wend + hd.w;
    base += 16 + (HALF ? 48 * h : 0);
    constexpr int ISTEP = HALF ? 96 : 48;
    const int ntrips = HALF ? (nitems >> 1) : nitems;
    // PEEL: the first item initialises the block (no zeroing pass, -4 % instructions) at the price of a second copy of the
    // item body; pays from twojmax 8 up, where a tile has enough work per fetched instruction
    if constexpr (PEEL) {
        blk_item<BX, BY, true>(Ulane, base, tr, ti);
        base += ISTEP;
    } else {
#pragma unroll
        for (int a = 0; a < BX; a++)
#pragma unroll
            for (int b = 0; b < BY; b++) { tr[a][b] = 0.0; ti[a][b] = 0.0; }
    }
    const int ifirst = PEEL ? 1 : 0;
#pragma unroll 1
    for (int i = ifirst; i < ntrips; i++) {
        blk_item<BX, BY, false>(Ulane, base, tr, ti);
        base += ISTEP;
    }
    if constexpr (HALF) base -= 48 * h;   // both halves read the same coefficients
    // z on the anti-diagonals of the block (coefficients = CG x fold weight, read where they are used: T dies element by
    // element, so the registers never hold the block and its coefficients together), dotted with conj(U^J[:, mb]) at once
    const unsigned char *ub = Ulane + uboff;
    double bs0 = 0.0, bs1 = 0.0;
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
        const double2 uu = *reinterpret_cast<const double2 *>(ub + d * RB);
        bs0 = fma(uu.x, zr, bs0);
        bs1 = fma(uu.y, zi, bs1);
    }
    rd.fill();   // only now: the requests overwrite ring words up to wpos, i.e. this unit's
    return bs0 + bs1;
}

template <int BX, int BY, bool PEEL, bool HALF>
__device__ __forceinline__ void blk_run_shape(const unsigned char *Ulane, const BlkTables &T, const int warp, const int lane, BlkReader &rd,
                                              double *P) {
    constexpr int shape = (BX - 1) * kBlkBY + (BY - 1);
    const int n = __ldg(T.wrange + warp * (kBlkShapes + 2) + shape);
#pragma unroll 1
    for (int k = 0; k < n; k++) {
        int slot;
        double b = blk_unit<BX, BY, PEEL, HALF>(Ulane, rd, slot, lane >> 4);
        if constexpr (HALF) {
            b += __shfl_xor_sync(0xffffffffu, b, 16);
            if (lane < 16) P[slot * 16 + lane] += b;
        } else {
            P[slot * 32 + lane] += b;
        }
    }
}

template <int BX, int BY, bool PEEL, bool HALF>
__device__ __forceinline__ void blk_run_all(const unsigned char *Ulane, const BlkTables &T, const int warp, const int lane, BlkReader &rd, double *P) {
    if constexpr (BX >= kBlkBXMin && BY >= kBlkBYMin) blk_run_shape<BX, BY, PEEL, HALF>(Ulane, T, warp, lane, rd, P);
    if constexpr (BY > 1) blk_run_all<BX, BY - 1, PEEL, HALF>(Ulane, T, warp, lane, rd, P);
    else if constexpr (BX > 1) blk_run_all<BX - 1, kBlkBY, PEEL, HALF>(Ulane, T, warp, lane, rd, P);
}

template <bool PEEL>
__global__ void __launch_bounds__(kBlkWarps * 32, 1)
compute_zi_bi_block_kernel(GridGeom g, SnapConst sc, DeviceTables tb, BlkTables T, ChunkBuffers cb, double *out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NW = kBlkWarps;
    const int nelem = sc.nelem, nt = sc.ntriples;
    double2 *U = reinterpret_cast<double2 *>(smem_raw + kBlkPadBytes);
    double *Bs = reinterpret_cast<double *>(U + (size_t)nelem * 32);
    double *P = Bs + 32 * nt;   // [nslots][32]
    int4 *rings = reinterpret_cast<int4 *>(P + (size_t)T.nslots * 32);   // [NW][kBlkRingWords]
    __shared__ uint64_t bar;
    __shared__ int s_slot;
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    for (int i = threadIdx.x; i < kBlkPadBytes / 8; i += NW * 32) reinterpret_cast<double *>(smem_raw)[i] = 0.0;
    for (int i = threadIdx.x; i < 32 * nt; i += NW * 32) Bs[i] = 0.0;   // the fold may read (times zero) past the last column
    uint32_t parity = 0;
    const int nactive = cb.counters[0];
    if (threadIdx.x == 0) s_slot = atomicAdd(&cb.counters[2], 1);
    for (;;) {
        __syncthreads();  // previous tile written out: Bs, P and U are free; s_slot is visible
        const int slot = s_slot;
        if (slot >= nactive) break;
        const int wt = cb.active[slot];
        __syncthreads();  // everybody has read s_slot
        if (threadIdx.x == 0) {
            tma_load_tile(U, cb.utot + (size_t)slot * nelem * 32, nelem, &bar);
            const int next = atomicAdd(&cb.counters[2], 1);   // claim the next tile now and pull its U_tot into L2
            s_slot = next;
            if (next < nactive) prefetch_l2_tile(cb.utot + (size_t)next * nelem * 32, nelem);
        }
        for (int i = threadIdx.x; i < T.nslots * 32; i += NW * 32) P[i] = 0.0;
        BlkReader rd;
        rd.src = T.stream + __ldg(T.wrange + warp * (kBlkShapes + 2) + kBlkShapes);
        rd.wtotal = __ldg(T.wrange + warp * (kBlkShapes + 2) + kBlkShapes + 1);
        rd.ring = smem_u32(rings + warp * kBlkRingWords);
        rd.lane = lane; rd.wpos = 0; rd.wreq = 0; rd.wready = 0;
        rd.fill();   // the first four chunks travel while the U_tot tile does
        mbar_wait(&bar, parity);
        parity ^= 1u;
        __syncthreads();  // P zeroed
        const unsigned char *Ulane = reinterpret_cast<const unsigned char *>(U + lane);
        blk_run_all<kBlkBX, kBlkBY, PEEL, false>(Ulane, T, warp, lane, rd, P);   // shapes in decreasing size: the order of the stream
        __syncthreads();
        for (int t = warp; t < nt; t += NW) {   // fixed-order sum of the slots of triple t
            double s = 0.0;
            for (int k = __ldg(T.tslot + t); k < __ldg(T.tslot + t + 1); k++) s += P[k * 32 + lane];
            Bs[lane * nt + t] = s;
        }
        __syncthreads();
        write_tile(g, cb.tile_begin + wt, Bs, nt, out, NW, cb.compact_out, wt);
    }
}

// twojmax 11..14: half tiles (16 points).  U_tot of the half tile (up to 167 KB at twojmax 14), the partial-sum slots and the
// rings fill the shared memory, so there is no staging of B: the sums of the slots go straight to global memory, a row of
// ntriples doubles per grid point.
#ifndef MALA_BLK_HALF_PEEL
#define MALA_BLK_HALF_PEEL true
#endif
__global__ void __launch_bounds__(kBlkWarps * 32, 1)
compute_zi_bi_block_half_kernel(GridGeom g, SnapConst sc, DeviceTables tb, BlkTables T, ChunkBuffers cb, double *out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NW = kBlkWarps;
    const int nelem = sc.nelem, nt = sc.ntriples;
    double2 *U = reinterpret_cast<double2 *>(smem_raw + kBlkPadBytes);          // [nelem][16]
    double *P = reinterpret_cast<double *>(U + (size_t)nelem * 16);              // [nslots][16]
    int4 *rings = reinterpret_cast<int4 *>(P + (size_t)T.nslots * 16);           // [NW][kBlkRingWords]
    __shared__ uint64_t bar;
    __shared__ int s_item;
    __shared__ long long s_dst[16];   // element offset of the output row of every point of the half tile, -1 = no such point
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    for (int i = threadIdx.x; i < kBlkPadBytes / 8; i += NW * 32) reinterpret_cast<double *>(smem_raw)[i] = 0.0;
    uint32_t parity = 0;
    const int nactive = cb.counters[0];
    const size_t half_elems = (size_t)nelem * 16;
    if (threadIdx.x == 0) s_item = atomicAdd(&cb.counters[2], 1);
    for (;;) {
        __syncthreads();  // previous half tile written out: P and U are free; s_item is visible
        const int item = s_item;
        const int slot = item >> 1, hh = item & 1;
        if (slot >= nactive) break;
        const int wt = cb.active[slot];
        __syncthreads();  // everybody has read s_item
        if (threadIdx.x == 0) {
            tma_load_bytes(U, cb.utot + (size_t)item * half_elems, (uint32_t)(half_elems * sizeof(double2)), &bar);
            s_item = atomicAdd(&cb.counters[2], 1);
        }
        if (threadIdx.x < 16) {
            long long off = -1;
            if (cb.compact_out) off = ((long long)wt * 32 + hh * 16 + threadIdx.x) * nt;
            else {
                int ix, iy, iz;
                bool valid;
                lane_point(g, cb.tile_begin + wt, hh * 16 + threadIdx.x, ix, iy, iz, valid);
                if (valid) off = ((long long)((long long)(iz - g.z0) * g.ny + iy) * g.nx + ix) * nt;
            }
            s_dst[threadIdx.x] = off;
        }
        for (int i = threadIdx.x; i < T.nslots * 16; i += NW * 32) P[i] = 0.0;
        BlkReader rd;
        rd.src = T.stream + __ldg(T.wrange + warp * (kBlkShapes + 2) + kBlkShapes);
        rd.wtotal = __ldg(T.wrange + warp * (kBlkShapes + 2) + kBlkShapes + 1);
        rd.ring = smem_u32(rings + warp * kBlkRingWords);
        rd.lane = lane; rd.wpos = 0; rd.wreq = 0; rd.wready = 0;
        rd.fill();
        mbar_wait(&bar, parity);
        parity ^= 1u;
        __syncthreads();  // P zeroed, s_dst written
        const unsigned char *Ulane = reinterpret_cast<const unsigned char *>(U + (lane & 15));
        blk_run_all<kBlkBX, kBlkBY, MALA_BLK_HALF_PEEL, true>(Ulane, T, warp, lane, rd, P);
        __syncthreads();
        for (int i = threadIdx.x; i < 16 * nt; i += NW * 32) {   // fixed-order sum of the slots of triple t, point p
            const int p = i / nt, t = i - p * nt;
            const long long off = s_dst[p];
            if (off < 0) continue;
            double sum = 0.0;
            for (int k = __ldg(T.tslot + t); k < __ldg(T.tslot + t + 1); k++) sum += P[k * 16 + p];
            __stcs(out + off + t, sum);
        }
    }
}

constexpr int kBlkHalfSmemMax = 232448 - 256;   // the 227 KB of an SM less the kernel's static shared memory
inline size_t compute_zi_block_half_smem_bytes(int nelem, int nslots) {
    return (size_t)kBlkPadBytes + (size_t)nelem * 16 * sizeof(double2) + (size_t)nslots * 16 * sizeof(double) + (size_t)kBlkWarps * kBlkRingWords * 16 + 16;
}

inline size_t compute_zi_block_smem_bytes(int nelem, int nt, int nslots) {
    return (size_t)kBlkPadBytes + (size_t)nelem * 32 * sizeof(double2) + (size_t)32 * nt * sizeof(double) + (size_t)nslots * 32 * sizeof(double) +
           (size_t)kBlkWarps * kBlkRingWords * 16 + 16;
}

}  // namespace mala
