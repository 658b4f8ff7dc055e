// snap_zi.cuh -- compute_zi / compute_bi kernels and the output writer (rows a5, a6, a7 of SURVEY.md 8(a)).
//
//   Z^{j}_{j1 j2}[ma][mb] = sum_{ma1,mb1} CG(j1 ma1 j2 ma2 ; j ma) CG(j1 mb1 j2 mb2 ; j mb) U^{j1}[ma1][mb1] U^{j2}[ma2][mb2]
//   B_{j1 j2 j}           = Re sum_{ma,mb} conj(U^{j}[ma][mb]) Z[ma][mb]            ("scalar triple products")
//
// evaluated over half columns (mb <= J/2; the middle column of an even J only for ma <= J/2) using
// u[J-ma][J-mb] = (-1)^(ma-mb) conj(u[ma][mb]).  Layout: one tile = 32 grid points = the 32 lanes of every warp;
// U_tot of the tile sits in shared memory as [element][lane] double2 (TMA bulk-loaded), the CG coefficients are
// warp-uniform.  Z is never stored: each warp owns whole triples, keeps one Z column in registers and folds
// it into B at once (compute_bi fused).
//
// Two kernels: a table-driven generic one (any twojmax <= 10) and one specialised at compile time per triple
// (twojmax = 10), where the inner double sum over (ma1, ma2) is a fully unrolled "CG-weighted convolution" of two
// register-resident columns with the CG values read from constant memory through uniform registers.
#pragma once
#include <utility>

#include "snap_common.cuh"

namespace mala {

// ---- TMA / mbarrier helpers (1-D bulk copies, sm_90+) -------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_1d(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// issue a bulk load of `total` bytes (a multiple of 16) in pieces of at most 32 KB, all completing on one mbarrier phase
__device__ __forceinline__ void tma_load_bytes(void *dst, const void *src, uint32_t total, uint64_t *bar) {
    mbar_expect_tx(bar, total);
    uint32_t done = 0;
    while (done < total) {
        const uint32_t n = min(total - done, 32768u);
        tma_load_1d(reinterpret_cast<unsigned char *>(dst) + done, reinterpret_cast<const unsigned char *>(src) + done, n, bar);
        done += n;
    }
}

// issue the bulk load of one U_tot tile (nelem*512 bytes) in pieces of at most 32 KB
__device__ __forceinline__ void tma_load_tile(double2 *dst, const double2 *src, int nelem, uint64_t *bar) {
    const uint32_t total = (uint32_t)nelem * 32u * (uint32_t)sizeof(double2);
    mbar_expect_tx(bar, total);
    uint32_t done = 0;
    while (done < total) {
        const uint32_t n = min(total - done, 32768u);
        tma_load_1d(reinterpret_cast<unsigned char *>(dst) + done, reinterpret_cast<const unsigned char *>(src) + done, n, bar);
        done += n;
    }
}

// L2 prefetch of one U_tot tile (no completion tracking: a hint)
__device__ __forceinline__ void prefetch_l2_tile(const double2 *src, int nelem) {
    const uint32_t total = (uint32_t)nelem * 32u * (uint32_t)sizeof(double2);
    for (uint32_t done = 0; done < total; done += 32768u) {
        const uint32_t n = min(total - done, 32768u);
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(reinterpret_cast<const unsigned char *>(src) + done), "r"(n) : "memory");
    }
}

// ---- writer (row a7): B of one tile, staged as Bs[lane][nt] in shared memory, to out[point][nt] --------------
// Points of one tile row (fixed iy, iz) are consecutive in x, so a row is one contiguous run of npx*nt doubles.
// compact (ChunkBuffers::compact_out): the tile's 32 x nt block goes, as it is, to out[wt * 32 ...] (wt = tile id in the chunk).
__device__ __forceinline__ void write_tile(const GridGeom &g, int tile, const double *Bs, int nt, double *out, int nwarps,
                                           int compact = 0, int wt = 0) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (compact) {
        double2 *d2 = reinterpret_cast<double2 *>(out + (size_t)wt * 32 * nt);   // 32 * nt * 8 bytes is a multiple of 16
        const double2 *s2 = reinterpret_cast<const double2 *>(Bs);
        for (int i = threadIdx.x; i < 16 * nt; i += nwarps * 32) __stcs(d2 + i, s2[i]);
        return;
    }
    const TileInfo ti = tile_info(g, tile);
    const int ix0 = ti.ix0;
    const int npx = min(ti.tx, ti.xend - ix0);
    for (int r = warp; r < ti.ty * ti.tz; r += nwarps) {
        const int iy = ti.iy0 + (r % ti.ty);
        const int iz = ti.iz0 + (r / ti.ty);
        if (iy >= ti.yend || iz >= g.z1) continue;
        double *dst = out + ((size_t)((size_t)(iz - g.z0) * g.ny + iy) * g.nx + ix0) * nt;
        const double *src = Bs + (size_t)(r * ti.tx) * nt;  // lanes r*tx .. r*tx+npx-1 are contiguous in Bs
        const int n = npx * nt;
        if (((((uintptr_t)dst) | ((uintptr_t)src)) & 15) == 0) {
            // 16-byte vector stores over the even part, scalar tail
            const int n2 = n >> 1;
            const double2 *s2 = reinterpret_cast<const double2 *>(src);
            double2 *d2 = reinterpret_cast<double2 *>(dst);
            for (int i = lane; i < n2; i += 32) __stcs(d2 + i, s2[i]);
            if ((n & 1) && lane == 0) __stcs(dst + n - 1, src[n - 1]);
            continue;
        }
        for (int i = lane; i < n; i += 32) __stcs(dst + i, src[i]);
    }
}

// =============================================================================================================
// Generic kernel: runtime twojmax, table-driven loops, one Z element at a time.
// =============================================================================================================
__device__ double triple_b_generic(const double2 *Ul, const int *uoff, int J1, int J2, int J, const double *cg) {
    const int sh = (J1 + J2 - J) / 2;
    double B = 0.0;
    for (int mb = 0; mb <= J / 2; mb++) {
        const bool mid = ((J & 1) == 0) && (mb == J / 2);
        const int mahi = mid ? J / 2 : J;
        const int mb1lo = max(0, mb + sh - J2), mb1hi = min(J1, mb + sh);
        for (int ma = 0; ma <= mahi; ma++) {
            double zr = 0.0, zi = 0.0;
            const int ma1lo = max(0, ma + sh - J2), ma1hi = min(J1, ma + sh);
            for (int mb1 = mb1lo; mb1 <= mb1hi; mb1++) {
                const int mb2 = mb + sh - mb1;
                const double cgb = cg[mb2 * (J1 + 1) + mb1];
                double sr = 0.0, si = 0.0;
                for (int ma1 = ma1lo; ma1 <= ma1hi; ma1++) {
                    const int ma2 = ma + sh - ma1;
                    const double cga = cg[ma2 * (J1 + 1) + ma1];
                    // symmetric loads, with level offsets from the table
                    double2 x, y;
                    if (mb1 <= J1 / 2) x = Ul[(size_t)(uoff[J1] + mb1 * (J1 + 1) + ma1) * 32];
                    else {
                        const double2 v = Ul[(size_t)(uoff[J1] + (J1 - mb1) * (J1 + 1) + (J1 - ma1)) * 32];
                        const double s = ((ma1 - mb1) & 1) ? -1.0 : 1.0;
                        x = make_double2(s * v.x, -s * v.y);
                    }
                    if (mb2 <= J2 / 2) y = Ul[(size_t)(uoff[J2] + mb2 * (J2 + 1) + ma2) * 32];
                    else {
                        const double2 v = Ul[(size_t)(uoff[J2] + (J2 - mb2) * (J2 + 1) + (J2 - ma2)) * 32];
                        const double s = ((ma2 - mb2) & 1) ? -1.0 : 1.0;
                        y = make_double2(s * v.x, -s * v.y);
                    }
                    sr += cga * (x.x * y.x - x.y * y.y);
                    si += cga * (x.x * y.y + x.y * y.x);
                }
                zr += cgb * sr;
                zi += cgb * si;
            }
            const double2 u = Ul[(size_t)(uoff[J] + mb * (J + 1) + ma) * 32];
            const double w = mid ? (ma < J / 2 ? 2.0 : 1.0) : 2.0;
            B += w * (u.x * zr + u.y * zi);
        }
    }
    return B;
}

constexpr int kZiWarps = 8;

__global__ void __launch_bounds__(kZiWarps * 32, 1)
compute_zi_bi_generic_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb, double *out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nelem = sc.nelem, nt = sc.ntriples;
    double2 *U = reinterpret_cast<double2 *>(smem_raw);
    double *Bs = reinterpret_cast<double *>(U + (size_t)nelem * 32);
    __shared__ uint64_t bar;
    __shared__ int s_slot, s_item;
    __shared__ int s_uoff[kMaxTwoJ + 2];
    const int lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        int o = 0;
        for (int J = 0; J <= kMaxTwoJ + 1; J++) {
            s_uoff[J] = o;
            o += (J + 1) * (J / 2 + 1);
        }
    }
    uint32_t parity = 0;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) {
            s_slot = atomicAdd(&cb.counters[2], 1);
            s_item = 0;
        }
        __syncthreads();
        const int slot = s_slot;
        if (slot >= cb.counters[0]) break;
        const int wt = cb.active[slot];
        if (threadIdx.x == 0) tma_load_tile(U, cb.utot + (size_t)slot * nelem * 32, nelem, &bar);
        mbar_wait(&bar, parity);
        parity ^= 1u;
        const double2 *Ul = U + lane;
        // triples are handed out dynamically in order of decreasing cost (longest first => balanced tail)
        for (;;) {
            int pos = 0;
            if (lane == 0) pos = atomicAdd(&s_item, 1);
            pos = __shfl_sync(0xffffffffu, pos, 0);
            if (pos >= nt) break;
            const int t = tb.order[pos];
            const int J1 = tb.triples[4 * t], J2 = tb.triples[4 * t + 1], J = tb.triples[4 * t + 2];
            const double b = triple_b_generic(Ul, s_uoff, J1, J2, J, tb.cg + tb.triples[4 * t + 3]);
            Bs[lane * nt + t] = b;
        }
        __syncthreads();
        write_tile(g, cb.tile_begin + wt, Bs, nt, out, kZiWarps, cb.compact_out, wt);
    }
}

inline size_t compute_zi_smem_bytes(int nelem, int nt) {
    return (size_t)nelem * 32 * sizeof(double2) + (size_t)32 * nt * sizeof(double) + 16;
}

}  // namespace mala
