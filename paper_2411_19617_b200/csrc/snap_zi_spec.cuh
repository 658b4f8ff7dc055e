// snap_zi_spec.cuh -- compute_zi/compute_bi specialised at compile time (rows a5 + a6), twojmax fixed by TJ.
//
// For a triple (J1,J2,J), output column mb and one (mb1, mb2 = mb + sh - mb1) pair, the inner sum over (ma1, ma2)
//     z[ma] += cgb * sum_{ma1 + ma2 - sh = ma} CG(ma1, ma2) * x[ma1] * y[ma2],   x = U^{J1}[:, mb1], y = U^{J2}[:, mb2]
// is a CG-weighted 1-D convolution of two columns.  Here x (<= 11 complex) and z (<= 11 complex) live in registers,
// y is streamed one element at a time (pre-multiplied by cgb and by the sign/conjugation of the column-flip
// symmetry), and the (ma1, ma2) loops are unrolled at compile time so every register index and every CG address is
// static; the CG values come from constant memory via uniform registers, costing neither shared-memory bandwidth
// nor vector registers.  6 FP64-pipe instructions per product term, ~0.3 B of shared-memory traffic per flop.
#pragma once
#include "snap_zi.cuh"

namespace mala {

constexpr int kSpecTJ = 10;
constexpr int kSpecNT = triple_count(kSpecTJ);
constexpr int kSpecCG = cg_block_off(kSpecTJ, kSpecNT);

__constant__ double c_cg_spec[kSpecCG];  // dense CG blocks of every triple, [m2][m1]
__constant__ int c_order_spec[kSpecNT];  // triples by decreasing cost

constexpr int kRowBytes = 32 * (int)sizeof(double2);  // bytes between consecutive elements of one lane

__device__ __forceinline__ double flip_sign(double v, unsigned mask) {
    return __hiloint2double(__double2hiint(v) ^ (int)mask, __double2loint(v));
}

// z[ma] += sum CG * x[ma1] * (scaled y[ma2]) for one (mb1, mb2) pair.  MID restricts to ma <= J/2.
template <int J1, int J2, int J, int CGOFF, bool MID>
__device__ __forceinline__ void cg_convolve(double (&zr)[J + 1], double (&zi)[J + 1], const double (&xr)[J1 + 1],
                                            const double (&xi)[J1 + 1], const unsigned char *ybase, const int ystep,
                                            const double sre0, const double sre1, const double sim0, const double sim1) {
    constexpr int SH = (J1 + J2 - J) / 2;
    constexpr int MAHI = MID ? J / 2 : J;
#pragma unroll
    for (int ma2 = 0; ma2 <= J2; ma2++) {
        const int lo = (SH - ma2) > 0 ? (SH - ma2) : 0;
        const int hi = (MAHI + SH - ma2) < J1 ? (MAHI + SH - ma2) : J1;
        if (lo <= hi) {
            const double2 yv = *reinterpret_cast<const double2 *>(ybase + ma2 * ystep);
            const double yr = yv.x * ((ma2 & 1) ? sre1 : sre0);
            const double yi = yv.y * ((ma2 & 1) ? sim1 : sim0);
#pragma unroll
            for (int ma1 = 0; ma1 <= J1; ma1++) {
                if (ma1 >= lo && ma1 <= hi) {
                    const int ma = ma1 + ma2 - SH;
                    const double cg = c_cg_spec[CGOFF + ma2 * (J1 + 1) + ma1];
                    const double tr = cg * xr[ma1];
                    const double ti = cg * xi[ma1];
                    zr[ma] = fma(tr, yr, zr[ma]);
                    zr[ma] = fma(-ti, yi, zr[ma]);
                    zi[ma] = fma(tr, yi, zi[ma]);
                    zi[ma] = fma(ti, yr, zi[ma]);
                }
            }
        }
    }
}

// one output column mb of one triple: returns its contribution to B
template <int J1, int J2, int J, int CGOFF, bool MID>
__device__ __forceinline__ double column_b(const unsigned char *Ulane, const int mb) {
    constexpr int SH = (J1 + J2 - J) / 2;
    double zr[J + 1], zi[J + 1];
#pragma unroll
    for (int k = 0; k <= J; k++) { zr[k] = 0.0; zi[k] = 0.0; }
    const int mb1lo = (mb + SH - J2) > 0 ? (mb + SH - J2) : 0;
    const int mb1hi = (mb + SH) < J1 ? (mb + SH) : J1;
    for (int mb1 = mb1lo; mb1 <= mb1hi; mb1++) {
        const int mb2 = mb + SH - mb1;
        const double cgb = c_cg_spec[CGOFF + mb2 * (J1 + 1) + mb1];
        // x = U^{J1}[:, mb1]; columns beyond the middle come from the stored half by
        // u[ma][mb] = (-1)^(ma-mb) conj(u[J-ma][J-mb])
        const bool fx = mb1 > J1 / 2;
        const int cx = fx ? J1 - mb1 : mb1;
        const unsigned char *xb = Ulane + (uhalf_off(J1) + cx * (J1 + 1) + (fx ? J1 : 0)) * kRowBytes;
        const int xstep = fx ? -kRowBytes : kRowBytes;
        // sign masks by parity of ma1: real part (-1)^(ma1-mb1), imaginary part the opposite (conjugation)
        const unsigned mxr0 = (fx && (mb1 & 1)) ? 0x80000000u : 0u;
        const unsigned mxr1 = (fx && !(mb1 & 1)) ? 0x80000000u : 0u;
        const unsigned mxi0 = fx ? (mxr0 ^ 0x80000000u) : 0u;
        const unsigned mxi1 = fx ? (mxr1 ^ 0x80000000u) : 0u;
        double xr[J1 + 1], xi[J1 + 1];
#pragma unroll
        for (int k = 0; k <= J1; k++) {
            const double2 v = *reinterpret_cast<const double2 *>(xb + k * xstep);
            xr[k] = flip_sign(v.x, (k & 1) ? mxr1 : mxr0);
            xi[k] = flip_sign(v.y, (k & 1) ? mxi1 : mxi0);
        }
        // y = U^{J2}[:, mb2], same symmetry, folded with cgb into four scale factors
        const bool fy = mb2 > J2 / 2;
        const int cy = fy ? J2 - mb2 : mb2;
        const unsigned char *yb = Ulane + (uhalf_off(J2) + cy * (J2 + 1) + (fy ? J2 : 0)) * kRowBytes;
        const int ystep = fy ? -kRowBytes : kRowBytes;
        const double p0 = (fy && (mb2 & 1)) ? -cgb : cgb;  // parity-0 rows, real part
        const double p1 = fy ? -p0 : cgb;                  // parity-1 rows, real part
        const double q0 = fy ? -p0 : cgb;                  // imaginary parts: conjugation flips the sign again
        const double q1 = fy ? -p1 : cgb;
        cg_convolve<J1, J2, J, CGOFF, MID>(zr, zi, xr, xi, yb, ystep, p0, p1, q0, q1);
    }
    // compute_bi: B += w * Re(conj(U^J[ma][mb]) * z[ma]);  w = 2 except on the middle column (2 below, 1 on, the centre)
    const unsigned char *ub = Ulane + (uhalf_off(J) + mb * (J + 1)) * kRowBytes;
    double b = 0.0;
#pragma unroll
    for (int ma = 0; ma <= (MID ? J / 2 : J); ma++) {
        const double2 u = *reinterpret_cast<const double2 *>(ub + ma * kRowBytes);
        const double w = (MID && ma == J / 2) ? 1.0 : 2.0;
        b = fma(w * u.x, zr[ma], b);
        b = fma(w * u.y, zi[ma], b);
    }
    return b;
}

template <int T>
__device__ __noinline__ double triple_b_spec(const unsigned char *Ulane) {
    constexpr Triple tr = triple_at(kSpecTJ, T);
    constexpr int J1 = tr.j1, J2 = tr.j2, J = tr.j;
    constexpr int CGOFF = cg_block_off(kSpecTJ, T);
    double b = 0.0;
    for (int mb = 0; mb < (J + 1) / 2; mb++) b += column_b<J1, J2, J, CGOFF, false>(Ulane, mb);
    if ((J & 1) == 0) b += column_b<J1, J2, J, CGOFF, true>(Ulane, J / 2);
    return b;
}

__device__ __forceinline__ double dispatch_triple(const int t, const unsigned char *Ulane) {
    double b = 0.0;
    switch (t) {
        // one case per triple
#define MALA_CASE(N) \
    case N:          \
        if (N < kSpecNT) b = triple_b_spec<(N < kSpecNT ? N : 0)>(Ulane); \
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

template <int NWARPS>
__global__ void __launch_bounds__(NWARPS * 32, 1)
compute_zi_bi_spec_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb, double *out) {
    static_assert(kSpecNT <= 100, "dispatch_triple covers 100 cases");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int nelem = uhalf_size(kSpecTJ), nt = kSpecNT;
    double2 *U = reinterpret_cast<double2 *>(smem_raw);
    double *Bs = reinterpret_cast<double *>(U + (size_t)nelem * 32);
    __shared__ uint64_t bar;
    __shared__ int s_slot, s_item;
    const int lane = threadIdx.x & 31;
    if (threadIdx.x == 0) mbar_init(&bar, 1);
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
        const unsigned char *Ulane = reinterpret_cast<const unsigned char *>(U + lane);
        for (;;) {
            int pos = 0;
            if (lane == 0) pos = atomicAdd(&s_item, 1);
            pos = __shfl_sync(0xffffffffu, pos, 0);
            if (pos >= nt) break;
            const int t = c_order_spec[pos];
            Bs[lane * nt + t] = dispatch_triple(t, Ulane);
        }
        __syncthreads();
        write_tile(g, cb.tile_begin + wt, Bs, nt, out, NWARPS);
    }
}

}  // namespace mala
