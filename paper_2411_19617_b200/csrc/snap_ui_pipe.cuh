// snap_ui_pipe.cuh -- the sampling compute_ui of snap_ui_dft.cuh as a producer / consumer pipeline (rows a3 + a4), twojmax 8..10.
//
// At these twojmax the sums of a sample fill the registers, one CTA of twojmax + 1 warps owns an SM, and everything in front of
// the accumulation -- claiming a tile, four dependent global loads for its candidates, distance tests, the pair geometry (a
// square root, two divisions, three trigonometric values per pair) -- is latency-bound work between barriers during which the
// FP64 pipe idles: about a third of the kernel.  twojmax + 1 = 9..11 warps also leave one of the four schedulers a warp short.
// Here that slot goes to a PRODUCER warp (lane = grid point) which prepares the neighbor queue of the NEXT tile while the
// twojmax + 1 CONSUMER warps (warp = sample point, as before) accumulate and transform the current one:
//
//   producer   claim tile -> candidates -> distance tests -> pair geometry -> geo[buf][entry][c, ar, ai, br, bi][lane]   -> full[buf]
//   consumers  full[buf] -> sums of chains mb < SPLIT -> S -> inverse DFT of those columns -> sums of the other chains
//              -> empty[buf] -> S -> inverse DFT of those columns
//
// Two queue buffers (mbarriers full / empty, the usual parities), consumer-only named barriers around the two uses of S.  The
// inverse DFT runs in two parts so that S holds the columns of one pass only: S (113 KB at twojmax 10) and two queues of
// kPipeCap entries (2 x 51 KB) fit the 227 KB of an SM.  A tile with more candidates than kPipeCap is sent window by window,
// once per pass.  The arithmetic of a sample is that of compute_ui_dft_kernel (dft_accumulate); summation order is fixed.
#pragma once
#include "snap_ui_dft.cuh"
#include "snap_zi.cuh"

namespace mala {

constexpr int kPipeCap = 40;     // candidates per window = entries of a queue buffer
constexpr int kPipeMaxTasks = 6; // pieces of columns one warp transforms per pass

constexpr int pipe_split(int tj) { return 2; }
constexpr int pipe_ka(int tj) { return dft_index(tj, pipe_split(tj), pipe_split(tj)); }                  // columns of the first pass
constexpr int pipe_kmax(int tj) { return pipe_ka(tj) > dft_njm(tj) - pipe_ka(tj) ? pipe_ka(tj) : dft_njm(tj) - pipe_ka(tj); }

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
template <int NTHREADS>
__device__ __forceinline__ void consumer_barrier() {
    asm volatile("bar.sync 1, %0;" ::"n"(NTHREADS) : "memory");
}

struct PipeTask { unsigned short scol, e0, k0, k1; };   // column index inside its pass, first element of the column, coefficients k0 <= k < k1

// inverse DFT of this warp's pieces of columns: q_k = (1/NW) sum_s S_s x_s^(-k) over conjugate sample pairs (snap_ui_dft.cuh),
// then the binomial normalisation and the self term.  S holds the columns of one pass: [column][sample][lane].
template <int TJ>
__device__ __forceinline__ void pipe_dft(const double2 *S, const PipeTask *tasks, const int ntasks, const int lane, const double2 *s_tw,
                                         double2 *dst, const double2 *s_norm) {
    constexpr int NW = TJ + 1, NP = (NW - 1) / 2;
    for (int ti = 0; ti < ntasks; ti++) {
        const PipeTask t = tasks[ti];
        const double2 *Sp = S + (size_t)t.scol * NW * 32 + lane;
        double pr_[NP], pi_[NP], mr_[NP], mi_[NP];
        const double2 v0 = Sp[0];
        double2 vh = make_double2(0.0, 0.0);   // the sample at x = -1 (even NW only)
        if constexpr (NW % 2 == 0) vh = Sp[(size_t)(NW / 2) * 32];
#pragma unroll
        for (int sI = 1; sI <= NP; sI++) {
            const double2 va = Sp[(size_t)sI * 32], vb = Sp[(size_t)(NW - sI) * 32];
            pr_[sI - 1] = va.x + vb.x; pi_[sI - 1] = va.y + vb.y;
            mr_[sI - 1] = va.x - vb.x; mi_[sI - 1] = va.y - vb.y;
        }
#pragma unroll 2
        for (int k = t.k0; k < t.k1; k++) {
            const double2 *tw = s_tw + k * NW;
            const double sg = (k & 1) ? -1.0 : 1.0;
            double sr = fma(sg, vh.x, v0.x), si = fma(sg, vh.y, v0.y);
#pragma unroll
            for (int sI = 1; sI <= NP; sI++) {
                const double2 w = tw[sI];
                sr = fma(pr_[sI - 1], w.x, sr); sr = fma(-mi_[sI - 1], w.y, sr);
                si = fma(pi_[sI - 1], w.x, si); si = fma(mr_[sI - 1], w.y, si);
            }
            const int e = t.e0 + k;
            const double2 nrm = s_norm[e];   // binomial normalisation / NW, self term of the diagonal elements
            dst[(size_t)e * 32 + lane] = make_double2(fma(sr, nrm.x, nrm.y), si * nrm.x);
        }
    }
}

template <int TJ>
__global__ void __launch_bounds__((TJ + 2) * 32, 1)
compute_ui_pipe_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb) {
    constexpr int NW = TJ + 1;          // consumer warps = sample points; warp NW is the producer
    constexpr int NJM = dft_njm(TJ);
    constexpr int nelem = uhalf_size(TJ);
    constexpr int SPLIT = pipe_split(TJ), KA = pipe_ka(TJ), KB = NJM - KA, KMAX = pipe_kmax(TJ);
    constexpr int GEO = kPipeCap * 5 * 32;   // doubles per queue buffer
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *S = reinterpret_cast<double2 *>(smem_raw);                       // [KMAX][NW][32]
    double *geo = reinterpret_cast<double *>(S + (size_t)KMAX * NW * 32);     // [2][kPipeCap][5][32]
    double *crec = geo + 2 * GEO;                                             // [kPipeCap][6], the producer's
    __shared__ uint64_t full[2], empty[2];
    __shared__ int s_cnt[2][32];          // entries of every lane's queue in the buffer
    __shared__ int s_meta[2][2];          // slot of the tile the buffer belongs to (-1: no more tiles), windows of that tile
    __shared__ double2 s_tw[NW * NW];     // [k][s] = x_s^(-k) = e^{-2 pi i s k / NW}
    __shared__ double2 s_norm[nelem];     // {unorm / NW, wself on the diagonal}
    __shared__ PipeTask s_task[2][NW][kPipeMaxTasks];
    __shared__ int s_ntask[2][NW];
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    if (threadIdx.x < NW * NW) {
        double sn, cs;
        sincospi(2.0 * (double)(((threadIdx.x / NW) * (threadIdx.x % NW)) % NW) / (double)NW, &sn, &cs);
        s_tw[threadIdx.x] = make_double2(cs, -sn);
    }
    for (int e = threadIdx.x; e < nelem; e += (NW + 1) * 32) s_norm[e] = make_double2(tb.unorm[e] * (1.0 / (double)NW), tb.udiag[e] ? sc.wself : 0.0);
    if (threadIdx.x == NW * 32) {
        mbar_init(&full[0], 32); mbar_init(&full[1], 32);
        mbar_init(&empty[0], NW); mbar_init(&empty[1], NW);
    }
    if (threadIdx.x == 0) {
        // the coefficients of a pass's columns, cut into NW runs of equal length: every warp transforms the same number of them
        for (int pass = 0; pass < 2; pass++) {
            const int mb0 = pass ? SPLIT : 0, mb1 = pass ? TJ / 2 + 1 : SPLIT;
            int total = 0;
            for (int mb = mb0; mb < mb1; mb++)
                for (int n = mb; n <= TJ - mb; n++) total += mb + n + 1;
            const int target = (total + NW - 1) / NW;
            int w = 0, room = target, scol = 0;
            for (int i = 0; i < NW; i++) s_ntask[pass][i] = 0;
            for (int mb = mb0; mb < mb1; mb++)
                for (int n = mb; n <= TJ - mb; n++, scol++) {
                    const int J = mb + n;
                    int k = 0;
                    while (k <= J) {
                        const int take = min(room, J + 1 - k);
                        PipeTask t;
                        t.scol = (unsigned short)scol; t.e0 = (unsigned short)(uhalf_off(J) + mb * (J + 1));
                        t.k0 = (unsigned short)k; t.k1 = (unsigned short)(k + take);
                        s_task[pass][w][s_ntask[pass][w]++] = t;
                        k += take; room -= take;
                        if (room == 0) { w++; room = target; }
                    }
                }
        }
    }
    __syncthreads();
    const int nactive = cb.counters[0];

    if (warp == NW) {
        // ---------------------------------------------------------------- producer: lane = grid point
        uint32_t it = 0;   // buffers handed over so far
        for (;;) {
            int slot = 0;
            if (lane == 0) slot = atomicAdd(&cb.counters[1], 1);
            slot = __shfl_sync(0xffffffffu, slot, 0);
            if (slot >= nactive) {
                const int buf = it & 1;
                mbar_wait(&empty[buf], ((it >> 1) & 1) ^ 1);
                if (lane == 0) s_meta[buf][0] = -1;
                mbar_arrive(&full[buf]);
                break;
            }
            const int wt = cb.active[slot];
            int ix, iy, iz;
            bool valid;
            lane_point(g, cb.tile_begin + wt, lane, ix, iy, iz, valid);
            ix = min(ix, g.nx - 1); iy = min(iy, g.ny - 1); iz = min(iz, g.z1 - 1);  // ragged tiles: a valid point whose result is never used
            double px, py, pz;
            point_position(g, ix, iy, iz, px, py, pz);
            const int nc = cb.ncand[wt];
            const int *mycand = cb.cand + (size_t)wt * cb.cand_cap;
            const int nwin = max(1, (nc + kPipeCap - 1) / kPipeCap);
            const int rounds = (nwin > 1 && KB > 0) ? 2 : 1;   // several windows are sent once per pass
            for (int round = 0; round < rounds; round++)
                for (int win = 0; win < nwin; win++, it++) {
                    const int wbase = win * kPipeCap, nw = min(kPipeCap, nc - wbase), buf = it & 1;
                    __syncwarp();
                    for (int k = lane; k < nw; k += 32) {
                        const Ghost gh = cb.ghosts[mycand[wbase + k]];
                        const double rc = tb.type_rcut[gh.type];
                        double *q = crec + k * 6;
                        q[0] = gh.x; q[1] = gh.y; q[2] = gh.z; q[3] = rc; q[4] = tb.type_w[gh.type]; q[5] = rc * rc;
                    }
                    __syncwarp();
                    unsigned long long hits = 0ull;
                    for (int k = 0; k < nw; k++) {
                        const double *q = crec + k * 6;
                        const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                        if (dx * dx + dy * dy + dz * dz < q[5]) hits |= 1ull << k;
                    }
                    mbar_wait(&empty[buf], ((it >> 1) & 1) ^ 1);   // the consumers are done with this buffer
                    double *gq = geo + (size_t)buf * GEO + lane;
                    for (unsigned long long r = hits; r != 0ull; r &= r - 1ull, gq += 5 * 32) {
                        const double *q = crec + (__ffsll((long long)r) - 1) * 6;
                        const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                        const double r2 = dx * dx + dy * dy + dz * dz;
                        double c, ar, ai, br, bi;
                        pair_geometry(dx, dy, dz, r2, q[3], q[4], sc.rfac0, sc.rmin0, c, ar, ai, br, bi);
                        gq[0] = c; gq[32] = ar; gq[64] = ai; gq[96] = br; gq[128] = bi;
                    }
                    s_cnt[buf][lane] = __popcll(hits);
                    if (lane == 0) { s_meta[buf][0] = slot; s_meta[buf][1] = nwin; }
                    mbar_arrive(&full[buf]);
                }
        }
        return;
    }

    // -------------------------------------------------------------------- consumers: warp = sample point, lane = grid point
    double xsr, xsi;                    // this warp's sample point x_s = e^{2 pi i s / NW}
    {
        double sn, cs;
        sincospi(2.0 * (double)warp / (double)NW, &sn, &cs);
        xsr = cs; xsi = sn;
    }
    uint32_t it = 0;   // buffers taken so far
    for (;;) {
        int buf = it & 1;
        mbar_wait(&full[buf], (it >> 1) & 1);
        const int slot = s_meta[buf][0];
        if (slot < 0) break;
        const int nwin = s_meta[buf][1];
        double2 *dst = cb.utot + (size_t)slot * nelem * 32;
        {   // first pass: chains mb < SPLIT
            double accr[NJM], acci[NJM];   // KA of them in use
#pragma unroll
            for (int k = 0; k < KA; k++) { accr[k] = 0.0; acci[k] = 0.0; }
            for (int win = 0;;) {
                dft_accumulate<TJ, 0, SPLIT>(geo + (size_t)buf * GEO, lane, s_cnt[buf][lane], xsr, xsi, accr, acci);
                if (nwin == 1 && KB > 0) break;   // a single window stays for the second pass
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[buf]);
                it++;
                if (++win == nwin) break;
                buf = it & 1;
                mbar_wait(&full[buf], (it >> 1) & 1);
            }
#pragma unroll
            for (int k = 0; k < KA; k++) S[((size_t)k * NW + warp) * 32 + lane] = make_double2(accr[k], acci[k]);
        }
        consumer_barrier<NW * 32>();
        pipe_dft<TJ>(S, s_task[0][warp], s_ntask[0][warp], lane, s_tw, dst, s_norm);
        if constexpr (KB > 0) {
            consumer_barrier<NW * 32>();   // S is free again
            double accr[NJM], acci[NJM];   // KB of them in use
#pragma unroll
            for (int k = 0; k < KB; k++) { accr[k] = 0.0; acci[k] = 0.0; }
            for (int win = 0;;) {
                if (nwin > 1) {
                    buf = it & 1;
                    mbar_wait(&full[buf], (it >> 1) & 1);
                }
                dft_accumulate<TJ, SPLIT, TJ / 2 + 1>(geo + (size_t)buf * GEO, lane, s_cnt[buf][lane], xsr, xsi, accr, acci);
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[buf]);
                it++;
                if (++win == nwin) break;
            }
#pragma unroll
            for (int k = 0; k < KB; k++) S[((size_t)k * NW + warp) * 32 + lane] = make_double2(accr[k], acci[k]);
            consumer_barrier<NW * 32>();
            pipe_dft<TJ>(S, s_task[1][warp], s_ntask[1][warp], lane, s_tw, dst, s_norm);
        }
        consumer_barrier<NW * 32>();   // S is free for the next tile
    }
}

template <int TJ>
inline size_t compute_ui_pipe_smem_bytes() {
    return (size_t)pipe_kmax(TJ) * (TJ + 1) * 32 * sizeof(double2) + (size_t)2 * kPipeCap * 5 * 32 * sizeof(double) +
           (size_t)kPipeCap * 6 * sizeof(double) + 16;
}

}  // namespace mala
