// snap_ui_pipe.cuh -- the sampling compute_ui of snap_ui_dft.cuh as a producer / consumer pipeline (rows a3 + a4), twojmax 8..14.
//
// At these twojmax the sums of a sample fill the registers, one CTA of twojmax + 1 warps owns an SM, and everything in front of
// the accumulation -- claiming a tile, four dependent global loads for its candidates, distance tests, the pair geometry (a
// square root, two divisions, three trigonometric values per pair) -- is latency-bound work between barriers during which the
// FP64 pipe idles: about a third of the kernel.  Here one more warp, the PRODUCER (lane = grid point), prepares the neighbor
// queue of the NEXT tile while the twojmax + 1 CONSUMER warps (warp = sample point, as before) accumulate and transform the
// current one:
//
//   producer   claim tile -> candidates -> distance tests -> pair geometry -> geo[buf][entry][c, ar, ai, br, bi][lane]   -> full[buf]
//   consumers  per pass (a group of whole chains sized to the registers, pipe_klim):
//              full[buf] -> sums of the pass's columns over the queue -> empty[buf] -> S -> inverse DFT of those columns
//
// Two queue buffers (mbarriers full / empty, the usual parities), consumer-only named barriers around the uses of S.  The
// inverse DFT runs pass by pass so that S holds the columns of one pass only: S (113 KB at twojmax 10) and two queues of
// pipe_cap entries per point (2 x 51 KB) fit the 227 KB of an SM.  A window takes up to 64 candidates and ends early where a
// point would get more neighbors than a queue holds.  A tile of one window stays in its buffer for every pass; a tile of
// several windows is sent once per pass -- from the second pass on out of global memory (ChunkBuffers::ui_spill), where the
// producer kept the geometry of the first pass.  Above twojmax 10 U_tot is written half tile by half tile (the layout the
// half-tile contraction kernels read).  The arithmetic of a sample is that of compute_ui_dft_kernel (dft_accumulate); the
// summation order is fixed, results are bit-reproducible.  Below twojmax 8 the one producer warp cannot feed the consumers
// (measured), so compute_ui_dft_kernel stays there.
#pragma once
#include "snap_ui_dft.cuh"
#include "snap_zi.cuh"

namespace mala {

constexpr int kPipeWin = 64;      // candidates per window of distance tests (hit masks are 64 bits)
constexpr int kPipeMaxTasks = 6;  // pieces of columns one warp transforms per pass
constexpr int kPipeMaxPass = 5;

// entries of a queue buffer per grid point (a window is cut short where a point would get more)
constexpr int pipe_cap(int tj) { return tj >= 14 ? 32 : 40; }
// doubles of one window kept in global memory for the later passes of a tile: its queue buffer, then the 32 entry counts
constexpr int pipe_spill_record(int tj) { return pipe_cap(tj) * 5 * 32 + 32; }
// columns whose sums a thread keeps in registers during one pass: whole chains (all n of one mb), as many as fit
constexpr int pipe_klim(int tj) { return tj <= 10 ? 20 : (tj == 11 ? 18 : 16); }
// first chain of pass p (p = number of passes: one past the last chain)
constexpr int pipe_pass_mb(int tj, int p) {
    int mb = 0;
    for (int i = 0; i < p; i++) {
        int cols = 0;
        while (mb <= tj / 2 && (cols == 0 || cols + (tj - 2 * mb + 1) <= pipe_klim(tj))) { cols += tj - 2 * mb + 1; mb++; }
    }
    return mb;
}
constexpr int pipe_npass(int tj) {
    int p = 0;
    while (pipe_pass_mb(tj, p) <= tj / 2) p++;
    return p;
}
constexpr int pipe_pass_col(int tj, int p) { return dft_index(tj, pipe_pass_mb(tj, p), pipe_pass_mb(tj, p)); }   // first column of pass p
constexpr int pipe_kmax(int tj) {
    int k = 0;
    for (int p = 0; p < pipe_npass(tj); p++)
        if (pipe_pass_col(tj, p + 1) - pipe_pass_col(tj, p) > k) k = pipe_pass_col(tj, p + 1) - pipe_pass_col(tj, p);
    return k;
}

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
// dst points at this lane's word of element 0 of the tile (ESTRIDE words per element: 32, or 16 in the half-tile layout).
template <int TJ, int ESTRIDE>
__device__ __forceinline__ void pipe_dft(const double2 *S, const PipeTask *tasks, const int ntasks, const int lane, const double2 *s_tw,
                                         double2 *dst, const double2 *norm) {
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
            const double2 nrm = norm[e];   // binomial normalisation / NW, self term of the diagonal elements
            dst[(size_t)e * ESTRIDE] = make_double2(fma(sr, nrm.x, nrm.y), si * nrm.x);
        }
    }
}

// most pieces a warp gets when the coefficients of a pass's columns are cut into twojmax + 1 runs of equal length (the deal
// of the kernel's prologue, replayed at compile time)
constexpr int pipe_max_tasks(int tj) {
    int worst = 0;
    for (int pass = 0; pass < pipe_npass(tj); pass++) {
        const int mb0 = pipe_pass_mb(tj, pass), mb1 = pipe_pass_mb(tj, pass + 1), nw = tj + 1;
        int total = 0;
        for (int mb = mb0; mb < mb1; mb++)
            for (int n = mb; n <= tj - mb; n++) total += mb + n + 1;
        const int target = (total + nw - 1) / nw;
        int room = target, count = 0;
        for (int mb = mb0; mb < mb1; mb++)
            for (int n = mb; n <= tj - mb; n++) {
                int k = 0;
                while (k <= mb + n) {
                    const int take = room < mb + n + 1 - k ? room : mb + n + 1 - k;
                    count++;
                    if (count > worst) worst = count;
                    k += take; room -= take;
                    if (room == 0) { room = target; count = 0; }
                }
            }
    }
    return worst;
}

// what the consumer warps share between the passes of a tile
template <int TJ>
struct PipeCtx {
    double2 *S;                 // [kmax][NW][32]
    const double *geo;          // [2][cap][5][32]
    uint64_t *full, *empty;     // [2] each
    const int (*cnt)[32];       // [2][32]
    const int (*meta)[2];       // [2]{slot, last window of its round}
    const PipeTask (*task)[TJ + 1][kPipeMaxTasks];
    const int (*ntask)[TJ + 1];
    const double2 *tw, *norm;
    double2 *dst;               // this lane's word of element 0 of the tile
    double xsr, xsi;
    uint32_t it;                // buffers taken so far
    int buf, lane, warp;
    bool single;                // the tile came in one window: its buffer serves every pass
};

// pass P of a tile and the passes behind it: sums of chains pipe_pass_mb(P) <= mb < pipe_pass_mb(P + 1) over every window,
// then those columns through S and the inverse DFT
template <int TJ, int P>
__device__ __forceinline__ void pipe_passes(PipeCtx<TJ> &c) {
    if constexpr (P < pipe_npass(TJ)) {
        constexpr int NW = TJ + 1, NJM = dft_njm(TJ), GEO = pipe_cap(TJ) * 5 * 32;
        constexpr int K = pipe_pass_col(TJ, P + 1) - pipe_pass_col(TJ, P);
        constexpr bool LAST = (P + 1 == pipe_npass(TJ));
        {
            double accr[NJM], acci[NJM];   // K of them in use
#pragma unroll
            for (int k = 0; k < K; k++) { accr[k] = 0.0; acci[k] = 0.0; }
            for (bool first = true;; first = false) {
                if (!(first && (P == 0 || c.single))) {   // the first window of a tile is taken by the caller; a single one stays
                    c.buf = c.it & 1;
                    mbar_wait(&c.full[c.buf], (c.it >> 1) & 1);
                }
                dft_accumulate<TJ, pipe_pass_mb(TJ, P), pipe_pass_mb(TJ, P + 1)>(c.geo + (size_t)c.buf * GEO, c.lane, c.cnt[c.buf][c.lane], c.xsr,
                                                                                  c.xsi, accr, acci);
                if (c.single && !LAST) break;
                const bool last = c.meta[c.buf][1] != 0;
                __syncwarp();
                if (c.lane == 0) mbar_arrive(&c.empty[c.buf]);
                c.it++;
                if (last) break;
            }
            consumer_barrier<NW * 32>();   // everybody is done with the inverse DFT of the previous pass: S is free
#pragma unroll
            for (int k = 0; k < K; k++) c.S[((size_t)k * NW + c.warp) * 32 + c.lane] = make_double2(accr[k], acci[k]);
        }
        consumer_barrier<NW * 32>();
        pipe_dft<TJ, (TJ > kFullTileTwoJ ? 16 : 32)>(c.S, c.task[P][c.warp], c.ntask[P][c.warp], c.lane, c.tw, c.dst, c.norm);
        pipe_passes<TJ, P + 1>(c);
    }
}

template <int TJ>
__global__ void __launch_bounds__((TJ + 2) * 32, 1)
compute_ui_pipe_kernel(GridGeom g, SnapConst sc, DeviceTables tb, ChunkBuffers cb) {
    constexpr int NW = TJ + 1;          // consumer warps = sample points; warp NW is the producer
    constexpr int nelem = uhalf_size(TJ);
    constexpr int NPASS = pipe_npass(TJ), KMAX = pipe_kmax(TJ), CAP = pipe_cap(TJ);
    constexpr int GEO = CAP * 5 * 32;   // doubles per queue buffer
    constexpr bool HALF = TJ > kFullTileTwoJ;   // U_tot is stored half tile by half tile
    static_assert(NPASS <= kPipeMaxPass && pipe_max_tasks(TJ) <= kPipeMaxTasks, "pass tables");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *S = reinterpret_cast<double2 *>(smem_raw);                       // [KMAX][NW][32]
    double *geo = reinterpret_cast<double *>(S + (size_t)KMAX * NW * 32);     // [2][CAP][5][32]
    double *crec = geo + 2 * GEO;                                             // [kPipeWin][6], the producer's
    __shared__ uint64_t full[2], empty[2];
    __shared__ int s_cnt[2][32];          // entries of every lane's queue in the buffer
    __shared__ int s_meta[2][2];          // slot of the tile the buffer belongs to (-1: no more tiles); last window of its round
    __shared__ double2 s_tw[NW * NW];     // [k][s] = x_s^(-k) = e^{-2 pi i s k / NW}
    __shared__ double2 s_norm[nelem];     // {unorm / NW, wself on the diagonal}
    __shared__ PipeTask s_task[NPASS][NW][kPipeMaxTasks];
    __shared__ int s_ntask[NPASS][NW];
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
        for (int pass = 0; pass < NPASS; pass++) {
            const int mb0 = pipe_pass_mb(TJ, pass), mb1 = pipe_pass_mb(TJ, pass + 1);
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
                        s_task[pass][w][s_ntask[pass][w]++] = t;   // at most pipe_max_tasks(TJ) per warp
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
        constexpr int REC = pipe_spill_record(TJ);
        const int wmax = cb.ui_spill ? cb.ui_spill_windows : 0;
        double *spill = wmax ? cb.ui_spill + (size_t)blockIdx.x * (size_t)wmax * REC : nullptr;
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
            int rounds = 1;   // a tile of several windows is sent once per pass
            int nkept = 0, wbase_kept = 0;   // windows of this tile kept in global memory, the candidate they end at
            bool kept_all = false;
            for (int round = 0; round < rounds; round++) {
                int wbase = 0, win = 0;
                bool last = false;
                if (round > 0 && nkept > 0) {
                    // later passes: the windows kept in round 0 come back from global memory (each lane reads what it wrote)
                    for (; win < nkept; win++, it++) {
                        const double *src = spill + (size_t)win * REC;
                        const int cnt = reinterpret_cast<const int *>(src + GEO)[lane];
                        const int buf = it & 1;
                        mbar_wait(&empty[buf], ((it >> 1) & 1) ^ 1);
                        double *gq = geo + (size_t)buf * GEO + lane;
                        const double *sq = src + lane;
                        for (int e = 0; e < cnt; e++, gq += 5 * 32, sq += 5 * 32) {
                            const double c = sq[0], ar = sq[32], ai = sq[64], br = sq[96], bi = sq[128];
                            gq[0] = c; gq[32] = ar; gq[64] = ai; gq[96] = br; gq[128] = bi;
                        }
                        s_cnt[buf][lane] = cnt;
                        last = kept_all && win == nkept - 1;
                        if (lane == 0) { s_meta[buf][0] = slot; s_meta[buf][1] = last ? 1 : 0; }
                        mbar_arrive(&full[buf]);
                    }
                    if (kept_all) continue;
                    wbase = wbase_kept;
                }
                do {
                    int nw = min(kPipeWin, nc - wbase);
                    __syncwarp();   // the geometry of the previous window has read crec
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
                    // the window ends where a point would get more entries than a buffer holds
                    while (__reduce_max_sync(0xffffffffu, (unsigned)__popcll(hits)) > (unsigned)CAP) {
                        nw--;
                        hits &= (1ull << nw) - 1ull;
                    }
                    last = wbase + nw >= nc;
                    if (round == 0 && wbase == 0 && !last) rounds = NPASS;
                    const int buf = it & 1;
                    mbar_wait(&empty[buf], ((it >> 1) & 1) ^ 1);   // the consumers are done with this buffer
                    double *gq = geo + (size_t)buf * GEO + lane;
                    const bool keep = round == 0 && rounds > 1 && win < wmax;
                    double *kq = keep ? spill + (size_t)win * REC + lane : gq;
                    for (unsigned long long r = hits; r != 0ull; r &= r - 1ull, gq += 5 * 32, kq += 5 * 32) {
                        const double *q = crec + (__ffsll((long long)r) - 1) * 6;
                        const double dx = q[0] - px, dy = q[1] - py, dz = q[2] - pz;
                        const double r2 = dx * dx + dy * dy + dz * dz;
                        double c, ar, ai, br, bi;
                        pair_geometry(dx, dy, dz, r2, q[3], q[4], sc.rfac0, sc.rmin0, c, ar, ai, br, bi);
                        gq[0] = c; gq[32] = ar; gq[64] = ai; gq[96] = br; gq[128] = bi;
                        if (keep) { kq[0] = c; kq[32] = ar; kq[64] = ai; kq[96] = br; kq[128] = bi; }
                    }
                    s_cnt[buf][lane] = __popcll(hits);
                    if (keep) {
                        reinterpret_cast<int *>(spill + (size_t)win * REC + GEO)[lane] = __popcll(hits);
                        nkept = win + 1; wbase_kept = wbase + nw; kept_all = last;
                    }
                    if (lane == 0) { s_meta[buf][0] = slot; s_meta[buf][1] = last ? 1 : 0; }
                    mbar_arrive(&full[buf]);
                    it++;
                    win++;
                    wbase += nw;
                } while (!last);
            }
        }
        return;
    }

    // -------------------------------------------------------------------- consumers: warp = sample point, lane = grid point
    PipeCtx<TJ> c;
    c.S = S; c.geo = geo; c.full = full; c.empty = empty; c.cnt = s_cnt; c.meta = s_meta; c.task = s_task; c.ntask = s_ntask;
    c.tw = s_tw; c.norm = s_norm; c.lane = lane; c.warp = warp; c.it = 0;
    {   // this warp's sample point x_s = e^{2 pi i s / NW}
        double sn, cs;
        sincospi(2.0 * (double)warp / (double)NW, &sn, &cs);
        c.xsr = cs; c.xsi = sn;
    }
    for (;;) {
        c.buf = c.it & 1;
        mbar_wait(&full[c.buf], (c.it >> 1) & 1);
        const int slot = s_meta[c.buf][0];
        if (slot < 0) break;
        c.single = s_meta[c.buf][1] != 0;
        c.dst = HALF ? cb.utot + ((size_t)(2 * slot + (lane >> 4)) * nelem) * 16 + (lane & 15) : cb.utot + (size_t)slot * nelem * 32 + lane;
        pipe_passes<TJ, 0>(c);
    }
}

template <int TJ>
inline size_t compute_ui_pipe_smem_bytes() {
    return (size_t)pipe_kmax(TJ) * (TJ + 1) * 32 * sizeof(double2) + (size_t)2 * pipe_cap(TJ) * 5 * 32 * sizeof(double) +
           (size_t)kPipeWin * 6 * sizeof(double) + 16;
}

}  // namespace mala
