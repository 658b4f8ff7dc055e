// mala_snap.cu -- C ABI of libmala_snap.so and the host planner (include/mala_snap.h documents every call).
//
// Host side per call: validate, wrap atoms, enumerate the periodic images that can reach the slab ("ghosts"),
// sort them into a Cartesian cell list, choose the tile shape and the chunking, then enqueue per chunk
//     tile_bin_kernel -> compute_ui_kernel -> compute_zi_bi_*_kernel
// on the caller's stream.  No step of the path runs on the CPU and there is no fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/mala_snap.h"
#include "snap_common.cuh"
#include "snap_internal.h"
#include "snap_tables.h"
#include "snap_ui.cuh"
#include "snap_ui_dft.cuh"
#include "snap_ui_pipe.cuh"
#include "snap_zi.cuh"
#include "snap_zi_coop.cuh"
#include "snap_zi_diag.cuh"
#include "snap_zi_block.cuh"
#include "snap_gauss.cuh"
#include "snap_force.cuh"
#include "snap_yi_block.cuh"
#include "snap_yi_fix.cuh"
#include "snap_dedr_dft.cuh"

using namespace mala;

static thread_local std::string g_last_error;

static int fail(int code, const std::string &msg) {
    g_last_error = msg;
    return code;
}

namespace mala {
int set_error(int code, const std::string &msg) { return fail(code, msg); }
}  // namespace mala

// Scratch of mala_gaussian_grid_static, the entry point that allocates nothing: ghost atoms, cell list, counters and the
// candidate lists of tile_bin_kernel live here instead of in the handle's stream-ordered workspace.  Every GPU that loads the
// library holds these bytes until exit.  In host code the name is a stand-in, not a device address: mala_snap_create resolves
// it once per handle (= per device, with that device current) through cudaGetSymbolAddress.
constexpr size_t kStaticScratchBytes = (size_t)16 << 20;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

#define CUDA_TRY(call)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess) {                                                                    \
            const int code_ = (e_ == cudaErrorMemoryAllocation) ? MALA_SNAP_ENOMEM : MALA_SNAP_ECUDA; \
            return fail(code_, std::string(#call) + ": " + cudaGetErrorString(e_));                 \
        }                                                                                           \
    } while (0)

namespace {

// Device buffer that only grows.  Tables are allocated once at create time (plain cudaMalloc); the per-call workspace
// grows through the stream-ordered allocator on the caller's stream, so enlarging it inside an enqueue-only call neither
// synchronises the device nor pulls memory from under kernels that are still queued on that stream.
template <typename T>
struct DevBuf {
    T *p = nullptr;
    size_t cap = 0;  // elements
    bool pooled = false;
    int reserve(size_t n, cudaStream_t st = nullptr, bool stream_ordered = false) {
        if (n <= cap) return 0;
        release(st);
        size_t want = n + n / 4 + 16;
        pooled = stream_ordered;
        cudaError_t e = stream_ordered ? cudaMallocAsync((void **)&p, want * sizeof(T), st) : cudaMalloc((void **)&p, want * sizeof(T));
        if (e != cudaSuccess) {
            cudaGetLastError();
            want = n;
            e = stream_ordered ? cudaMallocAsync((void **)&p, want * sizeof(T), st) : cudaMalloc((void **)&p, want * sizeof(T));
        }
        if (e != cudaSuccess) {
            cudaGetLastError();
            p = nullptr;
            return -1;
        }
        cap = want;
        return 0;
    }
    void release(cudaStream_t st = nullptr) {
        if (p) {
            if (pooled) cudaFreeAsync(p, st);
            else cudaFree(p);
        }
        p = nullptr;
        cap = 0;
    }
};

}  // namespace

struct mala_snap {
    // parameters
    int twojmax = 0, ntypes = 0;
    double rcutfac = 0, rfac0 = 0, rmin0 = 0, wself = 0;
    std::vector<double> rcut, wj;
    double rcutmax = 0;
    SnapTables tab;
    SnapConst sc{};
    int device = 0, num_sms = 0;
    unsigned char *static_scratch = nullptr;   // device address of g_static_scratch on this handle's device
    // options
    int zi_impl = 0;
    int ui_impl = 0;   // 0 automatic (sampling kernel for twojmax 1..10, pipelined from 8 up), 1 column kernel, 2 sampling kernel, 3 pipelined sampling kernel
    // tables of the anti-diagonal kernels (per handle, global memory)
    std::vector<double> k_dcg;
    std::vector<DiagTriple> k_dtriple;
    std::vector<unsigned short> k_dsched, k_ditems;
    DevBuf<double> d_dcg;
    DevBuf<DiagTriple> d_dtriple;
    DevBuf<unsigned short> d_dsched, d_ditems;
    // tables of the block kernel (snap_zi_block.cuh)
    DevBuf<int4> d_bstream;
    DevBuf<int> d_bwrange, d_btslot;
    int blk_nslots = 0;
    bool blk_ready = false;
    BlkTables blk_tables() const {
        BlkTables t;
        t.stream = d_bstream.p; t.wrange = d_bwrange.p; t.tslot = d_btslot.p; t.nslots = blk_nslots;
        return t;
    }
    long long workspace_mb = 4096;
    long long host_chunk_mb = 256;
    // device tables
    DevBuf<int> d_triples, d_udiag, d_order;
    DevBuf<double> d_cg, d_unorm, d_rcut, d_w, d_bconst;
    // per-call buffers
    // ghosts + cell list are double-buffered (set = call parity) and uploaded on a private stream, so that a
    // call never waits on the host for the kernels of the previous call
    DevBuf<Ghost> d_ghosts[2];
    DevBuf<int> d_cell_start[2];
    cudaStream_t upload_stream = nullptr;
    cudaEvent_t ev_upload = nullptr, ev_call_done[2] = {nullptr, nullptr};
    bool call_done_valid[2] = {false, false};
    unsigned long long ncalls = 0;
    int cur = 0;  // buffer set of the current call
    std::vector<int> h_cell_start;
    DevBuf<int> d_cand, d_ncand, d_active, d_counters;
    DevBuf<double> d_uispill;   // compute_ui_pipe_kernel: window geometry of multi-window tiles, per CTA
    DevBuf<int> d_status;          // kStatus* bits raised by the kernels; never cleared by a chunk
    int *h_status = nullptr;       // pinned mirror, refreshed at the end of every call
    int sticky_status = 0;         // bits seen so far (a raised bit makes every later call fail)
    int cand_cap_limit = 0;        // test hook: clamp the candidate capacity (0 = off) to provoke the overflow path
    DevBuf<double2> d_utot;
    DevBuf<double> d_bstage;       // fused network: descriptors of one chunk, [tile][32][ncomp]
    // row f3 (force adjoint): tables of compute_yi and the Y workspace
    DevBuf<YTerm> d_yterms;
    DevBuf<int> d_ylevel, d_yorder;
    DevBuf<double> d_ycg, d_yweight;
    DevBuf<double2> d_ytot;
    DevBuf<int4> d_ybstream;          // compute_yi on the block machinery (snap_yi_block.cuh)
    DevBuf<int> d_ybwrange, d_ybpass, d_ybmirror;
    int yb_npasses = 0, yb_yacc = 0;
    int yi_impl = 0;                  // 0 automatic (2), 1 table-driven kernel, 2 block kernel with Y in fixed point, 3 block kernel with fp64 atomics
    int dedr_impl = 0;                // 0 automatic (sampling kernel for twojmax 1..10), 1 column kernel
    YBlkTables yblk_tables() const {
        YBlkTables t;
        t.stream = d_ybstream.p; t.wrange = d_ybwrange.p; t.pass_elem = d_ybpass.p; t.yweight = d_yweight.p; t.mirror = d_ybmirror.p;
        t.npasses = yb_npasses; t.yacc_elems = yb_yacc;
        return t;
    }
    bool force_ready = false;
    ForceTables force_tables() const {
        ForceTables f;
        f.terms = d_yterms.p; f.level_begin = d_ylevel.p; f.cg = d_ycg.p; f.eorder = d_yorder.p; f.yweight = d_yweight.p;
        return f;
    }
    DevBuf<double> d_stage[2];
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_done[2] = {nullptr, nullptr}, ev_copied[2] = {nullptr, nullptr};
    // plan of the current call
    GridGeom geom{};
    long long total_tiles = 0;
    int cand_cap = 0;
    long long stats[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    // optional per-kernel timing ("timing" option): event pairs around every launch of the last call
    bool timing = false;
    struct Span { int kind; cudaEvent_t a, b; };
    std::vector<Span> spans;           // recorded during the last call
    std::vector<cudaEvent_t> ev_pool;  // reusable timing events
    size_t ev_used = 0;

    DeviceTables tables() const {
        DeviceTables t;
        t.triples = d_triples.p; t.cg = d_cg.p; t.unorm = d_unorm.p; t.udiag = d_udiag.p; t.order = d_order.p;
        t.type_rcut = d_rcut.p; t.type_w = d_w.p; t.bconst = d_bconst.p;
        return t;
    }
    DiagTables diag_tables() const {
        DiagTables t;
        t.cg2 = reinterpret_cast<const double2 *>(d_dcg.p); t.triple = d_dtriple.p; t.sched = d_dsched.p; t.items = d_ditems.p;
        return t;
    }
    // twojmax above kFullTileTwoJ: U_tot of 32 points does not fit one SM's shared memory; half-tile layout and kernel
    bool half_tiles() const { return twojmax > kFullTileTwoJ; }
    // 0 = automatic: the block kernel (on half tiles above twojmax = 10)
    bool use_block() const { return (zi_impl == 4 || zi_impl == 0) && blk_ready; }
    bool use_ui_pipe() const { return twojmax >= 8 && (ui_impl == 0 || ui_impl == 3); }
    bool use_ui_dft() const { return (twojmax >= 1 && twojmax <= kFullTileTwoJ && ui_impl != 1) || use_ui_pipe(); }
    bool use_spec() const { return zi_impl == 2; }
    bool use_diag() const { return zi_impl == 3 || (zi_impl == 0 && !use_block()); }
};

namespace {


template <typename T>
int upload(DevBuf<T> &b, const std::vector<T> &v) {
    if (b.reserve(std::max<size_t>(v.size(), 1))) return fail(MALA_SNAP_ENOMEM, "cudaMalloc (table) failed");
    if (!v.empty()) CUDA_TRY(cudaMemcpy(b.p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
    return 0;
}

int set_kernel_attributes(mala_snap *h) {
    const int ui_smem = (int)compute_ui_smem_bytes(kFullTileTwoJ);
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_kernel<kFullTileTwoJ, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, ui_smem));
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_kernel<kFullTileTwoJ, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, ui_smem));
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_kernel<kMaxTwoJ, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)compute_ui_smem_bytes(kMaxTwoJ)));
#define MALA_DFT_ATTR(TJ) \
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_dft_kernel<TJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_ui_dft_smem_bytes<TJ>()));
    MALA_DFT_ATTR(1) MALA_DFT_ATTR(2) MALA_DFT_ATTR(3) MALA_DFT_ATTR(4) MALA_DFT_ATTR(5)
    MALA_DFT_ATTR(6) MALA_DFT_ATTR(7) MALA_DFT_ATTR(8) MALA_DFT_ATTR(9) MALA_DFT_ATTR(10)
#undef MALA_DFT_ATTR
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_pipe_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_ui_pipe_smem_bytes<8>()));
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_pipe_kernel<9>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_ui_pipe_smem_bytes<9>()));
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_pipe_kernel<10>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_ui_pipe_smem_bytes<10>()));
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_pipe_kernel<11>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_ui_pipe_smem_bytes<11>()));
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_pipe_kernel<12>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_ui_pipe_smem_bytes<12>()));
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_pipe_kernel<13>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_ui_pipe_smem_bytes<13>()));
    CUDA_TRY(cudaFuncSetAttribute(compute_ui_pipe_kernel<14>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_ui_pipe_smem_bytes<14>()));
    const int zi_smem = (int)compute_zi_smem_bytes(uhalf_size(kFullTileTwoJ), triple_count(kFullTileTwoJ));
    CUDA_TRY(cudaFuncSetAttribute(compute_zi_bi_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, zi_smem));
    CUDA_TRY(cudaFuncSetAttribute(compute_zi_bi_coop_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_zi_coop_smem_bytes()));
    CUDA_TRY(cudaFuncSetAttribute(compute_zi_bi_diag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)compute_zi_diag_smem_bytes(uhalf_size(kFullTileTwoJ), triple_count(kFullTileTwoJ))));
    CUDA_TRY(cudaFuncSetAttribute(compute_zi_bi_diag_half_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)compute_zi_diag_half_smem_bytes(uhalf_size(kMaxTwoJ), triple_count(kMaxTwoJ))));
    CUDA_TRY(cudaFuncSetAttribute(compute_zi_bi_block_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)compute_zi_block_smem_bytes(uhalf_size(kFullTileTwoJ), triple_count(kFullTileTwoJ), kBlkMaxSlots)));
    CUDA_TRY(cudaFuncSetAttribute(compute_zi_bi_block_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)compute_zi_block_smem_bytes(uhalf_size(kFullTileTwoJ), triple_count(kFullTileTwoJ), kBlkMaxSlots)));
    CUDA_TRY(cudaFuncSetAttribute(compute_zi_bi_block_half_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kBlkHalfSmemMax));
    (void)h;
    return 0;
}

// kernel classes reported by mala_snap_kernel_times
enum { kKindBin = 0, kKindUi = 1, kKindZi = 2, kKindOther = 3 };

cudaEvent_t timing_event(mala_snap *h) {
    if (h->ev_used == h->ev_pool.size()) {
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        h->ev_pool.push_back(e);
    }
    return h->ev_pool[h->ev_used++];
}

// RAII bracket: records an event pair around the launches made while it is alive (no-op unless timing is on)
struct TimedSpan {
    mala_snap *h; cudaStream_t st; cudaEvent_t a = nullptr, b = nullptr; int kind;
    TimedSpan(mala_snap *h_, cudaStream_t st_, int kind_) : h(h_), st(st_), kind(kind_) {
        if (!h->timing) return;
        a = timing_event(h); b = timing_event(h);
        if (a && b) cudaEventRecord(a, st);
    }
    ~TimedSpan() {
        if (!h->timing || !a || !b) return;
        cudaEventRecord(b, st);
        h->spans.push_back({kind, a, b});
    }
};

// processing order (J1 descending, then cost), padded CG blocks and the per-warp item schedule of the diag kernel
int build_diag_schedule(mala_snap *h) {
    const SnapTables &T = h->tab;
    const int nt = T.ntriples;
    const int NWD = h->half_tiles() ? kDiagHalfWarps : kDiagWarps;  // warps of the kernel this handle will launch
    // CG blocks with an even row stride (16-byte rows: two coefficients per uniform load)
    std::vector<int> cgoff(nt, 0);
    h->k_dcg.clear();
    for (int t = 0; t < nt; t++) {
        const int J1 = T.triples[4 * t], J2 = T.triples[4 * t + 1], src = T.triples[4 * t + 3], S = diag_stride(J1);
        cgoff[t] = (int)h->k_dcg.size();
        for (int m2 = 0; m2 <= J2; m2++)
            for (int m1 = 0; m1 < S; m1++) h->k_dcg.push_back(m1 <= J1 ? T.cg[src + m2 * (J1 + 1) + m1] : 0.0);
    }
    h->k_dcg.resize(h->k_dcg.size() + 16, 0.0);
    // cost model in issue cycles (an FP64 instruction holds the issue port for two cycles, anything else for one):
    // one row of an item = 6 (J1+1) FP64 + (J1+1) constant loads + ~4; an item adds its x loads and set-up; every
    // column segment a warp starts pays for zeroing and folding the 2 J1 + 1 accumulators; every call ~120.
    std::vector<double> tcost(nt, 0.0), segcost(nt, 0.0);
    std::vector<std::vector<double>> icost(nt);
    std::vector<std::vector<int>> icol(nt);
    const double kCallCost = 120.0;
    for (int t = 0; t < nt; t++) {
        const int J1 = T.triples[4 * t], J2 = T.triples[4 * t + 1], J = T.triples[4 * t + 2];
        segcost[t] = 7.0 * (2 * J1 + 1) + 40.0;
        for (int mb = 0; mb <= J / 2; mb++) {
            int lo, hi;
            diag_item_range(J1, J2, J, mb, lo, hi);
            for (int i = lo; i <= hi; i++) {
                icost[t].push_back((J2 + 1) * (13.0 * (J1 + 1) + 4.0) + 4.0 * (J1 + 1) + 60.0);
                icol[t].push_back(mb);
            }
            if (hi >= lo) tcost[t] += segcost[t];
        }
        for (double c : icost[t]) tcost[t] += c;
    }
    // item descriptors (16-point kernel): item -> last-of-column flag | mb << 8 | mb1, items numbered column by column
    std::vector<int> itemoff(nt, 0);
    h->k_ditems.clear();
    for (int t = 0; t < nt; t++) {
        const int J1 = T.triples[4 * t], J2 = T.triples[4 * t + 1], J = T.triples[4 * t + 2];
        itemoff[t] = (int)h->k_ditems.size();
        for (int mb = 0; mb <= J / 2; mb++) {
            int lo, hi;
            diag_item_range(J1, J2, J, mb, lo, hi);
            for (int i = lo; i <= hi; i++)
                h->k_ditems.push_back((unsigned short)((i == hi ? 0x8000u : 0u) | ((unsigned)mb << 8) | (unsigned)i));
        }
    }
    h->k_ditems.push_back(0);
    std::vector<int> order(nt);
    for (int i = 0; i < nt; i++) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
        if (T.triples[4 * a] != T.triples[4 * b]) return T.triples[4 * a] > T.triples[4 * b];
        return tcost[a] > tcost[b];
    });
    h->k_dtriple.assign(nt, DiagTriple{});
    h->k_dsched.assign((size_t)nt * NWD * 2, 0);
    const int teams = (NWD % kDiagTeams == 0) ? kDiagTeams : 1;
    const int tw = NWD / teams;
    // balanced per reduction group, like the per-triple kernel: team split by exhaustive search, per-group running loads
    std::vector<int> pos_team(nt, 0);
    for (int g0 = 0; g0 < nt; g0 += kDiagGroup) {
        const int gn = std::min(kDiagGroup, nt - g0);
        if (teams == 2 && gn <= 16) {
            double total = 0.0, best = 1e300;
            for (int i = 0; i < gn; i++) total += tcost[order[g0 + i]];
            unsigned best_mask = 0;
            for (unsigned mask = 0; mask < (1u << gn); mask++) {
                double a = 0.0;
                for (int i = 0; i < gn; i++)
                    if (mask >> i & 1u) a += tcost[order[g0 + i]];
                if (std::fabs(2.0 * a - total) < best) { best = std::fabs(2.0 * a - total); best_mask = mask; }
            }
            for (int i = 0; i < gn; i++) pos_team[g0 + i] = (int)(best_mask >> i & 1u);
        } else {
            std::vector<double> tl(teams, 0.0);
            for (int i = 0; i < gn; i++) {
                int team = 0;
                for (int k = 1; k < teams; k++)
                    if (tl[k] < tl[team]) team = k;
                tl[team] += tcost[order[g0 + i]];
                pos_team[g0 + i] = team;
            }
        }
        std::vector<double> load(NWD, 0.0);
        for (int pos = g0; pos < g0 + gn; pos++) {
            const int t = order[pos], team = pos_team[pos];
            DiagTriple &d = h->k_dtriple[pos];
            d.J1 = (short)T.triples[4 * t]; d.J2 = (short)T.triples[4 * t + 1]; d.J = (short)T.triples[4 * t + 2];
            d.index = (short)t; d.cgoff = cgoff[t]; d.itemoff = itemoff[t];
            const std::vector<double> &cost = icost[t];
            const int n = (int)cost.size();
            double sum_load = tcost[t] + 0.5 * tw * kCallCost;
            for (int k = 0; k < tw; k++) sum_load += load[team * tw + k];
            const double target = sum_load / tw;
            int i = 0;
            for (int k = 0; k < tw; k++) {
                const int w = team * tw + k;
                const int begin = i;
                double acc = 0.0;
                const bool last = (k == tw - 1);
                const double want = target - load[w];
                while (i < n) {
                    const bool newseg = (i == begin) || (icol[t][i] != icol[t][i - 1]);
                    const double c = cost[i] + (newseg ? segcost[t] : 0.0) + (i == begin ? kCallCost : 0.0);
                    if (!last && acc + 0.5 * c > want) break;
                    acc += c;
                    i++;
                }
                load[w] += acc;
                h->k_dsched[((size_t)pos * NWD + w) * 2] = (unsigned short)begin;
                h->k_dsched[((size_t)pos * NWD + w) * 2 + 1] = (unsigned short)i;
            }
        }
    }
    int rc = 0;
    if ((rc = upload(h->d_dcg, h->k_dcg))) return rc;
    if ((rc = upload(h->d_dtriple, h->k_dtriple))) return rc;
    if ((rc = upload(h->d_dsched, h->k_dsched))) return rc;
    if ((rc = upload(h->d_ditems, h->k_ditems))) return rc;
    return 0;
}

// Tables of the block kernel (snap_zi_block.cuh): the units (blocks of the (ma1, ma2) rectangle of a triple and column, with
// their items and packed coefficients), their deal to the warps, one record stream per warp and the partial-sum slots.
int build_block_schedule(mala_snap *h) {
    const SnapTables &T = h->tab;
    const int nt = T.ntriples, NW = kBlkWarps;
    const bool half = h->half_tiles();   // 16-point items: the two half-warps take the items of a unit alternately
    const int RB = (half ? 16 : 32) * (int)sizeof(double2);
    struct HostItem { int ex, ey; bool fx, fy; int mb1, mb2; double w; };   // element index of row 0 of each column as it is read
    struct HostUnit { int triple, items_first, nitems, a0, b0, bx, by, ub_elem; std::vector<double> coef; double cost; };
    std::vector<HostItem> items;
    std::vector<std::vector<HostUnit>> tunits(nt);
    std::vector<double> tcost(nt, 0.0);
    auto chunks = [](int len, int mx) {
        std::vector<std::pair<int, int>> out;
        const int k = (len + mx - 1) / mx, base = len / k, rem = len % k;
        int s = 0;
        for (int i = 0; i < k; i++) { const int c = base + (i < rem ? 1 : 0); out.push_back({s, c}); s += c; }
        return out;
    };
    for (int t = 0; t < nt; t++) {
        const int J1 = T.triples[4 * t], J2 = T.triples[4 * t + 1], J = T.triples[4 * t + 2], cg0 = T.triples[4 * t + 3];
        const int sh = (J1 + J2 - J) / 2;
        for (int mb = 0; mb <= J / 2; mb++) {
            int lo, hi;
            diag_item_range(J1, J2, J, mb, lo, hi);
            if (hi < lo) continue;
            const bool mid = (J % 2 == 0) && (mb == J / 2);
            const int items_first = (int)items.size();
            for (int mb1 = lo; mb1 <= hi; mb1++) {
                const int mb2 = mb + sh - mb1;
                double w = T.cg[cg0 + mb2 * (J1 + 1) + mb1];
                if (J == J1 && J1 == J2) {   // one item per S3 x Z2 class (diag_weight3)
                    const int mu1 = mb1 - J / 2, mu3 = J / 2 - mb, mu2 = -mu1 - mu3;
                    const int perms = (mu1 == mu2 && mu2 == mu3) ? 1 : ((mu1 == mu2 || mu2 == mu3) ? 3 : 6);
                    w *= (double)(perms * ((mu2 == 0) ? 1 : 2)) / (mid ? 1.0 : 2.0);
                } else if (J1 == J2 && mb1 != mb2) w += w;
                if (J == J1 && J1 != J2 && mb1 != mb && mb1 != J - mb) w += w;
                HostItem it;
                it.fx = mb1 > J1 / 2; it.fy = mb2 > J2 / 2; it.mb1 = mb1; it.mb2 = mb2; it.w = w;
                it.ex = it.fx ? uhalf_off(J1) + (J1 - mb1) * (J1 + 1) + J1 : uhalf_off(J1) + mb1 * (J1 + 1);
                it.ey = it.fy ? uhalf_off(J2) + (J2 - mb2) * (J2 + 1) + J2 : uhalf_off(J2) + mb2 * (J2 + 1);
                items.push_back(it);
            }
            const int n = hi - lo + 1;
            // coefficient of (ma1, ma2): CG x weight of row ma in the fold (2; in the middle column 2 below the centre, 1 on it, 0 above)
            auto cf = [&](int m1, int m2) {
                const int ma = m1 + m2 - sh;
                if (ma < 0 || ma > J) return 0.0;
                const double wf = mid ? (ma < J / 2 ? 2.0 : (ma == J / 2 ? 1.0 : 0.0)) : 2.0;
                return wf * T.cg[cg0 + m2 * (J1 + 1) + m1];
            };
            for (auto cx : chunks(J1 + 1, kBlkBX))
                for (auto cy : chunks(J2 + 1, kBlkBY)) {
                    int a_lo = 1 << 30, a_hi = -1, b_lo = 1 << 30, b_hi = -1;   // bounding box of the non-zero coefficients
                    for (int a = cx.first; a < cx.first + cx.second; a++)
                        for (int b = cy.first; b < cy.first + cy.second; b++)
                            if (cf(a, b) != 0.0) { a_lo = std::min(a_lo, a); a_hi = std::max(a_hi, a); b_lo = std::min(b_lo, b); b_hi = std::max(b_hi, b); }
                    if (a_hi < 0) continue;
                    HostUnit hu;
                    hu.triple = t; hu.items_first = items_first; hu.nitems = n;
                    // pad to the smallest shape the kernel has a body for: shift the origin back where the column is long enough,
                    // else run past its end (those reads hit other finite words of the tile and meet zero coefficients)
                    int bx = a_hi - a_lo + 1, by = b_hi - b_lo + 1;
                    if (bx < kBlkBXMin) { a_lo = std::max(0, std::min(a_lo, J1 + 1 - kBlkBXMin)); bx = kBlkBXMin; }
                    if (by < kBlkBYMin) { b_lo = std::max(0, std::min(b_lo, J2 + 1 - kBlkBYMin)); by = kBlkBYMin; }
                    hu.a0 = a_lo; hu.b0 = b_lo; hu.bx = bx; hu.by = by;
                    hu.ub_elem = uhalf_off(J) + mb * (J + 1) + (a_lo + b_lo - sh);   // row of the first anti-diagonal (may lie before the column)
                    for (int d = 0; d <= hu.bx + hu.by - 2; d++)   // in the order the kernel consumes them (blk_coef_index)
                        for (int a = 0; a < hu.bx; a++) {
                            const int b = d - a;
                            if (b < 0 || b >= hu.by) continue;
                            hu.coef.push_back((a_lo + a >= cx.first && a_lo + a < cx.first + cx.second && b_lo + b >= cy.first && b_lo + b < cy.first + cy.second)
                                                  ? cf(a_lo + a, b_lo + b) : 0.0);
                        }
                    // issue cycles: an FP64 instruction holds the port for two, anything else for one
                    hu.cost = (half ? (n + 1) / 2 : n) * (2.0 * (4 * bx * by + 2 * by) + 3.0 * bx + 2.0 * by + 14.0) + 2.0 * (2 * bx * by + 2 * (bx + by - 1)) + 0.5 * bx * by +
                              bx + by + 2.0 * bx * by + 40.0;
                    tcost[t] += hu.cost;
                    tunits[t].push_back(std::move(hu));
                }
        }
    }
    // pieces: whole triples, the heaviest ones cut into parts of at most half a warp's share
    double total = 0.0;
    for (double c : tcost) total += c;
    const double share = total / NW;
    struct Piece { int triple, begin, end; double cost; };
    std::vector<Piece> pieces;
    for (int t = 0; t < nt; t++) {
        const int nu = (int)tunits[t].size();
        if (nu == 0) continue;
        const int parts = std::max(1, std::min(nu, (int)std::ceil(tcost[t] / (0.5 * share))));
        int i = 0;
        double run = 0.0;
        for (int k = 0; k < parts; k++) {
            const double want = tcost[t] * (k + 1) / parts;
            Piece pc{t, i, i, 0.0};
            while (i < nu && (k == parts - 1 || run + 0.5 * tunits[t][i].cost <= want)) { run += tunits[t][i].cost; pc.cost += tunits[t][i].cost; i++; }
            pc.end = i;
            if (pc.end > pc.begin) pieces.push_back(pc);
        }
    }
    std::stable_sort(pieces.begin(), pieces.end(), [](const Piece &a, const Piece &b) { return a.cost > b.cost; });
    std::vector<double> load(NW, 0.0);
    std::vector<int> piece_warp(pieces.size(), 0);
    for (size_t i = 0; i < pieces.size(); i++) {
        int w = 0;
        for (int k = 1; k < NW; k++)
            if (load[k] < load[w]) w = k;
        load[w] += pieces[i].cost;
        piece_warp[i] = w;
    }
    // slots: the pieces of a triple, in piece order; triples without work keep an empty range
    std::vector<int> tslot(nt + 1, 0), piece_slot(pieces.size(), 0);
    int nslots = 0;
    for (int t = 0; t < nt; t++) {
        tslot[t] = nslots;
        for (size_t i = 0; i < pieces.size(); i++)
            if (pieces[i].triple == t) piece_slot[i] = nslots++;
    }
    tslot[nt] = nslots;
    if (half ? compute_zi_block_half_smem_bytes(h->sc.nelem, nslots) > (size_t)kBlkHalfSmemMax : nslots > kBlkMaxSlots)
        return fail(MALA_SNAP_ECUDA, "internal: too many partial-sum slots");
    // one record stream per warp, units by decreasing shape (the order in which the kernel runs its shape loops)
    std::vector<int4> stream;
    std::vector<int> wrange((size_t)NW * (kBlkShapes + 2), 0);
    auto push_d2 = [&](double a, double b) {
        int4 v;
        std::memcpy(&v.x, &a, 8);
        std::memcpy(&v.z, &b, 8);
        stream.push_back(v);
    };
    for (int w = 0; w < NW; w++) {
        const size_t w0 = stream.size();
        wrange[(size_t)w * (kBlkShapes + 2) + kBlkShapes] = (int)w0;
        size_t last_header = 0;
        bool have_header = false;
        for (int bx = kBlkBX; bx >= 1; bx--)
            for (int by = kBlkBY; by >= 1; by--) {
                int count = 0;
                for (size_t i = 0; i < pieces.size(); i++) {
                    if (piece_warp[i] != w) continue;
                    for (int q = pieces[i].begin; q < pieces[i].end; q++) {
                        const HostUnit &u = tunits[pieces[i].triple][q];
                        if (u.bx != bx || u.by != by) continue;
                        count++;
                        // a unit must not straddle the end of the ring: the unit before it skips the words up to the boundary
                        const int nit = half ? (u.nitems + 1) & ~1 : u.nitems;   // half tiles: an even count, the last item repeated at weight zero
                        const int words = 1 + 3 * nit + (bx * by + 1) / 2;
                        const size_t pos = stream.size() - w0;
                        if (pos / kBlkRingWords != (pos + words - 1) / kBlkRingWords) {
                            const int skip = (int)(kBlkRingWords - pos % kBlkRingWords);
                            if (!have_header) return fail(MALA_SNAP_ECUDA, "internal: block stream starts with an oversized unit");
                            stream[last_header].w += skip;
                            for (int k = 0; k < skip; k++) stream.push_back(make_int4(0, 0, 0, 0));
                        }
                        last_header = stream.size();
                        have_header = true;
                        stream.push_back(make_int4(nit, u.ub_elem * RB, piece_slot[i], 0));
                        for (int k = 0; k < nit; k++) {
                            HostItem it = items[u.items_first + std::min(k, u.nitems - 1)];
                            if (k >= u.nitems) it.w = 0.0;
                            const int xe = it.fx ? it.ex - u.a0 : it.ex + u.a0, ye = it.fy ? it.ey - u.b0 : it.ey + u.b0;
                            // x = (-1)^(ma1 - mb1) conj(v) on a mirrored column: sign masks of the real part by the parity of the local row
                            const unsigned sgn = 0x80000000u;
                            const unsigned me = it.fx ? (((u.a0 + it.mb1) & 1) ? sgn : 0u) : 0u, mo = it.fx ? (me ^ sgn) : 0u;
                            stream.push_back(make_int4(xe * RB, it.fx ? -RB : RB, ye * RB, it.fy ? -RB : RB));
                            stream.push_back(make_int4((int)me, (int)mo, it.fx ? 1 : 0, 0));
                            const double pe = (it.fy && ((u.b0 + it.mb2) & 1)) ? -it.w : it.w, po = it.fy ? -pe : it.w;
                            push_d2(pe, po);
                        }
                        for (size_t k = 0; k < u.coef.size(); k += 2) push_d2(u.coef[k], k + 1 < u.coef.size() ? u.coef[k + 1] : 0.0);
                    }
                }
                wrange[(size_t)w * (kBlkShapes + 2) + (bx - 1) * kBlkBY + (by - 1)] = count;
            }
        while ((stream.size() - w0) % 32) stream.push_back(make_int4(0, 0, 0, 0));  // whole 512-byte chunks
        wrange[(size_t)w * (kBlkShapes + 2) + kBlkShapes + 1] = (int)(stream.size() - w0);
    }
    int rc = 0;
    if ((rc = upload(h->d_bstream, stream))) return rc;
    if ((rc = upload(h->d_bwrange, wrange))) return rc;
    if ((rc = upload(h->d_btslot, tslot))) return rc;
    h->blk_nslots = nslots;
    h->blk_ready = true;
    return 0;
}

// enqueue the sampling compute_ui (snap_ui_dft.cuh) for one chunk: whole tiles, twojmax + 1 warps
int launch_ui_dft(mala_snap *h, const GridGeom &g, const DeviceTables &tb, const ChunkBuffers &cb_in, cudaStream_t st) {
    ChunkBuffers cb = cb_in;
    if (h->use_ui_pipe()) {   // twojmax 8..14: one CTA per SM, a producer warp ahead of the sample warps (snap_ui_pipe.cuh)
        const int grid = std::max(1, std::min(h->num_sms, cb.ntiles));
        // A tile with more than 64 candidates, or a point with more neighbors than a queue buffer holds, comes in several windows
        // and once per accumulation pass: the producer keeps the geometry of the first pass in global memory (per CTA, at most
        // cand_cap / queue length windows; L2-resident) instead of preparing it again.
        const int cap = pipe_cap(h->twojmax);
        if (h->cand_cap > cap) {
            const int windows = std::min(16, (h->cand_cap + cap - 1) / cap);
            if (h->d_uispill.reserve((size_t)h->num_sms * windows * pipe_spill_record(h->twojmax), st, true))
                return fail(MALA_SNAP_ENOMEM, "cudaMallocAsync (compute_ui window spill) failed");
            cb.ui_spill = h->d_uispill.p;
            cb.ui_spill_windows = windows;
        }
        switch (h->twojmax) {
#define MALA_PIPE_CASE(TJ) \
    case TJ: compute_ui_pipe_kernel<TJ><<<grid, (TJ + 2) * 32, compute_ui_pipe_smem_bytes<TJ>(), st>>>(g, h->sc, tb, cb); break;
            MALA_PIPE_CASE(8) MALA_PIPE_CASE(9) MALA_PIPE_CASE(10) MALA_PIPE_CASE(11) MALA_PIPE_CASE(12) MALA_PIPE_CASE(13) MALA_PIPE_CASE(14)
#undef MALA_PIPE_CASE
            default: break;
        }
        return 0;
    }
    switch (h->twojmax) {
#define MALA_DFT_CASE(TJ) \
    case TJ: \
        compute_ui_dft_kernel<TJ><<<std::max(1, std::min(dft_ctas(TJ) * h->num_sms, cb.ntiles)), (TJ + 1) * 32, compute_ui_dft_smem_bytes<TJ>(), st>>>(g, h->sc, tb, cb); \
        break;
        MALA_DFT_CASE(1) MALA_DFT_CASE(2) MALA_DFT_CASE(3) MALA_DFT_CASE(4) MALA_DFT_CASE(5)
        MALA_DFT_CASE(6) MALA_DFT_CASE(7) MALA_DFT_CASE(8) MALA_DFT_CASE(9) MALA_DFT_CASE(10)
#undef MALA_DFT_CASE
        default: break;
    }
    return 0;
}

// enqueue compute_zi_bi for one chunk
int launch_zi(mala_snap *h, const ChunkBuffers &cb, double *out, cudaStream_t st) {
    const int grid = std::max(1, std::min(h->num_sms, h->half_tiles() ? 2 * cb.ntiles : cb.ntiles));
    TimedSpan span(h, st, kKindZi);
    if (h->use_block() && h->half_tiles())
        compute_zi_bi_block_half_kernel<<<grid, kBlkWarps * 32, compute_zi_block_half_smem_bytes(h->sc.nelem, h->blk_nslots), st>>>(
            h->geom, h->sc, h->tables(), h->blk_tables(), cb, out);
    else if (h->use_block()) {
        const size_t smem = compute_zi_block_smem_bytes(h->sc.nelem, h->sc.ntriples, h->blk_nslots);
        if (h->twojmax >= 8) compute_zi_bi_block_kernel<true><<<grid, kBlkWarps * 32, smem, st>>>(h->geom, h->sc, h->tables(), h->blk_tables(), cb, out);
        else compute_zi_bi_block_kernel<false><<<grid, kBlkWarps * 32, smem, st>>>(h->geom, h->sc, h->tables(), h->blk_tables(), cb, out);
    }
    else if (h->half_tiles())
        compute_zi_bi_diag_half_kernel<<<grid, kDiagHalfWarps * 32, compute_zi_diag_half_smem_bytes(h->sc.nelem, h->sc.ntriples), st>>>(
            h->geom, h->sc, h->tables(), h->diag_tables(), cb, out);
    else if (h->use_diag())
        compute_zi_bi_diag_kernel<<<grid, kDiagWarps * 32, compute_zi_diag_smem_bytes(h->sc.nelem, h->sc.ntriples), st>>>(
            h->geom, h->sc, h->tables(), h->diag_tables(), cb, out);
    else if (h->use_spec())
        compute_zi_bi_coop_kernel<<<grid, kCoopWarps * 32, compute_zi_coop_smem_bytes(), st>>>(h->geom, h->sc, h->tables(), cb, out);
    else
        compute_zi_bi_generic_kernel<<<grid, kZiWarps * 32, compute_zi_smem_bytes(h->sc.nelem, h->sc.ntriples), st>>>(h->geom, h->sc, h->tables(), cb, out);
    CUDA_TRY(cudaGetLastError());
    h->stats[0]++;
    return 0;
}

// B of a point without neighbors, computed by the same kernel that handles every other point.  Set-up time only
// (create, set_option): drains the device first, works on private temporaries and synchronises before returning.
int compute_bconst(mala_snap *h) {
    const int nelem = h->sc.nelem, nt = h->sc.ntriples, P = kTilePoints;
    CUDA_TRY(cudaDeviceSynchronize());
    std::vector<double2> u((size_t)nelem * P);  // [nelem][32], or [2][nelem][16] in the half-tile layout
    for (int e = 0; e < nelem; e++)
        for (int l = 0; l < P; l++) {
            const size_t at = h->half_tiles() ? ((size_t)(l >> 4) * nelem + e) * 16 + (l & 15) : (size_t)e * P + l;
            u[at] = make_double2(h->tab.udiag[e] ? h->wself : 0.0, 0.0);
        }
    DevBuf<double2> t_utot;
    DevBuf<int> t_active, t_counters;
    DevBuf<double> tmp;
    auto cleanup = [&]() { t_utot.release(); t_active.release(); t_counters.release(); tmp.release(); };
    if (t_utot.reserve(u.size()) || t_active.reserve(1) || t_counters.reserve(4) || tmp.reserve((size_t)32 * nt) || h->d_bconst.reserve(nt)) {
        cleanup();
        return fail(MALA_SNAP_ENOMEM, "cudaMalloc failed");
    }
    const int zero = 0;
    const int counters[4] = {1, 0, 0, 0};
    cudaError_t e = cudaMemcpy(t_utot.p, u.data(), u.size() * sizeof(double2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t_active.p, &zero, sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t_counters.p, counters, sizeof(counters), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cleanup(); return fail(MALA_SNAP_ECUDA, std::string("compute_bconst: ") + cudaGetErrorString(e)); }
    GridGeom g{};
    g.a1[0] = g.a2[1] = g.a3[2] = 1.0;
    g.nx = 4; g.ny = 4; g.nz = P / 16; g.z0 = 0; g.z1 = P / 16;
    g.nreg = 1; g.total_tiles = 1;
    g.reg[0].x0 = 0; g.reg[0].y0 = 0; g.reg[0].nxr = 4; g.reg[0].nyr = 4; g.reg[0].tx = 4; g.reg[0].ty = 4; g.reg[0].tz = P / 16;
    g.reg[0].ntx = g.reg[0].nty = g.reg[0].ntz = 1; g.reg[0].tile_begin = 0;
    const GridGeom saved = h->geom;
    h->geom = g;
    ChunkBuffers cb{};
    cb.active = t_active.p; cb.counters = t_counters.p; cb.status = h->d_status.p; cb.utot = t_utot.p; cb.tile_begin = 0; cb.ntiles = 1;
    cb.utot_half = h->half_tiles() ? 1 : 0;
    int rc = launch_zi(h, cb, tmp.p, nullptr);
    h->geom = saved;
    if (rc) { cleanup(); return rc; }
    e = cudaMemcpy(h->d_bconst.p, tmp.p, nt * sizeof(double), cudaMemcpyDeviceToDevice);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    cleanup();
    if (e != cudaSuccess) return fail(MALA_SNAP_ECUDA, std::string("compute_bconst: ") + cudaGetErrorString(e));
    return 0;
}

inline double dot3(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
inline void cross3(const double *a, const double *b, double *c) {
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

struct CallArgs {
    int natoms;
    const double *pos;
    const int *types;
    const double *box, *origin;
    const int *pbc, *ngrid;
    int z_begin, z_end;
};

int validate(const mala_snap *h, const CallArgs &a, bool need_out, const void *out) {
    if (!h) return fail(MALA_SNAP_EINVAL, "handle is NULL");
    if (a.natoms < 0) return fail(MALA_SNAP_EINVAL, "natoms < 0");
    if (a.natoms > 0 && (!a.pos || !a.types)) return fail(MALA_SNAP_EINVAL, "pos/types is NULL");
    if (!a.box || !a.origin || !a.pbc || !a.ngrid) return fail(MALA_SNAP_EINVAL, "box/origin/pbc/ngrid is NULL");
    for (int i = 0; i < 3; i++)
        if (a.ngrid[i] <= 0) return fail(MALA_SNAP_EINVAL, "ngrid must be positive");
    if (a.z_begin < 0 || a.z_end > a.ngrid[2] || a.z_begin > a.z_end) return fail(MALA_SNAP_EINVAL, "z range outside [0, nz]");
    if ((double)a.ngrid[0] * a.ngrid[1] * (double)(a.z_end - a.z_begin) * h->sc.ntriples > 9.0e15)
        return fail(MALA_SNAP_EINVAL, "grid too large");
    for (int i = 0; i < 9; i++)
        if (!std::isfinite(a.box[i])) return fail(MALA_SNAP_EINVAL, "box is not finite");
    for (int i = 0; i < 3; i++)
        if (!std::isfinite(a.origin[i])) return fail(MALA_SNAP_EINVAL, "origin is not finite");
    double c23[3];
    cross3(a.box + 3, a.box + 6, c23);
    const double det = dot3(a.box, c23);
    const double scale = std::sqrt(dot3(a.box, a.box) * dot3(a.box + 3, a.box + 3) * dot3(a.box + 6, a.box + 6));
    if (!(std::fabs(det) > 1e-12 * scale) || !(scale > 0)) return fail(MALA_SNAP_EINVAL, "box is singular");
    for (int n = 0; n < a.natoms; n++) {
        if (a.types[n] < 0 || a.types[n] >= h->ntypes) return fail(MALA_SNAP_EINVAL, "atom type out of range");
        for (int k = 0; k < 3; k++)
            if (!std::isfinite(a.pos[3 * n + k])) return fail(MALA_SNAP_EINVAL, "atom position is not finite");
    }
    if (need_out && !out && (a.z_end > a.z_begin)) return fail(MALA_SNAP_EINVAL, "out is NULL");
    return 0;
}

// Host half of build_plan: ghost atoms sorted by cell and the cell starts of the slab [z_begin, z_end); fills h->geom (except
// the tile fields) and picks the buffer set of the call.
int plan_host(mala_snap *h, const CallArgs &a, std::vector<Ghost> &sorted, std::vector<int> &start) {
    GridGeom &g = h->geom;
    h->spans.clear();
    h->ev_used = 0;
    h->cur = (int)(h->ncalls & 1ull);
    h->ncalls++;
    std::memset(&g, 0, sizeof(g));
    for (int k = 0; k < 3; k++) {
        g.a1[k] = a.box[k]; g.a2[k] = a.box[3 + k]; g.a3[k] = a.box[6 + k]; g.origin[k] = a.origin[k];
    }
    g.nx = a.ngrid[0]; g.ny = a.ngrid[1]; g.nz = a.ngrid[2];
    g.rcutmax = h->rcutmax;
    // reciprocal rows and plane spacings
    double c23[3], c31[3], c12[3];
    cross3(g.a2, g.a3, c23); cross3(g.a3, g.a1, c31); cross3(g.a1, g.a2, c12);
    const double det = dot3(g.a1, c23);
    const double *rec[3] = {c23, c31, c12};
    double hgt[3];
    for (int i = 0; i < 3; i++) hgt[i] = std::fabs(det) / std::sqrt(dot3(rec[i], rec[i]));
    // fractional extent of the grid points of the slab, widened by the cutoff
    const int n3[3] = {g.nx, g.ny, g.nz};
    double flo[3], fhi[3];
    for (int i = 0; i < 3; i++) {
        const double lo = (i == 2) ? (double)a.z_begin / n3[i] : 0.0;
        const double hi = (i == 2) ? (double)(std::max(a.z_end - 1, a.z_begin)) / n3[i] : (double)(n3[i] - 1) / n3[i];
        const double m = h->rcutmax / hgt[i] * (1.0 + 1e-12) + 1e-12;
        flo[i] = lo - m;
        fhi[i] = hi + m;
    }
    std::vector<Ghost> ghosts;
    ghosts.reserve((size_t)a.natoms * 2 + 16);
    const double *rows[3] = {g.a1, g.a2, g.a3};
    for (int n = 0; n < a.natoms; n++) {
        double x[3] = {a.pos[3 * n] - g.origin[0], a.pos[3 * n + 1] - g.origin[1], a.pos[3 * n + 2] - g.origin[2]};
        double f[3];
        int ilo[3], ihi[3];
        bool keep = true;
        for (int i = 0; i < 3; i++) {
            f[i] = dot3(x, rec[i]) / det;
            if (a.pbc[i]) {
                f[i] -= std::floor(f[i]);  // wrap into [0,1)  (reading #14)
                ilo[i] = (int)std::ceil(flo[i] - f[i]);
                ihi[i] = (int)std::floor(fhi[i] - f[i]);
                if (ilo[i] > ihi[i]) keep = false;
            } else {
                ilo[i] = ihi[i] = 0;
                if (f[i] < flo[i] || f[i] > fhi[i]) keep = false;
            }
        }
        if (!keep) continue;
        for (int i1 = ilo[0]; i1 <= ihi[0]; i1++)
            for (int i2 = ilo[1]; i2 <= ihi[1]; i2++)
                for (int i3 = ilo[2]; i3 <= ihi[2]; i3++) {
                    const double ff[3] = {f[0] + i1, f[1] + i2, f[2] + i3};
                    Ghost gh;
                    gh.x = g.origin[0] + ff[0] * rows[0][0] + ff[1] * rows[1][0] + ff[2] * rows[2][0];
                    gh.y = g.origin[1] + ff[0] * rows[0][1] + ff[1] * rows[1][1] + ff[2] * rows[2][1];
                    gh.z = g.origin[2] + ff[0] * rows[0][2] + ff[1] * rows[1][2] + ff[2] * rows[2][2];
                    gh.type = a.types[n];
                    gh.pad = n;  // the atom this image belongs to
                    ghosts.push_back(gh);
                    if (ghosts.size() > 400000000u) return fail(MALA_SNAP_ENOMEM, "too many periodic images");
                }
    }
    const size_t ng = ghosts.size();
    // Cartesian cell list
    double lo[3] = {0, 0, 0}, hi[3] = {1, 1, 1};
    if (ng > 0) {
        lo[0] = hi[0] = ghosts[0].x; lo[1] = hi[1] = ghosts[0].y; lo[2] = hi[2] = ghosts[0].z;
        for (const Ghost &gh : ghosts) {
            lo[0] = std::min(lo[0], gh.x); hi[0] = std::max(hi[0], gh.x);
            lo[1] = std::min(lo[1], gh.y); hi[1] = std::max(hi[1], gh.y);
            lo[2] = std::min(lo[2], gh.z); hi[2] = std::max(hi[2], gh.z);
        }
    }
    int nc[3];
    double target = std::max(0.5 * h->rcutmax, 1e-6);
    for (;;) {
        double total = 1.0;
        for (int d = 0; d < 3; d++) {
            const double ext = hi[d] - lo[d];
            nc[d] = (int)std::min(1024.0, std::max(1.0, std::floor(ext / target)));
            total *= nc[d];
        }
        if (total <= 4.0e6) break;
        target *= 1.26;
    }
    for (int d = 0; d < 3; d++) {
        const double ext = hi[d] - lo[d];
        g.cell_lo[d] = lo[d];
        g.cell_inv[d] = (ext > 1e-9) ? nc[d] / ext : 0.0;  // degenerate extent: one cell, every index maps to 0
    }
    g.ncx = nc[0]; g.ncy = nc[1]; g.ncz = nc[2];
    const size_t ncell = (size_t)nc[0] * nc[1] * nc[2];
    std::vector<int> cell_of(ng);
    start.assign(ncell + 1, 0);
    auto cidx = [&](double v, int d) {
        int i = (int)std::floor((v - g.cell_lo[d]) * g.cell_inv[d]);
        return std::min(std::max(i, 0), nc[d] - 1);
    };
    for (size_t i = 0; i < ng; i++) {
        const int c = (cidx(ghosts[i].z, 2) * nc[1] + cidx(ghosts[i].y, 1)) * nc[0] + cidx(ghosts[i].x, 0);
        cell_of[i] = c;
        start[c + 1]++;
    }
    for (size_t c = 0; c < ncell; c++) start[c + 1] += start[c];
    sorted.resize(ng);
    {
        std::vector<int> fill(start.begin(), start.end() - 1);
        for (size_t i = 0; i < ng; i++) sorted[fill[cell_of[i]]++] = ghosts[i];
    }
    return 0;
}

// Ghost atoms + cell list for the slab [z_begin, z_end) on the device; fills h->geom (except the tile fields).
int build_plan(mala_snap *h, const CallArgs &a, cudaStream_t st) {
    std::vector<Ghost> sorted;
    std::vector<int> start;
    int rc = plan_host(h, a, sorted, start);
    if (rc) return rc;
    const int cur = h->cur;
    const size_t ng = sorted.size(), ncell = start.size() - 1;
    // The workspace (U_tot, candidate lists, counters) is one set per handle: a call on another stream must not start
    // before the previous call on this handle has drained (calls on one handle are serialised, whatever their streams).
    if (h->call_done_valid[cur ^ 1]) CUDA_TRY(cudaStreamWaitEvent(st, h->ev_call_done[cur ^ 1], 0));
    // upload on the private stream once the call that last used this buffer set has drained
    if (h->call_done_valid[cur]) CUDA_TRY(cudaStreamWaitEvent(h->upload_stream, h->ev_call_done[cur], 0));
    if (h->d_ghosts[cur].reserve(std::max<size_t>(ng, 1), h->upload_stream, true) ||
        h->d_cell_start[cur].reserve(ncell + 1, h->upload_stream, true))
        return fail(MALA_SNAP_ENOMEM, "cudaMallocAsync (ghosts) failed");
    if (ng) CUDA_TRY(cudaMemcpyAsync(h->d_ghosts[cur].p, sorted.data(), ng * sizeof(Ghost), cudaMemcpyHostToDevice, h->upload_stream));
    CUDA_TRY(cudaMemcpyAsync(h->d_cell_start[cur].p, start.data(), (ncell + 1) * sizeof(int), cudaMemcpyHostToDevice, h->upload_stream));
    // (pageable sources: cudaMemcpyAsync returns only after they have been staged, so they may die with this scope)
    CUDA_TRY(cudaEventRecord(h->ev_upload, h->upload_stream));
    CUDA_TRY(cudaStreamWaitEvent(st, h->ev_upload, 0));
    h->stats[3] = (long long)ng;
    h->h_cell_start.swap(start);
    return 0;
}

}  // namespace

namespace {

// Tile shapes: 32 points as a small brick.  The (x, y) extent is split into the part the main brick covers exactly, the
// strips left over along x and along y, and their corner; every part gets the brick that minimises
// (number of tiles) x (1 + radius / rcut)^3 -- wasted lanes cost whole tiles, a larger radius costs candidate tests.
void choose_tiles(mala_snap *h, int z0, int z1) {
    GridGeom &g = h->geom;
    static const int shapes[][3] = {{4, 4, 2}, {4, 2, 4}, {2, 4, 4}, {8, 2, 2}, {2, 8, 2}, {2, 2, 8}, {8, 4, 1}, {4, 8, 1},
                                    {16, 2, 1}, {2, 16, 1}, {32, 1, 1}, {1, 32, 1}, {1, 1, 32}, {16, 1, 2}, {1, 16, 2},
                                    {8, 1, 4}, {1, 8, 4}, {4, 1, 8}, {1, 4, 8}, {2, 1, 16}, {1, 2, 16}};
    constexpr int nshapes = (int)(sizeof(shapes) / sizeof(shapes[0]));
    const int nzs = std::max(z1 - z0, 1);
    const double rcut = std::max(h->rcutmax, 1e-9);
    // radius of a brick: half its longest body diagonal
    auto radius_of = [&](const int *t) {
        double e[3][3];
        for (int k = 0; k < 3; k++) {
            e[0][k] = g.a1[k] * (t[0] - 1) / g.nx;
            e[1][k] = g.a2[k] * (t[1] - 1) / g.ny;
            e[2][k] = g.a3[k] * (t[2] - 1) / g.nz;
        }
        double r = 0.0;
        for (int sg = 0; sg < 4; sg++) {
            const double s1 = (sg & 1) ? -1.0 : 1.0, s2 = (sg & 2) ? -1.0 : 1.0;
            double d[3];
            for (int k = 0; k < 3; k++) d[k] = e[0][k] + s1 * e[1][k] + s2 * e[2][k];
            r = std::max(r, 0.5 * std::sqrt(dot3(d, d)));
        }
        return r * (1.0 + 1e-9) + 1e-12;
    };
    auto cost_of = [&](int nxr, int nyr, const int *t) {
        if (nxr <= 0 || nyr <= 0) return 0.0;
        const double tiles = (double)((nxr + t[0] - 1) / t[0]) * ((nyr + t[1] - 1) / t[1]) * ((nzs + t[2] - 1) / t[2]);
        const double reach = 1.0 + radius_of(t) / rcut;
        return tiles * reach * reach * reach;
    };
    auto best_shape = [&](int nxr, int nyr, double &cost) {
        int best = 0;
        cost = 1e300;
        for (int s = 0; s < nshapes; s++) {
            const double c = cost_of(nxr, nyr, shapes[s]);
            if (c < cost * (1.0 - 1e-12)) { cost = c; best = s; }
        }
        return best;
    };
    double best_cost = 1e300;
    int pick[4] = {0, 0, 0, 0}, X0 = 0, Y0 = 0;
    for (int s = 0; s < nshapes; s++) {
        const int *t = shapes[s];
        const int x0 = g.nx / t[0] * t[0], y0 = g.ny / t[1] * t[1];
        double c1, c2, c3;
        const int s1 = best_shape(g.nx - x0, y0, c1), s2 = best_shape(x0, g.ny - y0, c2), s3 = best_shape(g.nx - x0, g.ny - y0, c3);
        const double c = cost_of(x0, y0, t) + c1 + c2 + c3;
        if (c < best_cost * (1.0 - 1e-12)) {
            best_cost = c;
            pick[0] = s; pick[1] = s1; pick[2] = s2; pick[3] = s3;
            X0 = x0; Y0 = y0;
        }
    }
    const int ext[4][4] = {{0, 0, X0, Y0}, {X0, 0, g.nx - X0, Y0}, {0, Y0, X0, g.ny - Y0}, {X0, Y0, g.nx - X0, g.ny - Y0}};
    g.z0 = z0; g.z1 = z1;
    g.nreg = 0;
    g.tile_radius = 0.0;
    long long total = 0;
    for (int r = 0; r < 4; r++) {
        if (ext[r][2] <= 0 || ext[r][3] <= 0) continue;
        GridGeom::Region &R = g.reg[g.nreg++];
        const int *t = shapes[pick[r]];
        R.x0 = ext[r][0]; R.y0 = ext[r][1]; R.nxr = ext[r][2]; R.nyr = ext[r][3];
        R.tx = t[0]; R.ty = t[1]; R.tz = t[2];
        R.ntx = (R.nxr + R.tx - 1) / R.tx; R.nty = (R.nyr + R.ty - 1) / R.ty; R.ntz = (nzs + R.tz - 1) / R.tz;
        R.tile_begin = (int)std::min<long long>(total, 2000000000LL);
        R.pad = 0;
        R.tile_radius = radius_of(t);
        g.tile_radius = std::max(g.tile_radius, R.tile_radius);
        total += (long long)R.ntx * R.nty * R.ntz;
    }
    h->total_tiles = total;
    g.total_tiles = (int)std::min<long long>(total, 2000000000LL);
}

// upper bound of the candidates tile_bin_kernel can collect for any tile: maximum ghost count over all windows
// of cells it may scan (summed-area table over the cell counts)
int candidate_bound(const mala_snap *h) {
    const GridGeom &g = h->geom;
    const int nc[3] = {g.ncx, g.ncy, g.ncz};
    const double reach = g.tile_radius + g.rcutmax;
    int w[3];
    for (int d = 0; d < 3; d++) w[d] = (int)std::min((double)nc[d], std::floor(2.0 * reach * g.cell_inv[d]) + 2.0);
    const size_t sx = nc[0] + 1, sy = nc[1] + 1, sz = nc[2] + 1;
    std::vector<long long> S(sx * sy * sz, 0);
    auto at = [&](int x, int y, int z) -> long long & { return S[((size_t)z * sy + y) * sx + x]; };
    const std::vector<int> &st = h->h_cell_start;
    for (int z = 1; z <= nc[2]; z++)
        for (int y = 1; y <= nc[1]; y++)
            for (int x = 1; x <= nc[0]; x++) {
                const size_t c = ((size_t)(z - 1) * nc[1] + (y - 1)) * nc[0] + (x - 1);
                const long long cnt = st[c + 1] - st[c];
                at(x, y, z) = cnt + at(x - 1, y, z) + at(x, y - 1, z) + at(x, y, z - 1) - at(x - 1, y - 1, z) - at(x - 1, y, z - 1) -
                              at(x, y - 1, z - 1) + at(x - 1, y - 1, z - 1);
            }
    long long best = 0;
    for (int z = w[2]; z <= nc[2]; z++)
        for (int y = w[1]; y <= nc[1]; y++)
            for (int x = w[0]; x <= nc[0]; x++) {
                const int x0 = x - w[0], y0 = y - w[1], z0 = z - w[2];
                const long long v = at(x, y, z) - at(x0, y, z) - at(x, y0, z) - at(x, y, z0) + at(x0, y0, z) + at(x0, y, z0) +
                                    at(x, y0, z0) - at(x0, y0, z0);
                best = std::max(best, v);
            }
    best = std::max<long long>(best, 1);
    best = (best + 31) / 32 * 32;
    if (best > (1 << 24)) return -1;  // caller reports it: no silent clamp
    if (h->cand_cap_limit > 0) best = std::min<long long>(best, h->cand_cap_limit);  // test hook (provokes kStatusCandOverflow)
    return (int)best;
}

// enqueue the whole path for the slab [z0, z1) into out (DEVICE, relative to z0); out == nullptr: stop after compute_ui
// and scatter U_tot into u_out (test hook)
// net != nullptr: the descriptors of every chunk go to a compact staging buffer and the network maps them to ldos (DEVICE,
// [points of the slab][w_out] fp32) before the next chunk starts; out is not used
int run_slab(mala_snap *h, int z0, int z1, double *out, double2 *u_out, cudaStream_t st, const mala_mlp *net = nullptr,
             float *ldos = nullptr) {
    if (z1 <= z0) return 0;
    choose_tiles(h, z0, z1);
    GridGeom &g = h->geom;
    h->cand_cap = candidate_bound(h);
    if (h->cand_cap < 0) return fail(MALA_SNAP_EINVAL, "more than 2^24 candidate atoms per tile; use a finer cell or smaller z-slabs");
    const long long total_tiles = h->total_tiles;
    if (total_tiles > 2000000000LL) return fail(MALA_SNAP_EINVAL, "slab has too many tiles; use smaller z-slabs");
    const size_t per_tile = (size_t)h->sc.nelem * 32 * sizeof(double2) + (size_t)h->cand_cap * sizeof(int) + 2 * sizeof(int) +
                            (net ? (size_t)32 * h->sc.ntriples * sizeof(double) : 0);
    const size_t budget = (size_t)std::max<long long>(h->workspace_mb, 1) << 20;
    long long chunk_tiles = (long long)std::max<size_t>(budget / per_tile, (size_t)h->num_sms);
    chunk_tiles = std::min(chunk_tiles, total_tiles);
    if (net && h->d_bstage.reserve((size_t)chunk_tiles * 32 * h->sc.ntriples, st, true))
        return fail(MALA_SNAP_ENOMEM, "cudaMallocAsync (descriptor staging) failed");
    if (net) out = h->d_bstage.p;
    if (h->d_utot.reserve((size_t)chunk_tiles * h->sc.nelem * 32, st, true) || h->d_cand.reserve((size_t)chunk_tiles * h->cand_cap, st, true) ||
        h->d_ncand.reserve(chunk_tiles, st, true) || h->d_active.reserve(chunk_tiles, st, true) || h->d_counters.reserve(4, st, true))
        return fail(MALA_SNAP_ENOMEM, "cudaMallocAsync (workspace) failed");
    h->stats[4] = h->cand_cap;
    h->stats[5] = (long long)(per_tile * (size_t)chunk_tiles);
    const DeviceTables tb = h->tables();
    for (long long t0 = 0; t0 < total_tiles; t0 += chunk_tiles) {
        ChunkBuffers cb{};
        cb.ghosts = h->d_ghosts[h->cur].p; cb.cell_start = h->d_cell_start[h->cur].p;
        cb.cand = h->d_cand.p; cb.ncand = h->d_ncand.p; cb.active = h->d_active.p; cb.counters = h->d_counters.p;
        cb.status = h->d_status.p;
        cb.utot = h->d_utot.p; cb.cand_cap = h->cand_cap;
        cb.utot_half = h->half_tiles() ? 1 : 0;
        cb.compact_out = net ? 1 : 0;
        cb.tile_begin = (int)t0;
        cb.ntiles = (int)std::min(chunk_tiles, total_tiles - t0);
        CUDA_TRY(cudaMemsetAsync(cb.counters, 0, 4 * sizeof(int), st));
        const int bin_blocks = (cb.ntiles + 7) / 8;
        {
            TimedSpan span(h, st, kKindBin);
            tile_bin_kernel<<<bin_blocks, 256, 0, st>>>(g, h->sc, tb, cb, out);
        }
        CUDA_TRY(cudaGetLastError());
        const int grid = std::max(1, std::min(h->num_sms, cb.ntiles));
        {
            TimedSpan span(h, st, kKindUi);
            if (h->half_tiles() && h->use_ui_pipe()) {  // twojmax 11..14: the pipelined sampling kernel, whole tiles stored as two halves
                if (int rc = launch_ui_dft(h, g, tb, cb, st)) return rc;
            } else if (h->half_tiles()) {  // the column kernel: eight column warps, one CTA per SM
                const int ui_grid = std::max(1, std::min(h->num_sms, 2 * cb.ntiles));
                compute_ui_kernel<kMaxTwoJ, false><<<ui_grid, (kMaxTwoJ / 2 + 1) * 32, compute_ui_smem_bytes(kMaxTwoJ), st>>>(g, h->sc, tb, cb);
            } else {
                const int ui_grid = std::max(1, std::min(2 * h->num_sms, 2 * cb.ntiles));  // half-tile items, two CTAs per SM
                if (h->use_ui_dft()) {   // twojmax 1..10: column polynomials sampled at the roots of unity (snap_ui_dft.cuh), whole tiles
                    if (int rc = launch_ui_dft(h, g, tb, cb, st)) return rc;
                } else if (h->twojmax == kFullTileTwoJ)
                    compute_ui_kernel<kFullTileTwoJ, true><<<ui_grid, (kFullTileTwoJ / 2 + 1) * 32, compute_ui_smem_bytes(kFullTileTwoJ), st>>>(g, h->sc, tb, cb);
                else  // smaller twojmax: same code with run-time guards on the levels
                    compute_ui_kernel<kFullTileTwoJ, false><<<ui_grid, (kFullTileTwoJ / 2 + 1) * 32, compute_ui_smem_bytes(kFullTileTwoJ), st>>>(g, h->sc, tb, cb);
            }
        }
        CUDA_TRY(cudaGetLastError());
        h->stats[0] += 2;
        if (out) {
            int rc = launch_zi(h, cb, out, st);
            if (rc) return rc;
            if (net) {
                MlpRows rows{};
                rows.nrows = (long long)cb.ntiles * 32; rows.x = out; rows.y = ldos; rows.compact = 1; rows.tile_begin = cb.tile_begin;
                rows.geom = g;
                TimedSpan span(h, st, kKindOther);
                if ((rc = mlp_launch(net, rows, st))) return rc;
                h->stats[0]++;
            }
        } else if (u_out) {
            TimedSpan span(h, st, kKindOther);
            utot_scatter_kernel<<<bin_blocks, 256, 0, st>>>(g, h->sc, tb, cb, u_out);
            CUDA_TRY(cudaGetLastError());
            h->stats[0]++;
        }
        h->stats[1]++;
    }
    h->stats[2] += total_tiles;
    h->stats[6] += (long long)g.nx * g.ny * (z1 - z0);
    return 0;
}

// Gaussian descriptors of the slab [z0, z1) into out (DEVICE, [points][ntypes]): tile binning + one pass over the candidates
int run_slab_gauss(mala_snap *h, int z0, int z1, double sigma, double *out, cudaStream_t st) {
    if (z1 <= z0) return 0;
    choose_tiles(h, z0, z1);
    GridGeom &g = h->geom;
    h->cand_cap = candidate_bound(h);
    if (h->cand_cap < 0) return fail(MALA_SNAP_EINVAL, "more than 2^24 candidate atoms per tile; use a finer cell or smaller z-slabs");
    const long long total_tiles = h->total_tiles;
    if (total_tiles > 2000000000LL) return fail(MALA_SNAP_EINVAL, "slab has too many tiles; use smaller z-slabs");
    const size_t per_tile = (size_t)h->cand_cap * sizeof(int) + 2 * sizeof(int);
    const size_t budget = (size_t)std::max<long long>(h->workspace_mb, 1) << 20;
    long long chunk_tiles = (long long)std::max<size_t>(budget / per_tile, (size_t)h->num_sms);
    chunk_tiles = std::min(chunk_tiles, total_tiles);
    if (h->d_cand.reserve((size_t)chunk_tiles * h->cand_cap, st, true) || h->d_ncand.reserve(chunk_tiles, st, true) ||
        h->d_active.reserve(chunk_tiles, st, true) || h->d_counters.reserve(4, st, true))
        return fail(MALA_SNAP_ENOMEM, "cudaMallocAsync (workspace) failed");
    const double pi = 3.14159265358979323846;
    const double pref = 1.0 / (std::pow(2.0 * pi, 1.5) * sigma * sigma * sigma), inv2s2 = 1.0 / (2.0 * sigma * sigma);
    const DeviceTables tb = h->tables();
    for (long long t0 = 0; t0 < total_tiles; t0 += chunk_tiles) {
        ChunkBuffers cb{};
        cb.ghosts = h->d_ghosts[h->cur].p; cb.cell_start = h->d_cell_start[h->cur].p;
        cb.cand = h->d_cand.p; cb.ncand = h->d_ncand.p; cb.active = h->d_active.p; cb.counters = h->d_counters.p;
        cb.status = h->d_status.p;
        cb.cand_cap = h->cand_cap;
        cb.tile_begin = (int)t0;
        cb.ntiles = (int)std::min(chunk_tiles, total_tiles - t0);
        CUDA_TRY(cudaMemsetAsync(cb.counters, 0, 4 * sizeof(int), st));
        const int blocks = (cb.ntiles + 7) / 8;
        {
            TimedSpan span(h, st, kKindBin);
            tile_bin_kernel<<<blocks, 256, 0, st>>>(g, h->sc, tb, cb, nullptr);
        }
        CUDA_TRY(cudaGetLastError());
        {
            TimedSpan span(h, st, kKindOther);
            gaussian_grid_kernel<<<blocks, 256, 0, st>>>(g, h->sc, tb, cb, inv2s2, pref, out);
        }
        CUDA_TRY(cudaGetLastError());
        h->stats[0] += 2;
        h->stats[1]++;
    }
    h->stats[2] += total_tiles;
    h->stats[4] = h->cand_cap;
    h->stats[6] += (long long)g.nx * g.ny * (z1 - z0);
    return 0;
}

struct YHostTerm { int A, B, C, index; double coef; int cgoff; };
int build_yi_block_schedule(mala_snap *h, const std::vector<YHostTerm> &terms, const std::vector<double> &cg);

// tables of compute_yi (snap_force.cuh): the (up to three, distinct) Z-type contributions per bispectrum component, grouped by target level
int build_force_tables(mala_snap *h) {
    if (h->force_ready) return 0;
    const SnapTables &T = h->tab;
    const int tj = h->twojmax, nt = T.ntriples;
    struct Raw { int A, B, C, index; double coef; };
    std::vector<Raw> raw;
    for (int t = 0; t < nt; t++) {
        const int j1 = T.triples[4 * t], j2 = T.triples[4 * t + 1], j = T.triples[4 * t + 2];
        // a triple with equal entries names the same contraction more than once (j1 == j2: the last two; j == j1: the first
        // two): one term with the sum of the coefficients
        const Raw three[3] = {{j1, j2, j, t, 1.0}, {j, j2, j1, t, (double)(j + 1) / (double)(j1 + 1)}, {j, j1, j2, t, (double)(j + 1) / (double)(j2 + 1)}};
        const size_t first = raw.size();
        for (const Raw &r : three) {
            bool merged = false;
            for (size_t k = first; k < raw.size() && !merged; k++)
                if (raw[k].A == r.A && raw[k].B == r.B && raw[k].C == r.C) { raw[k].coef += r.coef; merged = true; }
            if (!merged) raw.push_back(r);
        }
    }
    std::stable_sort(raw.begin(), raw.end(), [](const Raw &a, const Raw &b) { return a.C < b.C; });
    std::vector<YTerm> terms;
    std::vector<double> cg;
    std::vector<int> level(tj + 2, 0);
    for (const Raw &r : raw) {
        YTerm y{};
        y.A = (short)r.A; y.B = (short)r.B; y.C = (short)r.C; y.index = (short)r.index; y.coef = r.coef;
        y.cgoff = (int)cg.size();
        const int sh = (r.A + r.B - r.C) / 2;
        for (int m2 = 0; m2 <= r.B; m2++)
            for (int m1 = 0; m1 <= r.A; m1++) {
                const int m = m1 + m2 - sh;
                cg.push_back((m >= 0 && m <= r.C) ? clebsch_gordan(r.A, 2 * m1 - r.A, r.B, 2 * m2 - r.B, r.C, 2 * m - r.C) : 0.0);
            }
        level[r.C + 1]++;
        terms.push_back(y);
    }
    for (int C = 0; C <= tj; C++) level[C + 1] += level[C];
    // cost of a Y element = product terms over its contributions; processing order by decreasing cost
    std::vector<double> cost(T.nelem, 0.0), yweight(T.nelem, 0.0);
    for (int C = 0; C <= tj; C++)
        for (int mb = 0; mb <= C / 2; mb++)
            for (int ma = 0; ma <= C; ma++) {
                const int e = uhalf_off(C) + mb * (C + 1) + ma;
                for (int k = level[C]; k < level[C + 1]; k++) {
                    const int A = terms[k].A, B = terms[k].B, sh = (A + B - C) / 2;
                    const int nb = std::min(A, mb + sh) - std::max(0, mb + sh - B) + 1, na = std::min(A, ma + sh) - std::max(0, ma + sh - B) + 1;
                    cost[e] += (double)std::max(nb, 0) * std::max(na, 0) + 4.0;
                }
                const bool mid = (C % 2 == 0) && (mb == C / 2);
                yweight[e] = T.unorm[e] * (mid ? 1.0 : 2.0);
            }
    std::vector<int> order(T.nelem);
    for (int e = 0; e < T.nelem; e++) order[e] = e;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cost[a] > cost[b]; });
    int rc = 0;
    if ((rc = upload(h->d_yterms, terms))) return rc;
    if ((rc = upload(h->d_ylevel, level))) return rc;
    if ((rc = upload(h->d_ycg, cg))) return rc;
    if ((rc = upload(h->d_yorder, order))) return rc;
    if ((rc = upload(h->d_yweight, yweight))) return rc;
    CUDA_TRY(cudaFuncSetAttribute(compute_yi_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)compute_yi_smem_bytes(uhalf_size(kFullTileTwoJ), triple_count(kFullTileTwoJ))));
    CUDA_TRY(cudaFuncSetAttribute(compute_dedr_kernel<kFullTileTwoJ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)compute_dedr_smem_bytes(kFullTileTwoJ)));
#define MALA_DD_ATTR(TJ) \
    CUDA_TRY(cudaFuncSetAttribute(compute_dedr_dft_kernel<TJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)compute_dedr_dft_smem_bytes<TJ>()));
    MALA_DD_ATTR(1) MALA_DD_ATTR(2) MALA_DD_ATTR(3) MALA_DD_ATTR(4) MALA_DD_ATTR(5)
    MALA_DD_ATTR(6) MALA_DD_ATTR(7) MALA_DD_ATTR(8) MALA_DD_ATTR(9) MALA_DD_ATTR(10)
#undef MALA_DD_ATTR
    {
        std::vector<YHostTerm> ht;
        for (const YTerm &y : terms) ht.push_back({y.A, y.B, y.C, y.index, y.coef, y.cgoff});
        if ((rc = build_yi_block_schedule(h, ht, cg))) return rc;
    }
    h->force_ready = true;
    return 0;
}

// Record streams of compute_yi_block_kernel (snap_yi_block.cuh): every term (A, B -> C) of Y is cut into units exactly as
// the triples of compute_zi are (build_block_schedule), without the symmetries that belong to B (only the swap of equal
// factors, A == B, halves the items) and without fold weights; the units of a pass (a group of target levels) are dealt to
// the warps by decreasing cost, pass by pass, because a barrier ends every pass.
int build_yi_block_schedule(mala_snap *h, const std::vector<YHostTerm> &terms, const std::vector<double> &cg) {
    const int tj = h->twojmax, NW = kBlkWarps;
    constexpr int RB = 32 * (int)sizeof(double2);
    // passes: consecutive levels from the top, as many as fit the accumulator (at least the top level alone)
    const int cap = std::max(64, (tj + 1) * (tj / 2 + 1));
    std::vector<int> pass_of_level(tj + 1, 0);
    std::vector<std::pair<int, int>> pass_levels;            // [lo level, hi level]
    for (int hi = tj; hi >= 0;) {
        int lo = hi, size = (hi + 1) * (hi / 2 + 1);
        while (lo - 1 >= 0 && size + lo * ((lo - 1) / 2 + 1) <= cap) { lo--; size += (lo + 1) * (lo / 2 + 1); }
        pass_levels.push_back({lo, hi});
        hi = lo - 1;
    }
    const int npasses = (int)pass_levels.size();
    if (npasses > kYBlkMaxPasses) return fail(MALA_SNAP_ECUDA, "internal: too many passes in compute_yi");
    for (int p = 0; p < npasses; p++)
        for (int L = pass_levels[p].first; L <= pass_levels[p].second; L++) pass_of_level[L] = p;
    struct HostItem { int ex, ey; bool fx, fy; int mb1, mb2; double w; };
    struct HostUnit { int items_first, nitems, a0, b0, bx, by, yelem, dlo, dhi, index; double coef; std::vector<double> c; double cost; };
    std::vector<HostItem> items;
    std::vector<std::vector<HostUnit>> punits(npasses);
    auto chunks = [](int len, int mx) {
        std::vector<std::pair<int, int>> out;
        const int k = (len + mx - 1) / mx, base = len / k, rem = len % k;
        int s = 0;
        for (int i = 0; i < k; i++) { const int c = base + (i < rem ? 1 : 0); out.push_back({s, c}); s += c; }
        return out;
    };
    for (const YHostTerm &t : terms) {
        const int A = t.A, B = t.B, C = t.C, sh = (A + B - C) / 2, pass = pass_of_level[C];
        const int e_pass = uhalf_off(pass_levels[pass].first);
        for (int mb = 0; mb <= C / 2; mb++) {
            int lo = std::max(0, mb + sh - B), hi = std::min(A, mb + sh);
            if (A == B && (mb + sh) / 2 < hi) hi = (mb + sh) / 2;   // items (mb1, mb2) and (mb2, mb1) contribute the same column
            if (hi < lo) continue;
            const int items_first = (int)items.size();
            for (int mb1 = lo; mb1 <= hi; mb1++) {
                const int mb2 = mb + sh - mb1;
                double w = cg[t.cgoff + mb2 * (A + 1) + mb1];
                if (A == B && mb1 != mb2) w += w;
                HostItem it;
                it.fx = mb1 > A / 2; it.fy = mb2 > B / 2; it.mb1 = mb1; it.mb2 = mb2; it.w = w;
                it.ex = it.fx ? uhalf_off(A) + (A - mb1) * (A + 1) + A : uhalf_off(A) + mb1 * (A + 1);
                it.ey = it.fy ? uhalf_off(B) + (B - mb2) * (B + 1) + B : uhalf_off(B) + mb2 * (B + 1);
                items.push_back(it);
            }
            const int n = hi - lo + 1;
            // the middle column of an even level is computed up to its centre row; the flush mirrors the rest (ma_hi rows)
            const int ma_hi = (C % 2 == 0 && mb == C / 2) ? C / 2 : C;
            auto cf = [&](int m1, int m2) {
                const int ma = m1 + m2 - sh;
                return (ma < 0 || ma > ma_hi) ? 0.0 : cg[t.cgoff + m2 * (A + 1) + m1];
            };
            for (auto cx : chunks(A + 1, kBlkBX))
                for (auto cy : chunks(B + 1, kBlkBY)) {
                    int a_lo = 1 << 30, a_hi = -1, b_lo = 1 << 30, b_hi = -1;
                    for (int a = cx.first; a < cx.first + cx.second; a++)
                        for (int b = cy.first; b < cy.first + cy.second; b++)
                            if (cf(a, b) != 0.0) { a_lo = std::min(a_lo, a); a_hi = std::max(a_hi, a); b_lo = std::min(b_lo, b); b_hi = std::max(b_hi, b); }
                    if (a_hi < 0) continue;
                    HostUnit u;
                    u.items_first = items_first; u.nitems = n; u.index = t.index; u.coef = t.coef;
                    int bx = a_hi - a_lo + 1, by = b_hi - b_lo + 1;
                    if (bx < kBlkBXMin) { a_lo = std::max(0, std::min(a_lo, A + 1 - kBlkBXMin)); bx = kBlkBXMin; }
                    if (by < kBlkBYMin) { b_lo = std::max(0, std::min(b_lo, B + 1 - kBlkBYMin)); by = kBlkBYMin; }
                    u.a0 = a_lo; u.b0 = b_lo; u.bx = bx; u.by = by;
                    const int ma0 = a_lo + b_lo - sh;
                    u.yelem = uhalf_off(C) + mb * (C + 1) + ma0 - e_pass;   // element of row ma0 in the pass's accumulator (may be negative)
                    u.dlo = std::max(0, -ma0); u.dhi = std::min(bx + by - 2, ma_hi - ma0);
                    for (int d = 0; d <= bx + by - 2; d++)   // in the order the kernel consumes them (blk_coef_index)
                        for (int a = 0; a < bx; a++) {
                            const int b = d - a;
                            if (b < 0 || b >= by) continue;
                            u.c.push_back((a_lo + a >= cx.first && a_lo + a < cx.first + cx.second && b_lo + b >= cy.first && b_lo + b < cy.first + cy.second)
                                              ? cf(a_lo + a, b_lo + b) : 0.0);
                        }
                    u.cost = n * (2.0 * (4 * bx * by + 2 * by) + 3.0 * bx + 2.0 * by + 14.0) + 2.0 * (2 * bx * by) + 12.0 * (bx + by - 1) + 2.0 * bx * by + 50.0;
                    punits[pass].push_back(std::move(u));
                }
        }
    }
    // deal: per pass, units by decreasing cost to the least loaded warp
    std::vector<std::vector<std::vector<const HostUnit *>>> mine(NW, std::vector<std::vector<const HostUnit *>>(npasses));
    for (int p = 0; p < npasses; p++) {
        std::vector<const HostUnit *> order;
        for (const HostUnit &u : punits[p]) order.push_back(&u);
        std::stable_sort(order.begin(), order.end(), [](const HostUnit *a, const HostUnit *b) { return a->cost > b->cost; });
        std::vector<double> load(NW, 0.0);
        for (const HostUnit *u : order) {
            int w = 0;
            for (int k = 1; k < NW; k++)
                if (load[k] < load[w]) w = k;
            load[w] += u->cost;
            mine[w][p].push_back(u);
        }
    }
    std::vector<int4> stream;
    std::vector<int> wrange((size_t)NW * npasses * kBlkShapes + 2 * NW, 0);
    auto push_d2 = [&](double a, double b) {
        int4 v;
        std::memcpy(&v.x, &a, 8);
        std::memcpy(&v.z, &b, 8);
        stream.push_back(v);
    };
    for (int w = 0; w < NW; w++) {
        const size_t w0 = stream.size();
        wrange[yblk_wrange_first(w, npasses)] = (int)w0;
        size_t last_header = 0;
        bool have_header = false;
        for (int p = 0; p < npasses; p++)
            for (int bx = kBlkBX; bx >= 1; bx--)
                for (int by = kBlkBY; by >= 1; by--) {
                    int count = 0;
                    for (const HostUnit *up : mine[w][p]) {
                        const HostUnit &u = *up;
                        if (u.bx != bx || u.by != by) continue;
                        count++;
                        const int words = 2 + 3 * u.nitems + (bx * by + 1) / 2;
                        const size_t pos = stream.size() - w0;
                        if (pos / kBlkRingWords != (pos + words - 1) / kBlkRingWords) {
                            const int skip = (int)(kBlkRingWords - pos % kBlkRingWords);
                            if (!have_header) return fail(MALA_SNAP_ECUDA, "internal: Y stream starts with an oversized unit");
                            stream[last_header].w += skip;
                            for (int k = 0; k < skip; k++) stream.push_back(make_int4(0, 0, 0, 0));
                        }
                        last_header = stream.size();
                        have_header = true;
                        stream.push_back(make_int4(u.nitems, u.yelem * RB, u.index, 0));
                        {
                            int4 h1;
                            h1.x = u.dlo; h1.y = u.dhi;
                            std::memcpy(&h1.z, &u.coef, 8);
                            stream.push_back(h1);
                        }
                        for (int k = 0; k < u.nitems; k++) {
                            const HostItem &it = items[u.items_first + k];
                            const int xe = it.fx ? it.ex - u.a0 : it.ex + u.a0, ye = it.fy ? it.ey - u.b0 : it.ey + u.b0;
                            const unsigned sgn = 0x80000000u;
                            const unsigned me = it.fx ? (((u.a0 + it.mb1) & 1) ? sgn : 0u) : 0u, mo = it.fx ? (me ^ sgn) : 0u;
                            stream.push_back(make_int4(xe * RB, it.fx ? -RB : RB, ye * RB, it.fy ? -RB : RB));
                            stream.push_back(make_int4((int)me, (int)mo, it.fx ? 1 : 0, 0));
                            const double pe = (it.fy && ((u.b0 + it.mb2) & 1)) ? -it.w : it.w, po = it.fy ? -pe : it.w;
                            push_d2(pe, po);
                        }
                        for (size_t k = 0; k < u.c.size(); k += 2) push_d2(u.c[k], k + 1 < u.c.size() ? u.c[k + 1] : 0.0);
                    }
                    wrange[yblk_wrange_count(w, p, (bx - 1) * kBlkBY + (by - 1), npasses)] = count;
                }
        while ((stream.size() - w0) % 32) stream.push_back(make_int4(0, 0, 0, 0));
        wrange[yblk_wrange_first(w, npasses) + 1] = (int)(stream.size() - w0);
    }
    std::vector<int> pe(npasses + 1, 0);
    int yacc = 0;
    for (int p = 0; p < npasses; p++) {
        pe[p] = uhalf_off(pass_levels[p].first);
        yacc = std::max(yacc, uhalf_off(pass_levels[p].second + 1) - uhalf_off(pass_levels[p].first));
    }
    // pass_elem[p+1] must be the END of pass p: passes run from the top level down, so ends are stored beside the starts
    std::vector<int> pass_elem(2 * npasses, 0);
    for (int p = 0; p < npasses; p++) { pass_elem[2 * p] = pe[p]; pass_elem[2 * p + 1] = uhalf_off(pass_levels[p].second + 1); }
    int rc = 0;
    if ((rc = upload(h->d_ybstream, stream))) return rc;
    if ((rc = upload(h->d_ybwrange, wrange))) return rc;
    if ((rc = upload(h->d_ybpass, pass_elem))) return rc;
    // rows above the centre of a middle column: Y[C - ma][C/2] = (-1)^(ma - C/2) conj(Y[ma][C/2]); entry = mirror element << 1 | odd sign
    std::vector<int> mirror(h->tab.nelem, -1);
    for (int C = 0; C <= tj; C += 2)
        for (int ma = C / 2 + 1; ma <= C; ma++) {
            const int e = uhalf_off(C) + (C / 2) * (C + 1) + ma, me = uhalf_off(C) + (C / 2) * (C + 1) + (C - ma);
            mirror[e] = (me << 1) | ((ma - C / 2) & 1);
        }
    if ((rc = upload(h->d_ybmirror, mirror))) return rc;
    h->yb_npasses = npasses;
    h->yb_yacc = yacc;
    CUDA_TRY(cudaFuncSetAttribute(compute_yi_fix_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)compute_yi_fix_smem_bytes(uhalf_size(kFullTileTwoJ), std::max(64, uhalf_off(kFullTileTwoJ + 1) - uhalf_off(kFullTileTwoJ)))));
    CUDA_TRY(cudaFuncSetAttribute(compute_yi_block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)compute_yi_block_smem_bytes(uhalf_size(kFullTileTwoJ), triple_count(kFullTileTwoJ), std::max(64, uhalf_off(kFullTileTwoJ + 1) - uhalf_off(kFullTileTwoJ)))));
    return 0;
}

// row f3 for the slab [z0, z1): tile binning -> compute_ui -> compute_yi (beta in, Y out) -> compute_dedr (adds into gout)
int run_slab_force(mala_snap *h, int z0, int z1, const double *beta, double *gout, cudaStream_t st) {
    if (z1 <= z0) return 0;
    choose_tiles(h, z0, z1);
    GridGeom &g = h->geom;
    h->cand_cap = candidate_bound(h);
    if (h->cand_cap < 0) return fail(MALA_SNAP_EINVAL, "more than 2^24 candidate atoms per tile; use a finer cell or smaller z-slabs");
    const long long total_tiles = h->total_tiles;
    if (total_tiles > 2000000000LL) return fail(MALA_SNAP_EINVAL, "slab has too many tiles; use smaller z-slabs");
    const size_t per_tile = (size_t)2 * h->sc.nelem * 32 * sizeof(double2) + (size_t)h->cand_cap * sizeof(int) + 2 * sizeof(int);
    const size_t budget = (size_t)std::max<long long>(h->workspace_mb, 1) << 20;
    long long chunk_tiles = (long long)std::max<size_t>(budget / per_tile, (size_t)h->num_sms);
    chunk_tiles = std::min(chunk_tiles, total_tiles);
    if (h->d_utot.reserve((size_t)chunk_tiles * h->sc.nelem * 32, st, true) || h->d_ytot.reserve((size_t)chunk_tiles * h->sc.nelem * 32, st, true) ||
        h->d_cand.reserve((size_t)chunk_tiles * h->cand_cap, st, true) || h->d_ncand.reserve(chunk_tiles, st, true) ||
        h->d_active.reserve(chunk_tiles, st, true) || h->d_counters.reserve(4, st, true))
        return fail(MALA_SNAP_ENOMEM, "cudaMallocAsync (workspace) failed");
    h->stats[4] = h->cand_cap;
    h->stats[5] = (long long)(per_tile * (size_t)chunk_tiles);
    const DeviceTables tb = h->tables();
    for (long long t0 = 0; t0 < total_tiles; t0 += chunk_tiles) {
        ChunkBuffers cb{};
        cb.ghosts = h->d_ghosts[h->cur].p; cb.cell_start = h->d_cell_start[h->cur].p;
        cb.cand = h->d_cand.p; cb.ncand = h->d_ncand.p; cb.active = h->d_active.p; cb.counters = h->d_counters.p;
        cb.status = h->d_status.p; cb.utot = h->d_utot.p; cb.cand_cap = h->cand_cap;
        cb.tile_begin = (int)t0;
        cb.ntiles = (int)std::min(chunk_tiles, total_tiles - t0);
        CUDA_TRY(cudaMemsetAsync(cb.counters, 0, 4 * sizeof(int), st));
        const int bin_blocks = (cb.ntiles + 7) / 8;
        {
            TimedSpan span(h, st, kKindBin);
            tile_bin_kernel<<<bin_blocks, 256, 0, st>>>(g, h->sc, tb, cb, nullptr);
        }
        CUDA_TRY(cudaGetLastError());
        const int grid2 = std::max(1, std::min(2 * h->num_sms, 2 * cb.ntiles));
        {
            TimedSpan span(h, st, kKindUi);
            if (h->use_ui_dft()) {
                if (int rc = launch_ui_dft(h, g, tb, cb, st)) return rc;
            } else if (h->twojmax == kFullTileTwoJ)
                compute_ui_kernel<kFullTileTwoJ, true><<<grid2, (kFullTileTwoJ / 2 + 1) * 32, compute_ui_smem_bytes(kFullTileTwoJ), st>>>(g, h->sc, tb, cb);
            else
                compute_ui_kernel<kFullTileTwoJ, false><<<grid2, (kFullTileTwoJ / 2 + 1) * 32, compute_ui_smem_bytes(kFullTileTwoJ), st>>>(g, h->sc, tb, cb);
        }
        CUDA_TRY(cudaGetLastError());
        {
            TimedSpan span(h, st, kKindZi);   // reported in the compute_zi_bi slot: the same kind of contraction
            const int grid = std::max(1, std::min(h->num_sms, cb.ntiles));
            if (h->yi_impl == 0 || h->yi_impl == 2) {   // the block kernel with Y in fixed point (snap_yi_fix.cuh)
                // |Z^C_AB component| <= (sum |CG|)^2 * 2 max|U component|^2 with sum |CG| <= sqrt(twojmax + 1); at most three terms per
                // bispectrum component, coefficients <= twojmax + 1
                const double bound = 2.0 * (h->twojmax + 1) * 3.0 * (h->twojmax + 1);
                compute_yi_fix_kernel<<<grid, kBlkWarps * 32, compute_yi_fix_smem_bytes(h->sc.nelem, h->yb_yacc), st>>>(g, h->sc, h->yblk_tables(), cb, beta,
                                                                                                                     h->d_ytot.p, bound);
            } else if (h->yi_impl == 1)
                compute_yi_kernel<<<grid, kYiWarps * 32, compute_yi_smem_bytes(h->sc.nelem, h->sc.ntriples), st>>>(g, h->sc, h->force_tables(), cb, beta,
                                                                                                                    h->d_ytot.p);
            else   // the same contraction on the register-tiled block machinery (snap_yi_block.cuh)
                compute_yi_block_kernel<<<grid, kBlkWarps * 32, compute_yi_block_smem_bytes(h->sc.nelem, h->sc.ntriples, h->yb_yacc), st>>>(
                    g, h->sc, h->yblk_tables(), cb, beta, h->d_ytot.p);
        }
        CUDA_TRY(cudaGetLastError());
        {
            TimedSpan span(h, st, kKindOther);
            if (h->dedr_impl == 0 && h->twojmax >= 1) {   // sampling form (snap_dedr_dft.cuh): whole tiles, twojmax + 1 warps
                switch (h->twojmax) {
#define MALA_DD_CASE(TJ) \
    case TJ: \
        compute_dedr_dft_kernel<TJ><<<std::max(1, std::min(dft_ctas(TJ) * h->num_sms, cb.ntiles)), (TJ + 1) * 32, compute_dedr_dft_smem_bytes<TJ>(), st>>>( \
            g, h->sc, tb, cb, h->d_ytot.p, gout); \
        break;
                    MALA_DD_CASE(1) MALA_DD_CASE(2) MALA_DD_CASE(3) MALA_DD_CASE(4) MALA_DD_CASE(5)
                    MALA_DD_CASE(6) MALA_DD_CASE(7) MALA_DD_CASE(8) MALA_DD_CASE(9) MALA_DD_CASE(10)
#undef MALA_DD_CASE
                    default: break;
                }
            } else
                compute_dedr_kernel<kFullTileTwoJ><<<grid2, (kFullTileTwoJ / 2 + 1) * 32, compute_dedr_smem_bytes(kFullTileTwoJ), st>>>(g, h->sc, tb, cb,
                                                                                                                                     h->d_ytot.p, gout);
        }
        CUDA_TRY(cudaGetLastError());
        h->stats[0] += 4;
        h->stats[1]++;
    }
    h->stats[2] += total_tiles;
    h->stats[6] += (long long)g.nx * g.ny * (z1 - z0);
    return 0;
}

int finish_call(mala_snap *h, cudaStream_t st) {
    // the status word travels back with every call: one 4-byte copy into pinned memory, ordered before ev_call_done
    CUDA_TRY(cudaMemcpyAsync(h->h_status, h->d_status.p, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaEventRecord(h->ev_call_done[h->cur], st));
    h->call_done_valid[h->cur] = true;
    return 0;
}

// Status of the calls issued so far.  wait = false: looks only at calls that have already drained (used at the start of an
// enqueue-only call, which must not block); wait = true: waits for the last call first.  A raised bit is sticky.
int check_status(mala_snap *h, bool wait) {
    const int last = (int)((h->ncalls + 1ull) & 1ull);  // buffer set of the most recent call
    if (h->ncalls > 0 && h->call_done_valid[last]) {
        cudaError_t e = wait ? cudaEventSynchronize(h->ev_call_done[last]) : cudaEventQuery(h->ev_call_done[last]);
        if (e == cudaSuccess) h->sticky_status |= *(volatile int *)h->h_status;
        else if (e != cudaErrorNotReady) return fail(MALA_SNAP_ECUDA, std::string("status check: ") + cudaGetErrorString(e));
        else cudaGetLastError();
    }
    if (h->sticky_status & kStatusCandOverflow)
        return fail(MALA_SNAP_ECUDA, "candidate overflow: tile_bin_kernel truncated a neighbor-candidate list in an earlier call on this "
                                     "handle (its results are invalid); the host bound was violated");
    return 0;
}

}  // namespace

// FP64 FMA-pipe probe: kDfmaChains independent dependent-chains per thread, nothing else in the loop
constexpr int kDfmaChains = 8;
__global__ void __launch_bounds__(256) dfma_probe_kernel(double *sink, int iters, double m) {
    double acc[kDfmaChains];
#pragma unroll
    for (int k = 0; k < kDfmaChains; k++) acc[k] = 1e-3 * (threadIdx.x + k);
    const double c = 1e-7;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int k = 0; k < kDfmaChains; k++) acc[k] = fma(acc[k], m, c);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < kDfmaChains; k++) s += acc[k];
    if (s == 123.456) sink[threadIdx.x] = s;  // never true; keeps the chains alive
}

// =============================================================================================================
// C ABI
// =============================================================================================================
extern "C" {

const char *mala_last_error(void) { return g_last_error.c_str(); }

double mala_snap_clebsch_gordan(int J1, int M1, int J2, int M2, int J, int M) { return clebsch_gordan(J1, M1, J2, M2, J, M); }

int mala_snap_create(mala_snap_t **handle, int twojmax, double rcutfac, double rfac0, double rmin0, double wself, int ntypes,
                     const double *radelem, const double *wj) {
    if (!handle) return fail(MALA_SNAP_EINVAL, "handle is NULL");
    *handle = nullptr;
    if (twojmax < 0 || twojmax > MALA_SNAP_MAX_TWOJMAX) return fail(MALA_SNAP_EINVAL, "twojmax outside [0, 14]");
    static_assert(MALA_SNAP_MAX_TWOJMAX == kMaxTwoJ, "header and kernels disagree on the largest twojmax");
    if (!(rcutfac > 0.0) || !std::isfinite(rcutfac)) return fail(MALA_SNAP_EINVAL, "rcutfac must be positive");
    if (!(rfac0 > 0.0) || !(rfac0 <= 1.0)) return fail(MALA_SNAP_EINVAL, "rfac0 must lie in (0, 1]");
    if (!std::isfinite(wself)) return fail(MALA_SNAP_EINVAL, "wself is not finite");
    if (ntypes < 1 || !radelem || !wj) return fail(MALA_SNAP_EINVAL, "ntypes < 1 or radelem/wj is NULL");
    mala_snap *h = new (std::nothrow) mala_snap();
    if (!h) return fail(MALA_SNAP_ENOMEM, "out of host memory");
    h->twojmax = twojmax; h->ntypes = ntypes; h->rcutfac = rcutfac; h->rfac0 = rfac0; h->rmin0 = rmin0; h->wself = wself;
    double rcutmin = 1e300;
    for (int t = 0; t < ntypes; t++) {
        if (!(radelem[t] > 0.0) || !std::isfinite(radelem[t]) || !std::isfinite(wj[t])) {
            delete h;
            return fail(MALA_SNAP_EINVAL, "radelem must be positive and wj finite");
        }
        h->rcut.push_back(2.0 * rcutfac * radelem[t]);
        h->wj.push_back(wj[t]);
        h->rcutmax = std::max(h->rcutmax, h->rcut.back());
        rcutmin = std::min(rcutmin, h->rcut.back());
    }
    if (!(rmin0 >= 0.0) || !(rmin0 < rcutmin)) {
        delete h;
        return fail(MALA_SNAP_EINVAL, "rmin0 must lie in [0, min rcut)");
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        delete h;
        return fail(MALA_SNAP_ECUDA, "no CUDA device: this library has no CPU fallback");
    }
    int rc = 0;
    auto body = [&]() -> int {
        CUDA_TRY(cudaGetDevice(&h->device));
        cudaDeviceProp prop;
        CUDA_TRY(cudaGetDeviceProperties(&prop, h->device));
        if (prop.major < 10) return fail(MALA_SNAP_ECUDA, "device is not sm_100 class (kernels are built for sm_100a only)");
        h->num_sms = prop.multiProcessorCount;
        CUDA_TRY(cudaGetSymbolAddress((void **)&h->static_scratch, g_static_scratch));
        h->tab = build_tables(twojmax);
        h->sc.twojmax = twojmax; h->sc.ntriples = h->tab.ntriples; h->sc.nelem = h->tab.nelem; h->sc.ntypes = ntypes;
        h->sc.rfac0 = rfac0; h->sc.rmin0 = rmin0; h->sc.wself = wself;
        if ((rc = upload(h->d_triples, h->tab.triples))) return rc;
        if ((rc = upload(h->d_cg, h->tab.cg))) return rc;
        if ((rc = upload(h->d_unorm, h->tab.unorm))) return rc;
        if ((rc = upload(h->d_udiag, h->tab.udiag))) return rc;
        if ((rc = upload(h->d_order, h->tab.order))) return rc;
        if ((rc = upload(h->d_rcut, h->rcut))) return rc;
        if ((rc = upload(h->d_w, h->wj))) return rc;
        if (twojmax == kSpecTJ) {
            if ((int)h->tab.cg.size() != kSpecCG || h->tab.ntriples != kSpecNT) return fail(MALA_SNAP_ECUDA, "internal: table size mismatch");
            CUDA_TRY(cudaMemcpyToSymbol(c_cg_spec, h->tab.cg.data(), sizeof(double) * kSpecCG));
            CUDA_TRY(cudaMemcpyToSymbol(c_order_spec, h->tab.order.data(), sizeof(int) * kSpecNT));
            {
                static double sq[kSpecTJ + 1][kSpecTJ + 1], isq[kSpecTJ + 1][kSpecTJ + 1];
                for (int J = 0; J <= kSpecTJ; J++)
                    for (int m = 0; m <= kSpecTJ; m++) {
                        sq[J][m] = (m <= J) ? std::sqrt(binom_d(J, m)) : 0.0;
                        isq[J][m] = (m <= J) ? 1.0 / std::sqrt(binom_d(J, m)) : 0.0;
                    }
                CUDA_TRY(cudaMemcpyToSymbol(c_sqbin, sq, sizeof(sq)));
                CUDA_TRY(cudaMemcpyToSymbol(c_isqbin, isq, sizeof(isq)));
            }
            // deal the (mb, mb1) items of every triple to the warps as contiguous runs (snap_zi_coop.cuh "Schedule"):
            // run boundaries are placed so that every warp's cumulative cost (product terms plus a fixed per-item
            // overhead) tracks the mean over the whole tile, not only within one triple
            static unsigned short sched[kSpecNT][kCoopWarps][2];
            // The warps form `teams` teams; a triple goes to the team with the smallest load (triples come in order of
            // decreasing cost) and its items are dealt to that team's warps as contiguous runs whose boundaries keep
            // every warp's cumulative cost on the team mean.  More teams = longer runs per call but more instruction
            // streams in flight: measured on B200 (config 2) 1 team 30.8 ms, 2 teams 28.9 ms, 3 teams 35.7 ms,
            // 4 teams 52.9 ms -- the 32 KB instruction cache holds two loop bodies, not three.
            // The CTA-wide barrier at the end of every reduction group (kCoopGroup triples) makes the group, not the tile,
            // the unit to balance: per group the triples are split between the teams so that the team totals are as equal
            // as possible (all subsets are tried), and the running loads that place the run boundaries start from zero
            // in every group.  Model idle time at the barriers: 15 % with tile-wide balancing, 6 % with this.
            const double kItemOverhead = 8.0;
            const int teams = kCoopTeams;  // compile-time: the kernel's reduction sums kTeamWarps partials
            const int tw = kCoopWarps / teams;  // warps per team
            std::vector<int> pos_team(kSpecNT, 0);
            std::vector<std::vector<double>> icost(kSpecNT);
            std::vector<double> tsum(kSpecNT, 0.0);
            for (int pos = 0; pos < kSpecNT; pos++) {
                const int t = h->tab.order[pos];
                const int J1 = h->tab.triples[4 * t], J2 = h->tab.triples[4 * t + 1], J = h->tab.triples[4 * t + 2];
                for (int mb = 0; mb <= J / 2; mb++) {
                    const int nb = item_hi(J1, J2, J, mb) - item_lo(J1, J2, J, mb) + 1;
                    for (int i = 0; i < nb; i++) icost[pos].push_back(item_terms(J1, J2, J, mb) + kItemOverhead);
                }
                for (double c : icost[pos]) tsum[pos] += c;
            }
            for (int g0 = 0; g0 < kSpecNT; g0 += kCoopGroup) {
                const int gn = std::min(kCoopGroup, kSpecNT - g0);
                // team of every triple of the group
                if (teams == 2 && gn <= 16) {
                    double total = 0.0, best = 1e300;
                    for (int i = 0; i < gn; i++) total += tsum[g0 + i];
                    unsigned best_mask = 0;
                    for (unsigned mask = 0; mask < (1u << gn); mask++) {
                        double a = 0.0;
                        for (int i = 0; i < gn; i++)
                            if (mask >> i & 1u) a += tsum[g0 + i];
                        if (std::fabs(2.0 * a - total) < best) { best = std::fabs(2.0 * a - total); best_mask = mask; }
                    }
                    for (int i = 0; i < gn; i++) pos_team[g0 + i] = (int)(best_mask >> i & 1u);
                } else {
                    std::vector<double> tl(teams, 0.0);
                    for (int i = 0; i < gn; i++) {
                        int team = 0;
                        for (int k = 1; k < teams; k++)
                            if (tl[k] < tl[team]) team = k;
                        tl[team] += tsum[g0 + i];
                        pos_team[g0 + i] = team;
                    }
                }
                std::vector<double> load(kCoopWarps, 0.0), team_load(teams, 0.0);
                for (int pos = g0; pos < g0 + gn; pos++) {
                    const std::vector<double> &cost = icost[pos];
                    const int n = (int)cost.size(), team = pos_team[pos];
                    team_load[team] += tsum[pos];
                    const double target = team_load[team] / tw;
                    for (int w = 0; w < kCoopWarps; w++) sched[pos][w][0] = sched[pos][w][1] = 0;
                    int i = 0;
                    for (int k = 0; k < tw; k++) {
                        const int w = team * tw + k;
                        const int begin = i;
                        double acc = 0.0;
                        if (k == tw - 1) {
                            for (; i < n; i++) acc += cost[i];
                        } else {
                            const double want = target - load[w];
                            while (i < n && acc + 0.5 * cost[i] <= want) acc += cost[i++];
                        }
                        load[w] += acc;
                        sched[pos][w][0] = (unsigned short)begin;
                        sched[pos][w][1] = (unsigned short)i;
                    }
                }
            }
            // flatten into one work list per warp (snap_zi_coop.cuh, c_wlist)
            static unsigned int wlist[kCoopWarps][kListMax];
            int wn[kCoopWarps];
            for (int w = 0; w < kCoopWarps; w++) wn[w] = 0;
            for (int pos = 0; pos < kSpecNT; pos++) {
                const int t = h->tab.order[pos];
                const int k = pos % kCoopGroup, buf = (pos / kCoopGroup) & 1;
                const int team = pos_team[pos];
                for (int q = 0; q < tw; q++) {
                    const int w = team * tw + q;
                    wlist[w][wn[w]++] = ((unsigned)(buf * kCoopGroup + k) << 23) | ((unsigned)sched[pos][w][1] << 15) |
                                        ((unsigned)sched[pos][w][0] << 7) | (unsigned)t;
                }
                if (k == kCoopGroup - 1 || pos == kSpecNT - 1)
                    for (int w = 0; w < kCoopWarps; w++)
                        wlist[w][wn[w]++] = 0x80000000u | ((unsigned)(pos - k) << 8) | ((unsigned)buf << 4) | (unsigned)k;
            }
            for (int w = 0; w < kCoopWarps; w++) {
                if (wn[w] >= kListMax) return fail(MALA_SNAP_ECUDA, "internal: work list overflow");
                for (int i = wn[w]; i < kListMax; i++) wlist[w][i] = 0xffffffffu;
            }
            CUDA_TRY(cudaMemcpyToSymbol(c_wlist, wlist, sizeof(wlist)));
        }
        if ((rc = build_diag_schedule(h))) return rc;
        if ((rc = build_block_schedule(h))) return rc;
        if ((rc = set_kernel_attributes(h))) return rc;
        if (h->d_status.reserve(1)) return fail(MALA_SNAP_ENOMEM, "cudaMalloc (status) failed");
        CUDA_TRY(cudaMemset(h->d_status.p, 0, sizeof(int)));
        CUDA_TRY(cudaMallocHost((void **)&h->h_status, sizeof(int)));
        *h->h_status = 0;
        {   // keep freed workspace blocks in the stream-ordered pool instead of returning them to the driver at every sync
            cudaMemPool_t pool = nullptr;
            if (cudaDeviceGetDefaultMemPool(&pool, h->device) == cudaSuccess) {
                unsigned long long keep = ~0ull;
                cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
            }
            cudaGetLastError();
        }
        CUDA_TRY(cudaStreamCreateWithFlags(&h->upload_stream, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
        CUDA_TRY(cudaEventCreateWithFlags(&h->ev_upload, cudaEventDisableTiming));
        for (int i = 0; i < 2; i++) {
            CUDA_TRY(cudaEventCreateWithFlags(&h->ev_call_done[i], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&h->ev_copied[i], cudaEventDisableTiming));
        }
        return compute_bconst(h);
    };
    rc = body();
    if (rc) {
        const std::string keep = g_last_error;
        mala_snap_destroy(h);
        g_last_error = keep;
        return rc;
    }
    *handle = h;
    return MALA_SNAP_OK;
}

int mala_snap_ncomp(const mala_snap_t *h) {
    if (!h) return fail(MALA_SNAP_EINVAL, "handle is NULL");
    return h->sc.ntriples;
}

int mala_snap_triples(const mala_snap_t *h, int *j1j2j) {
    if (!h || !j1j2j) return fail(MALA_SNAP_EINVAL, "handle or output is NULL");
    for (int t = 0; t < h->tab.ntriples; t++)
        for (int k = 0; k < 3; k++) j1j2j[3 * t + k] = h->tab.triples[4 * t + k];
    return MALA_SNAP_OK;
}

int mala_snap_set_option(mala_snap_t *h, const char *name, long long value) {
    if (!h || !name) return fail(MALA_SNAP_EINVAL, "handle or name is NULL");
    const std::string n(name);
    if (n == "dedr_impl") {
        if (value < 0 || value > 1) return fail(MALA_SNAP_EINVAL, "dedr_impl must be 0 or 1");
        h->dedr_impl = (int)value;
        return MALA_SNAP_OK;
    }
    if (n == "yi_impl") {
        if (value < 0 || value > 3) return fail(MALA_SNAP_EINVAL, "yi_impl must be 0 .. 3");
        h->yi_impl = (int)value;
        return MALA_SNAP_OK;
    }
    if (n == "ui_impl") {
        if (value < 0 || value > 3) return fail(MALA_SNAP_EINVAL, "ui_impl must be 0 .. 3");
        if (value == 3 && h->twojmax < 8) return fail(MALA_SNAP_EINVAL, "the pipelined sampling compute_ui kernel covers twojmax 8..14");
        if (value == 2 && (h->twojmax < 1 || h->twojmax > kFullTileTwoJ)) return fail(MALA_SNAP_EINVAL, "the sampling compute_ui kernel covers twojmax 1..10");
        h->ui_impl = (int)value;
        return MALA_SNAP_OK;
    }
    if (n == "zi_impl") {
        if (value < 0 || value > 4) return fail(MALA_SNAP_EINVAL, "zi_impl must be 0 .. 4");
        if (value == 2 && h->twojmax != kSpecTJ) return fail(MALA_SNAP_EINVAL, "the specialised kernel exists for twojmax = 10 only");
        if ((value == 1 || value == 2) && h->half_tiles())
            return fail(MALA_SNAP_EINVAL, "twojmax > 10 runs on half tiles: only the anti-diagonal and the block kernel (zi_impl 0, 3, 4) support them");
        if (value == 4 && !h->blk_ready) return fail(MALA_SNAP_EINVAL, "the block kernel has no tables for this handle");
        h->zi_impl = (int)value;
        return compute_bconst(h);
    }
    if (n == "timing") {
        h->timing = (value != 0);
        return MALA_SNAP_OK;
    }
    if (n == "workspace_mb") {
        if (value < 1) return fail(MALA_SNAP_EINVAL, "workspace_mb must be >= 1");
        h->workspace_mb = value;
        return MALA_SNAP_OK;
    }
    if (n == "cand_cap_limit") {  // test hook: see mala_snap.h
        if (value < 0 || value > (1 << 24)) return fail(MALA_SNAP_EINVAL, "cand_cap_limit must lie in [0, 2^24]");
        h->cand_cap_limit = (int)value;
        return MALA_SNAP_OK;
    }
    if (n == "host_chunk_mb") {
        if (value < 1) return fail(MALA_SNAP_EINVAL, "host_chunk_mb must be >= 1");
        h->host_chunk_mb = value;
        return MALA_SNAP_OK;
    }
    return fail(MALA_SNAP_EINVAL, "unknown option: " + n);
}

int mala_snap_last_stats(mala_snap_t *h, long long stats[8]) {
    if (!h || !stats) return fail(MALA_SNAP_EINVAL, "handle or stats is NULL");
    const int rc = check_status(h, true);  // waits for the last call: its status word is part of the answer
    h->stats[7] = h->sticky_status;
    for (int i = 0; i < 8; i++) stats[i] = h->stats[i];
    return rc;
}

int mala_snap_kernel_times(mala_snap_t *h, double ms[4], long long launches[4]) {
    if (!h || !ms || !launches) return fail(MALA_SNAP_EINVAL, "handle or output is NULL");
    for (int k = 0; k < 4; k++) { ms[k] = 0.0; launches[k] = 0; }
    for (const mala_snap::Span &s : h->spans) {
        CUDA_TRY(cudaEventSynchronize(s.b));
        float t = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&t, s.a, s.b));
        ms[s.kind] += (double)t;
        launches[s.kind]++;
    }
    return MALA_SNAP_OK;
}

const char *mala_snap_zi_kernel(const mala_snap_t *h) {
    if (!h) return "";
    if (h->use_block()) return "compute_zi_bi_block_kernel";
    if (h->half_tiles()) return "compute_zi_bi_diag_half_kernel";
    return h->use_diag() ? "compute_zi_bi_diag_kernel" : (h->use_spec() ? "compute_zi_bi_coop_kernel" : "compute_zi_bi_generic_kernel");
}

int mala_snap_fp64_peak(double *tflops, double *sm_mhz_effective, void *cuda_stream) {
    if (!tflops) return fail(MALA_SNAP_EINVAL, "tflops is NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double *sink = nullptr;
    CUDA_TRY(cudaMalloc((void **)&sink, sizeof(double) * 1024));
    cudaEvent_t a = nullptr, b = nullptr;
    cudaEventCreate(&a); cudaEventCreate(&b);
    const int blocks = sms * 4, threads = 256, iters = 1 << 15;
    double best = 0.0;
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 6 && e == cudaSuccess; rep++) {
        cudaEventRecord(a, st);
        dfma_probe_kernel<<<blocks, threads, 0, st>>>(sink, iters, 1.0 + 1e-9 * rep);
        cudaEventRecord(b, st);
        e = cudaEventSynchronize(b);
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, a, b);
        const double flop = 2.0 * kDfmaChains * (double)iters * blocks * threads;
        if (rep > 0 && t > 0.f) best = std::max(best, flop / (t * 1e-3) / 1e12);
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(sink);
    if (e != cudaSuccess) return fail(MALA_SNAP_ECUDA, std::string("fp64 probe: ") + cudaGetErrorString(e));
    *tflops = best;
    // clock the rate implies if every SM retires 64 DFMA per cycle
    if (sm_mhz_effective) *sm_mhz_effective = best * 1e12 / (2.0 * 64.0 * sms) / 1e6;
    return MALA_SNAP_OK;
}

int mala_bispectrum_grid(mala_snap_t *h, int natoms, const double *pos, const int *types, const double box[9],
                         const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end, double *out,
                         void *cuda_stream) {
    const CallArgs a{natoms, pos, types, box, origin, pbc, ngrid, z_begin, z_end};
    int rc = validate(h, a, true, out);
    if (rc) return rc;
    if ((rc = check_status(h, false))) return rc;
    std::fill(h->stats, h->stats + 8, 0LL);
    if (z_end == z_begin) return MALA_SNAP_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = build_plan(h, a, st))) return rc;
    if ((rc = run_slab(h, z_begin, z_end, out, nullptr, st))) return rc;
    return finish_call(h, st);
}

int mala_bispectrum_grid_host(mala_snap_t *h, int natoms, const double *pos, const int *types, const double box[9],
                              const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end,
                              double *out_host, void *cuda_stream) {
    const CallArgs a{natoms, pos, types, box, origin, pbc, ngrid, z_begin, z_end};
    int rc = validate(h, a, true, out_host);
    if (rc) return rc;
    if ((rc = check_status(h, false))) return rc;
    std::fill(h->stats, h->stats + 8, 0LL);
    if (z_end == z_begin) return MALA_SNAP_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = build_plan(h, a, st))) return rc;
    const size_t plane = (size_t)ngrid[0] * ngrid[1] * h->sc.ntriples;  // doubles per z-plane
    const size_t budget = ((size_t)h->host_chunk_mb << 20) / sizeof(double);
    const int planes_max = (int)std::max<size_t>(1, std::min<size_t>(budget / std::max<size_t>(plane, 1), (size_t)(z_end - z_begin)));
    // The device->host copy of a chunk overlaps the kernels of the next one, so only the last chunk's copy is exposed, and
    // every chunk costs the tails of its three persistent kernels.  Hence chunks that shrink: a third of what is left, in whole
    // tile layers (multiples of eight planes), at least eight planes, at most what a staging buffer holds -- config 2: 24, 16,
    // 16, 8, 8, 8, 8, 2 planes (equal chunks of 8 planes: 23.5 ms end to end).  Small outputs go in one piece.
    const size_t total = plane * (size_t)(z_end - z_begin);
    const bool split = total * sizeof(double) > ((size_t)96 << 20);
    auto next_planes = [&](int left) {
        int p = planes_max;
        if (split) p = std::min(p, std::max(8, left / 3));
        if (p >= 8) p = p / 8 * 8;  // whole tiles for every tile shape
        return std::min(p, left);
    };
    for (int b = 0; b < 2; b++)
        if (h->d_stage[b].reserve(plane * (size_t)next_planes(z_end - z_begin), st, true)) return fail(MALA_SNAP_ENOMEM, "cudaMallocAsync (staging) failed");
    bool used[2] = {false, false};
    int i = 0;
    for (int z = z_begin; z < z_end; i++) {
        const int b = i & 1;
        const int ze = z + next_planes(z_end - z);
        if (used[b]) CUDA_TRY(cudaStreamWaitEvent(st, h->ev_copied[b], 0));
        if ((rc = run_slab(h, z, ze, h->d_stage[b].p, nullptr, st))) return rc;
        CUDA_TRY(cudaEventRecord(h->ev_done[b], st));
        CUDA_TRY(cudaStreamWaitEvent(h->copy_stream, h->ev_done[b], 0));
        CUDA_TRY(cudaMemcpyAsync(out_host + (size_t)(z - z_begin) * plane, h->d_stage[b].p, (size_t)(ze - z) * plane * sizeof(double),
                                 cudaMemcpyDeviceToHost, h->copy_stream));
        CUDA_TRY(cudaEventRecord(h->ev_copied[b], h->copy_stream));
        used[b] = true;
        z = ze;
    }
    if ((rc = finish_call(h, st))) return rc;
    CUDA_TRY(cudaStreamSynchronize(h->copy_stream));
    CUDA_TRY(cudaStreamSynchronize(st));
    return check_status(h, true);
}

int mala_bispectrum_ldos_grid(mala_snap_t *h, mala_mlp_t *net, int natoms, const double *pos, const int *types, const double box[9],
                              const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end, float *ldos,
                              void *cuda_stream) {
    const CallArgs a{natoms, pos, types, box, origin, pbc, ngrid, z_begin, z_end};
    int rc = validate(h, a, true, ldos);
    if (rc) return rc;
    if (!net) return fail(MALA_SNAP_EINVAL, "net is NULL");
    if (mlp_in_width(net) != h->sc.ntriples)
        return fail(MALA_SNAP_EINVAL, "the network's input width differs from the number of bispectrum components of this handle");
    if ((rc = check_status(h, false))) return rc;
    std::fill(h->stats, h->stats + 8, 0LL);
    if (z_end == z_begin) return MALA_SNAP_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = build_plan(h, a, st))) return rc;
    if ((rc = run_slab(h, z_begin, z_end, nullptr, nullptr, st, net, ldos))) return rc;
    return finish_call(h, st);
}

int mala_bispectrum_force_adjoint(mala_snap_t *h, int natoms, const double *pos, const int *types, const double box[9],
                                  const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end, const double *beta,
                                  double *g, void *cuda_stream) {
    const CallArgs a{natoms, pos, types, box, origin, pbc, ngrid, z_begin, z_end};
    int rc = validate(h, a, true, beta);
    if (rc) return rc;
    if (natoms > 0 && !g) return fail(MALA_SNAP_EINVAL, "g is NULL");
    if (h->half_tiles()) return fail(MALA_SNAP_EINVAL, "mala_bispectrum_force_adjoint supports twojmax <= 10");
    if ((rc = check_status(h, false))) return rc;
    std::fill(h->stats, h->stats + 8, 0LL);
    if (z_end == z_begin || natoms == 0) return MALA_SNAP_OK;
    if ((rc = build_force_tables(h))) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = build_plan(h, a, st))) return rc;
    if ((rc = run_slab_force(h, z_begin, z_end, beta, g, st))) return rc;
    return finish_call(h, st);
}

int mala_gaussian_grid(mala_snap_t *h, double sigma, int natoms, const double *pos, const int *types, const double box[9],
                       const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end, double *out,
                       void *cuda_stream) {
    const CallArgs a{natoms, pos, types, box, origin, pbc, ngrid, z_begin, z_end};
    int rc = validate(h, a, true, out);
    if (rc) return rc;
    if ((rc = check_status(h, false))) return rc;
    if (!(sigma > 0.0) || !std::isfinite(sigma)) return fail(MALA_SNAP_EINVAL, "sigma must be positive");
    if (h->ntypes > kGaussMaxTypes) return fail(MALA_SNAP_EINVAL, "mala_gaussian_grid supports at most 4 atom types");
    std::fill(h->stats, h->stats + 8, 0LL);
    if (z_end == z_begin) return MALA_SNAP_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = build_plan(h, a, st))) return rc;
    if ((rc = run_slab_gauss(h, z_begin, z_end, sigma, out, st))) return rc;
    return finish_call(h, st);
}

int mala_gaussian_grid_static(mala_snap_t *h, double sigma, int natoms, const double *pos, const int *types, const double box[9],
                              const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end, double *out,
                              void *cuda_stream) {
    const CallArgs a{natoms, pos, types, box, origin, pbc, ngrid, z_begin, z_end};
    int rc = validate(h, a, true, out);
    if (rc) return rc;
    if ((rc = check_status(h, false))) return rc;
    if (!(sigma > 0.0) || !std::isfinite(sigma)) return fail(MALA_SNAP_EINVAL, "sigma must be positive");
    if (h->ntypes > kGaussMaxTypes) return fail(MALA_SNAP_EINVAL, "mala_gaussian_grid_static supports at most 4 atom types");
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev != h->device || !h->static_scratch) return fail(MALA_SNAP_EINVAL, "mala_gaussian_grid_static: the handle's device is not current");
    std::fill(h->stats, h->stats + 8, 0LL);
    if (z_end == z_begin) return MALA_SNAP_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    std::vector<Ghost> sorted;   // host memory only
    std::vector<int> start;
    if ((rc = plan_host(h, a, sorted, start))) return rc;
    const size_t ng = sorted.size(), ncell1 = start.size();
    h->h_cell_start.swap(start);   // candidate_bound reads the cell counts of this call
    choose_tiles(h, z_begin, z_end);
    const GridGeom &g = h->geom;
    h->cand_cap = candidate_bound(h);
    if (h->cand_cap < 0) return fail(MALA_SNAP_EINVAL, "more than 2^24 candidate atoms per tile; use a finer cell or smaller z-slabs");
    const long long total_tiles = h->total_tiles;
    if (total_tiles > 2000000000LL) return fail(MALA_SNAP_EINVAL, "slab has too many tiles; use smaller z-slabs");
    // carve the static array: ghosts | cell starts | counters | per-tile lists of one chunk (every piece 256-byte aligned)
    auto up = [](size_t n) { return (n + 255) & ~(size_t)255; };
    const size_t off_cells = up(std::max<size_t>(ng, 1) * sizeof(Ghost)), off_counters = off_cells + up(ncell1 * sizeof(int));
    const size_t off_tiles = off_counters + 256;
    const size_t per_tile = (size_t)h->cand_cap * sizeof(int) + 2 * sizeof(int);
    const long long want_tiles = std::min<long long>(total_tiles, h->num_sms);   // smallest chunk worth launching
    if (off_tiles + 768 + (size_t)want_tiles * per_tile > kStaticScratchBytes) {
        char msg[320];
        std::snprintf(msg, sizeof msg, "mala_gaussian_grid_static: %zu ghost atoms, %zu cells and the candidate lists of %lld tiles (%d entries "
                      "each) need %zu bytes, the static scratch holds %zu; use mala_gaussian_grid or smaller z-slabs",
                      ng, ncell1 - 1, want_tiles, h->cand_cap, off_tiles + 768 + (size_t)want_tiles * per_tile, kStaticScratchBytes);
        return fail(MALA_SNAP_EINVAL, msg);
    }
    const long long chunk_tiles = std::min<long long>(total_tiles, (long long)((kStaticScratchBytes - off_tiles - 768) / per_tile));
    unsigned char *base = h->static_scratch;
    Ghost *d_ghosts = reinterpret_cast<Ghost *>(base);
    int *d_cells = reinterpret_cast<int *>(base + off_cells), *d_counters = reinterpret_cast<int *>(base + off_counters);
    int *d_ncand = reinterpret_cast<int *>(base + off_tiles);
    int *d_active = reinterpret_cast<int *>(base + off_tiles + up((size_t)chunk_tiles * sizeof(int)));
    int *d_cand = reinterpret_cast<int *>(base + off_tiles + 2 * up((size_t)chunk_tiles * sizeof(int)));
    // calls on one handle are serialised whatever their streams (status word, geometry); the scratch itself is shared by every
    // handle of the device: calls that overlap on the GPU race (see include/mala_snap.h)
    if (h->call_done_valid[h->cur ^ 1]) CUDA_TRY(cudaStreamWaitEvent(st, h->ev_call_done[h->cur ^ 1], 0));
    if (h->call_done_valid[h->cur]) CUDA_TRY(cudaStreamWaitEvent(st, h->ev_call_done[h->cur], 0));
    // pageable sources: cudaMemcpyAsync returns once they are staged, so the vectors may die with this scope
    if (ng) CUDA_TRY(cudaMemcpyAsync(d_ghosts, sorted.data(), ng * sizeof(Ghost), cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(d_cells, h->h_cell_start.data(), ncell1 * sizeof(int), cudaMemcpyHostToDevice, st));
    h->stats[3] = (long long)ng;
    const double pi = 3.14159265358979323846;
    const double pref = 1.0 / (std::pow(2.0 * pi, 1.5) * sigma * sigma * sigma), inv2s2 = 1.0 / (2.0 * sigma * sigma);
    const DeviceTables tb = h->tables();
    for (long long t0 = 0; t0 < total_tiles; t0 += chunk_tiles) {
        ChunkBuffers cb{};
        cb.ghosts = d_ghosts; cb.cell_start = d_cells;
        cb.cand = d_cand; cb.ncand = d_ncand; cb.active = d_active; cb.counters = d_counters;
        cb.status = h->d_status.p;
        cb.cand_cap = h->cand_cap;
        cb.tile_begin = (int)t0;
        cb.ntiles = (int)std::min(chunk_tiles, total_tiles - t0);
        CUDA_TRY(cudaMemsetAsync(cb.counters, 0, 4 * sizeof(int), st));   // the array keeps the last call's contents
        const int blocks = (cb.ntiles + 7) / 8;
        tile_bin_kernel<<<blocks, 256, 0, st>>>(g, h->sc, tb, cb, nullptr);
        CUDA_TRY(cudaGetLastError());
        gaussian_grid_kernel<<<blocks, 256, 0, st>>>(g, h->sc, tb, cb, inv2s2, pref, out);
        CUDA_TRY(cudaGetLastError());
        h->stats[0] += 2;
        h->stats[1]++;
    }
    h->stats[2] += total_tiles;
    h->stats[4] = h->cand_cap;
    h->stats[6] += (long long)g.nx * g.ny * (z_end - z_begin);
    return finish_call(h, st);
}

int mala_snap_debug_utot(mala_snap_t *h, int natoms, const double *pos, const int *types, const double box[9],
                         const double origin[3], const int pbc[3], const int ngrid[3], int z_begin, int z_end, double *u_out,
                         void *cuda_stream) {
    const CallArgs a{natoms, pos, types, box, origin, pbc, ngrid, z_begin, z_end};
    int rc = validate(h, a, true, u_out);
    if (rc) return rc;
    if ((rc = check_status(h, false))) return rc;
    std::fill(h->stats, h->stats + 8, 0LL);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (z_end > z_begin) {
        if ((rc = build_plan(h, a, st))) return rc;
        if ((rc = run_slab(h, z_begin, z_end, nullptr, reinterpret_cast<double2 *>(u_out), st))) return rc;
        if ((rc = finish_call(h, st))) return rc;
    }
    CUDA_TRY(cudaStreamSynchronize(st));
    if ((rc = check_status(h, true))) return rc;
    return h->sc.nelem;
}

void mala_snap_destroy(mala_snap_t *h) {
    if (!h) return;
    cudaDeviceSynchronize();
    h->d_triples.release(); h->d_udiag.release(); h->d_order.release();
    h->d_cg.release(); h->d_unorm.release(); h->d_rcut.release(); h->d_w.release(); h->d_bconst.release();
    for (int i = 0; i < 2; i++) {
        h->d_ghosts[i].release(); h->d_cell_start[i].release(); h->d_stage[i].release();
        if (h->ev_call_done[i]) cudaEventDestroy(h->ev_call_done[i]);
        if (h->ev_done[i]) cudaEventDestroy(h->ev_done[i]);
        if (h->ev_copied[i]) cudaEventDestroy(h->ev_copied[i]);
    }
    h->d_cand.release(); h->d_ncand.release(); h->d_active.release(); h->d_counters.release(); h->d_utot.release(); h->d_uispill.release();
    h->d_status.release(); h->d_bstage.release();
    h->d_yterms.release(); h->d_ylevel.release(); h->d_yorder.release(); h->d_ycg.release(); h->d_yweight.release(); h->d_ytot.release();
    h->d_dcg.release(); h->d_dtriple.release(); h->d_dsched.release(); h->d_ditems.release();
    h->d_bstream.release(); h->d_bwrange.release(); h->d_btslot.release();
    h->d_ybstream.release(); h->d_ybwrange.release(); h->d_ybpass.release(); h->d_ybmirror.release();
    if (h->h_status) cudaFreeHost(h->h_status);
    for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
    if (h->ev_upload) cudaEventDestroy(h->ev_upload);
    if (h->upload_stream) cudaStreamDestroy(h->upload_stream);
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    cudaGetLastError();
    delete h;
}

}  // extern "C"
