// mala_mlp.cu -- the feed-forward network that maps a descriptor vector to the LDOS vector, point by point
// (Eqs. (18)-(19) PAPER.md:164-168), on the 5th-generation tensor cores.
//
// One persistent CTA per SM walks over row tiles of 128 grid points.  Per tile the layers run one after the other:
//     D[128][N_l] (TMEM, fp32) = A[128][K_l] (shared memory, TF32) x W_l[N_l][K_l]^T (shared memory ring, TF32)
// issued as tcgen05.mma.cta_group::1.kind::tf32 (M = 128, N = N_l, K = 8 per instruction) by one elected thread; the
// weights of the whole network stream through a 4-stage ring of 1-D bulk copies (cp.async.bulk + mbarrier) from an image
// that the host packed once in exactly the shared-memory order the MMA descriptors expect; four epilogue warps read the
// accumulator rows back with tcgen05.ld (thread = row = TMEM lane), add the bias, apply sigma, round to TF32 and write the
// row as the next layer's A operand -- activations never leave the SM between layers.  The last layer's rows are staged in
// shared memory and written as contiguous rows of w_L floats.
//
// Shared-memory operand layout (no swizzle, K-major "interleaved" canonical form): a K-chunk is 16 bytes (4 TF32); chunk c
// of row r sits at  c * (rows * 16) + r * 16,  i.e. 8 consecutive rows of one chunk form one contiguous 128-byte core matrix,
// the stride between 8-row groups (SBO) is 128 bytes and the stride between K-chunks (LBO) is rows * 16 bytes.
//
// Precision: TF32 operands (10-bit mantissa, round-to-nearest on both sides), fp32 accumulation, fp32 bias/activation.
// PyTorch's default for fp32 matmuls is full fp32; tcgen05 has no fp32-operand mode, so this is the
// torch.set_float32_matmul_precision("high") arithmetic.  DESIGN.md section 13 derives the tolerance used by the tests.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/mala_snap.h"
#include "snap_internal.h"

namespace mala {

constexpr int kMlpMaxLayers = 8;
constexpr int kMlpMaxWidth = 256;   // one MMA covers N <= 256; the A operand of 128 rows x 256 TF32 takes 128 KB
constexpr int kMlpRows = 128;       // rows per tile = MMA M = TMEM lanes
constexpr int kMlpBK = 16;          // K elements per ring stage (two MMA K-steps of 8)
constexpr int kMlpStages = 4;
constexpr int kMlpRowWarps = 8;     // warps 0-7: loader + epilogue; warp w works on rows 32 (w & 3) .. + 31 (its TMEM subpartition) and
                                    // on the column half w >> 2 of every accumulator
constexpr int kMlpThreads = (kMlpRowWarps + 2) * 32;  // + warp 8: weight producer, warp 9: TMEM allocation + MMA issue
constexpr int kMlpTmemCols = 256;
constexpr int kMlpABytes = kMlpRows * (kMlpMaxWidth + 1) * 4;  // A operand (128 KB); as output staging [128][w_out | 1] fp32 it needs 514 B more

struct MlpParams {
    int nlayers;
    int act, activate_last;
    int w_in, w_out;
    int K[kMlpMaxLayers], N[kMlpMaxLayers];   // padded: K to 16, N to 32 (two column halves of whole 16-column TMEM loads)
    int woff[kMlpMaxLayers];                  // float offset of layer l in the packed weight image
    int boff[kMlpMaxLayers];                  // float offset of layer l in the bias array
    const float *wpacked;                     // [layer][K block][chunk 0..3][n][4] TF32-rounded, zero padded
    const float *bias;                        // [layer][N] zero padded
    const double *in_shift, *in_scale;        // [w_in]
};

// ---- PTX helpers ----------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t s32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mb_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s32(bar)), "r"(count));
}
__device__ __forceinline__ void mb_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(s32(bar)) : "memory");
}
__device__ __forceinline__ void mb_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s32(bar)), "r"(bytes) : "memory");
}
// bounded wait: a protocol error must end in a trap (reported as a launch failure), never in a hung GPU
__device__ __forceinline__ void mb_wait(uint64_t *bar, uint32_t parity) {
    for (uint32_t spin = 0; spin < (1u << 26); spin++) {
        uint32_t done;
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(s32(bar)), "r"(parity)
            : "memory");
        if (done) return;
    }
    __trap();
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(s32(dst)), "l"(src),
                 "r"(bytes), "r"(s32(bar))
                 : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// K-major, no swizzle: start address, LBO (between the two 16-byte K-chunks of one MMA), SBO (between 8-row groups)
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((addr >> 4) & 0x3fffu) | ((uint64_t)((lbo_bytes >> 4) & 0x3fffu) << 16) | ((uint64_t)((sbo_bytes >> 4) & 0x3fffu) << 32) |
           (1ull << 46);  // descriptor version 1 (sm_100); base offset 0, layout type 0 = no swizzle
}
// instruction descriptor of kind::tf32: D fp32, A/B TF32, both K-major, M = 128
__device__ __forceinline__ uint32_t instr_desc_tf32(int n) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(kMlpRows >> 4) << 24);
}
__device__ __forceinline__ void mma_tf32(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void mma_commit(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(s32(bar)) : "memory");
}
// 16 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
        "tcgen05.wait::ld.sync.aligned;\n"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
#pragma unroll
    for (int i = 0; i < 16; i++) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ float to_tf32(float v) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(v));
    return __uint_as_float(r);
}
template <int ACT>
__device__ __forceinline__ float activate(float v) {
    if (ACT == 1) return fmaxf(v, 0.f);
    if (ACT == 2) return v > 0.f ? v : 0.01f * v;
    if (ACT == 3) return 1.f / (1.f + __expf(-v));
    return v;
}

// ---- the kernel -----------------------------------------------------------------------------------------------
// dynamic shared memory: A operand [Kmax/4][128][16 B] | ring [stages][16 KB] | biases | barriers
template <int ACT>
__global__ void __launch_bounds__(kMlpThreads, 1) mlp_forward_kernel(MlpParams P, MlpRows R) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char *Abuf = smem;                                   // kMlpMaxWidth / 4 chunks x 2048 B = 128 KB (+ staging slack)
    unsigned char *ring = Abuf + kMlpABytes;                         // kMlpStages x (kMlpBK / 4 chunks x 256 rows x 16 B = 16 KB)
    float *bias_s = reinterpret_cast<float *>(ring + kMlpStages * (kMlpBK / 4) * kMlpMaxWidth * 16);
    uint64_t *bars = reinterpret_cast<uint64_t *>(bias_s + kMlpMaxLayers * kMlpMaxWidth);
    uint64_t *full = bars, *empty = bars + kMlpStages, *a_ready = bars + 2 * kMlpStages, *d_full = a_ready + 1;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(d_full + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long ntiles = (R.nrows + kMlpRows - 1) / kMlpRows;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kMlpStages; s++) { mb_init(&full[s], 1); mb_init(&empty[s], 1); }
        mb_init(a_ready, kMlpRowWarps * 32);
        mb_init(d_full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = threadIdx.x; i < P.nlayers * kMlpMaxWidth; i += kMlpThreads) {
        const int l = i / kMlpMaxWidth, n = i % kMlpMaxWidth;
        bias_s[i] = (n < P.N[l]) ? P.bias[P.boff[l] + n] : 0.f;
    }
    if (warp == kMlpRowWarps + 1) {  // TMEM: one warp allocates (and frees at the end)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(s32(tmem_slot)), "n"(kMlpTmemCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == kMlpRowWarps) {
        // ===== weight producer: the same sequence of K-blocks for every tile =====
        if (lane == 0) {
            uint32_t it = 0;
            for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x)
                for (int l = 0; l < P.nlayers; l++) {
                    const uint32_t bytes = (uint32_t)(kMlpBK / 4) * P.N[l] * 16;
                    const float *src = P.wpacked + P.woff[l];
                    for (int kb = 0; kb < P.K[l] / kMlpBK; kb++, it++) {
                        const int s = it % kMlpStages;
                        mb_wait(&empty[s], ((it / kMlpStages) & 1u) ^ 1u);
                        mb_expect_tx(&full[s], bytes);
                        bulk_g2s(ring + (size_t)s * (kMlpBK / 4) * kMlpMaxWidth * 16, src + (size_t)kb * (bytes / 4), bytes, &full[s]);
                    }
                }
        }
    } else if (warp == kMlpRowWarps + 1) {
        // ===== MMA issuer =====
        if (lane == 0) {
            uint32_t it = 0, step = 0;
            for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x)
                for (int l = 0; l < P.nlayers; l++, step++) {
                    mb_wait(a_ready, step & 1u);  // A of this layer written, accumulator of the previous one drained
                    tc_fence_after();
                    const uint32_t idesc = instr_desc_tf32(P.N[l]);
                    const uint32_t b_lbo = (uint32_t)P.N[l] * 16;
                    for (int kb = 0; kb < P.K[l] / kMlpBK; kb++, it++) {
                        const int s = it % kMlpStages;
                        mb_wait(&full[s], (it / kMlpStages) & 1u);
                        tc_fence_after();
                        const uint32_t b_addr = s32(ring + (size_t)s * (kMlpBK / 4) * kMlpMaxWidth * 16);
#pragma unroll
                        for (int k8 = 0; k8 < kMlpBK / 8; k8++) {
                            const uint32_t a_addr = s32(Abuf) + (uint32_t)(kb * (kMlpBK / 4) + k8 * 2) * (kMlpRows * 16);
                            mma_tf32(tmem_base, smem_desc(a_addr, kMlpRows * 16, 128), smem_desc(b_addr + (uint32_t)k8 * 2 * b_lbo, b_lbo, 128),
                                     idesc, (kb | k8) ? 1u : 0u);
                        }
                        mma_commit(&empty[s]);  // the stage is free once these MMAs have read it
                    }
                    mma_commit(d_full);         // accumulator of layer l complete
                }
        }
    } else {
        // ===== rows: load the descriptors, then one epilogue per layer =====
        const int sub = warp & 3, half = warp >> 2;
        const int row = sub * 32 + lane;  // the TMEM lane (= tile row) this thread reads
        uint32_t step = 0;
        float *stage_out = reinterpret_cast<float *>(Abuf);  // last layer: [row][ostride] fp32
        const int ostride = P.w_out | 1;                     // odd stride: conflict-free row-per-thread writes
        for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const long long row0 = tile * kMlpRows;
            // ---- layer-0 operand: x = (descriptor - shift) * scale, rounded to TF32.  Warp w takes rows w, w + 8, ...; a lane owns
            // the features k = lane, lane + 32, ... of every row (coalesced 8-byte loads), eight rows of loads in flight at a time
#pragma unroll 1
            for (int k = lane; k < P.K[0]; k += 32) {
                const bool kin = k < P.w_in;
                const double sh = kin ? P.in_shift[k] : 0.0, sc = kin ? P.in_scale[k] : 0.0;  // padded features become exact zeros
                unsigned char *dstk = Abuf + (size_t)(k >> 2) * (kMlpRows * 16) + (k & 3) * 4;
#pragma unroll 1
                for (int rb = 0; rb < kMlpRows / kMlpRowWarps; rb += 8) {
                    double xv[8];
#pragma unroll
                    for (int i = 0; i < 8; i++) {
                        const long long gr = row0 + warp + kMlpRowWarps * (rb + i);
                        xv[i] = (kin && gr < R.nrows) ? __ldcs(R.x + gr * P.w_in + k) : 0.0;
                    }
#pragma unroll
                    for (int i = 0; i < 8; i++)
                        *reinterpret_cast<float *>(dstk + (warp + kMlpRowWarps * (rb + i)) * 16) = to_tf32((float)((xv[i] - sh) * sc));
                }
            }
            fence_async_smem();
            mb_arrive(a_ready);
            for (int l = 0; l < P.nlayers; l++, step++) {
                mb_wait(d_full, step & 1u);
                tc_fence_after();
                const bool last = (l == P.nlayers - 1);
                const bool act_on = !last || P.activate_last;
                const int nh = P.N[l] >> 1;               // this warp's column half: [half * nh, half * nh + nh)
                const uint32_t taddr = tmem_base + ((uint32_t)(sub * 32) << 16) + (uint32_t)(half * nh);
                const float *bl = bias_s + l * kMlpMaxWidth + half * nh;
                if (!last) {
                    unsigned char *arow = Abuf + (size_t)((half * nh) >> 2) * (kMlpRows * 16) + row * 16;
                    for (int n0 = 0; n0 < nh; n0 += 16) {
                        float v[16];
                        tmem_ld16(taddr + (uint32_t)n0, v);
#pragma unroll
                        for (int c = 0; c < 4; c++) {
                            const float4 b4 = *reinterpret_cast<const float4 *>(bl + n0 + 4 * c);
                            float4 q = make_float4(v[4 * c] + b4.x, v[4 * c + 1] + b4.y, v[4 * c + 2] + b4.z, v[4 * c + 3] + b4.w);
                            if (act_on) q = make_float4(activate<ACT>(q.x), activate<ACT>(q.y), activate<ACT>(q.z), activate<ACT>(q.w));
                            q = make_float4(to_tf32(q.x), to_tf32(q.y), to_tf32(q.z), to_tf32(q.w));
                            *reinterpret_cast<float4 *>(arow + (size_t)((n0 >> 2) + c) * (kMlpRows * 16)) = q;
                        }
                    }
                } else {
                    float *orow = stage_out + row * ostride + half * nh;
                    const int nvalid = P.w_out - half * nh;   // columns of this half that exist
                    for (int n0 = 0; n0 < nh && n0 < nvalid; n0 += 16) {
                        float v[16];
                        tmem_ld16(taddr + (uint32_t)n0, v);
#pragma unroll
                        for (int j = 0; j < 16; j++) {
                            float q = v[j] + bl[n0 + j];
                            if (act_on) q = activate<ACT>(q);
                            if (n0 + j < nvalid) orow[n0 + j] = q;
                        }
                    }
                }
                tc_fence_before();  // the accumulator reads above are ordered before the next layer's MMAs
                if (!last) {
                    fence_async_smem();
                    mb_arrive(a_ready);
                }
            }
            // ---- write the tile: one warp per row, w_out contiguous floats
            asm volatile("bar.sync 1, %0;" ::"n"(kMlpRowWarps * 32) : "memory");
            for (int r = warp; r < kMlpRows; r += kMlpRowWarps) {
                const long long gr = row0 + r;
                if (gr >= R.nrows) break;
                long long orow = gr;
                if (R.compact) {
                    int ix, iy, iz;
                    bool valid;
                    lane_point(R.geom, R.tile_begin + (int)(gr >> 5), (int)(gr & 31), ix, iy, iz, valid);
                    if (!valid) continue;
                    orow = ((long long)(iz - R.geom.z0) * R.geom.ny + iy) * R.geom.nx + ix;
                }
                float *dst = R.y + orow * P.w_out;
                for (int n = lane; n < P.w_out; n += 32) __stcs(dst + n, stage_out[r * ostride + n]);
            }
            asm volatile("bar.sync 1, %0;" ::"n"(kMlpRowWarps * 32) : "memory");  // staging area is the next tile's A operand
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == kMlpRowWarps + 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kMlpTmemCols));
}

constexpr size_t kMlpSmemBytes = (size_t)kMlpABytes + (size_t)kMlpStages * (kMlpBK / 4) * kMlpMaxWidth * 16 +
                                 (size_t)kMlpMaxLayers * kMlpMaxWidth * sizeof(float) + (2 * kMlpStages + 2) * sizeof(uint64_t) + 16;

}  // namespace mala

// =============================================================================================================
// host side
// =============================================================================================================
struct mala_mlp {
    mala::MlpParams P{};
    float *d_w = nullptr, *d_b = nullptr;
    double *d_shift = nullptr, *d_scale = nullptr;
    int num_sms = 0;
    long long flop_per_row = 0;   // 2 * sum_l w_l * w_{l+1}
};

namespace mala {

static float round_tf32(double x) {  // round-to-nearest-even onto 10 explicit mantissa bits, as cvt.rna does up to ties
    float f = (float)x;
    uint32_t u;
    std::memcpy(&u, &f, 4);
    if ((u & 0x7f800000u) == 0x7f800000u) return f;
    u += 0x00000fffu + ((u >> 13) & 1u);
    u &= 0xffffe000u;
    std::memcpy(&f, &u, 4);
    return f;
}

int mlp_in_width(const mala_mlp *net) { return net->P.w_in; }
int mlp_out_width(const mala_mlp *net) { return net->P.w_out; }

int mlp_launch(const mala_mlp *net, const MlpRows &rows, cudaStream_t st) {
    if (rows.nrows <= 0) return 0;
    const long long ntiles = (rows.nrows + kMlpRows - 1) / kMlpRows;
    const int grid = (int)std::min<long long>(ntiles, net->num_sms);
    switch (net->P.act) {
        case 1: mlp_forward_kernel<1><<<grid, kMlpThreads, kMlpSmemBytes, st>>>(net->P, rows); break;
        case 2: mlp_forward_kernel<2><<<grid, kMlpThreads, kMlpSmemBytes, st>>>(net->P, rows); break;
        case 3: mlp_forward_kernel<3><<<grid, kMlpThreads, kMlpSmemBytes, st>>>(net->P, rows); break;
        default: mlp_forward_kernel<0><<<grid, kMlpThreads, kMlpSmemBytes, st>>>(net->P, rows); break;
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_error(MALA_SNAP_ECUDA, std::string("mlp_forward_kernel: ") + cudaGetErrorString(e));
    return 0;
}

}  // namespace mala

extern "C" {

int mala_mlp_create(mala_mlp_t **net, int nlayers, const int *sizes, const double *const *weights, const double *const *biases,
                    int activation, int activate_last, const double *in_shift, const double *in_scale) {
    using namespace mala;
    if (!net) return set_error(MALA_SNAP_EINVAL, "net is NULL");
    *net = nullptr;
    if (nlayers < 1 || nlayers > kMlpMaxLayers) return set_error(MALA_SNAP_EINVAL, "nlayers must lie in [1, 8]");
    if (!sizes || !weights || !biases) return set_error(MALA_SNAP_EINVAL, "sizes/weights/biases is NULL");
    if (activation < 0 || activation > 3) return set_error(MALA_SNAP_EINVAL, "activation must be 0 (identity), 1 (ReLU), 2 (leaky ReLU) or 3 (sigmoid)");
    for (int l = 0; l <= nlayers; l++)
        if (sizes[l] < 1 || sizes[l] > kMlpMaxWidth) return set_error(MALA_SNAP_EINVAL, "layer widths must lie in [1, 256]");
    for (int l = 0; l < nlayers; l++)
        if (!weights[l] || !biases[l]) return set_error(MALA_SNAP_EINVAL, "a weight or bias pointer is NULL");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return set_error(MALA_SNAP_ECUDA, "no CUDA device: this library has no CPU fallback");
    }
    mala_mlp *m = new (std::nothrow) mala_mlp();
    if (!m) return set_error(MALA_SNAP_ENOMEM, "out of host memory");
    MlpParams &P = m->P;
    P.nlayers = nlayers; P.act = activation; P.activate_last = activate_last ? 1 : 0;
    P.w_in = sizes[0]; P.w_out = sizes[nlayers];
    std::vector<float> wp, bp;
    for (int l = 0; l < nlayers; l++) {
        const int wk = sizes[l], wn = sizes[l + 1];
        const int K = (l == 0) ? (wk + 15) / 16 * 16 : P.N[l - 1];   // = the padded width of the layer before
        const int N = (wn + 31) / 32 * 32;
        P.K[l] = K; P.N[l] = N;
        P.woff[l] = (int)wp.size(); P.boff[l] = (int)bp.size();
        m->flop_per_row += 2LL * wk * wn;
        // image of the ring stages: [K block of 16][chunk of 4 k][n][4 k], exactly what one bulk copy drops into shared memory
        for (int kb = 0; kb < K / kMlpBK; kb++)
            for (int c = 0; c < kMlpBK / 4; c++)
                for (int n = 0; n < N; n++)
                    for (int q = 0; q < 4; q++) {
                        const int k = kb * kMlpBK + c * 4 + q;
                        double v = (n < wn && k < wk) ? weights[l][(size_t)n * wk + k] : 0.0;
                        if (!std::isfinite(v)) { delete m; return set_error(MALA_SNAP_EINVAL, "a weight is not finite"); }
                        wp.push_back(round_tf32(v));
                    }
        for (int n = 0; n < N; n++) {
            const double v = n < wn ? biases[l][n] : 0.0;
            if (!std::isfinite(v)) { delete m; return set_error(MALA_SNAP_EINVAL, "a bias is not finite"); }
            bp.push_back((float)v);
        }
    }
    std::vector<double> sh(P.w_in, 0.0), sc(P.w_in, 1.0);
    for (int k = 0; k < P.w_in; k++) {
        if (in_shift) sh[k] = in_shift[k];
        if (in_scale) sc[k] = in_scale[k];
        if (!std::isfinite(sh[k]) || !std::isfinite(sc[k])) { delete m; return set_error(MALA_SNAP_EINVAL, "input shift/scale is not finite"); }
    }
    auto cleanup = [&](int code, const std::string &msg) {
        mala_mlp_destroy(m);
        return set_error(code, msg);
    };
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return cleanup(MALA_SNAP_ECUDA, "cudaGetDeviceProperties failed");
    if (prop.major < 10) return cleanup(MALA_SNAP_ECUDA, "device is not sm_100 class (tcgen05 kernels are built for sm_100a only)");
    m->num_sms = prop.multiProcessorCount;
    cudaError_t e = cudaMalloc((void **)&m->d_w, wp.size() * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc((void **)&m->d_b, bp.size() * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc((void **)&m->d_shift, sh.size() * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&m->d_scale, sc.size() * sizeof(double));
    if (e != cudaSuccess) { cudaGetLastError(); return cleanup(MALA_SNAP_ENOMEM, "cudaMalloc (network) failed"); }
    e = cudaMemcpy(m->d_w, wp.data(), wp.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(m->d_b, bp.data(), bp.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(m->d_shift, sh.data(), sh.size() * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(m->d_scale, sc.data(), sc.size() * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mlp_forward_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMlpSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mlp_forward_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMlpSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mlp_forward_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMlpSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mlp_forward_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMlpSmemBytes);
    if (e != cudaSuccess) return cleanup(MALA_SNAP_ECUDA, std::string("network upload: ") + cudaGetErrorString(e));
    P.wpacked = m->d_w; P.bias = m->d_b; P.in_shift = m->d_shift; P.in_scale = m->d_scale;
    *net = m;
    return MALA_SNAP_OK;
}

int mala_mlp_widths(const mala_mlp_t *net, int *w_in, int *w_out) {
    if (!net) return mala::set_error(MALA_SNAP_EINVAL, "net is NULL");
    if (w_in) *w_in = net->P.w_in;
    if (w_out) *w_out = net->P.w_out;
    return MALA_SNAP_OK;
}

int mala_mlp_forward(mala_mlp_t *net, long long npoints, const double *x, float *y, void *cuda_stream) {
    if (!net) return mala::set_error(MALA_SNAP_EINVAL, "net is NULL");
    if (npoints < 0) return mala::set_error(MALA_SNAP_EINVAL, "npoints < 0");
    if (npoints > 0 && (!x || !y)) return mala::set_error(MALA_SNAP_EINVAL, "x or y is NULL");
    mala::MlpRows rows{};
    rows.nrows = npoints; rows.x = x; rows.y = y; rows.compact = 0;
    return mala::mlp_launch(net, rows, (cudaStream_t)cuda_stream);
}

void mala_mlp_destroy(mala_mlp_t *net) {
    if (!net) return;
    cudaDeviceSynchronize();
    if (net->d_w) cudaFree(net->d_w);
    if (net->d_b) cudaFree(net->d_b);
    if (net->d_shift) cudaFree(net->d_shift);
    if (net->d_scale) cudaFree(net->d_scale);
    cudaGetLastError();
    delete net;
}

}  // extern "C"
