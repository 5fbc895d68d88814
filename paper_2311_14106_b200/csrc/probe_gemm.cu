// probe_gemm.cu — harness kernels OUTSIDE the hot path: skeletons of the k-tile loop of the grouped
// GEMM kernel, used to measure what a given staging scheme and tile shape can reach on this box before
// (and after) it is built into heff_kernels.cu.  Every CTA runs `ktiles` full k-tiles (BK = 16) of a
// dense C += A·Bᵀ with A, B tiles streamed from an L2-resident buffer; no ragged edges, no segment
// switches, no epilogue — so the result is the ceiling of the loop, not a product number.
//
//   kind 0: 64×64 CTA tile, 2×2 warps of 32×32, cp.async (LDGSTS) 16-byte copies issued by every
//           thread, 3 stages, one __syncthreads per k-tile, padded shared strides (the round-1 kernel)
//   kind 1: 64×64 CTA tile, 2×2 warps of 32×32, tiles fetched by ONE elected thread with
//           cp.async.bulk (the TMA unit; SASS UBLKCP) completing on an mbarrier, 4 stages, full/empty
//           mbarriers instead of __syncthreads, dense 128-byte shared rows with the 32-byte-group XOR
//           swizzle already present in global memory (panel layout)
//   kind 2: as kind 1 with a 128×64 CTA tile, 2×2 warps of 64×32 (8×4 fragments), 3 stages
//   kind 3: 128×64 tile, row-major source, cp.async issued by a dedicated fifth (producer) warp and
//           signalled through mbarriers; 160 threads, 2 CTAs per SM
//   kind 4: kind 2 at 2 CTAs per SM with 4 stages;   kind 5: kind 1 at 2 CTAs per SM
#include "internal.h"

namespace dmrgk {

namespace pg {

constexpr int BK = 16;
constexpr int NTHREADS = 128;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// ---- kind 0: the round-1 loop (cp.async, padded strides) ----------------------------------------
constexpr int K0_STRIDE = 20, K0_STAGES = 3, K0_OPER = 64 * K0_STRIDE, K0_SMEM = K0_STAGES * 2 * K0_OPER * 8;

__global__ void __launch_bounds__(NTHREADS, 3)
probe_loop_cpasync(const double* __restrict__ buf, long long span_tiles, int ktiles, double* sink) {
    extern __shared__ __align__(128) double smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, wm = warp >> 1, wn = warp & 1, g = lane >> 2, t4 = lane & 3;
    const double* A = buf + (long long)(blockIdx.x % 32) * span_tiles * 1024;
    const double* B = buf + (long long)(32 + (blockIdx.x / 32) % 32) * span_tiles * 1024;
    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const uint32_t sbase = smem_u32(smem);
    const int row = tid >> 3, ch = tid & 7;
    auto load = [&](int stage, int kt) {
        const long long t = kt % span_tiles;
#pragma unroll
        for (int op = 0; op < 2; ++op) {
            const double* src = (op ? B : A) + t * 1024 + row * 16 + ch * 2;
            const uint32_t dst = sbase + ((stage * 2 + op) * K0_OPER + row * K0_STRIDE + ch * 2) * 8;
#pragma unroll
            for (int j = 0; j < 4; ++j)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst + j * 16 * K0_STRIDE * 8), "l"(src + j * 256));
        }
    };
#pragma unroll
    for (int s = 0; s < K0_STAGES - 1; ++s) {
        load(s, s);
        asm volatile("cp.async.commit_group;\n" ::);
    }
    int stage = 0;
    for (int it = 0; it < ktiles; ++it) {
        asm volatile("cp.async.wait_group %0;\n" ::"n"(K0_STAGES - 2));
        __syncthreads();
        {
            int ns = stage + K0_STAGES - 1;
            if (ns >= K0_STAGES) ns -= K0_STAGES;
            if (it + K0_STAGES - 1 < ktiles) load(ns, it + K0_STAGES - 1);
            asm volatile("cp.async.commit_group;\n" ::);
        }
        const double* pa = smem + (stage * 2) * K0_OPER + (wm * 32 + g) * K0_STRIDE + t4;
        const double* pb = smem + (stage * 2 + 1) * K0_OPER + (wn * 32 + g) * K0_STRIDE + t4;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
            double af[4], bf[4];
#pragma unroll
            for (int f = 0; f < 4; ++f) af[f] = pa[f * 8 * K0_STRIDE + ks * 4];
#pragma unroll
            for (int f = 0; f < 4; ++f) bf[f] = pb[f * 8 * K0_STRIDE + ks * 4];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
        if (++stage == K0_STAGES) stage = 0;
    }
    asm volatile("cp.async.wait_group 0;\n" ::);
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s += acc[i][j][0] + acc[i][j][1];
    if (s == 123.456) sink[0] = s;
}

// ---- kinds 1, 2: bulk copies by one elected thread, full/empty mbarriers --------------------------
// Shared stage: A tile [BM rows][16] then B tile [64 rows][16], dense 128-byte rows; element (row, k)
// sits at row·16 + (k ^ ((row & 3) << 2)) — the swizzle is in the global panel, the copy is verbatim.
// Lane (g, t4) of a fragment reads row (…+g), k = 4·ks + t4 → offset 4·(ks ^ (g & 3)) + t4: the 16 lanes
// of a half-warp hit 16 distinct 8-byte banks.
template <int FM, int STAGES, int MINB>
__global__ void __launch_bounds__(NTHREADS, MINB)
probe_loop_bulk(const double* __restrict__ buf, long long span_tiles, int ktiles, double* sink) {
    constexpr int BM = FM * 16;                      // 2 warps along M, FM fragments of 8 rows each
    constexpr int A_DOUBLES = BM * BK, B_DOUBLES = 64 * BK, STAGE_DOUBLES = A_DOUBLES + B_DOUBLES;
    extern __shared__ __align__(128) double smem[];
    __shared__ __align__(8) unsigned long long bars[2 * STAGES];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, wm = warp >> 1, wn = warp & 1, g = lane >> 2, t4 = lane & 3;
    const double* A = buf + (long long)(blockIdx.x % 32) * span_tiles * A_DOUBLES;
    const double* B = buf + (long long)(32 + (blockIdx.x / 32) % 32) * span_tiles * A_DOUBLES;
    const uint32_t sbase = smem_u32(smem), bar0 = smem_u32(bars);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar0 + s * 8, 1);                   // full[s]: the producer's arrive + the copies' bytes
            mbar_init(bar0 + (STAGES + s) * 8, 4);        // empty[s]: one arrive per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    double acc[FM][4][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    auto produce = [&](int kt) {                          // called by ONE thread
        const int s = kt % STAGES;
        const long long t = kt % span_tiles;
        const uint32_t full = bar0 + s * 8;
        mbar_expect_tx(full, STAGE_DOUBLES * 8);
        bulk_g2s(sbase + s * STAGE_DOUBLES * 8, A + t * A_DOUBLES, A_DOUBLES * 8, full);
        bulk_g2s(sbase + (s * STAGE_DOUBLES + A_DOUBLES) * 8, B + t * B_DOUBLES, B_DOUBLES * 8, full);
    };
    // producer role rotates over the warps (tile kt is fetched by lane 0 of warp kt & 3) so that no
    // warp — and no SM sub-partition — carries the whole issue overhead
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < STAGES - 1; ++s)
            if (s < ktiles && (s & 3) == warp) produce(s);
    }
    const int g3 = g & 3;
    int offA[4], offB[4];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
        offA[ks] = (wm * (FM * 8) + g) * 16 + 4 * (ks ^ g3) + t4;
        offB[ks] = A_DOUBLES + (wn * 32 + g) * 16 + 4 * (ks ^ g3) + t4;
    }
    for (int it = 0; it < ktiles; ++it) {
        const int s = it % STAGES;
        const uint32_t ph = (it / STAGES) & 1;
        // refill: tile it+STAGES−1 goes into the stage tile it−1 used; its consumers must be done
        const int nt = it + STAGES - 1;
        if (lane == 0 && nt < ktiles && (nt & 3) == warp) {
            if (it >= 1) mbar_wait(bar0 + (STAGES + (nt % STAGES)) * 8, ((it - 1) / STAGES) & 1);
            produce(nt);
        }
        __syncwarp();
        mbar_wait(bar0 + s * 8, ph);
        const double* st = smem + s * STAGE_DOUBLES;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
            double af[FM], bf[4];
#pragma unroll
            for (int f = 0; f < FM; ++f) af[f] = st[offA[ks] + f * 128];
#pragma unroll
            for (int f = 0; f < 4; ++f) bf[f] = st[offB[ks] + f * 128];
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar0 + (STAGES + s) * 8);
    }
    double sum = 0.0;
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) sum += acc[i][j][0] + acc[i][j][1];
    if (sum == 123.456) sink[0] = sum;
}

// ---- kind 3: cp.async issued by a dedicated PRODUCER WARP, full/empty mbarriers --------------------
// Keeps the row-major global layout (tile rows are `ld` apart; here ld = 16) and the padded shared
// strides of kind 0, but the four compute warps carry no loader state: a fifth warp issues every
// 16-byte cp.async of the stage (48 per lane for a 128×64 tile pair) and lets the copies arrive on the
// stage's full barrier (cp.async.mbarrier.arrive.noinc).  160 threads, 2 CTAs per SM.
constexpr int K3_STRIDE = 20, K3_STAGES = 3, K3_A = 128 * K3_STRIDE, K3_B = 64 * K3_STRIDE;
constexpr int K3_STAGE = K3_A + K3_B, K3_SMEM = K3_STAGES * K3_STAGE * 8;

__global__ void __launch_bounds__(160, 2)
probe_loop_producer_warp(const double* __restrict__ buf, long long span_tiles, int ktiles, double* sink) {
    extern __shared__ __align__(128) double smem[];
    __shared__ __align__(8) unsigned long long bars[2 * K3_STAGES];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double* A = buf + (long long)(blockIdx.x % 32) * span_tiles * 2048;
    const double* B = buf + (long long)(32 + (blockIdx.x / 32) % 32) * span_tiles * 2048;
    const uint32_t sbase = smem_u32(smem), bar0 = smem_u32(bars);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < K3_STAGES; ++s) {
            mbar_init(bar0 + s * 8, 32);                     // full[s]: one deferred arrive per producer lane
            mbar_init(bar0 + (K3_STAGES + s) * 8, 4);        // empty[s]: one arrive per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    if (warp == 4) {
        // producer: lane owns chunk ch = lane & 7 of rows (lane >> 3) + 4·j
        const int r0 = lane >> 3, ch = lane & 7;
        for (int kt = 0; kt < ktiles; ++kt) {
            const int s = kt % K3_STAGES;
            if (kt >= K3_STAGES) mbar_wait(bar0 + (K3_STAGES + s) * 8, ((kt / K3_STAGES) - 1) & 1);
            const long long t = kt % span_tiles;
            const double* srcA = A + t * 2048 + r0 * 16 + ch * 2;
            const double* srcB = B + t * 1024 + r0 * 16 + ch * 2;
            const uint32_t dA = sbase + (s * K3_STAGE + r0 * K3_STRIDE + ch * 2) * 8;
            const uint32_t dB = dA + K3_A * 8;
#pragma unroll 8
            for (int j = 0; j < 32; ++j)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dA + j * 4 * K3_STRIDE * 8), "l"(srcA + j * 64));
#pragma unroll 8
            for (int j = 0; j < 16; ++j)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dB + j * 4 * K3_STRIDE * 8), "l"(srcB + j * 64));
            asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar0 + s * 8) : "memory");
        }
        asm volatile("cp.async.wait_all;\n" ::: "memory");
        return;
    }
    const int wm = warp >> 1, wn = warp & 1, g = lane >> 2, t4 = lane & 3;
    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    for (int it = 0; it < ktiles; ++it) {
        const int s = it % K3_STAGES;
        mbar_wait(bar0 + s * 8, (it / K3_STAGES) & 1);
        const double* pa = smem + s * K3_STAGE + (wm * 64 + g) * K3_STRIDE + t4;
        const double* pb = smem + s * K3_STAGE + K3_A + (wn * 32 + g) * K3_STRIDE + t4;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
            double af[8], bf[4];
#pragma unroll
            for (int f = 0; f < 8; ++f) af[f] = pa[f * 8 * K3_STRIDE + ks * 4];
#pragma unroll
            for (int f = 0; f < 4; ++f) bf[f] = pb[f * 8 * K3_STRIDE + ks * 4];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar0 + (K3_STAGES + s) * 8);
    }
    double sum = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) sum += acc[i][j][0] + acc[i][j][1];
    if (sum == 123.456) sink[0] = sum;
}

}  // namespace pg
}  // namespace dmrgk

using namespace dmrgk;

extern "C" int32_t dmrgk_probe_gemm_loop(dmrgk_ctx* ctx, int32_t kind, int32_t ktiles, const double* buf_dev,
                                         int64_t buf_doubles, double* sink_dev, double* flops, void* stream) {
    if (!ctx || !buf_dev || !sink_dev || ktiles < 1) return fail(DMRGK_EINVAL, "probe_gemm_loop: bad argument");
    if (!aligned128(buf_dev)) return fail(DMRGK_EALIGN, "probe_gemm_loop: buffer not 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    const int grid = ctx->n_sm * 3;
    cudaStream_t st = (cudaStream_t)stream;
    // 64 spans (32 for A, 32 for B) of span_tiles tiles each; a tile is ≤ 2048 doubles
    const long long span_tiles = buf_doubles / (64LL * 2048);
    if (span_tiles < 1) return fail(DMRGK_EINVAL, "probe_gemm_loop: buffer too small (need ≥ 1 MiB)");
    int bm = 64, ctas = 3;
    if (kind == 0) {
        DMRGK_CUDA(cudaFuncSetAttribute(pg::probe_loop_cpasync, cudaFuncAttributeMaxDynamicSharedMemorySize, pg::K0_SMEM));
        pg::probe_loop_cpasync<<<grid, pg::NTHREADS, pg::K0_SMEM, st>>>(buf_dev, span_tiles, ktiles, sink_dev);
    } else if (kind == 1 || kind == 5) {
        constexpr int smem = 4 * (64 + 64) * 16 * 8;
        if (kind == 1) {
            DMRGK_CUDA(cudaFuncSetAttribute(pg::probe_loop_bulk<4, 4, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            pg::probe_loop_bulk<4, 4, 3><<<grid, pg::NTHREADS, smem, st>>>(buf_dev, span_tiles, ktiles, sink_dev);
        } else {
            ctas = 2;
            DMRGK_CUDA(cudaFuncSetAttribute(pg::probe_loop_bulk<4, 4, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            pg::probe_loop_bulk<4, 4, 2><<<ctx->n_sm * 2, pg::NTHREADS, smem, st>>>(buf_dev, span_tiles, ktiles, sink_dev);
        }
    } else if (kind == 2 || kind == 4) {
        bm = 128;
        if (kind == 2) {
            constexpr int smem = 3 * (128 + 64) * 16 * 8;
            DMRGK_CUDA(cudaFuncSetAttribute(pg::probe_loop_bulk<8, 3, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            pg::probe_loop_bulk<8, 3, 3><<<grid, pg::NTHREADS, smem, st>>>(buf_dev, span_tiles, ktiles, sink_dev);
        } else {
            ctas = 2;
            constexpr int smem = 4 * (128 + 64) * 16 * 8;
            DMRGK_CUDA(cudaFuncSetAttribute(pg::probe_loop_bulk<8, 4, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            pg::probe_loop_bulk<8, 4, 2><<<ctx->n_sm * 2, pg::NTHREADS, smem, st>>>(buf_dev, span_tiles, ktiles, sink_dev);
        }
    } else if (kind == 3) {
        bm = 128;
        ctas = 2;
        DMRGK_CUDA(cudaFuncSetAttribute(pg::probe_loop_producer_warp, cudaFuncAttributeMaxDynamicSharedMemorySize, pg::K3_SMEM));
        pg::probe_loop_producer_warp<<<ctx->n_sm * 2, 160, pg::K3_SMEM, st>>>(buf_dev, span_tiles, ktiles, sink_dev);
    } else {
        return fail(DMRGK_EINVAL, "probe_gemm_loop: kind must be 0 … 5");
    }
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    if (flops) *flops = double(ctx->n_sm) * ctas * double(ktiles) * 2.0 * bm * 64 * 16;
    return DMRGK_OK;
}
