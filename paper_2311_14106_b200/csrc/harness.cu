// harness.cu — kernels OUTSIDE the hot path: seeded synthetic inputs and FP64 pipe probes.
//
// The fill kernels implement the same counter-based generator as workloads/rng.py (normal12:
// SplitMix64 of (seed, stream, element index), twelve 32-bit uniforms summed exactly, one exact
// power-of-two scaling), so that operator arenas too large to ship from the host (SURVEY.md §8(d):
// configs 3-5 hold 39-187 GB) can be generated in place and the oracle can regenerate any block on
// the CPU bit for bit.  Integer arithmetic only until the final int64→double conversion.
#include "internal.h"
#include <cmath>

namespace dmrgk {

__host__ __device__ inline unsigned long long splitmix64(unsigned long long x) {
    unsigned long long z = x + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__host__ __device__ inline double normal12(unsigned long long base, unsigned long long idx) {
    unsigned long long acc = 0, c0 = base + idx * 6ull;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        unsigned long long h = splitmix64(c0 + j);
        acc += (h >> 32) + (h & 0xFFFFFFFFull);
    }
    long long centred = (long long)acc - 6ll * 4294967295ll;
    return (double)centred * (1.0 / 4294967296.0);
}

// One CTA row of work per (block, row-chunk): grid.y = block index, grid.x strides rows·ld.
__global__ void fill_normal_kernel(const DevBlock* __restrict__ table, double* __restrict__ arena,
                                   unsigned long long base, int scale_mode, int symmetric) {
    const DevBlock b = table[blockIdx.y];
    const double scale = scale_mode == 1 ? 1.0 / sqrt((double)b.cols) : scale_mode == 2 ? 1.0 / sqrt((double)b.rows) : 1.0;
    const long long total = (long long)b.rows_pad * b.ld;      // every stored double, padding included
    const long long panel = (long long)b.rows_pad * 16;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        // inverse of panel_off: storage position e → element (r, c)
        const int p = int(e / panel), rem = int(e % panel);
        const int r = rem >> 4, pos = rem & 15;
        const int c = p * 16 + (pos ^ ((r & 3) << 2));
        double v = 0.0;
        if (r < b.rows && c < b.cols) {
            double gv = normal12(base, (unsigned long long)(b.uoff + (long long)r * b.cols + c));
            if (symmetric && b.square_diag) {
                const double gt = normal12(base, (unsigned long long)(b.uoff + (long long)c * b.cols + r));
                gv = (gv + gt) * 0.5;
            }
            v = gv * scale;
        }
        arena[b.off + e] = v;
    }
}

static int32_t fill(const DevBlock* table, const std::vector<Block>& blocks, double* arena,
                    uint64_t seed, uint64_t stream_id, int scale_mode, int symmetric, cudaStream_t st) {
    if (blocks.empty()) return DMRGK_OK;
    if (!arena) return fail(DMRGK_EINVAL, "fill_normal: arena is NULL");
    const unsigned long long base = splitmix64((unsigned long long)seed ^ splitmix64((unsigned long long)stream_id));
    // blocks are launched in slabs of ≤ 65535 (grid.y limit)
    for (size_t b0 = 0; b0 < blocks.size(); b0 += 65535) {
        const unsigned nb = unsigned(std::min<size_t>(65535, blocks.size() - b0));
        int64_t biggest = 0;
        for (size_t i = b0; i < b0 + nb; ++i) biggest = std::max<int64_t>(biggest, blocks[i].size());
        const unsigned gx = unsigned(std::max<int64_t>(1, std::min<int64_t>(1024, (biggest + 255) / 256)));
        fill_normal_kernel<<<dim3(gx, nb), 256, 0, st>>>(table + b0, arena, base, scale_mode, symmetric);
        count_launch();
        DMRGK_CUDA(cudaGetLastError());
    }
    return DMRGK_OK;
}

// ---- FP64 pipe probes --------------------------------------------------------------------------
__global__ void __launch_bounds__(256) probe_dmma_kernel(long long iters, double* sink) {
    double acc[16][2];
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i][0] = acc[i][1] = 0.0;
    double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(acc[i][0]), "+d"(acc[i][1])
                         : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += acc[i][0] + acc[i][1];
    if (s == 123.456) sink[0] = s;
}

__global__ void __launch_bounds__(256) probe_dfma_kernel(long long iters, double* sink) {
    double acc[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) acc[i] = 1e-3 * i;
    const double a = 1.0 + 1e-12 * threadIdx.x, b = 1e-9;
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 32; ++i) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 32; ++i) s += acc[i];
    if (s == 123.456) sink[0] = s;
}

}  // namespace dmrgk

using namespace dmrgk;

extern "C" {

int32_t dmrgk_op_fill_normal(const dmrgk_op* op, double* arena_dev, uint64_t seed, uint64_t stream_id,
                             int32_t scale_mode, int32_t symmetric, void* stream) {
    if (!op) return fail(DMRGK_EINVAL, "op_fill_normal: op is NULL");
    if (!aligned128(arena_dev)) return fail(DMRGK_EALIGN, "op_fill_normal: arena not 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(op->ctx->device));
    return fill(op->dev_table, op->blocks, arena_dev, seed, stream_id, scale_mode, symmetric, (cudaStream_t)stream);
}

int32_t dmrgk_layout_fill_normal(const dmrgk_layout* l, double* arena_dev, uint64_t seed,
                                 uint64_t stream_id, void* stream) {
    if (!l) return fail(DMRGK_EINVAL, "layout_fill_normal: layout is NULL");
    if (!aligned128(arena_dev)) return fail(DMRGK_EALIGN, "layout_fill_normal: arena not 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(l->ctx->device));
    return fill(l->dev_table, l->blocks, arena_dev, seed, stream_id, 0, 0, (cudaStream_t)stream);
}

int32_t dmrgk_iso_fill_normal(const dmrgk_iso* phi, double* arena_dev, uint64_t seed, uint64_t stream_id,
                              void* stream) {
    if (!phi) return fail(DMRGK_EINVAL, "iso_fill_normal: phi is NULL");
    if (!aligned128(arena_dev)) return fail(DMRGK_EALIGN, "iso_fill_normal: arena not 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(phi->ctx->device));
    return fill(phi->dev_table, phi->blocks, arena_dev, seed, stream_id, 2, 0, (cudaStream_t)stream);
}

int32_t dmrgk_probe_fp64(dmrgk_ctx* ctx, int32_t kind, int64_t iters, double* sink_dev, double* flops,
                         void* stream) {
    if (!ctx || !sink_dev || iters < 0) return fail(DMRGK_EINVAL, "probe_fp64: bad argument");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    int blocks = ctx->n_sm * 4, threads = 256;
    if (kind == 0 || (kind >= 2 && kind <= 4)) {
        // kind 0: 4 CTAs × 8 warps per SM; kinds 2-4: 1, 2, 3 CTAs × 4 warps per SM (3 × 4 is the
        // residency of the GEMM kernel) — the DMMA rate a box shows depends on the shape
        if (kind >= 2) {
            blocks = ctx->n_sm * (kind - 1);
            threads = 128;
        }
        probe_dmma_kernel<<<blocks, threads, 0, (cudaStream_t)stream>>>(iters, sink_dev);
        count_launch();
        if (flops) *flops = double(blocks) * (threads / 32) * double(iters) * 16.0 * 512.0;
    } else if (kind == 1) {
        probe_dfma_kernel<<<blocks, threads, 0, (cudaStream_t)stream>>>(iters, sink_dev);
        count_launch();
        if (flops) *flops = double(blocks) * threads * double(iters) * 32.0 * 2.0;
    } else {
        return fail(DMRGK_EINVAL, "probe_fp64: kind must be 0, 2, 3, 4 (DMMA shapes) or 1 (DFMA)");
    }
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

}  // extern "C"

// ---- host-only views of the planner's tiling rules (tests of the host logic) ------------------------
extern "C" int32_t dmrgk_plan_tile_cuts(int32_t extent, int32_t tile_max, int32_t* cuts, int32_t cap) {
    if (extent < 0 || (tile_max != 64 && tile_max != 128) || !cuts)
        return dmrgk::fail(DMRGK_EINVAL, "plan_tile_cuts: extent ≥ 0, tile_max 64 or 128, cuts not NULL");
    std::vector<int> c;
    dmrgk::tile_cuts(extent, tile_max, c);
    if (int32_t(c.size()) > cap) return dmrgk::fail(DMRGK_EINVAL, "plan_tile_cuts: %d boundaries need cap ≥ %d", int(c.size()), int(c.size()));
    for (size_t i = 0; i < c.size(); ++i) cuts[i] = c[i];
    return int32_t(c.size()) - 1;
}

extern "C" int32_t dmrgk_plan_tile_cost(int32_t rows, int32_t cols) {
    if (rows < 1 || cols < 1 || rows > 128 || cols > 64) return dmrgk::fail(DMRGK_EINVAL, "plan_tile_cost: 1 ≤ rows ≤ 128, 1 ≤ cols ≤ 64");
    return int32_t(dmrgk::tile_cost(rows, cols));
}
