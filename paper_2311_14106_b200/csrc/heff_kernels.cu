// heff_kernels.cu — a5/a6/a7/a4: the grouped FP64 GEMM kernel of σ = Σ_k c_k (L_k ⊗ R_k) ψ
// (§II.A; 142, 158 §III.B: the quantum-number-decomposed "matrix and tensor algebra";
// BASELINE.json north_star: block-sparse dense GEMM pairs L_k·ψ·R_kᵀ).
//
// One kernel serves both phases.  A work unit is a ≤64×≤64 tile of an output block, summed over a
// list of segments (phase 1: one segment, T_k = c_k s · L_k ψ; phase 2: every task of the output
// block, σ += [T_1 … T_n]·[R_1 … R_n]ᵀ — the stacked-k form, so accumulators never leave registers
// between tasks).  FP64 tensor cores on sm_100a are reached through mma.sync.m8n8k4.f64 (SASS
// DMMA.8x8x4; tcgen05.mma has no f64 kind), so accumulators live in registers, operands are staged
// global→shared by cp.async in a multi-stage ring that runs across segment boundaries, and every
// fragment load is one conflict-free LDS.64 per lane (padded tile strides, see smem layout below).
#include "internal.h"

namespace dmrgk {

constexpr int BM = TILE_M, BN = TILE_N, BK = TILE_K;
constexpr int NTHREADS = 128;           // 4 warps as 2×2, each a 32×32 warp tile = 4×4 DMMA frags
constexpr int STAGES = 3;
constexpr int NCOPY = BK / 4;            // 16-byte copies per thread per operand per stage
constexpr int KM_CPR = BK / 2;           // 16-byte chunks per row of a K-major tile
constexpr int KM_RPP = NTHREADS / KM_CPR;  // rows covered by one pass of the CTA
// Shared tile layouts (doubles).  K-major operand tile: [64 rows][BK] with row stride 20
// (20·2 words ≡ 8 mod 32 → the 4 rows × 4 k of a half-warp LDS.64 hit 16 distinct bank pairs).
// MN-major operand tile: [BK rows][64] with row stride 68 (68·2 ≡ 8 mod 32, same argument with
// the roles of row and k exchanged).
constexpr int KM_STRIDE = BK + 4;       // 20
constexpr int MN_STRIDE = BM + 4;       // 68
constexpr int OPER_DOUBLES = (BM * KM_STRIDE > BK * MN_STRIDE) ? BM * KM_STRIDE : BK * MN_STRIDE;  // 1280
constexpr int STAGE_DOUBLES = 2 * OPER_DOUBLES;
constexpr int SMEM_BYTES = STAGES * STAGE_DOUBLES * 8;   // 61440 → 3 CTAs per SM

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, bool pred) {
    unsigned s = static_cast<unsigned>(__cvta_generic_to_shared(smem));
    int n = pred ? 16 : 0;   // src-size 0 → 16 bytes of zeros
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(n));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// ---- loader ------------------------------------------------------------------------------------
// Per-thread copy plan of one operand for the current segment: every stage this thread issues four
// 16-byte cp.async; everything that does not change from k-tile to k-tile is computed once per segment
// so the per-stage cost is a pointer bump and four predicated copies.
struct OpPlan {
    const char* ptr;      // source of copy j = 0 for the next k-tile (bytes)
    const char* safe;     // a valid address for predicated-off copies (block origin)
    long long step_j;     // source distance between copies j and j+1 (bytes)
    long long step_k;     // source advance per k-tile (bytes)
    uint32_t dst;         // destination of copy j = 0 inside the operand tile (bytes)
    uint32_t dst_step;    // destination distance between copies (bytes)
    int32_t mask;         // bit j: copy j is inside the operand along the M/N direction
    int32_t krow;         // MN-major: k-row of copy 0 (copy j is krow + 4j); K-major: −64 (never cut by klen)
};

// Operand tile origin `o0` (row/column offset of the tile in the block), `ext` = block extent in that
// direction (rows for K-major predication; ld for MN-major), `mn_major` = the tile is stored [k][i].
__device__ __forceinline__ void make_plan(OpPlan& p, const char* base, int ld, bool mn_major, int o0, int ext,
                                          int tid) {
    p.safe = base;
    if (!mn_major) {
        const int row = tid / KM_CPR, ch = tid % KM_CPR;   // copies j: rows row + KM_RPP·j, chunk ch
        p.ptr = base + (int64_t(o0 + row) * ld + ch * 2) * 8;
        p.step_j = int64_t(KM_RPP) * ld * 8;
        p.step_k = BK * 8;
        p.dst = (row * KM_STRIDE + ch * 2) * 8;
        p.dst_step = KM_RPP * KM_STRIDE * 8;
        int m = 0;
#pragma unroll
        for (int j = 0; j < NCOPY; ++j) m |= ((o0 + row + KM_RPP * j) < ext) << j;
        p.mask = m;
        p.krow = -64;
    } else {
        const int row = tid >> 5, ch = tid & 31;           // copies j: k-rows row + 4 j, chunk ch
        p.ptr = base + (int64_t(row) * ld + o0 + ch * 2) * 8;
        p.step_j = int64_t(4) * ld * 8;
        p.step_k = int64_t(BK) * ld * 8;
        p.dst = (row * MN_STRIDE + ch * 2) * 8;
        p.dst_step = 4 * MN_STRIDE * 8;
        p.mask = (o0 + ch * 2) < ext ? ((1 << NCOPY) - 1) : 0;
        p.krow = row;
    }
}

// Issue the four copies of one operand for a k-tile with `rem` contraction elements left (≥ 1).
__device__ __forceinline__ void issue_plan(OpPlan& p, uint32_t smem_operand, int rem) {
#pragma unroll
    for (int j = 0; j < NCOPY; ++j) {
        const bool ok = ((p.mask >> j) & 1) && (p.krow + 4 * j) < rem;
        const char* src = ok ? p.ptr + j * p.step_j : p.safe;
        const int n = ok ? 16 : 0;   // src-size 0 → 16 bytes of zeros
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(smem_operand + p.dst + j * p.dst_step),
                     "l"(src), "r"(n));
    }
    p.ptr += p.step_k;
}

// ---- consumer ----------------------------------------------------------------------------------
// One k-tile (BK = 16, `nks` steps of 4) of a warp tile of FM × FN fragments.  FM, FN and the operand
// layouts are compile-time: accumulator indices are static, no DMMA carries a guard, and every LDS.64
// has an immediate offset.  Element (i, k) of A sits at i·20 + k (K-major) or k·68 + i (M-major);
// the same for B with j.
template <int FM, int FN, bool AM, bool BN_, bool FULLK>
__device__ __forceinline__ void mma_ktile(const double* __restrict__ pa, const double* __restrict__ pb, int nks,
                                          double (&acc)[4][4][2]) {
    constexpr int a_fs = 8 * (AM ? 1 : KM_STRIDE), a_ks4 = 4 * (AM ? MN_STRIDE : 1);
    constexpr int b_fs = 8 * (BN_ ? 1 : KM_STRIDE), b_ks4 = 4 * (BN_ ? MN_STRIDE : 1);
    if (FULLK) {
#pragma unroll
        for (int ks = 0; ks < BK / 4; ++ks) {
            double af[FM], bf[FN];
#pragma unroll
            for (int f = 0; f < FM; ++f) af[f] = pa[f * a_fs + ks * a_ks4];
#pragma unroll
            for (int f = 0; f < FN; ++f) bf[f] = pb[f * b_fs + ks * b_ks4];
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    } else {
#pragma unroll 1
        for (int ks = 0; ks < nks; ++ks) {
            double af[FM], bf[FN];
#pragma unroll
            for (int f = 0; f < FM; ++f) af[f] = pa[f * a_fs];
#pragma unroll
            for (int f = 0; f < FN; ++f) bf[f] = pb[f * b_fs];
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
            pa += a_ks4;
            pb += b_ks4;
        }
    }
}

template <int FM, bool AM, bool BN_>
__device__ __forceinline__ void mma_ktile_n(int nfn, const double* pa, const double* pb, int nks,
                                            double (&acc)[4][4][2]) {
    switch (nfn) {
        case 1: mma_ktile<FM, 1, AM, BN_, false>(pa, pb, nks, acc); break;
        case 2: mma_ktile<FM, 2, AM, BN_, false>(pa, pb, nks, acc); break;
        case 3: mma_ktile<FM, 3, AM, BN_, false>(pa, pb, nks, acc); break;
        default: mma_ktile<FM, 4, AM, BN_, false>(pa, pb, nks, acc); break;
    }
}

// All fragment shapes of one operand-layout combination; branches are warp-uniform.
template <bool AM, bool BN_>
__device__ __forceinline__ void mma_layout(int nfm, int nfn, int nks, const double* sA, const double* sB, int wm,
                                           int wn, int g, int t4, double (&acc)[4][4][2]) {
    const double* pa = sA + (wm * 32 + g) * (AM ? 1 : KM_STRIDE) + t4 * (AM ? MN_STRIDE : 1);
    const double* pb = sB + (wn * 32 + g) * (BN_ ? 1 : KM_STRIDE) + t4 * (BN_ ? MN_STRIDE : 1);
    if (nfm == 4 && nfn == 4 && nks == BK / 4) {
        mma_ktile<4, 4, AM, BN_, true>(pa, pb, BK / 4, acc);
    } else {
        switch (nfm) {
            case 1: mma_ktile_n<1, AM, BN_>(nfn, pa, pb, nks, acc); break;
            case 2: mma_ktile_n<2, AM, BN_>(nfn, pa, pb, nks, acc); break;
            case 3: mma_ktile_n<3, AM, BN_>(nfn, pa, pb, nks, acc); break;
            default: mma_ktile_n<4, AM, BN_>(nfn, pa, pb, nks, acc); break;
        }
    }
}

// Per-stage note left by the loader for the consumers (read after the barrier that publishes the stage).
struct StageNote {
    uint32_t flags;   // segment flags (operand majors)
    int32_t nks;      // k-steps of 4 that hold data in this k-tile (1..4)
};

__global__ void __launch_bounds__(NTHREADS, 3)
heff_gemm_dmma_kernel(const Unit* __restrict__ units, const Seg* __restrict__ segs, Bases bases) {
    extern __shared__ __align__(16) double smem[];
    __shared__ StageNote notes[STAGES];
    const Unit u = units[blockIdx.x];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp >> 1, wn = warp & 1;
    const int g = lane >> 2, t4 = lane & 3;
    const uint32_t smem_base = static_cast<uint32_t>(__cvta_generic_to_shared(smem));

    // rows / columns of this tile that hold data, in 8-wide fragments, for this warp
    const int rows_t = min(BM, u.mrows - u.i0);
    const int cols_t = min(BN, u.ncols_st - u.j0);
    const int nfm = max(0, min(4, (rows_t - wm * 32 + 7) >> 3));
    const int nfn = max(0, min(4, (min(BN, u.ncols - u.j0) - wn * 32 + 7) >> 3));
    const bool busy = nfm > 0 && nfn > 0;

    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // loader state: segment cursor, remaining contraction length of the segment, the two copy plans
    int ld_seg = u.seg_begin, ld_rem = 0;
    uint32_t ld_flags = 0;
    OpPlan planA, planB;
    auto open_segment = [&]() {
        while (ld_seg < u.seg_end) {
            const Seg sg = segs[ld_seg];
            if (sg.klen > 0) {
                ld_rem = sg.klen;
                ld_flags = sg.flags;
                const char* A = reinterpret_cast<const char*>(bases.b[(sg.flags >> SEG_A_SEL_SHIFT) & 3u] + sg.A);
                const char* B = reinterpret_cast<const char*>(bases.b[(sg.flags >> SEG_B_SEL_SHIFT) & 3u] + sg.B);
                const bool am = (sg.flags & SEG_A_MMAJOR) != 0, bn = (sg.flags & SEG_B_NMAJOR) != 0;
                make_plan(planA, A, sg.lda, am, u.i0, am ? sg.lda : u.mrows, tid);
                make_plan(planB, B, sg.ldb, bn, u.j0, bn ? sg.ldb : u.ncols, tid);
                return;
            }
            ++ld_seg;
        }
    };
    open_segment();
    const int total = u.nkt;

    auto load_next = [&](int stage) {
        const uint32_t sA = smem_base + stage * (STAGE_DOUBLES * 8);
        issue_plan(planA, sA, ld_rem);
        issue_plan(planB, sA + OPER_DOUBLES * 8, ld_rem);
        if (tid == 0) {
            notes[stage].flags = ld_flags;
            notes[stage].nks = min(BK / 4, (ld_rem + 3) >> 2);
        }
        ld_rem -= BK;
        if (ld_rem <= 0) {
            ++ld_seg;
            open_segment();
        }
    };

    // prologue: STAGES−1 stages in flight
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < total) load_next(s);
        cp_async_commit();
    }

    int stage = 0;
    for (int it = 0; it < total; ++it) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            int ns = stage + STAGES - 1;
            if (ns >= STAGES) ns -= STAGES;
            if (it + STAGES - 1 < total) load_next(ns);
            cp_async_commit();
        }
        if (busy) {
            const StageNote note = notes[stage];
            const double* sA = smem + stage * STAGE_DOUBLES;
            const double* sB = sA + OPER_DOUBLES;
            switch (note.flags & (SEG_A_MMAJOR | SEG_B_NMAJOR)) {
                case 0: mma_layout<false, false>(nfm, nfn, note.nks, sA, sB, wm, wn, g, t4, acc); break;
                case SEG_A_MMAJOR: mma_layout<true, false>(nfm, nfn, note.nks, sA, sB, wm, wn, g, t4, acc); break;
                case SEG_B_NMAJOR: mma_layout<false, true>(nfm, nfn, note.nks, sA, sB, wm, wn, g, t4, acc); break;
                default: mma_layout<true, true>(nfm, nfn, note.nks, sA, sB, wm, wn, g, t4, acc); break;
            }
        }
        if (++stage == STAGES) stage = 0;
    }
    cp_async_wait<0>();

    // epilogue: lane holds C[row g][cols 2·t4, 2·t4+1] of each 8×8 fragment
    double* C = reinterpret_cast<double*>(bases.b[(u.mode >> UNIT_C_SEL_SHIFT) & 3u] + u.C);
    const bool accum = (u.mode & UNIT_ACCUM) != 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = wm * 32 + i * 8 + g;
        if (r >= rows_t) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int c = wn * 32 + j * 8 + 2 * t4;
            if (c >= cols_t) continue;
            double2* p = reinterpret_cast<double2*>(C + int64_t(r) * u.ldc + c);
            double2 v;
            v.x = (u.j0 + c < u.ncols) ? u.alpha * acc[i][j][0] : 0.0;
            v.y = (u.j0 + c + 1 < u.ncols) ? u.alpha * acc[i][j][1] : 0.0;
            if (accum) {
                double2 o = *p;
                v.x += o.x;
                v.y += o.y;
            }
            *p = v;
        }
    }
}

// Scalar check kernel over the same work lists: one thread per 4×8 patch, plain FMA loops reading
// global memory directly.  A debugging aid (dmrgk_heff_opts.kernel = 1), never the product path.
__global__ void __launch_bounds__(NTHREADS)
heff_gemm_scalar_kernel(const Unit* __restrict__ units, const Seg* __restrict__ segs, Bases bases) {
    const Unit u = units[blockIdx.x];
    const int rows_t = min(BM, u.mrows - u.i0);
    const int cols_t = min(BN, u.ncols_st - u.j0);
    double* C = reinterpret_cast<double*>(bases.b[(u.mode >> UNIT_C_SEL_SHIFT) & 3u] + u.C);
    for (int e = threadIdx.x; e < rows_t * cols_t; e += NTHREADS) {
        const int r = e / cols_t, c = e % cols_t;
        const int i = u.i0 + r, j = u.j0 + c;
        double s = 0.0;
        if (j < u.ncols) {
            for (int sidx = u.seg_begin; sidx < u.seg_end; ++sidx) {
                const Seg sg = segs[sidx];
                const double* A = reinterpret_cast<const double*>(bases.b[(sg.flags >> SEG_A_SEL_SHIFT) & 3u] + sg.A);
                const double* B = reinterpret_cast<const double*>(bases.b[(sg.flags >> SEG_B_SEL_SHIFT) & 3u] + sg.B);
                for (int k = 0; k < sg.klen; ++k) {
                    double a = (sg.flags & SEG_A_MMAJOR) ? A[int64_t(k) * sg.lda + i] : A[int64_t(i) * sg.lda + k];
                    double b = (sg.flags & SEG_B_NMAJOR) ? B[int64_t(k) * sg.ldb + j] : B[int64_t(j) * sg.ldb + k];
                    s = fma(a, b, s);
                }
            }
        }
        double v = u.alpha * s;
        double* p = C + int64_t(r) * u.ldc + c;
        if (u.mode & UNIT_ACCUM) v += *p;
        *p = v;
    }
}

// a7: fixed-order sum of split-k partial tiles, σ_tile += Σ_s P_s (s ascending).  Eight CTAs per tile
// (one 8-row slab each, one double2 per thread) so that even a handful of output tiles fills the GPU;
// the partial loads of four splits are issued together, the additions stay in split order.
constexpr int RED_SLABS = BM / 8;
__global__ void __launch_bounds__(256)
heff_reduce_kernel(const RUnit* __restrict__ runits, Bases bases) {
    const RUnit u = runits[blockIdx.x / RED_SLABS];
    const int r = (blockIdx.x % RED_SLABS) * 8 + (threadIdx.x >> 5);
    const int c = (threadIdx.x & 31) * 2;
    if (r >= u.rows || c >= u.cols) return;   // cols is even (multiple of 16 or the tile width 64)
    double2* p = reinterpret_cast<double2*>(reinterpret_cast<double*>(bases.b[BASE_SIGMA] + u.C) + int64_t(r) * u.ldc + c);
    const double2* P = reinterpret_cast<const double2*>(reinterpret_cast<const double*>(bases.b[BASE_WS] + u.P) + r * BN + c);
    double2 v = *p;
    int s = 0;
    for (; s + 4 <= u.n_split; s += 4) {
        double2 q[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) q[j] = P[int64_t(s + j) * (BM * BN / 2)];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            v.x += q[j].x;
            v.y += q[j].y;
        }
    }
    for (; s < u.n_split; ++s) {
        const double2 q = P[int64_t(s) * (BM * BN / 2)];
        v.x += q.x;
        v.y += q.y;
    }
    *p = v;
}

// a4: diag(H_eff)[i, j] += Σ_t alpha_t · L_t[i, i] · R_t[j, j] over the block's diagonal tasks.
// grid = (tiles of 32×32 over the largest block, n_blocks); tasks are staged 64 at a time.
__global__ void __launch_bounds__(256)
heff_diag_kernel(const DiagBlock* __restrict__ blocks, const DiagTask* __restrict__ tasks,
                 double* __restrict__ diag, Bases bases) {
    const DiagBlock b = blocks[blockIdx.y];
    const int tiles_c = (b.cols + 31) / 32, tiles_r = (b.rows + 31) / 32;
    __shared__ double sl[64][32], sr[64][33];
    for (int tile = blockIdx.x; tile < tiles_r * tiles_c; tile += gridDim.x) {
        const int i0 = (tile / tiles_c) * 32, j0 = (tile % tiles_c) * 32;
        const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 8 rows of 32 lanes
        double acc[4] = {0, 0, 0, 0};
        for (int t0 = b.t_begin; t0 < b.t_end; t0 += 64) {
            const int nt = min(64, b.t_end - t0);
            __syncthreads();
            for (int e = threadIdx.x; e < nt * 32; e += 256) {
                const int t = e >> 5, x = e & 31;
                const DiagTask tk = tasks[t0 + t];
                const double* L = reinterpret_cast<const double*>(bases.b[tk.sel & 3u] + tk.L);
                const double* R = reinterpret_cast<const double*>(bases.b[(tk.sel >> 2) & 3u] + tk.R);
                sl[t][x] = (i0 + x < b.rows) ? tk.alpha * L[int64_t(i0 + x) * (tk.ldl + 1)] : 0.0;
                sr[t][x] = (j0 + x < b.cols) ? R[int64_t(j0 + x) * (tk.ldr + 1)] : 0.0;
            }
            __syncthreads();
            for (int t = 0; t < nt; ++t) {
                const double r = sr[t][tx];
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[q] = fma(sl[t][ty + 8 * q], r, acc[q]);
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int i = i0 + ty + 8 * q, j = j0 + tx;
            if (i < b.rows && j < b.cols) diag[b.off + int64_t(i) * b.ld + j] += acc[q];
        }
    }
}

int32_t gemm_kernel_setup() {
    DMRGK_CUDA(cudaFuncSetAttribute(heff_gemm_dmma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
    return DMRGK_OK;
}

int32_t launch_gemm_units(int kernel, const Unit* units_dev, const Seg* segs_dev, int64_t n_units,
                          const Bases& bases, cudaStream_t st) {
    if (n_units <= 0) return DMRGK_OK;
    if (n_units > 0x7fffffffLL) return fail(DMRGK_EINVAL, "too many work units in one launch: %lld", (long long)n_units);
    if (kernel == 1)
        heff_gemm_scalar_kernel<<<unsigned(n_units), NTHREADS, 0, st>>>(units_dev, segs_dev, bases);
    else
        heff_gemm_dmma_kernel<<<unsigned(n_units), NTHREADS, SMEM_BYTES, st>>>(units_dev, segs_dev, bases);
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

int32_t launch_reduce(const RUnit* runits_dev, int64_t n, const Bases& bases, cudaStream_t st) {
    if (n <= 0) return DMRGK_OK;
    heff_reduce_kernel<<<unsigned(n * RED_SLABS), 256, 0, st>>>(runits_dev, bases);
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

int32_t launch_diag(const DiagBlock* blocks_dev, const DiagTask* tasks_dev, int64_t n_blocks,
                    double* diag, const Bases& bases, cudaStream_t st) {
    if (n_blocks <= 0) return DMRGK_OK;
    dim3 grid(64, unsigned(n_blocks));
    heff_diag_kernel<<<grid, 256, 0, st>>>(blocks_dev, tasks_dev, diag, bases);
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

}  // namespace dmrgk
