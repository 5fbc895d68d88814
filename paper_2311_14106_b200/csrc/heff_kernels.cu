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

constexpr int BM = TILE_M, BN = TILE_N, BK = 16;
constexpr int NTHREADS = 128;           // 4 warps as 2×2, each a 32×32 warp tile = 4×4 DMMA frags
constexpr int STAGES = 3;
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

// Load one BK-deep stage of segment `sg` (k-tile kt) for tile (i0, j0) into sA / sB.
__device__ __forceinline__ void load_stage(const Seg& sg, const Bases& bases, int kt, int i0, int j0,
                                           int mrows, int ncols, double* sA, double* sB, int tid) {
    const double* A = reinterpret_cast<const double*>(bases.b[(sg.flags >> SEG_A_SEL_SHIFT) & 3u] + sg.A);
    const double* B = reinterpret_cast<const double*>(bases.b[(sg.flags >> SEG_B_SEL_SHIFT) & 3u] + sg.B);
    const int k0 = kt * BK;
    if (!(sg.flags & SEG_A_MMAJOR)) {
        // K-major: 64 rows × 8 chunks of 16 B; the k direction is covered by the zero padding of lda
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int c = tid + NTHREADS * j, row = c >> 3, ch = c & 7;
            bool p = (i0 + row) < mrows;
            const double* src = p ? A + int64_t(i0 + row) * sg.lda + k0 + ch * 2 : A;
            cp_async16(sA + row * KM_STRIDE + ch * 2, src, p);
        }
    } else {
        // M-major: 16 k-rows × 32 chunks
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int c = tid + NTHREADS * j, row = c >> 5, ch = c & 31;
            bool p = (k0 + row) < sg.klen && (i0 + ch * 2) < sg.lda;
            const double* src = p ? A + int64_t(k0 + row) * sg.lda + i0 + ch * 2 : A;
            cp_async16(sA + row * MN_STRIDE + ch * 2, src, p);
        }
    }
    if (!(sg.flags & SEG_B_NMAJOR)) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int c = tid + NTHREADS * j, row = c >> 3, ch = c & 7;
            bool p = (j0 + row) < ncols;
            const double* src = p ? B + int64_t(j0 + row) * sg.ldb + k0 + ch * 2 : B;
            cp_async16(sB + row * KM_STRIDE + ch * 2, src, p);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int c = tid + NTHREADS * j, row = c >> 5, ch = c & 31;
            bool p = (k0 + row) < sg.klen && (j0 + ch * 2) < sg.ldb;
            const double* src = p ? B + int64_t(k0 + row) * sg.ldb + j0 + ch * 2 : B;
            cp_async16(sB + row * MN_STRIDE + ch * 2, src, p);
        }
    }
}

// One k-tile (BK = 16, `nks` steps of 4) of a warp tile of FM × FN fragments.  FM, FN are compile-time
// so the accumulator indices are static and no DMMA carries a guard; the caller branches once per
// k-tile (warp-uniform) into the variant that matches the data this warp really holds.
template <int FM, int FN, bool FULLK>
__device__ __forceinline__ void mma_ktile(const double* __restrict__ pa, const double* __restrict__ pb,
                                          int a_fs, int b_fs, int a_ks4, int b_ks4, int nks,
                                          double (&acc)[4][4][2]) {
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
            for (int f = 0; f < FM; ++f) af[f] = pa[f * a_fs + ks * a_ks4];
#pragma unroll
            for (int f = 0; f < FN; ++f) bf[f] = pb[f * b_fs + ks * b_ks4];
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
}

template <int FM>
__device__ __forceinline__ void mma_ktile_n(int nfn, const double* pa, const double* pb, int a_fs, int b_fs,
                                            int a_ks4, int b_ks4, int nks, double (&acc)[4][4][2]) {
    switch (nfn) {
        case 1: mma_ktile<FM, 1, false>(pa, pb, a_fs, b_fs, a_ks4, b_ks4, nks, acc); break;
        case 2: mma_ktile<FM, 2, false>(pa, pb, a_fs, b_fs, a_ks4, b_ks4, nks, acc); break;
        case 3: mma_ktile<FM, 3, false>(pa, pb, a_fs, b_fs, a_ks4, b_ks4, nks, acc); break;
        default: mma_ktile<FM, 4, false>(pa, pb, a_fs, b_fs, a_ks4, b_ks4, nks, acc); break;
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

    // loader cursor: segment index, its descriptor (kept in registers), k-tile inside it
    int ld_seg = u.seg_begin, ld_kt = 0, ld_nkt = 0;
    Seg sg;
    sg.klen = 0;
    while (ld_seg < u.seg_end) {
        sg = segs[ld_seg];
        ld_nkt = (sg.klen + BK - 1) / BK;
        if (ld_nkt) break;
        ++ld_seg;
    }
    const int total = u.nkt;

    auto load_next = [&](int stage) {
        load_stage(sg, bases, ld_kt, u.i0, u.j0, u.mrows, u.ncols, smem + stage * STAGE_DOUBLES,
                   smem + stage * STAGE_DOUBLES + OPER_DOUBLES, tid);
        if (tid == 0) {
            notes[stage].flags = sg.flags;
            notes[stage].nks = min(BK / 4, (sg.klen - ld_kt * BK + 3) >> 2);
        }
        if (++ld_kt == ld_nkt) {
            ld_kt = 0;
            ld_nkt = 0;
            ++ld_seg;
            while (ld_seg < u.seg_end) {
                sg = segs[ld_seg];
                ld_nkt = (sg.klen + BK - 1) / BK;
                if (ld_nkt) break;
                ++ld_seg;
            }
        }
    };

    // prologue: STAGES−1 stages in flight
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < total) load_next(s);
        cp_async_commit();
    }

    uint32_t cur_flags = 0xffffffffu;
    int a_fs = 0, a_ks4 = 0, b_fs = 0, b_ks4 = 0, a_off = 0, b_off = 0;
    int stage = 0;
    for (int it = 0; it < total; ++it) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            const int nx = it + STAGES - 1;
            int ns = stage + STAGES - 1;
            if (ns >= STAGES) ns -= STAGES;
            if (nx < total) load_next(ns);
            cp_async_commit();
        }
        const StageNote note = notes[stage];
        if (note.flags != cur_flags) {
            cur_flags = note.flags;
            // element (i, k) of A: K-major i·20 + k, M-major k·68 + i; same for B with j
            const int a_is = (cur_flags & SEG_A_MMAJOR) ? 1 : KM_STRIDE;
            const int a_ks = (cur_flags & SEG_A_MMAJOR) ? MN_STRIDE : 1;
            const int b_js = (cur_flags & SEG_B_NMAJOR) ? 1 : KM_STRIDE;
            const int b_ks = (cur_flags & SEG_B_NMAJOR) ? MN_STRIDE : 1;
            a_off = (wm * 32 + g) * a_is + t4 * a_ks;
            b_off = (wn * 32 + g) * b_js + t4 * b_ks;
            a_fs = 8 * a_is;
            b_fs = 8 * b_js;
            a_ks4 = 4 * a_ks;
            b_ks4 = 4 * b_ks;
        }
        if (busy) {
            const double* pa = smem + stage * STAGE_DOUBLES + a_off;
            const double* pb = smem + stage * STAGE_DOUBLES + OPER_DOUBLES + b_off;
            if (nfm == 4 && nfn == 4 && note.nks == 4) {
                mma_ktile<4, 4, true>(pa, pb, a_fs, b_fs, a_ks4, b_ks4, 4, acc);
            } else {
                switch (nfm) {
                    case 1: mma_ktile_n<1>(nfn, pa, pb, a_fs, b_fs, a_ks4, b_ks4, note.nks, acc); break;
                    case 2: mma_ktile_n<2>(nfn, pa, pb, a_fs, b_fs, a_ks4, b_ks4, note.nks, acc); break;
                    case 3: mma_ktile_n<3>(nfn, pa, pb, a_fs, b_fs, a_ks4, b_ks4, note.nks, acc); break;
                    default: mma_ktile_n<4>(nfn, pa, pb, a_fs, b_fs, a_ks4, b_ks4, note.nks, acc); break;
                }
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

// a7: fixed-order sum of split-k partial tiles, σ_tile += Σ_s P_s (s ascending).
__global__ void __launch_bounds__(256)
heff_reduce_kernel(const RUnit* __restrict__ runits, Bases bases) {
    const RUnit u = runits[blockIdx.x];
    double* C = reinterpret_cast<double*>(bases.b[BASE_SIGMA] + u.C);
    const double* P = reinterpret_cast<const double*>(bases.b[BASE_WS] + u.P);
    const int half_cols = u.cols >> 1;   // cols is even (multiple of 16 or tile width 64)
    for (int e = threadIdx.x; e < u.rows * half_cols; e += 256) {
        const int r = e / half_cols, c = (e % half_cols) * 2;
        double2* p = reinterpret_cast<double2*>(C + int64_t(r) * u.ldc + c);
        double2 v = *p;
        for (int s = 0; s < u.n_split; ++s) {
            const double2 q = *reinterpret_cast<const double2*>(P + int64_t(s) * (BM * BN) + r * BN + c);
            v.x += q.x;
            v.y += q.y;
        }
        *p = v;
    }
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
    heff_reduce_kernel<<<unsigned(n), 256, 0, st>>>(runits_dev, bases);
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
