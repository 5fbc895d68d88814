// heff_kernels.cu — a5/a6/a7/a4: the grouped FP64 GEMM kernel of σ = Σ_k c_k (L_k ⊗ R_k) ψ
// (§II.A; 142, 158 §III.B: the quantum-number-decomposed "matrix and tensor algebra";
// BASELINE.json north_star: block-sparse dense GEMM pairs L_k·ψ·R_kᵀ).
//
// One kernel serves both phases.  A work unit is a ≤64×≤64 tile of an output block, summed over a
// list of segments (phase 1: one segment, T_k = c_k s · L_k ψ; phase 2: every task of the output
// block, σ += [T_1 … T_n]·[R_1 … R_n]ᵀ — the stacked-k form, so accumulators never leave registers
// between tasks).  FP64 tensor cores on sm_100a are reached through mma.sync.m8n8k4.f64 (SASS
// DMMA.8x8x4; tcgen05.mma has no f64 kind), so accumulators live in registers.
//
// Staging (round 2): operand tiles are fetched by the TMA unit.  Every block is stored in the panel
// layout (internal.h), in which a ≤64×16 K-major tile — and each 16×16 piece of an MN-major one — is
// one contiguous chunk, already swizzled; one elected lane of a dedicated PRODUCER warp issues 2–8
// cp.async.bulk copies (SASS UBLKCP) per k-tile of 32 that complete on the stage's `full` mbarrier, the four
// CONSUMER warps wait on it, run LDS.64 + DMMA only, and release the stage through its `empty` mbarrier.
// There is no __syncthreads and no per-thread address arithmetic in the k-loop.  The kernel is persistent:
// 3 CTAs per SM (2 stages of 32 KB each) claim work units from a device-side queue; the units of a block are
// balanced tiles whose fragments are split evenly over the warp rows and columns (internal.h tile_cuts).
// Design choices and their measurements: DESIGN.md §4.1, profiles/r2_tma_summary.md, r2_ragged.md,
// r2_final_summary.md.
#include "internal.h"
#include <algorithm>

namespace dmrgk {

// The kernel is a template on WM, the 8-row fragments a warp holds along M: WM = 4 gives the 64×64 CTA
// tile (2×2 warps of 32×32), WM = 8 the tall 128×64 tile (2×2 warps of 64×32).
constexpr int BN = TILE_N, BK = TILE_K;
constexpr int NTHREADS = 128;
constexpr int B_DOUBLES = BN * BK;       // the B operand tile, dense 128-byte rows
constexpr int MN_PANEL = BK * 16;        // doubles of one 16-column panel of an MN-major tile (BK k-rows)
constexpr int stage_doubles(int wm) { return wm * 16 * BK + B_DOUBLES; }
constexpr int smem_bytes(int wm, int stages) { return stages * stage_doubles(wm) * 8; }

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
// TMA bulk copy global → shared, completing `bytes` on the mbarrier (bytes a multiple of 16)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// ---- consumer ----------------------------------------------------------------------------------
// Shared image of an operand tile (doubles from the operand's origin in the stage):
//   K-major  (stored [i][k]): element (i, k) at (k >> 4)·1024 + i·16 + ((k & 15) xor ((i & 3) << 2))
//                                                            [BK/16 k-panels × tile rows (64 | 128) × 16]
//   MN-major (stored [k][i]): element (i, k) at (i >> 4)·16·BK + k·16 + ((i & 15) xor ((k & 3) << 2))
//                                                                    [4 panels × BK k-rows × 16]
// A warp owns the 8-row fragments F0 … F0 + n − 1 of its operand tile (F0 = 0 for warp row/column 0, the
// tile's fragments are split evenly over the two warp rows/columns, per unit).  A lane (g = lane >> 2,
// t4 = lane & 3) of the warp's fragment f reads row i = (F0 + f)·8 + g at k = 4·ks + t4:
//   K-major : k0 + f·128 + (ks >> 2)·1024 + (((ks & 3) xor (g & 3)) << 2)    with k0 = (F0·8 + g)·16 + t4
//   MN-major: m[f & 1] + (f >> 1)·16·BK + ks·64     with m[h] = ((F0 + h) >> 1)·16·BK + t4·16 + ((8·((F0 + h) & 1) + g) xor (t4 << 2))
// In both cases the 16 lanes of a half-warp hit 16 distinct 8-byte banks.
struct FragBase {
    int k0, m0, m1;
};
__device__ __forceinline__ FragBase make_frag_base(int origin, int F0, int g, int t4) {
    FragBase b;
    b.k0 = origin + (F0 * 8 + g) * 16 + t4;
    b.m0 = origin + (F0 >> 1) * MN_PANEL + t4 * 16 + ((8 * (F0 & 1) + g) ^ (t4 << 2));
    b.m1 = origin + ((F0 + 1) >> 1) * MN_PANEL + t4 * 16 + ((8 * ((F0 + 1) & 1) + g) ^ (t4 << 2));
    return b;
}
// KSTRIDE: doubles between the 16-column k-panels of a K-major operand tile (its rows × 16)
template <bool MN, int KSTRIDE>
__device__ __forceinline__ double frag(const double* __restrict__ st, const FragBase& b, int g3, int f, int ks) {
    if (MN) return st[((f & 1) ? b.m1 : b.m0) + (f >> 1) * MN_PANEL + ks * 64];
    return st[b.k0 + f * 128 + (ks >> 2) * KSTRIDE + (((ks & 3) ^ g3) << 2)];
}

// One k-tile (BK = 16, `nks` steps of 4) of a warp tile of FM × FN fragments.  FM, FN and the operand
// layouts are compile-time: accumulator indices are static and no DMMA carries a guard.
template <int WM, int FM, int FN, bool AM, bool BN_, bool FULLK>
__device__ __forceinline__ void mma_ktile(const double* __restrict__ st, const FragBase& fa, const FragBase& fb, int g3,
                                          int nks, double (&acc)[WM][4][2]) {
    constexpr int KA = WM * 256, KB = 1024;
    if (FULLK) {
#pragma unroll
        for (int ks = 0; ks < BK / 4; ++ks) {
            double af[FM], bf[FN];
#pragma unroll
            for (int f = 0; f < FM; ++f) af[f] = frag<AM, KA>(st, fa, g3, f, ks);
#pragma unroll
            for (int f = 0; f < FN; ++f) bf[f] = frag<BN_, KB>(st, fb, g3, f, ks);
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
            for (int f = 0; f < FM; ++f) af[f] = frag<AM, KA>(st, fa, g3, f, ks);
#pragma unroll
            for (int f = 0; f < FN; ++f) bf[f] = frag<BN_, KB>(st, fb, g3, f, ks);
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
}

template <int WM, int FM, bool AM, bool BN_>
__device__ __forceinline__ void mma_ktile_n(int nfn, const double* st, const FragBase& fa, const FragBase& fb, int g3,
                                            int nks, double (&acc)[WM][4][2]) {
    switch (nfn) {
        case 1: mma_ktile<WM, FM, 1, AM, BN_, false>(st, fa, fb, g3, nks, acc); break;
        case 2: mma_ktile<WM, FM, 2, AM, BN_, false>(st, fa, fb, g3, nks, acc); break;
        case 3: mma_ktile<WM, FM, 3, AM, BN_, false>(st, fa, fb, g3, nks, acc); break;
        default: mma_ktile<WM, FM, 4, AM, BN_, false>(st, fa, fb, g3, nks, acc); break;
    }
}

// All fragment shapes of one operand-layout combination; branches are warp-uniform.
template <int WM, bool AM, bool BN_>
__device__ __forceinline__ void mma_layout(int nfm, int nfn, int nks, const double* st, const FragBase& fa,
                                           const FragBase& fb, int g3, double (&acc)[WM][4][2]) {
    if (nfm == WM && nfn == 4 && nks == BK / 4) {
        mma_ktile<WM, WM, 4, AM, BN_, true>(st, fa, fb, g3, BK / 4, acc);
    } else {
        if constexpr (WM > 4) {
            switch (nfm) {
                case 1: mma_ktile_n<WM, 1, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                case 2: mma_ktile_n<WM, 2, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                case 3: mma_ktile_n<WM, 3, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                case 4: mma_ktile_n<WM, 4, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                case 5: mma_ktile_n<WM, 5, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                case 6: mma_ktile_n<WM, 6, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                case 7: mma_ktile_n<WM, 7, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                default: mma_ktile_n<WM, 8, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
            }
        } else {
            switch (nfm) {
                case 1: mma_ktile_n<WM, 1, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                case 2: mma_ktile_n<WM, 2, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                case 3: mma_ktile_n<WM, 3, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
                default: mma_ktile_n<WM, 4, AM, BN_>(nfn, st, fa, fb, g3, nks, acc); break;
            }
        }
    }
}

// Per-stage note left by the producer for the consumers (published by the stage's full barrier).
struct StageNote {
    uint32_t flags;   // segment flags (operand majors)
    int32_t nks;      // k-steps of 4 that hold data in this k-tile (1..BK/4)
};

// ---- persistent, warp-specialised form (the product path) ------------------------------------------
// grid = CTAS_PER_SM · n_SM CTAs of 5 warps.  Warp 4 is the PRODUCER: it claims work units from a
// device-side queue (atomicAdd on a per-launch counter; units are sorted longest first, so this is LPT
// list scheduling), publishes each unit's descriptor in a small shared-memory ring and streams the
// operand tiles of unit after unit through the stage ring with cp.async.bulk — it never waits for a
// unit to finish, so the pipeline does not drain between units and the unit-descriptor, segment-
// descriptor and first-tile latencies that a one-unit-per-CTA launch pays at every CTA start are
// hidden.  Warps 0-3 are CONSUMERS: wait full → LDS.64 + DMMA → arrive empty; at a unit's end each
// warp stores its own fragment rows and moves on (no CTA-wide barrier anywhere after the prologue).
// The stop signal is a descriptor with nkt = 0 published through the same ring on a data-less tile.
constexpr int P_NTHREADS = 160;
constexpr int EAGER = 1 << 30;           // LOOKAHEAD value: claim whole units ahead (variant 5)
constexpr int LATE = 8;                  // LOOKAHEAD of the product path, in k-tiles

template <int WM, int STAGES, int MIN_CTAS, int LOOKAHEAD>
__global__ void __launch_bounds__(P_NTHREADS, MIN_CTAS)
heff_gemm_dmma_persistent_kernel(const Unit* __restrict__ units, const Seg* __restrict__ segs, int n_units,
                                 int* __restrict__ queue_head, Bases bases) {
    constexpr int RING = STAGES + 1;       // a unit has ≥ 1 tile, the producer runs ≤ STAGES tiles ahead
    constexpr int A_DOUBLES = WM * 16 * BK, STAGE_DOUBLES = A_DOUBLES + B_DOUBLES;
    extern __shared__ __align__(128) double smem[];
    __shared__ __align__(8) unsigned long long bars[2 * STAGES];   // full[0..S), empty[S..2S)
    __shared__ StageNote notes[STAGES];
    __shared__ __align__(16) Unit ring[RING];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t smem_base = smem_u32(smem), bar0 = smem_u32(bars);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar0 + s * 8, 1);                   // full: the producer's arrive (+ the copies' bytes)
            mbar_init(bar0 + (STAGES + s) * 8, 4);        // empty: one arrive per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    if (warp == 4) {
        // ================================ PRODUCER ================================
        auto load_unit = [&](int idx, int4 (&w)[4]) {
            const int4* p = reinterpret_cast<const int4*>(units + idx);
#pragma unroll
            for (int q = 0; q < 4; ++q) w[q] = __ldg(p + q);
        };
        auto load_seg = [&](int seg, int4& lo, int4& hi) {
            lo = __ldg(reinterpret_cast<const int4*>(segs + seg));
            hi = __ldg(reinterpret_cast<const int4*>(segs + seg) + 1);
        };
        auto claim_async = [&]() -> int {      // only lane 0 holds the result until it is broadcast
            int v = 0;
            if (lane == 0) v = atomicAdd(queue_head, 1);
            return v;
        };
        // Look-ahead: the dependent loads between two units — queue index (atomic), unit descriptor, first
        // segment descriptor — are requested ahead of time so that no global-memory latency sits between
        // units.  Two schemes (template parameter LOOKAHEAD):
        //  * LATE, the product path, works in k-tiles: the next unit is claimed only when fewer than
        //    LOOKAHEAD tiles of the current one are left to issue, its descriptor follows two and its first
        //    segment four tiles later (a unit shorter than that pays the latencies).  A unit then starts a
        //    few tile times after its claim, so queue neighbours — the tiles of one (output block, k-range),
        //    which read the same T row tiles and R column tiles — run at the same time on different SMs and
        //    share those reads in L2.
        //  * EAGER (variant 5, kept for measurement) works in whole units: the index of the unit three
        //    ahead, the descriptors of the units one and two ahead and the first segment of the unit one
        //    ahead are in flight, each requested one unit before it is used.  Nothing ever blocks, but a
        //    CTA runs queue neighbours one after the other instead of next to other CTAs: same speed on
        //    config 4 (bound by the DMMA pipe), 1.6× the DRAM traffic (23 against 14 GB per launch,
        //    profiles/r2_final_summary.md).
        int4 uw[4];
        int4 s_lo = make_int4(0, 0, 0, 0), s_hi = s_lo, ns_lo = s_lo, ns_hi = s_lo;
        int nxt = 0, nx2 = 0, nx3 = 0;                  // EAGER: queue indices of the units one, two, three ahead
        int4 nw[4], n2w[4];                              //        descriptors of the units one and two ahead
        int idA = 0, stA = 0;                           // LATE:  the claimed next unit; 0 none, 1 claimed, 2 descriptor
        bool ended = false;                              //        requested, 4 first segment requested, 5 end of queue
        int4 wA[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) uw[q] = nw[q] = n2w[q] = wA[q] = s_lo;
        // LATE only, once per issued tile: one chain step when its trigger point is reached — claim with
        // LOOKAHEAD tiles left, descriptor two tiles later, first segment two tiles after that
        auto chain_claim = [&]() {
            idA = claim_async();
            stA = 1;
        };
        auto chain_desc = [&]() {
            idA = __shfl_sync(0xffffffffu, idA, 0);
            if (idA >= n_units) {
                stA = 5;
                ended = true;
            } else {
                load_unit(idA, wA);
                stA = 2;
            }
        };
        auto chain_seg = [&]() {
            load_seg(wA[2].z, ns_lo, ns_hi);
            stA = 4;
        };
        auto feed = [&](int tiles_left) {
            if (stA == 0) {
                if (!ended && tiles_left < LOOKAHEAD) chain_claim();
            } else if (stA == 1) {
                if (tiles_left < LOOKAHEAD - 2) chain_desc();
            } else if (stA == 2) {
                if (tiles_left < LOOKAHEAD - 4) chain_seg();
            }
        };
        // make the next unit current (uw, s_lo, s_hi); false at the end of the queue
        auto rotate = [&]() -> bool {
            if constexpr (LOOKAHEAD == EAGER) {
                const int cur = nxt;
                if (cur >= n_units) return false;
                s_lo = ns_lo;
                s_hi = ns_hi;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    uw[q] = nw[q];
                    nw[q] = n2w[q];
                }
                nxt = nx2;
                if (nxt < n_units) load_seg(nw[2].z, ns_lo, ns_hi);
                nx2 = nx3;
                if (nx2 < n_units) load_unit(nx2, n2w);
                nx3 = __shfl_sync(0xffffffffu, claim_async(), 0);
                return true;
            } else {
                if (stA == 0) {                        // finish whatever is missing, synchronously
                    if (ended) return false;
                    chain_claim();
                }
                if (stA == 1) chain_desc();
                if (stA == 5) return false;
                if (stA == 2) chain_seg();
                s_lo = ns_lo;
                s_hi = ns_hi;
#pragma unroll
                for (int q = 0; q < 4; ++q) uw[q] = wA[q];
                stA = 0;
                return true;
            }
        };
        if constexpr (LOOKAHEAD == EAGER) {             // prime the chain: units 0, 1, 2 of this CTA and the index of the fourth
            nxt = __shfl_sync(0xffffffffu, claim_async(), 0);
            nx2 = __shfl_sync(0xffffffffu, claim_async(), 0);
            nx3 = __shfl_sync(0xffffffffu, claim_async(), 0);
            if (nxt < n_units) load_unit(nxt, nw);
            if (nx2 < n_units) load_unit(nx2, n2w);
            if (nxt < n_units) load_seg(nw[2].z, ns_lo, ns_hi);
        }
        int T = 0, stage = 0, ring_pos = 0;
        uint32_t eph = 1;                                 // parity to wait for on empty[stage]: (T/S − 1) & 1
        auto advance_stage = [&]() {
            ++T;
            if (++stage == STAGES) {
                stage = 0;
                eph ^= 1u;
            }
        };
        bool more = rotate();
        while (more) {
            // fields of the unit (Unit layout: C, alpha | c_rp, i0, j0, mrows | ncols, ncols_st, seg_begin, seg_end | mode, nkt, -, tile)
            const int i0 = uw[1].y, j0 = uw[1].z, ncols = uw[2].x;
            const int seg_begin = uw[2].z, seg_end = uw[2].w;
            const int rows_a = int(uint32_t(uw[3].w) & 0xffffu), cols_b = min(int(uint32_t(uw[3].w) >> 16), ncols - j0);
            const int npa = (rows_a + 15) >> 4, npb = (cols_b + 15) >> 4;
            int tiles_left = uw[3].y;                            // nkt of the unit
            bool first = true;
            for (int sg = seg_begin; sg < seg_end; ++sg) {       // (s_lo, s_hi) hold segment sg
                const unsigned long long sA = (unsigned long long)(unsigned)s_lo.x | ((unsigned long long)(unsigned)s_lo.y << 32);
                const unsigned long long sB = (unsigned long long)(unsigned)s_lo.z | ((unsigned long long)(unsigned)s_lo.w << 32);
                const int a_rp = s_hi.x, b_rp = s_hi.y, klen = s_hi.z;
                const uint32_t flags = uint32_t(s_hi.w);
                if (sg + 1 < seg_end) {                   // the next descriptor travels while this segment streams
                    s_lo = __ldg(reinterpret_cast<const int4*>(segs + sg + 1));
                    s_hi = __ldg(reinterpret_cast<const int4*>(segs + sg + 1) + 1);
                }
                const bool am = (flags & SEG_A_MMAJOR) != 0, bn = (flags & SEG_B_NMAJOR) != 0;
                const char* A = reinterpret_cast<const char*>(bases.b[(flags >> SEG_A_SEL_SHIFT) & 3u] + sA);
                const char* B = reinterpret_cast<const char*>(bases.b[(flags >> SEG_B_SEL_SHIFT) & 3u] + sB);
                for (int k0 = 0; k0 < klen; k0 += BK) {
                    if (T >= STAGES) mbar_wait(bar0 + (STAGES + stage) * 8, eph);
                    const int nk = min(BK, klen - k0), nk4 = (nk + 3) & ~3, nkp = (nk + 15) >> 4;
                    const uint32_t bytes_a = am ? uint32_t(npa * nk4 * 128) : uint32_t(nkp * rows_a * 128);
                    const uint32_t bytes_b = bn ? uint32_t(npb * nk4 * 128) : uint32_t(nkp * cols_b * 128);
                    const uint32_t full = bar0 + stage * 8;
                    if (lane == 0) {
                        if (first) {
                            int4* slot = reinterpret_cast<int4*>(&ring[ring_pos]);
#pragma unroll
                            for (int q = 0; q < 4; ++q) slot[q] = uw[q];
                        }
                        notes[stage].flags = flags;
                        notes[stage].nks = nk4 >> 2;
                        mbar_expect_tx(full, bytes_a + bytes_b);
                    }
                    // copies of this tile: a K-major operand is BK/16 k-panels of (rows × 128 B), an MN-major
                    // one is ceil(extent/16) panels of (nk4 × 128 B); the elected lane issues them one by one
                    // (UBLKCP takes uniform operands, so spreading them over lanes would be serialised anyway)
                    if (lane == 0) {
                        const uint32_t dA = smem_base + stage * (STAGE_DOUBLES * 8), dB = dA + A_DOUBLES * 8;
                        if (!am) {
                            for (int kp = 0; kp < nkp; ++kp)
                                bulk_g2s(dA + kp * (WM * 2048), A + (int64_t((k0 >> 4) + kp) * a_rp + i0) * 128, uint32_t(rows_a * 128), full);
                        } else {
                            for (int pp = 0; pp < npa; ++pp)
                                bulk_g2s(dA + pp * (MN_PANEL * 8), A + (int64_t((i0 >> 4) + pp) * a_rp + k0) * 128, uint32_t(nk4 * 128), full);
                        }
                        if (!bn) {
                            for (int kp = 0; kp < nkp; ++kp)
                                bulk_g2s(dB + kp * 8192, B + (int64_t((k0 >> 4) + kp) * b_rp + j0) * 128, uint32_t(cols_b * 128), full);
                        } else {
                            for (int pp = 0; pp < npb; ++pp)
                                bulk_g2s(dB + pp * (MN_PANEL * 8), B + (int64_t((j0 >> 4) + pp) * b_rp + k0) * 128, uint32_t(nk4 * 128), full);
                        }
                    }
                    if (first) {
                        first = false;
                        if (++ring_pos == RING) ring_pos = 0;
                    }
                    advance_stage();
                    if constexpr (LOOKAHEAD != EAGER) feed(--tiles_left);
                }
            }
            more = rotate();
        }
        // stop sentinel on a data-less tile
        if (T >= STAGES) mbar_wait(bar0 + (STAGES + stage) * 8, eph);
        if (lane == 0) {
            int4* slot = reinterpret_cast<int4*>(&ring[ring_pos]);
#pragma unroll
            for (int q = 0; q < 4; ++q) slot[q] = make_int4(0, 0, 0, 0);      // nkt = 0
            mbar_arrive(bar0 + stage * 8);
        }
        return;
    }

    // ================================ CONSUMERS ================================
    const int wm = warp >> 1, wn = warp & 1;
    const int g = lane >> 2, t4 = lane & 3, g3 = g & 3;
    int stage = 0, ring_pos = 0;
    uint32_t ph = 0;
    while (true) {
        mbar_wait(bar0 + stage * 8, ph);                  // first tile of the next unit (or the stop tile)
        const Unit u = ring[ring_pos];
        if (++ring_pos == RING) ring_pos = 0;
        if (u.nkt == 0) break;
        // the tile's fragments, split evenly over the two warp rows and the two warp columns
        const int rows_t = int(u.tile & 0xffffu), cols_t = int(u.tile >> 16);      // cols_t: stored columns (padded ld)
        const int cols_b = min(cols_t, u.ncols - u.j0);                             // columns that hold data
        const int fmt = (rows_t + 7) >> 3, fnt = (cols_b + 7) >> 3, fm0 = (fmt + 1) >> 1, fn0 = (fnt + 1) >> 1;
        const int Fm = wm ? fm0 : 0, nfm = wm ? fmt - fm0 : fm0;
        const int Fn = wn ? fn0 : 0, nfn = wn ? fnt - fn0 : fn0;
        const int nfn_st = wn ? (cols_t >> 3) - fn0 : fn0;                          // incl. all-padding column fragments
        const FragBase fa = make_frag_base(0, Fm, g, t4), fb = make_frag_base(A_DOUBLES, Fn, g, t4);
        const bool busy = nfm > 0 && nfn > 0;
        double acc[WM][4][2];
#pragma unroll
        for (int i = 0; i < WM; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll 1
        for (int it = 0; it < u.nkt; ++it) {
            if (it > 0) mbar_wait(bar0 + stage * 8, ph);
            if (busy) {
                const StageNote note = notes[stage];
                const double* st = smem + stage * STAGE_DOUBLES;
                switch (note.flags & (SEG_A_MMAJOR | SEG_B_NMAJOR)) {
                    case 0: mma_layout<WM, false, false>(nfm, nfn, note.nks, st, fa, fb, g3, acc); break;
                    case SEG_A_MMAJOR: mma_layout<WM, true, false>(nfm, nfn, note.nks, st, fa, fb, g3, acc); break;
                    case SEG_B_NMAJOR: mma_layout<WM, false, true>(nfm, nfn, note.nks, st, fa, fb, g3, acc); break;
                    default: mma_layout<WM, true, true>(nfm, nfn, note.nks, st, fa, fb, g3, acc); break;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar0 + (STAGES + stage) * 8);
            if (++stage == STAGES) {
                stage = 0;
                ph ^= 1u;
            }
        }
        // epilogue: lane holds C[row g][cols 2·t4, 2·t4+1] of each 8×8 fragment
        double* C = reinterpret_cast<double*>(bases.b[(u.mode >> UNIT_C_SEL_SHIFT) & 3u] + u.C);
        const bool accum = (u.mode & UNIT_ACCUM) != 0, plain = (u.mode & UNIT_C_PLAIN) != 0;
        // the block's last row tile also writes the padding rows (zeros)
        const int rows_st = (plain || u.i0 + rows_t < u.mrows) ? rows_t : u.c_rp - u.i0;
#pragma unroll
        for (int i = 0; i < WM; ++i) {
            const int r = (Fm + i) * 8 + g;
            if (i >= nfm || r >= rows_st) continue;
            const bool live = r < rows_t;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int c = (Fn + j) * 8 + 2 * t4;
                if (j >= nfn_st) continue;
                double2* p = reinterpret_cast<double2*>(plain ? C + r * BN + c : C + panel_off(u.i0 + r, u.j0 + c, u.c_rp));
                double2 v;
                v.x = (live && u.j0 + c < u.ncols) ? u.alpha * acc[i][j][0] : 0.0;
                v.y = (live && u.j0 + c + 1 < u.ncols) ? u.alpha * acc[i][j][1] : 0.0;
                if (accum) {
                    double2 o = *p;
                    v.x += o.x;
                    v.y += o.y;
                }
                *p = v;
            }
        }
    }
}

// Scalar check kernel over the same work lists: one thread per output element, plain FMA loops reading
// global memory directly through panel_off.  A debugging aid (dmrgk_heff_opts.kernel = 1), never the
// product path.
__global__ void __launch_bounds__(NTHREADS)
heff_gemm_scalar_kernel(const Unit* __restrict__ units, const Seg* __restrict__ segs, Bases bases) {
    const Unit u = units[blockIdx.x];
    const int tr = int(u.tile & 0xffffu);
    const int rows_t = ((u.mode & UNIT_C_PLAIN) || u.i0 + tr < u.mrows) ? tr : u.c_rp - u.i0;   // incl. padding rows
    const int cols_t = int(u.tile >> 16);
    double* C = reinterpret_cast<double*>(bases.b[(u.mode >> UNIT_C_SEL_SHIFT) & 3u] + u.C);
    for (int e = threadIdx.x; e < rows_t * cols_t; e += NTHREADS) {
        const int r = e / cols_t, c = e % cols_t;
        const int i = u.i0 + r, j = u.j0 + c;
        double s = 0.0;
        if (i < u.mrows && j < u.ncols) {
            for (int sidx = u.seg_begin; sidx < u.seg_end; ++sidx) {
                const Seg sg = segs[sidx];
                const double* A = reinterpret_cast<const double*>(bases.b[(sg.flags >> SEG_A_SEL_SHIFT) & 3u] + sg.A);
                const double* B = reinterpret_cast<const double*>(bases.b[(sg.flags >> SEG_B_SEL_SHIFT) & 3u] + sg.B);
                for (int k = 0; k < sg.klen; ++k) {
                    double a = (sg.flags & SEG_A_MMAJOR) ? A[panel_off(k, i, sg.a_rp)] : A[panel_off(i, k, sg.a_rp)];
                    double b = (sg.flags & SEG_B_NMAJOR) ? B[panel_off(k, j, sg.b_rp)] : B[panel_off(j, k, sg.b_rp)];
                    s = fma(a, b, s);
                }
            }
        }
        double v = u.alpha * s;
        double* p = (u.mode & UNIT_C_PLAIN) ? C + r * BN + c : C + panel_off(i, j, u.c_rp);
        if (u.mode & UNIT_ACCUM) v += *p;
        *p = v;
    }
}

// a7: fixed-order sum of split-k partial tiles, σ_tile += Σ_s P_s (s ascending).  Eight CTAs per tile
// (one 8-row slab each, one double2 per thread; 16 for the tall tile) so that even a handful of output tiles fills the GPU;
// the partial loads of four splits are issued together, the additions stay in split order.
__global__ void __launch_bounds__(256)
heff_reduce_kernel(const RUnit* __restrict__ runits, Bases bases, int slabs) {      // slabs = tile rows / 8
    const RUnit u = runits[blockIdx.x / slabs];
    const int r = (blockIdx.x % slabs) * 8 + (threadIdx.x >> 5);
    const int64_t tile_d2 = int64_t(slabs) * 8 * BN / 2;                             // double2s per partial tile
    const int c = (threadIdx.x & 31) * 2;
    if (r >= u.rows || c >= u.cols) return;   // cols is even (multiple of 16 or the tile width 64)
    double2* p = reinterpret_cast<double2*>(reinterpret_cast<double*>(bases.b[BASE_SIGMA] + u.C) + panel_off(u.i0 + r, u.j0 + c, u.c_rp));
    const double2* P = reinterpret_cast<const double2*>(reinterpret_cast<const double*>(bases.b[BASE_WS] + u.P) + r * BN + c);
    double2 v = *p;
    int s = 0;
    for (; s + 4 <= u.n_split; s += 4) {
        double2 q[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) q[j] = P[int64_t(s + j) * tile_d2];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            v.x += q[j].x;
            v.y += q[j].y;
        }
    }
    for (; s < u.n_split; ++s) {
        const double2 q = P[int64_t(s) * tile_d2];
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
                sl[t][x] = (i0 + x < b.rows) ? tk.alpha * L[panel_off(i0 + x, i0 + x, tk.l_rp)] : 0.0;
                sr[t][x] = (j0 + x < b.cols) ? R[panel_off(j0 + x, j0 + x, tk.r_rp)] : 0.0;
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
            if (i < b.rows && j < b.cols) diag[b.off + panel_off(i, j, b.rows_pad)] += acc[q];
        }
    }
}

static int g_gemm_ctas_per_sm = 0;
int gemm_ctas_per_sm() { return g_gemm_ctas_per_sm; }

// Kernel variants (dmrgk_heff_opts.kernel): 0 = 64×64 tiles, 3 CTAs per SM with 64 KB of stages each;
// 1 = scalar check kernel; 2 = 64×64, 2 CTAs per SM with 96 KB of stages; 3 = 64×64, 2 CTAs per SM with
// 64 KB; 4 = the tall 128×64 tile (2×2 warps of 64×32: 128 accumulator registers), 2 CTAs per SM with 96 KB
// of stages — a CTA of 5 warps at 2 CTAs per SM is capped at 168 registers, so this variant spills and is
// slower than variant 0 on every shape measured (profiles/r2_ragged.md); kept, like 2 and 3, for measurement;
// 5 = variant 0 with EAGER unit claims (see the producer's look-ahead comment).
constexpr int ST64 = 65536 / (stage_doubles(4) * 8), ST96 = 98304 / (stage_doubles(4) * 8), ST96T = 98304 / (stage_doubles(8) * 8);
template <class K>
static int32_t setup_kernel(K* fn, int threads, int smem, int min_ctas, int* resident) {
    DMRGK_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    // the L1/shared split must leave room for min_ctas CTAs: ask for the largest shared-memory carve-out
    // and verify the residency instead of trusting the driver's heuristic
    DMRGK_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    int n = 0;
    DMRGK_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, fn, threads, smem));
    if (resident) *resident = n;
    if (n < min_ctas)
        return fail(DMRGK_ECUDA, "gemm kernel <%d B of stages, %d CTAs>: only %d CTA(s) per SM resident", smem, min_ctas, n);
    return DMRGK_OK;
}

// Set up at context creation.  Only the product variants (0 and its eager-claim twin 5) are required: a
// measurement variant that misses its residency target on some device is recorded as unavailable and
// refused where it is asked for (gemm_kernel_available), it does not take the whole library down.
static bool g_variant_ok[6] = {false, true, false, false, false, false};   // 1 = scalar check kernel, no set-up needed

int32_t gemm_kernel_setup() {
    DMRGK_TRY(setup_kernel(heff_gemm_dmma_persistent_kernel<4, ST64, 3, LATE>, P_NTHREADS, smem_bytes(4, ST64), 3, &g_gemm_ctas_per_sm));
    DMRGK_TRY(setup_kernel(heff_gemm_dmma_persistent_kernel<4, ST64, 3, EAGER>, P_NTHREADS, smem_bytes(4, ST64), 3, nullptr));
    g_variant_ok[0] = g_variant_ok[5] = true;
    g_variant_ok[2] = setup_kernel(heff_gemm_dmma_persistent_kernel<4, ST96, 2, LATE>, P_NTHREADS, smem_bytes(4, ST96), 2, nullptr) == DMRGK_OK;
    g_variant_ok[3] = setup_kernel(heff_gemm_dmma_persistent_kernel<4, ST64, 2, LATE>, P_NTHREADS, smem_bytes(4, ST64), 2, nullptr) == DMRGK_OK;
    g_variant_ok[4] = setup_kernel(heff_gemm_dmma_persistent_kernel<8, ST96T, 2, LATE>, P_NTHREADS, smem_bytes(8, ST96T), 2, nullptr) == DMRGK_OK;
    return DMRGK_OK;
}

bool gemm_kernel_available(int kernel) { return kernel >= 0 && kernel <= 5 && g_variant_ok[kernel]; }

int gemm_tile_m(int kernel) { return kernel == 4 ? 128 : 64; }
int gemm_ctas(int kernel) { return (kernel == 0 || kernel == 1 || kernel == 5) ? 3 : 2; }

int32_t launch_gemm_units(int kernel, const Unit* units_dev, const Seg* segs_dev, int64_t n_units,
                          const Bases& bases, cudaStream_t st, int* counter_dev, int n_sm, bool short_units) {
    if (n_units <= 0) return DMRGK_OK;
    if (kernel == 0 && short_units) kernel = 5;      // units too short for the late look-ahead chain: claim eagerly
    if (n_units > 0x7fffffffLL) return fail(DMRGK_EINVAL, "too many work units in one launch: %lld", (long long)n_units);
    const int nu = int(n_units);
    auto pgrid = [&](int ctas) { return unsigned(std::min<int64_t>(n_units, int64_t(n_sm) * ctas)); };
    if (kernel != 1 && !counter_dev) return fail(DMRGK_EINVAL, "launch_gemm_units: the persistent kernel needs a queue counter");
    switch (kernel) {
        case 1: heff_gemm_scalar_kernel<<<unsigned(n_units), NTHREADS, 0, st>>>(units_dev, segs_dev, bases); break;
        case 2: heff_gemm_dmma_persistent_kernel<4, ST96, 2, LATE><<<pgrid(2), P_NTHREADS, smem_bytes(4, ST96), st>>>(units_dev, segs_dev, nu, counter_dev, bases); break;
        case 3: heff_gemm_dmma_persistent_kernel<4, ST64, 2, LATE><<<pgrid(2), P_NTHREADS, smem_bytes(4, ST64), st>>>(units_dev, segs_dev, nu, counter_dev, bases); break;
        case 4: heff_gemm_dmma_persistent_kernel<8, ST96T, 2, LATE><<<pgrid(2), P_NTHREADS, smem_bytes(8, ST96T), st>>>(units_dev, segs_dev, nu, counter_dev, bases); break;
        case 5: heff_gemm_dmma_persistent_kernel<4, ST64, 3, EAGER><<<pgrid(3), P_NTHREADS, smem_bytes(4, ST64), st>>>(units_dev, segs_dev, nu, counter_dev, bases); break;
        default: heff_gemm_dmma_persistent_kernel<4, ST64, 3, LATE><<<pgrid(3), P_NTHREADS, smem_bytes(4, ST64), st>>>(units_dev, segs_dev, nu, counter_dev, bases); break;
    }
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

int32_t launch_reduce(const RUnit* runits_dev, int64_t n, const Bases& bases, cudaStream_t st, int tile_m) {
    if (n <= 0) return DMRGK_OK;
    const int slabs = tile_m / 8;
    heff_reduce_kernel<<<unsigned(n * slabs), 256, 0, st>>>(runits_dev, bases, slabs);
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
