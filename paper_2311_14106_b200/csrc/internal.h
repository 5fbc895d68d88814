// internal.h — private structures of libdmrgk (not part of the ABI; see include/dmrgk.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include <unordered_map>
#include "../../include/dmrgk.h"
#include "../../include/dmrgk_harness.h"

namespace dmrgk {

// ---- error plumbing ----------------------------------------------------------------------------
int32_t fail(int32_t code, const char* fmt, ...);
#define DMRGK_CUDA(call)                                                                         \
    do {                                                                                         \
        cudaError_t e__ = (call);                                                                \
        if (e__ != cudaSuccess)                                                                  \
            return dmrgk::fail(DMRGK_ECUDA, "%s failed: %s (%s:%d)", #call,                      \
                               cudaGetErrorString(e__), __FILE__, __LINE__);                     \
    } while (0)
#define DMRGK_TRY(call)                                                                          \
    do {                                                                                         \
        int32_t s__ = (call);                                                                    \
        if (s__ != DMRGK_OK) return s__;                                                         \
    } while (0)

// Number of kernels the library has launched in this process (dmrgk_launch_count).
void count_launch(int64_t n = 1);

static inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
static inline bool aligned128(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 127u) == 0; }

constexpr int LD_PAD = 16;   // column counts are padded to multiples of 16 doubles (one 128-byte panel row)
constexpr int ROW_PAD = 4;   // row counts are padded to multiples of 4 (one DMMA k-step) with zero rows

// ---- panel layout of a stored block ------------------------------------------------
// A block (rows × cols) is stored as ceil(cols/16) column PANELS, panel after panel; a panel holds
// rows_pad = round_up(rows, 4) rows of 16 doubles (128 bytes), so a (≤64 rows × 16 columns) operand tile
// — and a (≤16 rows × 16 columns) piece of a transposed one — is ONE contiguous chunk that a single
// cp.async.bulk moves to shared memory.  Inside a row the 32-byte groups are XOR-swizzled with the row
// index, so that the shared-memory copy (taken verbatim) is read conflict-free by the DMMA fragment
// loads both K-major and MN-major (heff_kernels.cu).  Padding rows and columns hold exact zeros.
__host__ __device__ inline int64_t panel_off(int r, int c, int rows_pad) {
    return (int64_t(c >> 4) * rows_pad + r) * 16 + ((c & 15) ^ ((r & 3) << 2));
}
static inline int32_t pad_rows(int32_t rows) { return (rows + ROW_PAD - 1) / ROW_PAD * ROW_PAD; }

// ---- a1: sectors and blocks --------------------------------------------------------------------
struct Block {
    int32_t r_idx, c_idx;  // sector indices (row, column); for ψ: (a, b)
    int32_t rows, cols, ld;   // ld = round_up(cols, 16): the padded column count
    int32_t rows_pad;         // round_up(rows, 4); the block occupies rows_pad·ld doubles
    int64_t off;           // doubles into the packed arena
    int64_t uoff;          // elements into the unpadded form
    int64_t size() const { return int64_t(rows_pad) * ld; }
};

// Block table mirrored on the device for the fill kernel.
struct DevBlock {
    int64_t off, uoff;
    int32_t rows, cols, ld, square_diag;
    int32_t rows_pad, pad_;
};

}  // namespace dmrgk

struct dmrgk_ctx {
    int device = 0;
    int n_sm = 0;
    int64_t l2_bytes = 0, hbm_bytes = 0;
    int smem_optin = 0;
};

struct dmrgk_space {
    dmrgk_ctx* ctx;
    int n_charges;
    std::vector<int32_t> q;     // [n][2] (second component 0 for one charge)
    std::vector<int32_t> dim;
    std::unordered_map<int64_t, int32_t> index;
    static int64_t key(int32_t a, int32_t b) { return (int64_t(a) << 32) ^ int64_t(uint32_t(b)); }
    int n() const { return int(dim.size()); }
    int find(int32_t a, int32_t b) const {
        auto it = index.find(key(a, b));
        return it == index.end() ? -1 : it->second;
    }
    int parity(int i) const { return (q[2 * i] + q[2 * i + 1]) & 1; }
};

struct dmrgk_layout {
    dmrgk_ctx* ctx;
    const dmrgk_space *A, *B;
    int32_t target[2];
    std::vector<dmrgk::Block> blocks;
    std::vector<int32_t> by_a;   // A sector → block index or −1
    int64_t n_elems = 0, n_padded = 0;
    dmrgk::DevBlock* dev_table = nullptr;
};

struct dmrgk_op {
    dmrgk_ctx* ctx;
    const dmrgk_space* space;
    int32_t dq[2];
    int32_t parity;
    std::vector<dmrgk::Block> blocks;
    std::vector<int32_t> by_col, by_row;   // sector → block index or −1
    int64_t n_elems = 0, n_padded = 0;
    const double* dev = nullptr;
    const double* pinned = nullptr;
    dmrgk::DevBlock* dev_table = nullptr;
};

struct dmrgk_iso {
    dmrgk_ctx* ctx;
    const dmrgk_space *enl, *kept;
    std::vector<dmrgk::Block> blocks;     // r_idx = enlarged sector, c_idx = kept sector
    std::vector<int32_t> by_enl;          // enlarged sector → block index or −1
    int64_t n_elems = 0, n_padded = 0;
    const double* dev = nullptr;
    dmrgk::DevBlock* dev_table = nullptr;
};

namespace dmrgk {

// ---- a2: device-side work descriptions ---------------------------------------------------------
// Pointers that depend on heff_apply arguments (ψ, σ, workspace) are stored as byte offsets plus a
// 2-bit base selector; the kernels add the base passed at launch (Bases).  Resident operator blocks
// are absolute addresses (selector 0, base 0).
enum : uint32_t { BASE_ABS = 0u, BASE_WS = 1u, BASE_PSI = 2u, BASE_SIGMA = 3u };
struct Bases {
    unsigned long long b[4];
};

// One GEMM "segment": C_tile += A[i, k]·B[k, j] over k < klen.  Operands are whole stored blocks in the
// panel layout; A is K-major (stored block = [i][k]) or M-major (stored block = [k][i], the transposed
// use of an operator); B is K-major (stored [j][k]) or N-major (stored [k][j]).
enum : uint32_t {
    SEG_A_MMAJOR = 1u,
    SEG_B_NMAJOR = 2u,
    SEG_A_TBUF = 4u,       // host only: A is the phase-1 intermediate (offset into the T buffer of its chunk)
    SEG_B_TBUF = 8u,       // host only: B is the phase-1 intermediate
    SEG_A_SEL_SHIFT = 4,   // bits 4-5: base selector of A
    SEG_B_SEL_SHIFT = 6    // bits 6-7: base selector of B
};
struct Seg {
    unsigned long long A, B;   // byte address / byte offset of the operand BLOCK origin
    int32_t a_rp, b_rp;        // rows_pad of the stored A / B block (panel stride = rows_pad·128 bytes)
    int32_t klen;
    uint32_t flags;
};  // 32 B

// One CTA work unit: a (≤64 × ≤64) tile of C summed over segments [seg_begin, seg_end).
// C is a block in the panel layout (origin + rows_pad) or, with UNIT_C_PLAIN, a private row-major
// 64×64 tile (split-k partial in the workspace).  Tiles of a block are BALANCED (tile_cuts): origins are
// multiples of 16 and extents differ by at most 16, so the tile's explicit extent travels in `tile`.
enum : uint32_t { UNIT_ACCUM = 1u, UNIT_C_PLAIN = 2u, UNIT_C_SEL_SHIFT = 4 };
struct Unit {
    unsigned long long C;   // byte address / offset of the C block origin (or of the plain tile)
    double alpha;
    int32_t c_rp;       // rows_pad of the C block
    int32_t i0, j0;     // tile origin inside the operand blocks and inside the C block
    int32_t mrows;      // block rows (A-operand row extent)
    int32_t ncols;      // block cols (B-operand column extent)
    int32_t ncols_st;   // columns to store (padded ld of the C block); columns ≥ ncols get zeros
    int32_t seg_begin, seg_end;
    uint32_t mode;      // UNIT_ACCUM | UNIT_C_PLAIN | selector << UNIT_C_SEL_SHIFT
    int32_t nkt;        // Σ over the unit's segments of ceil(klen/TILE_K); ≥ 1 (0 marks the stop sentinel)
    int32_t pad_;
    uint32_t tile;      // tile rows | tile columns << 16 (columns over the padded ld: the STORED extent)
};  // 64 B: four 16-byte words (the persistent kernel passes descriptors through shared memory)
static_assert(sizeof(Unit) == 64, "Unit must be 64 bytes");

// Fixed-order reduction of split-k partial tiles into σ: σ_block[i0 + r, j0 + c] += Σ_s P[s][r·64 + c].
struct RUnit {
    unsigned long long C;   // byte offset into σ of the BLOCK origin
    unsigned long long P;   // byte offset into the workspace of the first partial tile (64×64 each)
    int32_t c_rp, i0, j0, rows, cols, n_split;
};  // 40 B

// diag(H_eff) work: ψ block `DiagBlock` sums alpha·L[i,i]·R[j,j] over tasks [t_begin, t_end).
struct DiagTask {
    unsigned long long L, R;   // block origins (panel layout)
    double alpha;
    int32_t l_rp, r_rp;        // rows_pad of the L / R block
    uint32_t sel;              // selector of L in bits 0-1, of R in bits 2-3
    int32_t pad_;
};
struct DiagBlock {
    int64_t off;               // doubles into the ψ-layout arena
    int32_t rows, cols, ld;
    int32_t t_begin, t_end;
    int32_t rows_pad;
};

constexpr int TILE_M = 64, TILE_N = 64;
constexpr int TILE_K = 32;   // contraction depth of one pipeline stage (k-tile); Unit::nkt counts these

// Balanced tiling of one block dimension: ceil(extent/tile_max) tiles (tile_max = 64, or 128 rows for the tall tile) with origins at multiples of 16 (a panel
// row group, so that an MN-major operand tile starts on a panel) and extents that differ by at most 16;
// the larger tiles come first, the ragged end of the block falls into one of the smaller ones.  A tile's
// 8-row fragments are then split evenly over the two warp rows (columns) of the CTA — the CTA advances at
// the pace of its fullest warp, so 64 + 10 rows cost two full tiles, 48 + 26 cost 3/4 + 1/2
// (profiles/r2_ragged.md).  `cuts` gets n + 1 entries, cuts[n] = extent.
static inline void tile_cuts(int extent, int tile_max, std::vector<int>& cuts) {
    cuts.clear();
    const int panels = (extent + 15) / 16, n = (extent + tile_max - 1) / tile_max;
    int p = 0;
    for (int t = 0; t < n; ++t) {
        cuts.push_back(p * 16);
        p += panels / n + (t < panels % n ? 1 : 0);
    }
    cuts.push_back(extent);
}
static inline uint32_t pack_tile(int rows, int cols) { return uint32_t(rows) | (uint32_t(cols) << 16); }
// cost of a tile per k-tile: the fragment products of its fullest warp × 4 (a full 64×64 tile costs 64), but
// never less than TILE_COST_FLOOR — a thin tile turns its stages over faster than the copies arrive, so its
// k-tile costs a latency, not its flops (profiles/r2_ragged.md).  Used for LPT ordering and the split-k plan.
constexpr int TILE_COST_FLOOR = 24;
static inline int64_t tile_cost(int rows, int cols) {
    const int fm = (rows + 7) / 8, fn = (cols + 7) / 8;
    const int64_t c = int64_t(4) * ((fm + 1) / 2) * ((fn + 1) / 2);
    return c < TILE_COST_FLOOR ? TILE_COST_FLOOR : c;
}

// kernel launchers (heff_kernels.cu)
// `counter_dev`: a zeroed int the persistent kernel uses as its unit queue head (one per launch in flight)
// `short_units`: the launch's units average fewer k-tiles than the late look-ahead needs (variant 0 then claims eagerly)
bool gemm_kernel_available(int kernel);   // false for a measurement variant whose residency target this device misses
int32_t launch_gemm_units(int kernel, const Unit* units_dev, const Seg* segs_dev, int64_t n_units,
                          const Bases& bases, cudaStream_t st, int* counter_dev, int n_sm, bool short_units);
constexpr int SHORT_UNIT_TILES = 8;   // = the late look-ahead of the GEMM kernel, in k-tiles
int32_t launch_reduce(const RUnit* runits_dev, int64_t n, const Bases& bases, cudaStream_t st, int tile_m);
int gemm_tile_m(int kernel);   // rows of the CTA tile of a kernel variant (64, or 128 for the tall tile)
int gemm_ctas(int kernel);     // CTAs per SM the variant is launched with
int32_t launch_diag(const DiagBlock* blocks_dev, const DiagTask* tasks_dev, int64_t n_blocks,
                    double* diag, const Bases& bases, cudaStream_t st);
int32_t gemm_kernel_setup();   // opt-in shared memory attribute, once
int gemm_ctas_per_sm();        // resident CTAs per SM of the GEMM kernel, as reported by the occupancy API

// chunk = contiguous range of operator pairs processed together
struct StageCopy {
    const double* src_host;
    int64_t ring_off;   // doubles into the ring half
    int64_t n;          // doubles
};
struct Chunk {
    int64_t p1_unit0 = 0, p1_units = 0, p1_seg0 = 0;
    int64_t p2_unit0 = 0, p2_units = 0, p2_seg0 = 0;
    bool p1_short = false, p2_short = false;   // mean unit length below SHORT_UNIT_TILES k-tiles
    int64_t r_unit0 = 0, r_units = 0;
    int64_t p1_segs = 0, p2_segs = 0;
    int64_t d_block0 = 0, d_blocks = 0;
    std::vector<StageCopy> copies;
    int64_t k_first = 0, k_count = 0;   // the chunk's range of operator pairs
    int ring_part = -1;   // which third of the staging ring holds this chunk's pinned operators
};

}  // namespace dmrgk

struct dmrgk_renorm {
    dmrgk_ctx* ctx;
    int kernel = 0;
    int64_t n_tasks = 0, t_bytes = 0, workspace_bytes = 0, n_launches = 0;
    double flops = 0;
    struct RChunk {
        int64_t p1_unit0 = 0, p1_units = 0, p2_unit0 = 0, p2_units = 0;
        bool p1_short = false, p2_short = false;
    };
    std::vector<RChunk> chunks;
    dmrgk::Unit* units_dev = nullptr;
    dmrgk::Seg* segs_dev = nullptr;
    int* counters_dev = nullptr;          // unit-queue heads of the persistent kernel, two per chunk
    // same choreography as dmrgk_heff_apply: phase 1 of chunk c+1 (lowest-priority stream) overlaps
    // phase 2 of chunk c (greatest-priority stream); T is double-buffered
    cudaStream_t s1 = nullptr, s2 = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_join1 = nullptr, ev_p1[2] = {nullptr, nullptr}, ev_p2[2] = {nullptr, nullptr};
};

struct dmrgk_heff {
    dmrgk_ctx* ctx;
    const dmrgk_layout* layout;
    dmrgk_heff_opts opts;
    int64_t n_tasks = 0, n_rfirst = 0;
    double flops_alg = 0, flops_exec = 0;
    int64_t op_bytes = 0;
    int64_t t_bytes = 0, partial_bytes = 0, ring_bytes = 0, ring_part_bytes = 0, workspace_bytes = 0;
    int64_t pp_base = 0, pp_bytes = 0, pp_vec_bytes = 0;   // per-pair σ_k buffers + dot scratch (dmrgk_heff_expect)
    int64_t K = 0;
    bool done_recorded[3] = {false, false, false};
    std::vector<dmrgk::Chunk> chunks;
    // device metadata (library-owned)
    dmrgk::Unit* units_dev = nullptr;
    dmrgk::Seg* segs_dev = nullptr;
    dmrgk::RUnit* runits_dev = nullptr;
    dmrgk::DiagBlock* dblocks_dev = nullptr;
    dmrgk::DiagTask* dtasks_dev = nullptr;
    int64_t n_dblocks = 0;
    double* ident_dev = nullptr;       // identity block for IDENT_L / IDENT_R factors
    int* counters_dev = nullptr;       // unit-queue heads of the persistent kernel, two per chunk (zeroed per apply)
    cudaEvent_t ev_copy[3] = {nullptr, nullptr, nullptr}, ev_done[3] = {nullptr, nullptr, nullptr};
    // phase 1 of chunk c+1 runs on a library-owned side stream concurrently with phase 2 of chunk c
    // (T is double-buffered), so the tail of one launch is filled by the CTAs of the other
    cudaStream_t side = nullptr;       // phase 1 (lowest priority)
    cudaStream_t side_hi = nullptr;    // phase 2 + reduce (greatest priority: its CTAs are dispatched first)
    cudaEvent_t ev_join = nullptr, ev_join1 = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_p1[2] = {nullptr, nullptr}, ev_p2[2] = {nullptr, nullptr};
    cudaEvent_t ev_span[2] = {nullptr, nullptr};
    bool span_open = false;
    int64_t n_launches = 0;
    bool has_pinned = false;
    // optional per-kernel timing (dmrgk_heff_profile): event pairs around every launch of apply
    bool prof_on = false, prof_serial = false;
    std::vector<cudaEvent_t> prof_ev;      // pool, two per launch
    std::vector<int> prof_kind;            // per recorded pair: 0 phase 1, 1 phase 2, 2 reduce, 3 whole-apply span
    size_t prof_used = 0;                  // pairs recorded since the last read
    double prof_ms[4] = {0, 0, 0, 0};
    int64_t prof_launches[4] = {0, 0, 0, 0};
};
