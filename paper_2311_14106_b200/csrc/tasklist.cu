// tasklist.cu — a2/a3/a5-a7 host side: the operator-pair task list and σ = H_eff ψ
// ("enumerate (k, input block) … group by output block, tile, split-k plan";
// PAPER.md:142 "Tables", "H2D IO" for the staging of pinned operators).
//
// For pair k and ψ block (a, b):   σ[a′, b′] += c_k·s · Lapp[a′, a] · ψ[a, b] · Rapp[b′, b]ᵀ,
// s = −1 iff the pair is fermionic (odd) and the INPUT A sector has odd particle number
// (SURVEY.md §8.0).  Work is cut into chunks of consecutive pairs; per chunk
//   phase 1:  T_t = c·s · Lapp ψ[a, b]                 one GEMM unit per 64×64 tile of T_t
//   phase 2:  σ[a′, b′] += [T_t …]·[Rapp_t …]ᵀ          tasks grouped by OUTPUT block and stacked
//             along the contraction axis; a tile is owned by one CTA, or split along the task list
//             into partial tiles that a fixed-order reduction kernel adds up — never atomics.
#include "internal.h"
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

using namespace dmrgk;

namespace {

struct Task {
    int32_t k;
    int32_t ib, ob;          // input / output ψ block
    int32_t mo, m, n, no;    // m′, m, n, n′
    Seg s1, s2;              // phase-1 / phase-2 segment templates (the intermediate's offset is set per chunk)
    double alpha;
    bool diag;
    bool rfirst;             // GEMM order: false (L ψ) Rᵀ, true L (ψ Rᵀ)
    int32_t t_rows, t_cols, t_ld;   // shape of the phase-1 intermediate (m′ × n, or m × n′ when rfirst)
    // where the L / R operand of the pair sits in the two segments
    unsigned long long& Laddr() { return rfirst ? s2.A : s1.A; }
    unsigned long long& Raddr() { return rfirst ? s1.B : s2.B; }
    int32_t Lrp() const { return rfirst ? s2.a_rp : s1.a_rp; }
    int32_t Rrp() const { return rfirst ? s1.b_rp : s2.b_rp; }
    uint32_t Lsel() const { return ((rfirst ? s2.flags : s1.flags) >> SEG_A_SEL_SHIFT) & 3u; }
    uint32_t Rsel() const { return ((rfirst ? s1.flags : s2.flags) >> SEG_B_SEL_SHIFT) & 3u; }
};

struct OpRef {               // where an operator block lives
    unsigned long long addr; // absolute byte address, or byte offset inside the ring half
    uint32_t sel;            // BASE_ABS or BASE_WS (ring offset still to be added)
    int ld;
};

int64_t cost_of(int rows, int cols, int64_t nkt) { return tile_cost(rows, cols) * nkt; }

template <class T>
int32_t upload(const std::vector<T>& v, T** out) {
    *out = nullptr;
    if (v.empty()) return DMRGK_OK;
    DMRGK_CUDA(cudaMalloc(out, v.size() * sizeof(T)));
    DMRGK_CUDA(cudaMemcpy(*out, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
    return DMRGK_OK;
}

}  // namespace

extern "C" {

void dmrgk_heff_destroy(dmrgk_heff* h) {
    if (!h) return;
    cudaFree(h->units_dev);
    cudaFree(h->segs_dev);
    cudaFree(h->runits_dev);
    cudaFree(h->dblocks_dev);
    cudaFree(h->dtasks_dev);
    cudaFree(h->ident_dev);
    cudaFree(h->counters_dev);
    for (int i = 0; i < 3; ++i) {
        if (h->ev_copy[i]) cudaEventDestroy(h->ev_copy[i]);
        if (h->ev_done[i]) cudaEventDestroy(h->ev_done[i]);
    }
    for (int i = 0; i < 2; ++i) {
        if (h->ev_p1[i]) cudaEventDestroy(h->ev_p1[i]);
        if (h->ev_p2[i]) cudaEventDestroy(h->ev_p2[i]);
    }
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    if (h->ev_join1) cudaEventDestroy(h->ev_join1);
    if (h->side) cudaStreamDestroy(h->side);
    if (h->side_hi) cudaStreamDestroy(h->side_hi);
    for (cudaEvent_t e : h->prof_ev) cudaEventDestroy(e);
    delete h;
}

int32_t dmrgk_heff_create(dmrgk_ctx* ctx, const dmrgk_layout* layout, int64_t K,
                          dmrgk_op* const* L_in, dmrgk_op* const* R_in, const double* coef,
                          const uint32_t* flags_in, const dmrgk_heff_opts* opts, dmrgk_heff** out) {
    return dmrgk_heff_create_blockcoef(ctx, layout, K, L_in, R_in, coef, nullptr, flags_in, opts, out);
}

int32_t dmrgk_heff_create_blockcoef(dmrgk_ctx* ctx, const dmrgk_layout* layout, int64_t K,
                                    dmrgk_op* const* L_in, dmrgk_op* const* R_in, const double* coef,
                                    const double* block_coef, const uint32_t* flags_in,
                                    const dmrgk_heff_opts* opts, dmrgk_heff** out) {
    if (!out) return fail(DMRGK_EINVAL, "heff_create: out is NULL");
    *out = nullptr;
    if (!ctx || !layout) return fail(DMRGK_EINVAL, "heff_create: NULL ctx or layout");
    if (K < 0 || (K > 0 && (!L_in || !R_in || !coef || !flags_in)))
        return fail(DMRGK_EINVAL, "heff_create: bad pair arrays (K = %lld)", (long long)K);
    // DMRGK_HC_OF_PREV: pair k re-uses the stored operators of pair k−1, applied transposed
    std::vector<dmrgk_op*> Lv(static_cast<size_t>(K)), Rv(static_cast<size_t>(K));
    std::vector<uint32_t> fv(static_cast<size_t>(K));
    for (int64_t k = 0; k < K; ++k) {
        if (flags_in[k] & DMRGK_HC_OF_PREV) {
            if (k == 0) return fail(DMRGK_EINVAL, "heff_create: pair 0 cannot be the h.c. of a previous pair");
            if (flags_in[k] & ~uint32_t(DMRGK_HC_OF_PREV))
                return fail(DMRGK_EINVAL, "heff_create: pair %lld: HC_OF_PREV excludes the other flags", (long long)k);
            Lv[k] = Lv[k - 1];
            Rv[k] = Rv[k - 1];
            uint32_t f = fv[k - 1];
            if (Lv[k]) f ^= DMRGK_TRANS_L;
            if (Rv[k]) f ^= DMRGK_TRANS_R;
            fv[k] = f;
        } else {
            Lv[k] = L_in[k];
            Rv[k] = R_in[k];
            fv[k] = flags_in[k];
        }
    }
    dmrgk_op* const* L = Lv.data();
    dmrgk_op* const* R = Rv.data();
    const uint32_t* flags = fv.data();
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    dmrgk_heff_opts o;
    memset(&o, 0, sizeof(o));
    if (opts) o = *opts;
    if (o.split_waves <= 0) o.split_waves = 32;   // units per CTA slot: the queue's tail is ≈ one unit long
    if (o.ring_bytes < 0 || (o.kernel < 0 || o.kernel > 5) || o.order_policy < 0 || o.order_policy > 2 ||
        (o.per_pair_output != 0 && o.per_pair_output != 1))
        return fail(DMRGK_EINVAL, "heff_create: bad options");
    if (!gemm_kernel_available(o.kernel))
        return fail(DMRGK_EINVAL, "heff_create: kernel variant %d is not resident on this device (use 0)", o.kernel);
    const int64_t ring_part = (o.ring_bytes / 3) / 128 * 128;   // three parts: see dmrgk_heff_apply

    const dmrgk_space *SA = layout->A, *SB = layout->B;
    const std::vector<Block>& pb = layout->blocks;

    // ---- validation of every pair (SURVEY §8(b) "validation errors that must be reported") ----
    for (int64_t k = 0; k < K; ++k) {
        const uint32_t f = flags[k];
        if (f & ~15u) return fail(DMRGK_EINVAL, "heff_create: pair %lld has unknown flag bits 0x%x", (long long)k, f);
        if (bool(f & DMRGK_IDENT_L) != (L[k] == nullptr) || bool(f & DMRGK_IDENT_R) != (R[k] == nullptr))
            return fail(DMRGK_EINVAL, "heff_create: pair %lld: IDENT flag and NULL operator must go together", (long long)k);
        if (L[k] && L[k]->space != SA) return fail(DMRGK_ESHAPE, "heff_create: pair %lld: L is not on the layout's A space", (long long)k);
        if (R[k] && R[k]->space != SB) return fail(DMRGK_ESHAPE, "heff_create: pair %lld: R is not on the layout's B space", (long long)k);
        int dl[2] = {0, 0}, dr[2] = {0, 0};
        if (L[k]) for (int c = 0; c < 2; ++c) dl[c] = (f & DMRGK_TRANS_L) ? -L[k]->dq[c] : L[k]->dq[c];
        if (R[k]) for (int c = 0; c < 2; ++c) dr[c] = (f & DMRGK_TRANS_R) ? -R[k]->dq[c] : R[k]->dq[c];
        if (dl[0] + dr[0] != 0 || dl[1] + dr[1] != 0)
            return fail(DMRGK_ECHARGE, "heff_create: pair %lld: applied shifts (%d,%d)+(%d,%d) do not cancel", (long long)k, dl[0], dl[1], dr[0], dr[1]);
        if (L[k] && R[k] && L[k]->parity != R[k]->parity)
            return fail(DMRGK_ECHARGE, "heff_create: pair %lld: parities of L and R differ", (long long)k);
        for (const dmrgk_op* op : {(const dmrgk_op*)L[k], (const dmrgk_op*)R[k]}) {
            if (!op || op->n_padded == 0) continue;
            if (!op->dev && !op->pinned) return fail(DMRGK_ESTATE, "heff_create: pair %lld has an unbound operator", (long long)k);
            if (op->pinned && ring_part == 0) return fail(DMRGK_ESTATE, "heff_create: pair %lld has a pinned operator but ring_bytes = 0", (long long)k);
            if (op->pinned && op->n_padded * 8 > ring_part)
                return fail(DMRGK_ENOMEM, "heff_create: pinned operator of %lld bytes exceeds a third of the ring (%lld)", (long long)(op->n_padded * 8), (long long)ring_part);
        }
        // both operators of a pair are staged into the SAME ring part: together they must fit it
        {
            int64_t need = 0;
            if (L[k] && L[k]->pinned && !L[k]->dev) need += round_up(L[k]->n_padded * 8, 128);
            if (R[k] && R[k]->pinned && !R[k]->dev && (const dmrgk_op*)R[k] != (const dmrgk_op*)L[k]) need += round_up(R[k]->n_padded * 8, 128);
            if (need > ring_part)
                return fail(DMRGK_ENOMEM, "heff_create: the pinned operators of pair %lld need %lld bytes together, more than a third of the ring (%lld)", (long long)k, (long long)need, (long long)ring_part);
        }
    }

    dmrgk_heff* h = new (std::nothrow) dmrgk_heff;
    if (!h) return fail(DMRGK_ENOMEM, "heff_create: out of host memory");
    h->ctx = ctx;
    h->layout = layout;
    h->opts = o;
    auto bail = [&](int32_t s) {
        dmrgk_heff_destroy(h);
        return s;
    };

    // identity block for IDENT factors
    int max_dim = 0;
    for (const Block& b : pb) max_dim = std::max(max_dim, std::max(b.rows, b.cols));
    const int ident_ld = int(round_up(std::max(max_dim, 1), LD_PAD));
    bool need_ident = false;
    for (int64_t k = 0; k < K; ++k) need_ident |= (flags[k] & (DMRGK_IDENT_L | DMRGK_IDENT_R)) != 0;
    if (need_ident) {
        std::vector<double> id(size_t(ident_ld) * ident_ld, 0.0);      // panel layout, rows_pad = ident_ld
        for (int i = 0; i < ident_ld; ++i) id[size_t(panel_off(i, i, ident_ld))] = 1.0;
        cudaError_t e = cudaMalloc(&h->ident_dev, id.size() * 8);
        if (e == cudaSuccess) e = cudaMemcpy(h->ident_dev, id.data(), id.size() * 8, cudaMemcpyHostToDevice);
        if (e != cudaSuccess) return bail(fail(DMRGK_ECUDA, "heff_create: identity block: %s", cudaGetErrorString(e)));
    }

    // ---- chunking of the pair list + task enumeration ----------------------------------------
    std::vector<Unit> units;
    std::vector<Seg> segs;
    std::vector<RUnit> runits;
    std::vector<DiagBlock> dblocks;
    std::vector<DiagTask> dtasks;
    const int tile_m = gemm_tile_m(o.kernel);            // rows of the CTA tile: 64, or 128 for the tall-tile variant
    const int64_t slots = int64_t(ctx->n_sm) * gemm_ctas(o.kernel);
    std::vector<int> cut_r, cut_c;                       // balanced tile boundaries of the block at hand (tile_cuts)
    int64_t max_t_bytes = 0, max_partial_tiles = 0, max_pairs = 0;
    const int64_t pp_vec_bytes = round_up(layout->n_padded * 8, 128);     // one σ_k buffer (per-pair mode)

    // Tasks of pair k (every ψ block whose L and R blocks exist and whose output block is in the layout)
    // and the bytes of their T intermediates.  Enumerated once for all pairs: the total decides the
    // default chunk size, the chunk loop below then only groups the pairs.
    auto tasks_of_pair = [&](int64_t k, std::vector<Task>& mine) -> int64_t {
        const uint32_t f = flags[k];
        int64_t tb = 0;
        for (int ib = 0; ib < int(pb.size()); ++ib) {
            const int a = pb[ib].r_idx, b = pb[ib].c_idx;
            Task t;
            memset(&t, 0, sizeof(t));
            t.k = int32_t(k);
            t.ib = ib;
            t.m = pb[ib].rows;
            t.n = pb[ib].cols;
            int ao, bo;
            // L applied to sector a
            if (!L[k]) {
                ao = a;
                t.mo = t.m;
                t.s1.A = (unsigned long long)(uintptr_t)h->ident_dev;
                t.s1.a_rp = ident_ld;
                t.s1.flags = BASE_ABS << SEG_A_SEL_SHIFT;
            } else {
                const int bi = (f & DMRGK_TRANS_L) ? L[k]->by_row[a] : L[k]->by_col[a];
                if (bi < 0) continue;
                const Block& lb = L[k]->blocks[bi];
                ao = (f & DMRGK_TRANS_L) ? lb.c_idx : lb.r_idx;
                t.mo = (f & DMRGK_TRANS_L) ? lb.cols : lb.rows;
                t.s1.a_rp = lb.rows_pad;
                t.s1.flags = (f & DMRGK_TRANS_L) ? SEG_A_MMAJOR : 0u;
                if (L[k]->dev) {
                    t.s1.A = (unsigned long long)(uintptr_t)(L[k]->dev + lb.off);
                    t.s1.flags |= BASE_ABS << SEG_A_SEL_SHIFT;
                } else {
                    t.s1.A = (unsigned long long)(lb.off * 8);   // ring offset added below
                    t.s1.flags |= BASE_WS << SEG_A_SEL_SHIFT;
                }
            }
            if (!R[k]) {
                bo = b;
                t.no = t.n;
                t.s2.B = (unsigned long long)(uintptr_t)h->ident_dev;
                t.s2.b_rp = ident_ld;
                t.s2.flags = BASE_ABS << SEG_B_SEL_SHIFT;
            } else {
                const int bi = (f & DMRGK_TRANS_R) ? R[k]->by_row[b] : R[k]->by_col[b];
                if (bi < 0) continue;
                const Block& rb = R[k]->blocks[bi];
                bo = (f & DMRGK_TRANS_R) ? rb.c_idx : rb.r_idx;
                t.no = (f & DMRGK_TRANS_R) ? rb.cols : rb.rows;
                t.s2.b_rp = rb.rows_pad;
                t.s2.flags = (f & DMRGK_TRANS_R) ? SEG_B_NMAJOR : 0u;
                if (R[k]->dev) {
                    t.s2.B = (unsigned long long)(uintptr_t)(R[k]->dev + rb.off);
                    t.s2.flags |= BASE_ABS << SEG_B_SEL_SHIFT;
                } else {
                    t.s2.B = (unsigned long long)(rb.off * 8);
                    t.s2.flags |= BASE_WS << SEG_B_SEL_SHIFT;
                }
            }
            const int ob = layout->by_a[ao];
            if (ob < 0 || pb[ob].c_idx != bo) continue;
            t.ob = ob;
            const int par = L[k] ? L[k]->parity : (R[k] ? R[k]->parity : 0);
            t.alpha = coef[k] * ((par && SA->parity(a)) ? -1.0 : 1.0);
            if (block_coef) {                               // recoupling scalar of (pair k, input block ib)
                t.alpha *= block_coef[size_t(k) * pb.size() + ib];
                if (t.alpha == 0.0) continue;               // structurally forbidden (e.g. a triangle rule)
            }
            t.diag = (ob == ib);
            // phase-1 B operand = ψ block (N-major), phase-2 A operand = T (K-major, set per chunk)
            t.s1.B = (unsigned long long)(pb[ib].off * 8);
            t.s1.b_rp = pb[ib].rows_pad;
            t.s1.klen = t.m;
            t.s1.flags |= SEG_B_NMAJOR | (BASE_PSI << SEG_B_SEL_SHIFT);
            t.s2.a_rp = pad_rows(t.mo);                     // T_t is a block (m′ × n) in the panel layout
            t.s2.klen = t.n;
            t.s2.flags |= SEG_A_TBUF | (BASE_WS << SEG_A_SEL_SHIFT);
            t.t_rows = t.mo;
            t.t_cols = t.n;
            t.t_ld = pb[ib].ld;
            // GEMM order: (L ψ) Rᵀ costs 2m′n(m + n′), L (ψ Rᵀ) costs 2mn′(n + m′)
            if (L[k] && R[k]) {
                const double cl = 2.0 * t.mo * t.n * (double(t.m) + t.no), cr = 2.0 * t.m * t.no * (double(t.n) + t.mo);
                t.rfirst = o.order_policy == 2 || (o.order_policy == 0 && cr < cl);
            }
            if (t.rfirst) {
                // phase 1: U = c·s · ψ[a,b] Rapp[b′,b]ᵀ (m × n′);  phase 2: σ[a′,b′] += Lapp[a′,a] U[a,b′]
                Seg p1, p2;
                memset(&p1, 0, sizeof(p1));
                memset(&p2, 0, sizeof(p2));
                p1.A = (unsigned long long)(pb[ib].off * 8);            // ψ block, K-major (stored [a][b])
                p1.a_rp = pb[ib].rows_pad;
                p1.B = t.s2.B;                                          // R: K-major stored [b′][b], N-major if transposed
                p1.b_rp = t.s2.b_rp;
                p1.klen = t.n;
                p1.flags = (BASE_PSI << SEG_A_SEL_SHIFT) | (t.s2.flags & (SEG_B_NMAJOR | (3u << SEG_B_SEL_SHIFT)));
                p2.A = t.s1.A;                                          // L: K-major stored [a′][a], M-major if transposed
                p2.a_rp = t.s1.a_rp;
                p2.B = 0;                                               // U_t (stored [a][b′] = N-major), offset set per chunk
                p2.b_rp = pad_rows(t.m);
                p2.klen = t.m;
                p2.flags = (t.s1.flags & (SEG_A_MMAJOR | (3u << SEG_A_SEL_SHIFT))) | SEG_B_NMAJOR | SEG_B_TBUF | (BASE_WS << SEG_B_SEL_SHIFT);
                t.s1 = p1;
                t.s2 = p2;
                t.t_rows = t.m;
                t.t_cols = t.no;
                t.t_ld = pb[ob].ld;
            }
            tb += int64_t(pad_rows(t.t_rows)) * t.t_ld * 8;
            mine.push_back(t);
        }
        return tb;
    };
    std::vector<std::vector<Task>> pair_tasks(static_cast<size_t>(K));
    std::vector<int64_t> pair_tb(static_cast<size_t>(K), 0);
    int64_t total_tb = 0;
    for (int64_t k = 0; k < K; ++k) {
        pair_tb[k] = tasks_of_pair(k, pair_tasks[k]);
        total_tb += pair_tb[k];
    }
    if (opts == nullptr || opts->t_chunk_bytes <= 0) {
        // default: about 16 chunks so that phase 1 of one chunk overlaps phase 2 of the previous one
        // (dmrgk_heff_apply), between 512 MiB (launches stay long against their tails) and 4 GiB
        o.t_chunk_bytes = std::min<int64_t>(int64_t(4) << 30, std::max<int64_t>(int64_t(512) << 20, total_tb / 16));
    }

    int64_t k0 = 0;
    while (k0 < K) {
        Chunk ch;
        ch.ring_part = int(h->chunks.size() % 3);
        std::vector<Task> tasks;
        std::unordered_map<const dmrgk_op*, int64_t> staged;   // pinned op → ring offset (bytes)
        int64_t ring_used = 0, t_bytes = 0;
        int64_t k = k0;
        for (; k < K; ++k) {
            const uint32_t f = flags[k];
            // staging need of this pair
            int64_t need = 0;
            for (const dmrgk_op* op : {(const dmrgk_op*)L[k], (const dmrgk_op*)R[k]})
                if (op && op->pinned && op->n_padded && !staged.count(op)) need += round_up(op->n_padded * 8, 128);
            const int64_t tb = pair_tb[k];
            std::vector<Task>& mine = pair_tasks[k];
            const bool nonempty = !tasks.empty() || !staged.empty();
            if (nonempty && (t_bytes + tb > o.t_chunk_bytes || ring_used + need > ring_part)) break;
            // per-pair outputs: one σ_k buffer per pair of the chunk
            if (o.per_pair_output && k > k0 && (k - k0 + 1) * pp_vec_bytes > std::max<int64_t>(o.t_chunk_bytes, pp_vec_bytes)) break;
            // accept pair k into the chunk
            for (const dmrgk_op* op : {(const dmrgk_op*)L[k], (const dmrgk_op*)R[k]})
                if (op && op->pinned && op->n_padded && !staged.count(op)) {
                    staged[op] = ring_used;
                    ch.copies.push_back({op->pinned, ring_used / 8, op->n_padded});
                    ring_used += round_up(op->n_padded * 8, 128);
                }
            for (Task& t : mine) {
                if (L[k] && !L[k]->dev) t.Laddr() += (unsigned long long)staged[L[k]];
                if (R[k] && !R[k]->dev) t.Raddr() += (unsigned long long)staged[R[k]];
                tasks.push_back(t);
            }
            t_bytes += tb;
        }
        ch.k_first = k0;
        ch.k_count = k - k0;
        max_pairs = std::max<int64_t>(max_pairs, k - k0);
        k0 = k;
        max_t_bytes = std::max(max_t_bytes, t_bytes);

        // ---- flop / byte accounting ----
        for (const Task& t : tasks) {
            const double mo = t.mo, m = t.m, n = t.n, no = t.no;
            const bool il = !L[t.k], ir = !R[t.k];
            if (il && ir) {
            } else if (il) {
                h->flops_alg += 2 * m * n * no;
            } else if (ir) {
                h->flops_alg += 2 * mo * m * n;
            } else {
                h->flops_alg += std::min(2 * mo * n * (m + no), 2 * m * no * (n + mo));
            }
            h->flops_exec += t.rfirst ? 2 * m * n * no + 2 * mo * m * no : 2 * mo * m * n + 2 * mo * n * no;
            h->n_rfirst += t.rfirst;
            if (!il) h->op_bytes += int64_t(8) * t.mo * t.m;
            if (!ir) h->op_bytes += int64_t(8) * t.no * t.n;
        }
        h->n_tasks += int64_t(tasks.size());

        // ---- phase 1: one segment + tiles per task; T laid out task after task ----
        ch.p1_unit0 = int64_t(units.size());
        ch.p1_seg0 = int64_t(segs.size());
        {
            std::vector<int64_t> t_off(tasks.size());
            int64_t off = 0;
            for (size_t i = 0; i < tasks.size(); ++i) {
                t_off[i] = off;
                off += int64_t(pad_rows(tasks[i].t_rows)) * tasks[i].t_ld * 8;
            }
            struct U1 {
                int64_t cost;
                Unit u;
            };
            std::vector<U1> tmp;
            for (size_t i = 0; i < tasks.size(); ++i) {
                Task& t = tasks[i];
                segs.push_back(t.s1);   // a staged A still lacks the ring base (added below)
                (t.rfirst ? t.s2.B : t.s2.A) = (unsigned long long)t_off[i];
                const int ldt = t.t_ld;
                const int64_t nkt = (t.s1.klen + TILE_K - 1) / TILE_K;
                tile_cuts(t.t_rows, tile_m, cut_r);
                tile_cuts(ldt, TILE_N, cut_c);
                for (size_t ti = 0; ti + 1 < cut_r.size(); ++ti)
                    for (size_t tj = 0; tj + 1 < cut_c.size(); ++tj) {
                        const int i0 = cut_r[ti], j0 = cut_c[tj], rt = cut_r[ti + 1] - i0, ct = cut_c[tj + 1] - j0;
                        Unit u;
                        memset(&u, 0, sizeof(u));
                        u.C = (unsigned long long)t_off[i];      // block origin of T_t
                        u.alpha = t.alpha;
                        u.c_rp = pad_rows(t.t_rows);
                        u.i0 = i0;
                        u.j0 = j0;
                        u.mrows = t.t_rows;
                        u.ncols = t.t_cols;
                        u.ncols_st = ldt;
                        u.seg_begin = int32_t(i);   // chunk-local, rebased below
                        u.seg_end = int32_t(i) + 1;
                        u.mode = BASE_WS << UNIT_C_SEL_SHIFT;
                        u.nkt = int32_t(nkt);
                        u.tile = pack_tile(rt, ct);
                        tmp.push_back({cost_of(rt, std::min(ct, t.t_cols - j0), nkt), u});
                    }
            }
            std::stable_sort(tmp.begin(), tmp.end(), [](const U1& a, const U1& b) { return a.cost > b.cost; });
            for (const U1& x : tmp) units.push_back(x.u);
            ch.p1_units = int64_t(tmp.size());
            {
                int64_t kt = 0;
                for (const U1& x : tmp) kt += x.u.nkt;
                ch.p1_short = kt < SHORT_UNIT_TILES * ch.p1_units;
            }
            ch.p1_segs = int64_t(tasks.size());
        }

        // ---- phase 2: group by output block, stack along k, split-k plan ----
        ch.p2_unit0 = int64_t(units.size());
        ch.p2_seg0 = int64_t(segs.size());
        ch.r_unit0 = int64_t(runits.size());
        {
            // a group = the tasks summed into one destination block: all tasks of an output block, or — with
            // per-pair outputs (dmrgk_heff_expect) — the single task of (pair k, output block), which
            // writes block ob of the pair's own σ_k buffer
            struct Group {
                int ob;
                std::vector<int> idx;
                long long c_extra;       // byte offset of the σ_k buffer inside the per-pair region
            };
            std::vector<Group> groups;
            if (!o.per_pair_output) {
                std::vector<std::vector<int>> by_ob(pb.size());
                for (size_t i = 0; i < tasks.size(); ++i) by_ob[tasks[i].ob].push_back(int(i));
                for (size_t ob = 0; ob < pb.size(); ++ob)
                    if (!by_ob[ob].empty()) groups.push_back({int(ob), std::move(by_ob[ob]), 0});
            } else {
                for (size_t i = 0; i < tasks.size(); ++i)
                    groups.push_back({tasks[i].ob, std::vector<int>(1, int(i)), (long long)(tasks[i].k - ch.k_first) * pp_vec_bytes});
            }
            // total cost → target cost of a unit
            int64_t total_cost = 0;
            for (const Group& gr : groups) {
                const int ob = gr.ob;
                int64_t nkt = 0;
                for (int i : gr.idx) nkt += (tasks[i].s2.klen + TILE_K - 1) / TILE_K;
                tile_cuts(pb[ob].rows, tile_m, cut_r);
                tile_cuts(pb[ob].ld, TILE_N, cut_c);
                for (size_t ti = 0; ti + 1 < cut_r.size(); ++ti)
                    for (size_t tj = 0; tj + 1 < cut_c.size(); ++tj)
                        total_cost += cost_of(cut_r[ti + 1] - cut_r[ti], std::min(cut_c[tj + 1], pb[ob].cols) - cut_c[tj], nkt);
            }
            const int64_t target = o.per_pair_output ? (int64_t(1) << 60)
                                 : std::max<int64_t>(64 * 256 / TILE_K, total_cost / std::max<int64_t>(1, slots * o.split_waves));
            // Launch order = the queue order of the persistent kernel: longest first (LPT), and among units
            // of equal cost those of one (output block, k-range) together, row tile by row tile — they run
            // at the same time and share their T row tiles and R column tiles in L2.
            struct U2 {
                int64_t cost;            // queue key: the cost of the LARGEST tile of the unit's (group, split)
                Unit u;
                int32_t grp, split;
            };
            std::vector<U2> tmp;
            int64_t partial_tiles = 0;
            int32_t gi = -1;
            for (const Group& gr : groups) {
                ++gi;
                const int ob = gr.ob;
                const int seg0 = int(segs.size() - ch.p2_seg0);
                std::vector<int64_t> prefix(1, 0);
                for (int i : gr.idx) {
                    segs.push_back(tasks[i].s2);
                    prefix.push_back(prefix.back() + (tasks[i].s2.klen + TILE_K - 1) / TILE_K);
                }
                const int ns = int(gr.idx.size());
                const int64_t nkt = prefix.back();
                const Block& B = pb[ob];
                tile_cuts(B.rows, tile_m, cut_r);
                tile_cuts(B.ld, TILE_N, cut_c);
                // One split plan per GROUP, taken from its largest tile (the first one): every tile of the block
                // is cut at the same segment boundaries, and all units of a (group, split) carry the same queue
                // key, so they are claimed together and stream the same T row tiles and R column tiles through
                // L2 at the same time (profiles/r2_final_summary.md: DRAM traffic).
                const int rt0 = cut_r[1] - cut_r[0], cc0 = std::min(cut_c[1] - cut_c[0], B.cols);
                const int64_t c = cost_of(rt0, cc0, nkt);
                int n_split = int(std::min<int64_t>(ns, (c + target - 1) / target));
                if (n_split < 1) n_split = 1;
                for (size_t ti = 0; ti + 1 < cut_r.size(); ++ti)
                    for (size_t tj = 0; tj + 1 < cut_c.size(); ++tj) {
                        const int i0 = cut_r[ti], j0 = cut_c[tj], rt = cut_r[ti + 1] - i0, ct = cut_c[tj + 1] - j0;
                        Unit u;
                        memset(&u, 0, sizeof(u));
                        u.alpha = 1.0;
                        u.i0 = i0;
                        u.j0 = j0;
                        u.mrows = B.rows;
                        u.ncols = B.cols;
                        u.ncols_st = B.ld;
                        u.tile = pack_tile(rt, ct);
                        const unsigned long long c_sigma = (unsigned long long)(B.off * 8);     // block origin in σ
                        u.c_rp = B.rows_pad;
                        if (o.per_pair_output) {
                            u.C = c_sigma + (unsigned long long)gr.c_extra;   // + base of the per-pair region (rebased below)
                            u.seg_begin = seg0;
                            u.seg_end = seg0 + ns;
                            u.mode = BASE_WS << UNIT_C_SEL_SHIFT;             // the only writer of this block: no accumulation
                            u.pad_ = 1;
                            u.nkt = int32_t(nkt);
                            tmp.push_back({c, u, gi, 0});
                        } else if (n_split == 1) {
                            u.C = c_sigma;
                            u.seg_begin = seg0;
                            u.seg_end = seg0 + ns;
                            u.mode = UNIT_ACCUM | (BASE_SIGMA << UNIT_C_SEL_SHIFT);
                            u.nkt = int32_t(nkt);
                            tmp.push_back({c, u, gi, 0});
                        } else {
                            RUnit r;
                            r.C = c_sigma;
                            r.P = (unsigned long long)(partial_tiles * tile_m * TILE_N * 8);   // rebased below
                            r.c_rp = B.rows_pad;
                            r.i0 = i0;
                            r.j0 = j0;
                            r.rows = rt;
                            r.cols = ct;
                            int made = 0, sb = 0;
                            for (int s = 0; s < n_split; ++s) {
                                // even split of the k-tiles along segment boundaries
                                const int64_t want = nkt * (s + 1) / n_split;
                                int se = sb;
                                while (se < ns && prefix[se] < want) ++se;
                                if (s == n_split - 1) se = ns;
                                if (se == sb) continue;
                                u.C = (unsigned long long)((partial_tiles + made) * tile_m * TILE_N * 8);
                                u.seg_begin = seg0 + sb;
                                u.seg_end = seg0 + se;
                                u.mode = UNIT_C_PLAIN | (BASE_WS << UNIT_C_SEL_SHIFT);
                                u.nkt = int32_t(prefix[se] - prefix[sb]);
                                tmp.push_back({cost_of(rt0, cc0, u.nkt), u, gi, made});
                                ++made;
                                sb = se;
                            }
                            r.n_split = made;
                            partial_tiles += made;
                            runits.push_back(r);
                        }
                    }
            }
            std::stable_sort(tmp.begin(), tmp.end(), [](const U2& a, const U2& b) {
                if (a.cost != b.cost) return a.cost > b.cost;
                if (a.grp != b.grp) return a.grp < b.grp;
                return a.split < b.split;                  // then generation order: i0, j0
            });
            for (const U2& x : tmp) units.push_back(x.u);
            ch.p2_units = int64_t(tmp.size());
            {
                int64_t kt = 0;
                for (const U2& x : tmp) kt += x.u.nkt;
                ch.p2_short = kt < SHORT_UNIT_TILES * ch.p2_units;
            }
            ch.p2_segs = int64_t(segs.size()) - ch.p2_seg0;
            ch.r_units = int64_t(runits.size()) - ch.r_unit0;
            max_partial_tiles = std::max(max_partial_tiles, partial_tiles);
        }

        // ---- a4: diagonal tasks of this chunk, grouped by block ----
        {
            std::vector<std::vector<int>> by_b(pb.size());
            for (size_t i = 0; i < tasks.size(); ++i)
                if (tasks[i].diag) by_b[tasks[i].ib].push_back(int(i));
            ch.d_block0 = int64_t(dblocks.size());
            for (size_t b = 0; b < pb.size(); ++b) {
                if (by_b[b].empty()) continue;
                DiagBlock d;
                d.off = pb[b].off;
                d.rows = pb[b].rows;
                d.cols = pb[b].cols;
                d.ld = pb[b].ld;
                d.rows_pad = pb[b].rows_pad;
                d.t_begin = int32_t(dtasks.size());
                for (int i : by_b[b]) {
                    Task& t = tasks[i];
                    DiagTask dt;
                    memset(&dt, 0, sizeof(dt));
                    dt.L = t.Laddr();
                    dt.R = t.Raddr();
                    dt.alpha = t.alpha;
                    dt.l_rp = t.Lrp();
                    dt.r_rp = t.Rrp();
                    dt.sel = t.Lsel() | (t.Rsel() << 2);
                    dtasks.push_back(dt);
                }
                d.t_end = int32_t(dtasks.size());
                dblocks.push_back(d);
            }
            ch.d_blocks = int64_t(dblocks.size()) - ch.d_block0;
        }
        h->chunks.push_back(std::move(ch));
    }

    // ---- workspace layout: [T | partial tiles | ring half 0 | ring half 1] --------------------
    h->t_bytes = round_up(max_t_bytes, 128);
    h->partial_bytes = max_partial_tiles * tile_m * TILE_N * 8;
    bool any_pinned = false;
    for (const Chunk& c : h->chunks) any_pinned |= !c.copies.empty();
    h->has_pinned = any_pinned;
    h->ring_bytes = any_pinned ? 3 * ring_part : 0;
    h->ring_part_bytes = ring_part;
    // workspace layout: [T buffer 0 | T buffer 1 | partial tiles | ring part 0 | 1 | 2]
    h->pp_vec_bytes = pp_vec_bytes;
    h->pp_bytes = o.per_pair_output ? max_pairs * pp_vec_bytes + round_up(dmrgk_vec_scratch_bytes(64), 128) : 0;
    h->pp_base = 2 * h->t_bytes + h->partial_bytes + h->ring_bytes;
    h->workspace_bytes = std::max<int64_t>(128, h->pp_base + h->pp_bytes);
    const unsigned long long part_base = (unsigned long long)(2 * h->t_bytes);
    const unsigned long long ring_base = part_base + (unsigned long long)h->partial_bytes;

    // rebase: chunk-local segment indices → global, partial offsets → workspace, ring offsets
    for (size_t ci = 0; ci < h->chunks.size(); ++ci) {
        const Chunk& c = h->chunks[ci];
        const unsigned long long ring = ring_base + (unsigned long long)(c.ring_part) * ring_part;
        const unsigned long long tbuf = (unsigned long long)(ci & 1) * (unsigned long long)h->t_bytes;
        for (int64_t i = c.p1_unit0; i < c.p1_unit0 + c.p1_units; ++i) {
            units[i].seg_begin += int32_t(c.p1_seg0);
            units[i].seg_end += int32_t(c.p1_seg0);
            units[i].C += tbuf;                                   // phase 1 writes T buffer ci mod 2
        }
        for (int64_t sgi = c.p2_seg0; sgi < c.p2_seg0 + c.p2_segs; ++sgi) {                      // phase 2 reads it
            if (segs[sgi].flags & SEG_A_TBUF) segs[sgi].A += tbuf;
            if (segs[sgi].flags & SEG_B_TBUF) segs[sgi].B += tbuf;
        }
        for (int64_t i = c.p2_unit0; i < c.p2_unit0 + c.p2_units; ++i) {
            units[i].seg_begin += int32_t(c.p2_seg0);
            units[i].seg_end += int32_t(c.p2_seg0);
            if (units[i].mode & UNIT_C_PLAIN) units[i].C += part_base;
            if (units[i].pad_) {
                units[i].C += (unsigned long long)h->pp_base;
                units[i].pad_ = 0;
            }
        }
        for (int64_t i = c.r_unit0; i < c.r_unit0 + c.r_units; ++i) runits[i].P += part_base;
        for (int64_t s = c.p1_seg0; s < c.p2_seg0 + c.p2_segs; ++s) {      // staged operator blocks (the two phases' segments are contiguous)
            if (((segs[s].flags >> SEG_A_SEL_SHIFT) & 3u) == BASE_WS && !(segs[s].flags & SEG_A_TBUF)) segs[s].A += ring;
            if (((segs[s].flags >> SEG_B_SEL_SHIFT) & 3u) == BASE_WS && !(segs[s].flags & SEG_B_TBUF)) segs[s].B += ring;
        }
        for (int64_t b = c.d_block0; b < c.d_block0 + c.d_blocks; ++b)
            for (int t = dblocks[b].t_begin; t < dblocks[b].t_end; ++t) {
                if ((dtasks[t].sel & 3u) == BASE_WS) dtasks[t].L += ring;
                if (((dtasks[t].sel >> 2) & 3u) == BASE_WS) dtasks[t].R += ring;
            }
    }
    if (int64_t(segs.size()) > 0x7fffffffLL) return bail(fail(DMRGK_EINVAL, "heff_create: too many segments"));

    h->K = K;
    h->n_launches = 1;
    for (const Chunk& c : h->chunks) h->n_launches += (c.p1_units > 0) + (c.p2_units > 0) + (c.r_units > 0);

    int32_t s = upload(units, &h->units_dev);
    if (s == DMRGK_OK) s = upload(segs, &h->segs_dev);
    if (s == DMRGK_OK) s = upload(runits, &h->runits_dev);
    if (s == DMRGK_OK) s = upload(dblocks, &h->dblocks_dev);
    if (s == DMRGK_OK) s = upload(dtasks, &h->dtasks_dev);
    if (s != DMRGK_OK) return bail(s);
    if (cudaMalloc(&h->counters_dev, (2 * h->chunks.size() + 2) * sizeof(int)) != cudaSuccess)
        return bail(fail(DMRGK_ECUDA, "heff_create: queue counters"));
    {
        int prio_lo = 0, prio_hi = 0;
        cudaError_t e = cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
        if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&h->side, cudaStreamNonBlocking, prio_lo);
        if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&h->side_hi, cudaStreamNonBlocking, prio_hi);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_join1, cudaEventDisableTiming);
        for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
            e = cudaEventCreateWithFlags(&h->ev_p1[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_p2[i], cudaEventDisableTiming);
        }
        for (int i = 0; i < 3 && e == cudaSuccess && any_pinned; ++i) {
            e = cudaEventCreateWithFlags(&h->ev_copy[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) return bail(fail(DMRGK_ECUDA, "heff_create: stream/event: %s", cudaGetErrorString(e)));
    }
    *out = h;
    return DMRGK_OK;
}

int32_t dmrgk_heff_query(const dmrgk_heff* h, int64_t* n_tasks, double* flops_alg, double* flops_exec,
                         int64_t* op_bytes, int64_t* workspace_bytes, int64_t* n_chunks,
                         int64_t* n_launches_per_apply) {
    if (!h) return fail(DMRGK_EINVAL, "heff_query: heff is NULL");
    if (n_tasks) *n_tasks = h->n_tasks;
    if (flops_alg) *flops_alg = h->flops_alg;
    if (flops_exec) *flops_exec = h->flops_exec;
    if (op_bytes) *op_bytes = h->op_bytes;
    if (workspace_bytes) *workspace_bytes = h->workspace_bytes;
    if (n_chunks) *n_chunks = int64_t(h->chunks.size());
    if (n_launches_per_apply) *n_launches_per_apply = h->n_launches;
    return DMRGK_OK;
}

}  // extern "C"

namespace dmrgk {

// Stage the pinned operators of chunk c into its ring half on the copy stream, ordered after the
// last compute that read that half and before the compute that needs it (a3).
static int32_t stage_chunk(dmrgk_heff* h, const Chunk& c, char* ws, cudaStream_t main, cudaStream_t copy,
                           cudaStream_t side = nullptr, cudaStream_t side2 = nullptr) {
    if (c.copies.empty()) return DMRGK_OK;
    const int hf = c.ring_part;
    char* ring = ws + 2 * h->t_bytes + h->partial_bytes + int64_t(hf) * h->ring_part_bytes;
    if (h->done_recorded[hf]) DMRGK_CUDA(cudaStreamWaitEvent(copy, h->ev_done[hf], 0));
    for (const StageCopy& sc : c.copies)
        DMRGK_CUDA(cudaMemcpyAsync(ring + sc.ring_off * 8, sc.src_host, size_t(sc.n) * 8, cudaMemcpyHostToDevice, copy));
    DMRGK_CUDA(cudaEventRecord(h->ev_copy[hf], copy));
    DMRGK_CUDA(cudaStreamWaitEvent(main, h->ev_copy[hf], 0));
    if (side) DMRGK_CUDA(cudaStreamWaitEvent(side, h->ev_copy[hf], 0));
    if (side2) DMRGK_CUDA(cudaStreamWaitEvent(side2, h->ev_copy[hf], 0));
    return DMRGK_OK;
}

// Profiling (dmrgk_heff_profile): an event pair around one launch; the pool grows on demand.
static int32_t prof_begin(dmrgk_heff* h, int kind, cudaStream_t st, size_t* slot) {
    *slot = 0;
    if (!h->prof_on) return DMRGK_OK;
    while (h->prof_ev.size() < 2 * (h->prof_used + 1)) {
        cudaEvent_t e;
        DMRGK_CUDA(cudaEventCreate(&e));
        h->prof_ev.push_back(e);
    }
    if (h->prof_kind.size() <= h->prof_used) h->prof_kind.resize(h->prof_used + 1);
    *slot = h->prof_used++;
    h->prof_kind[*slot] = kind;
    DMRGK_CUDA(cudaEventRecord(h->prof_ev[2 * *slot], st));
    return DMRGK_OK;
}
static int32_t prof_end(dmrgk_heff* h, size_t slot, cudaStream_t st) {
    if (!h->prof_on) return DMRGK_OK;
    DMRGK_CUDA(cudaEventRecord(h->prof_ev[2 * slot + 1], st));
    return DMRGK_OK;
}
// Fold the recorded pairs into the running sums (synchronises on the last event).
static int32_t prof_collect(dmrgk_heff* h) {
    for (size_t i = 0; i < h->prof_used; ++i) {
        DMRGK_CUDA(cudaEventSynchronize(h->prof_ev[2 * i + 1]));
        float ms = 0.f;
        DMRGK_CUDA(cudaEventElapsedTime(&ms, h->prof_ev[2 * i], h->prof_ev[2 * i + 1]));
        h->prof_ms[h->prof_kind[i]] += ms;
        ++h->prof_launches[h->prof_kind[i]];
    }
    h->prof_used = 0;
    return DMRGK_OK;
}

static int32_t chunk_done(dmrgk_heff* h, const Chunk& c, cudaStream_t main) {
    if (c.copies.empty()) return DMRGK_OK;
    DMRGK_CUDA(cudaEventRecord(h->ev_done[c.ring_part], main));
    h->done_recorded[c.ring_part] = true;
    return DMRGK_OK;
}

}  // namespace dmrgk


// σ = H_eff ψ (expect_dev == NULL) or the per-pair expectation values (sigma_dev == NULL)
static int32_t run_plan(dmrgk_heff* h, const double* psi_dev, double* sigma_dev, double* expect_dev, void* workspace_dev,
                        void* stream_main, void* stream_copy) {
    const int64_t n = h->layout->n_padded;
    if (n == 0) return DMRGK_OK;
    const bool expect = expect_dev != nullptr;
    if (!psi_dev || (!expect && !sigma_dev)) return fail(DMRGK_EINVAL, "heff_apply: NULL vector");
    if (!expect && psi_dev == sigma_dev) return fail(DMRGK_EINVAL, "heff_apply: psi and sigma alias");
    if (!workspace_dev && h->n_tasks) return fail(DMRGK_EINVAL, "heff_apply: NULL workspace");
    if (!aligned128(psi_dev) || (sigma_dev && !aligned128(sigma_dev)) || !aligned128(workspace_dev))
        return fail(DMRGK_EALIGN, "heff_apply: pointers must be 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(h->ctx->device));
    cudaStream_t main = (cudaStream_t)stream_main, copy = (cudaStream_t)stream_copy;
    if (h->has_pinned && copy == main)
        return fail(DMRGK_EINVAL, "heff_apply: pinned operators need a copy stream distinct from the main stream");
    Bases bases;
    bases.b[BASE_ABS] = 0;
    bases.b[BASE_WS] = (unsigned long long)(uintptr_t)workspace_dev;
    bases.b[BASE_PSI] = (unsigned long long)(uintptr_t)psi_dev;
    bases.b[BASE_SIGMA] = (unsigned long long)(uintptr_t)sigma_dev;
    if (!expect) DMRGK_CUDA(cudaMemsetAsync(sigma_dev, 0, size_t(n) * 8, main));
    DMRGK_CUDA(cudaMemsetAsync(h->counters_dev, 0, (2 * h->chunks.size() + 2) * sizeof(int), main));
    // Stream choreography (all ordering by events; s1 and s2 are library-owned, non-blocking):
    //   s1 (lowest priority)  : p1(0)            p1(1)              p1(2) …   phase 1 of chunk c → T buffer c mod 2
    //   s2 (greatest priority):        p2(0) r(0)       p2(1) r(1) …          phase 2 + reduce of chunk c
    // p2(c) waits for p1(c); p1(c+2) waits for p2(c) (T buffer re-use); p1(c+1) overlaps p2(c).  s2's
    // priority makes the block scheduler dispatch the few long stacked-k units of p2(c) first and fill
    // the remaining slots — and the tail — with the many short units of p1(c+1).  The caller's stream
    // forks into s1/s2 after the memset of σ and joins them before apply returns, so the caller only
    // ever has to order against `main`.
    // Copies of chunk c+1 are enqueued before the compute of chunk c so that they overlap it.
    const size_t nc = h->chunks.size();
    const bool serial = h->prof_on && h->prof_serial;   // diagnostic mode: one stream, per-launch events
    cudaStream_t s1 = serial ? main : h->side, s2 = serial ? main : h->side_hi;
    size_t span_slot = 0, slot = 0;
    DMRGK_TRY(prof_begin(h, 3, main, &span_slot));
    DMRGK_CUDA(cudaEventRecord(h->ev_fork, main));
    if (!serial) {
        DMRGK_CUDA(cudaStreamWaitEvent(s1, h->ev_fork, 0));
        DMRGK_CUDA(cudaStreamWaitEvent(s2, h->ev_fork, 0));
    }
    // The chunk loop runs inside a lambda so that EVERY exit path — also a failed launch or event call
    // half-way — joins the library-owned streams back into `main` and closes the profiling span: the
    // caller only orders against `main` and may free ψ / σ / workspace right after an error return.
    auto enqueue_chunks = [&]() -> int32_t {
    if (nc) DMRGK_TRY(stage_chunk(h, h->chunks[0], (char*)workspace_dev, main, copy, s1, s2));
    for (size_t c = 0; c < nc; ++c) {
        const Chunk& ch = h->chunks[c];
        if (ch.p1_units) {
            if (c >= 2) DMRGK_CUDA(cudaStreamWaitEvent(s1, h->ev_p2[c & 1], 0));
            if (serial) DMRGK_TRY(prof_begin(h, 0, s1, &slot));
            DMRGK_TRY(launch_gemm_units(h->opts.kernel, h->units_dev + ch.p1_unit0, h->segs_dev, ch.p1_units, bases, s1, h->counters_dev + 2 * c, h->ctx->n_sm, ch.p1_short));
            if (serial) DMRGK_TRY(prof_end(h, slot, s1));
            DMRGK_CUDA(cudaEventRecord(h->ev_p1[c & 1], s1));
            DMRGK_CUDA(cudaStreamWaitEvent(s2, h->ev_p1[c & 1], 0));
        }
        if (expect && ch.k_count)       // blocks of σ_k that no task writes must read as zero
            DMRGK_CUDA(cudaMemsetAsync((char*)workspace_dev + h->pp_base, 0, size_t(ch.k_count) * h->pp_vec_bytes, s2));
        if (serial && ch.p2_units) DMRGK_TRY(prof_begin(h, 1, s2, &slot));
        DMRGK_TRY(launch_gemm_units(h->opts.kernel, h->units_dev + ch.p2_unit0, h->segs_dev, ch.p2_units, bases, s2, h->counters_dev + 2 * c + 1, h->ctx->n_sm, ch.p2_short));
        if (serial && ch.p2_units) DMRGK_TRY(prof_end(h, slot, s2));
        if (serial && ch.r_units) DMRGK_TRY(prof_begin(h, 2, s2, &slot));
        DMRGK_TRY(launch_reduce(h->runits_dev + ch.r_unit0, ch.r_units, bases, s2, gemm_tile_m(h->opts.kernel)));
        if (serial && ch.r_units) DMRGK_TRY(prof_end(h, slot, s2));
        if (expect) {
            // out[k] = ⟨σ_k, ψ⟩ for the pairs of this chunk, 64 at a time (fused, fixed-order dots)
            char* pp = (char*)workspace_dev + h->pp_base;
            void* scratch = pp + h->pp_bytes - round_up(dmrgk_vec_scratch_bytes(64), 128);
            for (int64_t g0 = 0; g0 < ch.k_count; g0 += 64) {
                const int cnt = int(std::min<int64_t>(64, ch.k_count - g0));
                DMRGK_TRY(dmrgk_vec_multi_dot(h->ctx, n, cnt, reinterpret_cast<const double*>(pp + g0 * h->pp_vec_bytes),
                                              h->pp_vec_bytes / 8, psi_dev, expect_dev + ch.k_first + g0, scratch, s2));
            }
        }
        DMRGK_CUDA(cudaEventRecord(h->ev_p2[c & 1], s2));
        DMRGK_TRY(chunk_done(h, ch, s2));
        if (c + 1 < nc) DMRGK_TRY(stage_chunk(h, h->chunks[c + 1], (char*)workspace_dev, main, copy, s1, s2));
    }
    return DMRGK_OK;
    };
    const int32_t status = enqueue_chunks();
    if (!serial) {
        // on success s2 has already waited for every p1 launch of s1; after an error it may not have,
        // so main waits for both streams explicitly
        cudaError_t e = cudaEventRecord(h->ev_join, s2);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(main, h->ev_join, 0);
        if (e == cudaSuccess) e = cudaEventRecord(h->ev_join1, s1);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(main, h->ev_join1, 0);
        if (e != cudaSuccess) {
            cudaStreamSynchronize(s1);                    // last resort: nothing may outlive the call
            cudaStreamSynchronize(s2);
            if (status == DMRGK_OK) return fail(DMRGK_ECUDA, "heff_apply: join failed: %s", cudaGetErrorString(e));
        }
    }
    {
        const int32_t ps = prof_end(h, span_slot, main);
        if (status != DMRGK_OK) return status;
        if (ps != DMRGK_OK) return ps;
    }
    if (h->prof_on && !serial) {
        for (const Chunk& ch : h->chunks) {
            h->prof_launches[0] += ch.p1_units > 0;
            h->prof_launches[1] += ch.p2_units > 0;
            h->prof_launches[2] += ch.r_units > 0;
        }
    }
    return DMRGK_OK;
}

extern "C" {

int32_t dmrgk_heff_apply(dmrgk_heff* h, const double* psi_dev, double* sigma_dev, void* workspace_dev,
                         void* stream_main, void* stream_copy) {
    if (!h) return fail(DMRGK_EINVAL, "heff_apply: heff is NULL");
    if (h->opts.per_pair_output) return fail(DMRGK_ESTATE, "heff_apply: the plan was created with per_pair_output (use heff_expect)");
    if (h->layout->n_padded && !sigma_dev) return fail(DMRGK_EINVAL, "heff_apply: NULL vector");
    return run_plan(h, psi_dev, sigma_dev, nullptr, workspace_dev, stream_main, stream_copy);
}

int32_t dmrgk_heff_expect(dmrgk_heff* h, const double* psi_dev, double* out_dev, void* workspace_dev,
                          void* stream_main, void* stream_copy) {
    if (!h) return fail(DMRGK_EINVAL, "heff_expect: heff is NULL");
    if (!h->opts.per_pair_output) return fail(DMRGK_ESTATE, "heff_expect: the plan was not created with per_pair_output");
    if (h->K == 0) return DMRGK_OK;
    if (!out_dev) return fail(DMRGK_EINVAL, "heff_expect: out is NULL");
    DMRGK_CUDA(cudaSetDevice(h->ctx->device));
    DMRGK_CUDA(cudaMemsetAsync(out_dev, 0, size_t(h->K) * 8, (cudaStream_t)stream_main));     // pairs without any task
    return run_plan(h, psi_dev, nullptr, out_dev, workspace_dev, stream_main, stream_copy);
}

int32_t dmrgk_heff_profile(dmrgk_heff* h, int32_t enable) {
    if (!h) return fail(DMRGK_EINVAL, "heff_profile: heff is NULL");
    if (h->prof_used) DMRGK_TRY(prof_collect(h));
    h->prof_on = enable != 0;
    h->prof_serial = enable == 2;
    for (int i = 0; i < 4; ++i) {
        h->prof_ms[i] = 0.0;
        h->prof_launches[i] = 0;
    }
    return DMRGK_OK;
}

int32_t dmrgk_heff_profile_read(dmrgk_heff* h, double* ms, int64_t* launches) {
    if (!h) return fail(DMRGK_EINVAL, "heff_profile_read: heff is NULL");
    DMRGK_TRY(prof_collect(h));
    for (int i = 0; i < 4; ++i) {
        if (ms) ms[i] = h->prof_ms[i];
        if (launches) launches[i] = h->prof_launches[i];
    }
    return DMRGK_OK;
}

int32_t dmrgk_heff_apply_host(dmrgk_heff* h, const double* psi_host, double* sigma_host,
                              double* psi_dev, double* sigma_dev, void* workspace_dev,
                              void* stream_main, void* stream_copy) {
    if (!h) return fail(DMRGK_EINVAL, "heff_apply_host: heff is NULL");
    const int64_t n = h->layout->n_padded;
    if (n == 0) return DMRGK_OK;
    if (!psi_host || !sigma_host || !psi_dev || !sigma_dev) return fail(DMRGK_EINVAL, "heff_apply_host: NULL buffer");
    DMRGK_CUDA(cudaSetDevice(h->ctx->device));
    cudaStream_t main = (cudaStream_t)stream_main;
    DMRGK_CUDA(cudaMemcpyAsync(psi_dev, psi_host, size_t(n) * 8, cudaMemcpyHostToDevice, main));
    DMRGK_TRY(dmrgk_heff_apply(h, psi_dev, sigma_dev, workspace_dev, stream_main, stream_copy));
    DMRGK_CUDA(cudaMemcpyAsync(sigma_host, sigma_dev, size_t(n) * 8, cudaMemcpyDeviceToHost, main));
    DMRGK_CUDA(cudaStreamSynchronize(main));
    return DMRGK_OK;
}

int32_t dmrgk_heff_diag(dmrgk_heff* h, double* diag_dev, void* workspace_dev, void* stream_main,
                        void* stream_copy) {
    if (!h) return fail(DMRGK_EINVAL, "heff_diag: heff is NULL");
    if (h->opts.per_pair_output) return fail(DMRGK_ESTATE, "heff_diag: the plan was created with per_pair_output");
    const int64_t n = h->layout->n_padded;
    if (n == 0) return DMRGK_OK;
    if (!diag_dev) return fail(DMRGK_EINVAL, "heff_diag: NULL vector");
    if (!aligned128(diag_dev) || !aligned128(workspace_dev)) return fail(DMRGK_EALIGN, "heff_diag: pointers must be 128-byte aligned");
    if (h->has_pinned && !workspace_dev) return fail(DMRGK_EINVAL, "heff_diag: NULL workspace");
    DMRGK_CUDA(cudaSetDevice(h->ctx->device));
    cudaStream_t main = (cudaStream_t)stream_main, copy = (cudaStream_t)stream_copy;
    if (h->has_pinned && copy == main)
        return fail(DMRGK_EINVAL, "heff_diag: pinned operators need a copy stream distinct from the main stream");
    Bases bases;
    bases.b[BASE_ABS] = 0;
    bases.b[BASE_WS] = (unsigned long long)(uintptr_t)workspace_dev;
    bases.b[BASE_PSI] = 0;
    bases.b[BASE_SIGMA] = 0;
    DMRGK_CUDA(cudaMemsetAsync(diag_dev, 0, size_t(n) * 8, main));
    for (const Chunk& ch : h->chunks) {
        if (ch.d_blocks == 0) continue;
        DMRGK_TRY(stage_chunk(h, ch, (char*)workspace_dev, main, copy));
        DMRGK_TRY(launch_diag(h->dblocks_dev + ch.d_block0, h->dtasks_dev, ch.d_blocks, diag_dev, bases, main));
        DMRGK_TRY(chunk_done(h, ch, main));
    }
    return DMRGK_OK;
}

}  // extern "C"
