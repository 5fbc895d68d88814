// renorm.cu — renormalisation step O′ = Φᵀ O Φ of block operators (
// PAPER.md:60 §II.A "the renormalization step", Fig. 7 "Ren_l", "Ren_r").
//
// Per stored block of operator i:   out_i[q+δ, q] = Φ[q+δ]ᵀ · in_i[q+δ, q] · Φ[q]
//   phase 1:  T = in_i[q+δ, q] · Φ[q]          A = operator block (K-major), B = Φ[q] (N-major)
//   phase 2:  out = Φ[q+δ]ᵀ · T                A = Φ[q+δ] (M-major),        B = T (N-major)
// Both phases are work lists for the grouped FP64 tensor-core kernel of heff_kernels.cu (one segment
// per unit, output written directly — every output tile has exactly one producer, so nothing is
// accumulated).  Operators are processed in chunks so that T fits its workspace.
#include "internal.h"
#include <algorithm>
#include <cstring>
#include <new>

using namespace dmrgk;

namespace {

struct RTask {
    const Block *ob, *pc, *pr;   // operator block, Φ[q] (column sector), Φ[q+δ] (row sector)
    const double *in, *out;      // device arenas of in_i / out_i
    const Block* outb;           // output block of out_i
};


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

void dmrgk_renorm_destroy(dmrgk_renorm* r) {
    if (!r) return;
    cudaFree(r->units_dev);
    cudaFree(r->segs_dev);
    cudaFree(r->counters_dev);
    for (int i = 0; i < 2; ++i) {
        if (r->ev_p1[i]) cudaEventDestroy(r->ev_p1[i]);
        if (r->ev_p2[i]) cudaEventDestroy(r->ev_p2[i]);
    }
    if (r->ev_fork) cudaEventDestroy(r->ev_fork);
    if (r->ev_join) cudaEventDestroy(r->ev_join);
    if (r->ev_join1) cudaEventDestroy(r->ev_join1);
    if (r->s1) cudaStreamDestroy(r->s1);
    if (r->s2) cudaStreamDestroy(r->s2);
    delete r;
}

int32_t dmrgk_renorm_create(dmrgk_ctx* ctx, const dmrgk_iso* phi, int64_t n_ops, dmrgk_op* const* in,
                            dmrgk_op* const* out, const dmrgk_renorm_opts* opts, dmrgk_renorm** plan) {
    if (!plan) return fail(DMRGK_EINVAL, "renorm_create: plan is NULL");
    *plan = nullptr;
    if (!ctx || !phi) return fail(DMRGK_EINVAL, "renorm_create: NULL ctx or phi");
    if (n_ops < 0 || (n_ops > 0 && (!in || !out))) return fail(DMRGK_EINVAL, "renorm_create: bad operator arrays");
    if (phi->n_padded && !phi->dev) return fail(DMRGK_ESTATE, "renorm_create: phi is not bound to a device arena");
    dmrgk_renorm_opts o;
    memset(&o, 0, sizeof(o));
    if (opts) o = *opts;
    const bool default_chunk = o.t_chunk_bytes <= 0;
    if (o.kernel < 0 || o.kernel > 5) return fail(DMRGK_EINVAL, "renorm_create: bad options");
    if (!gemm_kernel_available(o.kernel))
        return fail(DMRGK_EINVAL, "renorm_create: kernel variant %d is not resident on this device (use 0)", o.kernel);
    for (int64_t i = 0; i < n_ops; ++i) {
        if (!in[i] || !out[i]) return fail(DMRGK_EINVAL, "renorm_create: operator %lld is NULL", (long long)i);
        if (in[i]->space != phi->enl) return fail(DMRGK_ESHAPE, "renorm_create: in[%lld] is not on phi's enlarged space", (long long)i);
        if (out[i]->space != phi->kept) return fail(DMRGK_ESHAPE, "renorm_create: out[%lld] is not on phi's kept space", (long long)i);
        if (in[i]->dq[0] != out[i]->dq[0] || in[i]->dq[1] != out[i]->dq[1] || in[i]->parity != out[i]->parity)
            return fail(DMRGK_ECHARGE, "renorm_create: in[%lld] and out[%lld] differ in charge shift or parity", (long long)i, (long long)i);
        if ((in[i]->n_padded && !in[i]->dev) || (out[i]->n_padded && !out[i]->dev))
            return fail(DMRGK_ESTATE, "renorm_create: operator %lld is not bound to a device arena", (long long)i);
    }
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    dmrgk_renorm* r = new (std::nothrow) dmrgk_renorm;
    if (!r) return fail(DMRGK_ENOMEM, "renorm_create: out of host memory");
    r->ctx = ctx;
    r->kernel = o.kernel;

    if (default_chunk) {   // about 16 chunks, between 256 MiB and 4 GiB (see dmrgk_heff_create)
        int64_t total = 0;
        for (int64_t i = 0; i < n_ops; ++i)
            for (const Block& ob : in[i]->blocks) {
                const int pc = phi->by_enl[ob.c_idx], pr = phi->by_enl[ob.r_idx];
                if (pc >= 0 && pr >= 0) total += int64_t(ob.rows_pad) * phi->blocks[pc].ld * 8;
            }
        o.t_chunk_bytes = std::min<int64_t>(int64_t(4) << 30, std::max<int64_t>(int64_t(256) << 20, total / 16));
    }
    std::vector<Unit> units;
    std::vector<Seg> segs;
    std::vector<int64_t> seg0_of_chunk;
    int64_t max_t = 0;
    int64_t i0 = 0;
    while (i0 < n_ops) {
        // ---- one chunk: operators [i0, i1) whose T intermediates fit o.t_chunk_bytes ----
        std::vector<RTask> tasks;
        int64_t t_bytes = 0, i1 = i0;
        for (; i1 < n_ops; ++i1) {
            std::vector<RTask> mine;
            int64_t tb = 0;
            for (const Block& ob : in[i1]->blocks) {
                const int pc = phi->by_enl[ob.c_idx], pr = phi->by_enl[ob.r_idx];
                if (pc < 0 || pr < 0) continue;
                const Block& bc = phi->blocks[pc];
                const Block& br = phi->blocks[pr];
                const int oi = out[i1]->by_col[bc.c_idx];
                if (oi < 0 || out[i1]->blocks[oi].r_idx != br.c_idx) {
                    dmrgk_renorm_destroy(r);
                    return fail(DMRGK_ESHAPE, "renorm_create: out[%lld] has no block for kept sectors (%d, %d)", (long long)i1, br.c_idx, bc.c_idx);
                }
                mine.push_back({&ob, &bc, &br, in[i1]->dev, out[i1]->dev, &out[i1]->blocks[oi]});
                tb += int64_t(ob.rows_pad) * bc.ld * 8;
            }
            if (!tasks.empty() && t_bytes + tb > o.t_chunk_bytes) break;
            tasks.insert(tasks.end(), mine.begin(), mine.end());
            t_bytes += tb;
        }
        i0 = i1;
        max_t = std::max(max_t, t_bytes);
        dmrgk_renorm::RChunk ch;
        seg0_of_chunk.push_back(int64_t(segs.size()));
        struct CU {
            int64_t cost;
            Unit u;
        };
        std::vector<CU> p1, p2;
        std::vector<int> cut_r, cut_c;
        const int tile_m = gemm_tile_m(o.kernel);
        int64_t t_off = 0;
        for (const RTask& t : tasks) {
            const int e_r = t.ob->rows, e_c = t.ob->cols, n_c = t.pc->cols, n_r = t.pr->cols;
            const int ldt = t.pc->ld;
            r->flops += 2.0 * e_r * e_c * n_c + 2.0 * n_r * e_r * n_c;
            ++r->n_tasks;
            // phase 1: T (e_r × n_c, ld ldt) = O (K-major) · Φ[q] (N-major)
            Seg s1;
            memset(&s1, 0, sizeof(s1));
            s1.A = (unsigned long long)(uintptr_t)(t.in + t.ob->off);
            s1.a_rp = t.ob->rows_pad;
            s1.B = (unsigned long long)(uintptr_t)(phi->dev + t.pc->off);
            s1.b_rp = t.pc->rows_pad;
            s1.klen = e_c;
            s1.flags = SEG_B_NMAJOR | (BASE_ABS << SEG_A_SEL_SHIFT) | (BASE_ABS << SEG_B_SEL_SHIFT);
            const int32_t si1 = int32_t(segs.size());
            segs.push_back(s1);
            const int64_t nkt1 = (e_c + TILE_K - 1) / TILE_K;
            tile_cuts(e_r, tile_m, cut_r);
            tile_cuts(ldt, TILE_N, cut_c);
            for (size_t ti = 0; ti + 1 < cut_r.size(); ++ti)
                for (size_t tj = 0; tj + 1 < cut_c.size(); ++tj) {
                    const int r0 = cut_r[ti], c0 = cut_c[tj], rt = cut_r[ti + 1] - r0, ct = cut_c[tj + 1] - c0;
                    Unit u;
                    memset(&u, 0, sizeof(u));
                    u.C = (unsigned long long)t_off;            // block origin of T (e_r × n_c, panel layout)
                    u.alpha = 1.0;
                    u.c_rp = pad_rows(e_r);
                    u.i0 = r0;
                    u.j0 = c0;
                    u.mrows = e_r;
                    u.ncols = n_c;
                    u.ncols_st = ldt;
                    u.seg_begin = si1;
                    u.seg_end = si1 + 1;
                    u.mode = BASE_WS << UNIT_C_SEL_SHIFT;
                    u.nkt = int32_t(nkt1);
                    u.tile = pack_tile(rt, ct);
                    p1.push_back({tile_cost(rt, std::min(ct, n_c - c0)) * nkt1, u});
                }
            // phase 2: out (n_r × n_c) = Φ[q+δ]ᵀ (M-major) · T (N-major)
            Seg s2;
            memset(&s2, 0, sizeof(s2));
            s2.A = (unsigned long long)(uintptr_t)(phi->dev + t.pr->off);
            s2.a_rp = t.pr->rows_pad;
            s2.B = (unsigned long long)t_off;
            s2.b_rp = pad_rows(e_r);
            s2.klen = e_r;
            s2.flags = SEG_A_MMAJOR | SEG_B_NMAJOR | (BASE_ABS << SEG_A_SEL_SHIFT) | (BASE_WS << SEG_B_SEL_SHIFT);
            const int32_t si2 = int32_t(segs.size());
            segs.push_back(s2);
            const int64_t nkt2 = (e_r + TILE_K - 1) / TILE_K;
            const int ldo = t.outb->ld;
            tile_cuts(n_r, tile_m, cut_r);
            tile_cuts(ldo, TILE_N, cut_c);
            for (size_t ti = 0; ti + 1 < cut_r.size(); ++ti)
                for (size_t tj = 0; tj + 1 < cut_c.size(); ++tj) {
                    const int r0 = cut_r[ti], c0 = cut_c[tj], rt = cut_r[ti + 1] - r0, ct = cut_c[tj + 1] - c0;
                    Unit u;
                    memset(&u, 0, sizeof(u));
                    u.C = (unsigned long long)(uintptr_t)(t.out + t.outb->off);     // block origin
                    u.alpha = 1.0;
                    u.c_rp = t.outb->rows_pad;
                    u.i0 = r0;
                    u.j0 = c0;
                    u.mrows = n_r;
                    u.ncols = n_c;
                    u.ncols_st = ldo;
                    u.seg_begin = si2;
                    u.seg_end = si2 + 1;
                    u.mode = BASE_ABS << UNIT_C_SEL_SHIFT;
                    u.nkt = int32_t(nkt2);
                    u.tile = pack_tile(rt, ct);
                    p2.push_back({tile_cost(rt, std::min(ct, n_c - c0)) * nkt2, u});
                }
            t_off += int64_t(pad_rows(e_r)) * ldt * 8;
        }
        auto by_cost = [](const CU& a, const CU& b) { return a.cost > b.cost; };
        std::stable_sort(p1.begin(), p1.end(), by_cost);
        std::stable_sort(p2.begin(), p2.end(), by_cost);
        ch.p1_unit0 = int64_t(units.size());
        for (const CU& x : p1) units.push_back(x.u);
        ch.p1_units = int64_t(p1.size());
        {
            int64_t k1 = 0, k2 = 0;
            for (const CU& x : p1) k1 += x.u.nkt;
            for (const CU& x : p2) k2 += x.u.nkt;
            ch.p1_short = k1 < SHORT_UNIT_TILES * int64_t(p1.size());
            ch.p2_short = k2 < SHORT_UNIT_TILES * int64_t(p2.size());
        }
        ch.p2_unit0 = int64_t(units.size());
        for (const CU& x : p2) units.push_back(x.u);
        ch.p2_units = int64_t(p2.size());
        r->chunks.push_back(ch);
    }
    if (int64_t(segs.size()) > 0x7fffffffLL) {
        dmrgk_renorm_destroy(r);
        return fail(DMRGK_EINVAL, "renorm_create: too many segments");
    }
    r->t_bytes = round_up(max_t, 128);
    r->workspace_bytes = std::max<int64_t>(128, 2 * r->t_bytes);      // two T buffers
    seg0_of_chunk.push_back(int64_t(segs.size()));
    for (size_t c = 1; c < r->chunks.size(); c += 2) {                // odd chunks use the second buffer
        const unsigned long long tbuf = (unsigned long long)r->t_bytes;
        const auto& ch = r->chunks[c];
        for (int64_t i = ch.p1_unit0; i < ch.p1_unit0 + ch.p1_units; ++i) units[i].C += tbuf;
        for (int64_t sgi = seg0_of_chunk[c]; sgi < seg0_of_chunk[c + 1]; ++sgi)
            if (((segs[sgi].flags >> SEG_B_SEL_SHIFT) & 3u) == BASE_WS) segs[sgi].B += tbuf;
    }
    {
        int lo = 0, hi = 0;
        cudaError_t e = cudaDeviceGetStreamPriorityRange(&lo, &hi);
        if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&r->s1, cudaStreamNonBlocking, lo);
        if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&r->s2, cudaStreamNonBlocking, hi);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&r->ev_fork, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&r->ev_join, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&r->ev_join1, cudaEventDisableTiming);
        for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
            e = cudaEventCreateWithFlags(&r->ev_p1[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&r->ev_p2[i], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) {
            dmrgk_renorm_destroy(r);
            return fail(DMRGK_ECUDA, "renorm_create: stream/event: %s", cudaGetErrorString(e));
        }
    }
    for (const auto& c : r->chunks) r->n_launches += (c.p1_units > 0) + (c.p2_units > 0);
    int32_t s = upload(units, &r->units_dev);
    if (s == DMRGK_OK) s = upload(segs, &r->segs_dev);
    if (s == DMRGK_OK && cudaMalloc(&r->counters_dev, (2 * r->chunks.size() + 2) * sizeof(int)) != cudaSuccess)
        s = fail(DMRGK_ECUDA, "renorm_create: queue counters");
    if (s != DMRGK_OK) {
        dmrgk_renorm_destroy(r);
        return s;
    }
    *plan = r;
    return DMRGK_OK;
}

int32_t dmrgk_renorm_query(const dmrgk_renorm* r, int64_t* n_tasks, double* flops, int64_t* workspace_bytes,
                           int64_t* n_launches_per_apply) {
    if (!r) return fail(DMRGK_EINVAL, "renorm_query: plan is NULL");
    if (n_tasks) *n_tasks = r->n_tasks;
    if (flops) *flops = r->flops;
    if (workspace_bytes) *workspace_bytes = r->workspace_bytes;
    if (n_launches_per_apply) *n_launches_per_apply = r->n_launches;
    return DMRGK_OK;
}

int32_t dmrgk_renorm_apply(dmrgk_renorm* r, void* workspace_dev, void* stream) {
    if (!r) return fail(DMRGK_EINVAL, "renorm_apply: plan is NULL");
    if (r->n_tasks == 0) return DMRGK_OK;
    if (!workspace_dev) return fail(DMRGK_EINVAL, "renorm_apply: NULL workspace");
    if (!aligned128(workspace_dev)) return fail(DMRGK_EALIGN, "renorm_apply: workspace must be 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(r->ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    Bases bases;
    bases.b[BASE_ABS] = 0;
    bases.b[BASE_WS] = (unsigned long long)(uintptr_t)workspace_dev;
    bases.b[BASE_PSI] = 0;
    bases.b[BASE_SIGMA] = 0;
    DMRGK_CUDA(cudaMemsetAsync(r->counters_dev, 0, (2 * r->chunks.size() + 2) * sizeof(int), st));
    DMRGK_CUDA(cudaEventRecord(r->ev_fork, st));
    DMRGK_CUDA(cudaStreamWaitEvent(r->s1, r->ev_fork, 0));
    DMRGK_CUDA(cudaStreamWaitEvent(r->s2, r->ev_fork, 0));
    // every exit path joins the library-owned streams back into the caller's stream (see dmrgk_heff_apply)
    auto enqueue_chunks = [&]() -> int32_t {
        for (size_t c = 0; c < r->chunks.size(); ++c) {
            const auto& ch = r->chunks[c];
            if (c >= 2) DMRGK_CUDA(cudaStreamWaitEvent(r->s1, r->ev_p2[c & 1], 0));     // T buffer re-use
            DMRGK_TRY(launch_gemm_units(r->kernel, r->units_dev + ch.p1_unit0, r->segs_dev, ch.p1_units, bases, r->s1, r->counters_dev + 2 * c, r->ctx->n_sm, ch.p1_short));
            DMRGK_CUDA(cudaEventRecord(r->ev_p1[c & 1], r->s1));
            DMRGK_CUDA(cudaStreamWaitEvent(r->s2, r->ev_p1[c & 1], 0));
            DMRGK_TRY(launch_gemm_units(r->kernel, r->units_dev + ch.p2_unit0, r->segs_dev, ch.p2_units, bases, r->s2, r->counters_dev + 2 * c + 1, r->ctx->n_sm, ch.p2_short));
            DMRGK_CUDA(cudaEventRecord(r->ev_p2[c & 1], r->s2));
        }
        return DMRGK_OK;
    };
    const int32_t status = enqueue_chunks();
    cudaError_t e = cudaEventRecord(r->ev_join, r->s2);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, r->ev_join, 0);
    if (e == cudaSuccess) e = cudaEventRecord(r->ev_join1, r->s1);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, r->ev_join1, 0);
    if (e != cudaSuccess) {
        cudaStreamSynchronize(r->s1);
        cudaStreamSynchronize(r->s2);
        if (status == DMRGK_OK) return fail(DMRGK_ECUDA, "renorm_apply: join failed: %s", cudaGetErrorString(e));
    }
    return status;
}

}  // extern "C"
