// enlarge.cu — the block-enlargement half of the renormalisation step (
// PAPER.md:60 §II.A "renormalized block operators", Fig. 7 "Ren_l"):
//
//        O_{A′} = Σ_j coef_j · (X_j · P^{π_j}) ⊗ y_j
//
// X_j: a stored operator on the KEPT space (or the identity, or the transpose of a stored operator),
// y_j: a d×d site operator, P = (−1)^{N} on the kept column index, π_j = 1 for a fermionic site factor.
// The enlarged space A′ = kept ⊗ site is sector-major; inside an enlarged sector q′ the states are ordered
// by kept sector (in the kept space's order), each kept sector k appearing with the one site state σ of
// charge q′ − q_k.  An enlarged block (q′_r, q′_c) is therefore a grid of sub-blocks (k_r σ_r | k_c σ_c), and
//
//        sub-block = Σ_j coef_j · y_j[σ_r, σ_c] · (−1)^{π_j N(q_{k_c})} · X_j[k_r, k_c] .
//
// The host groups the contributions by DESTINATION sub-block (no atomics, bit-reproducible); the kernel
// is a scaled gather: each CTA owns a 32×32 tile of one sub-block, sums its sources in list order and
// writes the tile once.  HBM-bound: bytes = 8·(Σ source elements + destination elements).
#include "internal.h"
#include <algorithm>
#include <cstring>
#include <map>
#include <new>
#include <tuple>

using namespace dmrgk;

namespace dmrgk {

enum : uint32_t { ESRC_TRANS = 1u, ESRC_IDENT = 2u };
struct ESrc {
    unsigned long long X;   // absolute address of the source block origin (panel layout); 0 for the identity
    double scale;
    int32_t rp;             // rows_pad of the source block
    uint32_t flags;
    int32_t pad_[2];
};  // 32 B
struct EUnit {
    unsigned long long C;   // absolute address of the destination block origin
    int32_t c_rp;           // rows_pad of the destination block
    int32_t r0, c0;         // tile origin inside the destination block
    int32_t rows, cols;     // tile extent (≤ 32 × ≤ 32)
    int32_t sr0, sc0;       // tile origin inside the sub-block (= inside every source block)
    int32_t src_begin, src_end;
    int32_t pad_;
};  // 48 B

__global__ void __launch_bounds__(256)
enlarge_gather_kernel(const EUnit* __restrict__ units, const ESrc* __restrict__ srcs) {
    __shared__ double tile[32][33];
    const EUnit u = units[blockIdx.x];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;      // 8 rows of 32 lanes; thread owns rows ty + 8q
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int s = u.src_begin; s < u.src_end; ++s) {
        const ESrc sc = srcs[s];
        if (sc.flags & ESRC_IDENT) {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (u.sr0 + ty + 8 * q == u.sc0 + tx) acc[q] += sc.scale;
        } else if (!(sc.flags & ESRC_TRANS)) {
            const double* X = reinterpret_cast<const double*>(sc.X);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = ty + 8 * q;
                if (i < u.rows && tx < u.cols) acc[q] = fma(sc.scale, X[panel_off(u.sr0 + i, u.sc0 + tx, sc.rp)], acc[q]);
            }
        } else {
            // destination (i, j) takes source (sc0 + j, sr0 + i): read the source tile row by row
            // (coalesced), turn it in shared memory
            const double* X = reinterpret_cast<const double*>(sc.X);
            __syncthreads();
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int jj = ty + 8 * q;                      // source row ↔ destination column
                tile[jj][tx] = (jj < u.cols && tx < u.rows) ? X[panel_off(u.sc0 + jj, u.sr0 + tx, sc.rp)] : 0.0;
            }
            __syncthreads();
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[q] = fma(sc.scale, tile[tx][ty + 8 * q], acc[q]);
        }
    }
    double* C = reinterpret_cast<double*>(u.C);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int i = ty + 8 * q;
        if (i < u.rows && tx < u.cols) C[panel_off(u.r0 + i, u.c0 + tx, u.c_rp)] = acc[q];
    }
}

}  // namespace dmrgk

struct dmrgk_enlarge {
    dmrgk_ctx* ctx;
    std::vector<std::pair<double*, int64_t>> zero;   // destination arenas (pointer, doubles) to clear
    EUnit* units_dev = nullptr;
    ESrc* srcs_dev = nullptr;
    int64_t n_units = 0, n_srcs = 0, bytes_read = 0, bytes_written = 0;
};

extern "C" {

void dmrgk_enlarge_destroy(dmrgk_enlarge* e) {
    if (!e) return;
    cudaFree(e->units_dev);
    cudaFree(e->srcs_dev);
    delete e;
}

int32_t dmrgk_enlarge_create(dmrgk_ctx* ctx, const dmrgk_space* kept, const dmrgk_space* enlarged, int32_t d,
                             const int32_t* site_charges, int32_t site_major, int64_t n_out, dmrgk_op* const* out, int64_t n_terms,
                             const int32_t* t_out, dmrgk_op* const* t_x, const uint32_t* t_flags,
                             const double* t_coef, const double* t_y, dmrgk_enlarge** plan) {
    if (!plan) return fail(DMRGK_EINVAL, "enlarge_create: plan is NULL");
    *plan = nullptr;
    if (!ctx || !kept || !enlarged || !site_charges || d < 1 || d > 16 || (site_major != 0 && site_major != 1))
        return fail(DMRGK_EINVAL, "enlarge_create: bad argument (d must be 1..16, site_major 0 or 1)");
    if (n_out < 0 || n_terms < 0 || (n_out && !out) || (n_terms && (!t_out || !t_x || !t_flags || !t_coef || !t_y)))
        return fail(DMRGK_EINVAL, "enlarge_create: bad arrays");
    if (kept->n_charges != enlarged->n_charges) return fail(DMRGK_ESHAPE, "enlarge_create: spaces differ in the number of charges");
    const int nc = kept->n_charges;
    auto sq = [&](int s, int c) { return c < nc ? site_charges[s * nc + c] : 0; };
    for (int a = 0; a < d; ++a)
        for (int b = a + 1; b < d; ++b)
            if (sq(a, 0) == sq(b, 0) && sq(a, 1) == sq(b, 1))
                return fail(DMRGK_EINVAL, "enlarge_create: site states %d and %d have the same charge", a, b);
    // ---- structure of the enlarged space: for (enlarged sector e, site state σ) the kept sector and the
    //      offset of its states inside e (kept sectors in kept order) ----
    const int nE = enlarged->n();
    std::vector<int32_t> sub_k(size_t(nE) * d, -1), sub_off(size_t(nE) * d, 0);
    for (int e = 0; e < nE; ++e) {
        std::vector<std::pair<int, int>> parts;      // (kept sector, site state)
        for (int s = 0; s < d; ++s) {
            const int k = kept->find(enlarged->q[2 * e] - sq(s, 0), enlarged->q[2 * e + 1] - sq(s, 1));
            if (k >= 0 && kept->dim[k] > 0) parts.push_back({k, s});
        }
        // left block (kept ⊗ site): by kept sector; right block (site ⊗ kept): by site state
        std::sort(parts.begin(), parts.end(), [&](const std::pair<int, int>& a, const std::pair<int, int>& b) {
            return site_major ? std::make_pair(a.second, a.first) < std::make_pair(b.second, b.first) : a < b;
        });
        int off = 0;
        for (auto& p : parts) {
            sub_k[size_t(e) * d + p.second] = p.first;
            sub_off[size_t(e) * d + p.second] = off;
            off += kept->dim[p.first];
        }
        if (off != enlarged->dim[e])
            return fail(DMRGK_ESHAPE, "enlarge_create: enlarged sector %d has %d states, kept ⊗ site gives %d", e, enlarged->dim[e], off);
    }
    for (int64_t i = 0; i < n_out; ++i) {
        if (!out[i] || out[i]->space != enlarged) return fail(DMRGK_ESHAPE, "enlarge_create: out[%lld] is not on the enlarged space", (long long)i);
        if (out[i]->n_padded && !out[i]->dev) return fail(DMRGK_ESTATE, "enlarge_create: out[%lld] is not bound to a device arena", (long long)i);
    }
    // ---- contributions, grouped by destination sub-block ----
    struct Dest {
        int64_t o;
        int32_t blk, sr, sc;
        bool operator<(const Dest& b) const { return std::tie(o, blk, sr, sc) < std::tie(b.o, b.blk, b.sr, b.sc); }
    };
    std::map<Dest, std::vector<ESrc>> groups;
    for (int64_t j = 0; j < n_terms; ++j) {
        const int64_t o = t_out[j];
        if (o < 0 || o >= n_out) return fail(DMRGK_EINVAL, "enlarge_create: term %lld targets operator %lld", (long long)j, (long long)o);
        const dmrgk_op* X = t_x[j];
        const uint32_t f = t_flags[j];
        if (f & ~7u) return fail(DMRGK_EINVAL, "enlarge_create: term %lld has unknown flag bits", (long long)j);
        if ((f & 2u) && site_major) return fail(DMRGK_EINVAL, "enlarge_create: term %lld: the kept-parity flag belongs to the left block form", (long long)j);
        const bool trans = (f & 1u) != 0, kept_sign = (f & 2u) != 0, site_odd = (f & 6u) != 0;
        if (X) {
            if (X->space != kept) return fail(DMRGK_ESHAPE, "enlarge_create: term %lld: X is not on the kept space", (long long)j);
            if (X->n_padded && !X->dev) return fail(DMRGK_ESTATE, "enlarge_create: term %lld: X is not bound to a device arena", (long long)j);
            if (out[o]->parity != (X->parity ^ int(site_odd)))
                return fail(DMRGK_ECHARGE, "enlarge_create: term %lld: parity of out ≠ parity(X) xor parity(site factor)", (long long)j);
        } else if (out[o]->parity != int(site_odd)) {
            return fail(DMRGK_ECHARGE, "enlarge_create: term %lld: parity of out ≠ parity of the site factor", (long long)j);
        }
        int dx[2] = {0, 0};
        if (X) for (int c = 0; c < 2; ++c) dx[c] = trans ? -X->dq[c] : X->dq[c];
        for (int sr = 0; sr < d; ++sr)
            for (int sc = 0; sc < d; ++sc) {
                const double yv = t_y[(size_t(j) * d + sr) * d + sc];
                if (yv == 0.0) continue;
                if (out[o]->dq[0] != dx[0] + sq(sr, 0) - sq(sc, 0) || out[o]->dq[1] != dx[1] + sq(sr, 1) - sq(sc, 1))
                    return fail(DMRGK_ECHARGE, "enlarge_create: term %lld: shift of X plus the site entry (%d,%d) is not the shift of out", (long long)j, sr, sc);
                for (size_t b = 0; b < out[o]->blocks.size(); ++b) {
                    const Block& ob = out[o]->blocks[b];
                    const int kr = sub_k[size_t(ob.r_idx) * d + sr], kc = sub_k[size_t(ob.c_idx) * d + sc];
                    if (kr < 0 || kc < 0) continue;
                    ESrc s;
                    memset(&s, 0, sizeof(s));
                    const double sign = (kept_sign && kept->parity(kc)) ? -1.0 : 1.0;
                    s.scale = t_coef[j] * yv * sign;
                    if (!X) {
                        if (kr != kc) continue;
                        s.flags = ESRC_IDENT;
                    } else {
                        const int bi = trans ? X->by_col[kr] : X->by_col[kc];
                        if (bi < 0) continue;
                        const Block& xb = X->blocks[bi];
                        if (xb.r_idx != (trans ? kc : kr)) continue;
                        s.X = (unsigned long long)(uintptr_t)(X->dev + xb.off);
                        s.rp = xb.rows_pad;
                        s.flags = trans ? ESRC_TRANS : 0u;
                    }
                    groups[Dest{o, int32_t(b), sr, sc}].push_back(s);
                }
            }
    }
    dmrgk_enlarge* e = new (std::nothrow) dmrgk_enlarge;
    if (!e) return fail(DMRGK_ENOMEM, "enlarge_create: out of host memory");
    e->ctx = ctx;
    for (int64_t i = 0; i < n_out; ++i)
        if (out[i]->n_padded) e->zero.push_back({const_cast<double*>(out[i]->dev), out[i]->n_padded});
    // destination arenas are usually slices of one allocation: clear contiguous ranges with ONE memset each
    // (a memset per operator is 137 launches on the config-4 enlargement: 5.5 → 5.0 ms per step)
    std::sort(e->zero.begin(), e->zero.end());
    {
        std::vector<std::pair<double*, int64_t>> merged;
        for (const auto& z : e->zero) {
            if (!merged.empty() && z.first <= merged.back().first + merged.back().second)      // adjacent or overlapping only
                merged.back().second = std::max(merged.back().second, int64_t(z.first - merged.back().first) + z.second);
            else
                merged.push_back(z);
        }
        e->zero.swap(merged);
    }
    std::vector<EUnit> units;
    std::vector<ESrc> srcs;
    for (auto& kv : groups) {
        const Dest& dst = kv.first;
        const dmrgk_op* O = out[dst.o];
        const Block& ob = O->blocks[dst.blk];
        const int kr = sub_k[size_t(ob.r_idx) * d + dst.sr], kc = sub_k[size_t(ob.c_idx) * d + dst.sc];
        const int rows = kept->dim[kr], cols = kept->dim[kc];
        const int roff = sub_off[size_t(ob.r_idx) * d + dst.sr], coff = sub_off[size_t(ob.c_idx) * d + dst.sc];
        const int32_t sb = int32_t(srcs.size());
        srcs.insert(srcs.end(), kv.second.begin(), kv.second.end());
        const int32_t se = int32_t(srcs.size());
        for (const ESrc& s : kv.second) e->bytes_read += (s.flags & ESRC_IDENT) ? 0 : int64_t(8) * rows * cols;
        e->bytes_written += int64_t(8) * rows * cols;
        for (int i0 = 0; i0 < rows; i0 += 32)
            for (int j0 = 0; j0 < cols; j0 += 32) {
                EUnit u;
                memset(&u, 0, sizeof(u));
                u.C = (unsigned long long)(uintptr_t)(O->dev + ob.off);
                u.c_rp = ob.rows_pad;
                u.r0 = roff + i0;
                u.c0 = coff + j0;
                u.rows = std::min(32, rows - i0);
                u.cols = std::min(32, cols - j0);
                u.sr0 = i0;
                u.sc0 = j0;
                u.src_begin = sb;
                u.src_end = se;
                units.push_back(u);
            }
    }
    e->n_units = int64_t(units.size());
    e->n_srcs = int64_t(srcs.size());
    if (e->n_units > 0x7fffffffLL) {
        dmrgk_enlarge_destroy(e);
        return fail(DMRGK_EINVAL, "enlarge_create: too many tiles");
    }
    cudaError_t err = cudaSuccess;
    if (!units.empty()) {
        err = cudaMalloc(&e->units_dev, units.size() * sizeof(EUnit));
        if (err == cudaSuccess) err = cudaMemcpy(e->units_dev, units.data(), units.size() * sizeof(EUnit), cudaMemcpyHostToDevice);
        if (err == cudaSuccess) err = cudaMalloc(&e->srcs_dev, srcs.size() * sizeof(ESrc));
        if (err == cudaSuccess) err = cudaMemcpy(e->srcs_dev, srcs.data(), srcs.size() * sizeof(ESrc), cudaMemcpyHostToDevice);
    }
    if (err != cudaSuccess) {
        dmrgk_enlarge_destroy(e);
        return fail(DMRGK_ECUDA, "enlarge_create: metadata upload: %s", cudaGetErrorString(err));
    }
    *plan = e;
    return DMRGK_OK;
}

int32_t dmrgk_enlarge_query(const dmrgk_enlarge* e, int64_t* n_tiles, int64_t* n_sources, int64_t* bytes_read,
                            int64_t* bytes_written) {
    if (!e) return fail(DMRGK_EINVAL, "enlarge_query: plan is NULL");
    if (n_tiles) *n_tiles = e->n_units;
    if (n_sources) *n_sources = e->n_srcs;
    if (bytes_read) *bytes_read = e->bytes_read;
    if (bytes_written) *bytes_written = e->bytes_written;
    return DMRGK_OK;
}

int32_t dmrgk_enlarge_apply(dmrgk_enlarge* e, void* stream) {
    if (!e) return fail(DMRGK_EINVAL, "enlarge_apply: plan is NULL");
    DMRGK_CUDA(cudaSetDevice(e->ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    for (auto& z : e->zero) DMRGK_CUDA(cudaMemsetAsync(z.first, 0, size_t(z.second) * 8, st));
    if (e->n_units) {
        enlarge_gather_kernel<<<unsigned(e->n_units), 256, 0, st>>>(e->units_dev, e->srcs_dev);
        count_launch();
        DMRGK_CUDA(cudaGetLastError());
    }
    return DMRGK_OK;
}

}  // extern "C"
