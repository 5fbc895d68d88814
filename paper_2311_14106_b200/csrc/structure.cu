// structure.cu — a1: context, sector spaces, ψ layout, stored operators (
// PAPER.md:142 "Tables": preparing the quantum-number-decomposed matrix and tensor algebra).
// Host bookkeeping only; the block tables are mirrored on the device for the seeded fill kernel.
#include "internal.h"
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <atomic>
#include <new>

namespace dmrgk {

static thread_local char g_err[512] = "";

int32_t fail(int32_t code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

static std::atomic<long long> g_launches{0};
void count_launch(int64_t n) { g_launches.fetch_add((long long)n, std::memory_order_relaxed); }

static int32_t upload_table(const std::vector<Block>& blocks, DevBlock** out) {
    *out = nullptr;
    if (blocks.empty()) return DMRGK_OK;
    std::vector<DevBlock> t(blocks.size());
    for (size_t i = 0; i < blocks.size(); ++i) {
        t[i].off = blocks[i].off;
        t[i].uoff = blocks[i].uoff;
        t[i].rows = blocks[i].rows;
        t[i].cols = blocks[i].cols;
        t[i].ld = blocks[i].ld;
        t[i].rows_pad = blocks[i].rows_pad;
        t[i].pad_ = 0;
        t[i].square_diag = (blocks[i].r_idx == blocks[i].c_idx && blocks[i].rows == blocks[i].cols);
    }
    DMRGK_CUDA(cudaMalloc(out, t.size() * sizeof(DevBlock)));
    DMRGK_CUDA(cudaMemcpy(*out, t.data(), t.size() * sizeof(DevBlock), cudaMemcpyHostToDevice));
    return DMRGK_OK;
}

static void pack_blocks(const std::vector<Block>& blocks, int64_t n_padded, const double* u, double* p) {
    memset(p, 0, size_t(n_padded) * sizeof(double));
    for (const Block& b : blocks)
        for (int r = 0; r < b.rows; ++r)
            for (int c = 0; c < b.cols; ++c)
                p[b.off + panel_off(r, c, b.rows_pad)] = u[b.uoff + int64_t(r) * b.cols + c];
}

}  // namespace dmrgk

using namespace dmrgk;

extern "C" {

const char* dmrgk_last_error(void) { return g_err; }
#ifndef DMRGK_SOURCE_HASH
#define DMRGK_SOURCE_HASH "unstamped"
#endif
const char* dmrgk_version(void) { return "dmrgk 0.2 sm_100a src:" DMRGK_SOURCE_HASH; }
int64_t dmrgk_launch_count(int32_t reset) {
    return reset ? g_launches.exchange(0) : g_launches.load();
}

int32_t dmrgk_ctx_create(int32_t device, dmrgk_ctx** out) {
    if (!out) return fail(DMRGK_EINVAL, "ctx_create: out is NULL");
    *out = nullptr;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0)
        return fail(DMRGK_ECUDA, "ctx_create: no CUDA device (%s); dmrgk has no CPU fallback",
                    e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
    if (device < 0 || device >= n) return fail(DMRGK_EINVAL, "ctx_create: device %d of %d", device, n);
    DMRGK_CUDA(cudaSetDevice(device));
    cudaDeviceProp p;
    DMRGK_CUDA(cudaGetDeviceProperties(&p, device));
    dmrgk_ctx* c = new (std::nothrow) dmrgk_ctx;
    if (!c) return fail(DMRGK_ENOMEM, "ctx_create: out of host memory");
    c->device = device;
    c->n_sm = p.multiProcessorCount;
    c->l2_bytes = p.l2CacheSize;
    c->hbm_bytes = int64_t(p.totalGlobalMem);
    c->smem_optin = int(p.sharedMemPerBlockOptin);
    int32_t s = gemm_kernel_setup();
    if (s != DMRGK_OK) {
        delete c;
        return s;
    }
    *out = c;
    return DMRGK_OK;
}

void dmrgk_ctx_destroy(dmrgk_ctx* ctx) { delete ctx; }

int32_t dmrgk_ctx_query(const dmrgk_ctx* ctx, int32_t* n_sm, int64_t* l2_bytes, int64_t* hbm_bytes) {
    if (!ctx) return fail(DMRGK_EINVAL, "ctx_query: ctx is NULL");
    if (n_sm) *n_sm = ctx->n_sm;
    if (l2_bytes) *l2_bytes = ctx->l2_bytes;
    if (hbm_bytes) *hbm_bytes = ctx->hbm_bytes;
    return DMRGK_OK;
}

int32_t dmrgk_space_create(dmrgk_ctx* ctx, int32_t n_charges, int32_t n_sectors,
                           const int32_t* charges, const int32_t* dims, dmrgk_space** out) {
    if (!out) return fail(DMRGK_EINVAL, "space_create: out is NULL");
    *out = nullptr;
    if (!ctx) return fail(DMRGK_EINVAL, "space_create: ctx is NULL");
    if (n_charges < 1 || n_charges > 2)
        return fail(DMRGK_EINVAL, "space_create: n_charges must be 1 or 2, got %d", n_charges);
    if (n_sectors < 0 || (n_sectors > 0 && (!charges || !dims)))
        return fail(DMRGK_EINVAL, "space_create: bad sector arrays");
    dmrgk_space* s = new (std::nothrow) dmrgk_space;
    if (!s) return fail(DMRGK_ENOMEM, "space_create: out of host memory");
    s->ctx = ctx;
    s->n_charges = n_charges;
    s->q.resize(size_t(n_sectors) * 2);
    s->dim.resize(n_sectors);
    for (int i = 0; i < n_sectors; ++i) {
        int32_t a = charges[i * n_charges], b = n_charges == 2 ? charges[i * 2 + 1] : 0;
        if (dims[i] < 0) {
            delete s;
            return fail(DMRGK_EINVAL, "space_create: negative dimension in sector %d", i);
        }
        if (!s->index.emplace(dmrgk_space::key(a, b), i).second) {
            delete s;
            return fail(DMRGK_EINVAL, "space_create: duplicate charge in sector %d", i);
        }
        s->q[2 * i] = a;
        s->q[2 * i + 1] = b;
        s->dim[i] = dims[i];
    }
    *out = s;
    return DMRGK_OK;
}

void dmrgk_space_destroy(dmrgk_space* s) { delete s; }

int32_t dmrgk_layout_create(dmrgk_ctx* ctx, const dmrgk_space* A, const dmrgk_space* B,
                            const int32_t* target, dmrgk_layout** out) {
    if (!out) return fail(DMRGK_EINVAL, "layout_create: out is NULL");
    *out = nullptr;
    if (!ctx || !A || !B || !target) return fail(DMRGK_EINVAL, "layout_create: NULL argument");
    if (A->n_charges != B->n_charges)
        return fail(DMRGK_ESHAPE, "layout_create: A has %d charges, B has %d", A->n_charges, B->n_charges);
    dmrgk_layout* l = new (std::nothrow) dmrgk_layout;
    if (!l) return fail(DMRGK_ENOMEM, "layout_create: out of host memory");
    l->ctx = ctx;
    l->A = A;
    l->B = B;
    l->target[0] = target[0];
    l->target[1] = A->n_charges == 2 ? target[1] : 0;
    l->by_a.assign(A->n(), -1);
    int64_t off = 0, uoff = 0;
    for (int a = 0; a < A->n(); ++a) {
        int b = B->find(l->target[0] - A->q[2 * a], l->target[1] - A->q[2 * a + 1]);
        if (b < 0 || A->dim[a] == 0 || B->dim[b] == 0) continue;
        Block k;
        k.r_idx = a;
        k.c_idx = b;
        k.rows = A->dim[a];
        k.cols = B->dim[b];
        k.ld = int32_t(round_up(k.cols, LD_PAD));
        k.rows_pad = pad_rows(k.rows);
        k.off = off;
        k.uoff = uoff;
        off += k.size();
        uoff += int64_t(k.rows) * k.cols;
        l->by_a[a] = int32_t(l->blocks.size());
        l->blocks.push_back(k);
    }
    l->n_elems = uoff;
    l->n_padded = off;
    int32_t s = upload_table(l->blocks, &l->dev_table);
    if (s != DMRGK_OK) {
        delete l;
        return s;
    }
    *out = l;
    return DMRGK_OK;
}

void dmrgk_layout_destroy(dmrgk_layout* l) {
    if (!l) return;
    if (l->dev_table) cudaFree(l->dev_table);
    delete l;
}

int32_t dmrgk_layout_query(const dmrgk_layout* l, int64_t* n_blocks, int64_t* n_elems, int64_t* n_padded) {
    if (!l) return fail(DMRGK_EINVAL, "layout_query: layout is NULL");
    if (n_blocks) *n_blocks = int64_t(l->blocks.size());
    if (n_elems) *n_elems = l->n_elems;
    if (n_padded) *n_padded = l->n_padded;
    return DMRGK_OK;
}

static void copy_table(const std::vector<Block>& bl, int32_t* r, int32_t* c, int32_t* rows, int32_t* cols,
                       int32_t* ld, int64_t* off) {
    for (size_t i = 0; i < bl.size(); ++i) {
        if (r) r[i] = bl[i].r_idx;
        if (c) c[i] = bl[i].c_idx;
        if (rows) rows[i] = bl[i].rows;
        if (cols) cols[i] = bl[i].cols;
        if (ld) ld[i] = bl[i].ld;
        if (off) off[i] = bl[i].off;
    }
}

int32_t dmrgk_layout_blocks(const dmrgk_layout* l, int32_t* a_idx, int32_t* b_idx, int32_t* rows,
                            int32_t* cols, int32_t* ld, int64_t* offset) {
    if (!l) return fail(DMRGK_EINVAL, "layout_blocks: layout is NULL");
    copy_table(l->blocks, a_idx, b_idx, rows, cols, ld, offset);
    return DMRGK_OK;
}

int32_t dmrgk_layout_pack(const dmrgk_layout* l, const double* u, double* p) {
    if (!l || (l->n_padded && (!u || !p))) return fail(DMRGK_EINVAL, "layout_pack: NULL argument");
    pack_blocks(l->blocks, l->n_padded, u, p);
    return DMRGK_OK;
}

int32_t dmrgk_layout_unpack(const dmrgk_layout* l, const double* p, double* u) {
    if (!l || (l->n_padded && (!u || !p))) return fail(DMRGK_EINVAL, "layout_unpack: NULL argument");
    for (const Block& b : l->blocks)
        for (int r = 0; r < b.rows; ++r)
            for (int c = 0; c < b.cols; ++c)
                u[b.uoff + int64_t(r) * b.cols + c] = p[b.off + panel_off(r, c, b.rows_pad)];
    return DMRGK_OK;
}

int32_t dmrgk_op_create(dmrgk_ctx* ctx, const dmrgk_space* space, const int32_t* dq, int32_t parity,
                        dmrgk_op** out) {
    if (!out) return fail(DMRGK_EINVAL, "op_create: out is NULL");
    *out = nullptr;
    if (!ctx || !space || !dq) return fail(DMRGK_EINVAL, "op_create: NULL argument");
    if (parity != 0 && parity != 1) return fail(DMRGK_EINVAL, "op_create: parity must be 0 or 1");
    dmrgk_op* op = new (std::nothrow) dmrgk_op;
    if (!op) return fail(DMRGK_ENOMEM, "op_create: out of host memory");
    op->ctx = ctx;
    op->space = space;
    op->dq[0] = dq[0];
    op->dq[1] = space->n_charges == 2 ? dq[1] : 0;
    op->parity = parity;
    op->by_col.assign(space->n(), -1);
    op->by_row.assign(space->n(), -1);
    int64_t off = 0, uoff = 0;
    for (int c = 0; c < space->n(); ++c) {
        int r = space->find(space->q[2 * c] + op->dq[0], space->q[2 * c + 1] + op->dq[1]);
        if (r < 0 || space->dim[c] == 0 || space->dim[r] == 0) continue;
        Block k;
        k.r_idx = r;
        k.c_idx = c;
        k.rows = space->dim[r];
        k.cols = space->dim[c];
        k.ld = int32_t(round_up(k.cols, LD_PAD));
        k.rows_pad = pad_rows(k.rows);
        k.off = off;
        k.uoff = uoff;
        off += k.size();
        uoff += int64_t(k.rows) * k.cols;
        op->by_col[c] = op->by_row[r] = int32_t(op->blocks.size());
        op->blocks.push_back(k);
    }
    op->n_elems = uoff;
    op->n_padded = off;
    int32_t s = upload_table(op->blocks, &op->dev_table);
    if (s != DMRGK_OK) {
        delete op;
        return s;
    }
    *out = op;
    return DMRGK_OK;
}

void dmrgk_op_destroy(dmrgk_op* op) {
    if (!op) return;
    if (op->dev_table) cudaFree(op->dev_table);
    delete op;
}

int32_t dmrgk_op_query(const dmrgk_op* op, int64_t* n_blocks, int64_t* n_elems, int64_t* n_padded) {
    if (!op) return fail(DMRGK_EINVAL, "op_query: op is NULL");
    if (n_blocks) *n_blocks = int64_t(op->blocks.size());
    if (n_elems) *n_elems = op->n_elems;
    if (n_padded) *n_padded = op->n_padded;
    return DMRGK_OK;
}

int32_t dmrgk_op_blocks(const dmrgk_op* op, int32_t* row_idx, int32_t* col_idx, int32_t* rows,
                        int32_t* cols, int32_t* ld, int64_t* offset) {
    if (!op) return fail(DMRGK_EINVAL, "op_blocks: op is NULL");
    copy_table(op->blocks, row_idx, col_idx, rows, cols, ld, offset);
    return DMRGK_OK;
}

int32_t dmrgk_op_pack(const dmrgk_op* op, const double* u, double* p) {
    if (!op || (op->n_padded && (!u || !p))) return fail(DMRGK_EINVAL, "op_pack: NULL argument");
    pack_blocks(op->blocks, op->n_padded, u, p);
    return DMRGK_OK;
}

int32_t dmrgk_op_unpack(const dmrgk_op* op, const double* p, double* u) {
    if (!op || (op->n_padded && (!u || !p))) return fail(DMRGK_EINVAL, "op_unpack: NULL argument");
    for (const Block& b : op->blocks)
        for (int r = 0; r < b.rows; ++r)
            for (int c = 0; c < b.cols; ++c)
                u[b.uoff + int64_t(r) * b.cols + c] = p[b.off + panel_off(r, c, b.rows_pad)];
    return DMRGK_OK;
}

int64_t dmrgk_block_size(int32_t rows, int32_t cols) {
    if (rows < 0 || cols < 0) return 0;
    return int64_t(pad_rows(rows)) * round_up(cols, LD_PAD);
}

int32_t dmrgk_block_unpack(int32_t rows, int32_t cols, const double* packed_host, double* dense_host) {
    if (rows < 0 || cols < 0 || ((rows && cols) && (!packed_host || !dense_host)))
        return fail(DMRGK_EINVAL, "block_unpack: bad argument");
    const int rp = pad_rows(rows);
    for (int r = 0; r < rows; ++r)
        for (int c = 0; c < cols; ++c) dense_host[int64_t(r) * cols + c] = packed_host[panel_off(r, c, rp)];
    return DMRGK_OK;
}

int32_t dmrgk_block_padding_is_zero(int32_t rows, int32_t cols, const double* packed_host) {
    if (rows < 0 || cols < 0 || ((rows && cols) && !packed_host)) return fail(DMRGK_EINVAL, "block_padding_is_zero: bad argument");
    const int rp = pad_rows(rows), ld = int(round_up(cols, LD_PAD));
    for (int r = 0; r < rp; ++r)
        for (int c = 0; c < ld; ++c)
            if ((r >= rows || c >= cols) && packed_host[panel_off(r, c, rp)] != 0.0) return 1;
    return DMRGK_OK;
}

int32_t dmrgk_op_bind_device(dmrgk_op* op, const double* arena_dev) {
    if (!op) return fail(DMRGK_EINVAL, "op_bind_device: op is NULL");
    if (op->n_padded && !arena_dev) return fail(DMRGK_EINVAL, "op_bind_device: arena is NULL");
    if (!aligned128(arena_dev)) return fail(DMRGK_EALIGN, "op_bind_device: arena %p not 128-byte aligned", (const void*)arena_dev);
    op->dev = arena_dev;
    op->pinned = nullptr;
    return DMRGK_OK;
}

int32_t dmrgk_op_bind_pinned(dmrgk_op* op, const double* arena_pinned_host) {
    if (!op) return fail(DMRGK_EINVAL, "op_bind_pinned: op is NULL");
    if (op->n_padded && !arena_pinned_host) return fail(DMRGK_EINVAL, "op_bind_pinned: arena is NULL");
    op->pinned = arena_pinned_host;
    op->dev = nullptr;
    return DMRGK_OK;
}

// ---- Φ: kept basis of one half (renormalisation) ----------------------------
int32_t dmrgk_iso_create(dmrgk_ctx* ctx, const dmrgk_space* enlarged, const dmrgk_space* kept, dmrgk_iso** out) {
    if (!out) return fail(DMRGK_EINVAL, "iso_create: out is NULL");
    *out = nullptr;
    if (!ctx || !enlarged || !kept) return fail(DMRGK_EINVAL, "iso_create: NULL argument");
    if (enlarged->n_charges != kept->n_charges)
        return fail(DMRGK_ESHAPE, "iso_create: the two spaces have different numbers of charges");
    dmrgk_iso* p = new (std::nothrow) dmrgk_iso;
    if (!p) return fail(DMRGK_ENOMEM, "iso_create: out of host memory");
    p->ctx = ctx;
    p->enl = enlarged;
    p->kept = kept;
    p->by_enl.assign(enlarged->n(), -1);
    // every kept sector that holds states needs its enlarged counterpart: otherwise the renormalised
    // blocks on that sector would have no producer and would silently keep stale values
    for (int k = 0; k < kept->n(); ++k) {
        if (kept->dim[k] == 0) continue;
        const int e = enlarged->find(kept->q[2 * k], kept->q[2 * k + 1]);
        if (e < 0 || enlarged->dim[e] == 0) {
            delete p;
            return fail(DMRGK_ESHAPE, "iso_create: kept sector %d (charge %d,%d; %d states) has no enlarged sector", k,
                        kept->q[2 * k], kept->q[2 * k + 1], kept->dim[k]);
        }
    }
    int64_t off = 0, uoff = 0;
    for (int e = 0; e < enlarged->n(); ++e) {
        const int k = kept->find(enlarged->q[2 * e], enlarged->q[2 * e + 1]);
        if (k < 0 || enlarged->dim[e] == 0 || kept->dim[k] == 0) continue;
        if (kept->dim[k] > enlarged->dim[e]) {
            delete p;
            return fail(DMRGK_ESHAPE, "iso_create: kept sector %d holds %d states, its enlarged sector only %d", k,
                        kept->dim[k], enlarged->dim[e]);
        }
        Block b;
        b.r_idx = e;
        b.c_idx = k;
        b.rows = enlarged->dim[e];
        b.cols = kept->dim[k];
        b.ld = int32_t(round_up(b.cols, LD_PAD));
        b.rows_pad = pad_rows(b.rows);
        b.off = off;
        b.uoff = uoff;
        off += b.size();
        uoff += int64_t(b.rows) * b.cols;
        p->by_enl[e] = int32_t(p->blocks.size());
        p->blocks.push_back(b);
    }
    p->n_elems = uoff;
    p->n_padded = off;
    int32_t s = upload_table(p->blocks, &p->dev_table);
    if (s != DMRGK_OK) {
        delete p;
        return s;
    }
    *out = p;
    return DMRGK_OK;
}

void dmrgk_iso_destroy(dmrgk_iso* phi) {
    if (!phi) return;
    if (phi->dev_table) cudaFree(phi->dev_table);
    delete phi;
}

int32_t dmrgk_iso_query(const dmrgk_iso* phi, int64_t* n_blocks, int64_t* n_elems, int64_t* n_padded) {
    if (!phi) return fail(DMRGK_EINVAL, "iso_query: phi is NULL");
    if (n_blocks) *n_blocks = int64_t(phi->blocks.size());
    if (n_elems) *n_elems = phi->n_elems;
    if (n_padded) *n_padded = phi->n_padded;
    return DMRGK_OK;
}

int32_t dmrgk_iso_blocks(const dmrgk_iso* phi, int32_t* enl_idx, int32_t* new_idx, int32_t* rows, int32_t* cols,
                         int32_t* ld, int64_t* offset) {
    if (!phi) return fail(DMRGK_EINVAL, "iso_blocks: phi is NULL");
    copy_table(phi->blocks, enl_idx, new_idx, rows, cols, ld, offset);
    return DMRGK_OK;
}

int32_t dmrgk_iso_pack(const dmrgk_iso* phi, const double* u, double* p) {
    if (!phi || (phi->n_padded && (!u || !p))) return fail(DMRGK_EINVAL, "iso_pack: NULL argument");
    pack_blocks(phi->blocks, phi->n_padded, u, p);
    return DMRGK_OK;
}

int32_t dmrgk_iso_bind_device(dmrgk_iso* phi, const double* arena_dev) {
    if (!phi) return fail(DMRGK_EINVAL, "iso_bind_device: phi is NULL");
    if (phi->n_padded && !arena_dev) return fail(DMRGK_EINVAL, "iso_bind_device: arena is NULL");
    if (!aligned128(arena_dev)) return fail(DMRGK_EALIGN, "iso_bind_device: arena %p not 128-byte aligned", (const void*)arena_dev);
    phi->dev = arena_dev;
    return DMRGK_OK;
}

}  // extern "C"
