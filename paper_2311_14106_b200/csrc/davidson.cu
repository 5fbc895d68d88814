// davidson.cu — a8 + a9: the Davidson iteration around σ = H_eff ψ (§II.A "iterative
// diagonalization of the effective Hamiltonian … Lánczos or Davidson"; ε_Davidson of PAPER.md:114,
// 118 read as the residual 2-norm; SURVEY.md §8(c) "Davidson, step by step").
//
//   V=[x0/‖x0‖]; W=[H V0]; m=1
//   step:  G=(VᵀW + WᵀV)/2 ; (θ,y) = lowest eigenpair of G (host, cyclic Jacobi, m ≤ 63)
//          r = W y − θ V y ; ρ = ‖r‖ ; ρ ≤ tol → converged
//          m == m_max → collapse: V=[V y], W=[W y]
//          t = r/(θ − d) guarded ; t ← t − V(Vᵀt) twice ; v = t/‖t‖ ; w = H v ; append
//
// Everything ψ-sized stays on the device; only the Rayleigh matrix entries (2(m+1) doubles), ‖r‖²,
// ‖t‖² come back and (y, θ) go up per step — two host synchronisations per step: after the residual (the
// convergence decision precedes the expensive apply) and after the Rayleigh entries.  G is kept on the host and extended by one row and
// column per step: its entries v_i·w_j never change while the basis is only appended to.
#include "internal.h"
#include <cmath>
#include <cstring>
#include <new>

using namespace dmrgk;

struct dmrgk_davidson {
    dmrgk_heff* h;
    dmrgk_ctx* ctx;
    int64_t n;
    int m_max, max_iter;
    double tol;
    double *V, *W;
    const double* diag;
    void* ws;
    cudaStream_t main, copy;
    // extra region
    double *r, *t, *u, *coef, *out;
    void* scratch;
    double* host;                 // pinned: [0..64) coef staging, [64..192) dot results
    std::vector<double> G;        // m_max × m_max, G[i·m_max + j] = v_i · w_j
    std::vector<double> y;
    int m = 0, n_apply = 0;
    bool started = false, converged = false;
    double theta = 0.0, rho = 0.0;
    dmrgk_allreduce_fn reduce = nullptr;   // k-sharding hook: makes W_j the sum over all ranks
    void* reduce_user = nullptr;
};

namespace {

// Lowest eigenpair of the symmetric m×m matrix A (row-major, destroyed) by cyclic Jacobi rotations.
void jacobi_lowest(std::vector<double>& A, int m, double* theta, std::vector<double>& y) {
    std::vector<double> Q(size_t(m) * m, 0.0);
    for (int i = 0; i < m; ++i) Q[size_t(i) * m + i] = 1.0;
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = 0.0, dg = 0.0;
        for (int i = 0; i < m; ++i)
            for (int j = 0; j < m; ++j) (i == j ? dg : off) += A[size_t(i) * m + j] * A[size_t(i) * m + j];
        if (off <= 1e-34 * (dg + off) || off == 0.0) break;
        for (int p = 0; p < m - 1; ++p)
            for (int q = p + 1; q < m; ++q) {
                const double apq = A[size_t(p) * m + q];
                if (apq == 0.0) continue;
                const double app = A[size_t(p) * m + p], aqq = A[size_t(q) * m + q];
                const double tau = (aqq - app) / (2.0 * apq);
                const double tt = (tau >= 0.0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
                const double c = 1.0 / std::sqrt(1.0 + tt * tt), s = tt * c;
                for (int k = 0; k < m; ++k) {   // columns p, q
                    const double akp = A[size_t(k) * m + p], akq = A[size_t(k) * m + q];
                    A[size_t(k) * m + p] = c * akp - s * akq;
                    A[size_t(k) * m + q] = s * akp + c * akq;
                }
                for (int k = 0; k < m; ++k) {   // rows p, q
                    const double apk = A[size_t(p) * m + k], aqk = A[size_t(q) * m + k];
                    A[size_t(p) * m + k] = c * apk - s * aqk;
                    A[size_t(q) * m + k] = s * apk + c * aqk;
                }
                for (int k = 0; k < m; ++k) {
                    const double qkp = Q[size_t(k) * m + p], qkq = Q[size_t(k) * m + q];
                    Q[size_t(k) * m + p] = c * qkp - s * qkq;
                    Q[size_t(k) * m + q] = s * qkp + c * qkq;
                }
            }
    }
    int best = 0;
    for (int i = 1; i < m; ++i)
        if (A[size_t(i) * m + i] < A[size_t(best) * m + best]) best = i;
    *theta = A[size_t(best) * m + best];
    y.resize(m);
    double nrm = 0.0;
    for (int k = 0; k < m; ++k) {
        y[k] = Q[size_t(k) * m + best];
        nrm += y[k] * y[k];
    }
    nrm = std::sqrt(nrm);
    for (int k = 0; k < m; ++k) y[k] /= nrm;
}

int32_t read_back(dmrgk_davidson* d, int count) {
    DMRGK_CUDA(cudaMemcpyAsync(d->host + 64, d->out, size_t(count) * 8, cudaMemcpyDeviceToHost, d->main));
    DMRGK_CUDA(cudaStreamSynchronize(d->main));
    return DMRGK_OK;
}

// w = H v on this rank's share of the pair list, then the all-reduce hook (if any) completes it
int32_t apply_h(dmrgk_davidson* d, const double* v, double* w) {
    DMRGK_TRY(dmrgk_heff_apply(d->h, v, w, d->ws, d->main, d->copy));
    if (d->reduce) {
        const int32_t s = d->reduce(w, d->n, (void*)d->main, d->reduce_user);
        if (s != 0) return fail(DMRGK_ESTATE, "davidson: the all-reduce hook failed (%d)", s);
    }
    d->n_apply += 1;
    return DMRGK_OK;
}

// t ← t − V (Vᵀ t), twice (classical Gram–Schmidt with re-orthogonalisation)
int32_t orthogonalise(dmrgk_davidson* d, double* t) {
    for (int pass = 0; pass < 2; ++pass) {
        DMRGK_TRY(dmrgk_vec_multi_dot(d->ctx, d->n, d->m, d->V, d->n, t, d->out, d->scratch, d->main));
        DMRGK_TRY(dmrgk_vec_multi_axpy(d->ctx, d->n, d->m, d->V, d->n, d->out, -1.0, 1.0, t, d->main));
    }
    return DMRGK_OK;
}

// Rayleigh-matrix entries of the newest basis vector (index j = m): G[i][j] = v_i·w_j, G[j][i] = w_i·v_j.
// The read-back also brings ‖t‖² of the step (slot TT_SLOT of `out`), so a step has two host syncs, not three.
constexpr int TT_SLOT = 160;
int32_t extend_G(dmrgk_davidson* d) {
    const int j = d->m, mm = d->m_max;
    DMRGK_TRY(dmrgk_vec_multi_dot(d->ctx, d->n, j + 1, d->V, d->n, d->W + int64_t(j) * d->n, d->out, d->scratch, d->main));
    DMRGK_TRY(dmrgk_vec_multi_dot(d->ctx, d->n, j + 1, d->W, d->n, d->V + int64_t(j) * d->n, d->out + 64, d->scratch, d->main));
    DMRGK_TRY(read_back(d, TT_SLOT + 1));
    for (int i = 0; i <= j; ++i) {
        d->G[size_t(i) * mm + j] = d->host[64 + i];
        d->G[size_t(j) * mm + i] = d->host[128 + i];
    }
    d->G[size_t(j) * mm + j] = 0.5 * (d->host[64 + j] + d->host[128 + j]);
    return DMRGK_OK;
}

}  // namespace

extern "C" {

int64_t dmrgk_davidson_extra_bytes(int32_t m_max, int64_t n_padded) {
    if (m_max < 1) m_max = 1;
    if (n_padded < 0) n_padded = 0;
    return 3 * round_up(n_padded * 8, 128) + 2048 + dmrgk_vec_scratch_bytes(m_max + 1);
}

int32_t dmrgk_davidson_create(dmrgk_heff* h, int32_t m_max, double tol, int32_t max_iter,
                              double* basis_V_dev, double* basis_W_dev, const double* diag_dev,
                              void* workspace_dev, void* stream_main, void* stream_copy,
                              dmrgk_davidson** out) {
    if (!out) return fail(DMRGK_EINVAL, "davidson_create: out is NULL");
    *out = nullptr;
    if (!h) return fail(DMRGK_EINVAL, "davidson_create: heff is NULL");
    if (m_max < 2 || m_max > 62) return fail(DMRGK_EINVAL, "davidson_create: m_max = %d outside [2, 62]", m_max);
    if (!(tol >= 0.0) || max_iter < 1) return fail(DMRGK_EINVAL, "davidson_create: bad tol / max_iter");
    const int64_t n = h->layout->n_padded;
    if (n == 0) return fail(DMRGK_ESHAPE, "davidson_create: the layout has no block");
    if (!basis_V_dev || !basis_W_dev || !diag_dev || !workspace_dev)
        return fail(DMRGK_EINVAL, "davidson_create: NULL buffer");
    if (!aligned128(basis_V_dev) || !aligned128(basis_W_dev) || !aligned128(diag_dev) || !aligned128(workspace_dev))
        return fail(DMRGK_EALIGN, "davidson_create: pointers must be 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(h->ctx->device));
    dmrgk_davidson* d = new (std::nothrow) dmrgk_davidson;
    if (!d) return fail(DMRGK_ENOMEM, "davidson_create: out of host memory");
    d->h = h;
    d->ctx = h->ctx;
    d->n = n;
    d->m_max = m_max;
    d->max_iter = max_iter;
    d->tol = tol;
    d->V = basis_V_dev;
    d->W = basis_W_dev;
    d->diag = diag_dev;
    d->ws = workspace_dev;
    d->main = (cudaStream_t)stream_main;
    d->copy = (cudaStream_t)stream_copy;
    char* extra = static_cast<char*>(workspace_dev) + round_up(h->workspace_bytes, 128);
    const int64_t vb = round_up(n * 8, 128);
    d->r = reinterpret_cast<double*>(extra);
    d->t = reinterpret_cast<double*>(extra + vb);
    d->u = reinterpret_cast<double*>(extra + 2 * vb);
    d->coef = reinterpret_cast<double*>(extra + 3 * vb);
    d->out = d->coef + 64;   // 192 doubles: two dot result rows of 64 + spare
    d->scratch = extra + 3 * vb + 2048;
    d->G.assign(size_t(m_max) * m_max, 0.0);
    cudaError_t e = cudaMallocHost(&d->host, 256 * sizeof(double));
    if (e != cudaSuccess) {
        delete d;
        return fail(DMRGK_ECUDA, "davidson_create: pinned scalars: %s", cudaGetErrorString(e));
    }
    *out = d;
    return DMRGK_OK;
}

void dmrgk_davidson_destroy(dmrgk_davidson* d) {
    if (!d) return;
    if (d->host) cudaFreeHost(d->host);
    delete d;
}

int32_t dmrgk_davidson_start(dmrgk_davidson* d, const double* x0_dev) {
    if (!d || !x0_dev) return fail(DMRGK_EINVAL, "davidson_start: NULL argument");
    if (!aligned128(x0_dev)) return fail(DMRGK_EALIGN, "davidson_start: x0 not 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(d->ctx->device));
    d->started = false;
    d->converged = false;
    d->m = 0;
    d->n_apply = 0;
    DMRGK_TRY(dmrgk_vec_multi_dot(d->ctx, d->n, 1, x0_dev, d->n, x0_dev, d->out, d->scratch, d->main));
    DMRGK_TRY(read_back(d, 1));
    if (!(d->host[64] > 0.0) || !std::isfinite(d->host[64]))
        return fail(DMRGK_EINVAL, "davidson_start: start vector has norm² = %g", d->host[64]);
    DMRGK_TRY(dmrgk_vec_scal_dev(d->ctx, d->n, d->out, 3, x0_dev, d->V, d->main));
    DMRGK_TRY(apply_h(d, d->V, d->W));
    DMRGK_TRY(extend_G(d));
    d->m = 1;
    d->started = true;
    return DMRGK_OK;
}

int32_t dmrgk_davidson_step(dmrgk_davidson* d, double* theta, double* resnorm, int32_t* converged) {
    if (!d) return fail(DMRGK_EINVAL, "davidson_step: solver is NULL");
    if (!d->started) return fail(DMRGK_ESTATE, "davidson_step: call davidson_start first");
    DMRGK_CUDA(cudaSetDevice(d->ctx->device));
    const int m = d->m, mm = d->m_max;
    // Rayleigh–Ritz on the host
    std::vector<double> A(size_t(m) * m);
    for (int i = 0; i < m; ++i)
        for (int j = 0; j < m; ++j) A[size_t(i) * m + j] = 0.5 * (d->G[size_t(i) * mm + j] + d->G[size_t(j) * mm + i]);
    jacobi_lowest(A, m, &d->theta, d->y);
    for (int j = 0; j < m; ++j) d->host[j] = d->y[j];
    d->host[m] = d->theta;
    DMRGK_CUDA(cudaMemcpyAsync(d->coef, d->host, size_t(m + 1) * 8, cudaMemcpyHostToDevice, d->main));
    DMRGK_TRY(dmrgk_vec_residual(d->ctx, d->n, m, d->V, d->W, d->n, d->coef, d->r, d->out, d->scratch, d->main));
    DMRGK_TRY(read_back(d, 1));
    d->rho = std::sqrt(d->host[64]);
    if (theta) *theta = d->theta;
    if (resnorm) *resnorm = d->rho;
    d->converged = d->rho <= d->tol;
    if (converged) *converged = d->converged ? 1 : 0;
    if (d->converged) return DMRGK_OK;

    const double* theta_dev = d->coef + m;
    if (m == mm) {   // collapse restart: V=[V y], W=[W y]
        DMRGK_TRY(dmrgk_vec_multi_axpy(d->ctx, d->n, m, d->V, d->n, d->coef, 1.0, 0.0, d->t, d->main));
        DMRGK_TRY(dmrgk_vec_multi_axpy(d->ctx, d->n, m, d->W, d->n, d->coef, 1.0, 0.0, d->u, d->main));
        DMRGK_CUDA(cudaMemcpyAsync(d->V, d->t, size_t(d->n) * 8, cudaMemcpyDeviceToDevice, d->main));
        DMRGK_CUDA(cudaMemcpyAsync(d->W, d->u, size_t(d->n) * 8, cudaMemcpyDeviceToDevice, d->main));
        std::fill(d->G.begin(), d->G.end(), 0.0);
        d->G[0] = d->theta;
        d->m = 1;
    }
    DMRGK_TRY(dmrgk_vec_precond(d->ctx, d->n, d->r, d->diag, theta_dev, d->t, d->main));
    DMRGK_TRY(orthogonalise(d, d->t));
    // ‖t‖² stays on the device: the new basis vector, its image and the Rayleigh entries are computed without
    // waiting for it, and it comes back with them; a vanished correction (rare) is detected then and redone
    double* tt_dev = d->out + TT_SLOT;
    DMRGK_TRY(dmrgk_vec_multi_dot(d->ctx, d->n, 1, d->t, d->n, d->t, tt_dev, d->scratch, d->main));
    double* v = d->V + int64_t(d->m) * d->n;
    double* w = d->W + int64_t(d->m) * d->n;
    DMRGK_TRY(dmrgk_vec_scal_dev(d->ctx, d->n, tt_dev, 3, d->t, v, d->main));
    DMRGK_TRY(apply_h(d, v, w));
    DMRGK_TRY(extend_G(d));
    // correction vanished: fall back to the residual.  The apply above was wasted on a zero or noise vector
    // (finite: the scaling kernel maps 1/0 to 0) and stays counted in n_apply — the count is of applies run.
    if (!(std::sqrt(d->host[64 + TT_SLOT]) >= 1e-14 * d->rho)) {
        DMRGK_CUDA(cudaMemcpyAsync(d->t, d->r, size_t(d->n) * 8, cudaMemcpyDeviceToDevice, d->main));
        DMRGK_TRY(orthogonalise(d, d->t));
        DMRGK_TRY(dmrgk_vec_multi_dot(d->ctx, d->n, 1, d->t, d->n, d->t, tt_dev, d->scratch, d->main));
        DMRGK_CUDA(cudaMemcpyAsync(d->host + 64 + TT_SLOT, tt_dev, 8, cudaMemcpyDeviceToHost, d->main));
        DMRGK_CUDA(cudaStreamSynchronize(d->main));
        if (!(d->host[64 + TT_SLOT] > 0.0)) return fail(DMRGK_ENOTCONV, "davidson_step: the search space is exhausted (‖t‖ = 0)");
        DMRGK_TRY(dmrgk_vec_scal_dev(d->ctx, d->n, tt_dev, 3, d->t, v, d->main));
        DMRGK_TRY(apply_h(d, v, w));
        DMRGK_TRY(extend_G(d));
    }
    d->m += 1;
    return DMRGK_OK;
}

int32_t dmrgk_davidson_solve(dmrgk_davidson* d, double* theta, double* resnorm, double* x_dev, int32_t* n_apply) {
    if (!d) return fail(DMRGK_EINVAL, "davidson_solve: solver is NULL");
    if (!d->started) return fail(DMRGK_ESTATE, "davidson_solve: call davidson_start first");
    if (x_dev && !aligned128(x_dev)) return fail(DMRGK_EALIGN, "davidson_solve: x not 128-byte aligned");
    int32_t conv = 0;
    double th = 0.0, rn = 0.0;
    int m_ritz = d->m;
    while (true) {
        m_ritz = d->m;
        DMRGK_TRY(dmrgk_davidson_step(d, &th, &rn, &conv));
        if (conv || d->n_apply >= d->max_iter) break;
    }
    if (!conv) {   // Ritz pair of the final basis
        m_ritz = d->m;
        const int mm = d->m_max, m = d->m;
        std::vector<double> A(size_t(m) * m);
        for (int i = 0; i < m; ++i)
            for (int j = 0; j < m; ++j) A[size_t(i) * m + j] = 0.5 * (d->G[size_t(i) * mm + j] + d->G[size_t(j) * mm + i]);
        jacobi_lowest(A, m, &d->theta, d->y);
        for (int j = 0; j < m; ++j) d->host[j] = d->y[j];
        d->host[m] = d->theta;
        DMRGK_CUDA(cudaMemcpyAsync(d->coef, d->host, size_t(m + 1) * 8, cudaMemcpyHostToDevice, d->main));
        DMRGK_TRY(dmrgk_vec_residual(d->ctx, d->n, m, d->V, d->W, d->n, d->coef, d->r, d->out, d->scratch, d->main));
        DMRGK_TRY(read_back(d, 1));
        th = d->theta;
        rn = d->rho = std::sqrt(d->host[64]);
    }
    if (x_dev) {
        DMRGK_TRY(dmrgk_vec_multi_axpy(d->ctx, d->n, m_ritz, d->V, d->n, d->coef, 1.0, 0.0, x_dev, d->main));
        DMRGK_CUDA(cudaStreamSynchronize(d->main));
    }
    if (theta) *theta = th;
    if (resnorm) *resnorm = rn;
    if (n_apply) *n_apply = d->n_apply;
    if (!conv) return fail(DMRGK_ENOTCONV, "davidson_solve: ‖r‖ = %.3e > tol = %.3e after %d applies", rn, d->tol, d->n_apply);
    return DMRGK_OK;
}

int32_t dmrgk_davidson_set_allreduce(dmrgk_davidson* d, dmrgk_allreduce_fn fn, void* user) {
    if (!d) return fail(DMRGK_EINVAL, "davidson_set_allreduce: solver is NULL");
    d->reduce = fn;
    d->reduce_user = user;
    return DMRGK_OK;
}

int32_t dmrgk_davidson_query(const dmrgk_davidson* d, int32_t* m, int32_t* n_apply) {
    if (!d) return fail(DMRGK_EINVAL, "davidson_query: solver is NULL");
    if (m) *m = d->m;
    if (n_apply) *n_apply = d->n_apply;
    return DMRGK_OK;
}

}  // extern "C"
