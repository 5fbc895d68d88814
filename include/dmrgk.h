/* dmrgk.h — C ABI of the B200-native H_eff·ψ / Davidson hot path of arXiv 2311.14106.
 *
 * What the library computes (§II.A: "iterative diagonalization of the effective
 * Hamiltonian built from renormalized block operators"; BASELINE.json north_star):
 *
 *     σ = Σ_k c_k (L_k ⊗ R_k) ψ ,   per block:
 *     σ[qA+δ_k, qB−δ_k] += c_k · (−1)^{π_k·N(qA)} · L_k[qA+δ_k, qA] · ψ[qA, qB] · R_k[qB−δ_k, qB]ᵀ
 *
 * ψ is the two-site wavefunction as a block-sparse matrix ψ[a, b] over the U(1) (or U(1)×U(1))
 * sectors of the enlarged left block A and the enlarged right block B, with blocks only where
 * q_A + q_B = target.  π_k is the fermion parity of pair k; N(q) is the particle number of the
 * INPUT A sector (sum of the charge components).  Everything is FP64.
 *
 * Conventions
 *  - Every function returns 0 (DMRGK_OK) or a negative dmrgk_status.  Nothing throws or aborts across
 *    the ABI.  dmrgk_last_error() returns a thread-local message for the last failure.
 *  - Handles are opaque; *_create writes the handle to *out; *_destroy(NULL) is a no-op.
 *  - OWNERSHIP: the caller owns every large buffer (operator arenas, ψ, σ, Davidson basis, workspace,
 *    pinned host arenas).  The library borrows raw pointers; buffers must stay alive until the stream
 *    work using them has completed.  The library owns only its metadata.  "dev" = device pointer,
 *    "host" = host pointer; every device pointer must be 128-byte aligned (DMRGK_EALIGN otherwise).
 *  - Streams are cudaStream_t passed as void* (NULL = legacy default stream).
 *  - ASYNCHRONY: heff_apply, heff_diag and the vec_* calls enqueue work and return; the
 *    davidson_* calls and *_host calls synchronise the stream (they read scalars back).
 *  - LAYOUT ("panel layout"): a block (rows × cols) occupies rows_pad·ld doubles with
 *    ld = round_up(cols, 16), rows_pad = round_up(rows, 4).  It is stored as ld/16 column PANELS one
 *    after the other; a panel holds rows_pad rows of 16 doubles (128 bytes each), and inside a row the
 *    four 32-byte groups are XOR-swizzled with the row index: element (r, c) sits at
 *        ((c / 16)·rows_pad + r)·16 + ((c mod 16) xor ((r mod 4)·4))          doubles from the block origin,
 *    so a (rows ≤ 64) × 16-column operand tile is ONE contiguous chunk for a bulk copy and its
 *    shared-memory image is read without bank conflicts.  Padding rows and columns must be zero
 *    (pack/fill write zeros; every kernel of the library preserves zeros there).  A block-sparse object
 *    is one packed arena plus a block table; block offsets (in doubles) are multiples of 64.  ψ, σ,
 *    diag(H_eff) and all Davidson vectors share the layout of dmrgk_layout, so vector kernels run over
 *    the flat padded arena.  Callers never index the packed form themselves: *_pack / *_unpack and
 *    dmrgk_block_unpack translate to and from the "unpadded" form — block after block in table order,
 *    each block rows×cols row-major with no padding — which is also what the seeded fill indexes.
 */
#ifndef DMRGK_H
#define DMRGK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum dmrgk_status {
    DMRGK_OK = 0,
    DMRGK_EINVAL = -1,   /* NULL pointer, negative size, bad flag                       */
    DMRGK_ESHAPE = -2,   /* operator space is not the layout's, sizes disagree           */
    DMRGK_ECHARGE = -3,  /* charge shifts of a pair do not cancel / parity mismatch      */
    DMRGK_EALIGN = -4,   /* device pointer not 128-byte aligned                          */
    DMRGK_ENOMEM = -5,   /* host or device allocation of library metadata failed         */
    DMRGK_ECUDA = -6,    /* a CUDA runtime call failed (message holds the CUDA error)    */
    DMRGK_ENOTCONV = -7, /* davidson_solve hit max_iter                                  */
    DMRGK_ESTATE = -8    /* call out of order (unbound operator, solver not started)     */
} dmrgk_status;

typedef struct dmrgk_ctx dmrgk_ctx;
typedef struct dmrgk_space dmrgk_space;
typedef struct dmrgk_layout dmrgk_layout;
typedef struct dmrgk_op dmrgk_op;
typedef struct dmrgk_heff dmrgk_heff;
typedef struct dmrgk_davidson dmrgk_davidson;

const char* dmrgk_last_error(void);
/* Library version string, "dmrgk <version> sm_100a src:<16 hex digits>": the hash identifies the sources
 * and compiler flags the binary was built from (paper_2311_14106_b200/build.py source_hash). */
const char* dmrgk_version(void);

/* Number of CUDA kernels this library has launched in the calling process so far (every launch site
 * counts; memcpys/memsets do not).  reset != 0 returns the count and zeroes it. */
int64_t dmrgk_launch_count(int32_t reset);

/* ---- context ------------------------------------------------------------------------------ */
/* Binds the library to CUDA device `device` (cudaSetDevice on every call that launches work).
 * Fails with DMRGK_ECUDA when no device is present: there is no CPU fallback. */
int32_t dmrgk_ctx_create(int32_t device, dmrgk_ctx** out);
void dmrgk_ctx_destroy(dmrgk_ctx* ctx);
/* Number of SMs and bytes of L2 of the bound device. */
int32_t dmrgk_ctx_query(const dmrgk_ctx* ctx, int32_t* n_sm, int64_t* l2_bytes, int64_t* hbm_bytes);

/* ---- a1: sector index / block layout ("Tables") ------------- */
/* One space per half (A, B).  charges is [n_sectors][n_charges] (n_charges 1 or 2), dims[i] ≥ 0
 * (dim 0 = empty sector, skipped everywhere).  Charge tuples must be distinct. */
int32_t dmrgk_space_create(dmrgk_ctx* ctx, int32_t n_charges, int32_t n_sectors,
                           const int32_t* charges, const int32_t* dims, dmrgk_space** out);
void dmrgk_space_destroy(dmrgk_space* s);

/* ψ layout: one block (a, b) for every A sector a (in A order) whose partner charge
 * target − q_a is a B sector, both dims > 0.  A layout with no block is valid (n_blocks = 0). */
int32_t dmrgk_layout_create(dmrgk_ctx* ctx, const dmrgk_space* A, const dmrgk_space* B,
                            const int32_t* target, dmrgk_layout** out);
void dmrgk_layout_destroy(dmrgk_layout* l);
/* n_elems = Σ rows·cols (unpadded), n_padded = doubles of the packed arena (multiple of 16). */
int32_t dmrgk_layout_query(const dmrgk_layout* l, int64_t* n_blocks, int64_t* n_elems,
                           int64_t* n_padded);
/* Block table; each output array has n_blocks entries (any may be NULL).  offset is in doubles
 * into the packed arena; block i occupies dmrgk_block_size(rows[i], cols[i]) doubles from there. */
int32_t dmrgk_layout_blocks(const dmrgk_layout* l, int32_t* a_idx, int32_t* b_idx, int32_t* rows,
                            int32_t* cols, int32_t* ld, int64_t* offset);
/* Host-side test aids: unpadded ↔ packed (host pointers; pack zero-fills the padding). */
int32_t dmrgk_layout_pack(const dmrgk_layout* l, const double* unpadded_host, double* packed_host);
int32_t dmrgk_layout_unpack(const dmrgk_layout* l, const double* packed_host, double* unpadded_host);

/* A stored operator on one half with charge shift dq: one block (q+dq, q) for every column sector
 * q (in sector order) such that q+dq is a sector and both dims > 0.  parity: 0 even, 1 odd. */
int32_t dmrgk_op_create(dmrgk_ctx* ctx, const dmrgk_space* space, const int32_t* dq, int32_t parity,
                        dmrgk_op** out);
void dmrgk_op_destroy(dmrgk_op* op);
int32_t dmrgk_op_query(const dmrgk_op* op, int64_t* n_blocks, int64_t* n_elems, int64_t* n_padded);
int32_t dmrgk_op_blocks(const dmrgk_op* op, int32_t* row_idx, int32_t* col_idx, int32_t* rows,
                        int32_t* cols, int32_t* ld, int64_t* offset);
int32_t dmrgk_op_pack(const dmrgk_op* op, const double* unpadded_host, double* packed_host);
int32_t dmrgk_op_unpack(const dmrgk_op* op, const double* packed_host, double* unpadded_host);
/* One block in isolation (host test aids; no handle needed): the number of doubles a rows×cols block
 * occupies, its dense row-major form from its packed form, and whether all its padding is zero
 * (returns 0 if so, 1 if not). */
int64_t dmrgk_block_size(int32_t rows, int32_t cols);
int32_t dmrgk_block_unpack(int32_t rows, int32_t cols, const double* packed_host, double* dense_host);
int32_t dmrgk_block_padding_is_zero(int32_t rows, int32_t cols, const double* packed_host);
/* Resident operator: packed arena in device memory (n_padded doubles, 128-B aligned). */
int32_t dmrgk_op_bind_device(dmrgk_op* op, const double* arena_dev);
/* Staged operator ("H2D IO"): packed arena in PINNED host memory;
 * heff_apply copies it through the staging ring on the copy stream each time it is needed. */
int32_t dmrgk_op_bind_pinned(dmrgk_op* op, const double* arena_pinned_host);

/* ---- a2: operator-pair task list ---------------------------------------- */
enum {
    DMRGK_TRANS_L = 1u, /* apply the transpose of the stored L operator (h.c. partner)  */
    DMRGK_TRANS_R = 2u, /* apply the transpose of the stored R operator                 */
    DMRGK_IDENT_L = 4u, /* L is the identity on A (L[k] must be NULL)                   */
    DMRGK_IDENT_R = 8u, /* R is the identity on B (R[k] must be NULL)                   */
    DMRGK_HC_OF_PREV = 16u /* pair k is the Hermitian conjugate of pair k−1: L[k], R[k] are ignored (may
                           be NULL) and the stored operators of pair k−1 are applied transposed
                           (its TRANS flags toggled, its IDENT flags kept); coef[k] is the caller's —
                           −coef[k−1] for a fermionic (odd) pair, +coef[k−1] for an even one */
};

typedef struct dmrgk_heff_opts {
    int64_t t_chunk_bytes;  /* cap on the L_k·ψ intermediate workspace per chunk of pairs
                               (0 = default: about 1/16 of the total, clamped to
                               [512 MiB, 4 GiB]); pairs are processed chunk by chunk and the
                               workspace holds two such buffers                             */
    int64_t ring_bytes;     /* staging ring for pinned operators, split in three parts
                               (0 = no ring: binding a pinned operator is then an error)     */
    int32_t kernel;         /* 0 = DMMA tensor-core kernel (product path),
                               1 = scalar check kernel (same task lists; debugging aid),
                               2, 3 = the DMMA kernel at other residencies (measurement aid),
                               4 = the DMMA kernel with a tall 128×64 CTA tile,
                               5 = variant 0 claiming work units eagerly (L2 sharing experiment) */
    int32_t split_waves;    /* phase-2 split-k target: units per CTA slot (0 = default 32)  */
    int32_t order_policy;   /* GEMM order per task: 0 = the cheaper of (Lψ)Rᵀ and
                               L(ψRᵀ) by flop count, 1 = always (Lψ)Rᵀ, 2 = always L(ψRᵀ); tasks
                               with an identity factor are a single product either way            */
    int32_t per_pair_output;/* 1: plan for dmrgk_heff_expect — every pair writes its own σ_k = c_k (L_k ⊗ R_k) ψ
                               (not summed); dmrgk_heff_apply / _diag / Davidson refuse such a plan  */
    int32_t reserved[2];
} dmrgk_heff_opts;

/* Builds the task list of σ = Σ_k coef[k] (L[k] ⊗ R[k]) ψ for the given layout: enumerates
 * (k, input block) pairs whose L and R blocks exist and whose output block is in the layout, folds
 * coef[k]·(−1)^{π_k N(q_A)} into one scalar per task, groups tasks by OUTPUT block (accumulation
 * needs no atomics), tiles, plans split-k, cuts the pair list into chunks, uploads the metadata.
 * Every operator must already be bound.  K = 0 is valid (σ = 0).
 * Errors: DMRGK_ESHAPE (operator space ≠ layout's), DMRGK_ECHARGE (applied shifts do not cancel, or
 * parities differ), DMRGK_ESTATE (unbound operator; pinned operator without ring), DMRGK_EINVAL. */
int32_t dmrgk_heff_create(dmrgk_ctx* ctx, const dmrgk_layout* layout, int64_t K,
                          dmrgk_op* const* L, dmrgk_op* const* R, const double* coef,
                          const uint32_t* flags, const dmrgk_heff_opts* opts, dmrgk_heff** out);
/* As dmrgk_heff_create, with one extra scalar per (pair, INPUT ψ block): the task of pair k on input block
 * ib gets coef[k] · block_coef[k·n_blocks + ib] (n_blocks and the block order are those of
 * dmrgk_layout_blocks); a zero entry removes the task.  This is the slot for the SU(2) recoupling
 * coefficients of spin-adapted DMRG (BASELINE.json north_star: "SU(2) recoupling folded
 * into per-block-pair scalar coefficients"): with reduced matrix elements as the stored blocks, the sectors
 * labelled by (N, 2j) — for a singlet target the B half by (N, −2j) so that charges add up to the target — and
 * a rank-k operator split into one stored operator per Δ(2j), the 6j/9j factor of each block pair goes here
 * (SURVEY §8(f) NEXT-3).  block_coef = NULL is dmrgk_heff_create. */
int32_t dmrgk_heff_create_blockcoef(dmrgk_ctx* ctx, const dmrgk_layout* layout, int64_t K,
                                    dmrgk_op* const* L, dmrgk_op* const* R, const double* coef,
                                    const double* block_coef, const uint32_t* flags,
                                    const dmrgk_heff_opts* opts, dmrgk_heff** out);
void dmrgk_heff_destroy(dmrgk_heff* h);
/* flops_alg = Σ_tasks min(2m′n(m+n′), 2mn′(n+m′)) (identity factor → one product),
 * flops_exec = flops of the products the kernels execute in the chosen GEMM order (= flops_alg with
 * order_policy 0),
 * op_bytes = 8·Σ_tasks (m′m + n′n), workspace_bytes = what heff_apply needs (128-B aligned). */
int32_t dmrgk_heff_query(const dmrgk_heff* h, int64_t* n_tasks, double* flops_alg,
                         double* flops_exec, int64_t* op_bytes, int64_t* workspace_bytes,
                         int64_t* n_chunks, int64_t* n_launches_per_apply);

/* ---- a3 + a5..a7: σ = H_eff ψ ------------------------------------------------------------- */
/* Overwrites sigma_dev (whole padded arena).  psi_dev and sigma_dev must not alias.
 * stream_copy is used only when pinned operators are present (may equal NULL otherwise). */
int32_t dmrgk_heff_apply(dmrgk_heff* h, const double* psi_dev, double* sigma_dev,
                         void* workspace_dev, void* stream_main, void* stream_copy);
/* End-to-end form with HOST buffers (packed layout, pinned recommended): H2D ψ, apply, D2H σ,
 * synchronises.  psi_dev / sigma_dev are device scratch arenas of n_padded doubles. */
int32_t dmrgk_heff_apply_host(dmrgk_heff* h, const double* psi_host, double* sigma_host,
                              double* psi_dev, double* sigma_dev, void* workspace_dev,
                              void* stream_main, void* stream_copy);
/* a4: diag(H_eff) in ψ layout: Σ over tasks whose input block = output block of
 * coef·sign·L[i,i]·R[j,j].  Pinned operators are read through the ring like in apply. */
int32_t dmrgk_heff_diag(dmrgk_heff* h, double* diag_dev, void* workspace_dev, void* stream_main,
                        void* stream_copy);

/* Expectation values of the operator pairs ("one- and two-particle reduced
 * density matrices … computed" on the same kernels): out_dev[k] = ⟨ψ, c_k (L_k ⊗ R_k) ψ⟩ for every pair k of a
 * plan created with per_pair_output = 1, e.g. γ_ij = ⟨c†_i c_j⟩ with the pair list {c†_i c_j as L ⊗ R}.
 * Phase 1 as in apply; phase 2 writes σ_k of each pair of a chunk into its own buffer in the workspace;
 * a fused multi-dot against ψ (fixed-order, bit-reproducible) gives the K numbers.  out_dev: K doubles in
 * device memory; asynchronous. */
int32_t dmrgk_heff_expect(dmrgk_heff* h, const double* psi_dev, double* out_dev, void* workspace_dev,
                          void* stream_main, void* stream_copy);

/* Measurement aid.  enable = 1: every later heff_apply brackets its whole GEMM region
 * (first phase-1 launch … last reduce) with one CUDA event pair on stream_main; the launches keep
 * their normal overlap (phase 1 of chunk c+1 runs concurrently with phase 2 of chunk c).
 * enable = 2 (diagnostic): apply runs every launch on stream_main, serialised, each inside its own
 * event pair.  enable = 0 switches profiling off.  Every call zeroes the sums.
 * profile_read synchronises on the recorded events and returns the accumulated device time in ms and
 * the launch counts since the last enable, as ms[4] / launches[4] = {phase-1 GEMM (a5), phase-2 GEMM
 * (a6), split-k reduce (a7), whole-apply span}; ms[0..2] are only filled in mode 2, launches[3]
 * counts applies.  Either pointer may be NULL. */
int32_t dmrgk_heff_profile(dmrgk_heff* h, int32_t enable);
int32_t dmrgk_heff_profile_read(dmrgk_heff* h, double* ms, int64_t* launches);

/* ---- a8: vector kernels over the flat padded arena (n doubles) ----------------------------
 * The iterative diagonalisation of H_eff ("Lánczos or Davidson", §II.A, thresholds
 * ε_Davidson of PAPER.md:114, 118) needs, besides σ = H_eff ψ, only BLAS-1 work on ψ-sized vectors: the
 * Rayleigh-matrix dots, the Ritz vector and residual, the diagonal preconditioner and the
 * Gram–Schmidt passes (SURVEY §8(a) a8, §8(c) "Davidson, step by step").  Fused multi-vector forms
 * first (what the driver uses), the plain BLAS-1 names of SURVEY §8(b) after them. */
/* Reductions are two-stage and fixed-order (bit-reproducible); scratch_dev needs
 * dmrgk_vec_scratch_bytes(nv) bytes; results land in out_dev[nv] (device) — asynchronous. */
int64_t dmrgk_vec_scratch_bytes(int32_t nv);
/* out[j] = Σ_i X[j·stride + i] · y[i], j < nv. */
int32_t dmrgk_vec_multi_dot(dmrgk_ctx* ctx, int64_t n, int32_t nv, const double* X_dev,
                            int64_t stride, const double* y_dev, double* out_dev,
                            void* scratch_dev, void* stream);
/* The same dots with no scratch argument, for callers that cannot allocate device memory: a sweep driver
 * whose operator arenas and staging ring already fill HBM, a host code that is handed a fixed set of
 * device buffers and owns no allocator, or a step running beside the side-stream operator copies, which
 * a cudaMalloc / cudaFree would stall by synchronising the device.  The per-CTA partial sums go to a
 * 592 KiB array inside the library image (held by every GPU that loads the library until exit), so:
 *   - nv ≤ 64, DMRGK_EINVAL beyond that (n is unlimited); arguments otherwise as dmrgk_vec_multi_dot's,
 *     same kernels, bit-identical results;
 *   - the call itself makes no cudaMalloc / cudaFree and no allocating library call;
 *   - the first call on each device looks the array's device address up (cudaGetSymbolAddress, with that
 *     device current); make that first call before any stream capture begins;
 *   - there is one array per GPU, shared by all calls: calls that may overlap on the GPU (different
 *     streams with no ordering between them) race on it — order them.  Nothing in it needs clearing: a
 *     call reads only the slots it has itself written. */
int32_t dmrgk_vec_multi_dot_noalloc(dmrgk_ctx* ctx, int64_t n, int32_t nv, const double* X_dev,
                                    int64_t stride, const double* y_dev, double* out_dev, void* stream);
/* y[i] = beta·y[i] + alpha·Σ_j coef_dev[j]·X[j·stride + i]  (coefficients read from device memory,
 * nv ≤ 64; beta = 0 overwrites without reading y). */
int32_t dmrgk_vec_multi_axpy(dmrgk_ctx* ctx, int64_t n, int32_t nv, const double* X_dev,
                             int64_t stride, const double* coef_dev, double alpha, double beta,
                             double* y_dev, void* stream);
/* y = alpha·x + beta·y with host scalars. */
int32_t dmrgk_vec_axpby(dmrgk_ctx* ctx, int64_t n, double alpha, const double* x_dev, double beta,
                        double* y_dev, void* stream);
/* y = f·x with f from a device scalar a = *alpha_dev: mode 0: f = a, 1: f = 1/a, 2: f = sqrt(a),
 * 3: f = 1/sqrt(a)  (normalisation by a squared norm without a host round trip).  y may alias x.
 * In the inverse modes a = 0 gives f = 0, not Inf: a vector that vanished stays a zero vector. */
int32_t dmrgk_vec_scal_dev(dmrgk_ctx* ctx, int64_t n, const double* alpha_dev, int32_t mode,
                           const double* x_dev, double* y_dev, void* stream);
/* out[0] = x·y ;  out[0] = ‖x‖₂ ;  y += alpha·x ;  x *= alpha  (host scalars; dot / nrm2 results land in
 * device memory like multi_dot's, scratch as for nv = 1). */
int32_t dmrgk_vec_dot(dmrgk_ctx* ctx, int64_t n, const double* x_dev, const double* y_dev,
                      double* out_dev, void* scratch_dev, void* stream);
int32_t dmrgk_vec_nrm2(dmrgk_ctx* ctx, int64_t n, const double* x_dev, double* out_dev,
                       void* scratch_dev, void* stream);
int32_t dmrgk_vec_axpy(dmrgk_ctx* ctx, int64_t n, double alpha, const double* x_dev, double* y_dev,
                       void* stream);
int32_t dmrgk_vec_scal(dmrgk_ctx* ctx, int64_t n, double alpha, double* x_dev, void* stream);
/* Davidson residual and correction (SURVEY §8(c) "Davidson, step by step"):
 *   r = Σ_j y[j]·(W_j − θ V_j);  out[0] = ‖r‖²  (y, θ from device: coef_dev[0..m) = y, coef_dev[m] = θ) */
int32_t dmrgk_vec_residual(dmrgk_ctx* ctx, int64_t n, int32_t m, const double* V_dev,
                           const double* W_dev, int64_t stride, const double* coef_dev,
                           double* r_dev, double* out_dev, void* scratch_dev, void* stream);
/*   t[i] = r[i] / den, den = θ − d[i], |den| < 1e-10 → ±1e-10 (sign of den, +0 → +). */
int32_t dmrgk_vec_precond(dmrgk_ctx* ctx, int64_t n, const double* r_dev, const double* diag_dev,
                          const double* theta_dev, double* t_dev, void* stream);

/* ---- a8 + a9: Davidson (ε_Davidson = residual 2-norm) ----- */
/* basis_V_dev / basis_W_dev hold m_max vectors of n_padded doubles each (caller-owned), diag_dev the
 * diagonal from dmrgk_heff_diag, workspace_dev the heff_apply workspace plus
 * dmrgk_davidson_extra_bytes(m_max, n_padded) bytes after it. */
int64_t dmrgk_davidson_extra_bytes(int32_t m_max, int64_t n_padded);
int32_t dmrgk_davidson_create(dmrgk_heff* h, int32_t m_max, double tol, int32_t max_iter,
                              double* basis_V_dev, double* basis_W_dev, const double* diag_dev,
                              void* workspace_dev, void* stream_main, void* stream_copy,
                              dmrgk_davidson** out);
void dmrgk_davidson_destroy(dmrgk_davidson* d);
/* V_0 = x0/‖x0‖, W_0 = H V_0, m = 1. */
int32_t dmrgk_davidson_start(dmrgk_davidson* d, const double* x0_dev);
/* One pass of the loop = exactly one H_eff apply (none if it converges first):
 * Rayleigh–Ritz on the current basis → θ, residual norm; if not converged: (collapse restart if
 * m = m_max), preconditioned correction, 2× Gram–Schmidt, normalise, apply, append. */
int32_t dmrgk_davidson_step(dmrgk_davidson* d, double* theta, double* resnorm, int32_t* converged);
/* Steps until ‖r‖ ≤ tol or max_iter applies; writes the Ritz vector to x_dev (n_padded doubles).
 * Returns DMRGK_ENOTCONV (θ and x still written) when max_iter is reached. */
int32_t dmrgk_davidson_solve(dmrgk_davidson* d, double* theta, double* resnorm, double* x_dev,
                             int32_t* n_apply);
/* Current subspace size m, and the number of H_eff applies run since davidson_start (the start's own
 * included).  A step runs exactly one apply, except when the preconditioned correction vanishes after
 * orthogonalisation (it lies in the span of the basis — e.g. an exactly diagonal H_eff): that is only
 * known when ‖t‖² comes back with the Rayleigh entries, so the step then redoes the new basis vector from
 * the residual and has run two. */
int32_t dmrgk_davidson_query(const dmrgk_davidson* d, int32_t* m, int32_t* n_apply);
/* Multi-GPU k-sharding hook (the sum over operator pairs
 * is split over the GPUs, ψ is replicated, σ is the sum of the ranks' partial results).  When set, fn
 * is called right after every H_eff apply of the driver with the freshly written W vector (device
 * pointer, n_padded doubles) and the main stream; it must turn the vector into the SUM over all ranks
 * in stream order (e.g. an NCCL all-reduce) and return 0.  Every rank then iterates on identical
 * data.  fn = NULL removes the hook.  The library itself never communicates. */
typedef int32_t (*dmrgk_allreduce_fn)(double* vec_dev, int64_t n, void* stream, void* user);
int32_t dmrgk_davidson_set_allreduce(dmrgk_davidson* d, dmrgk_allreduce_fn fn, void* user);

/* ---- renormalisation step ("the renormalization step",
 *      PAPER.md:142 Fig. 7 "Ren_l", "Ren_r"):  O′ = Φᵀ O Φ  for every operator kept -------------- */
/* Φ: the kept basis of one half, a charge-block-diagonal map from the NEW space (kept states) into
 * the ENLARGED space: one block (dim_enl(q) × dim_new(q)) for every enlarged sector (in enlarged
 * order) whose charge is also a sector of the new space, both dims > 0.  Same packed layout rules as
 * operators (panel layout, zero padding). */
typedef struct dmrgk_iso dmrgk_iso;
int32_t dmrgk_iso_create(dmrgk_ctx* ctx, const dmrgk_space* enlarged, const dmrgk_space* kept,
                         dmrgk_iso** out);
void dmrgk_iso_destroy(dmrgk_iso* phi);
int32_t dmrgk_iso_query(const dmrgk_iso* phi, int64_t* n_blocks, int64_t* n_elems, int64_t* n_padded);
/* enl_idx / new_idx: sector indices in the enlarged / kept space. */
int32_t dmrgk_iso_blocks(const dmrgk_iso* phi, int32_t* enl_idx, int32_t* new_idx, int32_t* rows,
                         int32_t* cols, int32_t* ld, int64_t* offset);
int32_t dmrgk_iso_pack(const dmrgk_iso* phi, const double* unpadded_host, double* packed_host);
int32_t dmrgk_iso_bind_device(dmrgk_iso* phi, const double* arena_dev);

typedef struct dmrgk_renorm dmrgk_renorm;
typedef struct dmrgk_renorm_opts {
    int64_t t_chunk_bytes;  /* cap on the O·Φ intermediate per chunk of operators (0 = default: total/16
                               in [256 MiB, 4 GiB]); the workspace holds two such buffers                */
    int32_t kernel;         /* 0 = DMMA kernel, 1 = scalar check kernel                               */
    int32_t reserved[5];
} dmrgk_renorm_opts;
/* Plans out[i] = Φᵀ in[i] Φ for n_ops operators: in[i] lives on the enlarged space of Φ, out[i] on the
 * kept space with the same charge shift and parity; per stored block
 *     out[i][q+δ, q] = Φ[q+δ]ᵀ · in[i][q+δ, q] · Φ[q]
 * as two grouped GEMMs (T = in·Φ, then Φᵀ·T) on the same FP64 tensor-core kernel as heff_apply.
 * Blocks whose row or column sector keeps no state are skipped.  Every in[i], out[i] and Φ must be
 * bound to DEVICE arenas; the arenas bound to out[i] are WRITTEN by dmrgk_renorm_apply (all blocks
 * including their zero padding).  Errors: DMRGK_ESHAPE (wrong space), DMRGK_ECHARGE (shift or parity
 * of in[i] and out[i] differ), DMRGK_ESTATE (unbound / pinned-only operand), DMRGK_EINVAL. */
int32_t dmrgk_renorm_create(dmrgk_ctx* ctx, const dmrgk_iso* phi, int64_t n_ops,
                            dmrgk_op* const* in, dmrgk_op* const* out,
                            const dmrgk_renorm_opts* opts, dmrgk_renorm** plan);
void dmrgk_renorm_destroy(dmrgk_renorm* plan);
/* flops = Σ_blocks 2·e′·e·n + 2·n′·e′·n (e, e′: enlarged dims; n, n′: kept dims). */
int32_t dmrgk_renorm_query(const dmrgk_renorm* plan, int64_t* n_tasks, double* flops,
                           int64_t* workspace_bytes, int64_t* n_launches_per_apply);
/* Enqueues the products and returns (asynchronous); all work is ordered after what `stream` holds at
 * the call and joined back into `stream` (two library-owned streams overlap the two phases). */
int32_t dmrgk_renorm_apply(dmrgk_renorm* plan, void* workspace_dev, void* stream);

/* ---- block enlargement (second half; "Ren_l") -------------
 * The next bond's enlarged block is A′ = (kept block) ⊗ (site).  Every operator on A′ is a sum of products
 *        O_{A′} = Σ_j coef_j · (X_j · P^{π_j}) ⊗ y_j ,
 * X_j a stored operator on the KEPT space (its transpose when flag bit 0 is set; the identity when
 * t_x[j] is NULL), y_j a d×d site operator (row-major, t_y[j·d·d …]), P = (−1)^N on the kept column index,
 * π_j = flag bit 1 (set when the site factor is fermionic: the site's Jordan–Wigner string runs over the
 * block).  Which products make up which operator — the complementary-operator sums over t and V — is
 * host bookkeeping (paper_2311_14106_b200/blockops.py: "complementary operators built on the host").
 *
 * site_major = 0 is this LEFT-block form.  site_major = 1 is the RIGHT block, B′ = (site) ⊗ (kept block) with
 * the site's modes first: a product is (y · P_s^{π_x}) ⊗ X with the parity on the small SITE factor, which the
 * caller folds into y (flag bit 1 must be clear; flag bit 2 marks a fermionic site factor for validation only).
 *
 * `enlarged` must be the sector-major product space: sector q′ holds every kept sector k for which q′ − q_k
 * is the charge of a site state — ordered by kept sector (in the kept space's order) for the left block, by
 * site state for the right block; site_charges is [d][n_charges], all distinct.  out[i] live on `enlarged`
 * and are bound to DEVICE arenas, which dmrgk_enlarge_apply overwrites completely (zero fill, then every
 * sub-block once — contributions are grouped by destination, no atomics).  Errors: DMRGK_ESHAPE (spaces /
 * sector dimensions inconsistent), DMRGK_ECHARGE (shift or parity of a product does not match its target),
 * DMRGK_ESTATE (unbound), DMRGK_EINVAL. */
typedef struct dmrgk_enlarge dmrgk_enlarge;
int32_t dmrgk_enlarge_create(dmrgk_ctx* ctx, const dmrgk_space* kept, const dmrgk_space* enlarged, int32_t d,
                             const int32_t* site_charges, int32_t site_major, int64_t n_out, dmrgk_op* const* out,
                             int64_t n_terms, const int32_t* t_out, dmrgk_op* const* t_x,
                             const uint32_t* t_flags, const double* t_coef, const double* t_y,
                             dmrgk_enlarge** plan);
void dmrgk_enlarge_destroy(dmrgk_enlarge* plan);
/* n_tiles: 32×32 destination tiles; n_sources: (sub-block, source) pairs; bytes = 8·elements moved. */
int32_t dmrgk_enlarge_query(const dmrgk_enlarge* plan, int64_t* n_tiles, int64_t* n_sources,
                            int64_t* bytes_read, int64_t* bytes_written);
int32_t dmrgk_enlarge_apply(dmrgk_enlarge* plan, void* stream);

/* The seeded input fills, the FP64 pipe probes and the host-only views of the planner that tests and
 * bench.py use are declared in dmrgk_harness.h: exported by the same library, not part of the product API. */

#ifdef __cplusplus
}
#endif
#endif /* DMRGK_H */
