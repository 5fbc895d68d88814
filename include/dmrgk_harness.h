/* dmrgk_harness.h — test and measurement aids exported by libdmrgk.so next to the product API of dmrgk.h:
 * the seeded input generators (bit-identical to workloads/rng.py, so that tests and bench.py can fill
 * 100-GB arenas on the device), the register-only FP64 pipe probes bench.py reports its ceilings from, and
 * host-only views of the planner's tiling rules for the CPU tests.  Nothing here is on the hot path
 * and a user of the library needs none of it.  Conventions as in dmrgk.h. */
#ifndef DMRGK_HARNESS_H
#define DMRGK_HARNESS_H
#include "dmrgk.h"
#ifdef __cplusplus
extern "C" {
#endif

/* Counter-based values, bit-identical to workloads/rng.py normal12(seed, stream, index): fills the
 * packed arena of an operator / a ψ layout from the UNPADDED element index of each entry, times
 * scale (scale_mode 0: 1, 1: 1/sqrt(cols of the block)); symmetric != 0: square diagonal-sector
 * blocks get 0.5·(g(r,c)+g(c,r)).  Padding is zero-filled. */
int32_t dmrgk_op_fill_normal(const dmrgk_op* op, double* arena_dev, uint64_t seed, uint64_t stream_id,
                             int32_t scale_mode, int32_t symmetric, void* stream);
int32_t dmrgk_layout_fill_normal(const dmrgk_layout* l, double* arena_dev, uint64_t seed,
                                 uint64_t stream_id, void* stream);
/* Φ blocks: normal12 / sqrt(rows of the block) (workloads.fill_phi_host). */
int32_t dmrgk_iso_fill_normal(const dmrgk_iso* phi, double* arena_dev, uint64_t seed, uint64_t stream_id,
                              void* stream);
/* Register-only FP64 pipe probes: every warp of a full grid issues `iters` rounds of 16 independent
 * mma.sync.m8n8k4.f64 (kind 0: 4 CTAs × 8 warps per SM; kinds 2, 3, 4: 1, 2, 3 CTAs × 4 warps per SM)
 * or 32 independent fma.rn.f64 per lane (kind 1).  Returns the flops issued in *flops; the caller
 * times the stream with events. */
int32_t dmrgk_probe_fp64(dmrgk_ctx* ctx, int32_t kind, int64_t iters, double* sink_dev,
                         double* flops, void* stream);
/* Host only (no device needed): the tile boundaries the task-list builder uses for a block dimension of
 * `extent` rows (tile_max = 64, or 128 for the tall-tile variant) or padded columns (tile_max = 64) — the
 * balanced tiling of DESIGN.md §4.1: ceil(extent/tile_max) tiles, origins at multiples of 16, extents that
 * differ by at most 16, larger tiles first.  Writes n + 1 boundaries (the last one = extent) to `cuts` if
 * cap ≥ n + 1 and returns n; DMRGK_EINVAL (negative) on bad arguments.  For tests of the host logic. */
int32_t dmrgk_plan_tile_cuts(int32_t extent, int32_t tile_max, int32_t* cuts, int32_t cap);
/* Host only: the cost per k-tile the planner assigns to a tile of rows × cols computed elements (fragment
 * products of its fullest warp × 4, with the latency floor for thin tiles; a full 64×64 tile costs 64). */
int32_t dmrgk_plan_tile_cost(int32_t rows, int32_t cols);

#ifdef __cplusplus
}
#endif
#endif /* DMRGK_HARNESS_H */
