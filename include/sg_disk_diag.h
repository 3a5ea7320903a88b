/*
 * sg_disk_diag.h -- diagnostics of libsg_disk.so used by the tests, bench.py and the profiling notes: launch-plan
 * replay, launch counts, kernel timing, the roofline model of the kernels as built, and an FP64 peak micro-benchmark.
 * None of these is part of the method (include/sg_disk.h is); same conventions as there.
 */
#ifndef SG_DISK_DIAG_H
#define SG_DISK_DIAG_H

#include "sg_disk.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Diagnostic of the SG_MODE_LATTICE launch plan (P = 16), computed on the host (works on a context created with
 * device < 0): replays the walk of the offset-table kernels over every target group and patch offset and counts
 * the (target patch, source patch) pairs it reaches.  out[16]:
 *   out[0..4]  pairs reached per pair class: same level, source one level coarser, one finer, two coarser, two finer
 *   out[5]     pairs reached more than once (must be 0)      out[6]  pairs of the wrong level distance (must be 0)
 *   out[7..9]  target groups in the three group lists         out[10] offsets visited (= offset tables at most)
 *   out[11]    1 if the plan exists (P = 16, patch maps fit), else 0 and everything else is 0
 *   out[12]    target patches that are not exactly once in a group list whose pair classes are launched (must be 0:
 *              every launched class writes the partial sums of every target)      out[13..15] reserved, 0
 * Every patch pair at most two levels apart must be reached exactly once; pairs farther apart are summed directly.
 * Only for layouts of at most 65,536 patches (larger: counts stay 0).
 */
int sg_lattice_plan_check(const sg_ctx *ctx, int64_t *out);

/*
 * Fill of the offset walk (P = 16), host only: per pair class V, out[3 V] = offsets visited by all target groups,
 * out[3 V + 1] = offsets at which at least one of the group's <= 8 target patches has a source patch (one table each),
 * out[3 V + 2] = patch pairs.  pairs / (8 * live offsets) is the fraction of warp slots with work when the warps of a
 * CTA move through the offsets in lock step (patch_offset_kernel); lattice_corr_kernel lets them drift apart by the
 * depth of its stage ring (profiles/r2_*).  out: host [15].
 */
int sg_lattice_plan_fill(const sg_ctx *ctx, int64_t *out);

/* Number of kernel launches one sg_set_density / one sg_force enqueues with the current settings. */
int sg_launch_counts(const sg_ctx *ctx, int *set_density_launches, int *force_launches);

/*
 * Kernel timing for the roofline line.  While enabled, every sg_force records a pair of CUDA events
 * on the caller's stream around the interaction kernel (S3) only; no synchronisation is added to
 * sg_force.  sg_get_kernel_times synchronises on the newest end event and returns the durations (ms)
 * of the sg_force calls made since timing was enabled, oldest first; at most 64 are kept.
 *   ms: host [capacity];  n: host, receives the number written.
 */
int sg_set_kernel_timing(sg_ctx *ctx, int enable);
int sg_get_kernel_times(sg_ctx *ctx, float *ms, int capacity, int *n);

/*
 * Roofline model of the interaction kernel(s) the current mode selects, as built (instruction counts are read off the
 * SASS and guarded by tests/test_sass_counts.py).  Any pointer may be NULL.
 *   pair_evaluations      ALGORITHMIC units one sg_force processes: count * N_v (target, deduplicated vertex) pairs
 *                          -- the unit roofline.achieved is computed from, in every mode.
 *   fp64_instr_per_pair   FP64-pipe warp instructions per unit; flops_per_pair: the same in FLOPs (FMA = 2).
 *                         Direct kernel 21.2 / 37.2 (1 sqrt + 2 ln), slope kernel 28.3 / 50.5, lattice mode 2 / 4
 *                         (the two DFMA of the correlation; offset tables and the directly summed far pairs are
 *                         not credited).
 *   executed_evaluations  pairs the kernels actually run: direct = count * vertex slots (incl. zero-weight padding);
 *                         lattice = count * n_patches * (P+1)^2 per-patch vertices, (P+1)^2/P^2 times the
 *                         deduplicated list.  executed / pair_evaluations is the redundancy of the formulation.
 */
int sg_kernel_model(const sg_ctx *ctx, double *fp64_instr_per_pair, double *flops_per_pair,
                    double *pair_evaluations, double *executed_evaluations);

/* The instruction-count constants behind sg_kernel_model, without a context: kernel 0 = interaction_kernel (direct,
 * zeroth order), 1 = interaction_lin_kernel (direct, slope terms).  tests/test_sass_counts.py recounts them from the
 * SASS of the built library.  SG_ERR_ARG for another kernel id. */
int sg_kernel_instruction_counts(int kernel, double *fp64_instr_per_pair, double *flops_per_pair);

/* Diagnostic: sustained DFMA rate of the device (8 independent chains per thread, full occupancy),
 * in FP64 TFLOP/s (FMA = 2), and the same as warp-instructions/s.  Synchronous. */
int sg_measure_fp64_peak(int device, double *tflops, double *warp_instr_per_s);

/* Diagnostic: FP64 tensor-core rate (mma.sync.m8n8k4.f64, 512 flop per warp instruction) alone, and the total rate
 * of a loop that interleaves one DFMA with every DMMA: if the two shared nothing the second would be the sum of the
 * DMMA and DFMA peaks (DESIGN.md 6b uses this to decide against a tensor-core formulation).  Synchronous. */
int sg_measure_fp64_mma_peak(int device, double *dmma_tflops, double *mixed_tflops);

#ifdef __cplusplus
}
#endif
#endif /* SG_DISK_DIAG_H */
