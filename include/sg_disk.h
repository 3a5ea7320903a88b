/*
 * sg_disk.h -- C ABI of the B200 (sm_100a) direct self-gravity library for a razor-thin disk on
 * block-structured AMR, after arXiv 2001.02765 (Tseng, Shang & Yen).  Citations are lines of
 * /root/reference/PAPER.md (the paper's text) with the section / equation they fall in.
 *
 * What the library computes (PAPER.md:57-69 Eq. 4-5, :86-94, :96-100, :104, :110; readings in DESIGN.md):
 * the domain is the disjoint union of axis-aligned leaf cells D_c = [x_l,x_r] x [y_d,y_u], each carrying
 * one surface density sigma_c (the zeroth-order Taylor coefficient of Eq. 6).  At the centre (x_t,y_t)
 * of EVERY leaf cell t
 *
 *     Fx_t = G * sum_c sigma_c * K_c^{x,0}(x_t,y_t),      Fy_t = G * sum_c sigma_c * K_c^{y,0}(x_t,y_t)
 *
 * where K_c^{x,0} = integral over D_c of (xbar-x_t)/r^3 = [[ -ln( (ybar-y_t) + r ) ]] is the closed-form
 * mixed corner difference of PAPER.md:90-94 (z = 0), K^{y,0} the same with x and y exchanged, and where
 * a target that lies on the extension of a source grid line (xbar == x_t, exact on the integer
 * lattice) uses the paper's modified primitive.  The sum runs over ALL leaves,
 * the target's own cell included.  Everything is FP64.
 *
 * Conventions
 *   - return value: SG_OK (0) or a negative SG_ERR_* code; sg_last_error() gives a message.
 *   - levels: level 0 is the coarsest; cell_width[l+1] == cell_width[l] / 2.
 *   - a patch is P x P leaf cells of one level; (level, i0, j0) is the index of its lower-left cell on
 *     that level's lattice counted from (x0, y0); i0 and j0 must be multiples of P.  Only LEAF patches
 *     are listed (a refined patch is replaced by its four children).
 *   - cell order, used by sigma, Fx, Fy and sg_cell_geometry: [patch][j][i], i (x) fastest, patches in
 *     the order given to sg_create.
 *   - "host" / "device" below says where a pointer must live.  The context never frees or keeps a
 *     caller pointer beyond the call (device work is enqueued on the caller's stream and reads/writes
 *     the caller's device buffers asynchronously: keep them alive until the stream has drained).
 *   - there is no CPU fallback: every call that computes runs CUDA kernels on the context's device.
 */
#ifndef SG_DISK_H
#define SG_DISK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SG_OK          0
#define SG_ERR_ARG    -1   /* null pointer, non-positive size, widths not halving, ...            */
#define SG_ERR_LAYOUT -2   /* patch off its lattice / overlapping / duplicate / too large          */
#define SG_ERR_CUDA   -3   /* a CUDA runtime call failed (message has the CUDA error string)       */
#define SG_ERR_STATE  -4   /* sg_force before sg_set_density                                       */

typedef struct sg_ctx sg_ctx;                        /* opaque; owns every device array of the layout */
typedef struct { int32_t level, i0, j0; } sg_patch;  /* lower-left cell of a P x P leaf patch          */

/*
 * S1, layout build (PAPER.md:57-67: the D_i are disjoint rectangles; :104-110: leaf zones and their
 * centres).  Host work + uploads; synchronous.  Validates the patch list (levels in range, i0/j0 >= 0
 * and multiples of P, no duplicate, no patch inside another -> SG_ERR_LAYOUT), puts every cell edge
 * and centre on one integer lattice of unit cell_width[n_levels-1]/2, deduplicates cell corners
 * into a global vertex list with the <= 4 signed adjacent cells of each, and builds the per-column /
 * per-row tables used by the coincidence-safe separable part ("Kernels").
 *   out            host, receives the context
 *   cell_width     host [n_levels], physical widths; only cell_width[n_levels-1] enters the result
 *   x0, y0         physical lower-left corner of the level-0 lattice (reported back by sg_cell_geometry;
 *                  forces are translation invariant)
 *   patch_cells    P >= 1
 *   leaf_patches   host [n_patches], copied
 *   G              gravitational constant multiplying the sums (PAPER.md:139 uses G = 1)
 *   device         CUDA device ordinal
 * 2:1 balance is NOT required by the sum (any disjoint cover is valid, e.g. the paper's Table 10
 * example); sg_layout_info reports whether the layout is balanced.
 */
int sg_create(sg_ctx **out, int n_levels, const double *cell_width, double x0, double y0,
              int patch_cells, const sg_patch *leaf_patches, int64_t n_patches, double G, int device);

void sg_destroy(sg_ctx *ctx);                        /* frees device and host memory; NULL is allowed */

int64_t sg_num_cells(const sg_ctx *ctx);             /* N = n_patches * P * P ; -1 on NULL            */
int64_t sg_num_vertices(const sg_ctx *ctx);          /* N_v, deduplicated cell corners                */

/* info[0]=N, [1]=N_v, [2]=#distinct vertex x, [3]=#distinct vertex y, [4]=#distinct target x,
 * [5]=#distinct target y, [6]=1 if 2:1 balanced across faces and corners else 0, [7]=bytes of device
 * memory held by the context.  info: host [8]. */
int sg_layout_info(const sg_ctx *ctx, int64_t *info);

/* Cell centres and widths in physical units, library cell order.  xc, yc, h: host [N], any may be NULL. */
int sg_cell_geometry(const sg_ctx *ctx, double *xc, double *yc, double *h);

/*
 * S2, sigma -> signed vertex weights (exact regrouping of the corner differences of PAPER.md:92-94:
 * sum_c sigma_c [[P]]_c = sum_v w_v P(v), w_v = sum over the cells that have v as a corner of
 * +sigma (NE or SW corner) / -sigma (NW or SE corner)), plus the per-column / per-row cumulative
 * weights of the separable part.   sigma_dev: device [N], library cell order, FP64.   Asynchronous on
 * cuda_stream (a cudaStream_t passed as void*, NULL = default stream).
 */
int sg_set_density(sg_ctx *ctx, const double *sigma_dev, void *cuda_stream);

/*
 * S2 with the first-order Taylor terms of Eq. 6: on leaf c the density is
 * sigma_c + dx_c (x - x_c) + dy_c (y - y_c), and the following sg_force calls sum
 *     Fx_t = G * sum_c [ sigma_c K^{x,0} + dx_c K^{x,x} + dy_c K^{x,y} ]
 * (same for y) -- the paper's second-order method.  sigma_dev, dx_dev, dy_dev: device [N], library cell
 * order, FP64; slopes in physical units (d sigma / d x).  The paper does not say how slopes are obtained
 * (its tables use the exact Taylor coefficients, R10): they are inputs here.  A later
 * sg_set_density switches back to the zeroth-order sum.  Asynchronous on cuda_stream.
 */
int sg_set_density_linear(sg_ctx *ctx, const double *sigma_dev, const double *dx_dev, const double *dy_dev,
                          void *cuda_stream);

/*
 * S3-S5, the all-pairs sum.  Fx_dev, Fy_dev: device [N] (or [count] when a
 * target range is set, see below), FP64, written in library cell order.  Asynchronous on
 * cuda_stream.  Deterministic: the same context and sigma give bit-identical results run to run
 * (no floating-point atomics).  SG_ERR_STATE if no density has been set.  In SG_MODE_LATTICE on a
 * multi-level layout the independent pair-class kernels run on side streams owned by the context,
 * forked from and joined back into cuda_stream by events, so for the caller the call still orders
 * like one piece of work on cuda_stream (and can be captured in a CUDA graph; a launch error after the fork
 * still joins the side streams before SG_ERR_CUDA is returned).  The caller's current device is left unchanged.
 * The call enqueues kernel launches (and event records / waits) only: the internal partial-sum buffer is sized by
 * sg_create, sg_set_interaction_mode, sg_set_target_range and the first sg_set_density_linear, all host-synchronous.
 * Test aid: with the environment variable SG_POISON_PARTIALS set, the internal partial-sum buffer is filled
 * with NaN on cuda_stream at the start of every sg_force, so that a partial sum no kernel wrote surfaces in Fx, Fy.
 * Debugging aid: with SG_DEBUG_SYNC set, lattice mode synchronises after every pair-class launch and names the one
 * that failed in sg_last_error (it serialises the launches; not for timing).  Both variables are read once, at
 * sg_create; sg_force itself reads no environment.
 */
int sg_force(sg_ctx *ctx, double *Fx_dev, double *Fy_dev, void *cuda_stream);

/*
 * Restrict sg_force to the targets [first, first+count) of the library cell order (all sources are
 * still summed).  Fx_dev/Fy_dev then hold count values.  This is how the path shards over GPUs:
 * targets are independent, each rank owns a slice, no collective is needed.
 * count == 0 is allowed (sg_force does nothing).  Default: first = 0, count = N.
 * The cost follows the slice in every mode; a regrouped layout (P = 1, 2, 4 in SG_MODE_LATTICE) evaluates the 16 x 16
 * blocks that hold the slice (the covering block range: tight when the patch list is sorted by level, row, column).
 * In the lattice modes a slice is bit-identical to the same targets of the full evaluation (the source lists are split
 * as for the full range); in SG_MODE_DIRECT the source split depends on the range and a slice agrees with the full
 * evaluation to rounding (1e-13 of max|F|).
 */
int sg_set_target_range(sg_ctx *ctx, int64_t first, int64_t count);

/*
 * How sg_force evaluates the O(N^2) interaction sum (S3).  Same sum and same tolerances in every mode (
 * the paper rules out FFT on AMR, :267, :295 -- lattice mode is the patch-wise counterpart that needs no uniform grid).
 *   SG_MODE_DIRECT   every (target, vertex) pair: 1 sqrt + 2 ln (the north_star kernel; always available; default)
 *   SG_MODE_LATTICE  lattice-offset reuse: for a (target patch, source patch) pair the pair function
 *                    depends on the lattice offset only, so the pairs reduce to 2 FMA each against a table.
 *                    P = 16: the tables are windows of per-layout function lattices that this call builds ONCE (device
 *                      memory; budget a quarter of the device, SG_LATTICE_TABLE_MIB overrides) and that sg_force
 *                      streams by TMA -- no square root or logarithm is evaluated in sg_force for patch pairs up to two
 *                      levels apart (farther pairs are summed directly).  Covers the slope path of
 *                      sg_set_density_linear too (three table planes, 6 FMA per pair).  Over the budget: as
 *                      SG_MODE_LATTICE_INCTA, and the slope path runs direct.
 *                    P = 1, 2, 4 (e.g. the paper's zone-wise quadtrees): the leaves are regrouped into padded 16 x 16
 *                      blocks of an inner context (needs a device); set the density AFTER selecting the mode, an
 *                      sg_force with a density set before returns SG_ERR_STATE.
 *                    P = 8: a lighter one-target-per-thread kernel with tables built on the fly (pairs up to one level
 *                      apart by table; zeroth-order path only, the slope path runs direct).
 *                    Other P: SG_ERR_ARG.
 *   SG_MODE_LATTICE_BLOCKED  as SG_MODE_LATTICE, but SG_ERR_ARG unless P = 16.  For tests and profiling.
 *   SG_MODE_LATTICE_INCTA    P = 16, offset tables built inside the CTAs at every sg_force (the round-1 kernels; no
 *                    table memory; zeroth-order path only).  Bit-identical to SG_MODE_LATTICE.
 * Per-patch weights of lattice mode (same sum either way): the zeroth-order path uses deduplicated weights owned on
 * 16 x 16 vertices of a patch on lattices of up to 4,096 units (extent / (h_fin / 2)), and weights from the patch's own
 * cells on all 17 x 17 vertices (every patch neutral: less rounding on steep, deep hierarchies, 7-8 % slower) beyond
 * -- the library switches by itself -- or everywhere when SG_LATTICE_NEUTRAL_WEIGHTS is set (read at sg_create).  The
 * slope path always uses the neutral weights: its planes enter multiplied by the lattice offset, and only neutral
 * patches keep it at the accuracy of the direct slope kernel (BASELINE config 4: rel. L2 1.7e-12 owned, gate 1e-12).
 * Host-synchronous: may allocate and build tables; not to be called during stream capture.
 */
#define SG_MODE_DIRECT  0
#define SG_MODE_LATTICE 1
#define SG_MODE_LATTICE_BLOCKED 2
#define SG_MODE_LATTICE_INCTA 3
int sg_set_interaction_mode(sg_ctx *ctx, int mode);

const char *sg_last_error(const sg_ctx *ctx);        /* ctx may be NULL: error of the last failed sg_create */
const char *sg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SG_DISK_H */
