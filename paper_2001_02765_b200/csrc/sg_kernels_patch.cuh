// sg_kernels_patch.cuh -- internal: lattice-offset reuse path, sg_kernels_patch.cu.
#pragma once
#include "sg_kernels.cuh"

namespace sg {

struct PatchInfo {                    // one leaf patch on the integer lattice
    int32_t X0, Y0;                   // lattice coordinates of its lower-left vertex
    int32_t cw;                       // cell width in lattice units (2 << (n_levels-1-level))
    int32_t level;
};

struct PatchLevel {                   // the leaf patches of one level (the patch list may be in any order)
    int32_t p0, n;                    // first patch of the level in the list, number of patches
    int32_t pimin, pjmin, npx, npy;   // bounding box of their positions in patch units (i0 / P, j0 / P)
    int32_t map_off;                  // pmap[map_off + (pj - pjmin) * npx + (pi - pimin)] = patch index or -1
    int32_t cw;                       // cell width in lattice units
};

// Pair classes of patch_offset_kernel<V>: source patches of the target's own level (V = 0), of the next coarser
// level (V = 1), the next finer level (V = 2), two levels coarser (V = 3), two levels finer (V = 4).
constexpr int kOffSame = 0, kOffCoarserSrc = 1, kOffFinerSrc = 2, kOffCoarserSrc4 = 3, kOffFinerSrc4 = 4;
constexpr int kOffClasses = 5;
// Target-patch groups come in three lists: 0 = any 8 patches of a level (classes 0, 2, 4), 1 = 8 patches of one
// residue class (pi % 2, pj % 2) (class 1), 2 = of one residue class mod 4 (class 3): for a coarser source the source
// patch of A at offset d is (A + d) / F, which must be integral for the whole group.
constexpr int offset_group_list(int V) { return V == kOffCoarserSrc ? 1 : V == kOffCoarserSrc4 ? 2 : 0; }

struct PatchGroup {                   // <= 8 target patches of one level (lists 1, 2: of one residue class)
    int32_t level, n;
    int32_t patch[8];                 // patch indices (unused entries: -1)
    int32_t pmin, pmax;               // smallest / largest patch index (target-range test)
    // per pair class: box of patch offsets d that can hit a source patch, in units of the FINER level's patch
    // size: {dpi_min, ndpi, dpj_min, ndpj}; classes 1 / 3 step d by 2 / 4 (A + d must be a multiple); ndpi = 0: absent
    int32_t box[kOffClasses][4];
};

constexpr int kPatchQStride = 17 * 18;   // doubles per patch in wQ

struct PatchArrays {
    bool enabled = false;             // P is 8 or 16
    bool blocked = false;             // P == 16: patch_offset_kernel available (dense per-level patch maps built)
    PatchLevel *levels = nullptr;     // [n_levels]
    PatchGroup *groups = nullptr;     // [n_groups], ordered by first patch
    int n_groups = 0;
    int32_t *pmap = nullptr;
    double *wQ = nullptr;             // [n_patches * kPatchQStride] per-patch weights, rows 18 apart
    int P = 0;
    int n_patches = 0;
    int wstride = 0;                  // doubles per patch in wP: (P+1)^2 rounded up to a multiple of 2
    PatchInfo *info = nullptr;        // [n_patches]
    double *wP = nullptr;             // [n_patches * wstride] per-patch (owned, deduplicated) vertex weights, [j][i]
    int32_t *far_list = nullptr;      // P = 16: per level, the patches >= 3 levels away (patch_far_kernel)
    int32_t *far_meta = nullptr;      // [2 n_levels]: first entry and count of every level's list
    int32_t *pflags = nullptr;        // [n_patches] bit 0: vertex row P owned somewhere; bit 1: vertex column P (rows < P)
    int32_t *pvmap = nullptr;         // [n_patches * (P+1)^2] global vertex owned by patch vertex (i, j), or -1
};

struct PatchPlan {
    int n_split = 1, patches_per_split = 0;
    int first_patch = 0, n_tpatches = 0;   // target patches touched by the target range
    int grid = 0;
    size_t smem = 0;
};

size_t patch_smem_bytes(int P, int tab_entries);
cudaError_t configure_patch_kernels(int P, int tab_entries);
// w: flat deduplicated vertex weights (DevLayout::w); wl: {W0, a, c} per vertex of the slope path (LinArrays::wl)
void launch_patch_weights(const PatchArrays &pa, const double *w, cudaStream_t s);
void launch_patch_weights_owncell(const PatchArrays &pa, const double *sigma, cudaStream_t s);
void launch_patch_weights_lin_owncell(const PatchArrays &pa, const double *sigma, const double *dx, const double *dy,
                                      const double *patch_hh, double unit, double *wS, cudaStream_t s);
void launch_patch_weights_lin(const PatchArrays &pa, const double *wl, double *wS, cudaStream_t s);
// skip_near: patch pairs fewer than skip_near levels apart are skipped (done by patch_offset_kernel); 0 = none
void launch_patch_interaction(const DevLayout &d, const PatchArrays &pa, const PatchPlan &pp, int64_t first,
                              int64_t count, double *part, int skip_near, cudaStream_t s);
// P = 16: pairs >= 3 levels apart summed directly; wq: pa.wQ (zeroth order) or the three slope planes (lin)
cudaError_t configure_patch_far(int tab_entries);
void launch_patch_far(bool lin, const DevLayout &d, const PatchArrays &pa, const double *wq, const PatchPlan &pp,
                      int64_t first, int64_t count, double *part, cudaStream_t s);
// register-blocked kernels with one offset table per CTA (P = 16), patch pairs at most two levels apart
struct OffsetPlan {
    int n_groups[3] = {0, 0, 0};      // sizes of the three group lists, stored back to back
    int n_split = 1;                  // splits of every group's offset list
    int first_patch = 0, last_patch = -1;   // target patches touched by the target range
    bool variant[kOffClasses] = {false, false, false, false, false};   // pair classes present for the target range
};
cudaError_t configure_patch_offset();
// pair class V writes po.n_split slots of [2][count] partial sums at `part` and uses queue counter 1 + V
void launch_patch_offset(int V, const DevLayout &d, const PatchArrays &pa, const OffsetPlan &po, int64_t first,
                         int64_t count, double *part, int sms, cudaStream_t s);

}  // namespace sg
