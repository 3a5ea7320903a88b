// sg_kernels_patch.cuh -- internal: lattice-offset reuse path, sg_kernels_patch.cu.
#pragma once
#include "sg_kernels.cuh"

namespace sg {

struct PatchInfo {                    // one leaf patch on the integer lattice
    int32_t X0, Y0;                   // lattice coordinates of its lower-left vertex
    int32_t cw;                       // cell width in lattice units (2 << (n_levels-1-level))
    int32_t level;
};

struct PatchLevel {                   // the leaf patches of one level (contiguous in the sorted patch list)
    int32_t p0, n;                    // patches [p0, p0 + n)
    int32_t pimin, pjmin, npx, npy;   // bounding box of their positions in patch units (i0 / P, j0 / P)
    int32_t map_off;                  // pmap[map_off + (pj - pjmin) * npx + (pi - pimin)] = patch index or -1
    int32_t cw;                       // cell width in lattice units
};

struct PatchGroup {                   // <= 8 consecutive target patches of one level: one CTA work item per split
    int32_t level, first, n;
    int32_t dpi_min, ndpi, dpj_min, ndpj;   // box of patch offsets d = B - A that can hit a source patch of the level
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
    double *wP = nullptr;             // [n_patches * wstride] per-patch signed vertex weights, [j][i]
};

struct PatchPlan {
    int n_split = 1, patches_per_split = 0;
    int first_patch = 0, n_tpatches = 0;   // target patches touched by the target range
    int grid = 0;
    size_t smem = 0;
};

size_t patch_smem_bytes(int P, int tab_entries);
cudaError_t configure_patch_kernels(int P, int tab_entries);
void launch_patch_weights(const PatchArrays &pa, const double *sigma, cudaStream_t s);
void launch_patch_interaction(const DevLayout &d, const PatchArrays &pa, const PatchPlan &pp, int64_t first,
                              int64_t count, double *part, int skip_same_level, cudaStream_t s);
// register-blocked same-level kernel with one offset table per CTA (P = 16); uses the second queue counter
// (d.queue + 1) and writes the first po.n_split slots of d.part
struct OffsetPlan {
    int g_first = 0, n_groups = 0;    // groups touched by the target range
    int n_split = 1;                  // splits of every group's offset list
    int grid = 0;
};
size_t patch_offset_smem_bytes();
cudaError_t configure_patch_offset();
void launch_patch_offset(const DevLayout &d, const PatchArrays &pa, const OffsetPlan &po, int64_t first, int64_t count,
                         cudaStream_t s);

}  // namespace sg
