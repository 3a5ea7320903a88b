// sg_kernels_patch.cuh -- internal: lattice-offset reuse path, sg_kernels_patch.cu.
#pragma once
#include "sg_kernels.cuh"

namespace sg {

struct PatchInfo {                    // one leaf patch on the integer lattice
    int32_t X0, Y0;                   // lattice coordinates of its lower-left vertex
    int32_t cw;                       // cell width in lattice units (2 << (n_levels-1-level))
    int32_t level;
};

struct PatchArrays {
    bool enabled = false;             // P is 8 or 16
    bool blocked = false;             // P == 16 and the per-warp tables + log table fit in shared memory
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
// register-blocked same-level kernel (P = 16); uses the second queue counter (d.queue + 1), writes d.part slots
size_t patch_blocked_smem_bytes(int tab_entries);
cudaError_t configure_patch_blocked(int tab_entries);
void launch_patch_same_level(const DevLayout &d, const PatchArrays &pa, const PatchPlan &pp, int64_t first,
                             int64_t count, cudaStream_t s);

}  // namespace sg
