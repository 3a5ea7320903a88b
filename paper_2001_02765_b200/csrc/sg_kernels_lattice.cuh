// sg_kernels_lattice.cuh -- internal: lattice mode with PRECOMPUTED pair-function lattices streamed by TMA
// (sg_kernels_lattice.cu).  Same pair classes, target groups and offset boxes as sg_kernels_patch.cuh.
#pragma once
#include "sg_kernels_patch.cuh"

namespace sg {

// The pair function of a pair class depends only on the lattice offset (u, v) between a source vertex and a target
// centre, and for a given (target level, class) every offset table of patch_offset_kernel is a window of ONE
// two-dimensional array ("function lattice") F[row][col]:
//     u(col) = (col + cmin - MMIN) g - cw_target / 2,    v(row) = (row + rmin - MMIN) g - cw_target / 2,
// g = min(target pitch, source pitch) in lattice units; the table of patch offset d = (dx, dy) is the window of
// M x M entries at (row, col) = (16 dy - rmin, 16 dx - cmin).  The arrays depend on the layout only: they are built
// once (sg_set_interaction_mode) and every sg_force streams windows of them into shared memory with TMA bulk copies.
// Planes: 0 = {T1, T2}, T1 = s(v) ln(|v|+r), T2 = s(u) ln(|u|+r)          (zeroth order, and -W0 of the slope path)
//         1 = {u T1 + v T2, u T2 - r}    (slope path, weights a)       2 = {v T1 - r, u T1 + v T2}    (weights c)
struct FnLattice {
    int64_t base;                     // first entry (double2) of plane 0 in the context's function-lattice buffer
    int64_t plane_stride;             // entries between planes
    int32_t ncols, nrows;
    int32_t cmin, rmin;               // 16 * (smallest dx / dy of any group box of this (level, class))
    int32_t present;                  // 0: class absent at this level
    int32_t pad;
};

struct LatticeArrays {
    bool ready = false;               // function lattices built for plane 0 (n_planes_built >= 1)
    int n_planes_built = 0;           // 1 (zeroth order) or 3 (with the slope planes)
    FnLattice *meta = nullptr;        // device [n_levels * kOffClasses]
    double2 *fn = nullptr;            // the function lattices
    int64_t fn_entries = 0;           // entries per plane (sum over (level, class))
    double *wS = nullptr;             // [3][n_patches * kPatchQStride] per-patch weights of the slope path: -W0, a, c
    bool lin_neutral = false;         // wS holds own-cell weights on all 17 x 17 vertices (sg_api.cu: neutral_weights)
};

constexpr int kFnPlanesLin = 3;

// bytes of dynamic shared memory of lattice_corr_kernel<V>
size_t lattice_smem_bytes(int V);
cudaError_t configure_lattice_kernels();
// build the planes [plane0, plane0 + n) of every function lattice (host metadata in `meta_host`, same order as device)
void launch_build_fn_lattices(const LatticeArrays &la, const FnLattice *meta_host, const PatchLevel *levels_host,
                              int n_levels, const DevLayout &d, int plane0, int n, cudaStream_t s);
// pair class V with tables from the function lattices; n_planes = 1: weights wQ (zeroth order); 3: weights la.wS
void launch_lattice_corr(int V, const DevLayout &d, const PatchArrays &pa, const LatticeArrays &la, const OffsetPlan &po,
                         int n_planes, int64_t first, int64_t count, double *part, int sms, cudaStream_t s);
}  // namespace sg
