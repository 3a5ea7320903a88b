// sg_kernels_lin.cuh -- internal: device arrays and launchers of the slope-term path (sg_kernels_lin.cu).
#pragma once
#include "sg_kernels.cuh"

namespace sg {

// tile of the slope path: double xc[kChunksPerTile]; then per slot {y, W0, a, c}  ->  8,320 bytes
constexpr int kTileLinDoubles = kChunksPerTile + 4 * kTileSlots;

struct LinArrays {                    // allocated on the first sg_set_density_linear
    bool allocated = false;
    double unit = 0.0;                // physical length of one lattice unit
    int cells_per_patch = 1;
    double *patch_hh = nullptr;       // [n_patches] half cell width in lattice units
    double *wl = nullptr;             // [3 Nv]  {W0, a, c}
    double *vtile = nullptr;          // [n_tiles * kTileLinDoubles]
    double *TBx3 = nullptr;           // [ntY][nX][3]
    double *TBy3 = nullptr;           // [ntX][nY][3]
};

size_t interaction_lin_smem_bytes(int tab_entries);
cudaError_t configure_lin_kernels(int tab_entries);
int lin_targets_per_thread();

void launch_weights_lin(const DevLayout &d, const LinArrays &l, const double *sigma, const double *dx, const double *dy,
                        cudaStream_t s);
void launch_interaction_lin(const DevLayout &d, const LinArrays &l, const ForcePlan &p, cudaStream_t s);
void launch_finalise_lin(const DevLayout &d, const LinArrays &l, const ForcePlan &p, double *Fx, double *Fy,
                         cudaStream_t s);

// per (target, vertex) pair: 22 DFMA + 3 DADD + 3 DMUL (+ 5 per (target, chunk)); see sg_kernels_lin.cu
constexpr double kLinFp64InstrPerPair = 28.0 + 5.0 / kChunk;
constexpr double kLinFlopsPerPair = 22 * 2 + 3 + 3 + 6.0 / kChunk;   // per chunk: 1 DFMA + 3 DADD + 1 DMUL

}  // namespace sg
