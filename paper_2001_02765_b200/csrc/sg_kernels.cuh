// sg_kernels.cuh -- internal interface between the C-ABI layer (sg_api.cu) and the kernels
// (sg_kernels.cu).  Device pointers only; no ownership here.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace sg {

constexpr int kTile = 256;            // vertices per shared-memory tile (one TMA bulk copy of 24*kTile B)
constexpr int kTileDoubles = 3 * kTile;   // tile layout: double2 xy[kTile]; double w[kTile]
constexpr int kStages = 3;            // tiles in flight per CTA
constexpr int kThreads = 256;         // threads per CTA of the interaction kernel
constexpr int kLogK = 9;              // mantissa bits in the log-table index (|f| <= 2^-10 -> degree 4)

struct DevLayout {
    int64_t N = 0, Nv = 0;
    int nX = 0, nY = 0, ntX = 0, ntY = 0;
    int n_tiles = 0;                  // ceil(Nv / kTile)
    double G = 1.0;
    // targets
    double2 *tgt = nullptr;           // [N] lattice (kx, ky) as FP64 (exact integers)
    int32_t *itx = nullptr, *ity = nullptr;   // [N] index of the target's x / y among the distinct ones
    // vertices
    int32_t *adj = nullptr;           // [4 Nv]
    int32_t *vkx = nullptr, *vky = nullptr;   // [Nv]
    double *vtile = nullptr;          // [n_tiles * kTileDoubles]
    double *w = nullptr;              // [Nv]
    int32_t *colX = nullptr, *colstart = nullptr;           // [nX], [nX+1]
    int32_t *rowY = nullptr, *rowstart = nullptr, *rowperm = nullptr;   // [nY], [nY+1], [Nv]
    int32_t *tX = nullptr, *tY = nullptr;                   // [ntX], [ntY]
    double *TBx = nullptr;            // [ntY][nX]  weight strictly below y_t on column X
    double *TBy = nullptr;            // [ntX][nY]  weight strictly left of x_t on row Y
    // log table: lntab[i] = -ln(c_i), c_i = rcp.approx of the centre of bin (tab_idx0 + i)
    double *lntab = nullptr;
    int tab_idx0 = 0, tab_entries = 0;
    // split-source partial sums [n_split][2][count]
    double *part = nullptr;
    int64_t part_capacity = 0;        // doubles
};

struct ForcePlan {
    int T = 4;                        // targets per thread
    int n_split = 1;                  // source splits
    int tiles_per_split = 0;
    int64_t first = 0, count = 0;     // target range
    int n_tblocks = 0;                // ceil(count / (kThreads*T))
    int grid = 0;                     // CTAs launched (persistent over work items)
    size_t smem = 0;
};

size_t interaction_smem_bytes(int tab_entries);
cudaError_t configure_kernels(int tab_entries);   // cudaFuncSetAttribute for the opt-in smem size

void launch_build_logtab(const DevLayout &d, cudaStream_t s);
void launch_fill_static_tiles(const DevLayout &d, cudaStream_t s);        // xy part of vtile (once)
void launch_vertex_weights(const DevLayout &d, const double *sigma, cudaStream_t s);
void launch_line_tables(const DevLayout &d, cudaStream_t s);
void launch_interaction(const DevLayout &d, const ForcePlan &p, cudaStream_t s);
void launch_finalise(const DevLayout &d, const ForcePlan &p, double *Fx, double *Fy, cudaStream_t s);
cudaError_t measure_dfma(double *tflops, double *warp_instr_per_s);

// FP64-pipe warp instructions and FLOPs per (target, vertex) pair of the interaction kernel as
// written (cross-checked against cuobjdump -sass in DESIGN.md "Roofline").
constexpr double kFp64InstrPerPair = 23.0;
constexpr double kFlopsPerPair = 39.0;   // 16 DFMA x 2 + 4 DADD + 3 DMUL

}  // namespace sg
