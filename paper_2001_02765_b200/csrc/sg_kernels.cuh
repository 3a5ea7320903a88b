// sg_kernels.cuh -- internal interface between the C-ABI layer (sg_api.cu) and the kernels
// (sg_kernels.cu).  Device pointers only; no ownership here.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "sg_layout.h"

namespace sg {

// One shared-memory tile = kChunksPerTile chunks of kChunk vertices that share their x:
//   double xc[kChunksPerTile];  double2 yw[kChunksPerTile * kChunk]  ( {y, w} per vertex slot )
// = 4,224 bytes, moved by ONE TMA bulk copy.
constexpr int kTileSlots = kChunksPerTile * kChunk;              // 256 vertex slots per tile
constexpr int kTileDoubles = kChunksPerTile + 2 * kTileSlots;    // 528 doubles
constexpr int kStages = 3;            // tiles in flight per CTA
constexpr int kThreads = 256;         // threads per CTA of the interaction kernel
constexpr int kQueues = 8;            // atomic work-item counters per context
constexpr int kLogK = 9;              // mantissa bits in the log-table index (|f| <= 2^-10 -> degree 4)

struct DevLayout {
    int64_t N = 0, Nv = 0;
    int nX = 0, nY = 0, ntX = 0, ntY = 0;
    int n_tiles = 0;                  // n_chunks / kChunksPerTile
    int64_t n_slots = 0;              // n_tiles * kTileSlots (>= Nv: padding slots carry w = 0)
    double G = 1.0;
    // targets
    double2 *tgt = nullptr;           // [N] lattice (kx, ky) as FP64 (exact integers)
    int32_t *itx = nullptr, *ity = nullptr;   // [N] index of the target's x / y among the distinct ones
    // vertices
    int32_t *adj = nullptr;           // [4 Nv]
    int32_t *vkx = nullptr, *vky = nullptr;   // [Nv]
    int32_t *chunk_x = nullptr;       // [n_tiles * kChunksPerTile]
    int32_t *slot_vertex = nullptr;   // [n_slots] vertex index or -1
    double *vtile = nullptr;          // [n_tiles * kTileDoubles]
    double *w = nullptr;              // [Nv]
    double *wcum = nullptr;           // [2 Nv] running sums of w along the columns, then along the rows (S2b scratch)
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
    unsigned int *queue = nullptr;    // kQueues work-item counters of the interaction kernels (reset by finalise)
    // ln of the integer lattice distances 0 .. lnint_n-1 (lnint[0] = 0) for the separable part; lnint_n = 0 when
    // the lattice is too large for a table (then finalise calls log())
    double *lnint = nullptr;
    int lnint_n = 0;
};

struct ForcePlan {
    int T = 4;                        // targets per thread
    int n_split = 1;                  // source splits
    int tiles_per_split = 0;
    int64_t first = 0, count = 0;     // target range
    int n_tblocks = 0;                // ceil(count / (kThreads*T))
    int grid = 0;                     // CTAs launched (persistent, pull work items from the queue)
    size_t smem = 0;
};

// Opt-in dynamic shared memory.  cudaFuncAttributeMaxDynamicSharedMemorySize is a per-function, process-wide
// setting, so it must not depend on the context that happens to be created last: every kernel gets the device's
// maximum (opt-in limit minus the kernel's static shared memory), the same value whichever context asks.
// `need_bytes` is what the asking context will launch with: cudaErrorInvalidValue if even the maximum is too small.
template <class Kernel>
inline cudaError_t opt_in_max_smem(Kernel kernel, size_t need_bytes) {
    int dev = 0, optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, kernel);
    if (e != cudaSuccess) return e;
    const int max_dyn = optin - int(fa.sharedSizeBytes);
    if (max_dyn < 0 || need_bytes > size_t(max_dyn)) return cudaErrorInvalidValue;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn);
}

size_t interaction_smem_bytes(int tab_entries);
cudaError_t configure_kernels(int tab_entries);   // opt-in smem (opt_in_max_smem) for the interaction kernels

void launch_build_logtab(const DevLayout &d, cudaStream_t s);
void launch_build_lnint(const DevLayout &d, cudaStream_t s);
void launch_fill_static_tiles(const DevLayout &d, cudaStream_t s);        // xc and y of vtile (once)
void launch_vertex_weights(const DevLayout &d, const double *sigma, cudaStream_t s);
void launch_line_tables(const DevLayout &d, cudaStream_t s);
void launch_interaction(const DevLayout &d, const ForcePlan &p, cudaStream_t s);
void launch_finalise(const DevLayout &d, const ForcePlan &p, double *Fx, double *Fy, cudaStream_t s);
cudaError_t measure_dfma(double *tflops, double *warp_instr_per_s);
cudaError_t measure_dmma(double *dmma_tflops, double *mixed_tflops);   // FP64 mma.sync alone / interleaved with DFMA
// regrouped layouts: caller cell order <-> padded block order (b, c may be null: sigma only)
void launch_scatter_cells(const double *a, const double *b, const double *c, const int32_t *inv, double *oa, double *ob,
                          double *oc, int64_t n_inner, cudaStream_t s);
void launch_gather_cells(const double *fx, const double *fy, const int32_t *map, int64_t base, int64_t first,
                         int64_t count, double *ox, double *oy, cudaStream_t s);

// FP64-pipe warp instructions and FLOPs per (target, vertex slot) of the interaction kernel as written
// (cross-checked against cuobjdump -sass): per pair 16 DFMA + 3 DADD + 2 DMUL,
// plus per (target, chunk) 2 DADD + 1 DMUL shared by kChunk pairs.
constexpr double kFp64InstrPerPair = 21.0 + 3.0 / kChunk;
constexpr double kFlopsPerPair = 16 * 2 + 3 + 2 + 3.0 / kChunk;

}  // namespace sg
