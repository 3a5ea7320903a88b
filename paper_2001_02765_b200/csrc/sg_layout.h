// sg_layout.h -- internal: host-side flattened AMR layout (S1 of DESIGN.md).  Not part of the C ABI.
//
// All coordinates are integers on one lattice whose unit is half the finest cell width, so every
// cell edge (even multiples of 2^(L-1-level)) and every cell centre is an integer and the paper's
// coincidence test "xbar == x" (sgn(|xbar-x|)) is an exact integer comparison.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/sg_disk.h"

namespace sg {

constexpr int32_t kMaxLattice = 1 << 26;   // u^2+v^2 < 2^53 stays an exact FP64 integer

struct HostLayout {
    int n_levels = 0, P = 0;
    double unit = 0.0, x0 = 0.0, y0 = 0.0;
    int64_t N = 0, Nv = 0;
    int32_t extent = 0;                    // max lattice coordinate of any vertex (>= 2)
    bool balanced = true;
    std::vector<sg_patch> patches;

    // targets (leaf-cell centres), library cell order [patch][j][i]
    std::vector<int32_t> tkx, tky;         // lattice coordinates
    std::vector<int32_t> itx, ity;         // index into tX / tY
    std::vector<int32_t> tX, tY;           // sorted distinct target x / y

    // vertices (deduplicated cell corners), sorted by (kx, ky): column c is the contiguous range
    // [colstart[c], colstart[c+1]) and is sorted by ky inside.
    std::vector<int32_t> vkx, vky;
    std::vector<int32_t> adj;              // [4*Nv]: (cell << 2) | corner, or -1; corner 0 NE(+) 1 NW(-) 2 SE(-) 3 SW(+)
    std::vector<int32_t> colX, colstart;   // distinct vertex x (sorted); [nX+1]
    std::vector<int32_t> rowY, rowstart;   // distinct vertex y (sorted); [nY+1]
    std::vector<int32_t> rowperm;          // vertex indices sorted by (ky, kx)

    // chunks: runs of <= kChunk consecutive vertices of ONE column (same x), so that u, u^2 and s(u)
    // are shared by the whole chunk in the interaction kernel.  slot_vertex[c*kChunk + j] is the vertex
    // in slot j of chunk c, or -1 for a padding slot (it gets w = 0 and the coordinates of the chunk's
    // first vertex).  The chunk count is padded to a multiple of kChunksPerTile with copies of chunk 0
    // whose slots are all -1.
    std::vector<int32_t> chunk_x;          // [n_chunks]
    std::vector<int32_t> slot_vertex;      // [n_chunks * kChunk]
};

constexpr int kChunk = 16;                 // vertices per chunk
constexpr int kChunksPerTile = 16;         // chunks per shared-memory tile (one TMA bulk copy)

// Returns SG_OK or SG_ERR_*; on error `err` holds the message.
// cell_present (optional, [n_patches * P * P], library cell order): a PADDED layout, used internally when a layout of
// small patches is regrouped into 16 x 16 blocks for lattice mode -- cells with 0 are holes (the block is only partly
// covered by leaves of its level): they are targets whose result is discarded and they are not sources (no vertex
// records, no adjacency), so patches of different levels may overlap in their holes and the overlap / balance checks
// are skipped (the layout was derived from one that passed them).
int build_layout(HostLayout &out, int n_levels, const double *cell_width, double x0, double y0,
                 int P, const sg_patch *patches, int64_t n_patches, std::string &err,
                 const uint8_t *cell_present = nullptr);

}  // namespace sg
