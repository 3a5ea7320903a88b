// sg_layout.cpp -- S1: flatten a leaf patch list into lattice targets + a deduplicated, signed vertex
// list (host).  Follows PAPER.md:57-67 (disjoint rectangles covering the domain), :104-110 (leaf zones,
// force at zone centres) and the corner-difference structure of PAPER.md:92-94:
//   [[f]]_c = f(x_r,y_u) - f(x_l,y_u) - f(x_r,y_d) + f(x_l,y_d)   =>   signs NE +, NW -, SE -, SW +.
#include "sg_layout.h"

#include <algorithm>
#include <cmath>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <unordered_set>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace sg {
namespace {

inline uint64_t patch_key(int level, int64_t pi, int64_t pj) {
    return (uint64_t(level) << 58) | (uint64_t(pi) << 29) | uint64_t(pj);
}

std::string fmt(const char *f, long long a = 0, long long b = 0, long long c = 0, long long d = 0) {
    char buf[256];
    std::snprintf(buf, sizeof buf, f, a, b, c, d);
    return buf;
}

// std::sort over chunks in parallel, then pairwise merges (the layout build is host work a regridding caller pays at
// every regrid: PAPER.md:265; the 4N-record sort was most of it)
template <class It, class Cmp>
void parallel_sort(It first, It last, Cmp cmp) {
    const int64_t n = last - first;
    int nt = 1;
#ifdef _OPENMP
    nt = std::max(1, std::min(omp_get_max_threads(), 32));
#endif
    if (n < (int64_t(1) << 16) || nt == 1) { std::sort(first, last, cmp); return; }
    int chunks = 1;
    while (chunks * 2 <= nt) chunks *= 2;
    std::vector<int64_t> cut(size_t(chunks) + 1);
    for (int c = 0; c <= chunks; ++c) cut[size_t(c)] = n * c / chunks;
#pragma omp parallel for schedule(static, 1)
    for (int c = 0; c < chunks; ++c) std::sort(first + cut[size_t(c)], first + cut[size_t(c) + 1], cmp);
    for (int width = 1; width < chunks; width *= 2) {
#pragma omp parallel for schedule(static, 1)
        for (int c = 0; c < chunks; c += 2 * width)
            std::inplace_merge(first + cut[size_t(c)], first + cut[size_t(c + width)], first + cut[size_t(c + 2 * width)], cmp);
    }
}

void sorted_unique(std::vector<int32_t> &v) {
    parallel_sort(v.begin(), v.end(), [](int32_t a, int32_t b) { return a < b; });
    v.erase(std::unique(v.begin(), v.end()), v.end());
}

}  // namespace

int build_layout(HostLayout &L, int n_levels, const double *cell_width, double x0, double y0, int P,
                 const sg_patch *patches, int64_t n_patches, std::string &err, const uint8_t *cell_present) {
    if (!cell_width || !patches) { err = "null pointer argument"; return SG_ERR_ARG; }
    if (n_levels < 1 || n_levels > 24) { err = "n_levels must be in 1..24"; return SG_ERR_ARG; }
    if (P < 1 || P > 4096) { err = "patch_cells must be in 1..4096"; return SG_ERR_ARG; }
    if (n_patches < 1) { err = "n_patches must be >= 1"; return SG_ERR_ARG; }
    for (int l = 0; l < n_levels; ++l) {
        if (!(cell_width[l] > 0.0) || !std::isfinite(cell_width[l])) {
            err = "cell_width must be positive and finite"; return SG_ERR_ARG;
        }
        if (l > 0 && std::fabs(cell_width[l] * 2.0 - cell_width[l - 1]) > 1e-12 * cell_width[l - 1]) {
            err = fmt("cell_width[%lld] is not half of cell_width[%lld]", l, l - 1); return SG_ERR_ARG;
        }
    }
    // SG_TIME_CREATE (debugging aid): print the duration of the phases of the layout build to stderr
    const bool timing = std::getenv("SG_TIME_CREATE") != nullptr;
    auto t_last = std::chrono::steady_clock::now();
    auto lap = [&](const char *what) {
        if (!timing) return;
        const auto now = std::chrono::steady_clock::now();
        std::fprintf(stderr, "  build_layout %-22s %8.1f ms\n", what, std::chrono::duration<double, std::milli>(now - t_last).count());
        t_last = now;
    };
    const int64_t N = n_patches * int64_t(P) * P;
    if (N >= (int64_t(1) << 29)) { err = "too many cells (limit 2^29)"; return SG_ERR_LAYOUT; }

    L = HostLayout();
    L.n_levels = n_levels; L.P = P; L.x0 = x0; L.y0 = y0; L.N = N;
    L.unit = cell_width[n_levels - 1] / 2.0;
    L.patches.assign(patches, patches + n_patches);

    // ---- validation: on-lattice, in range, no duplicates, no patch inside another -------------
    std::unordered_set<uint64_t> leafset;
    leafset.reserve(size_t(n_patches) * 2);
    for (int64_t p = 0; p < n_patches; ++p) {
        const sg_patch &q = patches[p];
        if (q.level < 0 || q.level >= n_levels) {
            err = fmt("patch %lld: level %lld out of range", p, q.level); return SG_ERR_LAYOUT;
        }
        if (q.i0 < 0 || q.j0 < 0 || q.i0 % P || q.j0 % P) {
            err = fmt("patch %lld: (i0,j0)=(%lld,%lld) must be >= 0 and multiples of P", p, q.i0, q.j0);
            return SG_ERR_LAYOUT;
        }
        const int64_t cw = int64_t(2) << (n_levels - 1 - q.level);      // cell width in lattice units
        if ((int64_t(q.i0) + P) * cw > kMaxLattice || (int64_t(q.j0) + P) * cw > kMaxLattice) {
            err = fmt("patch %lld: lattice coordinate exceeds 2^26", p); return SG_ERR_LAYOUT;
        }
        if (!leafset.insert(patch_key(q.level, q.i0 / P, q.j0 / P)).second) {
            err = fmt("patch %lld: duplicate of an earlier patch", p); return SG_ERR_LAYOUT;
        }
    }
    auto covering_level = [&](int level, int64_t pi, int64_t pj) -> int {   // level of the leaf that
        for (int l = level; l >= 0; --l, pi >>= 1, pj >>= 1)                  // covers (pi,pj), looking
            if (leafset.count(patch_key(l, pi, pj))) return l;                // at `level` and coarser
        return -1;
    };
    if (!cell_present) {
        int64_t bad = -1;
        int unbalanced = 0;
#pragma omp parallel for schedule(static) reduction(max : bad) reduction(| : unbalanced)
        for (int64_t p = 0; p < n_patches; ++p) {                         // read-only look-ups in leafset
            const sg_patch &q = patches[p];
            const int64_t pi = q.i0 / P, pj = q.j0 / P;
            if (q.level > 0 && covering_level(q.level - 1, pi >> 1, pj >> 1) >= 0) bad = std::max(bad, p);
            if (q.level < 2) continue;                                    // a neighbour two levels coarser needs level >= 2
            for (int dj = -1; dj <= 1; ++dj)
                for (int di = -1; di <= 1; ++di) {
                    if ((!di && !dj) || pi + di < 0 || pj + dj < 0) continue;
                    const int c = covering_level(q.level, pi + di, pj + dj);
                    if (c >= 0 && c < q.level - 1) unbalanced |= 1;
                }
        }
        if (bad >= 0) {
            err = fmt("patch %lld (level %lld) lies inside a coarser leaf patch: leaves overlap", bad, patches[bad].level);
            return SG_ERR_LAYOUT;
        }
        L.balanced = unbalanced == 0;
    }

    lap("validation");
    // ---- targets ------------------------------------------------------------------------------
    L.tkx.resize(N); L.tky.resize(N);
    {
        int64_t c = 0;
        for (int64_t p = 0; p < n_patches; ++p) {
            const sg_patch &q = patches[p];
            const int32_t cw = int32_t(2) << (n_levels - 1 - q.level);
            for (int j = 0; j < P; ++j)
                for (int i = 0; i < P; ++i, ++c) {
                    L.tkx[c] = (q.i0 + i) * cw + cw / 2;
                    L.tky[c] = (q.j0 + j) * cw + cw / 2;
                }
        }
    }
    if (cell_present) {
        // holes of a padded layout: their results are discarded, but the direct kernels and finalise still run on them.
        // Give them the position of a real cell (the previous present one, the first for leading holes), so that no hole
        // can sit on a vertex (r = 0) or outside the range of the log tables; the lattice kernels take target positions
        // from the patch geometry and do not read these arrays.  The extent below still covers the blocks' full area.
        for (int64_t c = 0; c < N; ++c) L.extent = std::max(L.extent, std::max(L.tkx[c], L.tky[c]) + 1);
        int64_t first_present = 0;
        while (first_present < N && !cell_present[first_present]) ++first_present;
        if (first_present == N) { err = "no leaf cell present"; return SG_ERR_ARG; }
        int64_t last = first_present;
        for (int64_t c = 0; c < N; ++c) {
            if (cell_present[c]) { last = c; continue; }
            L.tkx[c] = L.tkx[last]; L.tky[c] = L.tky[last];
        }
    }
    L.tX = L.tkx; sorted_unique(L.tX);
    L.tY = L.tky; sorted_unique(L.tY);
    L.itx.resize(N); L.ity.resize(N);
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < N; ++c) {
        L.itx[c] = int32_t(std::lower_bound(L.tX.begin(), L.tX.end(), L.tkx[c]) - L.tX.begin());
        L.ity[c] = int32_t(std::lower_bound(L.tY.begin(), L.tY.end(), L.tky[c]) - L.tY.begin());
    }

    lap("targets");
    // ---- vertices: sort the 4N (corner key, cell, corner) records, merge equal keys ------------
    // corner id: 0 = NE (+), 1 = NW (-), 2 = SE (-), 3 = SW (+)
    struct Rec { uint64_t key; uint32_t cc; };
    std::vector<Rec> rec;
    rec.reserve(size_t(N) * 4);
    {
        int64_t c = 0;
        for (int64_t p = 0; p < n_patches; ++p) {
            const sg_patch &q = patches[p];
            const int32_t cw = int32_t(2) << (n_levels - 1 - q.level);
            for (int j = 0; j < P; ++j)
                for (int i = 0; i < P; ++i, ++c) {
                    if (cell_present && !cell_present[c]) continue;       // a hole of a padded layout: not a source
                    const uint64_t xl = uint64_t(q.i0 + i) * cw, xr = xl + cw;
                    const uint64_t yd = uint64_t(q.j0 + j) * cw, yu = yd + cw;
                    rec.push_back({(xr << 32) | yu, uint32_t(c << 2) | 0u});
                    rec.push_back({(xl << 32) | yu, uint32_t(c << 2) | 1u});
                    rec.push_back({(xr << 32) | yd, uint32_t(c << 2) | 2u});
                    rec.push_back({(xl << 32) | yd, uint32_t(c << 2) | 3u});
                }
        }
    }
    if (rec.empty()) { err = "no leaf cell present"; return SG_ERR_ARG; }
    lap("corner records");
    parallel_sort(rec.begin(), rec.end(), [](const Rec &a, const Rec &b) {
        return a.key != b.key ? a.key < b.key : a.cc < b.cc;
    });
    lap("record sort");
    L.vkx.reserve(N + N / 8); L.vky.reserve(N + N / 8); L.adj.reserve(4 * (N + N / 8));
    for (size_t r = 0; r < rec.size();) {
        size_t e = r;
        while (e < rec.size() && rec[e].key == rec[r].key) ++e;
        if (e - r > 4) {   // cannot happen for disjoint rectangles; a second line of defence
            err = "a vertex is shared by more than four cells: leaves overlap"; return SG_ERR_LAYOUT;
        }
        L.vkx.push_back(int32_t(rec[r].key >> 32));
        L.vky.push_back(int32_t(rec[r].key & 0xffffffffu));
        for (size_t k = 0; k < 4; ++k) {
            if (r + k < e) {
                const uint32_t cc = rec[r + k].cc;
                // (cell << 2) | corner; corner 0 = NE (+), 1 = NW (-), 2 = SE (-), 3 = SW (+)
                L.adj.push_back(int32_t(cc));
            } else {
                L.adj.push_back(-1);
            }
        }
        r = e;
    }
    L.Nv = int64_t(L.vkx.size());
    rec.clear(); rec.shrink_to_fit();

    lap("vertex merge");
    // columns: vertices are already sorted by (kx, ky)
    for (int64_t v = 0; v < L.Nv; ++v) {
        if (v == 0 || L.vkx[v] != L.vkx[v - 1]) { L.colX.push_back(L.vkx[v]); L.colstart.push_back(int32_t(v)); }
        L.extent = std::max(L.extent, std::max(L.vkx[v], L.vky[v]));
    }
    L.colstart.push_back(int32_t(L.Nv));
    // rows: permutation sorted by (ky, kx)
    L.rowperm.resize(L.Nv);
    for (int64_t v = 0; v < L.Nv; ++v) L.rowperm[v] = int32_t(v);
    parallel_sort(L.rowperm.begin(), L.rowperm.end(), [&](int32_t a, int32_t b) {
        return L.vky[a] != L.vky[b] ? L.vky[a] < L.vky[b] : L.vkx[a] < L.vkx[b];
    });
    for (int64_t r = 0; r < L.Nv; ++r) {
        const int32_t v = L.rowperm[r];
        if (r == 0 || L.vky[v] != L.vky[L.rowperm[r - 1]]) { L.rowY.push_back(L.vky[v]); L.rowstart.push_back(int32_t(r)); }
    }
    L.rowstart.push_back(int32_t(L.Nv));

    lap("columns and rows");
    // chunks: cut every column into runs of kChunk vertices; pad the last run of a column with -1
    for (size_t c = 0; c + 1 < L.colstart.size(); ++c)
        for (int32_t s = L.colstart[c]; s < L.colstart[c + 1]; s += kChunk) {
            L.chunk_x.push_back(L.colX[c]);
            for (int j = 0; j < kChunk; ++j)
                L.slot_vertex.push_back(s + j < L.colstart[c + 1] ? s + j : -1);
        }
    while (L.chunk_x.size() % kChunksPerTile) {          // whole tiles only
        L.chunk_x.push_back(L.chunk_x[0]);
        for (int j = 0; j < kChunk; ++j) L.slot_vertex.push_back(-1);
    }

    // a target can never sit on a vertex (it is strictly inside its own leaf and leaves are disjoint):
    // cheap necessary check on the lattice -- both coordinates of a target being vertex coordinates is
    // only possible if some vertex lies inside a leaf, i.e. an overlap the patch test did not see.
    {
        // the vertices are sorted by (kx, ky): look the target's position up in its column
        int64_t bad = -1;
#pragma omp parallel for schedule(static) reduction(max : bad)
        for (int64_t c = 0; c < N; ++c) {
            if (cell_present && !cell_present[c]) continue;
            const auto cx = std::lower_bound(L.colX.begin(), L.colX.end(), L.tkx[c]);
            if (cx == L.colX.end() || *cx != L.tkx[c]) continue;
            const size_t col = size_t(cx - L.colX.begin());
            const auto b0 = L.vky.begin() + L.colstart[col], b1 = L.vky.begin() + L.colstart[col + 1];
            if (std::binary_search(b0, b1, L.tky[c])) bad = std::max(bad, c);
        }
        if (bad >= 0) {
            err = fmt("cell %lld: centre coincides with a vertex of another leaf: leaves overlap", bad);
            return SG_ERR_LAYOUT;
        }
    }
    lap("chunks and vertex check");
    return SG_OK;
}

}  // namespace sg
