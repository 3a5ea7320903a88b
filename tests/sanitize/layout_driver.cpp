// layout_driver.cpp -- TEST CODE: runs the library's host layout builder (paper_2001_02765_b200/csrc/sg_layout.cpp,
// CUDA-free) under AddressSanitizer + UndefinedBehaviorSanitizer (tests/test_host_sanitizers.py builds and runs it).
// stdin: n_levels P n_patches, then n_levels cell widths, then n_patches rows "level i0 j0".
// stdout: "rc N Nv nX nY ntX ntY balanced extent checksum" (checksum over every array the builder fills), or
// "rc message" for a refused layout.  A sanitizer finding aborts with a non-zero exit status.
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../../paper_2001_02765_b200/csrc/sg_layout.h"

static uint64_t mix(uint64_t h, const std::vector<int32_t> &v) {
    for (int32_t x : v) h = (h ^ uint64_t(uint32_t(x))) * 1099511628211ull;
    return h;
}

int main() {
    int n_levels = 0, P = 0;
    long long n_patches = 0;
    if (std::scanf("%d %d %lld", &n_levels, &P, &n_patches) != 3 || n_levels < 0 || n_levels > 64 || n_patches < 0) return 2;
    std::vector<double> cw(size_t(n_levels), 0.0);
    for (double &w : cw) if (std::scanf("%lf", &w) != 1) return 2;
    std::vector<sg_patch> patches(size_t(n_patches), sg_patch{0, 0, 0});
    for (sg_patch &p : patches) if (std::scanf("%d %d %d", &p.level, &p.i0, &p.j0) != 3) return 2;
    sg::HostLayout h;
    std::string err;
    const int rc = sg::build_layout(h, n_levels, cw.data(), -1.0, -1.0, P, patches.data(), n_patches, err);
    if (rc != SG_OK) { std::printf("%d %s\n", rc, err.c_str()); return 0; }
    uint64_t sum = 1469598103934665603ull;
    for (const std::vector<int32_t> *v : {&h.tkx, &h.tky, &h.itx, &h.ity, &h.tX, &h.tY, &h.vkx, &h.vky, &h.adj, &h.colX,
                                          &h.colstart, &h.rowY, &h.rowstart, &h.rowperm, &h.chunk_x, &h.slot_vertex})
        sum = mix(sum, *v);
    std::printf("%d %lld %lld %zu %zu %zu %zu %d %d %llu\n", rc, (long long)h.N, (long long)h.Nv, h.colX.size(),
                h.rowY.size(), h.tX.size(), h.tY.size(), int(h.balanced), int(h.extent), (unsigned long long)sum);
    return 0;
}
