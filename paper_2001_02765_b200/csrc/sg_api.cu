// sg_api.cu -- the C ABI of include/sg_disk.h: context ownership, uploads, launch planning.
#include <algorithm>
#include <climits>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <string>
#include <vector>

#include "sg_kernels.cuh"
#include "sg_kernels_lin.cuh"
#include "sg_kernels_patch.cuh"
#include "sg_kernels_lattice.cuh"
#include "sg_layout.h"
#include "../../include/sg_disk_diag.h"

using namespace sg;

struct sg_ctx {
    HostLayout host;
    DevLayout dev;
    int device = -1;             // < 0: host-only context (layout queries work, compute calls fail)
    int sm_count = 148;
    bool density_set = false;
    bool linear = false;         // last density call carried slopes (sg_set_density_linear)
    LinArrays lin;
    PatchArrays patch;           // lattice-offset reuse path (P = 8 or 16)
    std::vector<PatchInfo> patch_info;      // host side of the lattice path (build_patch_plan)
    std::vector<PatchLevel> patch_levels;
    std::vector<int32_t> patch_pmap;
    std::vector<int32_t> patch_flags;       // per patch: bit 0 row P / bit 1 column P of its vertex lattice carries owned vertices
    bool patch_plan_ok = false;             // P == 16 and the per-level patch maps fit
    std::vector<PatchGroup> patch_groups;   // the three group lists back to back (offset_group_list)
    int patch_n_groups[3] = {0, 0, 0};      // sizes of the three group lists (offset_group_list)
    bool use_patch = false;      // sg_set_interaction_mode
    bool neutral_weights = false; // SG_LATTICE_NEUTRAL_WEIGHTS at sg_create: own-cell per-patch weights (sg_kernels_patch.cu)
    // environment switches, latched at sg_create (sg_force reads no environment)
    bool poison_partials = false;     // SG_POISON_PARTIALS: NaN-fill the partial sums before every sg_force (test aid)
    bool debug_sync = false;          // SG_DEBUG_SYNC: synchronise after every pair-class launch (debugging aid)
    bool owned_slope_weights = false; // SG_LATTICE_OWNED_SLOPE_WEIGHTS: round-2 owned weights on the lattice slope path
    bool force_incta = false;    // SG_MODE_LATTICE_INCTA: offset tables built inside the CTAs even if the lattices exist
    LatticeArrays lat;           // precomputed function lattices of the pair classes (sg_kernels_lattice.cu)
    std::vector<FnLattice> lat_meta;        // host copy, [n_levels * kOffClasses]
    int64_t lat_entries = 0;                // entries per plane; 0: no plan (P != 16) or over the memory budget
    // regrouped lattice mode (P = 1, 2 or 4, e.g. the paper's zone-wise quadtrees): the leaves are packed into padded
    // 16 x 16 blocks of an inner context that runs the lattice kernels; cell data is permuted in and out
    sg_ctx *inner = nullptr;
    int32_t *rg_map = nullptr, *rg_inv = nullptr;       // device: caller cell -> inner cell; inner cell -> caller cell or -1
    std::vector<int32_t> rg_map_host;                   // host copy of rg_map (sg_set_target_range -> inner block range)
    int64_t rg_first = 0;                               // first inner cell of the inner context's target range
    double *rg_in[3] = {nullptr, nullptr, nullptr};     // sigma, dx, dy in inner cell order
    double *rg_f[2] = {nullptr, nullptr};               // Fx, Fy in inner cell order
    int64_t first = 0, count = 0;
    int64_t dev_bytes = 0;
    std::vector<void *> allocs;
    std::string err;
    // kernel timing ring (sg_set_kernel_timing)
    bool timing = false;
    int64_t timed_calls = 0;
    std::vector<cudaEvent_t> ev0, ev1;
    // lattice mode: the pair-class kernels of one sg_force run concurrently (fork / join around the caller's stream),
    // so that the tail of one class overlaps the start of the next
    std::vector<cudaStream_t> side;
    cudaEvent_t fork_ev = nullptr;
    std::vector<cudaEvent_t> join_ev;
};

constexpr int kTimingRing = 64;

static thread_local std::string g_create_error;

namespace {

#define SG_CUDA(ctx, call)                                                              \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess) {                                                        \
            (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e_);            \
            return SG_ERR_CUDA;                                                         \
        }                                                                               \
    } while (0)

// The library works on the context's device and leaves the caller's current device as it found it.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        err = cudaSetDevice(device);
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

template <class T>
int dev_alloc(sg_ctx *c, T **p, int64_t n) {
    const size_t bytes = size_t(std::max<int64_t>(n, 1)) * sizeof(T);
    SG_CUDA(c, cudaMalloc(reinterpret_cast<void **>(p), bytes));
    c->allocs.push_back(*p);
    c->dev_bytes += int64_t(bytes);
    return SG_OK;
}

template <class T>
int upload(sg_ctx *c, T **p, const std::vector<T> &h) {
    int rc = dev_alloc(c, p, int64_t(h.size()));
    if (rc) return rc;
    if (!h.empty()) SG_CUDA(c, cudaMemcpy(*p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    return SG_OK;
}

// Work items = target blocks x source splits, pulled from an atomic queue by a persistent grid of
// 2 CTAs per SM (about 16 items per CTA).  Pick the split count that keeps the last round fullest.
ForcePlan make_plan(const sg_ctx *c, bool linear) {
    ForcePlan p;
    p.first = c->first; p.count = c->count;
    p.smem = linear ? interaction_lin_smem_bytes(c->dev.tab_entries) : interaction_smem_bytes(c->dev.tab_entries);
    if (p.count == 0 || c->dev.n_tiles == 0) return p;                 // nothing to do / host-only context
    p.T = linear ? lin_targets_per_thread() : (p.count > 16384 ? 4 : 1);
    const int64_t per_block = int64_t(kThreads) * p.T;
    p.n_tblocks = int((p.count + per_block - 1) / per_block);
    const int slots = c->sm_count * 2;
    const int n_tiles = c->dev.n_tiles;
    int best_split = 1; double best_eff = -1.0;
    const int want = std::max(1, std::min(n_tiles, (16 * slots + p.n_tblocks - 1) / p.n_tblocks));
    for (int s = want; s <= std::min(n_tiles, want + 12); ++s) {
        const int tps = (n_tiles + s - 1) / s, ns = (n_tiles + tps - 1) / tps;
        const int64_t items = int64_t(ns) * p.n_tblocks;
        const int64_t rounds = (items + slots - 1) / slots;
        // cost ~ rounds * tiles per item; ideal ~ items * tps / slots
        const double eff = double(n_tiles) * p.n_tblocks / (double(rounds) * slots * tps);
        if (eff > best_eff + 1e-9) { best_eff = eff; best_split = ns; }
    }
    p.tiles_per_split = (n_tiles + best_split - 1) / best_split;
    p.n_split = (n_tiles + p.tiles_per_split - 1) / p.tiles_per_split;
    const int64_t items = int64_t(p.n_split) * p.n_tblocks;
    p.grid = int(std::min<int64_t>(items, slots));
    return p;
}

// The partial-sum buffer [n_split][2][count].  It is sized by reserve_partials() from the host-synchronous calls that
// change the plan (sg_create, sg_set_interaction_mode, sg_set_target_range, the first sg_set_density_linear), so that
// sg_force itself never allocates or synchronises (CUDA-graph capture).  grow_partials is the fallback for
// a plan nobody announced: refused during stream capture (a captured graph would keep the freed pointer).
int grow_partials(sg_ctx *c, int64_t need, cudaStream_t capturing_on) {
    if (need <= c->dev.part_capacity) return SG_OK;
    if (capturing_on != nullptr || c->dev.part) {
        cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(capturing_on, &st) == cudaSuccess && st != cudaStreamCaptureStatusNone) {
            c->err = "sg_force during stream capture needs a larger partial-sum buffer: call sg_force once with the same "
                     "mode and target range before capturing";
            return SG_ERR_STATE;
        }
    }
    if (c->dev.part) {
        SG_CUDA(c, cudaDeviceSynchronize());
        cudaFree(c->dev.part);
        c->allocs.erase(std::remove(c->allocs.begin(), c->allocs.end(), (void *)c->dev.part), c->allocs.end());
        c->dev_bytes -= c->dev.part_capacity * 8;
        c->dev.part = nullptr; c->dev.part_capacity = 0;
    }
    int rc = dev_alloc(c, &c->dev.part, need);
    if (rc) return rc;
    c->dev.part_capacity = need;
    return SG_OK;
}

// Lattice-offset path: one work item = (target patch, split of the source patch list).
PatchPlan make_patch_plan(const sg_ctx *c) {
    PatchPlan pp;
    const PatchArrays &pa = c->patch;
    const int64_t PP = int64_t(pa.P) * pa.P;
    pp.smem = patch_smem_bytes(pa.P, c->dev.tab_entries);
    if (c->count == 0) return pp;
    pp.first_patch = int(c->first / PP);
    pp.n_tpatches = int((c->first + c->count - 1) / PP) - pp.first_patch + 1;
    const int slots = c->sm_count * (pa.P == 16 ? 2 : 4);
    // The split of the source list is that of the FULL evaluation whatever the target range: a slice then adds the
    // same partial sums in the same order as the unsharded call, so rank slices are bit-identical to it.
    int want = (8 * slots + pa.n_patches - 1) / std::max(1, pa.n_patches);  // about 8 items per resident CTA (full range)
    want = std::max(1, std::min(want, std::max(1, pa.n_patches / 4)));     // but >= 4 source patches per item
    pp.patches_per_split = (pa.n_patches + want - 1) / want;
    pp.n_split = (pa.n_patches + pp.patches_per_split - 1) / pp.patches_per_split;
    pp.grid = int(std::min<int64_t>(int64_t(pp.n_split) * pp.n_tpatches, slots));
    return pp;
}

// Blocked kernels (patch pairs at most two levels apart): one work item = (group of <= 8 target patches, split of the
// group's offset box), per pair class.
int offset_classes(const OffsetPlan &po) {
    int n = 0;
    for (int v = 0; v < kOffClasses; ++v) n += int(po.variant[v]);
    return n;
}

OffsetPlan make_offset_plan(const sg_ctx *c, const PatchPlan &pp) {
    OffsetPlan po;
    if (c->count == 0) return po;
    for (int q = 0; q < 3; ++q) po.n_groups[q] = c->patch_n_groups[q];
    po.first_patch = pp.first_patch;
    po.last_patch = pp.first_patch + pp.n_tpatches - 1;
    bool any[kOffClasses] = {false, false, false, false, false};
    for (size_t i = 0; i < c->patch_groups.size(); ++i) {
        const PatchGroup &g = c->patch_groups[i];
        for (int v = 0; v < kOffClasses; ++v) any[v] = any[v] || g.box[v][1] > 0;
        if (g.pmax < po.first_patch || g.pmin > po.last_patch) continue;
        for (int v = 0; v < kOffClasses; ++v) po.variant[v] = po.variant[v] || g.box[v][1] > 0;
    }
    // n_split is chosen for the FULL evaluation (all groups, all N targets) whatever the target range: every group's
    // offset list is then cut the same way in a slice as in the unsharded call and the partial sums are added in the
    // same order, so rank slices (sg_set_target_range, regrouped layouts included) are bit-identical to it.  A rank
    // of an N-GPU run gets 1/N of the ~16 items per resident CTA.
    const int touched = po.n_groups[0];
    int64_t classes = 0;
    for (int v = 0; v < kOffClasses; ++v) classes += any[v] ? 1 : 0;
    classes = std::max<int64_t>(1, classes);
    // splits of every group's offset list: about 16 work items per resident CTA (items of sparse levels differ a lot in
    // weight; the queue is dynamic), and among the next few counts the one whose item count fills the last wave of the
    // persistent grid best (on a uniform level all items weigh the same: 512 groups x 4 splits ran 13 % faster than
    // x 3, and x 6 slower than x 4)
    const int slots = c->sm_count * 2;
    const int64_t mem_cap = std::max<int64_t>(1, (int64_t(1) << 30) / (classes * 16 * std::max<int64_t>(1, c->host.N)));
    const int cap = int(std::min<int64_t>(64, mem_cap));              // partial sums stay below 1 GiB
    const int want = std::max(1, std::min(cap, (16 * slots + touched - 1) / std::max(1, touched)));
    double best = -1.0;
    for (int sp = want; sp <= std::min(cap, want + 8); ++sp) {
        const int64_t items = int64_t(sp) * std::max(1, touched), waves = (items + slots - 1) / slots;
        const double eff = double(items) / double(waves * slots);
        if (eff > best + 1e-9) { best = eff; po.n_split = sp; }
    }
    return po;
}

// P = 16: the register-blocked offset-table kernels for pairs <= 2 levels apart (measured faster than the generic
// kernel at every size, cfg 1: 25 vs 37 us, cfg 3: 2.6 vs 4.0 ms), the generic kernel only for the direct sum of
// the pairs >= 3 levels apart; P = 8: generic kernel (tables for pairs <= 1 level apart, direct sum beyond)
bool use_blocked(const sg_ctx *c, const PatchPlan &) { return c->patch.blocked; }

// Function lattices (sg_kernels_lattice.cuh): extents per (target level, pair class) = the union of the offset boxes
// of the level's target groups.  Host only; returns the entries per plane (0 if the plan does not exist).
int64_t plan_fn_lattices(sg_ctx *c) {
    c->lat_meta.assign(size_t(c->host.n_levels) * kOffClasses, FnLattice{0, 0, 0, 0, 0, 0, 0, 0});
    if (!c->patch_plan_ok) return 0;
    const int M_of[kOffClasses] = {32, 48, 47, 80, 77}, TROW_of[kOffClasses] = {33, 49, 49, 81, 79};
    const int ROWS_of[kOffClasses] = {32, 48, 48, 80, 80};
    struct Ext { int64_t xlo = INT64_MAX, xhi = INT64_MIN, ylo = INT64_MAX, yhi = INT64_MIN; };
    std::vector<Ext> ext(c->lat_meta.size());
    for (const PatchGroup &g : c->patch_groups)
        for (int v = 0; v < kOffClasses; ++v) {
            if (g.box[v][1] <= 0 || g.box[v][3] <= 0) continue;
            const int step = (v == kOffCoarserSrc) ? 2 : (v == kOffCoarserSrc4) ? 4 : 1;
            Ext &e = ext[size_t(g.level) * kOffClasses + v];
            e.xlo = std::min<int64_t>(e.xlo, g.box[v][0]);
            e.xhi = std::max<int64_t>(e.xhi, g.box[v][0] + int64_t(step) * (g.box[v][1] - 1));
            e.ylo = std::min<int64_t>(e.ylo, g.box[v][2]);
            e.yhi = std::max<int64_t>(e.yhi, g.box[v][2] + int64_t(step) * (g.box[v][3] - 1));
        }
    int64_t total = 0;
    for (size_t k = 0; k < ext.size(); ++k) {
        const Ext &e = ext[k];
        if (e.xlo > e.xhi) continue;
        const int v = int(k % kOffClasses);
        const int64_t ncols = 16 * (e.xhi - e.xlo) + TROW_of[v], nrows = 16 * (e.yhi - e.ylo) + std::max(ROWS_of[v], M_of[v]);
        if (ncols > INT32_MAX / 2 || nrows > INT32_MAX / 2) return 0;
        FnLattice &m = c->lat_meta[k];
        m.base = total; m.ncols = int32_t(ncols); m.nrows = int32_t(nrows);
        m.cmin = int32_t(16 * e.xlo); m.rmin = int32_t(16 * e.ylo); m.present = 1;
        total += ncols * nrows;
        total = (total + 7) & ~int64_t(7);                       // every lattice starts on a 128-byte boundary
    }
    return total;
}

// Memory budget of the function lattices (all planes): SG_LATTICE_TABLE_MIB, default a quarter of the device's memory
// (45 GB on a B200) or what is free right now, whichever is less.  Over it, lattice mode builds its offset tables
// inside the CTAs (patch_offset_kernel) and the slope path stays direct.
int64_t fn_budget_bytes() {
    if (const char *e = std::getenv("SG_LATTICE_TABLE_MIB")) return std::max<int64_t>(0, std::atoll(e)) << 20;
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) return int64_t(16) << 30;
    return int64_t(std::min(free_b, total_b / 4));
}

// Build (or extend to the slope planes) the function lattices.  Host-synchronous; no-op when they exist already.
// Never fails for lack of memory: over the budget, or when the allocation itself fails, whatever lattice exists stays
// in place (a 1-plane lattice keeps serving the zeroth-order path) and the caller's path falls back as sg_disk.h says
// (in-CTA tables / direct slope kernel).  The new buffer is allocated BEFORE the old one is released.
int ensure_fn_lattices(sg_ctx *c, int n_planes) {
    if (c->device < 0 || !c->patch.blocked || c->lat_entries == 0) return SG_OK;
    if (c->lat.n_planes_built >= n_planes) return SG_OK;
    const int64_t need = c->lat_entries * 16 * n_planes;
    if (need > fn_budget_bytes()) return SG_OK;                                // stays on the fallback
    SG_CUDA(c, cudaDeviceSynchronize());
    void *fresh = nullptr;
    if (cudaMalloc(&fresh, size_t(need)) != cudaSuccess) {
        cudaGetLastError();                                                    // not sticky: clear it, keep what exists
        return SG_OK;
    }
    if (c->lat.fn) {
        cudaFree(c->lat.fn);
        c->allocs.erase(std::remove(c->allocs.begin(), c->allocs.end(), (void *)c->lat.fn), c->allocs.end());
        c->dev_bytes -= c->lat_entries * 16 * c->lat.n_planes_built;
        c->lat.n_planes_built = 0; c->lat.ready = false;
    }
    c->lat.fn = static_cast<decltype(c->lat.fn)>(fresh);
    c->allocs.push_back(fresh);
    c->dev_bytes += need;
    int rc;
    for (FnLattice &m : c->lat_meta) m.plane_stride = c->lat_entries;
    if (!c->lat.meta) {
        if ((rc = upload(c, &c->lat.meta, c->lat_meta))) return rc;
        SG_CUDA(c, configure_lattice_kernels());
    } else {
        SG_CUDA(c, cudaMemcpy(c->lat.meta, c->lat_meta.data(), c->lat_meta.size() * sizeof(FnLattice), cudaMemcpyHostToDevice));
    }
    c->lat.fn_entries = c->lat_entries;
    launch_build_fn_lattices(c->lat, c->lat_meta.data(), c->patch_levels.data(), c->host.n_levels, c->dev, 0, n_planes, nullptr);
    SG_CUDA(c, cudaGetLastError());
    SG_CUDA(c, cudaDeviceSynchronize());
    c->lat.n_planes_built = n_planes;
    c->lat.ready = true;
    return SG_OK;
}

// Source vertices the lattice kernels run through per target: (P + 1)^2 per patch in the generic kernel; in the
// offset-table kernels (P = 16) vertex row 16 / column 16 of a patch only where it owns vertices there (pflags).
double executed_patch_vertices(const sg_ctx *c, bool all_vertices = false) {
    const int P = c->host.P;
    if (all_vertices || c->patch_flags.size() != c->host.patches.size()) return double(c->host.patches.size()) * double((P + 1) * (P + 1));
    double n = 0.0;
    for (int32_t f : c->patch_flags) n += double(P + (f & 1)) * double(P + ((f >> 1) & 1));
    return n;
}

// Everything one sg_force launches with the current mode and target range.
struct StepPlan {
    ForcePlan p;                           // direct / slope kernel, and the finalise kernel (p.n_split partial sums per target)
    PatchPlan pp;                          // generic kernel: everything (P = 8) or the pairs >= 3 levels apart (P = 16)
    OffsetPlan po;                         // blocked kernels: pairs at most two levels apart
    bool by_patch = false, blocked = false, far = true;
    bool fn = false;                       // blocked kernels read precomputed function lattices (lattice_corr_kernel)
    int n_planes = 1;                      // 3: slope path in lattice mode
    int64_t partials() const { return int64_t(p.n_split) * 2 * p.count; }
};

StepPlan make_step_plan(const sg_ctx *c, bool linear) {
    StepPlan sp;
    sp.p = make_plan(c, linear);
    // the slope path runs in lattice mode only through the function lattices (three planes)
    const bool lin_lattice = c->patch.blocked && !c->force_incta && c->lat.n_planes_built >= kFnPlanesLin;
    // (a regrouped context, c->inner, hands lattice mode to its inner context and plans only its own direct kernels)
    sp.by_patch = c->use_patch && c->patch.enabled && !c->inner && (!linear || lin_lattice);
    sp.n_planes = linear ? kFnPlanesLin : 1;
    if (sp.by_patch) {
        sp.pp = make_patch_plan(c);
        sp.blocked = use_blocked(c, sp.pp);
        sp.fn = sp.blocked && c->lat.ready && !c->force_incta;
        if (sp.blocked) {
            sp.po = make_offset_plan(c, sp.pp);
            sp.far = c->host.n_levels > 3;                     // pairs >= 3 levels apart exist only then
            sp.p.n_split = offset_classes(sp.po) * sp.po.n_split + (sp.far ? sp.pp.n_split : 0);
        } else {
            sp.p.n_split = sp.pp.n_split;
        }
    }
    return sp;
}

// Called from the host-synchronous calls that change the plan: the buffer fits the zeroth-order and the slope path.
int reserve_partials(sg_ctx *c) {
    if (c->device < 0) return SG_OK;
    const int64_t need = std::max(make_step_plan(c, false).partials(), make_step_plan(c, true).partials());
    return grow_partials(c, need, nullptr);
}

// Host-side plan of the offset-table kernels (P = 16): per-patch lattice info, per-level dense patch maps, target
// groups with their offset boxes per pair class.  No CUDA: also built for host-only contexts (sg_lattice_plan_check).
bool build_patch_plan(sg_ctx *c) {
    const HostLayout &h = c->host;
    std::vector<PatchInfo> &info = c->patch_info;
    info.resize(h.patches.size());
    for (size_t p = 0; p < info.size(); ++p) {
        const int32_t cw = int32_t(2) << (h.n_levels - 1 - h.patches[p].level);
        info[p] = PatchInfo{h.patches[p].i0 * cw, h.patches[p].j0 * cw, cw, h.patches[p].level};
    }
    if (h.P != 16) return false;
    {
        // per level: dense map patch position -> patch index; groups of <= 8 consecutive patches with the box of
        // patch offsets that can reach a source patch of the same level (patch_offset_kernel)
        std::vector<PatchLevel> &lev = c->patch_levels;
        lev.assign(size_t(h.n_levels), PatchLevel{0, 0, 0, 0, 0, 0, 0, 0});
        std::vector<int32_t> &pmap = c->patch_pmap;
        pmap.clear();
        std::vector<PatchGroup> &groups = c->patch_groups;
        groups.clear();
        int64_t map_total = 0;
        bool ok = true;
        // the patch list may come in any order: collect the patches of every level (PatchLevel.p0 is unused then)
        std::vector<std::vector<int32_t>> of_level(size_t(h.n_levels));
        for (size_t p = 0; p < info.size(); ++p) of_level[size_t(h.patches[p].level)].push_back(int32_t(p));
        for (int L = 0; L < h.n_levels && ok; ++L) {
            const std::vector<int32_t> &m = of_level[size_t(L)];
            if (m.empty()) continue;
            int imin = INT32_MAX, imax = INT32_MIN, jmin = INT32_MAX, jmax = INT32_MIN;
            for (int32_t r : m) {
                imin = std::min(imin, h.patches[size_t(r)].i0 / h.P); imax = std::max(imax, h.patches[size_t(r)].i0 / h.P);
                jmin = std::min(jmin, h.patches[size_t(r)].j0 / h.P); jmax = std::max(jmax, h.patches[size_t(r)].j0 / h.P);
            }
            PatchLevel &l = lev[size_t(L)];
            l = PatchLevel{m.front(), int32_t(m.size()), imin, jmin, imax - imin + 1, jmax - jmin + 1,
                           int32_t(map_total), info[size_t(m.front())].cw};
            map_total += int64_t(l.npx) * l.npy;
            if (map_total > (int64_t(1) << 26)) { ok = false; break; }
            pmap.resize(size_t(map_total), -1);
            for (int32_t r : m)
                pmap[size_t(l.map_off) + size_t(h.patches[size_t(r)].j0 / h.P - jmin) * l.npx + (h.patches[size_t(r)].i0 / h.P - imin)] = r;
        }
        // groups of 8 target patches in sorted order with their offset boxes.  List 0 (any patches of a level) serves
        // the pair classes "same level" and "finer source"; lists 1 / 2 (patches of one residue class of (pi, pj)
        // mod F = 2 / 4) serve the sources F times coarser, where A + d must be a multiple of F for the whole group.
        std::vector<PatchGroup> glist[3];
        auto level_ok = [&](int L) { return L >= 0 && L < h.n_levels && lev[size_t(L)].n > 0; };
        for (int L = 0; L < h.n_levels && ok; ++L) {
            const PatchLevel &l = lev[size_t(L)];
            if (l.n == 0) continue;
            for (int list = 0; list < 3 && ok; ++list) {
                const int F = 1 << list;                                // residue classes mod F
                // a level without a source level `list` levels up still gets its groups in that list (with an empty
                // box): every launched class must write its partial-sum slots for EVERY target patch
                const bool has_src = list == 0 || level_ok(L - list);
                for (int cls = 0; cls < F * F && ok; ++cls) {
                    const int cx = cls % F, cy = cls / F;
                    std::vector<int32_t> members;
                    for (int32_t r : of_level[size_t(L)])
                        if ((h.patches[size_t(r)].i0 / h.P) % F == cx && (h.patches[size_t(r)].j0 / h.P) % F == cy)
                            members.push_back(r);
                    // 8 consecutive members should be a compact 4 x 2 block of the class's own patch lattice (pitch F):
                    // the offset box of a group grows with the group's spread, and every offset costs one table
                    std::stable_sort(members.begin(), members.end(), [&](int32_t a, int32_t b) {
                        const sg_patch &pa_ = h.patches[size_t(a)], &pb_ = h.patches[size_t(b)];
                        const int ai = pa_.i0 / h.P / F, aj = pa_.j0 / h.P / F, bi = pb_.i0 / h.P / F, bj = pb_.j0 / h.P / F;
                        if ((aj >> 1) != (bj >> 1)) return (aj >> 1) < (bj >> 1);
                        if ((ai >> 2) != (bi >> 2)) return (ai >> 2) < (bi >> 2);
                        if (aj != bj) return aj < bj;
                        return ai < bi;
                    });
                    for (size_t m0 = 0; m0 < members.size() && ok; m0 += 8) {
                        PatchGroup gr;
                        std::memset(&gr, 0, sizeof gr);
                        gr.level = L;
                        gr.n = int(std::min<size_t>(8, members.size() - m0));
                        int64_t gimin = INT32_MAX, gimax = INT32_MIN, gjmin = INT32_MAX, gjmax = INT32_MIN;
                        gr.pmin = INT32_MAX; gr.pmax = INT32_MIN;
                        for (int w = 0; w < 8; ++w) {
                            // warp w runs on SM sub-partition w % 4: rotate the block's second row by one so that the two
                            // patches of a block column (idle together at the edge of the level) sit on different ones
                            const int src = (gr.n == 8 && w >= 4) ? 4 + ((w - 4 + 3) & 3) : w;
                            gr.patch[w] = w < gr.n ? members[m0 + size_t(src)] : -1;
                            if (w >= gr.n) continue;
                            const sg_patch &q = h.patches[size_t(gr.patch[w])];
                            gimin = std::min<int64_t>(gimin, q.i0 / h.P); gimax = std::max<int64_t>(gimax, q.i0 / h.P);
                            gjmin = std::min<int64_t>(gjmin, q.j0 / h.P); gjmax = std::max<int64_t>(gjmax, q.j0 / h.P);
                            gr.pmin = std::min(gr.pmin, gr.patch[w]); gr.pmax = std::max(gr.pmax, gr.patch[w]);
                        }
                        // d ranges over [lo, hi] per axis in steps of `step`, starting where A + d is a multiple of it
                        auto set_box = [&](int v, int64_t lox, int64_t hix, int64_t loy, int64_t hiy, int step) {
                            while (((lox + cx) % step + step) % step != 0) ++lox;
                            while (((loy + cy) % step + step) % step != 0) ++loy;
                            const int64_t nx = hix >= lox ? (hix - lox) / step + 1 : 0, ny = hiy >= loy ? (hiy - loy) / step + 1 : 0;
                            if (nx * ny > (int64_t(1) << 30)) { ok = false; return; }
                            gr.box[v][0] = int32_t(lox); gr.box[v][1] = int32_t(nx * ny > 0 ? nx : 0);
                            gr.box[v][2] = int32_t(loy); gr.box[v][3] = int32_t(nx * ny > 0 ? ny : 0);
                        };
                        auto hi_i = [](const PatchLevel &q) { return int64_t(q.pimin) + q.npx - 1; };
                        auto hi_j = [](const PatchLevel &q) { return int64_t(q.pjmin) + q.npy - 1; };
                        if (list == 0) {
                            set_box(kOffSame, l.pimin - gimax, hi_i(l) - gimin, l.pjmin - gjmax, hi_j(l) - gjmin, 1);
                            for (int dl = 1; dl <= 2; ++dl) {            // source patch F A + d inside the finer level's box
                                if (!level_ok(L + dl)) continue;
                                const PatchLevel &f0 = lev[size_t(L + dl)];
                                const int64_t Ff = 1 << dl;
                                set_box(dl == 1 ? kOffFinerSrc : kOffFinerSrc4, f0.pimin - Ff * gimax, hi_i(f0) - Ff * gimin,
                                        f0.pjmin - Ff * gjmax, hi_j(f0) - Ff * gjmin, 1);
                            }
                        } else if (has_src) {                            // source patch (A + d) / F inside the coarser level's box
                            const PatchLevel &c0 = lev[size_t(L - list)];
                            set_box(list == 1 ? kOffCoarserSrc : kOffCoarserSrc4, F * int64_t(c0.pimin) - gimax, F * hi_i(c0) - gimin,
                                    F * int64_t(c0.pjmin) - gjmax, F * hi_j(c0) - gjmin, F);
                        }
                        glist[list].push_back(gr);
                    }
                }
            }
        }
        groups.clear();
        for (int list = 0; list < 3; ++list) {
            c->patch_n_groups[list] = int(glist[list].size());
            groups.insert(groups.end(), glist[list].begin(), glist[list].end());
        }
        return ok;
    }
}

int upload_patches(sg_ctx *c) {
    const HostLayout &h = c->host;
    PatchArrays &pa = c->patch;
    if (h.P != 8 && h.P != 16) return SG_OK;                               // direct kernel only
    pa.P = h.P;
    pa.n_patches = int(h.patches.size());
    pa.wstride = ((h.P + 1) * (h.P + 1) + 1) & ~1;
    int rc;
    if ((rc = upload(c, &pa.info, c->patch_info))) return rc;
    if ((rc = dev_alloc(c, &pa.wP, int64_t(pa.n_patches) * pa.wstride))) return rc;
    {
        // owner patch of every vertex: the finest patch that has it on its (P+1)^2 lattice; among patches of that level
        // the one that holds it in its lower-left P x P block (i < P and j < P), then i < P, then the lowest index.  On a
        // uniform level every patch then owns exactly its P x P lower-left vertices, and row P / column P of a patch
        // carry weights only where no patch of the level continues above / to the right: the offset-table kernels skip
        // them otherwise (pflags: bit 0 = row P owned somewhere, bit 1 = column P owned in a row below P).
        const int P1 = h.P + 1;
        auto vertex_of = [&](int32_t x, int32_t y) -> int32_t {
            const auto cx = std::lower_bound(h.colX.begin(), h.colX.end(), x);
            if (cx == h.colX.end() || *cx != x) return -1;
            const size_t col = size_t(cx - h.colX.begin());
            const auto b0 = h.vky.begin() + h.colstart[col], b1 = h.vky.begin() + h.colstart[col + 1];
            const auto it = std::lower_bound(b0, b1, y);
            return (it == b1 || *it != y) ? -1 : int32_t(it - h.vky.begin());
        };
        std::vector<int32_t> pv(size_t(pa.n_patches) * P1 * P1, -1), owner(size_t(h.Nv), -1);
        std::vector<int8_t> owner_rank(size_t(h.Nv), 127);
#pragma omp parallel for schedule(static)
        for (int p = 0; p < pa.n_patches; ++p) {                   // the look-ups (read only), in parallel
            const PatchInfo &q = c->patch_info[size_t(p)];
            for (int j = 0; j < P1; ++j)
                for (int i = 0; i < P1; ++i)
                    pv[(size_t(p) * P1 + j) * P1 + i] = vertex_of(q.X0 + i * q.cw, q.Y0 + j * q.cw);
        }
        for (int p = 0; p < pa.n_patches; ++p) {
            const PatchInfo &q = c->patch_info[size_t(p)];
            for (int j = 0; j < P1; ++j)
                for (int i = 0; i < P1; ++i) {
                    const int32_t v = pv[(size_t(p) * P1 + j) * P1 + i];
                    if (v < 0) continue;                           // a lattice point of a padded block that no cell touches
                    const int8_t rank = int8_t((j == h.P ? 2 : 0) + (i == h.P ? 1 : 0));
                    int32_t &o = owner[size_t(v)];
                    if (o < 0 || c->patch_info[size_t(o)].level < q.level ||
                        (c->patch_info[size_t(o)].level == q.level && rank < owner_rank[size_t(v)])) {
                        o = p;
                        owner_rank[size_t(v)] = rank;
                    }
                }
        }
        std::vector<int32_t> pflags(size_t(pa.n_patches), 0);
        for (int p = 0; p < pa.n_patches; ++p)
            for (int e = 0; e < P1 * P1; ++e) {
                int32_t &v = pv[size_t(p) * P1 * P1 + e];
                if (v >= 0 && owner[size_t(v)] != p) v = -1;
                if (v >= 0 && e / P1 == h.P) pflags[size_t(p)] |= 1;
                if (v >= 0 && e / P1 < h.P && e % P1 == h.P) pflags[size_t(p)] |= 2;
            }
        // Per-patch weights of lattice mode: owned deduplicated weights on 16 x 16 vertices (fast: cfg 5 162.7 ms), or
        // "neutral" weights from the patch's own cells on all 17 x 17 vertices (176.2 ms), with which every patch's
        // weights sum to zero and the rounding error does not grow with the lattice: 12 M-leaf config 4 (extent 16,384
        // lattice units) 1.4e-12 -> 5e-14 of max|F|, slope path on the 6 M-leaf quadtrees 1.4e-11 -> < 1e-11
        // (DESIGN.md 6c, 8).  Neutral on lattices of more than 4,096 units, or when SG_LATTICE_NEUTRAL_WEIGHTS is set
        // (read at sg_create); owned below, where both agree to ~1e-13.
        c->neutral_weights = std::getenv("SG_LATTICE_NEUTRAL_WEIGHTS") != nullptr || h.extent > 4096;
        if (c->neutral_weights) for (auto &f : pflags) f = 3;
        c->patch_flags = pflags;
        if ((rc = upload(c, &pa.pflags, pflags))) return rc;
        if ((rc = upload(c, &pa.pvmap, pv))) return rc;
    }
    SG_CUDA(c, configure_patch_kernels(pa.P, c->dev.tab_entries));
    if (pa.P == 16) {
        const bool ok = c->patch_plan_ok;
        const std::vector<PatchLevel> &lev = c->patch_levels;
        const std::vector<int32_t> &pmap = c->patch_pmap;
        const std::vector<PatchGroup> &groups = c->patch_groups;
        if (ok) {
            if ((rc = upload(c, &pa.levels, lev)) || (rc = upload(c, &pa.groups, groups)) || (rc = upload(c, &pa.pmap, pmap)))
                return rc;
            if ((rc = dev_alloc(c, &pa.wQ, int64_t(pa.n_patches) * kPatchQStride))) return rc;
            // per level: the patches at least three levels away (patch_far_kernel)
            std::vector<int32_t> far_list, far_meta(size_t(2 * h.n_levels), 0);
            for (int L = 0; L < h.n_levels; ++L) {
                far_meta[size_t(2 * L)] = int32_t(far_list.size());
                for (int M2 = 0; M2 < h.n_levels; ++M2) {
                    if (std::abs(M2 - L) < 3) continue;
                    for (size_t q = 0; q < h.patches.size(); ++q)
                        if (h.patches[q].level == M2) far_list.push_back(int32_t(q));
                }
                far_meta[size_t(2 * L + 1)] = int32_t(far_list.size()) - far_meta[size_t(2 * L)];
            }
            if ((rc = upload(c, &pa.far_list, far_list)) || (rc = upload(c, &pa.far_meta, far_meta))) return rc;
            SG_CUDA(c, configure_patch_far(c->dev.tab_entries));
            pa.n_groups = int(groups.size());
            SG_CUDA(c, configure_patch_offset());
            pa.blocked = true;
        }
    }
    pa.enabled = true;
    return SG_OK;
}

int upload_layout(sg_ctx *c) {
    const HostLayout &h = c->host;
    DevLayout &d = c->dev;
    d.N = h.N; d.Nv = h.Nv;
    d.nX = int(h.colX.size()); d.nY = int(h.rowY.size());
    d.ntX = int(h.tX.size()); d.ntY = int(h.tY.size());
    d.n_tiles = int(h.chunk_x.size() / kChunksPerTile);
    d.n_slots = int64_t(d.n_tiles) * kTileSlots;
    const int64_t tb_bytes = (int64_t(d.ntY) * d.nX + int64_t(d.ntX) * d.nY) * 8;
    if (tb_bytes > (int64_t(48) << 30)) {
        c->err = "line tables would need more than 48 GiB: layout too large for this build";
        return SG_ERR_LAYOUT;
    }
    std::vector<double2> tgt(size_t(h.N));
    for (int64_t i = 0; i < h.N; ++i) tgt[i] = make_double2(double(h.tkx[i]), double(h.tky[i]));
    int rc;
    if ((rc = upload(c, &d.tgt, tgt))) return rc;
    if ((rc = upload(c, &d.itx, h.itx)) || (rc = upload(c, &d.ity, h.ity))) return rc;
    if ((rc = upload(c, &d.adj, h.adj))) return rc;
    if ((rc = upload(c, &d.vkx, h.vkx)) || (rc = upload(c, &d.vky, h.vky))) return rc;
    if ((rc = upload(c, &d.colX, h.colX)) || (rc = upload(c, &d.colstart, h.colstart))) return rc;
    if ((rc = upload(c, &d.rowY, h.rowY)) || (rc = upload(c, &d.rowstart, h.rowstart))) return rc;
    if ((rc = upload(c, &d.rowperm, h.rowperm))) return rc;
    if ((rc = upload(c, &d.chunk_x, h.chunk_x)) || (rc = upload(c, &d.slot_vertex, h.slot_vertex))) return rc;
    if ((rc = dev_alloc(c, &d.queue, kQueues))) return rc;
    SG_CUDA(c, cudaMemset(d.queue, 0, kQueues * sizeof(unsigned int)));
    if ((rc = upload(c, &d.tX, h.tX)) || (rc = upload(c, &d.tY, h.tY))) return rc;
    if ((rc = dev_alloc(c, &d.vtile, int64_t(d.n_tiles) * kTileDoubles))) return rc;
    if ((rc = dev_alloc(c, &d.w, h.Nv))) return rc;
    if ((rc = dev_alloc(c, &d.wcum, 2 * h.Nv))) return rc;
    if ((rc = dev_alloc(c, &d.TBx, int64_t(d.ntY) * d.nX))) return rc;
    if ((rc = dev_alloc(c, &d.TBy, int64_t(d.ntX) * d.nY))) return rc;

    // log-table range: arguments a = |v| + r with r >= 1 (a target never sits on a vertex) and
    // a <= (1 + sqrt 2) * extent, all in lattice units.
    const double a_max = 2.5 * double(h.extent) + 2.0;
    int e_max = 0;
    std::frexp(a_max, &e_max);                       // a_max < 2^e_max
    d.tab_idx0 = 0x3ff << kLogK;                     // a = 1.0
    d.tab_entries = (e_max + 1) << kLogK;
    if ((rc = dev_alloc(c, &d.lntab, d.tab_entries))) return rc;
    SG_CUDA(c, configure_kernels(d.tab_entries));
    d.lnint_n = h.extent < (1 << 21) ? h.extent + 2 : 0;        // all |vertex - target| lattice distances
    if (d.lnint_n > 0 && (rc = dev_alloc(c, &d.lnint, d.lnint_n))) return rc;
    launch_build_logtab(d, nullptr);
    launch_build_lnint(d, nullptr);
    launch_fill_static_tiles(d, nullptr);
    SG_CUDA(c, cudaGetLastError());
    SG_CUDA(c, cudaDeviceSynchronize());
    if ((rc = upload_patches(c))) return rc;
    return SG_OK;
}

}  // namespace

extern "C" {

static int create_ctx(sg_ctx **out, int n_levels, const double *cell_width, double x0, double y0, int patch_cells,
                      const sg_patch *leaf_patches, int64_t n_patches, double G, int device, const uint8_t *cell_present) {
    if (!out) { g_create_error = "out is NULL"; return SG_ERR_ARG; }
    *out = nullptr;
    if (!std::isfinite(G)) { g_create_error = "G must be finite"; return SG_ERR_ARG; }
    sg_ctx *c = new sg_ctx();
    int rc = build_layout(c->host, n_levels, cell_width, x0, y0, patch_cells, leaf_patches, n_patches, c->err, cell_present);
    if (rc == SG_OK) {
        c->device = device;
        c->dev.G = G;
        c->first = 0; c->count = c->host.N;
        c->poison_partials = std::getenv("SG_POISON_PARTIALS") != nullptr;
        c->debug_sync = std::getenv("SG_DEBUG_SYNC") != nullptr;
        c->owned_slope_weights = std::getenv("SG_LATTICE_OWNED_SLOPE_WEIGHTS") != nullptr;
        c->patch_plan_ok = build_patch_plan(c);
        c->lat_entries = plan_fn_lattices(c);
        if (device >= 0) {
            DeviceGuard guard(device);
            cudaError_t e = guard.err;
            if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
            if (e != cudaSuccess) {
                c->err = std::string("cudaSetDevice: ") + cudaGetErrorString(e);
                rc = SG_ERR_CUDA;
            } else {
                rc = upload_layout(c);
                if (rc == SG_OK) rc = reserve_partials(c);
            }
        }
    }
    if (rc != SG_OK) {
        g_create_error = c->err;
        sg_destroy(c);
        return rc;
    }
    *out = c;
    return SG_OK;
}

int sg_create(sg_ctx **out, int n_levels, const double *cell_width, double x0, double y0, int patch_cells,
              const sg_patch *leaf_patches, int64_t n_patches, double G, int device) {
    return create_ctx(out, n_levels, cell_width, x0, y0, patch_cells, leaf_patches, n_patches, G, device, nullptr);
}

static int apply_inner_range(sg_ctx *c);

// Regrouping for lattice mode (P = 1, 2, 4): every leaf cell of level l at (ci, cj) on its level's lattice goes to
// the aligned 16 x 16 block (l, ci >> 4, cj >> 4); a block that is only partly covered by leaves of its level is
// padded with holes (targets whose result is discarded, no sources: build_layout's cell_present).  The inner context
// is an ordinary P = 16 context on that padded layout.
static int build_regrouped(sg_ctx *c) {
    const HostLayout &h = c->host;
    const int P = h.P;
    std::vector<uint64_t> keys(size_t(h.N));
    std::vector<uint32_t> within(size_t(h.N));
    {
        int64_t cell = 0;
        for (size_t p = 0; p < h.patches.size(); ++p) {
            const sg_patch &q = h.patches[p];
            for (int j = 0; j < P; ++j)
                for (int i = 0; i < P; ++i, ++cell) {
                    const uint64_t ci = uint64_t(q.i0 + i), cj = uint64_t(q.j0 + j);
                    keys[size_t(cell)] = (uint64_t(q.level) << 56) | ((cj >> 4) << 28) | (ci >> 4);   // sorts by (level, bj, bi)
                    within[size_t(cell)] = uint32_t((cj & 15) * 16 + (ci & 15));
                }
        }
    }
    std::vector<uint64_t> blocks(keys);
    std::sort(blocks.begin(), blocks.end());
    blocks.erase(std::unique(blocks.begin(), blocks.end()), blocks.end());
    const int64_t nb = int64_t(blocks.size()), n_inner = nb * 256;
    if (n_inner >= (int64_t(1) << 29)) { c->err = "regrouped layout too large"; return SG_ERR_LAYOUT; }
    std::vector<sg_patch> bp;
    bp.resize(size_t(nb));
    for (int64_t b = 0; b < nb; ++b) {
        const uint64_t k = blocks[size_t(b)];
        bp[size_t(b)] = sg_patch{int32_t(k >> 56), int32_t((k & 0xfffffffu) * 16), int32_t(((k >> 28) & 0xfffffffu) * 16)};
    }
    std::vector<int32_t> map(size_t(h.N)), inv(size_t(n_inner), -1);
    std::vector<uint8_t> present(size_t(n_inner), 0);
    for (int64_t cell = 0; cell < h.N; ++cell) {
        const int64_t b = std::lower_bound(blocks.begin(), blocks.end(), keys[size_t(cell)]) - blocks.begin();
        const int64_t k = b * 256 + within[size_t(cell)];
        map[size_t(cell)] = int32_t(k);
        inv[size_t(k)] = int32_t(cell);
        present[size_t(k)] = 1;
    }
    std::vector<double> cw(size_t(h.n_levels));
    for (int l = 0; l < h.n_levels; ++l) cw[size_t(l)] = h.unit * double(int64_t(2) << (h.n_levels - 1 - l));
    sg_ctx *in = nullptr;
    int rc = create_ctx(&in, h.n_levels, cw.data(), h.x0, h.y0, 16, bp.data(), nb, c->dev.G, c->device, present.data());
    if (rc != SG_OK) { c->err = "regrouped layout: " + g_create_error; return rc; }
    // c->inner is what marks the regrouping as built (sg_set_interaction_mode, sg_set_density, sg_force): it is set
    // only once every permutation buffer exists; on a failure the inner context goes and a later call starts over
    // (buffers already allocated stay owned by c and are freed by sg_destroy)
    rc = upload(c, &c->rg_map, map);
    if (rc == SG_OK) rc = upload(c, &c->rg_inv, inv);
    for (int k = 0; k < 3 && rc == SG_OK; ++k) rc = dev_alloc(c, &c->rg_in[k], n_inner);
    for (int k = 0; k < 2 && rc == SG_OK; ++k) rc = dev_alloc(c, &c->rg_f[k], n_inner);
    if (rc != SG_OK) {
        sg_destroy(in);
        c->rg_map = c->rg_inv = nullptr;
        for (double *&q : c->rg_in) q = nullptr;
        for (double *&q : c->rg_f) q = nullptr;
        return rc;
    }
    c->inner = in;
    c->rg_map_host = std::move(map);
    return apply_inner_range(c);                                  // a target range set before the mode was chosen
}

// Regrouped lattice mode: a target slice must cost a slice (targets are shared out over GPUs).  The
// caller's range [first, first + count) is turned into the range of inner blocks that hold its cells, and the inner
// context evaluates only those: the caller's cell order (level, row, column) and the block order (level, block row,
// block column) run alike when the patch list is sorted that way (the usual case; any order is still correct, the
// covering range just grows), so the covering block range exceeds the slice by about two block rows per level touched.  rg_first is the inner cell the slice-relative rg_f buffers start at (gather_cells_kernel subtracts it).
static int apply_inner_range(sg_ctx *c) {
    if (!c->inner) return SG_OK;
    int64_t f = 0, n = 0;
    if (c->count > 0) {
        int32_t kmin = INT32_MAX, kmax = -1;
        const int32_t *m = c->rg_map_host.data() + c->first;
        for (int64_t i = 0; i < c->count; ++i) { kmin = std::min(kmin, m[i]); kmax = std::max(kmax, m[i]); }
        f = int64_t(kmin / 256) * 256;
        n = (int64_t(kmax / 256) + 1) * 256 - f;
    }
    c->rg_first = f;
    const int rc = sg_set_target_range(c->inner, f, n);
    if (rc) c->err = c->inner->err;
    return rc;
}

static bool regroupable(const sg_ctx *c) { return c->host.P == 1 || c->host.P == 2 || c->host.P == 4; }

void sg_destroy(sg_ctx *c) {
    if (!c) return;
    if (c->inner) { sg_destroy(c->inner); c->inner = nullptr; }
    if (c->device >= 0) {
        DeviceGuard guard(c->device);
        cudaDeviceSynchronize();
        for (void *p : c->allocs) cudaFree(p);
        for (cudaEvent_t e : c->ev0) cudaEventDestroy(e);
        for (cudaEvent_t e : c->ev1) cudaEventDestroy(e);
        for (cudaStream_t st : c->side) cudaStreamDestroy(st);
        for (cudaEvent_t e : c->join_ev) cudaEventDestroy(e);
        if (c->fork_ev) cudaEventDestroy(c->fork_ev);
    }
    delete c;
}

int64_t sg_num_cells(const sg_ctx *c) { return c ? c->host.N : -1; }
int64_t sg_num_vertices(const sg_ctx *c) { return c ? c->host.Nv : -1; }

int sg_layout_info(const sg_ctx *c, int64_t *info) {
    if (!c || !info) return SG_ERR_ARG;
    info[0] = c->host.N; info[1] = c->host.Nv;
    info[2] = int64_t(c->host.colX.size()); info[3] = int64_t(c->host.rowY.size());
    info[4] = int64_t(c->host.tX.size()); info[5] = int64_t(c->host.tY.size());
    info[6] = c->host.balanced ? 1 : 0;
    info[7] = c->dev_bytes + (c->inner ? c->inner->dev_bytes : 0);
    return SG_OK;
}

int sg_cell_geometry(const sg_ctx *c, double *xc, double *yc, double *h) {
    if (!c) return SG_ERR_ARG;
    const HostLayout &L = c->host;
    const int64_t PP = int64_t(L.P) * L.P;
    for (int64_t i = 0; i < L.N; ++i) {
        if (xc) xc[i] = L.x0 + double(L.tkx[i]) * L.unit;
        if (yc) yc[i] = L.y0 + double(L.tky[i]) * L.unit;
        if (h) h[i] = L.unit * double(int64_t(2) << (L.n_levels - 1 - L.patches[i / PP].level));
    }
    return SG_OK;
}

int sg_set_density(sg_ctx *c, const double *sigma_dev, void *cuda_stream) {
    if (!c) return SG_ERR_ARG;
    if (!sigma_dev) { c->err = "sigma_dev is NULL"; return SG_ERR_ARG; }
    if (c->device < 0) { c->err = "host-only context (device < 0): no CUDA path, and there is no CPU fallback"; return SG_ERR_CUDA; }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    DeviceGuard guard(c->device);
    SG_CUDA(c, guard.err);
    launch_vertex_weights(c->dev, sigma_dev, s);
    launch_line_tables(c->dev, s);
    if (c->patch.enabled) {
        if (c->neutral_weights) launch_patch_weights_owncell(c->patch, sigma_dev, s);
        else launch_patch_weights(c->patch, c->dev.w, s);
    }
    SG_CUDA(c, cudaGetLastError());
    c->density_set = true;
    c->linear = false;
    if (c->inner) {                                           // regrouped lattice mode: the same sigma in block order
        launch_scatter_cells(sigma_dev, nullptr, nullptr, c->rg_inv, c->rg_in[0], nullptr, nullptr, c->inner->host.N, s);
        const int rc = sg_set_density(c->inner, c->rg_in[0], cuda_stream);
        if (rc) { c->err = c->inner->err; return rc; }
    }
    return SG_OK;
}

int sg_set_density_linear(sg_ctx *c, const double *sigma_dev, const double *dx_dev, const double *dy_dev,
                          void *cuda_stream) {
    if (!c) return SG_ERR_ARG;
    if (!sigma_dev || !dx_dev || !dy_dev) { c->err = "sigma_dev / dx_dev / dy_dev is NULL"; return SG_ERR_ARG; }
    if (c->device < 0) { c->err = "host-only context (device < 0): no CUDA path, and there is no CPU fallback"; return SG_ERR_CUDA; }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    DeviceGuard guard(c->device);
    SG_CUDA(c, guard.err);
    LinArrays &l = c->lin;
    if (!l.allocated) {
        const HostLayout &h = c->host;
        const DevLayout &d = c->dev;
        l.unit = h.unit;
        l.cells_per_patch = h.P * h.P;
        std::vector<double> hh(h.patches.size());
        for (size_t p = 0; p < hh.size(); ++p) hh[p] = double(int64_t(1) << (h.n_levels - 1 - h.patches[p].level));
        int rc;
        if ((rc = upload(c, &l.patch_hh, hh))) return rc;
        if ((rc = dev_alloc(c, &l.wl, 3 * h.Nv))) return rc;
        if ((rc = dev_alloc(c, &l.vtile, int64_t(d.n_tiles) * kTileLinDoubles))) return rc;
        if ((rc = dev_alloc(c, &l.TBx3, int64_t(d.ntY) * d.nX * 3))) return rc;
        if ((rc = dev_alloc(c, &l.TBy3, int64_t(d.ntX) * d.nY * 3))) return rc;
        SG_CUDA(c, configure_lin_kernels(d.tab_entries));
        if (c->patch.blocked && (rc = dev_alloc(c, &c->lat.wS, int64_t(kFnPlanesLin) * c->patch.n_patches * kPatchQStride)))
            return rc;
        // lattice mode is on already: add the slope planes to the function lattices (host-synchronous, first call only)
        if (c->use_patch && !c->force_incta && (rc = ensure_fn_lattices(c, kFnPlanesLin))) return rc;
        if ((rc = reserve_partials(c))) return rc;
        l.allocated = true;                                       // only now: a failed set-up is retried by the next call
    }
    launch_weights_lin(c->dev, l, sigma_dev, dx_dev, dy_dev, s);
    if (c->lat.wS) {
        // slope path in lattice mode: ALWAYS own-cell (neutral) per-patch weights on all 17 x 17 vertices.  The slope
        // planes a_v, c_v enter multiplied by the lattice offset u, v, so owned 16 x 16 weights (patches not neutral)
        // cancel across patches and lose digits with extent / h: BASELINE config 4 (extent 2,048) rel. L2 1.7e-12
        // owned against 7e-13 with the direct slope kernel and the 1e-12 gate; neutral weights are as accurate as the
        // direct kernel at every extent.  Costs 289 instead of 256 vertices per patch pair on this path
        // only; the zeroth-order path keeps the choice made in upload_patches.  SG_LATTICE_OWNED_SLOPE_WEIGHTS (read at
        // sg_create) brings the owned weights back on lattices of up to 4,096 units: a test aid that reproduces the
        // comparison table of DESIGN.md 8, not a supported mode.
        c->lat.lin_neutral = c->neutral_weights || !c->owned_slope_weights;
        if (c->lat.lin_neutral) launch_patch_weights_lin_owncell(c->patch, sigma_dev, dx_dev, dy_dev, l.patch_hh, l.unit, c->lat.wS, s);
        else launch_patch_weights_lin(c->patch, l.wl, c->lat.wS, s);
    }
    SG_CUDA(c, cudaGetLastError());
    c->density_set = true;
    c->linear = true;
    if (c->inner) {
        launch_scatter_cells(sigma_dev, dx_dev, dy_dev, c->rg_inv, c->rg_in[0], c->rg_in[1], c->rg_in[2], c->inner->host.N, s);
        const int rc = sg_set_density_linear(c->inner, c->rg_in[0], c->rg_in[1], c->rg_in[2], cuda_stream);
        if (rc) { c->err = c->inner->err; return rc; }
    }
    return SG_OK;
}

int sg_force(sg_ctx *c, double *Fx_dev, double *Fy_dev, void *cuda_stream) {
    if (!c) return SG_ERR_ARG;
    if (c->device < 0) { c->err = "host-only context (device < 0): no CUDA path, and there is no CPU fallback"; return SG_ERR_CUDA; }
    if (!c->density_set) { c->err = "sg_force called before sg_set_density"; return SG_ERR_STATE; }
    if (c->count == 0) return SG_OK;
    if (!Fx_dev || !Fy_dev) { c->err = "Fx_dev / Fy_dev is NULL"; return SG_ERR_ARG; }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    DeviceGuard guard(c->device);
    SG_CUDA(c, guard.err);
    if (c->use_patch && c->inner) {
        // regrouped lattice mode: the inner context evaluates the blocks that hold the caller's target range
        // (apply_inner_range), the caller's targets are picked out of its slice-relative result
        if (!c->inner->density_set || c->inner->linear != c->linear) {
            c->err = "regrouped lattice mode: set the density after sg_set_interaction_mode(SG_MODE_LATTICE)";
            return SG_ERR_STATE;
        }
        const int rc = sg_force(c->inner, c->rg_f[0], c->rg_f[1], cuda_stream);
        if (rc) { c->err = c->inner->err; return rc; }
        launch_gather_cells(c->rg_f[0], c->rg_f[1], c->rg_map, c->rg_first, c->first, c->count, Fx_dev, Fy_dev, s);
        SG_CUDA(c, cudaGetLastError());
        return SG_OK;
    }
    const StepPlan sp = make_step_plan(c, c->linear);
    const ForcePlan &p = sp.p;
    int rc = grow_partials(c, sp.partials(), s);           // no-op: reserve_partials() sized it (fallback otherwise)
    if (rc) return rc;
    // test aid (tests/conftest.py sets it): NaN-fill the partial sums on the caller's stream before EVERY evaluation,
    // so that a slot no kernel writes shows up in the forces instead of passing as the previous call's value
    if (c->poison_partials)
        SG_CUDA(c, cudaMemsetAsync(c->dev.part, 0xFF, size_t(sp.partials()) * sizeof(double), s));
    const int slot = int(c->timed_calls % kTimingRing);
    if (c->timing) SG_CUDA(c, cudaEventRecord(c->ev0[slot], s));
    if (c->linear && !sp.by_patch) launch_interaction_lin(c->dev, c->lin, p, s);
    else if (sp.by_patch) {
        // every launch writes its own n_split slots of [2][count] partial sums and has its own work queue, so the
        // launches are independent: the first runs on the caller's stream, the others on side streams that wait for
        // an event recorded on the caller's stream and are joined back into it (capturable in a CUDA graph)
        const OffsetPlan &po = sp.po;
        double *part = c->dev.part;
        const bool debug_sync = c->debug_sync;                 // debugging aid: name the failing launch
        const int n_total = (sp.blocked ? offset_classes(po) : 0) + ((!sp.blocked || sp.far) ? 1 : 0);
        if (n_total > 1) {
            while (int(c->side.size()) < n_total - 1) {
                cudaStream_t st; cudaEvent_t ev;
                SG_CUDA(c, cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
                c->side.push_back(st);
                SG_CUDA(c, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
                c->join_ev.push_back(ev);
            }
            if (!c->fork_ev) SG_CUDA(c, cudaEventCreateWithFlags(&c->fork_ev, cudaEventDisableTiming));
            SG_CUDA(c, cudaEventRecord(c->fork_ev, s));
        }
        // from here on a failure must still join the side streams back (a dangling fork would break a stream capture
        // and leave the work queues undrained): remember the first error, keep going, join, then return it
        cudaError_t first_err = cudaSuccess;
        std::string where;
        auto note = [&](cudaError_t e, const char *what) {
            if (e != cudaSuccess && first_err == cudaSuccess) { first_err = e; where = what; }
        };
        int n_launch = 0;
        auto on_stream = [&](int idx) -> cudaStream_t {
            if (idx == 0) return s;
            cudaStream_t st = c->side[size_t(idx - 1)];
            note(cudaStreamWaitEvent(st, c->fork_ev, 0), "cudaStreamWaitEvent(fork)");
            return st;
        };
        if (sp.blocked && sp.far) {
            // pairs >= 3 levels apart, directly: the longest launch of a deep hierarchy goes first, so that the short
            // table classes fill in beside and after it (its partial sums are the LAST slots of `part`)
            double *far_part = part + int64_t(offset_classes(po)) * po.n_split * 2 * c->count;
            launch_patch_far(c->linear, c->dev, c->patch, c->linear ? c->lat.wS : c->patch.wQ, sp.pp, c->first, c->count, far_part,
                             on_stream(n_launch));
            ++n_launch;
        }
        if (sp.blocked)
            for (int v = 0; v < kOffClasses; ++v)
                if (po.variant[v]) {
                    if (sp.fn)
                        launch_lattice_corr(v, c->dev, c->patch, c->lat, po, sp.n_planes, c->first, c->count, part, c->sm_count,
                                            on_stream(n_launch));
                    else
                        launch_patch_offset(v, c->dev, c->patch, po, c->first, c->count, part, c->sm_count, on_stream(n_launch));
                    ++n_launch;
                    part += int64_t(po.n_split) * 2 * c->count;
                    if (debug_sync && first_err == cudaSuccess) {
                        const cudaError_t e = cudaDeviceSynchronize();
                        if (e != cudaSuccess) { first_err = e; where = std::string(sp.fn ? "lattice_corr_kernel<" : "patch_offset_kernel<") + std::to_string(v) + ">"; }
                    }
                }
        if (!sp.blocked) {                              // P = 8: everything in the generic kernel
            launch_patch_interaction(c->dev, c->patch, sp.pp, c->first, c->count, part, 0, on_stream(n_launch));
            ++n_launch;
        }
        note(cudaGetLastError(), "pair-class kernel launch");
        for (int i = 1; i < n_launch; ++i) {
            note(cudaEventRecord(c->join_ev[size_t(i - 1)], c->side[size_t(i - 1)]), "cudaEventRecord(join)");
            note(cudaStreamWaitEvent(s, c->join_ev[size_t(i - 1)], 0), "cudaStreamWaitEvent(join)");
        }
        if (first_err != cudaSuccess) {
            // the queues may be half drained: reset them so that the next call starts clean
            cudaMemsetAsync(c->dev.queue, 0, kQueues * sizeof(unsigned int), s);
            c->err = where + ": " + cudaGetErrorString(first_err);
            return SG_ERR_CUDA;
        }
    }
    else launch_interaction(c->dev, p, s);
    if (c->timing) {
        SG_CUDA(c, cudaEventRecord(c->ev1[slot], s));
        ++c->timed_calls;
    }
    if (c->linear) launch_finalise_lin(c->dev, c->lin, p, Fx_dev, Fy_dev, s);
    else launch_finalise(c->dev, p, Fx_dev, Fy_dev, s);
    SG_CUDA(c, cudaGetLastError());
    return SG_OK;
}

int sg_set_interaction_mode(sg_ctx *c, int mode) {
    if (!c) return SG_ERR_ARG;
    if (mode != SG_MODE_DIRECT && mode != SG_MODE_LATTICE && mode != SG_MODE_LATTICE_BLOCKED && mode != SG_MODE_LATTICE_INCTA) {
        c->err = "unknown interaction mode"; return SG_ERR_ARG;
    }
    if (mode == SG_MODE_LATTICE && regroupable(c) && c->device >= 0) {
        // small patches (the paper's zone-wise quadtrees): pack the leaves into padded 16 x 16 blocks once
        DeviceGuard guard(c->device);
        SG_CUDA(c, guard.err);
        if (!c->inner) {
            const int rc = build_regrouped(c);
            if (rc) return rc;
        }
        const int rc = sg_set_interaction_mode(c->inner, SG_MODE_LATTICE);
        if (rc) { c->err = c->inner->err; return rc; }
        c->use_patch = true;
        return SG_OK;
    }
    if (mode == SG_MODE_LATTICE && c->host.P != 8 && c->host.P != 16) {
        c->err = "SG_MODE_LATTICE needs patches of 8 x 8 or 16 x 16 cells (or of 1, 2 or 4 cells, regrouped on a device)";
        return SG_ERR_ARG;
    }
    if ((mode == SG_MODE_LATTICE_BLOCKED || mode == SG_MODE_LATTICE_INCTA) &&
        (c->host.P != 16 || (c->device >= 0 && !c->patch.blocked))) {
        c->err = "SG_MODE_LATTICE_BLOCKED / _INCTA need patches of 16 x 16 cells (and per-level patch maps that fit)";
        return SG_ERR_ARG;
    }
    c->use_patch = mode != SG_MODE_DIRECT;
    c->force_incta = mode == SG_MODE_LATTICE_INCTA;
    if (c->device < 0) return SG_OK;
    DeviceGuard guard(c->device);
    SG_CUDA(c, guard.err);
    if (c->use_patch && !c->force_incta) {
        const int rc = ensure_fn_lattices(c, c->lin.allocated ? kFnPlanesLin : 1);
        if (rc) return rc;
    }
    return reserve_partials(c);
}

int sg_set_target_range(sg_ctx *c, int64_t first, int64_t count) {
    if (!c) return SG_ERR_ARG;
    if (first < 0 || count < 0 || first + count > c->host.N) {
        c->err = "target range outside [0, N)"; return SG_ERR_ARG;
    }
    c->first = first; c->count = count;
    if (c->device < 0) return SG_OK;
    DeviceGuard guard(c->device);
    SG_CUDA(c, guard.err);
    const int rc = apply_inner_range(c);
    if (rc) return rc;
    return reserve_partials(c);
}

int sg_lattice_plan_check(const sg_ctx *c, int64_t *out) {
    if (!c || !out) return SG_ERR_ARG;
    for (int i = 0; i < 16; ++i) out[i] = 0;
    if (!c->patch_plan_ok) return SG_OK;
    out[11] = 1;
    const HostLayout &h = c->host;
    const int64_t np = int64_t(h.patches.size());
    if (np * np > (int64_t(1) << 32)) return SG_OK;                       // diagnostic for test-sized layouts
    std::vector<uint8_t> hits(size_t(np * np), 0);
    const int F_of[kOffClasses] = {1, 2, 2, 4, 4}, dl_of[kOffClasses] = {0, -1, 1, -2, 2};
    size_t g0 = 0;
    for (int list = 0; list < 3; ++list) {
        out[7 + list] = c->patch_n_groups[list];
        // a list whose classes are launched must hold every patch exactly once (each launch writes the partial sums
        // of all targets, zeros included)
        bool launched = false;
        std::vector<int> seen(size_t(np), 0);
        for (size_t gi = g0; gi < g0 + size_t(c->patch_n_groups[list]); ++gi) {
            const PatchGroup &g = c->patch_groups[gi];
            for (int v = 0; v < kOffClasses; ++v) launched = launched || (offset_group_list(v) == list && g.box[v][1] > 0);
            for (int w = 0; w < g.n; ++w) ++seen[size_t(g.patch[w])];
        }
        if (launched)
            for (int64_t q = 0; q < np; ++q) out[12] += seen[size_t(q)] != 1;
        for (size_t gi = g0; gi < g0 + size_t(c->patch_n_groups[list]); ++gi) {
            const PatchGroup &g = c->patch_groups[gi];
            for (int v = 0; v < kOffClasses; ++v) {
                if (offset_group_list(v) != list) continue;
                const int ndpi = g.box[v][1], ndpj = g.box[v][3];
                if (ndpi * ndpj == 0) continue;
                const int F = F_of[v], step = dl_of[v] < 0 ? F : 1;
                const PatchLevel &slev = c->patch_levels[size_t(g.level + dl_of[v])];
                out[10] += int64_t(ndpi) * ndpj;
                for (int n = 0; n < ndpi * ndpj; ++n)                          // the walk of patch_offset_kernel<v>
                    for (int w = 0; w < g.n; ++w) {
                        const int api = h.patches[size_t(g.patch[w])].i0 / h.P, apj = h.patches[size_t(g.patch[w])].j0 / h.P;
                        const int dx = g.box[v][0] + step * (n % ndpi), dy = g.box[v][2] + step * (n / ndpi);
                        int bi, bj;
                        if (dl_of[v] < 0) {
                            if ((api + dx) % F != 0 || (apj + dy) % F != 0) { ++out[6]; continue; }
                            bi = (api + dx) / F; bj = (apj + dy) / F;
                        } else { bi = F * api + dx; bj = F * apj + dy; }
                        bi -= slev.pimin; bj -= slev.pjmin;
                        if (bi < 0 || bi >= slev.npx || bj < 0 || bj >= slev.npy) continue;
                        const int b = c->patch_pmap[size_t(slev.map_off) + size_t(bj) * slev.npx + bi];
                        if (b < 0) continue;
                        if (h.patches[size_t(b)].level - g.level != dl_of[v]) ++out[6];
                        if (hits[size_t(g.patch[w]) * np + b]++) ++out[5];
                        ++out[v];
                    }
            }
        }
        g0 += size_t(c->patch_n_groups[list]);
    }
    return SG_OK;
}

int sg_lattice_plan_fill(const sg_ctx *c, int64_t *out) {
    if (!c || !out) return SG_ERR_ARG;
    for (int i = 0; i < 3 * kOffClasses; ++i) out[i] = 0;
    if (!c->patch_plan_ok) return SG_OK;
    const HostLayout &h = c->host;
    const int F_of[kOffClasses] = {1, 2, 2, 4, 4}, dl_of[kOffClasses] = {0, -1, 1, -2, 2};
    size_t g0 = 0;
    for (int list = 0; list < 3; ++list) {
        for (size_t gi = g0; gi < g0 + size_t(c->patch_n_groups[list]); ++gi) {
            const PatchGroup &g = c->patch_groups[gi];
            for (int v = 0; v < kOffClasses; ++v) {
                if (offset_group_list(v) != list) continue;
                const int ndpi = g.box[v][1], ndpj = g.box[v][3];
                if (ndpi * ndpj == 0) continue;
                const int F = F_of[v], step = dl_of[v] < 0 ? F : 1;
                const PatchLevel &slev = c->patch_levels[size_t(g.level + dl_of[v])];
                for (int n = 0; n < ndpi * ndpj; ++n) {
                    int hits = 0;
                    for (int w = 0; w < g.n; ++w) {
                        const int api = h.patches[size_t(g.patch[w])].i0 / h.P, apj = h.patches[size_t(g.patch[w])].j0 / h.P;
                        const int dx = g.box[v][0] + step * (n % ndpi), dy = g.box[v][2] + step * (n / ndpi);
                        int bi, bj;
                        if (dl_of[v] < 0) { bi = (api + dx) / F; bj = (apj + dy) / F; }
                        else { bi = F * api + dx; bj = F * apj + dy; }
                        bi -= slev.pimin; bj -= slev.pjmin;
                        if (bi < 0 || bi >= slev.npx || bj < 0 || bj >= slev.npy) continue;
                        hits += c->patch_pmap[size_t(slev.map_off) + size_t(bj) * slev.npx + bi] >= 0;
                    }
                    out[3 * v] += 1;
                    out[3 * v + 1] += hits > 0;
                    out[3 * v + 2] += hits;
                }
            }
        }
        g0 += size_t(c->patch_n_groups[list]);
    }
    return SG_OK;
}

// Launches of the context's OWN path (as if it had no inner context); read-only on the context.
static void own_launch_counts(const sg_ctx *c, int *set_density_launches, int *force_launches) {
    // vertex weights, running sums and look-ups per direction (+ per-patch weights when the lattice-offset path exists);
    // with slopes: weights, column tables, row tables (+ per-patch slope weights)
    if (set_density_launches) *set_density_launches = c->linear ? 3 + (c->lat.wS ? 1 : 0) : 5 + (c->patch.enabled ? 1 : 0);
    if (force_launches) {                                         // interaction kernel(s) + finalise
        int n = 1;
        if (c->count > 0) {
            const StepPlan sp = make_step_plan(c, c->linear);
            if (sp.by_patch && sp.blocked) n = offset_classes(sp.po) + (sp.far ? 1 : 0);
        }
        *force_launches = c->count > 0 ? n + 1 : 0;
    }
}

int sg_launch_counts(const sg_ctx *c, int *set_density_launches, int *force_launches) {
    if (!c) return SG_ERR_ARG;
    if (c->inner) {                                               // + the permutation kernels
        int a = 0, b = 0, a2 = 0, b2 = 0;
        sg_launch_counts(c->inner, &a, &b);
        own_launch_counts(c, &a2, &b2);
        if (set_density_launches) *set_density_launches = a2 + 1 + a;
        if (force_launches) *force_launches = c->use_patch ? (c->count > 0 ? b + 1 : 0) : b2;
        return SG_OK;
    }
    own_launch_counts(c, set_density_launches, force_launches);
    return SG_OK;
}

int sg_set_kernel_timing(sg_ctx *c, int enable) {
    if (!c) return SG_ERR_ARG;
    if (c->inner) {
        const int rc = sg_set_kernel_timing(c->inner, enable);
        if (rc) { c->err = c->inner->err; return rc; }
    }
    if (c->device < 0) { c->err = "host-only context"; return SG_ERR_CUDA; }
    DeviceGuard guard(c->device);
    SG_CUDA(c, guard.err);
    if (enable && c->ev0.empty()) {
        c->ev0.resize(kTimingRing); c->ev1.resize(kTimingRing);
        for (int i = 0; i < kTimingRing; ++i) {
            SG_CUDA(c, cudaEventCreate(&c->ev0[i]));
            SG_CUDA(c, cudaEventCreate(&c->ev1[i]));
        }
    }
    c->timing = enable != 0;
    c->timed_calls = 0;
    return SG_OK;
}

int sg_get_kernel_times(sg_ctx *c, float *ms, int capacity, int *n) {
    if (!c || !ms || !n || capacity < 0) return SG_ERR_ARG;
    *n = 0;
    if (c->inner && c->use_patch) return sg_get_kernel_times(c->inner, ms, capacity, n);
    if (c->device < 0) { c->err = "host-only context"; return SG_ERR_CUDA; }
    const int64_t have = std::min<int64_t>(c->timed_calls, kTimingRing);
    const int64_t take = std::min<int64_t>(have, capacity);
    if (take == 0) return SG_OK;
    DeviceGuard guard(c->device);
    SG_CUDA(c, guard.err);
    SG_CUDA(c, cudaEventSynchronize(c->ev1[(c->timed_calls - 1) % kTimingRing]));
    for (int64_t k = 0; k < take; ++k) {
        const int slot = int((c->timed_calls - take + k) % kTimingRing);
        SG_CUDA(c, cudaEventElapsedTime(&ms[k], c->ev0[slot], c->ev1[slot]));
    }
    *n = int(take);
    return SG_OK;
}

int sg_kernel_model(const sg_ctx *c, double *fp64_instr_per_pair, double *flops_per_pair, double *pair_evaluations,
                    double *executed_evaluations) {
    if (!c) return SG_ERR_ARG;
    // algorithmic unit: one (target, deduplicated vertex) pair; one launch processes count * N_v
    const double alg = double(c->count) * double(c->host.Nv);
    if (pair_evaluations) *pair_evaluations = alg;
    if (c->inner && c->use_patch)                                 // regrouped: the blocks' work, the caller's units
        return sg_kernel_model(c->inner, fp64_instr_per_pair, flops_per_pair, nullptr, executed_evaluations);
    const StepPlan sp = make_step_plan(c, c->linear);
    if (sp.by_patch && c->linear) {
        // slope path in lattice mode: three planes, 6 DFMA per pair (sg_kernels_lattice.cu)
        if (fp64_instr_per_pair) *fp64_instr_per_pair = 6.0;
        if (flops_per_pair) *flops_per_pair = 12.0;
        if (executed_evaluations) *executed_evaluations = double(c->count) * executed_patch_vertices(c, c->lat.lin_neutral);
        return SG_OK;
    }
    if (sp.by_patch) {
        // lattice-offset path: a pair costs the 2 DFMA of the correlation.  The kernels work on per-patch vertex
        // sets, (P+1)^2 / P^2 more pairs than the deduplicated list: reported separately as executed work, not
        // credited.  Not credited either: the offset tables and the pairs >= 3 levels apart that are summed
        // directly (21 FP64 instructions each), so the algorithmic fraction is a lower bound on deep hierarchies.
        if (fp64_instr_per_pair) *fp64_instr_per_pair = 2.0;
        if (flops_per_pair) *flops_per_pair = 4.0;
        if (executed_evaluations) *executed_evaluations = double(c->count) * executed_patch_vertices(c);
        return SG_OK;
    }
    if (fp64_instr_per_pair) *fp64_instr_per_pair = c->linear ? kLinFp64InstrPerPair : kFp64InstrPerPair;
    if (flops_per_pair) *flops_per_pair = c->linear ? kLinFlopsPerPair : kFlopsPerPair;
    if (executed_evaluations) *executed_evaluations = double(c->count) * double(c->host.slot_vertex.size());   // incl. padding slots
    return SG_OK;
}

int sg_kernel_instruction_counts(int kernel, double *fp64_instr_per_pair, double *flops_per_pair) {
    if (kernel != 0 && kernel != 1) return SG_ERR_ARG;
    if (fp64_instr_per_pair) *fp64_instr_per_pair = kernel ? kLinFp64InstrPerPair : kFp64InstrPerPair;
    if (flops_per_pair) *flops_per_pair = kernel ? kLinFlopsPerPair : kFlopsPerPair;
    return SG_OK;
}

int sg_measure_fp64_peak(int device, double *tflops, double *warp_instr_per_s) {
    DeviceGuard guard(device);
    cudaError_t e = guard.err;
    if (e == cudaSuccess) e = measure_dfma(tflops, warp_instr_per_s);
    if (e != cudaSuccess) { g_create_error = std::string("sg_measure_fp64_peak: ") + cudaGetErrorString(e); return SG_ERR_CUDA; }
    return SG_OK;
}

int sg_measure_fp64_mma_peak(int device, double *dmma_tflops, double *mixed_tflops) {
    DeviceGuard guard(device);
    cudaError_t e = guard.err;
    if (e == cudaSuccess) e = measure_dmma(dmma_tflops, mixed_tflops);
    if (e != cudaSuccess) { g_create_error = std::string("sg_measure_fp64_mma_peak: ") + cudaGetErrorString(e); return SG_ERR_CUDA; }
    return SG_OK;
}

const char *sg_last_error(const sg_ctx *c) { return c ? c->err.c_str() : g_create_error.c_str(); }
const char *sg_version(void) { return "sg-disk-b200 0.1 (sm_100a)"; }

}  // extern "C"
