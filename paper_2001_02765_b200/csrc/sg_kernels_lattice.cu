// sg_kernels_lattice.cu -- S3 by lattice-offset reuse with PRECOMPUTED function lattices ((f1 x f2)).
//
// sg_kernels_patch.cu tabulates the pair function T(d) of a patch offset d inside the CTA, every time a target group
// walks over d.  But T depends on the LAYOUT only (on the pair class and the lattice offset), not on sigma: for a
// (target level, class) all offset tables are windows of one two-dimensional array F (sg_kernels_lattice.cuh).  Here F
// is built once per context and the interaction kernel contains no square root and no logarithm at all:
//
//   lattice_corr_kernel<V>: a CTA = 8 warps = a group of <= 8 target patches, as in patch_offset_kernel<V>, same
//   register-blocked correlation (8 targets per thread, 16 DFMA per LDS.128, weights through L1).  The windows arrive
//   through a ring of K shared-memory stages filled by TMA bulk copies (one cp.async.bulk per table row, issued by the
//   32 lanes of one warp, completion counted on the stage's mbarrier).  There is no CTA-wide barrier per offset: a warp
//   whose target patch has no source patch at an offset only waits for that stage and releases it, so the warps of a
//   CTA drift apart by up to K stages, which absorbs most of the idle time that irregular AMR levels cause in the
//   lock-step kernel (measured in profiles/r2_*).  The warp that releases a stage last issues the copies of the stage
//   K ahead; the lists of live offsets (any warp has a source patch) are made per chunk of kChunkOffsets offsets by
//   all threads together.
//
//   Slope terms (Eq. 6): with planes {T1,T2}, {uT1+vT2, uT2-r}, {vT1-r, uT1+vT2} of F and per-patch
//   weights -W0, a, c (patch_weights_kernel)   Fx/G = sum -W0 T1 + a (uT1+vT2) + c (vT1-r),   Fy/G = sum -W0 T2 + a (uT2-r)
//   + c (uT1+vT2): the same kernel with three stages per offset (plane p correlated with weight array p), 6 DFMA per
//   pair instead of the 28 FP64 + 15 other instructions of interaction_lin_kernel.
#include <algorithm>

#include "sg_kernels_lattice.cuh"
#include "sg_patch_device.cuh"

namespace sg {

// ------------------------------------------------------------------------------------------------
// function lattices: one thread per entry and plane set
// ------------------------------------------------------------------------------------------------
__global__ void build_fn_lattice_kernel(double2 *__restrict__ F, int64_t plane_stride, int ncols, int nrows, int cmin,
                                        int rmin, int mmin, double g, double half_cw, int plane0, int n_planes,
                                        const double *__restrict__ lntab_g, int tab_idx0, uint32_t keep) {
    const int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (e >= int64_t(ncols) * nrows) return;
    const int col = int(e % ncols), row = int(e / ncols);
    const double u = fma(double(col + cmin - mmin), g, -half_cw);
    const double v = fma(double(row + rmin - mmin), g, -half_cw);
    double2 T = make_double2(0.0, 0.0);
    double r = 0.0;
    if (u != 0.0 || v != 0.0) {                          // (0, 0): a target on a vertex, never inside a used window
        T = pair_terms_g(u, v, lntab_g, tab_idx0, keep);
        const double q = fma(u, u, v * v);
        const double y0 = rsqrt_approx(q);
        const double t = q * y0;
        const double ee = fma(-t, y0, 1.0);
        r = fma(t, fma(0.375, ee, 0.5) * ee, t);
    }
    for (int p = plane0; p < plane0 + n_planes; ++p) {
        double2 o;
        const double mix = fma(u, T.x, v * T.y);         // u T1 + v T2
        if (p == 0) o = T;
        else if (p == 1) o = make_double2(mix, fma(u, T.y, -r));
        else o = make_double2(fma(v, T.x, -r), mix);
        F[int64_t(p) * plane_stride + e] = o;
    }
}

void launch_build_fn_lattices(const LatticeArrays &la, const FnLattice *meta_host, const PatchLevel *levels_host,
                              int n_levels, const DevLayout &d, int plane0, int n, cudaStream_t s) {
    const int mmin_of[kOffClasses] = {OffCls<0>::MMIN, OffCls<1>::MMIN, OffCls<2>::MMIN, OffCls<3>::MMIN, OffCls<4>::MMIN};
    const int ldist_of[kOffClasses] = {OffCls<0>::LDIST, OffCls<1>::LDIST, OffCls<2>::LDIST, OffCls<3>::LDIST, OffCls<4>::LDIST};
    for (int L = 0; L < n_levels; ++L)
        for (int v = 0; v < kOffClasses; ++v) {
            const FnLattice &m = meta_host[L * kOffClasses + v];
            if (!m.present) continue;
            const int cw_t = levels_host[L].cw, cw_s = levels_host[L + ldist_of[v]].cw;
            const int64_t n_e = int64_t(m.ncols) * m.nrows;
            build_fn_lattice_kernel<<<unsigned((n_e + 255) / 256), 256, 0, s>>>(
                la.fn + m.base, m.plane_stride, m.ncols, m.nrows, m.cmin, m.rmin, mmin_of[v], double(std::min(cw_t, cw_s)),
                0.5 * double(cw_t), plane0, n, d.lntab, d.tab_idx0, kLogKeepMask);
        }
}

// ------------------------------------------------------------------------------------------------
// the correlation kernel
// ------------------------------------------------------------------------------------------------
constexpr int kChunkOffsets = 64;                       // offsets whose source patches are looked up together
constexpr int kLatAuxBytes = kChunkOffsets * 8 * 4      // sB: source patch of (offset, warp)
                             + kChunkOffsets * 4        // sLive: offsets of the chunk with any source patch
                             + 8 * 8 + 8 * 4            // full[] mbarriers, done[] counters
                             + 16 * 4 + 8 * 4;          // patch positions of the group, item / live count
// dynamic shared memory per CTA with two CTAs per SM: (228 KB - 2 x 1 KB reserved) / 2, minus a little static room
// Deepest ring.  4 stages of the same-level class leave ~45 KB of the SM's 256 KB to L1, where the warps' weight rows
// live (16 warps x 2.4 KB); with 6 stages the L1 hit rate of the weight loads was 63 % and cfg 5 ran 1.3 % slower, and
// the AMR configs gained nothing from the deeper ring (cfg 4: 40.1 vs 40.3 ms).
#ifndef SG_LAT_KMAX
#define SG_LAT_KMAX 4
#endif
constexpr int kLatSmemBudget = 115712 - 256;

// A stage of the ring holds a whole table (classes at most one level apart) or a SUB-BLOCK of its rows: the 80-row
// tables of the classes two levels apart (104 KB) would leave room for one stage only, i.e. lock step.
//   source two levels coarser (V = 3): source row j needs table rows 4 j .. 4 j + 15; sub-block s = the rows of source
//       rows 4 s .. 4 s + 3 = table rows 16 s .. 16 s + 27 (s = 4: row 16 only, table rows 64 .. 79); 5 sub-blocks that
//       overlap by 12 rows (the rows are fetched twice; TMA traffic is not the bottleneck)
//   source two levels finer (V = 4): the table is stored by residue class of the source row (j mod 4), and the source
//       rows are correlated class by class (OffCls::JPASSES): sub-block c = the 20 stored rows of class c
template <int V>
struct LatCls {
    using C = OffCls<V>;
    static constexpr int NSUB = V == kOffCoarserSrc4 ? 5 : V == kOffFinerSrc4 ? 4 : 1;
    static constexpr int SLOT_ROWS = V == kOffCoarserSrc4 ? 28 : V == kOffFinerSrc4 ? C::RPC : C::ROWS;
    static constexpr int SLOT_ENTRIES = SLOT_ROWS * C::TROW;
    static constexpr int STAGE_BYTES = SLOT_ENTRIES * 16;
    static constexpr int K_FIT = (kLatSmemBudget - kLatAuxBytes) / STAGE_BYTES;
    static constexpr int K = K_FIT < 1 ? 1 : (K_FIT > SG_LAT_KMAX ? SG_LAT_KMAX : K_FIT);        // ring depth: 4, 3, 3, 3, 4
    static constexpr size_t smem = size_t(K) * STAGE_BYTES + kLatAuxBytes;
};

template <int V>
__global__ void __launch_bounds__(kOffWarps * 32, 2)
lattice_corr_kernel(const PatchInfo *__restrict__ info, const PatchLevel *__restrict__ levels,
                    const PatchGroup *__restrict__ groups, const int32_t *__restrict__ pmap,
                    const double *__restrict__ wq, int64_t w_plane_stride, const int32_t *__restrict__ pflags,
                    const double2 *__restrict__ fn,
                    const FnLattice *__restrict__ meta, int n_planes, int flags_or, int n_groups, int n_split, int first_patch,
                    int last_patch, int64_t first, int64_t count, double *__restrict__ part,
                    unsigned int *__restrict__ queue) {
    using C = OffCls<V>;
    constexpr int P = 16, F = C::F, TROW = C::TROW, TBUF = LatCls<V>::SLOT_ENTRIES, K = LatCls<V>::K;
    constexpr int NSUB = LatCls<V>::NSUB;
    constexpr int STEP = C::coarser ? F : 1;                              // offsets keep A + d a multiple of F
    constexpr int NCLS = C::coarser ? F / 2 : 1, MT = kBlkR / NCLS;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2 *ring = reinterpret_cast<double2 *>(smem_raw);                 // [K][TBUF]
    int *sB = reinterpret_cast<int *>(ring + K * TBUF);                    // [kChunkOffsets][8]
    int *sLive = sB + kChunkOffsets * 8;                                   // [kChunkOffsets]
    uint64_t *full = reinterpret_cast<uint64_t *>(sLive + kChunkOffsets);  // [4] "full": the stage's TMA bytes have landed
    uint64_t *empty = full + 4;                                            // [4] "empty": all 8 warps are done reading it
    static_assert(K <= 4, "full[] and empty[] share eight mbarrier slots");
    int *sDone = reinterpret_cast<int *>(full + 8);                        // [8]
    int *sPos = sDone + 8;                                                 // [8][2] patch position of target patch w
    int *sMisc = sPos + 16;                                                // [0] item, [1] live offsets of the chunk
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int l = lane & 15, h = lane >> 4;

    if (tid == 0) {
        for (int k = 0; k < K; ++k) { mbar_init(&full[k], 1); mbar_init(&empty[k], kOffWarps); sDone[k] = 0; }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    uint32_t gs = 0;                  // stages this CTA has been through (the same in every warp): slot and parity

    const int n_items = n_groups * n_split;
    while (true) {
        __syncthreads();
        if (tid == 0) sMisc[0] = int(atomicAdd(queue, 1u));
        __syncthreads();
        const int item = sMisc[0];
        if (item >= n_items) break;
        const int gi = item / n_split, sp = item - gi * n_split;
        const PatchGroup *gp = groups + gi;
        if (gp->pmax < first_patch || gp->pmin > last_patch) continue;          // no target of the range in this group
        const int grp_n = gp->n, grp_level = gp->level;
        const PatchLevel lev = levels[grp_level];
        const int dpi_min = gp->box[V][0], ndpi = gp->box[V][1], dpj_min = gp->box[V][2], ndpj = gp->box[V][3];
        const int n_off = ndpi * ndpj, per = (n_off + n_split - 1) / n_split;   // 0 when the class is absent here
        const int n0 = sp * per, n1 = min(n_off, n0 + per);
        const PatchLevel slev = levels[n_off > 0 ? grp_level + C::LDIST : grp_level];
        const FnLattice fm = meta[grp_level * kOffClasses + V];
        if (tid < grp_n) {
            const PatchInfo A = info[gp->patch[tid]];
            sPos[2 * tid] = A.X0 / (P * lev.cw);
            sPos[2 * tid + 1] = A.Y0 / (P * lev.cw);
        }
        const int my_patch = warp < grp_n ? gp->patch[warp] : -1;
        double ax[kBlkR], ay[kBlkR];
#pragma unroll
        for (int r = 0; r < kBlkR; ++r) { ax[r] = 0.0; ay[r] = 0.0; }

        // the copies of stage s of the current chunk: stage = (live offset m, plane pl, sub-block sub), by one warp
        auto issue_stage = [&](int s, int cb) {
            const int sub = NSUB == 1 ? 0 : s % NSUB, sp2 = NSUB == 1 ? s : s / NSUB;
            const int m = n_planes == 1 ? sp2 : sp2 / n_planes, pl = sp2 - m * n_planes;
            const int n = cb + sLive[m];
            const int dx = dpi_min + STEP * (n % ndpi), dy = dpj_min + STEP * (n / ndpi);
            const double2 *src = fn + fm.base + int64_t(pl) * fm.plane_stride +
                                 int64_t(P * dy - fm.rmin) * fm.ncols + (P * dx - fm.cmin);
            const uint32_t g = gs + uint32_t(s), slot = g % K;
            const int nrows = V == kOffCoarserSrc4 ? (sub < 4 ? 28 : 16) : LatCls<V>::SLOT_ROWS;
            // Producer acquire: the slot's previous use (stage g - K) was read through the generic proxy by all eight
            // warps, each of which arrived on empty[slot] afterwards; the TMA writes below go through the async proxy
            // and are issued only after that phase has completed -- the mbarrier empty / full protocol, for the
            // refills inside a chunk and for the first K stages of a chunk alike.
            if (g >= uint32_t(K)) mbar_wait(&empty[slot], ((g / K) - 1u) & 1u);
            if (lane == 0) mbar_expect_tx(&full[slot], uint32_t(nrows) * TROW * 16);
            __syncwarp();
            for (int r = lane; r < nrows; r += 32) {
                // table row held by slot row r
                const int nn = V == kOffCoarserSrc4 ? 16 * sub + r
                             : V == kOffFinerSrc4   ? r * C::RA + sub
                                                    : (r % C::RPC) * C::RA + r / C::RPC;
                tma_bulk_g2s(ring + slot * TBUF + r * TROW, src + int64_t(nn) * fm.ncols, TROW * 16, &full[slot]);
            }
        };
        // correlation of target patch `my_patch` with the vertices of source patch b (weights of plane pl) through
        // the table T: correlate_patch, shared with patch_offset_kernel
        auto consume = [&](int b, int pl, int sub, const double2 *T) {
            const double2 *src = reinterpret_cast<const double2 *>(wq + int64_t(pl) * w_plane_stride + int64_t(b) * kPatchQStride);
            const int flags = __ldg(pflags + b) | flags_or;    // flags_or = 3: all 17 x 17 vertices (own-cell weights)
            if (V == kOffCoarserSrc4)            // slot row 0 = table row 16 sub; source rows 4 sub .. 4 sub + 3
                correlate_patch<V>(T - 16 * sub * TROW, src, flags, l, h, ax, ay, 4 * sub, min(4 * sub + 3, P), 1);
            else if (V == kOffFinerSrc4)         // slot row 0 = stored row sub RPC; source rows sub, sub + 4, ...
                correlate_patch<V>(T - sub * C::RPC * TROW, src, flags, l, h, ax, ay, sub, P, 4);
            else
                correlate_patch<V>(T, src, flags, l, h, ax, ay, 0, P, 1);
        };
        __syncthreads();                                                  // sPos is visible

        for (int cb = n0; cb < n1; cb += kChunkOffsets) {
            const int nc = min(kChunkOffsets, n1 - cb);
            // (1) source patch of every (offset, target patch) of the chunk, all threads
            for (int idx = tid; idx < nc * 8; idx += kOffWarps * 32) {
                const int c = idx >> 3, w = idx & 7, n = cb + c;
                int b = -1;
                if (w < grp_n) {
                    const int dx = dpi_min + STEP * (n % ndpi), dy = dpj_min + STEP * (n / ndpi);
                    int bi, bj;
                    if (C::coarser) { bi = (sPos[2 * w] + dx) / F; bj = (sPos[2 * w + 1] + dy) / F; }   // exact: A + d is a multiple of F
                    else { bi = F * sPos[2 * w] + dx; bj = F * sPos[2 * w + 1] + dy; }
                    bi -= slev.pimin; bj -= slev.pjmin;
                    if (bi >= 0 && bi < slev.npx && bj >= 0 && bj < slev.npy) b = pmap[slev.map_off + bj * slev.npx + bi];
                }
                sB[idx] = b;
            }
            __syncthreads();
            // (2) the live offsets of the chunk, in order (warp 0)
            if (warp == 0) {
                int cnt = 0;
                for (int c0 = 0; c0 < nc; c0 += 32) {
                    const int c = c0 + lane;
                    bool live = false;
                    if (c < nc) {
#pragma unroll
                        for (int w = 0; w < 8; ++w) live = live || sB[c * 8 + w] >= 0;
                    }
                    const uint32_t mask = __ballot_sync(0xffffffffu, live);
                    if (live) sLive[cnt + __popc(mask & ((1u << lane) - 1u))] = c;
                    cnt += __popc(mask);
                }
                if (lane == 0) sMisc[1] = cnt;
            }
            __syncthreads();
            const int S = sMisc[1] * n_planes * NSUB;                     // stages of this chunk
            // (3) the ring: warp 0 fills the first K stages, afterwards the last warp to release a stage refills it
            // (full[slot]: TMA complete_tx -> consumers; empty[slot]: 8 consumer arrivals -> the issuing warp)
            if (warp == 0)
                for (int s = 0; s < min(K, S); ++s) issue_stage(s, cb);
            for (int s = 0; s < S; ++s) {
                const int sub = NSUB == 1 ? 0 : s % NSUB, sp2 = NSUB == 1 ? s : s / NSUB;
                const int m = n_planes == 1 ? sp2 : sp2 / n_planes, pl = sp2 - m * n_planes;
                const int b = sB[sLive[m] * 8 + warp];
                const uint32_t g = gs + uint32_t(s), slot = g % K;
                mbar_wait(&full[slot], (g / K) & 1u);                     // also for a warp without work: a warp
                if (my_patch >= 0 && b >= 0) consume(b, pl, sub, ring + slot * TBUF);   // never runs more than K stages ahead
                __syncwarp();
                // Consumer release: every warp arrives on empty[slot] (this is what orders its reads of the stage before
                // the refill, see issue_stage).  The counter only ELECTS the refilling warp -- the one that arrived last,
                // so that no warp waits for a slower one here; its wait on empty[slot] returns at once.
                int last = 0;
                if (lane == 0) {
                    mbar_arrive(&empty[slot]);
                    __threadfence_block();
                    last = atomicAdd(&sDone[slot], 1) == kOffWarps - 1;
                    if (last) atomicExch(&sDone[slot], 0);
                }
                last = __shfl_sync(0xffffffffu, last, 0);
                if (last && s + K < S) issue_stage(s + K, cb);
            }
            gs += uint32_t(S);
            __syncthreads();                                              // the chunk is drained: sB / sLive are free
        }
        if (my_patch >= 0) {
#pragma unroll
            for (int r = 0; r < kBlkR; ++r) {
                const int k = C::coarser ? F * (r % MT) + NCLS * h + r / MT : 8 * h + r;
                const int64_t lt = (int64_t(my_patch) * (P * P) + l * P + k) - first;
                if (lt >= 0 && lt < count) {
                    part[(int64_t(sp) * 2 + 0) * count + lt] = ax[r];
                    part[(int64_t(sp) * 2 + 1) * count + lt] = ay[r];
                }
            }
        }
    }
}

size_t lattice_smem_bytes(int V) {
    switch (V) {
        case 0: return LatCls<0>::smem;
        case 1: return LatCls<1>::smem;
        case 2: return LatCls<2>::smem;
        case 3: return LatCls<3>::smem;
        default: return LatCls<4>::smem;
    }
}

cudaError_t configure_lattice_kernels() {
    cudaError_t e = opt_in_max_smem(lattice_corr_kernel<0>, LatCls<0>::smem);
    if (e == cudaSuccess) e = opt_in_max_smem(lattice_corr_kernel<1>, LatCls<1>::smem);
    if (e == cudaSuccess) e = opt_in_max_smem(lattice_corr_kernel<2>, LatCls<2>::smem);
    if (e == cudaSuccess) e = opt_in_max_smem(lattice_corr_kernel<3>, LatCls<3>::smem);
    if (e == cudaSuccess) e = opt_in_max_smem(lattice_corr_kernel<4>, LatCls<4>::smem);
    return e;
}

template <int V>
void launch_lattice_corr_one(const DevLayout &d, const PatchArrays &pa, const LatticeArrays &la, const OffsetPlan &po,
                             int n_planes, int64_t first, int64_t count, double *part, int sms, cudaStream_t s) {
    const int list = offset_group_list(V);
    const int n_groups = po.n_groups[list];
    if (n_groups == 0) return;
    const PatchGroup *groups = pa.groups;
    for (int q = 0; q < list; ++q) groups += po.n_groups[q];
    const int grid = int(std::min<int64_t>(int64_t(po.n_split) * n_groups, int64_t(2) * sms));
    const double *wq = n_planes == 1 ? pa.wQ : la.wS;
    lattice_corr_kernel<V><<<grid, kOffWarps * 32, LatCls<V>::smem, s>>>(
        pa.info, pa.levels, groups, pa.pmap, wq, int64_t(pa.n_patches) * kPatchQStride, pa.pflags, la.fn, la.meta, n_planes,
        (n_planes > 1 && la.lin_neutral) ? 3 : 0, n_groups, po.n_split, po.first_patch, po.last_patch, first, count, part, d.queue + 1 + V);
}

void launch_lattice_corr(int V, const DevLayout &d, const PatchArrays &pa, const LatticeArrays &la, const OffsetPlan &po,
                         int n_planes, int64_t first, int64_t count, double *part, int sms, cudaStream_t s) {
    if (count == 0) return;
    switch (V) {
        case kOffSame: launch_lattice_corr_one<kOffSame>(d, pa, la, po, n_planes, first, count, part, sms, s); break;
        case kOffCoarserSrc: launch_lattice_corr_one<kOffCoarserSrc>(d, pa, la, po, n_planes, first, count, part, sms, s); break;
        case kOffFinerSrc: launch_lattice_corr_one<kOffFinerSrc>(d, pa, la, po, n_planes, first, count, part, sms, s); break;
        case kOffCoarserSrc4: launch_lattice_corr_one<kOffCoarserSrc4>(d, pa, la, po, n_planes, first, count, part, sms, s); break;
        default: launch_lattice_corr_one<kOffFinerSrc4>(d, pa, la, po, n_planes, first, count, part, sms, s); break;
    }
}

}  // namespace sg
