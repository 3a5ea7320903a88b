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
constexpr int kLatSmemBudget = 115712 - 256;

template <int V>
struct LatCls {
    using C = OffCls<V>;
    static constexpr int STAGE_BYTES = C::TBUF * 16;
    static constexpr int K_FIT = (kLatSmemBudget - kLatAuxBytes) / STAGE_BYTES;
    static constexpr int K = K_FIT < 1 ? 1 : (K_FIT > 6 ? 6 : K_FIT);        // ring depth: 6, 3, 3, 1, 1
    static constexpr size_t smem = size_t(K) * STAGE_BYTES + kLatAuxBytes;
};

template <int V>
__global__ void __launch_bounds__(kOffWarps * 32, 2)
lattice_corr_kernel(const PatchInfo *__restrict__ info, const PatchLevel *__restrict__ levels,
                    const PatchGroup *__restrict__ groups, const int32_t *__restrict__ pmap,
                    const double *__restrict__ wq, int64_t w_plane_stride, const int32_t *__restrict__ pflags,
                    const double2 *__restrict__ fn,
                    const FnLattice *__restrict__ meta, int n_planes, int n_groups, int n_split, int first_patch,
                    int last_patch, int64_t first, int64_t count, double *__restrict__ part,
                    unsigned int *__restrict__ queue) {
    using C = OffCls<V>;
    constexpr int P = 16, F = C::F, TROW = C::TROW, TBUF = C::TBUF, K = LatCls<V>::K;
    constexpr int STEP = C::coarser ? F : 1;                              // offsets keep A + d a multiple of F
    constexpr int NCLS = C::coarser ? F / 2 : 1, MT = kBlkR / NCLS;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2 *ring = reinterpret_cast<double2 *>(smem_raw);                 // [K][TBUF]
    int *sB = reinterpret_cast<int *>(ring + K * TBUF);                    // [kChunkOffsets][8]
    int *sLive = sB + kChunkOffsets * 8;                                   // [kChunkOffsets]
    uint64_t *full = reinterpret_cast<uint64_t *>(sLive + kChunkOffsets);  // [8]
    int *sDone = reinterpret_cast<int *>(full + 8);                        // [8]
    int *sPos = sDone + 8;                                                 // [8][2] patch position of target patch w
    int *sMisc = sPos + 16;                                                // [0] item, [1] live offsets of the chunk
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int l = lane & 15, h = lane >> 4;

    if (tid == 0) {
        for (int k = 0; k < K; ++k) { mbar_init(&full[k], 1); sDone[k] = 0; }
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

        // the copies of stage s of the current chunk (offset sLive[s / n_planes], plane s % n_planes), by one warp
        auto issue_stage = [&](int s, int cb) {
            const int m = n_planes == 1 ? s : s / n_planes, pl = s - m * n_planes;
            const int n = cb + sLive[m];
            const int dx = dpi_min + STEP * (n % ndpi), dy = dpj_min + STEP * (n / ndpi);
            const double2 *src = fn + fm.base + int64_t(pl) * fm.plane_stride +
                                 int64_t(P * dy - fm.rmin) * fm.ncols + (P * dx - fm.cmin);
            const uint32_t slot = (gs + uint32_t(s)) % K;
            if (lane == 0) mbar_expect_tx(&full[slot], C::ROWS * TROW * 16);
            __syncwarp();
            for (int pos = lane; pos < C::ROWS; pos += 32) {
                const int nn = (pos % C::RPC) * C::RA + pos / C::RPC;       // stored row pos holds table row nn
                tma_bulk_g2s(ring + slot * TBUF + pos * TROW, src + int64_t(nn) * fm.ncols, TROW * 16, &full[slot]);
            }
        };
        // correlation of target patch `my_patch` with the vertices of source patch b (weights of plane pl) through
        // the table T: correlate_patch, shared with patch_offset_kernel
        auto consume = [&](int b, int pl, const double2 *T) {
            const double2 *src = reinterpret_cast<const double2 *>(wq + int64_t(pl) * w_plane_stride + int64_t(b) * kPatchQStride);
            correlate_patch<V>(T, src, __ldg(pflags + b), l, h, ax, ay);
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
            const int S = sMisc[1] * n_planes;                            // stages of this chunk
            // (3) the ring: warp 0 fills the first K stages, afterwards the last warp to release a stage refills it
            if (warp == 0)
                for (int s = 0; s < min(K, S); ++s) issue_stage(s, cb);
            for (int s = 0; s < S; ++s) {
                const int m = n_planes == 1 ? s : s / n_planes, pl = s - m * n_planes;
                const int b = sB[sLive[m] * 8 + warp];
                const uint32_t g = gs + uint32_t(s), slot = g % K;
                mbar_wait(&full[slot], (g / K) & 1u);                     // also for a warp without work: a warp
                if (my_patch >= 0 && b >= 0) consume(b, pl, ring + slot * TBUF);   // never runs more than K stages ahead
                __syncwarp();
                int last = 0;
                if (lane == 0) {
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
        n_groups, po.n_split, po.first_patch, po.last_patch, first, count, part, d.queue + 1 + V);
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
