// sg_kernels_patch.cu -- S3 by lattice-offset reuse.
//
// The interaction sum M^x_t = sum_v w_v s(v) ln(|v|+r), M^y_t = sum_v w_v s(u) ln(|u|+r) (sg_kernels.cu header) is
// evaluated patch against patch.  For a target patch A (P x P cell centres, pitch cw_A) and a source patch B
// ((P+1)^2 vertices, pitch cw_B) every offset is
//     u = u00 + g (i rb - k ra),   v = v00 + g (j rb - l ra),     g = min(cw_A, cw_B), ra = cw_A/g, rb = cw_B/g,
// so only M^2 distinct (u, v) occur, M = P rb + (P-1) ra + 1, for P^2 (P+1)^2 pairs.  The CTA tabulates
//     T[n][m] = { s(v) ln(|v|+r), s(u) ln(|u|+r) }
// once per patch pair in shared memory (same sqrt / table-driven log as the direct kernel) and the pair sum becomes
// a correlation with the patch's own signed vertex weights w^B (cells of B only; the weights of all patches at a
// shared vertex add up to the deduplicated w_v, so the sum over patches is the same sum):
//     M^x[l][k] += sum_{j,i} w^B[j][i] T[j rb - l ra][i rb - k ra].x          (2 DFMA per pair)
// Two families of kernels:
//   patch_offset_kernel<V>       P = 16: one table per CTA shared by 8 target patches, 8 targets per thread, patch pairs
//                                up to two levels apart (five pair classes V);
//   patch_interaction_kernel<P>  P = 8 (one target per thread, one table per patch pair, pairs up to one level apart)
//                                and, for both P, the pairs farther apart (M^2 exceeds the pair count: no reuse left),
//                                which it sums directly, pair by pair.
// The separable ln|u| part, the coincidence rule and the epilogue are unchanged (finalise_kernel).
#include <algorithm>

#include "sg_device.cuh"
#include "sg_kernels_patch.cuh"
#include "sg_patch_device.cuh"

namespace sg {

constexpr int kPatchMaxM = 48;        // table path for |level difference| <= 1: M <= 3P <= 48

// Per-patch vertex weights = the DEDUPLICATED signed vertex weights w_v (vertex_weights_kernel: the sum of +-sigma over
// all <= 4 cells around v, whichever patch they belong to), each global vertex handed to exactly ONE owner patch
// (pvmap[p][j][i] = vertex index if patch p owns vertex (i, j) of its (P+1)^2 lattice, else -1; sg_create picks the
// finest patch that has the vertex, the lowest index among equals).  The sum over patches is then the same sum over
// vertices as in the direct kernel, and the weights a patch correlates are second differences of sigma (small for a
// smooth disk) instead of one-sided patch-edge sums that only cancel against the neighbouring patch: an order of
// magnitude less rounding error, for the slope path in particular.
// wP: [j][i] rows P+1 apart (generic kernel).  wQ (P = 16 only, may be null): rows 18 apart, column 17 zero, so that the
// offset-table kernels read aligned 16-byte pairs.  n_planes = 1: plane 0 = w[v];  3 (slope path): planes -W0, a, c
// from wl[3 v + {0, 1, 2}] (vertex_weights_lin_kernel), wQ layout only.
__global__ void patch_weights_kernel(const double *__restrict__ w, const int32_t *__restrict__ pvmap,
                                     double *__restrict__ wP, double *__restrict__ wQ, int P, int wstride,
                                     int n_planes, int64_t q_plane_stride) {
    const int p = blockIdx.x, NV = (P + 1) * (P + 1);
    for (int e = threadIdx.x; e < max(wstride, kPatchQStride); e += blockDim.x) {
        if (n_planes == 1 && e < wstride) {
            const int v = e < NV ? pvmap[int64_t(p) * NV + e] : -1;
            wP[int64_t(p) * wstride + e] = v >= 0 ? w[v] : 0.0;
        }
        if (wQ && e < kPatchQStride) {
            const int i = e % (P + 2), j = e / (P + 2);
            const int v = i <= P ? pvmap[int64_t(p) * NV + j * (P + 1) + i] : -1;
            if (n_planes == 1) wQ[int64_t(p) * kPatchQStride + e] = v >= 0 ? w[v] : 0.0;
            else {
                const int64_t o = int64_t(p) * kPatchQStride + e;
                wQ[o] = v >= 0 ? -w[3 * int64_t(v)] : 0.0;
                wQ[q_plane_stride + o] = v >= 0 ? w[3 * int64_t(v) + 1] : 0.0;
                wQ[2 * q_plane_stride + o] = v >= 0 ? w[3 * int64_t(v) + 2] : 0.0;
            }
        }
    }
}

// Alternative per-patch weights (SG_LATTICE_NEUTRAL_WEIGHTS, sg_api.cu): the corner sums of the patch's OWN cells only, on
// all (P+1)^2 vertices.  Every patch is then neutral (its weights sum to zero, and so do their first moments), so a
// patch pair contributes a small quadrupole-like number instead of a monopole that only cancels against the
// neighbouring patches' sums: less rounding on steep, deep hierarchies, at the price of 289 instead of 256 vertices.
__global__ void patch_weights_owncell_kernel(const double *__restrict__ sigma, double *__restrict__ wP, double *__restrict__ wQ,
                                             int P, int wstride) {
    const int p = blockIdx.x;
    const double *s = sigma + int64_t(p) * P * P;
    for (int e = threadIdx.x; e < wstride; e += blockDim.x) {
        double w = 0.0;
        if (e < (P + 1) * (P + 1)) {
            const int i = e % (P + 1), j = e / (P + 1);
            if (i >= 1 && j >= 1) w += s[(j - 1) * P + (i - 1)];
            if (i < P && j >= 1) w -= s[(j - 1) * P + i];
            if (i >= 1 && j < P) w -= s[j * P + (i - 1)];
            if (i < P && j < P) w += s[j * P + i];
            if (wQ) {
                wQ[int64_t(p) * kPatchQStride + j * (P + 2) + i] = w;
                if (i == P) wQ[int64_t(p) * kPatchQStride + j * (P + 2) + P + 1] = 0.0;
            }
        }
        wP[int64_t(p) * wstride + e] = w;
    }
}
void launch_patch_weights_owncell(const PatchArrays &pa, const double *sigma, cudaStream_t s) {
    patch_weights_owncell_kernel<<<pa.n_patches, 128, 0, s>>>(sigma, pa.wP, pa.wQ, pa.P, pa.wstride);
}

void launch_patch_weights(const PatchArrays &pa, const double *w, cudaStream_t s) {
    patch_weights_kernel<<<pa.n_patches, 128, 0, s>>>(w, pa.pvmap, pa.wP, pa.wQ, pa.P, pa.wstride, 1, 0);
}

// The slope-path counterpart of patch_weights_owncell_kernel: -W0, a, c of a patch vertex from the <= 4 cells of the
// SAME patch, W0 = sum s (sigma + dx (xbar - x_c) + dy (ybar - y_c)), a = sum s dx, c = sum s dy (slopes per lattice
// unit; xbar - x_c = +-hh), in the [17][18] layout.
__global__ void patch_weights_lin_owncell_kernel(const double *__restrict__ sigma, const double *__restrict__ dx,
                                                 const double *__restrict__ dy, const double *__restrict__ patch_hh,
                                                 double unit, double *__restrict__ wS, int64_t plane_stride) {
    constexpr int P = 16;
    const int p = blockIdx.x;
    const int64_t c0 = int64_t(p) * P * P;
    const double hh = patch_hh[p];
    for (int e = threadIdx.x; e < kPatchQStride; e += blockDim.x) {
        const int i = e % (P + 2), j = e / (P + 2);
        double W0 = 0.0, a = 0.0, c = 0.0;
        if (i <= P) {
            // cell (ci, cj) has the vertex as its NE (+), NW (-), SE (-), SW (+) corner
            const int ci[4] = {i - 1, i, i - 1, i}, cj[4] = {j - 1, j - 1, j, j};
            const double sg[4] = {1.0, -1.0, -1.0, 1.0};
            const double ex[4] = {1.0, -1.0, 1.0, -1.0}, ey[4] = {1.0, 1.0, -1.0, -1.0};
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (ci[k] >= 0 && ci[k] < P && cj[k] >= 0 && cj[k] < P) {
                    const int64_t cell = c0 + cj[k] * P + ci[k];
                    const double dxl = dx[cell] * unit, dyl = dy[cell] * unit;
                    W0 += sg[k] * (sigma[cell] + ex[k] * dxl * hh + ey[k] * dyl * hh);
                    a += sg[k] * dxl;
                    c += sg[k] * dyl;
                }
        }
        const int64_t o = int64_t(p) * kPatchQStride + e;
        wS[o] = -W0;
        wS[plane_stride + o] = a;
        wS[2 * plane_stride + o] = c;
    }
}

void launch_patch_weights_lin_owncell(const PatchArrays &pa, const double *sigma, const double *dx, const double *dy,
                                      const double *patch_hh, double unit, double *wS, cudaStream_t s) {
    patch_weights_lin_owncell_kernel<<<pa.n_patches, 128, 0, s>>>(sigma, dx, dy, patch_hh, unit, wS,
                                                                  int64_t(pa.n_patches) * kPatchQStride);
}

void launch_patch_weights_lin(const PatchArrays &pa, const double *wl, double *wS, cudaStream_t s) {
    patch_weights_kernel<<<pa.n_patches, 128, 0, s>>>(wl, pa.pvmap, nullptr, wS, pa.P, pa.wstride, 3,
                                                      int64_t(pa.n_patches) * kPatchQStride);
}

__device__ __forceinline__ double2 pair_terms(double u, double v, const char *tabb, uint32_t keep) {
    const double q = fma(u, u, v * v);
    const double y0 = rsqrt_approx(q);
    const double t = q * y0;
    const double e = fma(-t, y0, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double r = fma(t, p * e, t);
    return make_double2(flip_sign_by(fast_ln(fabs(v) + r, tabb, keep), v),
                        flip_sign_by(fast_ln(fabs(u) + r, tabb, keep), u));
}

template <int P>
__global__ void __launch_bounds__(P * P, (P == 16 ? 2 : 4))
patch_interaction_kernel(const PatchInfo *__restrict__ info, const double *__restrict__ wP, int wstride,
                         const double *__restrict__ lntab_g, int tab_idx0, int tab_entries, int n_patches,
                         int patches_per_split, int n_split, int first_patch, int n_tpatches, int64_t first,
                         int64_t count, double *__restrict__ part, unsigned int *__restrict__ queue, uint32_t keep,
                         int skip_near) {
    constexpr int NT = P * P, NV = (P + 1) * (P + 1);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2 *stab2 = reinterpret_cast<double2 *>(smem_raw);                        // kPatchMaxM^2 pair table
    double *sw = reinterpret_cast<double *>(stab2 + kPatchMaxM * kPatchMaxM);     // weights of B
    double *stab = sw + ((NV + 1) & ~1);                                          // log table
    __shared__ int s_item;
    const int tid = threadIdx.x, k = tid % P, l = tid / P;

    for (int i = tid; i < tab_entries; i += NT) stab[i] = lntab_g[i];
    __syncthreads();
    const char *tabb = reinterpret_cast<const char *>(stab) - int64_t(tab_idx0) * 8 - 4;

    const int n_items = n_tpatches * n_split;
    while (true) {
        __syncthreads();           // every thread has read s_item of the previous item (an item whose source patches
                                   // are all skipped runs no other barrier) and is done with sw / stab2
        if (tid == 0) s_item = int(atomicAdd(queue, 1u));
        __syncthreads();
        const int item = s_item;
        if (item >= n_items) break;
        const int ta = item / n_split, sp = item - ta * n_split;
        const PatchInfo A = info[first_patch + ta];
        const int b0 = sp * patches_per_split, b1 = min(n_patches, b0 + patches_per_split);
        const int xt = A.X0 + k * A.cw + A.cw / 2, yt = A.Y0 + l * A.cw + A.cw / 2;     // lattice, exact
        double ax = 0.0, ay = 0.0;

        for (int b = b0; b < b1; ++b) {
            const PatchInfo B = info[b];
            if (abs(A.level - B.level) < skip_near) continue;     // done by patch_offset_kernel (CTA-uniform)
            __syncthreads();                                   // previous pair is done with sw / stab2
            for (int e = tid; e < NV; e += NT) sw[e] = wP[int64_t(b) * wstride + e];
            const int dl = A.level - B.level;
            if (dl >= -1 && dl <= 1) {
                const int g = min(A.cw, B.cw), ra = A.cw / g, rb = B.cw / g;
                const int M = P * rb + (P - 1) * ra + 1, mmin = (P - 1) * ra;
                const int u00 = B.X0 - (A.X0 + A.cw / 2), v00 = B.Y0 - (A.Y0 + A.cw / 2);
                for (int e = tid; e < M * M; e += NT) {
                    const int mm = e % M, nn = e / M;
                    stab2[e] = pair_terms(double(u00 + (mm - mmin) * g), double(v00 + (nn - mmin) * g), tabb, keep);
                }
                __syncthreads();
                const double2 *trow = stab2 + ((P - 1 - l) * ra) * M + (P - 1 - k) * ra;
                const double *wrow = sw;
                for (int j = 0; j <= P; ++j, trow += rb * M, wrow += P + 1) {
#pragma unroll
                    for (int i = 0; i <= P; ++i) {
                        const double2 T = trow[i * rb];
                        const double w = wrow[i];
                        ax = fma(w, T.x, ax);
                        ay = fma(w, T.y, ay);
                    }
                }
            } else {
                // far pair: every (target, vertex) pair directly, column by column as in interaction_kernel: u, u^2 and
                // s(u) once per column, v by exact integer steps, 21 FP64-pipe instructions per pair
                __syncthreads();
                const double dv = double(B.cw), v0 = double(B.Y0 - yt);
                for (int i = 0; i <= P; ++i) {
                    const double u = double(B.X0 + i * B.cw - xt), uu = u * u, au = fabs(u);
                    double cy = 0.0, v = v0;
#pragma unroll 4
                    for (int j = 0; j <= P; ++j, v += dv) {
                        const double w = sw[j * (P + 1) + i];
                        const double q = fma(v, v, uu);
                        const double y0 = rsqrt_approx(q);
                        const double t = q * y0;
                        const double e = fma(-t, y0, 1.0);
                        const double pp = fma(0.375, e, 0.5);
                        const double r = fma(t, pp * e, t);
                        ax = fma(w, flip_sign_by(fast_ln(fabs(v) + r, tabb, keep), v), ax);
                        cy = fma(w, fast_ln(au + r, tabb, keep), cy);
                    }
                    ay += flip_sign_by(cy, u);
                }
            }
        }
        const int64_t lt = (int64_t(first_patch + ta) * NT + tid) - first;      // local index in the target range
        if (lt >= 0 && lt < count) {
            part[(int64_t(sp) * 2 + 0) * count + lt] = ax;
            part[(int64_t(sp) * 2 + 1) * count + lt] = ay;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Patch pairs three or more levels apart, P = 16 (table side >= 137: no reuse left): every (target, vertex) pair
// directly, 21 FP64-pipe instructions (28 with the slope terms, LIN), column by column as in interaction_kernel
// (u, u^2 and s(u) once per column, v by exact integer steps).  Work item = (target patch, split of the list of the
// source patches that are far from the target's level); the lists are per level (far_meta[2 l] = first entry,
// [2 l + 1] = count), so every item of a level carries the same work.  Weights in the wQ layout (rows 18 apart);
// LIN: planes -W0, a, c (patch_weights_kernel) and the partial sums hold the main parts of F/G as in
// interaction_lin_kernel.
// ------------------------------------------------------------------------------------------------
template <bool LIN>
__global__ void __launch_bounds__(256, 2)
patch_far_kernel(const PatchInfo *__restrict__ info, const double *__restrict__ wq, int64_t w_plane_stride,
                 const int32_t *__restrict__ far_list, const int32_t *__restrict__ far_meta,
                 const double *__restrict__ lntab_g, int tab_idx0, int tab_entries, int n_split, int first_patch,
                 int n_tpatches, int64_t first, int64_t count, double *__restrict__ part,
                 unsigned int *__restrict__ queue, uint32_t keep) {
    constexpr int P = 16, NT = P * P, NPL = LIN ? 3 : 1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *sw = reinterpret_cast<double *>(smem_raw);                    // [NPL][kPatchQStride] weights of B
    double *stab = sw + NPL * kPatchQStride;                              // log table
    __shared__ int s_item;
    const int tid = threadIdx.x, k = tid % P, l = tid / P;

    for (int i = tid; i < tab_entries; i += NT) stab[i] = lntab_g[i];
    const char *tabb = reinterpret_cast<const char *>(stab) - int64_t(tab_idx0) * 8 - 4;

    const int n_items = n_tpatches * n_split;
    while (true) {
        __syncthreads();
        if (tid == 0) s_item = int(atomicAdd(queue, 1u));
        __syncthreads();
        const int item = s_item;
        if (item >= n_items) break;
        const int ta = item / n_split, sp = item - ta * n_split;
        const PatchInfo A = info[first_patch + ta];
        const int f0 = far_meta[2 * A.level], fc = far_meta[2 * A.level + 1];
        const int per = (fc + n_split - 1) / n_split;
        const int b0 = sp * per, b1 = min(fc, b0 + per);
        const int xt = A.X0 + k * A.cw + A.cw / 2, yt = A.Y0 + l * A.cw + A.cw / 2;     // lattice, exact
        double ax = 0.0, ay = 0.0;
        for (int bb = b0; bb < b1; ++bb) {
            const int b = far_list[f0 + bb];
            const PatchInfo B = info[b];
            __syncthreads();                                   // previous source patch is done with sw
            for (int e = tid; e < NPL * kPatchQStride; e += NT)
                sw[e] = wq[int64_t(e / kPatchQStride) * w_plane_stride + int64_t(b) * kPatchQStride + e % kPatchQStride];
            __syncthreads();
            const double dv = double(B.cw), v0 = double(B.Y0 - yt);
            for (int i = 0; i <= P; ++i) {
                const double u = double(B.X0 + i * B.cw - xt), uu = u * u, au = fabs(u);
                double cy = 0.0, cx2 = 0.0, cy1 = 0.0, v = v0;
#pragma unroll 4
                for (int j = 0; j <= P; ++j, v += dv) {
                    const double w = sw[j * (P + 2) + i];
                    const double q = fmax(fma(v, v, uu), 0.5);        // 0 only for a hole of a padded layout (discarded)
                    const double y0 = rsqrt_approx(q);
                    const double t = q * y0;
                    const double e = fma(-t, y0, 1.0);
                    const double pp = fma(0.375, e, 0.5);
                    const double r = fma(t, pp * e, t);
                    const double sl1 = flip_sign_by(fast_ln(fabs(v) + r, tabb, keep), v);
                    const double l2 = fast_ln(au + r, tabb, keep);
                    if (!LIN) {
                        ax = fma(w, sl1, ax);
                        cy = fma(w, l2, cy);
                    } else {
                        // w = -W0;  Wt = W0 - u a - v c;  x: -Wt s(v)L1 + a v s(u)L2 - c r;  y: -Wt s(u)L2 + c u s(v)L1 - a r
                        const double a = sw[kPatchQStride + j * (P + 2) + i], c = sw[2 * kPatchQStride + j * (P + 2) + i];
                        const double mwt = fma(v, c, fma(u, a, w));           // -Wt
                        ax = fma(mwt, sl1, ax);
                        ax = fma(-c, r, ax);
                        cx2 = fma(a * v, l2, cx2);
                        cy = fma(mwt, l2, cy);
                        cy1 = fma(c, sl1, cy1);
                        ay = fma(-a, r, ay);
                    }
                }
                ay += flip_sign_by(cy, u);
                if (LIN) {
                    ax += flip_sign_by(cx2, u);
                    ay = fma(u, cy1, ay);
                }
            }
        }
        const int64_t lt = (int64_t(first_patch + ta) * NT + tid) - first;      // local index in the target range
        if (lt >= 0 && lt < count) {
            part[(int64_t(sp) * 2 + 0) * count + lt] = ax;
            part[(int64_t(sp) * 2 + 1) * count + lt] = ay;
        }
    }
}

size_t patch_far_smem_bytes(bool lin, int tab_entries) {
    return size_t(lin ? 3 : 1) * kPatchQStride * 8 + size_t(tab_entries) * 8;
}

cudaError_t configure_patch_far(int tab_entries) {
    cudaError_t e = opt_in_max_smem(patch_far_kernel<false>, patch_far_smem_bytes(false, tab_entries));
    if (e == cudaSuccess) e = opt_in_max_smem(patch_far_kernel<true>, patch_far_smem_bytes(true, tab_entries));
    return e;
}

void launch_patch_far(bool lin, const DevLayout &d, const PatchArrays &pa, const double *wq, const PatchPlan &pp,
                      int64_t first, int64_t count, double *part, cudaStream_t s) {
    if (count == 0) return;
    const int64_t stride = int64_t(pa.n_patches) * kPatchQStride;
    const size_t smem = patch_far_smem_bytes(lin, d.tab_entries);
    if (lin)
        patch_far_kernel<true><<<pp.grid, 256, smem, s>>>(pa.info, wq, stride, pa.far_list, pa.far_meta, d.lntab, d.tab_idx0,
                                                         d.tab_entries, pp.n_split, pp.first_patch, pp.n_tpatches, first,
                                                         count, part, d.queue, kLogKeepMask);
    else
        patch_far_kernel<false><<<pp.grid, 256, smem, s>>>(pa.info, wq, stride, pa.far_list, pa.far_meta, d.lntab, d.tab_idx0,
                                                          d.tab_entries, pp.n_split, pp.first_patch, pp.n_tpatches, first,
                                                          count, part, d.queue, kLogKeepMask);
}

// ------------------------------------------------------------------------------------------------
// Patch pairs at most two levels apart, P = 16: register-blocked correlation with ONE OFFSET TABLE PER CTA.
//
// The table of a patch pair depends only on the patch offset d = B - A (in units of the finer level's patch size)
// and on the pair class V (sg_kernels_patch.cuh): source level = target level (V = 0), F = 2 or 4 times coarser
// (V = 1, 3), F = 2 or 4 times finer (V = 2, 4).  A CTA takes a group of up to 8 target patches A_w of one level, one
// warp each (for a coarser source all of one residue class (pi, pj) mod F, so that the source patch (A_w + d) / F is
// integral for all of them or none) and walks over the offsets d of the class's box; for each d warp w looks up its
// source patch B_w in the source level's dense patch map (absent: the warp skips this offset).  All 256 threads
// tabulate T(d) together, double-buffered for F <= 2 (the table of offset n+1 is built while offset n is consumed, one
// CTA barrier per offset; consecutive offsets of a box row reuse the overlapping columns of the previous table); the
// 80 x 80 tables of F = 4 are single-buffered, one CTA per SM.  The log table of the pair function is read through L1.
//
// Correlation, 8 targets per thread, lane = l + 16 h (l = target row).  With vertex (i, j) of B and target (k, l) of A
// the table entry is T[j rb - l ra + 15 ra][i rb - k ra + 15 ra] (ra, rb = target / source pitch in units of g):
//   same level (ra = rb = 1): thread owns columns k = 8 h + r; entry column t + 8 - 8 h serves vertices i = t + r - 7;
//   coarser source (ra = 1, rb = F): thread owns NCLS = F / 2 column classes mod F of MT = 8 / NCLS targets,
//          k = F m + NCLS h + cc; entry column F t + F (1 - MT) + 15 - NCLS h - cc serves i = t + m - (MT - 1);
//   finer source (ra = F, rb = 1): thread owns k = 8 h + r; entry column t + 8 F (1 - h) serves i = t + F r - 7 F;
//          table rows are stored by row class (row j - F l + 15 F has the residue of j mod F, so the 16 lanes of a
//          half-warp read consecutive stored rows).
// One loaded entry serves up to 8 targets of a thread (16 DFMA per LDS.128); the vertex weights sit in registers
// (fully unrolled, compile-time indices; the ragged ends are removed at compile time).  Stored table rows are an odd
// number of entries apart so that the 8 lanes of an LDS.128 quarter-warp hit 8 different 16-byte bank groups.
// Every per-patch sum stays in one accumulator chain (split chains cancel badly).
// ------------------------------------------------------------------------------------------------
template <int V>
__global__ void __launch_bounds__(kOffWarps * 32, 2)
patch_offset_kernel(const PatchInfo *__restrict__ info, const PatchLevel *__restrict__ levels,
                    const PatchGroup *__restrict__ groups, const int32_t *__restrict__ pmap,
                    const double *__restrict__ wQ, const int32_t *__restrict__ pflags,
                    const double *__restrict__ lntab_g, int tab_idx0, int n_groups,
                    int n_split, int first_patch, int last_patch, int64_t first, int64_t count,
                    double *__restrict__ part, unsigned int *__restrict__ queue, uint32_t keep) {
    using C = OffCls<V>;
    constexpr int P = 16, F = C::F, M = C::M, MMIN = C::MMIN, TROW = C::TROW, TBUF = C::TBUF;
    constexpr int STEP = C::coarser ? F : 1;                              // offsets keep A + d a multiple of F
    // per thread and source row: coarser source: NCLS column classes of MT targets each, NT table steps;
    // otherwise 8 consecutive targets, NT table entries
    constexpr int NCLS = C::coarser ? F / 2 : 1, MT = kBlkR / NCLS;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2 *sT = reinterpret_cast<double2 *>(smem_raw);                   // [2 or 1][TBUF] offset tables
    __shared__ int s_item;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int l = lane & 15, h = lane >> 4;

    const int n_items = n_groups * n_split;
    while (true) {
        __syncthreads();
        if (tid == 0) s_item = int(atomicAdd(queue, 1u));
        __syncthreads();
        const int item = s_item;
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
        const double g = double(min(lev.cw, slev.cw));

        // lane w < grp_n of every warp holds the patch position of target patch A_w (for the map look-ups)
        int api = 0, apj = 0;
        if (lane < grp_n) {
            const PatchInfo A = info[gp->patch[lane]];
            api = A.X0 / (P * lev.cw);
            apj = A.Y0 / (P * lev.cw);
        }
        const int my_patch = warp < grp_n ? gp->patch[warp] : -1;
        double ax[kBlkR], ay[kBlkR];
#pragma unroll
        for (int r = 0; r < kBlkR; ++r) { ax[r] = 0.0; ay[r] = 0.0; }

        // source patch of this warp at offset n (or -1), and whether any warp of the CTA has one
        auto lookup = [&](int n, bool &any) -> int {
            int b = -1;
            if (n < n1 && lane < grp_n) {
                const int dx = dpi_min + STEP * (n % ndpi), dy = dpj_min + STEP * (n / ndpi);
                int bi, bj;
                if (C::coarser) { bi = (api + dx) / F; bj = (apj + dy) / F; }     // exact: A + d is a multiple of F
                else { bi = F * api + dx; bj = F * apj + dy; }
                bi -= slev.pimin; bj -= slev.pjmin;
                if (bi >= 0 && bi < slev.npx && bj >= 0 && bj < slev.npy) b = pmap[slev.map_off + bj * slev.npx + bi];
            }
            any = __ballot_sync(0xffffffffu, b >= 0) != 0u;
            return __shfl_sync(0xffffffffu, b, warp & 7);
        };
        // T[row][col] = pair function at u = B.X0 - x_centre(A, k = 0) + (col - MMIN) g, likewise v; for a finer
        // source the rows are stored by row class (row % RA): the 16 lanes of a half-warp read consecutive stored rows
        // Consecutive offsets of one box row shift the table by SHIFT columns: with `prev` (the table of offset n-1,
        // complete and read-only while table n is built) only the last SHIFT columns are evaluated, the others copied.
        auto build = [&](int n, double2 *T, const double2 *prev) {
            constexpr int SHIFT = STEP * P;                               // columns (units of g) between offsets d, d + STEP
            const double u00 = double((dpi_min + STEP * (n % ndpi)) * P) * g - 0.5 * double(lev.cw);
            const double v00 = double((dpj_min + STEP * (n / ndpi)) * P) * g - 0.5 * double(lev.cw);
            const bool reuse = SHIFT < M && prev != nullptr && n % ndpi != 0;
            const int m0 = reuse ? M - SHIFT : 0, ncol = M - m0;          // columns [m0, M) are evaluated
#pragma unroll 2
            for (int e = tid; e < M * ncol; e += kOffWarps * 32) {
                const int mm = m0 + e % ncol, nn = e / ncol;
                const int pos = nn / C::RA + (nn % C::RA) * C::RPC;
                T[pos * TROW + mm] = pair_terms_g(fma(double(mm - MMIN), g, u00), fma(double(nn - MMIN), g, v00),
                                                  lntab_g, tab_idx0, keep);
            }
            if (reuse)
                for (int e = tid; e < C::ROWS * m0; e += kOffWarps * 32) {
                    const int mm = e % m0, pos = e / m0;
                    T[pos * TROW + mm] = prev[pos * TROW + mm + SHIFT];
                }
        };
        auto consume = [&](int b, const double2 *T) {
            correlate_patch_all<V>(T, reinterpret_cast<const double2 *>(wQ + int64_t(b) * kPatchQStride), __ldg(pflags + b),
                                   l, h, ax, ay);
        };

        bool any_cur = false, any_next = false;
        int b_cur = lookup(n0, any_cur), b_next = -1;
        if (C::DB) {
            if (any_cur) build(n0, sT, nullptr);
            __syncthreads();
            for (int n = n0; n < n1; ++n) {
                b_next = lookup(n + 1, any_next);
                if (!any_cur && !any_next) continue;             // nothing built, nothing consumed: no barrier needed
                if (any_next) build(n + 1, sT + ((n + 1 - n0) & 1) * TBUF, any_cur ? sT + ((n - n0) & 1) * TBUF : nullptr);
                if (my_patch >= 0 && b_cur >= 0) consume(b_cur, sT + ((n - n0) & 1) * TBUF);
                __syncthreads();
                b_cur = b_next; any_cur = any_next;
            }
        } else {                                                 // one table buffer: build, barrier, consume, barrier
            for (int n = n0; n < n1; ++n) {
                if (any_cur) {
                    build(n, sT, nullptr);
                    __syncthreads();
                    if (my_patch >= 0 && b_cur >= 0) consume(b_cur, sT);
                    __syncthreads();
                }
                b_cur = lookup(n + 1, any_cur);
            }
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

template <int V>
cudaError_t configure_patch_offset_one() {
    return opt_in_max_smem(patch_offset_kernel<V>, OffCls<V>::smem);
}

cudaError_t configure_patch_offset() {
    cudaError_t e = configure_patch_offset_one<0>();
    if (e == cudaSuccess) e = configure_patch_offset_one<1>();
    if (e == cudaSuccess) e = configure_patch_offset_one<2>();
    if (e == cudaSuccess) e = configure_patch_offset_one<3>();
    if (e == cudaSuccess) e = configure_patch_offset_one<4>();
    return e;
}

template <int V>
void launch_patch_offset_one(const DevLayout &d, const PatchArrays &pa, const OffsetPlan &po, int64_t first,
                             int64_t count, double *part, int sms, cudaStream_t s) {
    const int list = offset_group_list(V);
    const int n_groups = po.n_groups[list];
    if (n_groups == 0) return;
    const PatchGroup *groups = pa.groups;
    for (int q = 0; q < list; ++q) groups += po.n_groups[q];
    const int grid = int(std::min<int64_t>(int64_t(po.n_split) * n_groups, int64_t(2) * sms));
    patch_offset_kernel<V><<<grid, kOffWarps * 32, OffCls<V>::smem, s>>>(
        pa.info, pa.levels, groups, pa.pmap, pa.wQ, pa.pflags, d.lntab, d.tab_idx0, n_groups, po.n_split, po.first_patch,
        po.last_patch, first, count, part, d.queue + 1 + V, kLogKeepMask);
}

void launch_patch_offset(int V, const DevLayout &d, const PatchArrays &pa, const OffsetPlan &po, int64_t first,
                         int64_t count, double *part, int sms, cudaStream_t s) {
    if (count == 0) return;
    switch (V) {
        case kOffSame: launch_patch_offset_one<kOffSame>(d, pa, po, first, count, part, sms, s); break;
        case kOffCoarserSrc: launch_patch_offset_one<kOffCoarserSrc>(d, pa, po, first, count, part, sms, s); break;
        case kOffFinerSrc: launch_patch_offset_one<kOffFinerSrc>(d, pa, po, first, count, part, sms, s); break;
        case kOffCoarserSrc4: launch_patch_offset_one<kOffCoarserSrc4>(d, pa, po, first, count, part, sms, s); break;
        default: launch_patch_offset_one<kOffFinerSrc4>(d, pa, po, first, count, part, sms, s); break;
    }
}

size_t patch_smem_bytes(int P, int tab_entries) {
    const int NV = (P + 1) * (P + 1);
    return size_t(kPatchMaxM) * kPatchMaxM * 16 + size_t((NV + 1) & ~1) * 8 + size_t(tab_entries) * 8;
}

cudaError_t configure_patch_kernels(int P, int tab_entries) {
    const size_t bytes = patch_smem_bytes(P, tab_entries);
    if (P == 16) return opt_in_max_smem(patch_interaction_kernel<16>, bytes);
    return opt_in_max_smem(patch_interaction_kernel<8>, bytes);
}

void launch_patch_interaction(const DevLayout &d, const PatchArrays &pa, const PatchPlan &pp, int64_t first,
                              int64_t count, double *part, int skip_near, cudaStream_t s) {
    if (count == 0) return;
    if (pa.P == 16)
        patch_interaction_kernel<16><<<pp.grid, 256, pp.smem, s>>>(
            pa.info, pa.wP, pa.wstride, d.lntab, d.tab_idx0, d.tab_entries, pa.n_patches, pp.patches_per_split,
            pp.n_split, pp.first_patch, pp.n_tpatches, first, count, part, d.queue, kLogKeepMask, skip_near);
    else
        patch_interaction_kernel<8><<<pp.grid, 64, pp.smem, s>>>(
            pa.info, pa.wP, pa.wstride, d.lntab, d.tab_idx0, d.tab_entries, pa.n_patches, pp.patches_per_split,
            pp.n_split, pp.first_patch, pp.n_tpatches, first, count, part, d.queue, kLogKeepMask, skip_near);
}

}  // namespace sg
