// sg_kernels_lin.cu -- the first-order (slope) terms of PAPER.md:71-94 (Eq. 6) on the GPU, SURVEY.md 8(f1).
//
// With sigma_c(x,y) = sigma_c + dx_c (x - x_c) + dy_c (y - y_c) on every leaf the force is
//   F^x_t = G sum_c [ sigma_c K^{x,0} + dx_c K^{x,x} + dy_c K^{x,y} ],
//   K^{x,x} = (x_t - x_c) K^{x,0} + [[ v ln(u + r) ]],   K^{x,y} = (y_t - y_c) K^{x,0} - [[ r ]]      (z = 0)
// and the same with x and y exchanged (readings R1-R3, R6 of DESIGN.md).  Writing x_t - x_c = (xbar - x_c) - u
// at each corner regroups the cell sums by vertex, in lattice units with slopes per lattice unit:
//   F^x_t / G = sum_v [ Wt_v P(u,v) + a_v v ln(u + r) - c_v r ],   Wt_v = W0_v - u a_v - v c_v,
//   F^y_t / G = sum_v [ Wt_v P(v,u) + c_v u ln(v + r) - a_v r ],
//   W0_v = sum_{c in v} s (sigma_c + dx_c (xbar - x_c) + dy_c (ybar - y_c)),  a_v = sum s dx_c,  c_v = sum s dy_c,
// s = +1 for NE / SW corners and -1 for NW / SE.  P and ln(u + r) are evaluated in the cancellation-free forms
//   P(u,v) = -s(v) ln(|v|+r) - [v<0] 2 ln|u|,     ln(u+r) = s(u) ln(|u|+r) + [u<0] 2 ln|v|,
// whose separable parts (dropped on u == 0, resp. v == 0: the paper's modified primitive)
// go to the finalise kernel through three cumulative line tables per direction.
#include "sg_device.cuh"
#include "sg_kernels_lin.cuh"

namespace sg {

__device__ __forceinline__ double *slot_lin(double *vtile, int64_t slot) {
    return vtile + (slot / kTileSlots) * kTileLinDoubles + kChunksPerTile + 4 * (slot % kTileSlots);
}

// S2a': one thread per tile slot.  Writes {y, W0, a, c} of the slot, the chunk abscissa, and the flat wl[3v..].
__global__ void vertex_weights_lin_kernel(const int32_t *__restrict__ adj, const int32_t *__restrict__ slot_vertex,
                                          const int32_t *__restrict__ vky, const int32_t *__restrict__ chunk_x,
                                          const double *__restrict__ sigma, const double *__restrict__ dx,
                                          const double *__restrict__ dy, const double *__restrict__ patch_hh,
                                          int cells_per_patch, double unit, double *__restrict__ wl,
                                          double *__restrict__ vtile, int64_t n_slots) {
    const int64_t s = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (s >= n_slots) return;
    const int v = slot_vertex[s];
    double W0 = 0.0, a = 0.0, c = 0.0;
    if (v >= 0) {
        const int4 q = reinterpret_cast<const int4 *>(adj)[v];
        const int e[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (e[k] >= 0) {
                const int cell = e[k] >> 2, corner = e[k] & 3;       // 0 NE, 1 NW, 2 SE, 3 SW
                const double sgn = (corner == 1 || corner == 2) ? -1.0 : 1.0;
                const double ex = (corner == 0 || corner == 2) ? 1.0 : -1.0;   // xbar - x_c = +- hh
                const double ey = corner < 2 ? 1.0 : -1.0;
                const double hh = patch_hh[cell / cells_per_patch];
                const double dxl = dx[cell] * unit, dyl = dy[cell] * unit;     // slopes per lattice unit
                W0 += sgn * (sigma[cell] + ex * dxl * hh + ey * dyl * hh);
                a += sgn * dxl;
                c += sgn * dyl;
            }
        wl[3 * int64_t(v) + 0] = W0; wl[3 * int64_t(v) + 1] = a; wl[3 * int64_t(v) + 2] = c;
    }
    int vy = v;
    if (vy < 0) vy = slot_vertex[(s / kChunk) * kChunk];
    if (vy < 0) vy = 0;
    double *o = slot_lin(vtile, s);
    o[0] = double(vky[vy]); o[1] = W0; o[2] = a; o[3] = c;
    if (s % kChunk == 0) {
        const int64_t ch = s / kChunk;
        vtile[(ch / kChunksPerTile) * kTileLinDoubles + (ch % kChunksPerTile)] = double(chunk_x[ch]);
    }
}

// S2b': cumulative line weights, three per line.  mode 0 (columns, strictly below y_t):
//   TB[(i*n + c)*3 + {0,1,2}] = sum of { W0 - y_v c_v,  c_v,  a_v };   mode 1 (rows, strictly left of x_t):
//   TB[(i*n + r)*3 + {0,1,2}] = sum of { W0 - x_v a_v,  a_v,  c_v }.
__global__ void line_tables_lin_kernel(const int32_t *__restrict__ start, const int32_t *__restrict__ perm,
                                       const int32_t *__restrict__ vcoord, const double *__restrict__ wl,
                                       const int32_t *__restrict__ tcoord, int n_lines, int n_t, int mode,
                                       double *__restrict__ TB) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_lines) return;
    int p = start[c];
    const int e = start[c + 1];
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int i = 0; i < n_t; ++i) {
        const int t = tcoord[i];
        while (p < e) {
            const int v = perm ? perm[p] : p;
            if (vcoord[v] >= t) break;
            const double W0 = wl[3 * int64_t(v)], a = wl[3 * int64_t(v) + 1], cc = wl[3 * int64_t(v) + 2];
            const double along = double(vcoord[v]);
            if (mode == 0) { s0 += W0 - along * cc; s1 += cc; s2 += a; }
            else           { s0 += W0 - along * a;  s1 += a;  s2 += cc; }
            ++p;
        }
        double *o = TB + (int64_t(i) * n_lines + c) * 3;
        o[0] = s0; o[1] = s1; o[2] = s2;
    }
}

void launch_weights_lin(const DevLayout &d, const LinArrays &l, const double *sigma, const double *dx, const double *dy,
                        cudaStream_t s) {
    vertex_weights_lin_kernel<<<unsigned((d.n_slots + 255) / 256), 256, 0, s>>>(
        d.adj, d.slot_vertex, d.vky, d.chunk_x, sigma, dx, dy, l.patch_hh, l.cells_per_patch, l.unit, l.wl, l.vtile,
        d.n_slots);
    line_tables_lin_kernel<<<(d.nX + 127) / 128, 128, 0, s>>>(d.colstart, nullptr, d.vky, l.wl, d.tY, d.nX, d.ntY, 0, l.TBx3);
    line_tables_lin_kernel<<<(d.nY + 127) / 128, 128, 0, s>>>(d.rowstart, d.rowperm, d.vkx, l.wl, d.tX, d.nY, d.ntX, 1, l.TBy3);
}

// ------------------------------------------------------------------------------------------------
// S3': all-pairs kernel with slope terms.  Same structure as interaction_kernel (persistent CTAs, item queue,
// TMA-staged chunk tiles, T targets per thread in registers); per pair 28 FP64-pipe instructions:
//   v, q (2)  sqrt (5)  a1, a2 (2)  two logs (10)  Wt = W0 - u a - v c (2)  a*v (1)  six accumulations (6).
// Terms whose sign is s(u) are summed per chunk (u is shared by the chunk) and signed once at its end.
// The partial sums hold the main parts of F/G directly:
//   x:  -Wt s(v) L1 + a v s(u) L2 - c r        y:  -Wt s(u) L2 + c u s(v) L1 - a r
// ------------------------------------------------------------------------------------------------
constexpr int kLinT = 4;
int lin_targets_per_thread() { return kLinT; }

template <int T>
__global__ void __launch_bounds__(kThreads, 2)
interaction_lin_kernel(const double2 *__restrict__ tgt, const double *__restrict__ vtile,
                       const double *__restrict__ lntab_g, int tab_idx0, int tab_entries, int n_tiles,
                       int tiles_per_split, int n_split, int n_tblocks, int64_t first, int64_t count,
                       double *__restrict__ part, unsigned int *__restrict__ queue, uint32_t keep) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *stile = reinterpret_cast<double *>(smem_raw);
    uint64_t *full = reinterpret_cast<uint64_t *>(stile + kStages * kTileLinDoubles);
    double *stab = reinterpret_cast<double *>(full + 8);
    __shared__ int s_item;
    const int tid = threadIdx.x;

    for (int i = tid; i < tab_entries; i += kThreads) stab[i] = lntab_g[i];
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const char *tabb = reinterpret_cast<const char *>(stab) - int64_t(tab_idx0) * 8 - 4;

    uint32_t it = 0;
    const int n_items = n_tblocks * n_split;
    while (true) {
        if (tid == 0) s_item = int(atomicAdd(queue, 1u));
        __syncthreads();
        const int item = s_item;
        if (item >= n_items) break;
        const int tb = item / n_split, sp = item - tb * n_split;
        const int tile0 = sp * tiles_per_split;
        const int ntile = min(tiles_per_split, n_tiles - tile0);

        double xt[T], yt[T], ax[T], ay[T];
#pragma unroll
        for (int k = 0; k < T; ++k) {
            int64_t lt = int64_t(tb) * (kThreads * T) + k * kThreads + tid;
            if (lt >= count) lt = count - 1;
            const double2 p = tgt[first + lt];
            xt[k] = p.x; yt[k] = p.y; ax[k] = 0.0; ay[k] = 0.0;
        }
        if (tid == 0) {
            const int pre = min(kStages, ntile);
            for (int i = 0; i < pre; ++i) {
                const uint32_t st = (it + i) % kStages;
                mbar_expect_tx(&full[st], kTileLinDoubles * 8);
                tma_bulk_g2s(stile + st * kTileLinDoubles, vtile + int64_t(tile0 + i) * kTileLinDoubles,
                             kTileLinDoubles * 8, &full[st]);
            }
        }
        for (int i = 0; i < ntile; ++i, ++it) {
            const uint32_t st = it % kStages;
            mbar_wait(&full[st], (it / kStages) & 1u);
            const double *sx = stile + st * kTileLinDoubles;
            const double2 *sv = reinterpret_cast<const double2 *>(sx + kChunksPerTile);
#pragma unroll 1
            for (int c = 0; c < kChunksPerTile; ++c) {
                const double xc = sx[c];
                double u[T], uu[T], cx2[T], cy[T], cy1[T];
#pragma unroll
                for (int k = 0; k < T; ++k) {
                    u[k] = xc - xt[k]; uu[k] = u[k] * u[k];
                    cx2[k] = 0.0; cy[k] = 0.0; cy1[k] = 0.0;
                }
#pragma unroll 4
                for (int j = 0; j < kChunk; ++j) {
                    const double2 yw = sv[2 * (c * kChunk + j)];          // {y, W0}
                    const double2 ac = sv[2 * (c * kChunk + j) + 1];      // {a, c}
#pragma unroll
                    for (int k = 0; k < T; ++k) {
                        const double v = yw.x - yt[k];
                        const double q = fma(v, v, uu[k]);
                        const double y0 = rsqrt_approx(q);
                        const double t = q * y0;
                        const double e = fma(-t, y0, 1.0);
                        const double p = fma(0.375, e, 0.5);
                        const double r = fma(t, p * e, t);
                        const double sl1 = flip_sign_by(fast_ln(fabs(v) + r, tabb, keep), v);   // s(v) L1
                        const double l2 = fast_ln(fabs(u[k]) + r, tabb, keep);
                        const double wt = fma(-v, ac.y, fma(-u[k], ac.x, yw.y));                // W0 - u a - v c
                        ax[k] = fma(-wt, sl1, ax[k]);
                        ax[k] = fma(-ac.y, r, ax[k]);
                        cx2[k] = fma(ac.x * v, l2, cx2[k]);
                        cy[k] = fma(wt, l2, cy[k]);
                        cy1[k] = fma(ac.y, sl1, cy1[k]);
                        ay[k] = fma(-ac.x, r, ay[k]);
                    }
                }
#pragma unroll
                for (int k = 0; k < T; ++k) {
                    ax[k] += flip_sign_by(cx2[k], u[k]);
                    ay[k] -= flip_sign_by(cy[k], u[k]);
                    ay[k] = fma(u[k], cy1[k], ay[k]);
                }
            }
            __syncthreads();
            if (tid == 0 && i + kStages < ntile) {
                mbar_expect_tx(&full[st], kTileLinDoubles * 8);
                tma_bulk_g2s(stile + st * kTileLinDoubles, vtile + int64_t(tile0 + i + kStages) * kTileLinDoubles,
                             kTileLinDoubles * 8, &full[st]);
            }
        }
#pragma unroll
        for (int k = 0; k < T; ++k) {
            const int64_t lt = int64_t(tb) * (kThreads * T) + k * kThreads + tid;
            if (lt < count) {
                part[(int64_t(sp) * 2 + 0) * count + lt] = ax[k];
                part[(int64_t(sp) * 2 + 1) * count + lt] = ay[k];
            }
        }
    }
}

size_t interaction_lin_smem_bytes(int tab_entries) {
    return size_t(kStages) * kTileLinDoubles * 8 + 64 + size_t(tab_entries) * 8;
}

cudaError_t configure_lin_kernels(int tab_entries) {
    return opt_in_max_smem(interaction_lin_kernel<kLinT>, interaction_lin_smem_bytes(tab_entries));
}

void launch_interaction_lin(const DevLayout &d, const LinArrays &l, const ForcePlan &p, cudaStream_t s) {
    if (p.count == 0) return;
    interaction_lin_kernel<kLinT><<<p.grid, kThreads, p.smem, s>>>(d.tgt, l.vtile, d.lntab, d.tab_idx0, d.tab_entries,
                                                                  d.n_tiles, p.tiles_per_split, p.n_split, p.n_tblocks,
                                                                  p.first, p.count, d.part, d.queue, kLogKeepMask);
}

// S4' + S5': separable parts through the line tables, split reduction, scaling by G (F = G (main + sep)).
//   sep_x = -2 sum_{X != x_t} ln|X-x_t| [T0 + y_t T1 - (X-x_t) T2] + 2 sum_{Y != y_t} (Y-y_t) ln|Y-y_t| R1
//   sep_y = -2 sum_{Y != y_t} ln|Y-y_t| [R0 + x_t R1 - (Y-y_t) R2] + 2 sum_{X != x_t} (X-x_t) ln|X-x_t| T1
__global__ void finalise_lin_kernel(const double2 *__restrict__ tgt, const int32_t *__restrict__ itx,
                                    const int32_t *__restrict__ ity, const int32_t *__restrict__ colX,
                                    const int32_t *__restrict__ rowY, const double *__restrict__ TBx3,
                                    const double *__restrict__ TBy3, int nX, int nY,
                                    const double *__restrict__ part, int n_split, int64_t first, int64_t count,
                                    double G, double *__restrict__ Fx, double *__restrict__ Fy,
                                    unsigned int *__restrict__ queue, const double *__restrict__ lnint,
                                    int lnint_n) {
    const int64_t lt = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (lt < kQueues) queue[lt] = 0u;                 // every work queue (lattice mode uses one per pair class)
    if (lt >= count) return;
    const int64_t t = first + lt;
    const double2 p = tgt[t];
    const int kx = int(p.x), ky = int(p.y);
    double mx = 0.0, my = 0.0;
    for (int s = 0; s < n_split; ++s) {
        mx += part[(int64_t(s) * 2 + 0) * count + lt];
        my += part[(int64_t(s) * 2 + 1) * count + lt];
    }
    double sx = 0.0, sy = 0.0;
    const double *bx = TBx3 + int64_t(ity[t]) * nX * 3;
    for (int c = 0; c < nX; ++c) {
        const int d = colX[c] - kx;
        if (d != 0) {
            const double ln = ln_lattice(d, lnint, lnint_n), dd = double(d);
            sx = fma(-2.0 * ln, bx[3 * c] + p.y * bx[3 * c + 1] - dd * bx[3 * c + 2], sx);
            sy = fma(2.0 * dd * ln, bx[3 * c + 1], sy);
        }
    }
    const double *by = TBy3 + int64_t(itx[t]) * nY * 3;
    for (int r = 0; r < nY; ++r) {
        const int d = rowY[r] - ky;
        if (d != 0) {
            const double ln = ln_lattice(d, lnint, lnint_n), dd = double(d);
            sy = fma(-2.0 * ln, by[3 * r] + p.x * by[3 * r + 1] - dd * by[3 * r + 2], sy);
            sx = fma(2.0 * dd * ln, by[3 * r + 1], sx);
        }
    }
    Fx[lt] = G * (mx + sx);
    Fy[lt] = G * (my + sy);
}

void launch_finalise_lin(const DevLayout &d, const LinArrays &l, const ForcePlan &p, double *Fx, double *Fy,
                         cudaStream_t s) {
    if (p.count == 0) return;
    finalise_lin_kernel<<<unsigned((p.count + 127) / 128), 128, 0, s>>>(d.tgt, d.itx, d.ity, d.colX, d.rowY, l.TBx3,
                                                                       l.TBy3, d.nX, d.nY, d.part, p.n_split, p.first,
                                                                       p.count, d.G, Fx, Fy, d.queue, d.lnint, d.lnint_n);
}

}  // namespace sg
