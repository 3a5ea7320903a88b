// sg_kernels.cu -- CUDA kernels (sm_100a) of the direct thin-disk self-gravity sum.
//
// Mathematics (derivation and readings in DESIGN.md):
//   F^x_t = G sum_c sigma_c [[ P ]]_c ,  P(u,v) = -ln(v + r),  u = xbar-x_t, v = ybar-y_t, r = sqrt(u^2+v^2)
// regrouped by vertex, sum_c sigma_c [[P]]_c = sum_v w_v P(u_v, v_v), and with P written in the
// cancellation-free form
//   P(u,v) = -s(v) ln(|v| + r) - [v < 0] * 2 ln|u|            s(v) = +1 for v >= 0, -1 for v < 0
// whose second, separable part is dropped when u == 0 (the paper's modified primitive, PAPER.md:96-100,
// up to a constant that cancels because the weights on each side of the target along a grid line sum
// to zero).  Hence, in lattice units (every u, v an exact integer held in FP64):
//   F^x_t = -G [ M^x_t + 2 S^x_t ],   M^x_t = sum_v w_v s(v_v) ln(|v_v| + r_v)          (interaction kernel)
//                                     S^x_t = sum_{X != x_t} ln|X - x_t| * Wbelow(X, y_t) (finalise kernel)
// and the same with x and y exchanged for F^y.  The additive constant ln(unit) cancels exactly
// (sum of all weights on a grid line is zero), so no scaling enters the hot loop.
#include "sg_kernels.cuh"
#include "sg_device.cuh"

#include <cstdio>

namespace sg {

__global__ void build_logtab_kernel(double *lntab, int idx0, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t hc = (uint32_t(idx0 + i) << kLogShift) | kLogHalfBin;
    const double c = rcp_approx(__hiloint2double(int(hc), 0));
    lntab[i] = -log(c);
}

__global__ void build_lnint_kernel(double *lnint, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) lnint[i] = i ? log(double(i)) : 0.0;
}

void launch_build_lnint(const DevLayout &d, cudaStream_t s) {
    if (d.lnint_n > 0) build_lnint_kernel<<<(d.lnint_n + 255) / 256, 256, 0, s>>>(d.lnint, d.lnint_n);
}

void launch_build_logtab(const DevLayout &d, cudaStream_t s) {
    build_logtab_kernel<<<(d.tab_entries + 255) / 256, 256, 0, s>>>(d.lntab, d.tab_idx0, d.tab_entries);
}

// ------------------------------------------------------------------------------------------------
// S2a: vertex weights.  w_v = sum of +-sigma over the <= 4 cells that have v as a corner, in the fixed
// order of the adjacency list (deterministic).  One thread per tile slot: writes the w half of the
// slot's {y, w} pair (0 for padding slots) and the flat array used by the line tables.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double *slot_yw(double *vtile, int64_t slot) {
    return vtile + (slot / kTileSlots) * kTileDoubles + kChunksPerTile + 2 * (slot % kTileSlots);
}

__global__ void vertex_weights_kernel(const int32_t *__restrict__ adj, const int32_t *__restrict__ slot_vertex,
                                      const double *__restrict__ sigma, double *__restrict__ w,
                                      double *__restrict__ vtile, int64_t n_slots) {
    const int64_t s = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (s >= n_slots) return;
    const int v = slot_vertex[s];
    double acc = 0.0;
    if (v >= 0) {
        const int4 a = reinterpret_cast<const int4 *>(adj)[v];
        const int e[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (e[k] >= 0) {
                const double sg = sigma[e[k] >> 2];
                const int corner = e[k] & 3;                    // 0 NE (+), 1 NW (-), 2 SE (-), 3 SW (+)
                acc += (corner == 1 || corner == 2) ? -sg : sg;
            }
        w[v] = acc;
    }
    slot_yw(vtile, s)[1] = acc;
}

void launch_vertex_weights(const DevLayout &d, const double *sigma, cudaStream_t s) {
    vertex_weights_kernel<<<unsigned((d.n_slots + 255) / 256), 256, 0, s>>>(d.adj, d.slot_vertex, sigma, d.w, d.vtile,
                                                                           d.n_slots);
}

// Static part of the tiles (lattice coordinates as FP64): xc per chunk, y per slot.  A padding slot takes
// the y of its chunk's first vertex (of vertex 0 in an all-padding chunk, whose x is chunk 0's): a real
// vertex position, so r > 0 against every target, and its w stays 0.
__global__ void fill_static_tiles_kernel(const int32_t *__restrict__ vky, const int32_t *__restrict__ chunk_x,
                                         const int32_t *__restrict__ slot_vertex, double *__restrict__ vtile,
                                         int64_t n_slots) {
    const int64_t s = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (s >= n_slots) return;
    int v = slot_vertex[s];
    if (v < 0) v = slot_vertex[(s / kChunk) * kChunk];
    if (v < 0) v = 0;
    double *yw = slot_yw(vtile, s);
    yw[0] = double(vky[v]);
    yw[1] = 0.0;
    if (s % kChunk == 0) {
        const int64_t c = s / kChunk;
        vtile[(c / kChunksPerTile) * kTileDoubles + (c % kChunksPerTile)] = double(chunk_x[c]);
    }
}

void launch_fill_static_tiles(const DevLayout &d, cudaStream_t s) {
    fill_static_tiles_kernel<<<unsigned((d.n_slots + 255) / 256), 256, 0, s>>>(d.vky, d.chunk_x, d.slot_vertex, d.vtile,
                                                                              d.n_slots);
}

// ------------------------------------------------------------------------------------------------
// S2b: cumulative line weights.
//   TBx[iy][c] = sum of w over the vertices of column c with y_v <  tY[iy]   (strictly below)
//   TBy[ix][r] = sum of w over the vertices of row    r with x_v <  tX[ix]   (strictly left)
// Two steps per direction: a running sum along every line (one thread per line, vertices in line order, so the
// rounding is that of a plain left-to-right sum), then one thread per (target coordinate, line) finds by bisection
// how many vertices of the line lie strictly before the coordinate and picks the running sum there.
// ------------------------------------------------------------------------------------------------
__global__ void line_prefix_kernel(const int32_t *__restrict__ start, const int32_t *__restrict__ perm,
                                   const double *__restrict__ w, int n_lines, double *__restrict__ wcum) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_lines) return;
    const int e = start[c + 1];
    double acc = 0.0;
    for (int p = start[c]; p < e; ++p) {
        acc += w[perm ? perm[p] : p];
        wcum[p] = acc;
    }
}

__global__ void line_lookup_kernel(const int32_t *__restrict__ start, const int32_t *__restrict__ perm,
                                   const int32_t *__restrict__ vcoord, const double *__restrict__ wcum,
                                   const int32_t *__restrict__ tcoord, int n_lines, int n_t, double *__restrict__ TB) {
    const int64_t idx = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (idx >= int64_t(n_lines) * n_t) return;
    const int c = int(idx % n_lines), i = int(idx / n_lines);
    const int t = tcoord[i], s0 = start[c];
    int lo = s0, hi = start[c + 1];                       // first position in [lo, hi) whose coordinate is >= t
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (vcoord[perm ? perm[mid] : mid] < t) lo = mid + 1; else hi = mid;
    }
    TB[idx] = lo > s0 ? wcum[lo - 1] : 0.0;
}

void launch_line_tables(const DevLayout &d, cudaStream_t s) {
    line_prefix_kernel<<<(d.nX + 63) / 64, 64, 0, s>>>(d.colstart, nullptr, d.w, d.nX, d.wcum);
    line_prefix_kernel<<<(d.nY + 63) / 64, 64, 0, s>>>(d.rowstart, d.rowperm, d.w, d.nY, d.wcum + d.Nv);
    const int64_t nx = int64_t(d.nX) * d.ntY, ny = int64_t(d.nY) * d.ntX;
    if (nx > 0)
        line_lookup_kernel<<<unsigned((nx + 255) / 256), 256, 0, s>>>(d.colstart, nullptr, d.vky, d.wcum, d.tY, d.nX,
                                                                     d.ntY, d.TBx);
    if (ny > 0)
        line_lookup_kernel<<<unsigned((ny + 255) / 256), 256, 0, s>>>(d.rowstart, d.rowperm, d.vkx, d.wcum + d.Nv, d.tX,
                                                                     d.nY, d.ntX, d.TBy);
}

// ------------------------------------------------------------------------------------------------
// S3: the all-pairs interaction kernel.
//
// Work item = (target block of kThreads*T targets, source split of tiles_per_split vertex tiles).
// A persistent grid (2 CTAs per SM) pulls items from an atomic counter; every item writes its own slot of
// `part`, so the result does not depend on which CTA ran it.  Per item each thread keeps T targets and
// their accumulators in registers; vertex tiles (4,224 bytes: 16 chunk abscissae + 256 {y, w} slots)
// arrive in shared memory through TMA bulk copies (cp.async.bulk + mbarrier complete_tx), kStages deep;
// every thread reads every slot as a warp-wide broadcast.
//
// A chunk is 16 vertices of one grid column, so u = xc - x_t, u^2 and the sign s(u) are shared by its
// pairs: per (target, chunk) 2 DADD + 1 DMUL, and per (target, vertex) pair 21 FP64-pipe instructions,
// no branch, no division, no libdevice call:
//   v, q = v^2 + u^2                                    2   (exact: integers < 2^53)
//   r = sqrt(q): MUFU.RSQ64H seed + one cubic step      5
//   a1 = |v|+r, a2 = |u|+r                              2
//   ln a_i = lntab[bin of a_i] + log1p(a_i*c - 1)       2 x 5   (c = MUFU.RCP64H of the bin centre)
//   ax += w * s(v) ln a1 ;  cy += w * ln a2             2   (s(v) by integer XOR; s(u) once per chunk)
// On sm_100 an FP64 instruction takes two issue cycles of a sub-partition and every other instruction
// one (measured), so the non-FP64 instructions are kept few as well: the bin-centre
// high word hc = (hi & keep) | half is both the MUFU.RCP64H operand and, shifted by 8, the table offset.
// ------------------------------------------------------------------------------------------------
template <int T>
__global__ void __launch_bounds__(kThreads, 2)
interaction_kernel(const double2 *__restrict__ tgt, const double *__restrict__ vtile,
                   const double *__restrict__ lntab_g, int tab_idx0, int tab_entries, int n_tiles,
                   int tiles_per_split, int n_split, int n_tblocks, int64_t first, int64_t count,
                   double *__restrict__ part, unsigned int *__restrict__ queue, uint32_t keep) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *stile = reinterpret_cast<double *>(smem_raw);                         // kStages tiles
    uint64_t *full = reinterpret_cast<uint64_t *>(stile + kStages * kTileDoubles); // kStages mbarriers
    double *stab = reinterpret_cast<double *>(full + 8);                          // log table
    __shared__ int s_item;
    const int tid = threadIdx.x;

    for (int i = tid; i < tab_entries; i += kThreads) stab[i] = lntab_g[i];
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const char *tabb = reinterpret_cast<const char *>(stab) - int64_t(tab_idx0) * 8 - 4;

    uint32_t it = 0;   // tiles consumed by this CTA so far (stage = it % kStages, parity from it / kStages)
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
                mbar_expect_tx(&full[st], kTileDoubles * 8);
                tma_bulk_g2s(stile + st * kTileDoubles, vtile + int64_t(tile0 + i) * kTileDoubles,
                             kTileDoubles * 8, &full[st]);
            }
        }
        for (int i = 0; i < ntile; ++i, ++it) {
            const uint32_t st = it % kStages;
            mbar_wait(&full[st], (it / kStages) & 1u);
            const double *sx = stile + st * kTileDoubles;
            const double2 *syw = reinterpret_cast<const double2 *>(sx + kChunksPerTile);
#pragma unroll 1
            for (int c = 0; c < kChunksPerTile; ++c) {
                const double xc = sx[c];
                double u[T], uu[T], cy[T];
#pragma unroll
                for (int k = 0; k < T; ++k) { u[k] = xc - xt[k]; uu[k] = u[k] * u[k]; cy[k] = 0.0; }
#pragma unroll 4
                for (int j = 0; j < kChunk; ++j) {
                    const double2 yw = syw[c * kChunk + j];
#pragma unroll
                    for (int k = 0; k < T; ++k) {
                        const double v = yw.x - yt[k];
                        const double q = fma(v, v, uu[k]);
                        const double y0 = rsqrt_approx(q);
                        const double t = q * y0;                 // ~sqrt(q)
                        const double e = fma(-t, y0, 1.0);       // 1 - q*y0^2
                        const double p = fma(0.375, e, 0.5);
                        const double r = fma(t, p * e, t);       // t * (1 + e/2 + 3e^2/8)
                        const double l1 = fast_ln(fabs(v) + r, tabb, keep);
                        const double l2 = fast_ln(fabs(u[k]) + r, tabb, keep);
                        ax[k] = fma(yw.y, flip_sign_by(l1, v), ax[k]);
                        cy[k] = fma(yw.y, l2, cy[k]);
                    }
                }
#pragma unroll
                for (int k = 0; k < T; ++k) ay[k] += flip_sign_by(cy[k], u[k]);
            }
            __syncthreads();   // every thread is done with stage st
            if (tid == 0 && i + kStages < ntile) {
                mbar_expect_tx(&full[st], kTileDoubles * 8);
                tma_bulk_g2s(stile + st * kTileDoubles, vtile + int64_t(tile0 + i + kStages) * kTileDoubles,
                             kTileDoubles * 8, &full[st]);
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

size_t interaction_smem_bytes(int tab_entries) {
    return size_t(kStages) * kTileDoubles * 8 + 64 + size_t(tab_entries) * 8;
}

cudaError_t configure_kernels(int tab_entries) {
    const size_t bytes = interaction_smem_bytes(tab_entries);
    cudaError_t e = opt_in_max_smem(interaction_kernel<4>, bytes);
    if (e != cudaSuccess) return e;
    return opt_in_max_smem(interaction_kernel<1>, bytes);
}

void launch_interaction(const DevLayout &d, const ForcePlan &p, cudaStream_t s) {
    if (p.count == 0) return;
    if (p.T == 4)
        interaction_kernel<4><<<p.grid, kThreads, p.smem, s>>>(d.tgt, d.vtile, d.lntab, d.tab_idx0, d.tab_entries,
                                                              d.n_tiles, p.tiles_per_split, p.n_split, p.n_tblocks,
                                                              p.first, p.count, d.part, d.queue, kLogKeepMask);
    else
        interaction_kernel<1><<<p.grid, kThreads, p.smem, s>>>(d.tgt, d.vtile, d.lntab, d.tab_idx0, d.tab_entries,
                                                              d.n_tiles, p.tiles_per_split, p.n_split, p.n_tblocks,
                                                              p.first, p.count, d.part, d.queue, kLogKeepMask);
}

// ------------------------------------------------------------------------------------------------
// S4 + S5: coincidence-safe separable part, split-source reduction, scaling by G.
//   S^x_t = sum over vertex columns X != x_t (exact integer test: this is where the paper's modified
//           primitive for xbar == x, takes effect) of ln|X - x_t| * TBx[iy_t][X]
//   F^x_t = -G ( sum_splits M^x + 2 S^x ),  same for y with rows.
// One thread per target; the partial sums are added in split order (deterministic, no atomics).
// ------------------------------------------------------------------------------------------------
__global__ void finalise_kernel(const double2 *__restrict__ tgt, const int32_t *__restrict__ itx,
                                const int32_t *__restrict__ ity, const int32_t *__restrict__ colX,
                                const int32_t *__restrict__ rowY, const double *__restrict__ TBx,
                                const double *__restrict__ TBy, int nX, int nY,
                                const double *__restrict__ part, int n_split, int64_t first, int64_t count,
                                double G, double *__restrict__ Fx, double *__restrict__ Fy,
                                unsigned int *__restrict__ queue, const double *__restrict__ lnint, int lnint_n) {
    const int64_t lt = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (lt < kQueues) queue[lt] = 0u;                 // drained by this call's interaction kernels; ready for the next
    if (lt >= count) return;
    const int64_t t = first + lt;
    const double2 p = tgt[t];
    const int kx = int(p.x), ky = int(p.y);
    double mx = 0.0, my = 0.0;
    for (int s = 0; s < n_split; ++s) {
        mx += part[(int64_t(s) * 2 + 0) * count + lt];
        my += part[(int64_t(s) * 2 + 1) * count + lt];
    }
    const double *bx = TBx + int64_t(ity[t]) * nX;
    double sx = 0.0;
    for (int c = 0; c < nX; ++c) {
        const int d = colX[c] - kx;
        sx = fma(ln_lattice(d, lnint, lnint_n), bx[c], sx);
    }
    const double *by = TBy + int64_t(itx[t]) * nY;
    double sy = 0.0;
    for (int r = 0; r < nY; ++r) {
        const int d = rowY[r] - ky;
        sy = fma(ln_lattice(d, lnint, lnint_n), by[r], sy);
    }
    Fx[lt] = -G * (mx + 2.0 * sx);
    Fy[lt] = -G * (my + 2.0 * sy);
}

void launch_finalise(const DevLayout &d, const ForcePlan &p, double *Fx, double *Fy, cudaStream_t s) {
    if (p.count == 0) return;
    finalise_kernel<<<unsigned((p.count + 127) / 128), 128, 0, s>>>(d.tgt, d.itx, d.ity, d.colX, d.rowY, d.TBx, d.TBy,
                                                                   d.nX, d.nY, d.part, p.n_split, p.first, p.count,
                                                                   d.G, Fx, Fy, d.queue, d.lnint, d.lnint_n);
}

// ------------------------------------------------------------------------------------------------
// Regrouped layouts (small patches packed into padded 16 x 16 blocks for lattice mode, sg_api.cu): cell data of the
// caller's order <-> the block order of the inner context.  inv[k] = caller cell of inner cell k, or -1 (hole).
// ------------------------------------------------------------------------------------------------
__global__ void scatter_cells_kernel(const double *__restrict__ a, const double *__restrict__ b,
                                     const double *__restrict__ c, const int32_t *__restrict__ inv,
                                     double *__restrict__ oa, double *__restrict__ ob, double *__restrict__ oc,
                                     int64_t n_inner) {
    const int64_t k = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (k >= n_inner) return;
    const int32_t s = inv[k];
    oa[k] = s >= 0 ? a[s] : 0.0;
    if (b) { ob[k] = s >= 0 ? b[s] : 0.0; oc[k] = s >= 0 ? c[s] : 0.0; }
}

__global__ void gather_cells_kernel(const double *__restrict__ fx, const double *__restrict__ fy,
                                    const int32_t *__restrict__ map, int64_t base, int64_t first, int64_t count,
                                    double *__restrict__ ox, double *__restrict__ oy) {
    const int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const int64_t k = int64_t(map[first + i]) - base;   // fx, fy hold the inner target range, which starts at `base`
    ox[i] = fx[k];
    oy[i] = fy[k];
}

void launch_scatter_cells(const double *a, const double *b, const double *c, const int32_t *inv, double *oa, double *ob,
                          double *oc, int64_t n_inner, cudaStream_t s) {
    scatter_cells_kernel<<<unsigned((n_inner + 255) / 256), 256, 0, s>>>(a, b, c, inv, oa, ob, oc, n_inner);
}

void launch_gather_cells(const double *fx, const double *fy, const int32_t *map, int64_t base, int64_t first,
                         int64_t count, double *ox, double *oy, cudaStream_t s) {
    if (count > 0) gather_cells_kernel<<<unsigned((count + 255) / 256), 256, 0, s>>>(fx, fy, map, base, first, count, ox, oy);
}

// ------------------------------------------------------------------------------------------------
// FP64 peak: 8 independent DFMA chains per thread, 4 CTAs of 256 threads per SM.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_kernel(double *out, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    const double sum = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (sum == 123.456) out[0] = sum;   // never true; keeps the chains alive
}

cudaError_t measure_dfma(double *tflops, double *warp_instr_per_s) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    double *out = nullptr;
    e = cudaMalloc(&out, 8);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = sms * 4, iters = 4096;
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        dfma_kernel<<<grid, 256>>>(out, iters, 0.999999, 1e-9);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    if (e != cudaSuccess) return e;
    const double fmas = double(grid) * 256.0 * double(iters) * 64.0;   // thread-level DFMAs
    if (tflops) *tflops = 2.0 * fmas / (best * 1e-3) / 1e12;
    if (warp_instr_per_s) *warp_instr_per_s = fmas / 32.0 / (best * 1e-3);
    return cudaSuccess;
}


// ------------------------------------------------------------------------------------------------
// FP64 tensor-core probe ("FP64 tensor cores do not help").  mma.sync.m8n8k4.f64 = 512 flop per warp
// instruction, four independent accumulator pairs per thread; MIX adds four independent DFMA chains per thread in
// the same loop (one DFMA per DMMA), to see whether the two add up or share one pipe.
// ------------------------------------------------------------------------------------------------
template <bool MIX>
__global__ void __launch_bounds__(256) dmma_kernel(double *out, int iters, double a, double b) {
    double c[4][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3;
    const double fa = a + 1e-9 * threadIdx.x, fb = b;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                             : "+d"(c[q][0]), "+d"(c[q][1]) : "d"(fa), "d"(fb));
            if (MIX) { x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b); }
        }
    }
    const double sum = c[0][0] + c[0][1] + c[1][0] + c[1][1] + c[2][0] + c[2][1] + c[3][0] + c[3][1] + x0 + x1 + x2 + x3;
    if (sum == 123.456) out[0] = sum;   // never true; keeps the chains alive
}

cudaError_t measure_dmma(double *dmma_tflops, double *mixed_tflops) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    double *out = nullptr;
    e = cudaMalloc(&out, 8);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = sms * 4, iters = 2048;
    double res[2] = {0.0, 0.0};
    for (int mix = 0; mix < 2 && e == cudaSuccess; ++mix) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {
            cudaEventRecord(e0);
            if (mix) dmma_kernel<true><<<grid, 256>>>(out, iters, 0.999999, 1e-9);
            else dmma_kernel<false><<<grid, 256>>>(out, iters, 0.999999, 1e-9);
            cudaEventRecord(e1);
            e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) break;
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        const double warps = double(grid) * 8.0, steps = double(iters) * 4.0;
        const double flop = warps * steps * (4.0 * 512.0 + (mix ? 4.0 * 32.0 * 2.0 : 0.0));   // per warp and step
        res[mix] = flop / (best * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    if (e != cudaSuccess) return e;
    if (dmma_tflops) *dmma_tflops = res[0];
    if (mixed_tflops) *mixed_tflops = res[1];
    return cudaSuccess;
}

}  // namespace sg
