// sg_patch_device.cuh -- internal device-side pieces shared by the two families of offset-table kernels
// (sg_kernels_patch.cu: tables built in the CTA; sg_kernels_lattice.cu: tables streamed from precomputed lattices):
// the compile-time description of the pair classes and the pair function evaluated through the L1-cached log table.
#pragma once
#include "sg_device.cuh"
#include "sg_kernels_patch.cuh"

namespace sg {

constexpr int kOffWarps = 8, kBlkR = 8, kBlkWRow = 32, kBlkW = 17 * kBlkWRow;

__device__ __forceinline__ double fast_ln_g(double a, const double *__restrict__ lntab_g, int tab_idx0, uint32_t keep) {
    const uint32_t hi = uint32_t(__double2hiint(a));
    const uint32_t hc = (hi & keep) | kLogHalfBin;
    const double tv = __ldg(lntab_g + (int(hc >> kLogShift) - tab_idx0));
    const double c = rcp_approx(__hiloint2double(int(hc), 0));
    const double f = fma(a, c, -1.0);
    double s = fma(f, -0.25, 1.0 / 3.0);
    s = fma(f, s, -0.5);
    s = fma(f, s, 1.0);
    return fma(f, s, tv);
}

__device__ __forceinline__ double2 pair_terms_g(double u, double v, const double *__restrict__ lntab_g, int tab_idx0,
                                                uint32_t keep) {
    // q >= 1 for every real pair (a target never sits on a vertex).  The clamp only matters for the holes of a padded
    // layout (regrouped small patches), whose discarded targets may coincide with a vertex: it keeps r finite and the
    // log-table index in range
    const double q = fmax(fma(u, u, v * v), 0.5);
    const double y0 = rsqrt_approx(q);
    const double t = q * y0;
    const double e = fma(-t, y0, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double r = fma(t, p * e, t);
    return make_double2(flip_sign_by(fast_ln_g(fabs(v) + r, lntab_g, tab_idx0, keep), v),
                        flip_sign_by(fast_ln_g(fabs(u) + r, lntab_g, tab_idx0, keep), u));
}

// compile-time description of pair class V (kOffSame, kOffCoarserSrc, kOffFinerSrc, kOffCoarserSrc4, kOffFinerSrc4)
template <int V>
struct OffCls {
    static constexpr int P = 16;
    static constexpr bool coarser = V == kOffCoarserSrc || V == kOffCoarserSrc4, finer = V == kOffFinerSrc || V == kOffFinerSrc4;
    static constexpr int F = V == kOffSame ? 1 : (V == kOffCoarserSrc || V == kOffFinerSrc) ? 2 : 4;   // pitch ratio
    static constexpr int RA = finer ? F : 1, RB = coarser ? F : 1;        // target / source pitch in units of g
    static constexpr int M = P * RB + (P - 1) * RA + 1, MMIN = (P - 1) * RA;      // table side 32, 48, 47, 80, 77
    static constexpr int RPC = (M + RA - 1) / RA;                         // stored rows per row class (finer source)
    static constexpr int ROWS = RA * RPC, TROW = (M | 1) == M ? M + 2 : M + 1;    // odd pitch >= M + 1
    static constexpr int TBUF = ROWS * TROW;
    static constexpr bool DB = F < 4;                                     // double-buffered tables (two CTAs per SM)
    static constexpr int LDIST = coarser ? -(F == 2 ? 1 : 2) : finer ? (F == 2 ? 1 : 2) : 0;   // source level - target level
    // weights are read straight from global memory (warp-uniform addresses: an L1 broadcast), shared memory holds tables only
    static constexpr size_t smem = size_t(DB ? 2 : 1) * TBUF * 16;
    // Order in which the source rows of a patch are correlated: natural, except for the source two levels finer, whose
    // table rows are stored by residue class of j mod 4 -- there class by class (j = c, c + 4, ...), so that one class
    // block of the table is needed at a time (lattice_corr_kernel streams it in four sub-blocks).
    static constexpr int JPASSES = V == kOffFinerSrc4 ? 4 : 1;
};

// Correlation of one target patch (this warp: lane = l + 16 h, l = target row, 8 targets per thread) with the vertices
// of one source patch through the offset table T of the patch pair; shared by patch_offset_kernel (tables built in the
// CTA) and lattice_corr_kernel (tables streamed from the function lattices), so that both give bit-identical sums.
// With vertex (i, j) of B and target (k, l) of A the table entry is T[j rb - l ra + 15 ra][i rb - k ra + 15 ra]:
//   same level (ra = rb = 1): thread owns columns k = 8 h + r; entry column t + 8 - 8 h serves vertices i = t + r - 7;
//   coarser source (ra = 1, rb = F): NCLS = F / 2 column classes mod F of MT = 8 / NCLS targets, k = F m + NCLS h + cc;
//          entry column F t + F (1 - MT) + 15 - NCLS h - cc serves i = t + m - (MT - 1);
//   finer source (ra = F, rb = 1): k = 8 h + r; entry column t + 8 F (1 - h) serves i = t + F r - 7 F; table rows are
//          stored by row class (row j - F l + 15 F has the residue of j mod F: a half-warp reads consecutive stored rows).
// One loaded entry serves up to 8 targets (16 DFMA per LDS.128); the weights of a source row sit in registers (fully
// unrolled, compile-time indices, ragged ends removed at compile time).  src: the patch's weights, [17] rows of 9
// double2 (vertices 2c, 2c+1; vertex 17 is zero padding).  flags (warp-uniform): bit 0 = vertex row 16 of the source
// patch carries owned vertices, bit 1 = vertex column 16 does (in a row below 16): on a uniform level a patch owns only
// its 16 x 16 lower-left vertices (sg_api.cu, owner rule), so row 16 and column 16 are skipped for almost every patch --
// 256 instead of 289 vertices.  Every per-patch sum stays in one accumulator chain.
// Source rows j0, j0 + jstep, ... <= j1 only (the whole patch: 0, 16, 1): lattice_corr_kernel streams the large
// tables of the classes two levels apart in sub-blocks of rows and correlates the source rows of one sub-block at a time.
template <int V>
__device__ __forceinline__ void correlate_patch(const double2 *__restrict__ T, const double2 *__restrict__ src, int flags,
                                                int l, int h, double (&ax)[kBlkR], double (&ay)[kBlkR], int j0, int j1,
                                                int jstep) {
    using C = OffCls<V>;
    constexpr int P = 16, F = C::F, TROW = C::TROW;
    constexpr int NCLS = C::coarser ? F / 2 : 1, MT = kBlkR / NCLS;
    constexpr int NT = C::finer ? P + F * (kBlkR - 1) : P + MT - 1;       // table steps that reach vertices 0 .. P-1
    if (C::coarser) T += (15 - l) * TROW + F * (1 - MT) + 15 - NCLS * h;  // column F t + this - cc
    else T += (15 - l) * TROW + 8 * F * (1 - h);                          // column t + this (F = 1: 8 - 8 h)
    const int jmax = min(j1, (flags & 1) ? P : P - 1);
#pragma unroll 1
    for (int j = j0; j <= jmax; j += jstep) {
        const double2 *trow = C::coarser ? T + F * j * TROW                                   // row F j - l + 15
                                         : T + (j / C::RA + (j % C::RA) * C::RPC) * TROW;      // row j - RA l + MMIN
        double wv[P];                                                     // compile-time indices only: registers
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            if ((t & 1) == 0 && t < P) {                                  // vertices t, t+1
                const double2 w2 = __ldg(src + j * 9 + t / 2);            // warp-uniform address: L1 broadcast
                wv[t] = w2.x;
                wv[t + 1] = w2.y;
            }
#pragma unroll
            for (int cc = 0; cc < NCLS; ++cc) {
                const double2 Tv = trow[C::coarser ? F * t - cc : t];
#pragma unroll
                for (int m = 0; m < MT; ++m) {
                    const int i = C::finer ? t + F * m - F * (kBlkR - 1) : t + m - (MT - 1);    // compile-time
                    if (i >= 0 && i < P) {
                        ax[cc * MT + m] = fma(wv[i], Tv.x, ax[cc * MT + m]);
                        ay[cc * MT + m] = fma(wv[i], Tv.y, ay[cc * MT + m]);
                    }
                }
            }
        }
        if ((flags & 2) || j == P) {                                      // vertex column 16 of this row
            const double w16 = __ldg(src + j * 9 + 8).x;
#pragma unroll
            for (int cc = 0; cc < NCLS; ++cc)
#pragma unroll
                for (int m = 0; m < MT; ++m) {
                    const int t = C::finer ? P - F * m + F * (kBlkR - 1) : P - m + (MT - 1);   // the step with i(t, m) = 16
                    const double2 Tv = trow[C::coarser ? F * t - cc : t];
                    ax[cc * MT + m] = fma(w16, Tv.x, ax[cc * MT + m]);
                    ay[cc * MT + m] = fma(w16, Tv.y, ay[cc * MT + m]);
                }
        }
    }
}

// the whole source patch, in the row order of the class (both kernel families: bit-identical sums)
template <int V>
__device__ __forceinline__ void correlate_patch_all(const double2 *__restrict__ T, const double2 *__restrict__ src,
                                                    int flags, int l, int h, double (&ax)[kBlkR], double (&ay)[kBlkR]) {
#pragma unroll 1
    for (int c = 0; c < OffCls<V>::JPASSES; ++c) correlate_patch<V>(T, src, flags, l, h, ax, ay, c, 16, OffCls<V>::JPASSES);
}


}  // namespace sg
