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
    const double q = fma(u, u, v * v);
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
    static constexpr bool WG = F == 4;                                    // weights straight from global / L1: the table
                                                                          // leaves no room for weight buffers at 2 CTAs per SM
    static constexpr size_t smem = size_t(DB ? 2 : 1) * TBUF * 16 + (WG ? 0 : size_t(kOffWarps) * kBlkW * 8);
};

}  // namespace sg
