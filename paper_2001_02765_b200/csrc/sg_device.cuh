// sg_device.cuh -- internal device helpers shared by sg_kernels.cu and sg_kernels_lin.cu:
// PTX wrappers (MUFU seeds, mbarrier, TMA bulk copy), the log-table binning and the table-driven logarithm.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "sg_kernels.cuh"

namespace sg {

// ------------------------------------------------------------------------------------------------
// PTX helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double rsqrt_approx(double x) {      // MUFU.RSQ64H
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}
__device__ __forceinline__ double rcp_approx(double x) {        // MUFU.RCP64H (uses the high word only)
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
// plain arrival (release.cta): a consumer hands a shared-memory stage back to its producer ("empty" barrier)
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void tma_bulk_g2s(void *smem_dst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ------------------------------------------------------------------------------------------------
// log table: bins are the top (11 exponent + kLogK mantissa) bits of the FP64 high word.
//   idx(a) = hi(a) >> (20 - kLogK);   centre of the bin: hi_c = (idx << (20-kLogK)) | (1 << (19-kLogK))
//   c = rcp.approx(hi_c : 0)  (a pure function of idx),   lntab[idx - idx0] = -ln(c)
// so that ln(a) = lntab + log1p(f), f = a*c - 1, |f| <= 2^-(kLogK+1) + rcp error.
// ------------------------------------------------------------------------------------------------
constexpr int kLogShift = 20 - kLogK;
constexpr uint32_t kLogHalfBin = 1u << (19 - kLogK);
constexpr uint32_t kLogKeep = ~((1u << kLogShift) - 1u);

constexpr uint32_t kLogKeepMask = kLogKeep;

// tabb = (const char*)stab - tab_idx0*8 - 4:  hc = idx << 11 | 0x400  =>  hc >> 8 = idx*8 + 4
__device__ __forceinline__ double fast_ln(double a, const char *tabb, uint32_t keep) {
    const uint32_t hi = uint32_t(__double2hiint(a));
    uint32_t hc;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(hc) : "r"(hi), "r"(keep), "r"(kLogHalfBin));   // (hi & keep) | half
    const double tv = *reinterpret_cast<const double *>(tabb + (hc >> 8));
    const double c = rcp_approx(__hiloint2double(int(hc), 0));
    const double f = fma(a, c, -1.0);
    double s = fma(f, -0.25, 1.0 / 3.0);
    s = fma(f, s, -0.5);
    s = fma(f, s, 1.0);
    return fma(f, s, tv);
}

__device__ __forceinline__ double flip_sign_by(double a, double x) {   // a * s(x), s(+0) = +1
    return __hiloint2double(__double2hiint(a) ^ (__double2hiint(x) & int(0x80000000u)), __double2loint(a));
}

// ln|d| of an integer lattice distance; 0 for d == 0 (the coincident grid line is skipped)
__device__ __forceinline__ double ln_lattice(int d, const double *__restrict__ lnint, int lnint_n) {
    const int a = abs(d);
    if (lnint_n > 0) return lnint[a];
    return a ? log(double(a)) : 0.0;
}

}  // namespace sg
