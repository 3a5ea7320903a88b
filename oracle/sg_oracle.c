/*
 * sg_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU evaluation of the force sum of arXiv 2001.02765
 * (Tseng, Shang & Yen), written from the paper.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or helper with the CUDA library under paper_2001_02765_b200/.
 *
 * What it computes (every symbol as in the paper):
 *   PAPER.md:57-69  (Eq. 4-5)  sigma = sum_i sigma_i chi_{D_i}, D_i = [x_l,x_r] x [y_d,y_u] disjoint leaves.
 *   PAPER.md:71-76  (Eq. 6)    sigma_i ~ sigma_i^0 + delta_i^x (x - x_i^c) + delta_i^y (y - y_i^c).
 *   PAPER.md:82-90             F^x ~ F^{x,0} + F^{x,x} + F^{x,y}, one kernel integral K per term and cell.
 *   PAPER.md:92-94             closed forms at z = 0 as mixed corner differences
 *                              [[f]] = f(x_r,y_u) - f(x_l,y_u) - f(x_r,y_d) + f(x_l,y_d):
 *        K^{x,0} = [[ -ln( v + r ) ]]                        u = xbar - x, v = ybar - y, r = sqrt(u^2+v^2)
 *        K^{x,x} = (x - x_c) K^{x,0} + [[ v ln(u + r) ]]
 *        K^{x,y} = (y - y_c) K^{x,0} - [[ r ]]
 *        K^{y,0}, K^{y,y}, K^{y,x}: the same with x and y exchanged.
 *   PAPER.md:96-100            when xbar == x the primitive of K^{x,0} is replaced by -sgn(v) ln|v|.
 *   PAPER.md:104,110           targets are the centres of the leaf zones.
 *
 * Readings of garbled / silent passages:
 *   R1 sign: F = + G sum sigma K (attractive; K^{x,0} is the integral of (xbar-x)/r^3).
 *   R2 integration limits printed |_{x^c}^{x^c}|_{y^d}^{y^a} are x_l..x_r, y_d..y_u.
 *   R3 the "(ybar-y)^2 + z^2" / "+ z^2" fragments inside K^{x,x}, K^{x,y} are extraction debris; the
 *      z = 0 forms above follow from direct integration and are pinned by quadrature in the tests.
 *   R4 -ln(v + r) is evaluated for v < 0 as ln(r - v) - 2 ln|u| (the same number, without the
 *      cancellation in v + r); the paper does not discuss conditioning.
 *   R5 K^{y,0} is modified on ybar == y by symmetry (the paper gives only the x case).
 *   R6 v ln(u + r) := 0 at v == 0 (its limit), u ln(v + r) := 0 at u == 0.
 *
 * Geometry is passed as integers on a lattice (unit = physical length of one lattice step) so
 * that "xbar == x" is an exact integer test, as the paper's sgn(|xbar - x|) requires.
 *
 * Floating type: REAL = long double (x87 80-bit) by default; -DSG_ORACLE_DOUBLE builds the same
 * source in double.  No blocking, no regrouping, no vertex sharing: cell by cell, four corners each.
 *
 * Pins (tests/test_oracle_pins.py): 2-D quadrature of the kernel integrands, far-field monopole,
 * antisymmetry, telescoping of constant sigma, refinement invariance, Table 1/2/3 values.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef SG_ORACLE_DOUBLE
typedef double REAL;
#define RLOG  log
#define RSQRT sqrt
#define RFABS fabs
#define SUFFIX(name) name##_f64
#else
typedef long double REAL;
#define RLOG  logl
#define RSQRT sqrtl
#define RFABS fabsl
#define SUFFIX(name) name##_f80
#endif

/* primitive of K^{x,0}: P(u,v) = -ln(v + r), with the paper's modification at u == 0 (ku is the
 * integer lattice difference so the test is exact) and reading R4 for v < 0. */
static REAL prim0(int64_t ku, int64_t kv, REAL unit)
{
    REAL u = (REAL)ku * unit, v = (REAL)kv * unit;
    if (ku == 0) {                       /* -(1 - sgn|u|) sgn(v) ln|v| */
        if (kv > 0) return -RLOG(v);
        if (kv < 0) return RLOG(-v);
        return 0;                        /* target on a vertex: excluded by the callers */
    }
    REAL r = RSQRT(u * u + v * v);
    if (kv >= 0) return -RLOG(v + r);
    return RLOG(r - v) - 2 * RLOG(RFABS(u));
}

/* primitive of the integral of u^2/r^3:  v ln(u + r)  (reading R3, R6; stable for u < 0) */
static REAL prim_vlog(int64_t ku, int64_t kv, REAL unit)
{
    if (kv == 0) return 0;
    REAL u = (REAL)ku * unit, v = (REAL)kv * unit;
    REAL r = RSQRT(u * u + v * v);
    if (ku >= 0) return v * RLOG(u + r);
    return v * (2 * RLOG(RFABS(v)) - RLOG(r - u));
}

static REAL prim_r(int64_t ku, int64_t kv, REAL unit)
{
    REAL u = (REAL)ku * unit, v = (REAL)kv * unit;
    return RSQRT(u * u + v * v);
}

#define CORNERS(f, a_l, a_r, b_d, b_u) \
    (f((a_r), (b_u), unit) - f((a_l), (b_u), unit) - f((a_r), (b_d), unit) + f((a_l), (b_d), unit))

/* The six z = 0 kernels of one cell seen from one target. Exposed for the pins. */
void SUFFIX(sg_oracle_cell_kernels)(int64_t kxl, int64_t kxr, int64_t kyd, int64_t kyu,
                                    int64_t ktx, int64_t kty, double unit_d, double *out6)
{
    REAL unit = unit_d;
    int64_t ul = kxl - ktx, ur = kxr - ktx, vd = kyd - kty, vu = kyu - kty;
    REAL xmxc = -(REAL)(ul + ur) * unit / 2;           /* x - x_c */
    REAL ymyc = -(REAL)(vd + vu) * unit / 2;           /* y - y_c */
    REAL Kx0 = CORNERS(prim0, ul, ur, vd, vu);
    /* y kernels: exchange the roles of x and y; the corner difference is symmetric in the exchange */
    REAL Ky0 = prim0(vu, ur, unit) - prim0(vu, ul, unit) - prim0(vd, ur, unit) + prim0(vd, ul, unit);
    REAL Ivl = CORNERS(prim_vlog, ul, ur, vd, vu);     /* [[ v ln(u+r) ]] */
    REAL Iul = prim_vlog(vu, ur, unit) - prim_vlog(vu, ul, unit) - prim_vlog(vd, ur, unit) + prim_vlog(vd, ul, unit);
    REAL Ir  = CORNERS(prim_r, ul, ur, vd, vu);        /* [[ r ]] */
    out6[0] = (double)Kx0;
    out6[1] = (double)(xmxc * Kx0 + Ivl);              /* K^{x,x} */
    out6[2] = (double)(ymyc * Kx0 - Ir);               /* K^{x,y} */
    out6[3] = (double)Ky0;
    out6[4] = (double)(xmxc * Ky0 - Ir);               /* K^{y,x} */
    out6[5] = (double)(ymyc * Ky0 + Iul);              /* K^{y,y} */
}

/*
 * F^x, F^y at n_t targets from n_c leaf cells (PAPER.md:86 with reading R1):
 *    Fx_t = G sum_c [ sigma_c K^{x,0} + dx_c K^{x,x} + dy_c K^{x,y} ],   likewise Fy.
 * dx, dy may be NULL (zeroth-order sum only: the hot path of BASELINE.json's north_star).
 * All cells are summed, including the one that contains the target (its K^{.,0} is 0 by symmetry).
 * Returns the number of threads used.
 */
int SUFFIX(sg_oracle_force)(int64_t n_c, const int64_t *kxl, const int64_t *kxr,
                            const int64_t *kyd, const int64_t *kyu,
                            const double *sigma, const double *dx, const double *dy,
                            int64_t n_t, const int64_t *ktx, const int64_t *kty,
                            double unit_d, double G, double *Fx, double *Fy, int n_threads)
{
    const REAL unit = unit_d;
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
    used = omp_get_max_threads();
#endif
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t t = 0; t < n_t; ++t) {
        REAL fx = 0, fy = 0;
        const int64_t tx = ktx[t], ty = kty[t];
        for (int64_t c = 0; c < n_c; ++c) {
            const int64_t ul = kxl[c] - tx, ur = kxr[c] - tx, vd = kyd[c] - ty, vu = kyu[c] - ty;
            REAL Kx0 = CORNERS(prim0, ul, ur, vd, vu);
            REAL Ky0 = prim0(vu, ur, unit) - prim0(vu, ul, unit) - prim0(vd, ur, unit) + prim0(vd, ul, unit);
            fx += (REAL)sigma[c] * Kx0;
            fy += (REAL)sigma[c] * Ky0;
            if (dx && dy) {
                REAL xmxc = -(REAL)(ul + ur) * unit / 2, ymyc = -(REAL)(vd + vu) * unit / 2;
                REAL Ivl = CORNERS(prim_vlog, ul, ur, vd, vu);
                REAL Iul = prim_vlog(vu, ur, unit) - prim_vlog(vu, ul, unit)
                         - prim_vlog(vd, ur, unit) + prim_vlog(vd, ul, unit);
                REAL Ir = CORNERS(prim_r, ul, ur, vd, vu);
                fx += (REAL)dx[c] * (xmxc * Kx0 + Ivl) + (REAL)dy[c] * (ymyc * Kx0 - Ir);
                fy += (REAL)dx[c] * (xmxc * Ky0 - Ir) + (REAL)dy[c] * (ymyc * Ky0 + Iul);
            }
        }
        Fx[t] = (double)((REAL)G * fx);
        Fy[t] = (double)((REAL)G * fy);
    }
    return used;
}
