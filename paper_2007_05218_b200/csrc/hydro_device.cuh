// hydro_device.cuh -- layout descriptor and per-zone / per-face device arithmetic of the
// hot path (steps O2..O7).  sm_100a only.  Shares nothing with oracle/.
//
// Every expression is written in the association DESIGN.md fixes (left to right, one
// IEEE operation per operator, reciprocal constants as multipliers), so that a build with
// -fmad=false reproduces the scheme's definition bit for bit and an FMA build differs by
// rounding only.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace hydro {

constexpr double HALF = 0.5;
constexpr double SIXTH = 1.0 / 6.0;

// One descriptor for the whole MultiFab, passed by value as a __grid_constant__ kernel
// parameter: no per-array bounds live in registers (the paper's Volta lesson,
// PAPER.md:59).
struct Geom {
    int nb[3];       // valid zones per box
    int nt[3];       // padded zones per box
    int NB[3];       // boxes per dimension
    int ndom[3];
    int bc_lo[3], bc_hi[3];
    int ng, nspec, nvar, nflux, nboxes, has_grav, flatten, evolve;
    long long cstride;   // doubles per (box, component) of a state     = nt0*nt1*nt2
    long long bstride;   // doubles per box of a state                  = cstride*nvar
    long long lcstride;  // doubles per (box, component) of the accumulator = nb0*nb1*nb2
    long long lbstride;  // = lcstride*nflux
    long long fbstride;  // doubles per box of the face mass-flux array = (nb0+1)(nb1+1)(nb2+1)
    double dxinv[3];
    double gamma, gm1, gm1inv, small_dens, small_pres, floor_rhoe, cfl, vol;
    double grav[3];
};

__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

// streaming loads/stores for data touched once per kernel
__device__ __forceinline__ double ldg(const double* p) { return __ldg(p); }

// ---- O3: limited van Leer slope (CW84 1.7-1.8) ---------------------------------------
__device__ __forceinline__ double ppm_slope(double am, double a, double ap)
{
    const double dp = ap - a;
    const double dm = a - am;
    const double dc = HALF * (ap - am);
    const double lim = dmin(fabs(dc), 2.0 * dmin(fabs(dp), fabs(dm)));   // = min(|dc|, 2|dp|, 2|dm|) exactly (x2 is exact)
    return (dp * dm > 0.0) ? copysign(lim, dc) : 0.0;
}

// ---- O3: fourth-order edge value between zones i and i+1 (CW84 1.6, uniform grid) ----
__device__ __forceinline__ double ppm_edge(double a, double ap, double s, double sp)
{
    return a + HALF * (ap - a) - SIXTH * (sp - s);
}

// ---- O4: monotonised parabola edges of one zone (CW84 1.10) --------------------------
// HYDRO_PPM_DIFF (default build only; the strict build keeps the definitional form below so that it stays equal to
// the oracle bit for bit): the same case analysis written on the edge differences dl = a - el, dr = er - a.  With
// d = dl + dr and a - (el + er)/2 = (dl - dr)/2, CW84's overshoot test d*(a - (el+er)/2) > d^2/6 is |dl| > 2|dr|
// (dl, dr of one sign, else the zone is flat), and 3a - 2er = a - 2dr: 7 FP64 operations instead of 13, the same
// three compares and four selects.  The two forms differ by rounding only (both branches are continuous).
#ifndef HYDRO_PPM_DIFF
#define HYDRO_PPM_DIFF 1
#endif
__device__ __forceinline__ void ppm_mono(double el, double er, double a, double& aL, double& aR)
{
#if !defined(HYDRO_STRICT) && HYDRO_PPM_DIFF
    const double dl = a - el, dr = er - a;
    const bool flat = dr * dl <= 0.0;
    const double dl2 = dl + dl, dr2 = dr + dr;
    const bool over_l = fabs(dl) > fabs(dr2);
    const bool over_r = fabs(dr) > fabs(dl2);
    const double l1 = over_l ? a - dr2 : el;
    const double r1 = over_r ? a + dl2 : er;
    aL = flat ? a : l1;
    aR = flat ? a : r1;
#else
    // branch-free: every candidate is evaluated and the CW84 (1.10) cases pick among them, so
    // the five variables of a zone stay in one basic block and interleave in the FP64 pipe.
    // The selected values are the same expressions as in the if/else form of the definition.
    const bool flat = (er - a) * (a - el) <= 0.0;
    const double d = er - el;
    const double m = a - HALF * (el + er);
    const double t = d * d * SIXTH;
    const double dm = d * m;
    const bool over_l = dm > t;
    const bool over_r = !over_l && (-t > dm);
#ifdef PPM_PRED
    double l1 = el, r1 = er;
    if (over_l) l1 = 3.0 * a - 2.0 * er;
    if (over_r) r1 = 3.0 * a - 2.0 * el;
    if (flat) { l1 = a; r1 = a; }
    aL = l1; aR = r1;
#else
    const double l1 = over_l ? 3.0 * a - 2.0 * er : el;
    const double r1 = over_r ? 3.0 * a - 2.0 * el : er;
    aL = flat ? a : l1;
    aR = flat ? a : r1;
#endif
#endif
}

// ---- division and square root ----------------------------------------------------------
// HYDRO_STRICT (the -fmad=false build): IEEE-correct '/' and sqrt(), bit-for-bit the scheme's
// definition.  Default build: branch-free Newton forms on the MUFU seeds (rcp/rsqrt.approx.f64),
// faithful to <= 1 ulp for the normal-range operands of this path (densities >= small_dens,
// pressures >= small_pres, wave-speed differences); no slow-path call, so no BSSY/BSYNC regions.
#ifdef HYDRO_STRICT
__device__ __forceinline__ double ddiv(double a, double b) { return a / b; }
__device__ __forceinline__ double drcp(double b) { return 1.0 / b; }
__device__ __forceinline__ double dsqrt(double x) { return sqrt(x); }
#else
__device__ __forceinline__ double drcp(double b)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
    double e = fma(-b, r, 1.0);      // seed is good to ~2^-20: two Newton steps reach 2^-80
    r = fma(r, e, r);
    e = fma(-b, r, 1.0);
    return fma(r, e, r);
}
__device__ __forceinline__ double ddiv(double a, double b)
{
    const double r = drcp(b);
    const double q = a * r;
    return fma(fma(-b, q, a), r, q);
}
__device__ __forceinline__ double dsqrt(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double g = x * y, h = 0.5 * y;
    double r = fma(-g, h, 0.5);      // coupled Newton on g ~ sqrt(x), h ~ 1/(2 sqrt(x))
    g = fma(g, r, g); h = fma(h, r, h);
    r = fma(-g, h, 0.5);
    g = fma(g, r, g); h = fma(h, r, h);
    g = fma(fma(-g, g, x), h, g);    // residual correction
    return x > 0.0 ? g : 0.0;
}
#endif

// ---- O5: HLLC flux of (rho, rho u, rho v, rho w, rho E) at one face ------------------
// DIR = face normal.  qL/qR = (rho, u, v, w, p) left/right states.
// uf = face-normal velocity of the fan (O11, reading G2): SM between the acoustic waves, else the upwind n.
template <int DIR>
__device__ __forceinline__ void hllc(const Geom& g, const double (&qL)[5], const double (&qR)[5],
                                     double (&F)[5], double& uf)
{
    const double rL = dmax(qL[0], g.small_dens), rR = dmax(qR[0], g.small_dens);
    const double pL = dmax(qL[4], g.small_pres), pR = dmax(qR[4], g.small_pres);
    const double nL = qL[1 + DIR], nR = qR[1 + DIR];
    const double rinvL = drcp(rL), rinvR = drcp(rR);
    const double cL = dsqrt(g.gamma * pL * rinvL), cR = dsqrt(g.gamma * pR * rinvR);
    const double SL = dmin(nL - cL, nR - cR);
    const double SR = dmax(nL + cL, nR + cR);
    const double EL = pL * g.gm1inv + HALF * rL * (qL[1] * qL[1] + qL[2] * qL[2] + qL[3] * qL[3]);
    const double ER = pR * g.gm1inv + HALF * rR * (qR[1] * qR[1] + qR[2] * qR[2] + qR[3] * qR[3]);

    // Star-region quantities are always evaluated (branch-free); when the face is supersonic
    // (SL >= 0 or SR <= 0) they are not selected.
    const bool star = !(SL >= 0.0) && !(SR <= 0.0);
    const double mL = rL * (SL - nL);
    const double mR = rR * (SR - nR);
    const double SM = ddiv(pR - pL + mL * nL - mR * nR, mL - mR);
    const bool left = star ? (SM >= 0.0) : (SL >= 0.0);
    const double rK = left ? rL : rR, pK = left ? pL : pR, nK = left ? nL : nR;
    const double EK = left ? EL : ER;
    double vK[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) vK[c] = left ? qL[1 + c] : qR[1 + c];

    const double rn = rK * nK;
    double FK[5], UK[5];
    FK[0] = rn;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        FK[1 + c] = rn * vK[c];
        if (c == DIR) FK[1 + c] = FK[1 + c] + pK;
        UK[1 + c] = rK * vK[c];
    }
    FK[4] = (EK + pK) * nK;
    UK[0] = rK;
    UK[4] = EK;
    const double rinvK = left ? rinvL : rinvR;
    const double S = left ? SL : SR;
    const double mK = left ? mL : mR;
    const double fac = ddiv(mK, S - SM);
    double Us[5];
    Us[0] = fac;
#pragma unroll
    for (int c = 0; c < 3; ++c) Us[1 + c] = fac * (c == DIR ? SM : vK[c]);
    Us[4] = fac * (EK * rinvK + (SM - nK) * (SM + ddiv(pK, mK)));
#pragma unroll
    for (int c = 0; c < 5; ++c) F[c] = star ? FK[c] + S * (Us[c] - UK[c]) : FK[c];
    uf = star ? SM : nK;
}

template <int DIR>
__device__ __forceinline__ void hllc(const Geom& g, const double (&qL)[5], const double (&qR)[5], double (&F)[5])
{
    double uf;
    hllc<DIR>(g, qL, qR, F, uf);
}

// ---- O2: conserved -> primitive for the five hydro variables -------------------------
__device__ __forceinline__ void cons_to_prim(const Geom& g, double rho, double mx, double my, double mz,
                                             double re, double (&q)[5], double& rinv)
{
    const double r = dmax(rho, g.small_dens);
    rinv = drcp(r);
    q[0] = r;
    q[1] = mx * rinv;
    q[2] = my * rinv;
    q[3] = mz * rinv;
    q[4] = dmax(g.gm1 * re, g.small_pres);
}

// ---- O7: stage combination (SSP-RK2, Shu-Osher form) ---------------------------------
template <int STAGE>
__device__ __forceinline__ double rk_combine(double us, double ubase, double dt, double L)
{
    if (STAGE == 0) return us + dt * L;
    return HALF * ubase + HALF * (us + dt * L);
}

}  // namespace hydro
