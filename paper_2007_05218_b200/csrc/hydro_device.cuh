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
    int ng, nspec, nvar, nflux, nboxes, has_grav;
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
    const double lim = dmin(fabs(dc), dmin(2.0 * fabs(dp), 2.0 * fabs(dm)));
    return (dp * dm > 0.0) ? copysign(lim, dc) : 0.0;
}

// ---- O3: fourth-order edge value between zones i and i+1 (CW84 1.6, uniform grid) ----
__device__ __forceinline__ double ppm_edge(double a, double ap, double s, double sp)
{
    return a + HALF * (ap - a) - SIXTH * (sp - s);
}

// ---- O4: monotonised parabola edges of one zone (CW84 1.10) --------------------------
__device__ __forceinline__ void ppm_mono(double el, double er, double a, double& aL, double& aR)
{
    double l = el, r = er;
    if ((r - a) * (a - l) <= 0.0) {
        l = a;
        r = a;
    } else {
        const double d = r - l;
        const double m = a - HALF * (l + r);
        const double t = d * d * SIXTH;
        const double dm = d * m;
        if (dm > t) l = 3.0 * a - 2.0 * r;
        else if (-t > dm) r = 3.0 * a - 2.0 * l;
    }
    aL = l;
    aR = r;
}

// ---- O5: HLLC flux of (rho, rho u, rho v, rho w, rho E) at one face ------------------
// DIR = face normal.  qL/qR = (rho, u, v, w, p) left/right states.
template <int DIR>
__device__ __forceinline__ void hllc(const Geom& g, const double (&qL)[5], const double (&qR)[5],
                                     double (&F)[5])
{
    const double rL = dmax(qL[0], g.small_dens), rR = dmax(qR[0], g.small_dens);
    const double pL = dmax(qL[4], g.small_pres), pR = dmax(qR[4], g.small_pres);
    const double nL = qL[1 + DIR], nR = qR[1 + DIR];
    const double rinvL = 1.0 / rL, rinvR = 1.0 / rR;
    const double cL = sqrt(g.gamma * pL * rinvL), cR = sqrt(g.gamma * pR * rinvR);
    const double SL = dmin(nL - cL, nR - cR);
    const double SR = dmax(nL + cL, nR + cR);
    const double EL = pL * g.gm1inv + HALF * rL * (qL[1] * qL[1] + qL[2] * qL[2] + qL[3] * qL[3]);
    const double ER = pR * g.gm1inv + HALF * rR * (qR[1] * qR[1] + qR[2] * qR[2] + qR[3] * qR[3]);

    // which side supplies the flux, and whether a star state is needed
    const bool star = !(SL >= 0.0) && !(SR <= 0.0);
    double SM = 0.0, mL = 0.0, mR = 0.0;
    bool left = (SL >= 0.0);
    if (star) {
        mL = rL * (SL - nL);
        mR = rR * (SR - nR);
        SM = (pR - pL + mL * nL - mR * nR) / (mL - mR);
        left = (SM >= 0.0);
    }
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
    if (star) {
        const double rinvK = left ? rinvL : rinvR;
        const double S = left ? SL : SR;
        const double mK = left ? mL : mR;
        const double fac = mK / (S - SM);
        double Us[5];
        Us[0] = fac;
#pragma unroll
        for (int c = 0; c < 3; ++c) Us[1 + c] = fac * (c == DIR ? SM : vK[c]);
        Us[4] = fac * (EK * rinvK + (SM - nK) * (SM + pK / mK));
#pragma unroll
        for (int c = 0; c < 5; ++c) F[c] = FK[c] + S * (Us[c] - UK[c]);
    } else {
#pragma unroll
        for (int c = 0; c < 5; ++c) F[c] = FK[c];
    }
}

// ---- O2: conserved -> primitive for the five hydro variables -------------------------
__device__ __forceinline__ void cons_to_prim(const Geom& g, double rho, double mx, double my, double mz,
                                             double re, double (&q)[5], double& rinv)
{
    const double r = dmax(rho, g.small_dens);
    rinv = 1.0 / r;
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
