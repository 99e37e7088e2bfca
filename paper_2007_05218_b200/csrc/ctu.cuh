// ctu.cuh -- the unsplit corner-transport-upwind update O12 (readings C1..C9; SURVEY 8(f)
// NEXT-2): PPM + characteristic tracing + transverse flux corrections + ONE conservative update per step.
//
// First CUDA path of this row: correct before fast.  Every kernel gives a thread one zone (or one face) of
// one box and keeps the intermediate fields in HBM, in arrays laid out like a state component (padded zones,
// i fastest, so every access is coalesced along x):
//   QM[d], QP[d]  traced states on the low / high face of every zone -1 .. nb, d = 0, 1, 2   (NQ components each)
//   F1[d]         first fluxes on the low face of zones 0 .. nb along d, -1 .. nb across       (NFLUX components)
//   F2[d]         final fluxes on the low face of zones 0 .. nb along d, valid across          (NFLUX components)
// = 12 * NQ padded arrays per box.  The 512^3 state would need 300 GB of them, so hydro_ctu_step works through
// the boxes in BATCHES that fit the scratch buffer the caller provides (boxes are independent within a step
// once the ghosts are filled).  Hydro variables and species are separate launches, as in the
// method-of-lines path: the species kernels read the mass flux the hydro kernels leave in F*[d][0].
//
// The arithmetic follows the oracle's expressions operator for operator (the strict build reproduces
// oracle_ctu_step bit for bit; tests/strict_bits_helper.py).
#pragma once
#include "hydro_device.cuh"

namespace hydro {

struct CtuArgs {
    const double* U;       // state at time n, ghosts filled
    double* Unew;          // state at time n+1 (valid zones written)
    double* Q;             // scratch of the batch: per box 12 * NQ padded arrays, see ctu_off
    const double* dt_dev;  // device dt
    int box0, nbatch;      // boxes box0 .. box0 + nbatch - 1 of the MultiFab
};

// offset of array (kind, d) of batch box bb: kind 0 QM, 1 QP, 2 F1, 3 F2; nq components each
__device__ __forceinline__ long long ctu_off(const Geom& g, int bb, int kind, int d)
{
    const long long nq = g.nflux;
    return ((long long)bb * 12 + kind * 3 + d) * nq * g.cstride;
}

constexpr int CTU_BY = 4;      // a CTA = 32 zones along x times CTU_BY rows

// block (32, CTU_BY), grid (ceil(n0/32) * nbatch, ceil(n1/CTU_BY), n2) with n_d = nb_d + 2*ext (+1 along `face`):
// zone / face indices lo .. of the batch box; returns false outside
__device__ __forceinline__ bool ctu_zone(const Geom& g, const int (&lo)[3], const int (&n)[3], int& bb, int (&ijk)[3])
{
    const int xblocks = (n[0] + 31) / 32;
    bb = blockIdx.x / xblocks;
    const int i = (blockIdx.x - bb * xblocks) * 32 + threadIdx.x;
    const int j = blockIdx.y * CTU_BY + threadIdx.y;
    if (i >= n[0] || j >= n[1]) return false;
    ijk[0] = lo[0] + i; ijk[1] = lo[1] + j; ijk[2] = lo[2] + blockIdx.z;
    return true;
}

__device__ __forceinline__ long long ctu_z(const Geom& g, const int (&ijk)[3])
{
    return ((long long)(ijk[2] + g.ng) * g.nt[1] + (ijk[1] + g.ng)) * g.nt[0] + (ijk[0] + g.ng);
}

// C2: parabola averages over the domain of dependence of a wave
__device__ __forceinline__ double ctu_Ip(double lam, double dtdx, double a, double aL, double aR)
{
    if (!(lam > 0.0)) return aR;
    const double sig = fabs(lam) * dtdx;
    const double da = aR - aL, a6 = 6.0 * (a - HALF * (aL + aR));
    return aR - HALF * sig * (da - (1.0 - (2.0 / 3.0) * sig) * a6);
}
__device__ __forceinline__ double ctu_Im(double lam, double dtdx, double a, double aL, double aR)
{
    if (!(lam < 0.0)) return aL;
    const double sig = fabs(lam) * dtdx;
    const double da = aR - aL, a6 = 6.0 * (a - HALF * (aL + aR));
    return aL + HALF * sig * (da + (1.0 - (2.0 / 3.0) * sig) * a6);
}

// monotonised parabola of the centre zone of five values (O3 + O4)
__device__ __forceinline__ void ctu_parabola(const double (&a)[5], double& aL, double& aR)
{
    const double sm = ppm_slope(a[0], a[1], a[2]), s0 = ppm_slope(a[1], a[2], a[3]), sp = ppm_slope(a[2], a[3], a[4]);
    const double el = ppm_edge(a[1], a[2], sm, s0), er = ppm_edge(a[2], a[3], s0, sp);
    ppm_mono(el, er, a[2], aL, aR);
}

// ---- C2-C5, hydro variables: traced states of zones -1 .. nb of every direction, along DIR ----------------------
template <int DIR>
__global__ void __launch_bounds__(32 * CTU_BY)
k_ctu_trace_hydro(const __grid_constant__ Geom g, const __grid_constant__ CtuArgs a)
{
    const int lo[3] = {-1, -1, -1}, n[3] = {g.nb[0] + 2, g.nb[1] + 2, g.nb[2] + 2};
    int bb, ijk[3];
    if (!ctu_zone(g, lo, n, bb, ijk)) return;
    const long long z = ctu_z(g, ijk);
    const long long st = DIR == 0 ? 1 : (DIR == 1 ? (long long)g.nt[0] : (long long)g.nt[0] * g.nt[1]);
    const double* Ub = a.U + (long long)(a.box0 + bb) * g.bstride + z;
    const double dtdx = *a.dt_dev * g.dxinv[DIR];
    double q[5][5];                                   // [variable][zone -2 .. +2]
#pragma unroll
    for (int m = 0; m < 5; ++m) {
        const double* Uz = Ub + (m - 2) * st;
        double qq[5], rinv;
        cons_to_prim(g, ldg(Uz), ldg(Uz + g.cstride), ldg(Uz + 2 * g.cstride), ldg(Uz + 3 * g.cstride), ldg(Uz + 5 * g.cstride), qq, rinv);
#pragma unroll
        for (int v = 0; v < 5; ++v) q[v][m] = qq[v];
    }
    double aL[5], aR[5], ac[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { ctu_parabola(q[v], aL[v], aR[v]); ac[v] = q[v][2]; }
    constexpr int in = 1 + DIR;
    const double rho = ac[0], un = ac[in], pr = ac[4];
#ifdef HYDRO_STRICT
    const double c = sqrt(g.gamma * pr / rho);
#else
    const double c = dsqrt(ddiv(g.gamma * pr, rho));
#endif
    const double lam[3] = {un - c, un, un + c};
    const int hv[3] = {0, in, 4};
    double* QM = a.Q + ctu_off(g, bb, 0, DIR) + z;
    double* QP = a.Q + ctu_off(g, bb, 1, DIR) + z;
#pragma unroll
    for (int side = 0; side < 2; ++side) {
        double I[3][3];
#pragma unroll
        for (int w = 0; w < 3; ++w)
#pragma unroll
            for (int v = 0; v < 3; ++v)
                I[w][v] = side ? ctu_Ip(lam[w], dtdx, ac[hv[v]], aL[hv[v]], aR[hv[v]]) : ctu_Im(lam[w], dtdx, ac[hv[v]], aL[hv[v]], aR[hv[v]]);
        const bool reaches = side ? (lam[2] > 0.0) : (lam[0] < 0.0);
        double ref[3];
#pragma unroll
        for (int v = 0; v < 3; ++v) ref[v] = reaches ? I[side ? 2 : 0][v] : ac[hv[v]];
        const double dum = ref[1] - I[0][1], dpm = ref[2] - I[0][2];
        const double drho0 = ref[0] - I[1][0], dp0 = ref[2] - I[1][2];
        const double dup = ref[1] - I[2][1], dpp = ref[2] - I[2][2];
        double am = HALF * (ddiv(dpm, rho * c) - dum) * ddiv(rho, c);
        double ap = HALF * (ddiv(dpp, rho * c) + dup) * ddiv(rho, c);
        double a0 = drho0 - ddiv(dp0, c * c);
        if (side) { am = lam[0] > 0.0 ? -am : 0.0; ap = lam[2] > 0.0 ? -ap : 0.0; a0 = lam[1] > 0.0 ? -a0 : 0.0; }
        else { am = lam[0] < 0.0 ? -am : 0.0; ap = lam[2] < 0.0 ? -ap : 0.0; a0 = lam[1] < 0.0 ? -a0 : 0.0; }
        double qf[5];
        qf[0] = dmax(ref[0] + ap + am + a0, g.small_dens);
        qf[in] = ref[1] + (ap - am) * ddiv(c, rho);
        qf[4] = dmax(ref[2] + (ap + am) * (c * c), g.small_pres);
#pragma unroll
        for (int v = 1; v < 4; ++v) {
            if (v == in) continue;
            if (side) qf[v] = lam[1] > 0.0 ? ctu_Ip(lam[1], dtdx, ac[v], aL[v], aR[v]) : ac[v];
            else qf[v] = lam[1] < 0.0 ? ctu_Im(lam[1], dtdx, ac[v], aL[v], aR[v]) : ac[v];
        }
        double* Qf = side ? QP : QM;
#pragma unroll
        for (int v = 0; v < 5; ++v) Qf[v * g.cstride] = qf[v];
    }
}

// ---- C4: all species of a zone (the five reciprocal densities of the stencil are formed once) -------------------
template <int DIR>
__global__ void __launch_bounds__(32 * CTU_BY)
k_ctu_trace_species(const __grid_constant__ Geom g, const __grid_constant__ CtuArgs a)
{
    const int lo[3] = {-1, -1, -1}, n[3] = {g.nb[0] + 2, g.nb[1] + 2, g.nb[2] + 2};
    int bb, ijk[3];
    if (!ctu_zone(g, lo, n, bb, ijk)) return;
    const long long z = ctu_z(g, ijk);
    const long long st = DIR == 0 ? 1 : (DIR == 1 ? (long long)g.nt[0] : (long long)g.nt[0] * g.nt[1]);
    const double* Ub = a.U + (long long)(a.box0 + bb) * g.bstride + z;
    const double dtdx = *a.dt_dev * g.dxinv[DIR];
    double rinv[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) rinv[m] = drcp(dmax(ldg(Ub + (m - 2) * st), g.small_dens));
    const double un = ldg(Ub + (long long)(1 + DIR) * g.cstride) * rinv[2];
    double* QM = a.Q + ctu_off(g, bb, 0, DIR) + z;
    double* QP = a.Q + ctu_off(g, bb, 1, DIR) + z;
#pragma unroll 2
    for (int s = 0; s < g.nspec; ++s) {
        const double* Xb = Ub + (long long)(6 + s) * g.cstride;
        double X[5];
#pragma unroll
        for (int m = 0; m < 5; ++m) X[m] = ldg(Xb + (m - 2) * st) * rinv[m];
        double aL, aR;
        ctu_parabola(X, aL, aR);
        QM[(long long)(5 + s) * g.cstride] = un < 0.0 ? ctu_Im(un, dtdx, X[2], aL, aR) : X[2];
        QP[(long long)(5 + s) * g.cstride] = un > 0.0 ? ctu_Ip(un, dtdx, X[2], aL, aR) : X[2];
    }
}

// ---- C6 / C7-C9: fluxes on the low face of a zone.  FINAL = false: first fluxes from the traced states (zones
// 0 .. nb along DIR, -1 .. nb across).  FINAL = true: transverse corrections + gravity, final fluxes (valid across).
__device__ __forceinline__ void ctu_correct(const Geom& g, const CtuArgs& a, int bb, int DIR, long long zz, double hdt,
                                            double (&q)[5])
{
    // conserved form of the face state, minus half a step of the transverse flux differences of the zone zz
    double Uc[5];
    Uc[0] = q[0];
    Uc[1] = q[0] * q[1]; Uc[2] = q[0] * q[2]; Uc[3] = q[0] * q[3];
    Uc[4] = q[4] * g.gm1inv + HALF * q[0] * (q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int dd = 0; dd < 3; ++dd) {
        if (dd == DIR) continue;
        const long long sd = dd == 0 ? 1 : (dd == 1 ? (long long)g.nt[0] : (long long)g.nt[0] * g.nt[1]);
        const double* F = a.Q + ctu_off(g, bb, 2, dd) + zz;
#pragma unroll
        for (int c = 0; c < 5; ++c) Uc[c] = Uc[c] - hdt * g.dxinv[dd] * (F[c * g.cstride + sd] - F[c * g.cstride]);
    }
    const double rho = dmax(Uc[0], g.small_dens);
    const double rinv = drcp(rho);
    q[0] = rho;
    q[1] = Uc[1] * rinv; q[2] = Uc[2] * rinv; q[3] = Uc[3] * rinv;
    const double K = HALF * (Uc[1] * Uc[1] + Uc[2] * Uc[2] + Uc[3] * Uc[3]) * rinv;
    q[4] = dmax(g.gm1 * (Uc[4] - K), g.small_pres);
    if (g.has_grav) { q[1] = q[1] + hdt * g.grav[0]; q[2] = q[2] + hdt * g.grav[1]; q[3] = q[3] + hdt * g.grav[2]; }
}

template <int DIR, bool FINAL>
__global__ void __launch_bounds__(32 * CTU_BY)
k_ctu_flux_hydro(const __grid_constant__ Geom g, const __grid_constant__ CtuArgs a)
{
    constexpr int E = FINAL ? 0 : 1;
    int lo[3] = {-E, -E, -E}, n[3] = {g.nb[0] + 2 * E, g.nb[1] + 2 * E, g.nb[2] + 2 * E};
    lo[DIR] = 0; n[DIR] = g.nb[DIR] + 1;
    int bb, ijk[3];
    if (!ctu_zone(g, lo, n, bb, ijk)) return;
    const long long z = ctu_z(g, ijk);
    const long long st = DIR == 0 ? 1 : (DIR == 1 ? (long long)g.nt[0] : (long long)g.nt[0] * g.nt[1]);
    const double* QP = a.Q + ctu_off(g, bb, 1, DIR) + z - st;      // high face of the zone below
    const double* QM = a.Q + ctu_off(g, bb, 0, DIR) + z;           // low face of this zone
    double qL[5], qR[5], F[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { qL[v] = QP[v * g.cstride]; qR[v] = QM[v * g.cstride]; }
    if (FINAL) {
        const double hdt = HALF * *a.dt_dev;
        ctu_correct(g, a, bb, DIR, z - st, hdt, qL);
        ctu_correct(g, a, bb, DIR, z, hdt, qR);
    }
    hllc<DIR>(g, qL, qR, F);
    double* Fo = a.Q + ctu_off(g, bb, FINAL ? 3 : 2, DIR) + z;
#pragma unroll
    for (int c = 0; c < 5; ++c) Fo[c * g.cstride] = F[c];
}

// species fluxes F_rho * X_upwind (S7) of all species of a face; FINAL: X of the corrected state = (rho*X)' / rho'
template <int DIR, bool FINAL>
__global__ void __launch_bounds__(32 * CTU_BY)
k_ctu_flux_species(const __grid_constant__ Geom g, const __grid_constant__ CtuArgs a)
{
    constexpr int E = FINAL ? 0 : 1;
    int lo[3] = {-E, -E, -E}, n[3] = {g.nb[0] + 2 * E, g.nb[1] + 2 * E, g.nb[2] + 2 * E};
    lo[DIR] = 0; n[DIR] = g.nb[DIR] + 1;
    int bb, ijk[3];
    if (!ctu_zone(g, lo, n, bb, ijk)) return;
    const long long z = ctu_z(g, ijk);
    const long long st = DIR == 0 ? 1 : (DIR == 1 ? (long long)g.nt[0] : (long long)g.nt[0] * g.nt[1]);
    constexpr int D1 = DIR == 0 ? 1 : 0, D2 = DIR == 2 ? 1 : 2;       // the other two directions, ascending
    const long long s1 = D1 == 0 ? 1 : (long long)g.nt[0];
    const long long s2 = D2 == 1 ? (long long)g.nt[0] : (long long)g.nt[0] * g.nt[1];
    const double* QPl = a.Q + ctu_off(g, bb, 1, DIR) + z - st;        // left state: high face of the zone below
    const double* QMr = a.Q + ctu_off(g, bb, 0, DIR) + z;             // right state: low face of this zone
    const double* F1a = a.Q + ctu_off(g, bb, 2, D1);
    const double* F1b = a.Q + ctu_off(g, bb, 2, D2);
    double* Fo = a.Q + ctu_off(g, bb, FINAL ? 3 : 2, DIR) + z;
    const double Frho = Fo[0];
    const double hdt = FINAL ? HALF * *a.dt_dev : 0.0;
    double rfL = 0.0, rfR = 0.0, rinvL = 0.0, rinvR = 0.0;
    if (FINAL) {      // corrected densities of the two face states (the expressions of ctu_correct)
        rfL = QPl[0]; rfR = QMr[0];
        double rL = rfL, rR = rfR;
        rL = rL - hdt * g.dxinv[D1] * (F1a[z - st + s1] - F1a[z - st]);
        rL = rL - hdt * g.dxinv[D2] * (F1b[z - st + s2] - F1b[z - st]);
        rR = rR - hdt * g.dxinv[D1] * (F1a[z + s1] - F1a[z]);
        rR = rR - hdt * g.dxinv[D2] * (F1b[z + s2] - F1b[z]);
        rinvL = drcp(dmax(rL, g.small_dens)); rinvR = drcp(dmax(rR, g.small_dens));
    }
#pragma unroll 2
    for (int s = 0; s < g.nspec; ++s) {
        const long long cs5 = (long long)(5 + s) * g.cstride;
        double XL = QPl[cs5], XR = QMr[cs5];
        if (FINAL) {
            double xl = rfL * XL, xr = rfR * XR;
            xl = xl - hdt * g.dxinv[D1] * (F1a[cs5 + z - st + s1] - F1a[cs5 + z - st]);
            xl = xl - hdt * g.dxinv[D2] * (F1b[cs5 + z - st + s2] - F1b[cs5 + z - st]);
            xr = xr - hdt * g.dxinv[D1] * (F1a[cs5 + z + s1] - F1a[cs5 + z]);
            xr = xr - hdt * g.dxinv[D2] * (F1b[cs5 + z + s2] - F1b[cs5 + z]);
            XL = xl * rinvL; XR = xr * rinvR;
        }
        Fo[cs5] = Frho * (Frho >= 0.0 ? XL : XR);
    }
}

// ---- C1 + C8 + O7: conservative update of the valid zones ----------------------------------------------------
__global__ void __launch_bounds__(32 * CTU_BY)
k_ctu_update_hydro(const __grid_constant__ Geom g, const __grid_constant__ CtuArgs a)
{
    const int lo[3] = {0, 0, 0}, n[3] = {g.nb[0], g.nb[1], g.nb[2]};
    int bb, ijk[3];
    if (!ctu_zone(g, lo, n, bb, ijk)) return;
    const long long z = ctu_z(g, ijk);
    const long long st[3] = {1, g.nt[0], (long long)g.nt[0] * g.nt[1]};
    const double dt = *a.dt_dev;
    const long long zo = (long long)(a.box0 + bb) * g.bstride + z;
    double us[5], L[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) {
        us[c] = a.U[zo + c * g.cstride];
        const double* F0 = a.Q + ctu_off(g, bb, 3, 0) + c * g.cstride + z;
        const double* F1 = a.Q + ctu_off(g, bb, 3, 1) + c * g.cstride + z;
        const double* F2 = a.Q + ctu_off(g, bb, 3, 2) + c * g.cstride + z;
        L[c] = -(F0[st[0]] - F0[0]) * g.dxinv[0] - (F1[st[1]] - F1[0]) * g.dxinv[1] - (F2[st[2]] - F2[0]) * g.dxinv[2];
    }
    if (g.has_grav) {
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            L[1 + e] += us[0] * g.grav[e];
            L[4] += (us[1 + e] + HALF * dt * us[0] * g.grav[e]) * g.grav[e];
        }
    }
    double un[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) { un[c] = us[c] + dt * L[c]; a.Unew[zo + c * g.cstride] = un[c]; }
    double re = un[4] - ddiv(HALF * (un[1] * un[1] + un[2] * un[2] + un[3] * un[3]), un[0]);
    if (re < g.floor_rhoe) re = g.floor_rhoe;
    a.Unew[zo + 5 * g.cstride] = re;
}

__global__ void __launch_bounds__(32 * CTU_BY)
k_ctu_update_species(const __grid_constant__ Geom g, const __grid_constant__ CtuArgs a)
{
    const int lo[3] = {0, 0, 0}, n[3] = {g.nb[0], g.nb[1], g.nb[2]};
    int bb, ijk[3];
    if (!ctu_zone(g, lo, n, bb, ijk)) return;
    const long long z = ctu_z(g, ijk);
    const long long st[3] = {1, g.nt[0], (long long)g.nt[0] * g.nt[1]};
    const double dt = *a.dt_dev;
#pragma unroll 2
    for (int s = 0; s < g.nspec; ++s) {
        const long long cs5 = (long long)(5 + s) * g.cstride;
        const double* F0 = a.Q + ctu_off(g, bb, 3, 0) + cs5 + z;
        const double* F1 = a.Q + ctu_off(g, bb, 3, 1) + cs5 + z;
        const double* F2 = a.Q + ctu_off(g, bb, 3, 2) + cs5 + z;
        const double L = -(F0[st[0]] - F0[0]) * g.dxinv[0] - (F1[st[1]] - F1[0]) * g.dxinv[1] - (F2[st[2]] - F2[0]) * g.dxinv[2];
        const long long zo = (long long)(a.box0 + bb) * g.bstride + (long long)(6 + s) * g.cstride + z;
        a.Unew[zo] = a.U[zo] + dt * L;
    }
}

}  // namespace hydro
