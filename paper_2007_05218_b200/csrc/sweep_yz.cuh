// sweep_yz.cuh -- y- and z-direction reconstruct + Riemann + flux-difference kernels.
//
// A thread owns one pencil along DIR (fixed i and fixed other transverse index) and MARCHES
// along it with a rolling register window: one new zone is loaded per step (coalesced along
// i across the warp) and each slope, edge value, monotonised parabola and face flux is
// computed exactly once -- the de-duplicated form PAPER.md:57 says the V100 port had not
// explored.  The flux difference of a zone is complete when its high face is done, so no
// face-flux array is ever written except the mass flux F_rho (8 B/face) that the species
// kernels upwind with.
//
// Accumulator protocol per stage: sweep_x writes Lacc, the y sweep does Lacc -= dFy*dyinv,
// the z sweep (FINAL) forms L = Lacc - dFz*dzinv (+ gravity), applies the SSP-RK2 stage
// combination, re-synchronises rho*e and writes the destination state.  This reproduces
// L = -(dFx)*dxinv - (dFy)*dyinv - (dFz)*dzinv in exactly that association (O6).
#pragma once
#include "hydro_device.cuh"
#include "flatten.cuh"

namespace hydro {

struct SweepArgs {
    const double* Us;      // stage state (ghosts filled), read
    const double* Ubase;   // U0 (stage 1 combination), read; may alias Uout zone-for-zone
    double* Uout;          // destination state (valid zones written)   [FINAL only]
    double* Lacc;          // accumulator, NFLUX per valid zone
    double* Frho;          // face mass flux of this direction
    const double* dt_dev;  // device dt (hydro_step) or nullptr
    double dt;             // host dt when dt_dev == nullptr
    int seglen;            // zones per pencil segment along DIR
    int sbase;             // first species of this launch (species kernels)
    int xends;             // FINAL ring kernels: also write the x-direction ghost images of every zone
    // stage-1 FINAL hydro ring kernel: also reduce the CFL signal speed of the state it writes (O8)
    // and leave the next step's dt in dt_next[0] (max t in dt_next[1]); nullptr = off
    unsigned long long* red;
    double* dt_next;
    const double* FL;      // O10 flattening coefficients (padded, one array per box) or nullptr
    int ngroups, n_hi;     // k_march_species_groups: species groups in the launch, and how many carry the larger count
    int lacc_shift;        // species kernels: accumulator component = 5 + sbase + lacc_shift (0 for species; the
                           // O11 energy launch uses sbase = -1, i.e. state component 5, and the slot after the fluxes)
};

// pencil decode shared by both kernels.  Returns false if the thread has no pencil.
template <int DIR>
__device__ __forceinline__ bool pencil(const Geom& g, int seglen, int& i, int& t, int& b, int& m0, int& m1)
{
    constexpr int T = (DIR == 1) ? 2 : 1;              // the other transverse dimension
    // grid.x = (CTAs per box) * boxes: the box index rides in blockIdx.x (no 65535 limit)
    const int tiles = gridDim.x / g.nboxes;
    b = blockIdx.x / tiles;
    const int pid = (blockIdx.x - b * tiles) * blockDim.x + threadIdx.x;
    if (pid >= g.nb[0] * g.nb[T]) return false;
    i = pid % g.nb[0];
    t = pid / g.nb[0];
    m0 = blockIdx.y * seglen;
    m1 = min(m0 + seglen, g.nb[DIR]);
    return true;
}

// ------------------------------------------------------------------------------------
// hydro variables: (rho, u, v, w, p) reconstruction, HLLC, flux difference
// ------------------------------------------------------------------------------------
template <int DIR, bool FINAL, int STAGE, int BS, bool EVOLVE = false>
__global__ void __launch_bounds__(BS)
k_sweep_hydro(const __grid_constant__ Geom g, const __grid_constant__ SweepArgs a)
{
    int i, t, b, m0, m1;
    if (!pencil<DIR>(g, a.seglen, i, t, b, m0, m1)) return;
    const int j = (DIR == 1) ? 0 : t, k = (DIR == 1) ? t : 0;      // index along DIR starts at 0
    const long long mstride = (DIR == 1) ? g.nt[0] : (long long)g.nt[0] * g.nt[1];
    const long long lmstride = (DIR == 1) ? g.nb[0] : (long long)g.nb[0] * g.nb[1];
    // padded offset of valid zone (i,j,k) with the DIR index = 0
    const long long z0 = ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0] + (i + g.ng);
    const long long l0 = ((long long)k * g.nb[1] + j) * g.nb[0] + i;
    const double* Ub = a.Us + (long long)b * g.bstride + z0;
    double* Lb = a.Lacc + (long long)b * g.lbstride + l0;
    // face array of direction DIR: dims nb + (1 along DIR); face f = low face of zone f
    const long long fmstride = (DIR == 1) ? g.nb[0] : (long long)g.nb[0] * g.nb[1];
    double* Fb = a.Frho + (long long)b * g.fbstride + ((DIR == 1) ? (long long)k * (g.nb[1] + 1) * g.nb[0] + i
                                                                   : (long long)j * g.nb[0] + i);
    const double dinv = g.dxinv[DIR];
    const double dt = a.dt_dev ? *a.dt_dev : a.dt;

    double a1[5], a2[5], s1[5], e1[5], aR1[5], Fp[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { a1[v] = a2[v] = s1[v] = e1[v] = aR1[v] = Fp[v] = 0.0; }
    double ufp = 0.0;                                  // O11: face velocity of the previous face

    for (int n = m0 - 3; n <= m1 + 2; ++n) {
        // load zone n, convert to primitives (O2)
        const double* Un = Ub + n * mstride;
        double q[5], rinv;
        cons_to_prim(g, ldg(Un), ldg(Un + g.cstride), ldg(Un + 2 * g.cstride), ldg(Un + 3 * g.cstride),
                     ldg(Un + 5 * g.cstride), q, rinv);
        double qL[5], qR[5];
        // O10 coefficient of zone n-2 (defined on zones -1 .. nb; the other parabolas are not used)
        const bool flat = a.FL != nullptr && n - 2 >= -1 && n - 2 <= g.nb[DIR];
        const double f2 = flat ? ldg(a.FL + (long long)b * g.cstride + z0 + (long long)(n - 2) * mstride) : 1.0;
        const double omf2 = 1.0 - f2;
        // window before the shift: a1 = a[n-1], a2 = a[n-2], s1 = s[n-2], e1 = e[n-5/2], aR1 = aR(n-3)
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double sn = ppm_slope(a2[v], a1[v], q[v]);        // s[n-1]     (n >= m0-1)
            const double en = ppm_edge(a2[v], a1[v], s1[v], sn);    // e[n-3/2]   (n >= m0)
            double aL, aR;
            ppm_mono(e1[v], en, a2[v], aL, aR);                     // zone n-2   (n >= m0+1)
            if (flat) flat_blend(f2, omf2, a2[v], aL, aR);
            qL[v] = aR1[v];                                         // face n-5/2 (n >= m0+2)
            qR[v] = aL;
            a2[v] = a1[v]; a1[v] = q[v]; s1[v] = sn; e1[v] = en; aR1[v] = aR;
        }
        if (n < m0 + 2) continue;                      // warp-uniform: window still filling
        double F[5], uf;
        hllc<DIR>(g, qL, qR, F, uf);                   // face between zones n-3 and n-2
        Fb[(long long)(n - 2) * fmstride] = F[0];
        if (n >= m0 + 3) {
            const int z = n - 3;                       // zone whose two faces are now known
            double* Lz = Lb + z * lmstride;
            // O11: div(u_face) so far + this direction's part (accumulator slot nflux + 1)
            double dsum = 0.0;
            if (EVOLVE) {
                dsum = Lz[(long long)(g.nflux + 1) * g.lcstride] + (uf - ufp) * dinv;
                Lz[(long long)(g.nflux + 1) * g.lcstride] = dsum;
            }
            if (!FINAL) {
#pragma unroll
                for (int c = 0; c < 5; ++c) Lz[c * g.lcstride] = Lz[c * g.lcstride] - (F[c] - Fp[c]) * dinv;
            } else {
                double L[5];
#pragma unroll
                for (int c = 0; c < 5; ++c) L[c] = Lz[c * g.lcstride] - (F[c] - Fp[c]) * dinv;
                const double* Uz = Ub + z * mstride;   // raw stage state of the zone (L1/L2 hit)
                double us[5];
#pragma unroll
                for (int c = 0; c < 5; ++c) us[c] = Uz[c * g.cstride];
                if (g.has_grav) {
                    L[1] += us[0] * g.grav[0];
                    L[2] += us[0] * g.grav[1];
                    L[3] += us[0] * g.grav[2];
                    L[4] += us[1] * g.grav[0] + us[2] * g.grav[1] + us[3] * g.grav[2];
                }
                const long long zo = (long long)b * g.bstride + z0 + z * mstride;
                double un[5];
#pragma unroll
                for (int c = 0; c < 5; ++c) {
                    const double ub = (STAGE == 1) ? a.Ubase[zo + c * g.cstride] : 0.0;
                    un[c] = rk_combine<STAGE>(us[c], ub, dt, L[c]);
                    a.Uout[zo + c * g.cstride] = un[c];
                }
                const double K = ddiv(HALF * (un[1] * un[1] + un[2] * un[2] + un[3] * un[3]), un[0]);
                double re = un[4] - K;
                if (EVOLVE) {      // rho*e is written by the energy launch; leave rho*E - K (slot nflux + 2) for its switch
                    double eE = re;
                    if (fabs(re - 1.0e-4 * un[4]) <= 1e-12 * fabs(un[4])) {
                        // within rounding of the switch threshold: K exactly as the definition forms it (march_ring.cuh)
                        const double m2 = __dadd_rn(__dadd_rn(__dmul_rn(un[1], un[1]), __dmul_rn(un[2], un[2])), __dmul_rn(un[3], un[3]));
                        eE = __dsub_rn(un[4], __ddiv_rn(__dmul_rn(HALF, m2), un[0]));
                    }
                    Lz[(long long)(g.nflux + 2) * g.lcstride] = eE;
                } else {
                    if (re < g.floor_rhoe) re = g.floor_rhoe;
                    a.Uout[zo + 5 * g.cstride] = re;
                }
            }
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) Fp[c] = F[c];
        ufp = uf;
    }
}

// ------------------------------------------------------------------------------------
// passive species: X_k reconstruction, upwinding with the face mass flux (S7)
// NS species per thread (a1.sbase .. sbase+NS-1)
// ------------------------------------------------------------------------------------
// ENERGY (NS = 1, launched with sbase = -1 and lacc_shift = nflux - 4): the one "species" is e = rho*e / rho of O11;
// its FINAL update adds -p div(u_face) and ends with the dual-energy switch (as k_march_species<ENERGY>).
template <int DIR, bool FINAL, int STAGE, int NS, int BS, bool ENERGY = false>
__global__ void __launch_bounds__(BS)
k_sweep_species(const __grid_constant__ Geom g, const __grid_constant__ SweepArgs a)
{
    int i, t, b, m0, m1;
    if (!pencil<DIR>(g, a.seglen, i, t, b, m0, m1)) return;
    const int j = (DIR == 1) ? 0 : t, k = (DIR == 1) ? t : 0;
    const long long mstride = (DIR == 1) ? g.nt[0] : (long long)g.nt[0] * g.nt[1];
    const long long lmstride = (DIR == 1) ? g.nb[0] : (long long)g.nb[0] * g.nb[1];
    const long long z0 = ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0] + (i + g.ng);
    const long long l0 = ((long long)k * g.nb[1] + j) * g.nb[0] + i;
    const double* Ub = a.Us + (long long)b * g.bstride + z0;
    const double* Xb = Ub + (long long)(6 + a.sbase) * g.cstride;
    double* Lb = a.Lacc + (long long)b * g.lbstride + l0 + (long long)(5 + a.sbase + a.lacc_shift) * g.lcstride;
    const long long fmstride = (DIR == 1) ? g.nb[0] : (long long)g.nb[0] * g.nb[1];
    const double* Fb = a.Frho + (long long)b * g.fbstride + ((DIR == 1) ? (long long)k * (g.nb[1] + 1) * g.nb[0] + i
                                                                         : (long long)j * g.nb[0] + i);
    const double dinv = g.dxinv[DIR];
    const double dt = a.dt_dev ? *a.dt_dev : a.dt;

    double a1[NS], a2[NS], s1[NS], e1[NS], aR1[NS], Fp[NS];
#pragma unroll
    for (int v = 0; v < NS; ++v) { a1[v] = a2[v] = s1[v] = e1[v] = aR1[v] = Fp[v] = 0.0; }

    for (int n = m0 - 3; n <= m1 + 2; ++n) {
        const double rinv = drcp(dmax(ldg(Ub + n * mstride), g.small_dens));
        const bool haveF = (n >= m0 + 2);
        const double Frho = haveF ? ldg(Fb + (long long)(n - 2) * fmstride) : 0.0;
        const bool upd = (n >= m0 + 3);
        const int z = n - 3;
        const bool flat = a.FL != nullptr && n - 2 >= -1 && n - 2 <= g.nb[DIR];
        const double f2 = flat ? ldg(a.FL + (long long)b * g.cstride + z0 + (long long)(n - 2) * mstride) : 1.0;
        const double omf2 = 1.0 - f2;
#pragma unroll
        for (int v = 0; v < NS; ++v) {
            const double X = ldg(Xb + n * mstride + v * g.cstride) * rinv;
            const double sn = ppm_slope(a2[v], a1[v], X);
            const double en = ppm_edge(a2[v], a1[v], s1[v], sn);
            double aL, aR;
            ppm_mono(e1[v], en, a2[v], aL, aR);
            if (flat) flat_blend(f2, omf2, a2[v], aL, aR);
            const double Fs = Frho * (Frho >= 0.0 ? aR1[v] : aL);
            a2[v] = a1[v]; a1[v] = X; s1[v] = sn; e1[v] = en; aR1[v] = aR;
            if (upd) {
                double* Lz = Lb + z * lmstride + v * g.lcstride;
                double L = *Lz - (Fs - Fp[v]) * dinv;
                if (!FINAL) {
                    *Lz = L;
                } else {
                    const long long zo = (long long)b * g.bstride + z0 + z * mstride +
                                         (long long)(6 + a.sbase + v) * g.cstride;
                    const double us = a.Us[zo];
                    const double ub = (STAGE == 1) ? a.Ubase[zo] : 0.0;
                    if (ENERGY) L = L - dmax(g.gm1 * us, g.small_pres) * Lz[g.lcstride];      // - p_c * div(u_face)
                    double un = rk_combine<STAGE>(us, ub, dt, L);
                    if (ENERGY) {                      // dual-energy switch on the new state, then the floor (G5)
                        const double eE = Lz[2 * g.lcstride], rEn = a.Uout[zo - g.cstride];
                        un = (eE > 1.0e-4 * rEn) ? eE : un;
                        if (un < g.floor_rhoe) un = g.floor_rhoe;
                    }
                    a.Uout[zo] = un;
                }
            }
            Fp[v] = Fs;
        }
    }
}

}  // namespace hydro
