// sweep_xc.cuh -- x-direction reconstruct + Riemann + flux-difference kernel, chunk-lane form.
//
// The padded x row of layout a1 is a whole number of 4-zone chunks when ng and nb_x are multiples of 4
// (136 = 34 chunks; chunks 1..32 are the valid zones, chunks 0 and 33 the x ghost zones), and the valid rows
// of a box follow one another in memory.  A lane owns ONE CHUNK: it loads its four zones of a component with
// one 256-bit load, runs the PPM stencil over them in registers (O3, O4) and needs from its two neighbour
// lanes only the values at the chunk ends -- six doubles per variable and chunk (a, slope and parabola edge at
// either end, the flux of the right neighbour's first face) against six doubles per variable and ZONE in the
// one-zone-per-lane form of sweep_x.cuh.  A warp takes 32 consecutive chunks of the flattened (row, chunk)
// sequence of a box; its first and last lane only feed their neighbours, so consecutive warps overlap by two
// chunks.  The x ghost chunks are ordinary lanes whose results are not stored: they are what separates the
// rows, so nothing is special at a row end.  Work per stored zone: 32/30 * 34/32 = 1.13 lane-zones
// (sweep_x.cuh: 32/26 * 130/128 = 1.25), and a quarter of its shuffles.
//
// Arithmetic: the same ppm_slope / ppm_edge / ppm_mono / hllc calls on the same operands as k_sweep_x, so the
// two kernels agree bit for bit in either build.  WRITES the accumulator Lacc_c = -(Fx_{i+1/2} - Fx_{i-1/2}) * dxinv.
#pragma once
#include "hydro_device.cuh"
#include "flatten.cuh"
#include "sweep_x.cuh"

namespace hydro {

#ifndef HYDRO_XC_WARPS
#define HYDRO_XC_WARPS 4
#endif
#ifndef HYDRO_XC_MINB
#define HYDRO_XC_MINB 3
#endif
#ifndef HYDRO_XC_PF
#define HYDRO_XC_PF 4
#endif
constexpr int XC_WARPS = HYDRO_XC_WARPS;
constexpr int XC_PF = HYDRO_XC_PF;  // species rows in flight per lane
constexpr int XC_LANES = 30;       // chunks stored per warp

struct d4 { double v[4]; };

__device__ __forceinline__ d4 xc_ld4(const double* p)
{
    d4 r;
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(r.v[0]), "=d"(r.v[1]), "=d"(r.v[2]), "=d"(r.v[3]) : "l"(p));
    return r;
}
__device__ __forceinline__ void xc_st4(double* p, double a, double b, double c, double d)
{
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" :: "l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// PPM over the four zones of this lane's chunk.  fL[i], fR[i]: left and right state of the face between zone
// i-1 and zone i (the LEFT face of zone i): fL[i] = aR(zone i-1), fR[i] = aL(zone i).  Valid for lanes 1..31
// (lane 31: faces 0 only as far as the right neighbour is not needed: fR[0], fL[0]).
template <bool FLAT>
__device__ __forceinline__ void ppm_chunk(const double (&a)[4], const double (&fl)[4], double (&fL)[4], double (&fR)[4])
{
    const double am = shfl_up1(a[3]), ap = shfl_dn1(a[0]);
    double s[4];
    s[0] = ppm_slope(am, a[0], a[1]);
    s[1] = ppm_slope(a[0], a[1], a[2]);
    s[2] = ppm_slope(a[1], a[2], a[3]);
    s[3] = ppm_slope(a[2], a[3], ap);
    const double sm = shfl_up1(s[3]), sp = shfl_dn1(s[0]);
    double e[5];                                       // e[i] = edge between zone i-1 and zone i
    e[0] = ppm_edge(am, a[0], sm, s[0]);               // the left neighbour forms the same value as its e[4]
    e[1] = ppm_edge(a[0], a[1], s[0], s[1]);
    e[2] = ppm_edge(a[1], a[2], s[1], s[2]);
    e[3] = ppm_edge(a[2], a[3], s[2], s[3]);
    e[4] = ppm_edge(a[3], ap, s[3], sp);
    double aR[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        ppm_mono(e[i], e[i + 1], a[i], fR[i], aR[i]);
        if (FLAT) flat_blend(fl[i], 1.0 - fl[i], a[i], fR[i], aR[i]);
    }
    fL[0] = shfl_up1(aR[3]);
    fL[1] = aR[0]; fL[2] = aR[1]; fL[3] = aR[2];
}

// grid (ceil(warps per box / XC_WARPS), gy, gz) with gy * gz >= boxes; warps per box = ceil(T / 30),
// T = nb_y * nb_z * nt_x / 4 chunks.
template <bool FLAT, bool EVOLVE>
__global__ void __launch_bounds__(XC_WARPS * 32, HYDRO_XC_MINB)
k_sweep_xc(const __grid_constant__ Geom g, const double* __restrict__ U, double* __restrict__ Lacc,
           const double* __restrict__ FL)
{
    const int lane = threadIdx.x & 31;
    const int b = blockIdx.z * gridDim.y + blockIdx.y;
    if (b >= g.nboxes) return;
    const int NC = g.nt[0] >> 2;
    const int T = g.nb[1] * g.nb[2] * NC;
    const int w = blockIdx.x * XC_WARPS + (threadIdx.x >> 5);
    if (w * XC_LANES >= T) return;                     // whole warp leaves together
    const int G0 = w * XC_LANES - 1 + lane;            // this lane's chunk in the flattened (row, chunk) sequence
    const int G = G0 < 0 ? 0 : (G0 > T - 1 ? T - 1 : G0);   // first / last lane of a box: any readable chunk
    const int r = G / NC, c = G - r * NC;              // valid row (k * nb_y + j) and chunk of the padded row
    const int k = r / g.nb[1], j = r - k * g.nb[1];
    const double* Ub = U + (long long)b * g.bstride + ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0] + 4 * c;
    const int cv = c - (g.ng >> 2);                    // chunk of the valid row
    const bool store = lane >= 1 && lane <= XC_LANES && G0 < T && cv >= 0 && cv < (g.nb[0] >> 2);
    double* Lb = Lacc + (long long)b * g.lbstride + (long long)r * g.nb[0] + 4 * cv;
    const double dxi = g.dxinv[0];

    // The species rows travel through a per-lane ring in shared memory filled by cp.async (32 bytes per lane and
    // row; a lane reads back only what it copied itself, so no barrier): completion is counted in order
    // (cp.async.wait_group), so XC_PF rows really are in flight, at no cost in registers, and the first XC_PF are
    // issued here, ahead of the whole hydro part.  Plain global loads cannot do this: ptxas puts every load of the
    // species loop on ONE scoreboard, so the first use of species n also waits for the load issued a moment ago
    // (ncu: 33-37 % of the stall samples there at any software prefetch depth 1..4).
    __shared__ __align__(16) double ring[XC_PF][2][XC_WARPS * 32][2];
    const int ns = g.nspec;
    const double* pl = Ub + 6 * g.cstride;                 // next species row to load
    auto issue = [&](int q) {
        const unsigned d0 = (unsigned)__cvta_generic_to_shared(&ring[q][0][threadIdx.x][0]);
        const unsigned d1 = (unsigned)__cvta_generic_to_shared(&ring[q][1][threadIdx.x][0]);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(d0), "l"(pl) : "memory");
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(d1), "l"(pl + 2) : "memory");
        pl += g.cstride;
    };
#pragma unroll
    for (int q = 0; q < XC_PF; ++q) {
        if (q < ns) issue(q);
        asm volatile("cp.async.commit_group;" ::: "memory");
    }

    double fl[4] = {1.0, 1.0, 1.0, 1.0};
    if (FLAT) {
        const d4 f = xc_ld4(FL + (long long)b * g.cstride + (Ub - (U + (long long)b * g.bstride)));
#pragma unroll
        for (int i = 0; i < 4; ++i) fl[i] = f.v[i];
    }
    double rinv[4], Frho[5];
    d4 re_raw;
    {
        const d4 rho = xc_ld4(Ub), mx = xc_ld4(Ub + g.cstride), my = xc_ld4(Ub + 2 * g.cstride), mz = xc_ld4(Ub + 3 * g.cstride);
        re_raw = xc_ld4(Ub + 5 * g.cstride);
        double q[5][4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            double qz[5];
            cons_to_prim(g, rho.v[i], mx.v[i], my.v[i], mz.v[i], re_raw.v[i], qz, rinv[i]);
#pragma unroll
            for (int v = 0; v < 5; ++v) q[v][i] = qz[v];
        }
        double fL[5][4], fR[5][4];
#pragma unroll
        for (int v = 0; v < 5; ++v) ppm_chunk<FLAT>(q[v], fl, fL[v], fR[v]);
        double F[5][4], uf[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {                  // the left face of zone i
            double qL[5], qR[5], Ff[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { qL[v] = fL[v][i]; qR[v] = fR[v][i]; }
            hllc<0>(g, qL, qR, Ff, uf[i]);
#pragma unroll
            for (int v = 0; v < 5; ++v) F[v][i] = Ff[v];
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double F4 = shfl_dn1(F[v][0]);       // the right face of zone 3 = the right neighbour's face 0
            if (v == 0) { Frho[0] = F[0][0]; Frho[1] = F[0][1]; Frho[2] = F[0][2]; Frho[3] = F[0][3]; Frho[4] = F4; }
            const double a0 = -(F[v][1] - F[v][0]) * dxi, a1 = -(F[v][2] - F[v][1]) * dxi;
            const double a2 = -(F[v][3] - F[v][2]) * dxi, a3 = -(F4 - F[v][3]) * dxi;
            if (store) xc_st4(Lb + v * g.lcstride, a0, a1, a2, a3);
        }
        if (EVOLVE) {     // O11: x part of div(u_face), accumulator slot nflux + 1
            const double u4 = shfl_dn1(uf[0]);
            const double D0 = (uf[1] - uf[0]) * dxi, D1 = (uf[2] - uf[1]) * dxi;
            const double D2 = (uf[3] - uf[2]) * dxi, D3 = (u4 - uf[3]) * dxi;
            if (store) xc_st4(Lb + (long long)(g.nflux + 1) * g.lcstride, D0, D1, D2, D3);
        }
    }
    // species (and, with O11, e = rho*e / rho as one more): X = raw / rho reconstructed, upwinded by the sign
    // of the face mass flux
    auto species = [&](const double (&X)[4], double* out) {
        double XL[4], XR[4];
        ppm_chunk<FLAT>(X, fl, XL, XR);
        double Fs[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) Fs[i] = Frho[i] * (Frho[i] >= 0.0 ? XL[i] : XR[i]);
        const double F4 = shfl_dn1(Fs[0]);
        const double a0 = -(Fs[1] - Fs[0]) * dxi, a1 = -(Fs[2] - Fs[1]) * dxi;
        const double a2 = -(Fs[3] - Fs[2]) * dxi, a3 = -(F4 - Fs[3]) * dxi;
        if (store) xc_st4(out, a0, a1, a2, a3);
    };
    double* ps = Lb + 5 * g.lcstride;                      // next accumulator row to store
    for (int s = 0; s < ns; s += XC_PF) {
#pragma unroll
        for (int q = 0; q < XC_PF; ++q) {
            if (s + q < ns) {                              // warp-uniform
                asm volatile("cp.async.wait_group %0;" :: "n"(XC_PF - 1) : "memory");
                const double2 lo = *reinterpret_cast<const double2*>(&ring[q][0][threadIdx.x][0]);
                const double2 hi = *reinterpret_cast<const double2*>(&ring[q][1][threadIdx.x][0]);
                double X[4];
                X[0] = lo.x * rinv[0]; X[1] = lo.y * rinv[1]; X[2] = hi.x * rinv[2]; X[3] = hi.y * rinv[3];
                if (s + q + XC_PF < ns) issue(q);
                asm volatile("cp.async.commit_group;" ::: "memory");
                species(X, ps);
                ps += g.lcstride;
            }
        }
    }
    if (EVOLVE) {
        double X[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) X[i] = re_raw.v[i] * rinv[i];
        species(X, Lb + (long long)g.nflux * g.lcstride);
    }
}

}  // namespace hydro
