// sweep_x.cuh -- x-direction reconstruct + Riemann + flux-difference kernel.
//
// x is the contiguous direction of layout a1, so a thread cannot own an x pencil without
// strided (uncoalesced) access.  Instead a warp owns 32 consecutive zones of one row and the
// PPM stencil is assembled with warp shuffles: each lane computes ITS zone's slope, edge
// and monotonised parabola exactly once and hands them to its neighbours (de-duplicated,
// unlike the one-thread-per-zone recompute of PAPER.md:51,57).  Lanes 3..28 produce zone
// updates (26 per warp); the 3-lane aprons are the PPM halo.
//
// First sweep of a stage: WRITES the accumulator  Lacc_c = -(Fx_{i+1/2} - Fx_{i-1/2}) * dxinv.
// Hydro variables and all species are handled here (species are transient per lane, so no
// face mass-flux array is needed in x).
#pragma once
#include "hydro_device.cuh"
#include "flatten.cuh"

namespace hydro {

constexpr int XW_VALID = 26;   // zones updated per warp
constexpr unsigned FULL = 0xffffffffu;
#ifndef HYDRO_XG
#define HYDRO_XG 4
#endif
constexpr int XG = HYDRO_XG;       // species per software-pipelined load group

__device__ __forceinline__ double shfl_up1(double v) { return __shfl_up_sync(FULL, v, 1); }
__device__ __forceinline__ double shfl_dn1(double v) { return __shfl_down_sync(FULL, v, 1); }

// PPM along the lanes: returns the face states of face i+1/2 (between this lane's zone
// and the next lane's): qLf = aR(i), qRf = aL(i+1).  Valid for lanes 2..28.
template <bool FLAT>
__device__ __forceinline__ void ppm_lanes(double a, double f, double omf, double& qLf, double& qRf)
{
    const double ap = shfl_dn1(a), am = shfl_up1(a);
    const double s = ppm_slope(am, a, ap);             // lanes 1..30
    const double sp = shfl_dn1(s);
    const double e = ppm_edge(a, ap, s, sp);           // e_{i+1/2}, lanes 1..29
    const double em = shfl_up1(e);                     // e_{i-1/2}, lanes 2..30
    double aL, aR;
    ppm_mono(em, e, a, aL, aR);                        // lanes 2..29
    if (FLAT) flat_blend(f, omf, a, aL, aR);           // O10 (this lane's zone)
    qLf = aR;
    qRf = shfl_dn1(aL);                                // lanes 2..28
}

template <int WARPS, bool FLAT, bool EVOLVE, bool FOLDB = false>
__global__ void __launch_bounds__(WARPS * 32)
k_sweep_x(const __grid_constant__ Geom g, const double* __restrict__ U, double* __restrict__ Lacc,
          const double* __restrict__ FL)
{
    const int lane = threadIdx.x & 31;
    const int nchunk = (g.nb[0] + XW_VALID - 1) / XW_VALID;
    // grid (nchunk * ceil(nb_y / WARPS), nb_z, boxes): the chunks of a row are consecutive blocks, the
    // warps of a block are WARPS consecutive rows; one 32-bit division per warp (a flat 64-bit warp
    // index cost ~150 instructions of division per warp, 8 % of the kernel).  FOLDB (more than 65535
    // boxes): the box index rides in blockIdx.x too, at the price of two more divisions per warp.
    int b, rb;
    if (FOLDB) {
        const int per_box = gridDim.x / g.nboxes;
        b = blockIdx.x / per_box;
        rb = blockIdx.x - b * per_box;
    } else {
        b = blockIdx.z;
        rb = blockIdx.x;
    }
    const int jb = rb / nchunk;
    const int chunk = rb - jb * nchunk;
    const int j = jb * WARPS + (threadIdx.x >> 5);
    if (j >= g.nb[1]) return;                          // whole warp leaves together
    const int k = blockIdx.y;

    const int i = chunk * XW_VALID + lane - 3;         // valid-zone index of this lane
    int ip = i + g.ng;                                 // padded index
    if (ip > g.nt[0] - 1) ip = g.nt[0] - 1;            // lanes past the halo: clamp (unused)
    const long long row = ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0];
    const double* Ub = U + (long long)b * g.bstride + row + ip;

    double fl = 1.0, omf = 0.0;
    if (FLAT) { fl = ldg(FL + (long long)b * g.cstride + row + ip); omf = 1.0 - fl; }
    double q[5], rinv;
    const double* p1 = Ub + g.cstride;
    const double* p2 = p1 + g.cstride;
    const double* p3 = p2 + g.cstride;
    const double re_raw = ldg(p3 + 2 * g.cstride);
    cons_to_prim(g, ldg(Ub), ldg(p1), ldg(p2), ldg(p3), re_raw, q, rinv);
    double qL[5], qR[5], F[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) ppm_lanes<FLAT>(q[v], fl, omf, qL[v], qR[v]);
    double uf;
    hllc<0>(g, qL, qR, F, uf);                         // face i+1/2, lanes 2..28

    const bool store = (lane >= 3) && (lane <= 2 + XW_VALID) && (i < g.nb[0]);
    double* Lb = Lacc + (long long)b * g.lbstride + ((long long)k * g.nb[1] + j) * g.nb[0] + i;
    {
        double* pa = Lb;
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            const double Fm = shfl_up1(F[c]);
            const double acc = -(F[c] - Fm) * g.dxinv[0];
            if (store) *pa = acc;
            pa += g.lcstride;
        }
        if (EVOLVE) {     // O11: x part of div(u_face), accumulator slot nflux + 1
            const double ufm = shfl_up1(uf);
            const double D = (uf - ufm) * g.dxinv[0];
            if (store) Lb[(long long)(g.nflux + 1) * g.lcstride] = D;
        }
    }
    // species: the loads of group n+1 are issued before group n is reconstructed, so the
    // global-load latency (ncu r01: 40 % of this kernel's stall samples sat on the first use of
    // a species load) is covered by XG species' worth of arithmetic.
    const double Frho = F[0];
    const double* pl = Ub + 6 * g.cstride;             // next species row to load
    double* ps = Lb + 5 * g.lcstride;                  // next accumulator row to store
    int lrem = g.nspec, rem = g.nspec;                 // species not yet loaded / not yet reconstructed
    auto load = [&](double (&x)[XG]) {
#pragma unroll
        for (int q = 0; q < XG; ++q) { x[q] = (q < lrem) ? ldg(pl) : 0.0; pl += g.cstride; }
        lrem -= XG;
    };
    auto species = [&](double raw) {
        const double X = raw * rinv;
        double XL, XR;
        ppm_lanes<FLAT>(X, fl, omf, XL, XR);
        const double Fs = Frho * (Frho >= 0.0 ? XL : XR);
        const double Fm = shfl_up1(Fs);
        const double acc = -(Fs - Fm) * g.dxinv[0];
        if (store) *ps = acc;
        ps += g.lcstride;
    };
    auto group = [&](const double (&x)[XG]) {
        if (rem >= XG) {                               // full group: no per-species guard
#pragma unroll
            for (int q = 0; q < XG; ++q) species(x[q]);
        } else {                                       // tail group (warp-uniform guard)
#pragma unroll
            for (int q = 0; q < XG - 1; ++q)
                if (q < rem) species(x[q]);
        }
        rem -= XG;
    };
    // two register sets alternate (no copies): load one while the other is reconstructed
    double xa[XG], xb[XG];
    load(xa);
    while (rem > 0) {
        load(xb);
        group(xa);
        if (rem <= 0) break;
        load(xa);
        group(xb);
    }
    // O11 (G1): e = rho*e / rho is reconstructed and upwinded like one more species; ps now points at
    // accumulator slot nflux
    if (EVOLVE) species(re_raw);
}

}  // namespace hydro
