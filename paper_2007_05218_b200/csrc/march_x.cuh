// march_x.cuh -- x-direction reconstruct + Riemann + flux-difference kernels that MARCH along x.
//
// x is the contiguous direction of layout a1.  The lane-parallel sweep of sweep_x.cuh keeps the
// accesses coalesced by giving every lane one zone of a row and assembling the PPM stencil with
// warp shuffles; it pays for that with 32/26 redundant lanes and twelve shuffles per variable
// (profiles/r01_ncu_final.md: issue-bound at 2 100 thread instructions per zone).  Here a THREAD
// owns a ROW (fixed j, k) and marches along i with the same rolling register window as the y/z
// kernels -- every slope, edge, parabola and face flux is computed once, nothing is exchanged
// between lanes.  The transposition this needs (a warp = 32 rows, consecutive zones of a row in
// one thread) is done by the TMA unit: one 5-D tensor copy per march step lands the box
// {XC = 4 zones, RJ x RK = 128 rows, NC components} of the stage state in a shared-memory ring
// slot, from which thread t reads its row's 32 bytes.  One ring step = four zones, unrolled, so
// the window rotation is register renaming and the per-step cost (mbarrier wait, CTA barrier,
// copy issue) is shared by four zones.  Results go back to global memory as one 32-byte sector
// per thread, variable and step (256-bit stores): the four accumulator values of an aligned
// group of four zones.
//
// First sweep of a stage: WRITES  Lacc_c = -(Fx_{i+1/2} - Fx_{i-1/2}) * dxinv  (as k_sweep_x).
// The hydro kernel also writes the face mass flux F_rho,x (array FX: rows of nb0 + 4 doubles,
// face f -- the low face of zone f -- in column f + 2, so that the four faces finished in a
// ring step are one aligned sector) for the species kernels to upwind with (S7).
//
// Geometry: nb0 % 4 == 0, ng even and >= 4, 128 % nb1 == 0 or nb1 % 128 == 0; other boxes (and
// the options O10 / O11) take k_sweep_x.
#pragma once
#include "hydro_device.cuh"
#include "march_ring.cuh"

#ifndef XM_MINB_H
#define XM_MINB_H 3        // CTAs per SM the hydro kernel's register allocation is capped for
#endif
#ifndef XM_MINB_S
#define XM_MINB_S 3        // same for the species kernels
#endif

namespace hydro {

constexpr int XC = 4;          // zones per ring step
constexpr int XBS = 128;       // threads = rows per CTA

struct XArgs {
    double* Lacc;          // accumulator, written
    double* FX;            // face mass flux of the x sweep: written by the hydro kernel, read by the species kernels
    int sbase;             // first species of this launch (species kernels)
};

struct XMaps {
    CUtensorMap a, b;      // {XC, RJ, RK, NCa, 1} and {XC, RJ, RK, NCb, 1} boxes of the stage state
    CUtensorMap fx;        // {XC, RJ, RK, 1} boxes of the face mass-flux array FX (species kernels)
};

__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}

// rows of the CTA: RJ consecutive j times RK consecutive k of one box
struct XRows {
    int b, j0, k0, j, k;
    bool active;
};

// row = index of the thread's row in the CTA's tile of ROWS rows (RJ = min(nb1, ROWS) along j, ROWS / RJ along k)
template <int ROWS>
__device__ __forceinline__ XRows xrows(const Geom& g, int row)
{
    XRows r;
    const int tiles = gridDim.x / g.nboxes;          // grid.x = (row tiles per box) * boxes
    r.b = blockIdx.x / tiles;
    const int tile = blockIdx.x - r.b * tiles;
    const int RJ = g.nb[1] < ROWS ? g.nb[1] : ROWS;
    const int jt = g.nb[1] / RJ;
    const int kt = tile / jt;
    r.j0 = (tile - kt * jt) * RJ;
    r.k0 = kt * (ROWS / RJ);
    const int rk = row / RJ;
    r.j = r.j0 + row - rk * RJ;
    r.k = r.k0 + rk;
    r.active = r.k < g.nb[2];
    return r;
}

__device__ __forceinline__ void st4(double* p, double x, double y, double z, double w)
{
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(x), "d"(y), "d"(z), "d"(w) : "memory");
}
__device__ __forceinline__ void ld4(const double* p, double& x, double& y, double& z, double& w)
{
    asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(x), "=d"(y), "=d"(z), "=d"(w) : "l"(p));
}

// ------------------------------------------------------------------------------------
// hydro variables.  Ring rows: rho, mx, my, mz (map a, 4 components) + rho*e (map b, 1 component).
// Ring step `it` holds zones 4(it-1) .. 4(it-1)+3, it = 0 .. nb0/4 + 1 (zones -4 .. nb0+3).  After
// zone n has been consumed the face between zones n-3 and n-2 (face index n-2) and the flux
// difference of zone n-3 are known, so step `it` finishes faces 4it-6 .. 4it-3 (columns 4(it-1) ..
// of FX) and zones 4it-7 .. 4it-4; zones 4(it-2) .. 4(it-2)+3 are stored, the last one is carried.
template <int D>
__global__ void __launch_bounds__(XBS, XM_MINB_H)
k_xmarch_hydro(const __grid_constant__ Geom g, const __grid_constant__ XArgs a, const __grid_constant__ XMaps tm)
{
    constexpr int NROW = 5;
    constexpr int SLOT = NROW * XBS * XC;            // doubles per ring slot
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* ring = reinterpret_cast<double*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)D * SLOT * 8);

    const int tid = threadIdx.x;
    const XRows r = xrows<XBS>(g, tid);
    const int nsteps = g.nb[0] / XC + 2;

    auto issue = [&](int it) {      // thread 0 only
        uint64_t* bar = &full[it % D];
        double* slot = ring + (size_t)(it % D) * SLOT;
        mbar_expect_tx(bar, (uint32_t)(SLOT * 8));
        const int c0 = XC * (it - 1) + g.ng;
        tma_load_5d(slot, &tm.a, bar, c0, r.j0 + g.ng, r.k0 + g.ng, 0, r.b);
        tma_load_5d(slot + 4 * XBS * XC, &tm.b, bar, c0, r.j0 + g.ng, r.k0 + g.ng, 5, r.b);
    };

    if (tid == 0) {
        tma_prefetch_desc(&tm.a);
        tma_prefetch_desc(&tm.b);
        for (int s = 0; s < D; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0)
        for (int it = 0; it < D && it < nsteps; ++it) issue(it);

    // row bases: group of step `it` at Lrow + XC*it (zones 4(it-2) ..), faces at Frow + XC*it (columns 4(it-1) ..)
    const long long rowid = (long long)r.k * g.nb[1] + r.j;
    double* Lrow = a.Lacc + (long long)r.b * g.lbstride + rowid * g.nb[0] - 2 * XC;
    double* Frow = a.FX + (long long)r.b * g.fbstride + rowid * (g.nb[0] + 4) - XC;
    const double dinv = g.dxinv[0];

    double a1[5], a2[5], s1[5], e1[5], aR1[5], Fp[5], carry[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { a1[v] = a2[v] = s1[v] = e1[v] = aR1[v] = Fp[v] = carry[v] = 0.0; }

    for (int it = 0; it < nsteps; ++it) {
        const double* sl = ring + (size_t)(it % D) * SLOT + tid * XC;
        mbar_wait(&full[it % D], (uint32_t)((it / D) & 1));
        double acc[5][XC], fr[XC];
#pragma unroll
        for (int q = 0; q < XC; ++q) {
            double qv[5], rinv;
            cons_to_prim(g, sl[q], sl[XBS * XC + q], sl[2 * XBS * XC + q], sl[3 * XBS * XC + q], sl[4 * XBS * XC + q], qv, rinv);
            double qL[5], qR[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                const double sn = ppm_slope(a2[v], a1[v], qv[v]);
                const double en = ppm_edge(a2[v], a1[v], s1[v], sn);
                double aL, aR;
                ppm_mono(e1[v], en, a2[v], aL, aR);
                qL[v] = aR1[v];
                qR[v] = aL;
                a2[v] = a1[v]; a1[v] = qv[v]; s1[v] = sn; e1[v] = en; aR1[v] = aR;
            }
            if (it > 0) {          // step 0 (zones -4 .. -1) only fills the window
                double F[5];
                hllc<0>(g, qL, qR, F);
                fr[q] = F[0];
#pragma unroll
                for (int c = 0; c < 5; ++c) { acc[c][q] = -(F[c] - Fp[c]) * dinv; Fp[c] = F[c]; }
            } else {
                fr[q] = 0.0;
#pragma unroll
                for (int c = 0; c < 5; ++c) acc[c][q] = 0.0;
            }
        }
        if (r.active && it >= 1) {
            st4(Frow + XC * it, fr[0], fr[1], fr[2], fr[3]);
            if (it >= 2) {
#pragma unroll
                for (int c = 0; c < 5; ++c) st4(Lrow + c * g.lcstride + XC * it, carry[c], acc[c][0], acc[c][1], acc[c][2]);
            }
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) carry[c] = acc[c][3];
        // release the slot: one CTA barrier per four zones, then thread 0 refills it
        __syncthreads();
        if (tid == 0 && it + D < nsteps) issue(it + D);
    }
}

// ------------------------------------------------------------------------------------
// Passive species.  A CTA of ROWS * SETS threads owns ROWS rows; thread set `set` (threads set*ROWS ..) marches
// NS species, sbase + set*NS .. of every row, so that the rows of rho are shared by SETS thread sets: more
// threads per row stream in flight (the L2 holds the 128-byte lines of which a step consumes 32 bytes; their
// number, not the thread count, is what has to stay small -- profiles/r02_xmarch.md).
// Ring rows: rho (map a, 1 component), F_rho,x of the four faces of the step (map fx), rho*X_k, k = sbase ..
// sbase + NS*SETS - 1 (map b): no thread loads anything from global memory.  The four reciprocal densities of a
// row and step are formed once (by different thread sets) and shared through shared memory.
template <int NS, int SETS, int ROWS, int D>
__global__ void __launch_bounds__(ROWS * SETS, XM_MINB_S)
k_xmarch_species(const __grid_constant__ Geom g, const __grid_constant__ XArgs a, const __grid_constant__ XMaps tm)
{
    // ring rows: rho, F_rho,x of the step's four faces (map fx over the FX array), then the NS * SETS species
    constexpr int NROW = 2 + NS * SETS;
    constexpr int SLOT = NROW * ROWS * XC;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* ring = reinterpret_cast<double*>(smem_raw);
    double* rinvs = ring + (size_t)D * SLOT;                     // 1 / rho of the step's zones, two buffers by step parity
    uint64_t* full = reinterpret_cast<uint64_t*>(rinvs + 2 * ROWS * XC);

    const int tid = threadIdx.x;
    const int set = tid / ROWS, row = tid - set * ROWS;
    const XRows r = xrows<ROWS>(g, row);
    const int nsteps = g.nb[0] / XC + 2;
    const int sbase = a.sbase;

    auto issue = [&](int it) {      // thread 0 only
        uint64_t* bar = &full[it % D];
        double* slot = ring + (size_t)(it % D) * SLOT;
        mbar_expect_tx(bar, (uint32_t)(SLOT * 8));
        const int c0 = XC * (it - 1) + g.ng;
        tma_load_5d(slot, &tm.a, bar, c0, r.j0 + g.ng, r.k0 + g.ng, 0, r.b);
        tma_load_4d(slot + ROWS * XC, &tm.fx, bar, XC * (it - 1), r.j0, r.k0, r.b);     // columns < 0 (step 0): zero fill
        tma_load_5d(slot + 2 * ROWS * XC, &tm.b, bar, c0, r.j0 + g.ng, r.k0 + g.ng, 6 + sbase, r.b);
    };

    if (tid == 0) {
        tma_prefetch_desc(&tm.a);
        tma_prefetch_desc(&tm.b);
        tma_prefetch_desc(&tm.fx);
        for (int s = 0; s < D; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0)
        for (int it = 0; it < D && it < nsteps; ++it) issue(it);

    const long long rowid = (long long)r.k * g.nb[1] + r.j;
    double* Lrow = a.Lacc + (long long)r.b * g.lbstride + (long long)(5 + sbase + set * NS) * g.lcstride + rowid * g.nb[0] - 2 * XC;
    const double dinv = g.dxinv[0];

    double a1[NS], a2[NS], s1[NS], e1[NS], aR1[NS], Fp[NS], carry[NS];
#pragma unroll
    for (int v = 0; v < NS; ++v) { a1[v] = a2[v] = s1[v] = e1[v] = aR1[v] = Fp[v] = carry[v] = 0.0; }

    for (int it = 0; it < nsteps; ++it) {
        const double* sl = ring + (size_t)(it % D) * SLOT + row * XC;
        const double* sx = sl + (2 + set * NS) * ROWS * XC;
        double* rs = rinvs + (it & 1) * ROWS * XC + row;          // [zone of the step][row]: conflict-free both ways
        mbar_wait(&full[it % D], (uint32_t)((it / D) & 1));
        // the reciprocal densities of the step's zones are formed once per row: thread set s takes zone s (, s + SETS ..)
        for (int q = set; q < XC; q += SETS) rs[q * ROWS] = drcp(dmax(sl[q], g.small_dens));
        __syncthreads();
        double acc[NS][XC];
#pragma unroll
        for (int q = 0; q < XC; ++q) {
            const double rinv = rs[q * ROWS];
            const double Frho = sl[ROWS * XC + q];
#pragma unroll
            for (int v = 0; v < NS; ++v) {
                const double X = sx[v * ROWS * XC + q] * rinv;
                const double sn = ppm_slope(a2[v], a1[v], X);
                const double en = ppm_edge(a2[v], a1[v], s1[v], sn);
                double aL, aR;
                ppm_mono(e1[v], en, a2[v], aL, aR);
                const double Fs = Frho * (Frho >= 0.0 ? aR1[v] : aL);
                a2[v] = a1[v]; a1[v] = X; s1[v] = sn; e1[v] = en; aR1[v] = aR;
                acc[v][q] = -(Fs - Fp[v]) * dinv;
                Fp[v] = Fs;
            }
        }
        if (r.active && it >= 2) {
#pragma unroll
            for (int v = 0; v < NS; ++v) st4(Lrow + v * g.lcstride + XC * it, carry[v], acc[v][0], acc[v][1], acc[v][2]);
        }
#pragma unroll
        for (int v = 0; v < NS; ++v) carry[v] = acc[v][3];
        __syncthreads();
        if (tid == 0 && it + D < nsteps) issue(it + D);
    }
}

}  // namespace hydro
