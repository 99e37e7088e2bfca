// march_ring.cuh -- y/z marching sweeps fed by a TMA tensor-copy ring in shared memory.
//
// Same arithmetic and accumulator protocol as sweep_yz.cuh (the generic fallback); what
// changes is how zones reach the registers.  A CTA of BS threads owns BS pencils laid out
// as R row segments of W contiguous zones (R consecutive rows of the plane normal to DIR).
// For every march step ONE thread issues one or two cp.async.bulk.tensor copies (TMA, 5-D
// tiled tensor map over a state: i, j, k, component, box; SASS UTMALDG) that bring the
// step's rows of all components the kernel reads -- a {W, R, NC} box -- into slot
// (step % D) of a D-deep ring, signalled through a "full" mbarrier with an expected-bytes
// count.  The copies run D-KEEP-1 steps ahead of the arithmetic, so the bytes in flight per
// SM are set by the ring depth and not by how many registers a thread can spare.  Slot reuse
// is ordered by one __syncthreads per step.  FINAL (z) kernels keep the last KEEP = 3 slots
// alive so that the update of zone n-3 reads its raw conserved state from shared memory.
//
// Measured dead ends (profiles/r01_experiments.md): per-row 1-D bulk copies issued by the 32
// lanes of warp 0 (ptxas serialises them through ELECT loops: ~10 instructions per copy on the
// critical warp); per-warp "empty" mbarriers instead of the CTA barrier, blocking or polled;
// L2 prefetch of the accumulator rows; the accumulator rows through the ring; unroll by 2 of
// the FINAL and species kernels (spills; only the y hydro kernel is unrolled).
#pragma once
#include <cuda.h>

#include "hydro_device.cuh"
#include "sweep_yz.cuh"
#include "ghost_reduce.cuh"
#include "flatten.cuh"

#ifndef RING_MINB
#define RING_MINB 3        // CTAs per SM the hydro kernels' register allocation is capped for
#endif
#ifndef RING_MINB_S
#define RING_MINB_S 4      // same for the species kernels (NS <= 5 species per thread fit 128 registers)
#endif

// species kernels: march steps by which the accumulator (and U0) values of a zone are fetched ahead through a
// per-thread cp.async ring in shared memory (0: plain loads at the top of the zone's own step); y sweep (not FINAL) and
// z sweep (FINAL) separately: the ring costs shared memory, which the z kernels (KEEP slots) cannot spare
#ifndef RING_LPD_Y
#define RING_LPD_Y 1
#endif
#ifndef RING_LPD_Z
#define RING_LPD_Z 0
#endif
#ifndef RING_UNROLL_S
#define RING_UNROLL_S 1     // unroll of the march loop of the species kernels
#endif
#ifndef RING_UNROLL_Z
#define RING_UNROLL_Z 1     // unroll of the march loop of the FINAL hydro kernels (2 spills at 168 registers)
#endif
#ifndef RING_UNROLL_Y
#define RING_UNROLL_Y 2     // unroll of the march loop of the non-FINAL hydro kernel
#endif

namespace hydro {

__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
// 5-D tiled tensor copy global -> shared, completion on an mbarrier (coordinates innermost first)
__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2,
                                            int c3, int c4)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}

// The two tensor maps of a launch (built on the host, hydro_api.cu): `a` and `b` view the
// stage state with boxes {W, R rows, NCa components} and {W, R rows, NCb components}.
struct RingMaps {
    CUtensorMap a, b, b2;
    CUtensorMap f;       // flattening coefficients (FLAT kernels): {W, R rows, 1} boxes of the FL array
};

// Decomposition of a CTA into R row segments of W zones.
struct RingMap {
    int W, R;        // zones per row segment, row segments per CTA
    int r, ii;       // this thread's row segment and position in it
    int i, t;        // pencil coordinates (t clamped into range)
    int x0, t0;      // first zone / first row of the CTA's tile
    bool active;     // pencil exists (t in range)
};

template <int DIR, int BS>
__device__ __forceinline__ RingMap ring_map(const Geom& g, int tid, int cta)
{
    constexpr int T = (DIR == 1) ? 2 : 1;
    RingMap m;
    m.W = g.nb[0] < BS ? g.nb[0] : BS;
    m.R = BS / m.W;
    m.r = tid / m.W;
    m.ii = tid - m.r * m.W;
    const int xchunks = g.nb[0] / m.W;       // > 1 only when W == BS (R == 1)
    const int rc0 = cta * m.R;
    m.t0 = rc0 / xchunks;
    m.x0 = (rc0 - m.t0 * xchunks) * m.W;
    int t = m.t0 + m.r;
    m.active = t < g.nb[T];
    if (!m.active) t = g.nb[T] - 1;
    m.t = t;
    m.i = m.x0 + m.ii;
    return m;
}

// padded offset of valid zone (i, t, n) for a DIR sweep (n = index along DIR)
template <int DIR>
__device__ __forceinline__ long long zone_off(const Geom& g, int i, int t, int n)
{
    const int j = (DIR == 1) ? n : t, k = (DIR == 1) ? t : n;
    return ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0] + (i + g.ng);
}

// offset of valid zone (i, t, n) in the unpadded accumulator / face arrays of a DIR sweep;
// ext = extent of the array along DIR (nb for the accumulator, nb+1 for the face array)
template <int DIR>
__device__ __forceinline__ long long flat_off(const Geom& g, int i, int t, int n, int ext)
{
    return (DIR == 1) ? ((long long)t * ext + n) * g.nb[0] + i : ((long long)n * g.nb[1] + t) * g.nb[0] + i;
}

// issue the tensor copy of march step `it` (one thread): rows of zone index n = m0-3+it
template <int DIR>
__device__ __forceinline__ void ring_issue(const Geom& g, const RingMap& m, const CUtensorMap* map, void* dst,
                                           uint64_t* bar, int n, int comp0, int box)
{
    const int j = (DIR == 1) ? n : m.t0, k = (DIR == 1) ? m.t0 : n;
    tma_load_5d(dst, map, bar, m.x0 + g.ng, j + g.ng, k + g.ng, comp0, box);
}

// x-direction ghost images of this thread's pencil (FINAL kernels with a.xends).  With boxes
// at least ng wide a zone has at most two groups of images, one per side; a group is a single
// ghost zone (box interface, periodic wrap, reflecting wall) or the run of ng consecutive ghost
// zones an outflow wall copies from its edge zone.  Group q: first image at offset d[q] from the
// zone, n[q] images, consecutive ones `step[q]` doubles apart, f[q] = reflected.
struct XEnds {
    long long d[2];
    int n[2], step[2];
    bool f[2];
    bool any;        // the zone has images
    bool single;     // exactly one image (group 0): the common case, unrolled in the kernels
};
__device__ __forceinline__ XEnds xends_setup(const Geom& g, bool on, int b, int i)
{
    // scalars only (no dynamically indexed arrays: the struct must stay in registers)
    long long d0 = 0, d1 = 0;
    int n0 = 0, n1 = 0, st0 = 1, st1 = 1;
    bool f0 = false, f1 = false;
    if (on) {
        const int bi = b % g.NB[0];
        int db, p, q = 0, ldb = 0, lp = 0;
        bool f;
        while (dim_image(g, 0, bi, i, q, db, p, f)) {
            const bool adj = q > 0 && db == ldb && (p == lp + 1 || p == lp - 1);
            if (n1 == 0 && n0 > 0 && adj && f == f0 && (n0 == 1 || p - lp == st0)) { st0 = p - lp; ++n0; }
            else if (n1 > 0 && adj && f == f1 && (n1 == 1 || p - lp == st1)) { st1 = p - lp; ++n1; }
            else if (n0 == 0) { d0 = (long long)(db - bi) * g.bstride + (p - (i + g.ng)); n0 = 1; f0 = f; }
            else if (n1 == 0) { d1 = (long long)(db - bi) * g.bstride + (p - (i + g.ng)); n1 = 1; f1 = f; }
            ldb = db; lp = p; ++q;
        }
    }
    XEnds x;
    x.d[0] = d0; x.d[1] = d1; x.n[0] = n0; x.n[1] = n1; x.step[0] = st0; x.step[1] = st1; x.f[0] = f0; x.f[1] = f1;
    x.any = (n0 | n1) != 0;
    x.single = n0 == 1 && n1 == 0;
    return x;
}

// ------------------------------------------------------------------------------------
// hydro variables.  Ring rows: non-FINAL  rho, mx, my, mz (map a, 4 components) + rho*e (map b,
// 1 component); FINAL  rho, mx, my, mz, rho*E, rho*e (map a, 6 components).
template <int DIR, bool FINAL, int STAGE, int BS, int D, bool FLAT, bool EVOLVE>
__global__ void __launch_bounds__(BS, RING_MINB)
k_march_hydro(const __grid_constant__ Geom g, const __grid_constant__ SweepArgs a, const __grid_constant__ RingMaps tm)
{
    constexpr int ROW_F = FINAL ? 6 : 5;      // ring row of the flattening coefficient (FLAT)
    constexpr int NROW = ROW_F + (FLAT ? 1 : 0);
    constexpr int KEEP = FINAL ? 3 : 0;
    constexpr int ROW_E = FINAL ? 5 : 4;       // ring row of rho*e
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* ring = reinterpret_cast<double*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)D * NROW * BS * 8);

    const int tid = threadIdx.x;
    const int tiles = gridDim.x / g.nboxes;      // grid.x = (CTAs per box) * boxes
    const int b = blockIdx.x / tiles;
    const RingMap m = ring_map<DIR, BS>(g, tid, blockIdx.x - b * tiles);
    const int m0 = blockIdx.y * a.seglen;
    const int m1 = min(m0 + a.seglen, g.nb[DIR]);
    const int nsteps = m1 - m0 + 6;
    const long long mstride = (DIR == 1) ? g.nt[0] : (long long)g.nt[0] * g.nt[1];
    const long long lmstride = (DIR == 1) ? g.nb[0] : (long long)g.nb[0] * g.nb[1];

    auto issue = [&](int it) {      // thread 0 only
        uint64_t* bar = &full[it % D];
        double* slot = ring + (size_t)(it % D) * NROW * BS;
        mbar_expect_tx(bar, (uint32_t)(NROW * BS * 8));
        if (FINAL) ring_issue<DIR>(g, m, &tm.a, slot, bar, m0 - 3 + it, 0, b);
        else {
            ring_issue<DIR>(g, m, &tm.a, slot, bar, m0 - 3 + it, 0, b);
            ring_issue<DIR>(g, m, &tm.b, slot + 4 * BS, bar, m0 - 3 + it, 5, b);
        }
        if (FLAT) ring_issue<DIR>(g, m, &tm.f, slot + ROW_F * BS, bar, m0 - 3 + it, 0, b);
    };

    if (tid == 0) {
        tma_prefetch_desc(&tm.a);
        if (!FINAL) tma_prefetch_desc(&tm.b);
        if (FLAT) tma_prefetch_desc(&tm.f);
        for (int s = 0; s < D; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0)
        for (int it = 0; it < D && it < nsteps; ++it) issue(it);

    // running offsets of zone z = m0-6+it (the zone updated at step it) and of face n-2
    long long lz = (long long)b * g.lbstride + flat_off<DIR>(g, m.i, m.t, m0 - 6, g.nb[DIR]);
    long long fz = (long long)b * g.fbstride + flat_off<DIR>(g, m.i, m.t, m0 - 5, g.nb[DIR] + 1);
    long long zo = (long long)b * g.bstride + zone_off<DIR>(g, m.i, m.t, m0 - 6);
    const double dinv = g.dxinv[DIR];
    const double dt = a.dt_dev ? *a.dt_dev : a.dt;

    double a1[5], a2[5], s1[5], e1[5], aR1[5], Fp[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { a1[v] = a2[v] = s1[v] = e1[v] = aR1[v] = Fp[v] = 0.0; }
    const XEnds xe = xends_setup(g, FINAL && a.xends && m.active, b, m.i);
    double f1 = 1.0, f2 = 1.0;               // O10 coefficients of zones n-1, n-2 (FLAT)
    double ufp = 0.0;                        // O11 face velocity of the previous face (EVOLVE)
    constexpr int NOUT = EVOLVE ? 5 : 6;     // with O11 rho*e is not written here
    constexpr bool CFL = FINAL && STAGE == 1;
    const bool cfl_on = CFL && a.dt_next != nullptr;
    double tmax = 0.0;
    bool tbad = false;

    // two steps per trip in the y kernel: the rolling-window rotation becomes register renaming
    // (8.1 -> 7.6 ms per step at 512^3); the FINAL kernels spill when unrolled and stay at 1
    constexpr int UNROLL = FINAL ? RING_UNROLL_Z : RING_UNROLL_Y;
#pragma unroll UNROLL
    for (int it = 0; it < nsteps; ++it, lz += lmstride, fz += lmstride, zo += mstride) {
        const bool upd = (it >= 6);
        // early, independent global loads for the update of zone z
        double lacc[5], ubase[5], ldiv = 0.0;
        if (upd) {
#pragma unroll
            for (int c = 0; c < 5; ++c) lacc[c] = a.Lacc[lz + c * g.lcstride];
            if (EVOLVE) ldiv = a.Lacc[lz + (long long)(g.nflux + 1) * g.lcstride];   // O11: div(u_face) so far
            if (FINAL && STAGE == 1) {
#pragma unroll
                for (int c = 0; c < 5; ++c) ubase[c] = a.Ubase[zo + c * g.cstride];
            }
        }
        const double* slot = ring + (size_t)(it % D) * NROW * BS;
        mbar_wait(&full[it % D], (uint32_t)((it / D) & 1));
        double q[5], rinv;
        cons_to_prim(g, slot[tid], slot[BS + tid], slot[2 * BS + tid], slot[3 * BS + tid], slot[ROW_E * BS + tid], q, rinv);
        const double fn = FLAT ? slot[ROW_F * BS + tid] : 1.0;   // O10 coefficient of the new zone
        const double omf2 = 1.0 - f2;
        double qL[5], qR[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double sn = ppm_slope(a2[v], a1[v], q[v]);
            const double en = ppm_edge(a2[v], a1[v], s1[v], sn);
            double aL, aR;
            ppm_mono(e1[v], en, a2[v], aL, aR);
            if (FLAT) flat_blend(f2, omf2, a2[v], aL, aR);
            qL[v] = aR1[v];
            qR[v] = aL;
            a2[v] = a1[v]; a1[v] = q[v]; s1[v] = sn; e1[v] = en; aR1[v] = aR;
        }
        f2 = f1; f1 = fn;
        if (it >= 5) {
            double F[5];
            double uf;
            hllc<DIR>(g, qL, qR, F, uf);
            double out[6];
            const double dsum = EVOLVE ? ldiv + (uf - ufp) * dinv : 0.0;
            double eE = 0.0;
            if (upd) {
#pragma unroll
                for (int c = 0; c < 5; ++c) out[c] = lacc[c] - (F[c] - Fp[c]) * dinv;
                if (FINAL) {
                    const double* sz = ring + (size_t)((it - 3) % D) * NROW * BS;   // raw state of zone z
                    double us[5];
                    us[0] = sz[tid]; us[1] = sz[BS + tid]; us[2] = sz[2 * BS + tid]; us[3] = sz[3 * BS + tid];
                    us[4] = sz[4 * BS + tid];
                    if (g.has_grav) {
                        out[1] += us[0] * g.grav[0];
                        out[2] += us[0] * g.grav[1];
                        out[3] += us[0] * g.grav[2];
                        out[4] += us[1] * g.grav[0] + us[2] * g.grav[1] + us[3] * g.grav[2];
                    }
#pragma unroll
                    for (int c = 0; c < 5; ++c) out[c] = rk_combine<STAGE>(us[c], (STAGE == 1) ? ubase[c] : 0.0, dt, out[c]);
                    const double K = ddiv(HALF * (out[1] * out[1] + out[2] * out[2] + out[3] * out[3]), out[0]);
                    double re = out[4] - K;
                    eE = re;                    // O11: rho*E - K before the floor, for the dual-energy switch
                    if (EVOLVE && fabs(re - 1.0e-4 * out[4]) <= 1e-12 * fabs(out[4])) {
                        // within rounding of the switch threshold: form K exactly as the definition does, so
                        // that the yes/no decision taken by the energy kernel is the definition's
                        const double m2 = __dadd_rn(__dadd_rn(__dmul_rn(out[1], out[1]), __dmul_rn(out[2], out[2])), __dmul_rn(out[3], out[3]));
                        eE = __dsub_rn(out[4], __ddiv_rn(__dmul_rn(HALF, m2), out[0]));
                    }
                    if (re < g.floor_rhoe) re = g.floor_rhoe;
                    out[5] = re;
                    if (CFL && cfl_on && m.active) {       // O8 on the zone just formed (same code as k_estimate_dt)
                        double qn[5], rn;
                        cons_to_prim(g, out[0], out[1], out[2], out[3], out[5], qn, rn);
                        const double cs = sqrt(g.gamma * qn[4] * rn);
                        const double t = (fabs(qn[1]) + cs) * g.dxinv[0] + (fabs(qn[2]) + cs) * g.dxinv[1] + (fabs(qn[3]) + cs) * g.dxinv[2];
                        if (!(t == t)) tbad = true;
                        if (t > tmax) tmax = t;
                    }
                }
            }
            if (m.active) {          // all stores of the step under one predicate
                a.Frho[fz] = F[0];
                if (upd) {
                    if (!FINAL) {
#pragma unroll
                        for (int c = 0; c < 5; ++c) a.Lacc[lz + c * g.lcstride] = out[c];
                        if (EVOLVE) a.Lacc[lz + (long long)(g.nflux + 1) * g.lcstride] = dsum;
                    } else {
                        if (EVOLVE) {   // rho*e is written by the energy kernel (k_march_species<ENERGY>)
                            a.Lacc[lz + (long long)(g.nflux + 1) * g.lcstride] = dsum;
                            a.Lacc[lz + (long long)(g.nflux + 2) * g.lcstride] = eE;
                        }
#pragma unroll
                        for (int c = 0; c < NOUT; ++c) a.Uout[zo + c * g.cstride] = out[c];
                        if (xe.single) {
                            const long long zi = zo + xe.d[0];
#pragma unroll
                            for (int c = 0; c < NOUT; ++c) a.Uout[zi + c * g.cstride] = (c == 1 && xe.f[0]) ? -out[c] : out[c];
                        } else if (xe.any) {
#pragma unroll 1
                            for (int qr = 0; qr < xe.n[0] + xe.n[1]; ++qr) {
                                const int qq = qr < xe.n[0] ? 0 : 1, r = qr - (qq ? xe.n[0] : 0);
                                const long long zi = zo + (qq ? xe.d[1] : xe.d[0]) + r * (qq ? xe.step[1] : xe.step[0]);
                                const bool fq = qq ? xe.f[1] : xe.f[0];
#pragma unroll
                                for (int c = 0; c < NOUT; ++c) a.Uout[zi + c * g.cstride] = (c == 1 && fq) ? -out[c] : out[c];
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) Fp[c] = F[c];
            ufp = uf;
        }
        // release slot (it-KEEP): one CTA barrier per step, then thread 0 refills it
        __syncthreads();
        if (tid == 0 && it >= KEEP && it - KEEP + D < nsteps) issue(it - KEEP + D);
    }
    if (CFL && cfl_on)
        cfl_reduce_finish(g, tbad, tmax, a.red, a.dt_next, reinterpret_cast<unsigned long long*>(ring));
}

// ------------------------------------------------------------------------------------
// NS passive species per thread.  Ring rows: rho (map a, 1 component) + rho*X_k, k = sbase..
// sbase+NS-1 (map b, NS components).
// ENERGY (NS = 1, FINAL, launched with sbase = -1): the one "species" is e = rho*e / rho of O11; the update adds
// -p div(u_face) and ends with the dual-energy switch (readings G3-G5).
// The march of one CTA: bx / gx = this CTA's index and the CTA count of ITS species group along grid.x
// ((CTAs per box) * boxes), sbase = first species of the group, mapb = tensor map with NS-component boxes.
template <int DIR, bool FINAL, int STAGE, int NS, int BS, int D, bool FLAT, bool ENERGY>
__device__ __forceinline__ void march_species_body(const Geom& g, const SweepArgs& a, const CUtensorMap* mapa,
                                                   const CUtensorMap* mapb, const CUtensorMap* mapf, int bx, int gx, int sbase)
{
    constexpr int ROW_F = 1 + NS;             // ring row of the flattening coefficient (FLAT)
    constexpr int NROW = ROW_F + (FLAT ? 1 : 0);
    constexpr int KEEP = FINAL ? 3 : 0;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* ring = reinterpret_cast<double*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)D * NROW * BS * 8);
    // accumulator / U0 values of the zone updated LPD steps from now, one double per thread and species: each thread
    // copies and reads back its own values only (cp.async, completion in order: no barrier, no registers held)
    constexpr int LPD = FINAL ? RING_LPD_Z : RING_LPD_Y, LSL = LPD + 1;
    constexpr bool UB = FINAL && STAGE == 1;
    constexpr int NL = NS * (UB ? 2 : 1);
    double* lring = reinterpret_cast<double*>(smem_raw + (size_t)D * NROW * BS * 8 + (size_t)D * 8);

    const int tid = threadIdx.x;
    const int tiles = gx / g.nboxes;
    const int b = bx / tiles;
    const RingMap m = ring_map<DIR, BS>(g, tid, bx - b * tiles);
    const int m0 = blockIdx.y * a.seglen;
    const int m1 = min(m0 + a.seglen, g.nb[DIR]);
    const int nsteps = m1 - m0 + 6;
    const long long mstride = (DIR == 1) ? g.nt[0] : (long long)g.nt[0] * g.nt[1];
    const long long lmstride = (DIR == 1) ? g.nb[0] : (long long)g.nb[0] * g.nb[1];

    auto issue = [&](int it) {      // thread 0 only
        uint64_t* bar = &full[it % D];
        double* slot = ring + (size_t)(it % D) * NROW * BS;
        mbar_expect_tx(bar, (uint32_t)(NROW * BS * 8));
        ring_issue<DIR>(g, m, mapa, slot, bar, m0 - 3 + it, 0, b);
        ring_issue<DIR>(g, m, mapb, slot + BS, bar, m0 - 3 + it, 6 + sbase, b);
        if (FLAT) ring_issue<DIR>(g, m, mapf, slot + ROW_F * BS, bar, m0 - 3 + it, 0, b);
    };

    if (tid == 0) {
        tma_prefetch_desc(mapa);
        tma_prefetch_desc(mapb);
        if (FLAT) tma_prefetch_desc(mapf);
        for (int s = 0; s < D; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0)
        for (int it = 0; it < D && it < nsteps; ++it) issue(it);

    // running offsets of zone z = m0-6+it (updated at step it) and of face n-2 = m0-5+it
    long long lz = (long long)b * g.lbstride + (long long)(5 + sbase + a.lacc_shift) * g.lcstride + flat_off<DIR>(g, m.i, m.t, m0 - 6, g.nb[DIR]);
    long long fz = (long long)b * g.fbstride + flat_off<DIR>(g, m.i, m.t, m0 - 5, g.nb[DIR] + 1);
    long long zo = (long long)b * g.bstride + (long long)(6 + sbase) * g.cstride + zone_off<DIR>(g, m.i, m.t, m0 - 6);
    const double dinv = g.dxinv[DIR];
    const double dt = a.dt_dev ? *a.dt_dev : a.dt;

    double a1[NS], a2[NS], s1[NS], e1[NS], aR1[NS], Fp[NS];
#pragma unroll
    for (int v = 0; v < NS; ++v) { a1[v] = a2[v] = s1[v] = e1[v] = aR1[v] = Fp[v] = 0.0; }
    const XEnds xe = xends_setup(g, FINAL && a.xends && m.active, b, m.i);
    // F_rho of the face handled at step `it` is loaded one step ahead (ncu r01: 23-25 % of this
    // kernel's stall samples sat on its first use when it was loaded at the top of its own step)
    double Fnext = 0.0;
    double f1 = 1.0, f2 = 1.0;               // O10 coefficients of zones n-1, n-2 (FLAT)

    constexpr int UNROLL_S = RING_UNROLL_S;
#pragma unroll UNROLL_S
    for (int it = 0; it < nsteps; ++it, lz += lmstride, fz += lmstride, zo += mstride) {
        const bool upd = (it >= 6);
        const double Frho = Fnext;
        if (it >= 4 && it + 1 < nsteps) Fnext = ldg(a.Frho + fz + lmstride);
        double lacc[NS], ubase[NS], ldiv = 0.0, eE = 0.0, rEn = 0.0;
        if (LPD > 0) {
            const int itp = it + LPD;
            if (itp >= 6 && itp < nsteps) {
                const uint32_t dst = smem_u32(lring + (size_t)(itp % LSL) * NL * BS + tid);
#pragma unroll
                for (int v = 0; v < NS; ++v)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + (uint32_t)(v * BS * 8)),
                                 "l"(a.Lacc + lz + LPD * lmstride + v * g.lcstride) : "memory");
                if (UB) {
#pragma unroll
                    for (int v = 0; v < NS; ++v)
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + (uint32_t)((NS + v) * BS * 8)),
                                     "l"(a.Ubase + zo + LPD * mstride + v * g.cstride) : "memory");
                }
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
        if (upd) {
            if (LPD == 0) {
#pragma unroll
                for (int v = 0; v < NS; ++v) lacc[v] = a.Lacc[lz + v * g.lcstride];
                if (UB) {
#pragma unroll
                    for (int v = 0; v < NS; ++v) ubase[v] = a.Ubase[zo + v * g.cstride];
                }
            }
            if (ENERGY) {     // div(u_face) and rho*E - K left by the z hydro kernel, and the new rho*E
                ldiv = a.Lacc[lz + g.lcstride];
                eE = a.Lacc[lz + 2 * g.lcstride];
                rEn = a.Uout[zo - g.cstride];
            }
        }
        const double* slot = ring + (size_t)(it % D) * NROW * BS;
        mbar_wait(&full[it % D], (uint32_t)((it / D) & 1));
        const double rinv = drcp(dmax(slot[tid], g.small_dens));
        const double fn = FLAT ? slot[ROW_F * BS + tid] : 1.0;
        const double omf2 = 1.0 - f2;
        // pass 1: reconstruction and face fluxes of all NS species (no global operand)
        double out[NS];
#pragma unroll
        for (int v = 0; v < NS; ++v) {
            const double X = slot[(1 + v) * BS + tid] * rinv;
            const double sn = ppm_slope(a2[v], a1[v], X);
            const double en = ppm_edge(a2[v], a1[v], s1[v], sn);
            double aL, aR;
            ppm_mono(e1[v], en, a2[v], aL, aR);
            if (FLAT) flat_blend(f2, omf2, a2[v], aL, aR);
            const double Fs = Frho * (Frho >= 0.0 ? aR1[v] : aL);
            a2[v] = a1[v]; a1[v] = X; s1[v] = sn; e1[v] = en; aR1[v] = aR;
            out[v] = Fs - Fp[v];
            Fp[v] = Fs;
        }
        f2 = f1; f1 = fn;
        // pass 2: accumulator / stage update (first use of this step's global loads)
        if (upd) {
            if (LPD > 0) {
                asm volatile("cp.async.wait_group %0;" ::"n"(LPD) : "memory");
                const double* src = lring + (size_t)(it % LSL) * NL * BS + tid;
#pragma unroll
                for (int v = 0; v < NS; ++v) lacc[v] = src[v * BS];
                if (UB) {
#pragma unroll
                    for (int v = 0; v < NS; ++v) ubase[v] = src[(NS + v) * BS];
                }
            }
#pragma unroll
            for (int v = 0; v < NS; ++v) out[v] = lacc[v] - out[v] * dinv;
            if (FINAL) {
                const double* sz = ring + (size_t)((it + D - 3) % D) * NROW * BS;   // zone z's slot
#pragma unroll
                for (int v = 0; v < NS; ++v) {
                    const double us = sz[(1 + v) * BS + tid];
                    if (ENERGY) out[v] = out[v] - dmax(g.gm1 * us, g.small_pres) * ldiv;
                    out[v] = rk_combine<STAGE>(us, (STAGE == 1) ? ubase[v] : 0.0, dt, out[v]);
                    if (ENERGY) {                      // dual-energy switch, then the floor (as O7)
                        double re = (eE > 1.0e-4 * rEn) ? eE : out[v];
                        if (re < g.floor_rhoe) re = g.floor_rhoe;
                        out[v] = re;
                    }
                }
            }
            if (m.active) {          // all stores of the step under one predicate
                if (!FINAL) {
#pragma unroll
                    for (int v = 0; v < NS; ++v) a.Lacc[lz + v * g.lcstride] = out[v];
                } else {
#pragma unroll
                    for (int v = 0; v < NS; ++v) a.Uout[zo + v * g.cstride] = out[v];
                    if (xe.single) {     // x ghost images of the zone (only the threads at the row ends)
                        const long long zi = zo + xe.d[0];
#pragma unroll
                        for (int v = 0; v < NS; ++v) a.Uout[zi + v * g.cstride] = out[v];
                    } else if (xe.any) {
#pragma unroll 1
                        for (int qr = 0; qr < xe.n[0] + xe.n[1]; ++qr) {
                            const int qq = qr < xe.n[0] ? 0 : 1, r = qr - (qq ? xe.n[0] : 0);
                            const long long zi = zo + (qq ? xe.d[1] : xe.d[0]) + r * (qq ? xe.step[1] : xe.step[0]);
#pragma unroll
                            for (int v = 0; v < NS; ++v) a.Uout[zi + v * g.cstride] = out[v];
                        }
                    }
                }
            }
        }
        __syncthreads();
        if (tid == 0 && it >= KEEP && it - KEEP + D < nsteps) issue(it - KEEP + D);
    }
}

// One species group per launch (also the O11 energy launch: ENERGY, NS = 1, sbase = -1).
template <int DIR, bool FINAL, int STAGE, int NS, int BS, int D, bool FLAT, bool ENERGY = false>
__global__ void __launch_bounds__(BS, RING_MINB_S)
k_march_species(const __grid_constant__ Geom g, const __grid_constant__ SweepArgs a, const __grid_constant__ RingMaps tm)
{
    march_species_body<DIR, FINAL, STAGE, NS, BS, D, FLAT, ENERGY>(g, a, &tm.a, &tm.b, &tm.f, blockIdx.x, gridDim.x, a.sbase);
}

// ALL species groups in one launch: CTA blockIdx.x works on group blockIdx.x % ngroups of tile blockIdx.x / ngroups,
// so that the CTAs which read the same rho and F_rho rows are dispatched together and march in step -- the rows one
// of them pulls from HBM are L2 hits for its siblings (the groups re-read rho and F_rho: 16 B per zone and group).
// The first a.n_hi groups carry NSA species, the others NSA - 1 (maps tm.b / tm.b2); CTA-uniform branch.
template <int DIR, bool FINAL, int STAGE, int NSA, int BS, int D, bool FLAT>
__global__ void __launch_bounds__(BS, RING_MINB_S)
k_march_species_groups(const __grid_constant__ Geom g, const __grid_constant__ SweepArgs a, const __grid_constant__ RingMaps tm)
{
    const int group = blockIdx.x % a.ngroups, bx = blockIdx.x / a.ngroups, gx = gridDim.x / a.ngroups;
    if (group < a.n_hi) {
        march_species_body<DIR, FINAL, STAGE, NSA, BS, D, FLAT, false>(g, a, &tm.a, &tm.b, &tm.f, bx, gx, group * NSA);
    } else {
        constexpr int NSB = NSA > 1 ? NSA - 1 : 1;
        march_species_body<DIR, FINAL, STAGE, NSB, BS, D, FLAT, false>(g, a, &tm.a, &tm.b2, &tm.f, bx, gx,
                                                                      a.n_hi * NSA + (group - a.n_hi) * NSB);
    }
}

}  // namespace hydro
