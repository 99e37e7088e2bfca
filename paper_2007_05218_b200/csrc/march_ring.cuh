// march_ring.cuh -- y/z marching sweeps fed by a TMA bulk-copy ring in shared memory.
//
// Same arithmetic and accumulator protocol as sweep_yz.cuh (the generic fallback); what
// changes is how zones reach the registers.  A CTA of BS threads owns BS pencils laid out
// as R row segments of W contiguous zones.  For every march step one elected set of
// threads issues cp.async.bulk (TMA, 1-D) copies of the step's rows -- W*8 contiguous
// bytes per component per row segment -- into slot (step % D) of a D-deep ring, signalled
// through a "full" mbarrier with an expected-bytes count.  The copies run D-KEEP-1 steps
// ahead of the arithmetic, so the bytes in flight per SM are set by the ring depth and not
// by how many registers a thread can spare: that is what the y/z sweeps lacked (ncu: 17 %
// occupancy, fp64 pipe 19-30 %, DRAM 25-35 % of peak with plain per-thread loads).
// Slot reuse is ordered by one __syncthreads per step (RING_CTASYNC=1, measured faster than
// per-warp "empty" mbarriers, RING_CTASYNC=0).  The accumulator / face-flux / U0 rows that the
// update needs are read with plain loads issued at the top of the step; pulling them into L2
// ahead of time with cp.async.bulk.prefetch.L2 (RING_PF=1) measured slower and is off.
// FINAL (z) kernels keep the last KEEP=3 slots alive so that the update of zone n-3 reads
// its raw conserved state from shared memory instead of going back to L2.
#pragma once
#include "hydro_device.cuh"
#include "sweep_yz.cuh"
#include "ghost_reduce.cuh"

// tuning switches (overridable with -D for experiments)
#ifndef RING_UNROLL
#define RING_UNROLL 1      // unroll factor of the march loop
#endif
#ifndef RING_PF
#define RING_PF 0          // cp.async.bulk.prefetch.L2 of the accumulator / face-flux / U0 rows
#endif
#ifndef RING_CTASYNC
#define RING_CTASYNC 1     // 1: __syncthreads per step instead of per-warp slot release
#endif
#ifndef RING_MINB
#define RING_MINB 3        // CTAs per SM the hydro kernels' register allocation is capped for
#endif
#ifndef RING_MINB_S
#define RING_MINB_S 4      // same for the species kernels (NS <= 5 species per thread fit 128 registers)
#endif
#define RING_STR2(x) #x
#define RING_STR(x) RING_STR2(x)

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
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
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

// non-blocking phase test by lane 0, broadcast to the warp
__device__ __forceinline__ bool mbar_test_warp(uint64_t* bar, uint32_t parity)
{
    uint32_t ok = 0;
    if ((threadIdx.x & 31) == 0) {
        asm volatile(
            "{\n"
            ".reg .pred P1;\n"
            "mbarrier.test_wait.parity.shared::cta.b64 P1, [%1], %2;\n"
            "selp.u32 %0, 1, 0, P1;\n"
            "}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    }
    return __shfl_sync(0xffffffffu, ok, 0) != 0;
}

// Decomposition of a CTA into R row segments of W zones.
struct RingMap {
    int W, R;        // zones per row segment, row segments per CTA
    int r, ii;       // this thread's row segment and position in it
    int i, t;        // pencil coordinates (t clamped into range)
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
    const int xchunks = g.nb[0] / m.W;
    const int rc = cta * m.R + m.r;
    int t = rc / xchunks;
    const int xc = rc - t * xchunks;
    m.active = t < g.nb[T];
    if (!m.active) t = g.nb[T] - 1;
    m.t = t;
    m.i = xc * m.W + m.ii;
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
    XEnds x;
    x.d[0] = x.d[1] = 0; x.n[0] = x.n[1] = 0; x.step[0] = x.step[1] = 1; x.f[0] = x.f[1] = false;
    if (on) {
        const int bi = b % g.NB[0];
        int db, p, q = 0, grp = -1, ldb = 0, lp = 0;
        bool f;
        while (dim_image(g, 0, bi, i, q, db, p, f)) {
            const bool run = grp >= 0 && db == ldb && f == x.f[grp] && (p == lp + 1 || p == lp - 1) &&
                             (x.n[grp] == 1 || p - lp == x.step[grp]);
            if (run) { x.step[grp] = p - lp; ++x.n[grp]; }
            else if (grp < 1) {
                ++grp;
                x.d[grp] = (long long)(db - bi) * g.bstride + (p - (i + g.ng));
                x.n[grp] = 1; x.f[grp] = f;
            }
            ldb = db; lp = p; ++q;
        }
    }
    x.any = (x.n[0] | x.n[1]) != 0;
    x.single = x.n[0] == 1 && x.n[1] == 0;
    return x;
}

// Copy / prefetch descriptors held by the lanes of warp 0 (at most 2 each): pointer for
// march step 0 and the destination offset inside a ring slot (copies), or the first step at
// which the row exists (prefetches).  Per step a lane only adds step*stride.
struct RingDesc {          // lives in shared memory: entry q*32 + lane
    const double* src[64];
    const double* pf[64];
    long long pf_stride[64];
    int dst[64];
    int pf_first[64];
};

// ------------------------------------------------------------------------------------
template <int DIR, bool FINAL, int STAGE, int BS, int D>
__global__ void __launch_bounds__(BS, RING_MINB)
k_march_hydro(const __grid_constant__ Geom g, const __grid_constant__ SweepArgs a)
{
    constexpr int T = (DIR == 1) ? 2 : 1;
    constexpr int NROW = FINAL ? 6 : 5;
    constexpr int KEEP = FINAL ? 3 : 0;
    constexpr int NPF = 5 + ((FINAL && STAGE == 1) ? 5 : 0);        // Lacc rows (+ U0 rows)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* ring = reinterpret_cast<double*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)D * NROW * BS * 8);
    uint64_t* empty = full + D;

    const int tid = threadIdx.x;
    const RingMap m = ring_map<DIR, BS>(g, tid, blockIdx.x);
    const int b = blockIdx.z;
    const int m0 = blockIdx.y * a.seglen;
    const int m1 = min(m0 + a.seglen, g.nb[DIR]);
    const int nsteps = m1 - m0 + 6;
    const double* Ub = a.Us + (long long)b * g.bstride;
    const long long mstride = (DIR == 1) ? g.nt[0] : (long long)g.nt[0] * g.nt[1];
    const long long lmstride = (DIR == 1) ? g.nb[0] : (long long)g.nb[0] * g.nb[1];
    double* Lbox = a.Lacc + (long long)b * g.lbstride;

    RingDesc& ds = *reinterpret_cast<RingDesc*>(empty + D);
    if (tid < 32) {
        const int xchunks = g.nb[0] / m.W;
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const int cpy = tid + 32 * q;
            ds.src[q * 32 + tid] = nullptr; ds.dst[q * 32 + tid] = 0; ds.pf[q * 32 + tid] = nullptr; ds.pf_first[q * 32 + tid] = 0; ds.pf_stride[q * 32 + tid] = 0;
            const int row = cpy / m.R, r = cpy - row * m.R;
            const int rc = blockIdx.x * m.R + r;
            int t = rc / xchunks;
            const int x0 = (rc - t * xchunks) * m.W;
            if (t >= g.nb[T]) t = g.nb[T] - 1;
            if (row < NROW) {
                const int comp = row < 4 ? row : (row == 4 ? 5 : 4);   // rho, mx, my, mz, rho*e, (rho*E)
                ds.src[q * 32 + tid] = Ub + (long long)comp * g.cstride + zone_off<DIR>(g, x0, t, m0 - 3);
                ds.dst[q * 32 + tid] = row * BS + r * m.W;
            }
            if (row < NPF) {     // row of zone n-3 = m0-6+it: exists from step 6 on
                ds.pf_first[q * 32 + tid] = 6;
                if (row < 5) {
                    ds.pf[q * 32 + tid] = Lbox + (long long)row * g.lcstride + flat_off<DIR>(g, x0, t, m0 - 6, g.nb[DIR]);
                    ds.pf_stride[q * 32 + tid] = lmstride;
                } else {
                    ds.pf[q * 32 + tid] = a.Ubase + (long long)b * g.bstride + (long long)(row - 5) * g.cstride +
                               zone_off<DIR>(g, x0, t, m0 - 6);
                    ds.pf_stride[q * 32 + tid] = mstride;
                }
            }
        }
    }
    auto issue = [&](int it) {      // warp 0 only
        uint64_t* bar = &full[it % D];
        double* slot = ring + (size_t)(it % D) * NROW * BS;
        if (tid == 0) mbar_expect_tx(bar, (uint32_t)(NROW * BS * 8));
        __syncwarp();
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const double* src = ds.src[q * 32 + tid];
            if (src) bulk_g2s(slot + ds.dst[q * 32 + tid], src + it * mstride, (uint32_t)(m.W * 8), bar);
#if RING_PF
            const double* pf = ds.pf[q * 32 + tid];
            if (pf && it >= ds.pf_first[q * 32 + tid])
                bulk_prefetch_l2(pf + it * ds.pf_stride[q * 32 + tid], (uint32_t)(m.W * 8));
#endif
        }
    };

    if (tid == 0) {
        for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], BS / 32); }
        mbar_fence_init();
    }
    __syncthreads();
    if (tid < 32)
        for (int it = 0; it < D && it < nsteps; ++it) issue(it);

    double* Lb = Lbox + flat_off<DIR>(g, m.i, m.t, 0, g.nb[DIR]);
    double* Fb = a.Frho + (long long)b * g.fbstride + flat_off<DIR>(g, m.i, m.t, 0, g.nb[DIR] + 1);
    const long long zo0 = (long long)b * g.bstride + zone_off<DIR>(g, m.i, m.t, 0);
    const double dinv = g.dxinv[DIR];
    const double dt = a.dt_dev ? *a.dt_dev : a.dt;

    double a1[5], a2[5], s1[5], e1[5], aR1[5], Fp[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { a1[v] = a2[v] = s1[v] = e1[v] = aR1[v] = Fp[v] = 0.0; }
    const XEnds xe = xends_setup(g, FINAL && a.xends && m.active, b, m.i);

    int next_issue = D;          // first step whose copies have not been issued (warp 0)
_Pragma(RING_STR(unroll RING_UNROLL))
    for (int it = 0; it < nsteps; ++it) {
        const int n = m0 - 3 + it;
        const int z = n - 3;
        const bool upd = (it >= 6);
        // early, independent global loads for the update of zone z (L2 hits: prefetched by warp 0)
        double lacc[5], ubase[5];
        if (upd) {
#pragma unroll
            for (int c = 0; c < 5; ++c) lacc[c] = Lb[z * lmstride + c * g.lcstride];
            if (FINAL && STAGE == 1) {
#pragma unroll
                for (int c = 0; c < 5; ++c) ubase[c] = a.Ubase[zo0 + z * mstride + c * g.cstride];
            }
        }
        const double* slot = ring + (size_t)(it % D) * NROW * BS;
        mbar_wait(&full[it % D], (uint32_t)((it / D) & 1));
        double q[5], rinv;
        cons_to_prim(g, slot[tid], slot[BS + tid], slot[2 * BS + tid], slot[3 * BS + tid], slot[4 * BS + tid], q, rinv);
        double qL[5], qR[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double sn = ppm_slope(a2[v], a1[v], q[v]);
            const double en = ppm_edge(a2[v], a1[v], s1[v], sn);
            double aL, aR;
            ppm_mono(e1[v], en, a2[v], aL, aR);
            qL[v] = aR1[v];
            qR[v] = aL;
            a2[v] = a1[v]; a1[v] = q[v]; s1[v] = sn; e1[v] = en; aR1[v] = aR;
        }
        if (it >= 5) {
            double F[5];
            hllc<DIR>(g, qL, qR, F);
            if (m.active) Fb[(long long)(n - 2) * lmstride] = F[0];
            if (upd) {
                if (!FINAL) {
                    if (m.active) {
#pragma unroll
                        for (int c = 0; c < 5; ++c) Lb[z * lmstride + c * g.lcstride] = lacc[c] - (F[c] - Fp[c]) * dinv;
                    }
                } else {
                    double L[5];
#pragma unroll
                    for (int c = 0; c < 5; ++c) L[c] = lacc[c] - (F[c] - Fp[c]) * dinv;
                    const double* sz = ring + (size_t)((it - 3) % D) * NROW * BS;   // raw state of zone z
                    double us[5];
                    us[0] = sz[tid]; us[1] = sz[BS + tid]; us[2] = sz[2 * BS + tid]; us[3] = sz[3 * BS + tid];
                    us[4] = sz[5 * BS + tid];
                    if (g.has_grav) {
                        L[1] += us[0] * g.grav[0];
                        L[2] += us[0] * g.grav[1];
                        L[3] += us[0] * g.grav[2];
                        L[4] += us[1] * g.grav[0] + us[2] * g.grav[1] + us[3] * g.grav[2];
                    }
                    double un[5];
#pragma unroll
                    for (int c = 0; c < 5; ++c) un[c] = rk_combine<STAGE>(us[c], (STAGE == 1) ? ubase[c] : 0.0, dt, L[c]);
                    const double K = ddiv(HALF * (un[1] * un[1] + un[2] * un[2] + un[3] * un[3]), un[0]);
                    double re = un[4] - K;
                    if (re < g.floor_rhoe) re = g.floor_rhoe;
                    if (m.active) {
                        const long long zo = zo0 + z * mstride;
#pragma unroll
                        for (int c = 0; c < 5; ++c) a.Uout[zo + c * g.cstride] = un[c];
                        a.Uout[zo + 5 * g.cstride] = re;
                        if (xe.single) {
                            const long long zi = zo + xe.d[0];
#pragma unroll
                            for (int c = 0; c < 5; ++c) a.Uout[zi + c * g.cstride] = (c == 1 && xe.f[0]) ? -un[c] : un[c];
                            a.Uout[zi + 5 * g.cstride] = re;
                        } else if (xe.any) {
#pragma unroll 1
                            for (int qr = 0; qr < xe.n[0] + xe.n[1]; ++qr) {
                                const int q = qr < xe.n[0] ? 0 : 1, r = qr - (q ? xe.n[0] : 0);
                                const long long zi = zo + (q ? xe.d[1] : xe.d[0]) + r * (q ? xe.step[1] : xe.step[0]);
                                const bool fq = q ? xe.f[1] : xe.f[0];
#pragma unroll
                                for (int c = 0; c < 5; ++c) a.Uout[zi + c * g.cstride] = (c == 1 && fq) ? -un[c] : un[c];
                                a.Uout[zi + 5 * g.cstride] = re;
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) Fp[c] = F[c];
        }
        // release slot (it-KEEP); warp 0 refills the slot released one step earlier
#if RING_CTASYNC == 2
        // Slot release without a CTA-wide barrier: every warp arrives on the slot's "empty"
        // mbarrier; warp 0 refills whatever slots have been released by all warps (non-blocking
        // test), and blocks only if the step it needs next has not been issued yet.
        if (it >= KEEP) {
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(&empty[(it - KEEP) % D]);
        }
        if (tid < 32) {
            while (next_issue < nsteps) {
                const int rel = next_issue - D;
                if (next_issue <= it + 1) mbar_wait(&empty[rel % D], (uint32_t)((rel / D) & 1));
                else if (!mbar_test_warp(&empty[rel % D], (uint32_t)((rel / D) & 1))) break;
                issue(next_issue);
                ++next_issue;
            }
        }
#elif RING_CTASYNC
        __syncthreads();
        if (tid < 32 && it >= KEEP && it - KEEP + D < nsteps) issue(it - KEEP + D);
#else
        if (it >= KEEP) {
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(&empty[(it - KEEP) % D]);
        }
        if (tid < 32) {
            const int rel = it - KEEP - 1;
            if (rel >= 0 && rel + D < nsteps) {
                mbar_wait(&empty[rel % D], (uint32_t)((rel / D) & 1));
                issue(rel + D);
            }
        }
#endif
    }
}

// ------------------------------------------------------------------------------------
template <int DIR, bool FINAL, int STAGE, int NS, int BS, int D>
__global__ void __launch_bounds__(BS, RING_MINB_S)
k_march_species(const __grid_constant__ Geom g, const __grid_constant__ SweepArgs a)
{
    constexpr int T = (DIR == 1) ? 2 : 1;
    constexpr int NROW = 1 + NS;
    constexpr int KEEP = FINAL ? 3 : 0;
    constexpr int NPF = 1 + NS + ((FINAL && STAGE == 1) ? NS : 0);  // F_rho, Lacc rows (+ U0 rows)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* ring = reinterpret_cast<double*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)D * NROW * BS * 8);
    uint64_t* empty = full + D;

    const int tid = threadIdx.x;
    const RingMap m = ring_map<DIR, BS>(g, tid, blockIdx.x);
    const int b = blockIdx.z;
    const int m0 = blockIdx.y * a.seglen;
    const int m1 = min(m0 + a.seglen, g.nb[DIR]);
    const int nsteps = m1 - m0 + 6;
    const int sbase = a.sbase;
    const double* Ub = a.Us + (long long)b * g.bstride;
    const long long mstride = (DIR == 1) ? g.nt[0] : (long long)g.nt[0] * g.nt[1];
    const long long lmstride = (DIR == 1) ? g.nb[0] : (long long)g.nb[0] * g.nb[1];
    double* Lbox = a.Lacc + (long long)b * g.lbstride + (long long)(5 + sbase) * g.lcstride;
    const double* Fbox = a.Frho + (long long)b * g.fbstride;

    RingDesc& ds = *reinterpret_cast<RingDesc*>(empty + D);
    if (tid < 32) {
        const int xchunks = g.nb[0] / m.W;
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const int cpy = tid + 32 * q;
            ds.src[q * 32 + tid] = nullptr; ds.dst[q * 32 + tid] = 0; ds.pf[q * 32 + tid] = nullptr; ds.pf_first[q * 32 + tid] = 0; ds.pf_stride[q * 32 + tid] = 0;
            const int row = cpy / m.R, r = cpy - row * m.R;
            const int rc = blockIdx.x * m.R + r;
            int t = rc / xchunks;
            const int x0 = (rc - t * xchunks) * m.W;
            if (t >= g.nb[T]) t = g.nb[T] - 1;
            if (row < NROW) {
                const int comp = row == 0 ? 0 : 5 + sbase + row;       // rho, then rho*X_k
                ds.src[q * 32 + tid] = Ub + (long long)comp * g.cstride + zone_off<DIR>(g, x0, t, m0 - 3);
                ds.dst[q * 32 + tid] = row * BS + r * m.W;
            }
            if (row < NPF) {
                if (row == 0) {          // F_rho of face n-2 = m0-5+it: exists from step 5 on
                    ds.pf[q * 32 + tid] = Fbox + flat_off<DIR>(g, x0, t, m0 - 5, g.nb[DIR] + 1);
                    ds.pf_first[q * 32 + tid] = 5; ds.pf_stride[q * 32 + tid] = lmstride;
                } else if (row <= NS) {  // Lacc of zone n-3
                    ds.pf[q * 32 + tid] = Lbox + (long long)(row - 1) * g.lcstride + flat_off<DIR>(g, x0, t, m0 - 6, g.nb[DIR]);
                    ds.pf_first[q * 32 + tid] = 6; ds.pf_stride[q * 32 + tid] = lmstride;
                } else {                 // U0 rho*X_k of zone n-3
                    ds.pf[q * 32 + tid] = a.Ubase + (long long)b * g.bstride + (long long)(6 + sbase + row - 1 - NS) * g.cstride +
                               zone_off<DIR>(g, x0, t, m0 - 6);
                    ds.pf_first[q * 32 + tid] = 6; ds.pf_stride[q * 32 + tid] = mstride;
                }
            }
        }
    }
    auto issue = [&](int it) {      // warp 0 only
        uint64_t* bar = &full[it % D];
        double* slot = ring + (size_t)(it % D) * NROW * BS;
        if (tid == 0) mbar_expect_tx(bar, (uint32_t)(NROW * BS * 8));
        __syncwarp();
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const double* src = ds.src[q * 32 + tid];
            if (src) bulk_g2s(slot + ds.dst[q * 32 + tid], src + it * mstride, (uint32_t)(m.W * 8), bar);
#if RING_PF
            const double* pf = ds.pf[q * 32 + tid];
            if (pf && it >= ds.pf_first[q * 32 + tid])
                bulk_prefetch_l2(pf + it * ds.pf_stride[q * 32 + tid], (uint32_t)(m.W * 8));
#endif
        }
    };

    if (tid == 0) {
        for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], BS / 32); }
        mbar_fence_init();
    }
    __syncthreads();
    if (tid < 32)
        for (int it = 0; it < D && it < nsteps; ++it) issue(it);

    double* Lb = Lbox + flat_off<DIR>(g, m.i, m.t, 0, g.nb[DIR]);
    const double* Fb = Fbox + flat_off<DIR>(g, m.i, m.t, 0, g.nb[DIR] + 1);
    const long long zo0 = (long long)b * g.bstride + zone_off<DIR>(g, m.i, m.t, 0) + (long long)(6 + sbase) * g.cstride;
    const double dinv = g.dxinv[DIR];
    const double dt = a.dt_dev ? *a.dt_dev : a.dt;

    double a1[NS], a2[NS], s1[NS], e1[NS], aR1[NS], Fp[NS];
#pragma unroll
    for (int v = 0; v < NS; ++v) { a1[v] = a2[v] = s1[v] = e1[v] = aR1[v] = Fp[v] = 0.0; }
    const XEnds xe = xends_setup(g, FINAL && a.xends && m.active, b, m.i);
    // F_rho of the face handled at step `it` is loaded one step ahead (ncu r01: 23-25 % of this
    // kernel's stall samples sat on its first use when it was loaded at the top of its own step)
    double Fnext = 0.0;

    int next_issue = D;          // first step whose copies have not been issued (warp 0)
_Pragma(RING_STR(unroll RING_UNROLL))
    for (int it = 0; it < nsteps; ++it) {
        const int n = m0 - 3 + it;
        const int z = n - 3;
        const bool upd = (it >= 6);
        const double Frho = Fnext;
        if (it >= 4 && it + 1 < nsteps) Fnext = ldg(Fb + (long long)(n - 1) * lmstride);
        double lacc[NS], ubase[NS];
        if (upd) {
#pragma unroll
            for (int v = 0; v < NS; ++v) lacc[v] = Lb[z * lmstride + v * g.lcstride];
            if (FINAL && STAGE == 1) {
#pragma unroll
                for (int v = 0; v < NS; ++v) ubase[v] = a.Ubase[zo0 + z * mstride + v * g.cstride];
            }
        }
        const double* slot = ring + (size_t)(it % D) * NROW * BS;
        mbar_wait(&full[it % D], (uint32_t)((it / D) & 1));
        const double rinv = drcp(dmax(slot[tid], g.small_dens));
        const double* sz = ring + (size_t)((it + D - 3) % D) * NROW * BS;       // zone z's slot (FINAL)
        // pass 1: reconstruction and face fluxes of all NS species (no global operand)
        double dF[NS];
#pragma unroll
        for (int v = 0; v < NS; ++v) {
            const double X = slot[(1 + v) * BS + tid] * rinv;
            const double sn = ppm_slope(a2[v], a1[v], X);
            const double en = ppm_edge(a2[v], a1[v], s1[v], sn);
            double aL, aR;
            ppm_mono(e1[v], en, a2[v], aL, aR);
            const double Fs = Frho * (Frho >= 0.0 ? aR1[v] : aL);
            a2[v] = a1[v]; a1[v] = X; s1[v] = sn; e1[v] = en; aR1[v] = aR;
            dF[v] = Fs - Fp[v];
            Fp[v] = Fs;
        }
        // pass 2: accumulator / stage update (first use of this step's global loads)
        if (upd) {
            if (!FINAL) {
#pragma unroll
                for (int v = 0; v < NS; ++v) {
                    const double L = lacc[v] - dF[v] * dinv;
                    if (m.active) Lb[z * lmstride + v * g.lcstride] = L;
                }
            } else {
                double un[NS];
                const long long zo = zo0 + z * mstride;
#pragma unroll
                for (int v = 0; v < NS; ++v) {
                    const double L = lacc[v] - dF[v] * dinv;
                    const double us = sz[(1 + v) * BS + tid];
                    un[v] = rk_combine<STAGE>(us, (STAGE == 1) ? ubase[v] : 0.0, dt, L);
                    if (m.active) a.Uout[zo + v * g.cstride] = un[v];
                }
                if (xe.single) {     // x ghost images of the zone (only the threads at the row ends)
                    const long long zi = zo + xe.d[0];
#pragma unroll
                    for (int v = 0; v < NS; ++v) a.Uout[zi + v * g.cstride] = un[v];
                } else if (xe.any) {
#pragma unroll 1
                    for (int qr = 0; qr < xe.n[0] + xe.n[1]; ++qr) {
                        const int q = qr < xe.n[0] ? 0 : 1, r = qr - (q ? xe.n[0] : 0);
                        const long long zi = zo + (q ? xe.d[1] : xe.d[0]) + r * (q ? xe.step[1] : xe.step[0]);
#pragma unroll
                        for (int v = 0; v < NS; ++v) a.Uout[zi + v * g.cstride] = un[v];
                    }
                }
            }
        }
#if RING_CTASYNC == 2
        // Slot release without a CTA-wide barrier: every warp arrives on the slot's "empty"
        // mbarrier; warp 0 refills whatever slots have been released by all warps (non-blocking
        // test), and blocks only if the step it needs next has not been issued yet.
        if (it >= KEEP) {
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(&empty[(it - KEEP) % D]);
        }
        if (tid < 32) {
            while (next_issue < nsteps) {
                const int rel = next_issue - D;
                if (next_issue <= it + 1) mbar_wait(&empty[rel % D], (uint32_t)((rel / D) & 1));
                else if (!mbar_test_warp(&empty[rel % D], (uint32_t)((rel / D) & 1))) break;
                issue(next_issue);
                ++next_issue;
            }
        }
#elif RING_CTASYNC
        __syncthreads();
        if (tid < 32 && it >= KEEP && it - KEEP + D < nsteps) issue(it - KEEP + D);
#else
        if (it >= KEEP) {
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(&empty[(it - KEEP) % D]);
        }
        if (tid < 32) {
            const int rel = it - KEEP - 1;
            if (rel >= 0 && rel + D < nsteps) {
                mbar_wait(&empty[rel % D], (uint32_t)((rel / D) & 1));
                issue(rel + D);
            }
        }
#endif
    }
}

}  // namespace hydro
