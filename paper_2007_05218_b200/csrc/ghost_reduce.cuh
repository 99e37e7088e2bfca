// ghost_reduce.cuh -- ghost-zone fill (O1), CFL reduction (O8), conservation totals (O9).
#pragma once
#include "hydro_device.cuh"

namespace hydro {

// ---- O1 ----------------------------------------------------------------------------
// Global index along dimension d -> the valid global index that supplies it; flip is set
// when a reflecting wall was crossed.
__device__ __forceinline__ int map_global(const Geom& g, int d, int gi, bool& flip)
{
    const int n = g.ndom[d];
    flip = false;
    if (gi >= 0 && gi < n) return gi;
    const int bc = gi < 0 ? g.bc_lo[d] : g.bc_hi[d];
    if (bc == 0) return ((gi % n) + n) % n;
    if (bc == 1) return gi < 0 ? 0 : n - 1;
    flip = true;
    return gi < 0 ? -1 - gi : 2 * n - 1 - gi;
}

// One CTA per (padded k-plane, component, box); the plane's ghost zones are enumerated as a
// flat task list so that consecutive threads touch consecutive zones.  A plane in the ghost
// k-range is filled whole; a plane in the valid k-range has 2*ng whole ghost rows plus the
// 2*ng end zones of each valid row.  The k mapping is done once per CTA.  Reads valid zones,
// writes ghost zones: disjoint, so one launch is race free.
__global__ void __launch_bounds__(256)
k_fill_ghosts(const __grid_constant__ Geom g, double* __restrict__ U)
{
    const int kl = blockIdx.x, c = blockIdx.y, b = blockIdx.z;
    const int bi = b % g.NB[0], bj = (b / g.NB[0]) % g.NB[1], bk = b / (g.NB[0] * g.NB[1]);
    bool fz;
    const int gz = map_global(g, 2, bk * g.nb[2] + kl - g.ng, fz);
    const int sbk = gz / g.nb[2];
    const int skl = gz - sbk * g.nb[2] + g.ng;
    const bool kghost = kl < g.ng || kl >= g.ng + g.nb[2];
    const int ng2 = 2 * g.ng;
    const int nA = kghost ? g.nt[1] * g.nt[0] : ng2 * g.nt[0];      // whole rows
    const int nB = kghost ? 0 : g.nb[1] * ng2;                        // row ends
    double* dplane = U + ((long long)b * g.nvar + c) * g.cstride + (long long)kl * g.nt[1] * g.nt[0];
    const double* splane = U + (long long)c * g.cstride + (long long)skl * g.nt[1] * g.nt[0];
    for (int idx = threadIdx.x; idx < nA + nB; idx += blockDim.x) {
        int jl, il;
        if (idx < nA) {
            const int row = idx / g.nt[0];
            il = idx - row * g.nt[0];
            jl = kghost ? row : (row < g.ng ? row : g.nb[1] + row);
        } else {
            const int r = idx - nA;
            const int row = r / ng2, l = r - row * ng2;
            jl = g.ng + row;
            il = l < g.ng ? l : g.nb[0] + l;
        }
        bool fx, fy;
        const int gx = map_global(g, 0, bi * g.nb[0] + il - g.ng, fx);
        const int gy = map_global(g, 1, bj * g.nb[1] + jl - g.ng, fy);
        const int sbi = gx / g.nb[0], sbj = gy / g.nb[1];
        const long long sb = ((long long)sbk * g.NB[1] + sbj) * g.NB[0] + sbi;
        double v = splane[sb * g.bstride + (long long)(gy - sbj * g.nb[1] + g.ng) * g.nt[0] + (gx - sbi * g.nb[0] + g.ng)];
        if ((c == 1 && fx) || (c == 2 && fy) || (c == 3 && fz)) v = -v;
        dplane[(long long)jl * g.nt[0] + il] = v;
    }
}

// ---- O8 ----------------------------------------------------------------------------
// red[0] = running max of t (as ordered bits), red[1] = blocks-done counter,
// dtslot[0] = dt, dtslot[1] = max t of the last reduction.
__global__ void __launch_bounds__(256)
k_estimate_dt(const __grid_constant__ Geom g, const double* __restrict__ U, unsigned long long* red,
              double* dtslot)
{
    const long long nzone = g.lcstride * g.nboxes;
    double tmax = 0.0;
    bool bad = false;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < nzone;
         v += (long long)gridDim.x * blockDim.x) {
        long long r = v;
        const int i = (int)(r % g.nb[0]); r /= g.nb[0];
        const int j = (int)(r % g.nb[1]); r /= g.nb[1];
        const int k = (int)(r % g.nb[2]);
        const long long b = r / g.nb[2];
        const double* Uz = U + b * g.bstride + ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0] + (i + g.ng);
        double q[5], rinv;
        cons_to_prim(g, ldg(Uz), ldg(Uz + g.cstride), ldg(Uz + 2 * g.cstride), ldg(Uz + 3 * g.cstride),
                     ldg(Uz + 5 * g.cstride), q, rinv);
        const double cs = sqrt(g.gamma * q[4] * rinv);
        const double t = (fabs(q[1]) + cs) * g.dxinv[0] + (fabs(q[2]) + cs) * g.dxinv[1] + (fabs(q[3]) + cs) * g.dxinv[2];
        if (!(t == t)) bad = true;
        if (t > tmax) tmax = t;
    }
    // t >= 0, so the IEEE bit pattern orders like the value; NaN is mapped above +inf
    unsigned long long bits = bad ? 0x7ff8000000000000ull : (unsigned long long)__double_as_longlong(tmax);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, bits, o);
        bits = other > bits ? other : bits;
    }
    __shared__ unsigned long long sm[8];
    __shared__ bool last;
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = bits;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int wv = 1; wv < (int)(blockDim.x >> 5); ++wv) bits = sm[wv] > bits ? sm[wv] : bits;
        atomicMax(red, bits);
        __threadfence();
        last = (atomicAdd(red + 1, 1ull) == gridDim.x - 1);
        if (last) {
            __threadfence();
            const unsigned long long m = atomicExch(red, 0ull);   // reset for the next call
            red[1] = 0ull;
            const double tm = __longlong_as_double((long long)m);
            dtslot[1] = tm;
            dtslot[0] = g.cfl / tm;
        }
    }
}

// ---- O9 ----------------------------------------------------------------------------
// error-free transformation: s + e == a + b exactly
__device__ __forceinline__ void two_sum(double a, double b, double& s, double& e)
{
    s = __dadd_rn(a, b);
    const double bb = __dsub_rn(s, a);
    e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}
__device__ __forceinline__ void dd_add(double& hi, double& lo, double xh, double xl)
{
    double s, e;
    two_sum(hi, xh, s, e);
    lo = __dadd_rn(__dadd_rn(lo, xl), e);
    hi = s;
}

// pass 1: grid (blocks, nflux); each block leaves a (hi, lo) partial in part[(c*blocks+blk)*2]
__global__ void __launch_bounds__(256)
k_totals_partial(const __grid_constant__ Geom g, const double* __restrict__ U, double* __restrict__ part)
{
    const int c = blockIdx.y;
    const int sc = c < 5 ? c : c + 1;
    const long long nzone = g.lcstride * g.nboxes;
    double hi = 0.0, lo = 0.0;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < nzone;
         v += (long long)gridDim.x * blockDim.x) {
        long long r = v;
        const int i = (int)(r % g.nb[0]); r /= g.nb[0];
        const int j = (int)(r % g.nb[1]); r /= g.nb[1];
        const int k = (int)(r % g.nb[2]);
        const long long b = r / g.nb[2];
        const double x = ldg(U + b * g.bstride + sc * g.cstride +
                             ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0] + (i + g.ng));
        dd_add(hi, lo, x, 0.0);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double oh = __shfl_xor_sync(0xffffffffu, hi, o), ol = __shfl_xor_sync(0xffffffffu, lo, o);
        dd_add(hi, lo, oh, ol);
    }
    __shared__ double sh[8], sl[8];
    if ((threadIdx.x & 31) == 0) { sh[threadIdx.x >> 5] = hi; sl[threadIdx.x >> 5] = lo; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int wv = 1; wv < (int)(blockDim.x >> 5); ++wv) dd_add(hi, lo, sh[wv], sl[wv]);
        part[((long long)c * gridDim.x + blockIdx.x) * 2] = hi;
        part[((long long)c * gridDim.x + blockIdx.x) * 2 + 1] = lo;
    }
}

// pass 2: one warp per component folds the partials in a fixed order
__global__ void __launch_bounds__(32)
k_totals_final(const __grid_constant__ Geom g, const double* __restrict__ part, int nblocks, double* __restrict__ out)
{
    const int c = blockIdx.x;
    double hi = 0.0, lo = 0.0;
    for (int p = threadIdx.x; p < nblocks; p += 32)
        dd_add(hi, lo, part[((long long)c * nblocks + p) * 2], part[((long long)c * nblocks + p) * 2 + 1]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double oh = __shfl_xor_sync(0xffffffffu, hi, o), ol = __shfl_xor_sync(0xffffffffu, lo, o);
        dd_add(hi, lo, oh, ol);
    }
    if (threadIdx.x == 0) out[c] = (hi + lo) * g.vol;
}

}  // namespace hydro
