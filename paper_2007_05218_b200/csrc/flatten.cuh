// flatten.cuh -- optional shock flattening (O10): the multi-dimensional
// flattening coefficient of every zone -1 .. nb (one ghost layer in each direction) of every box,
// written to FL (one padded array per box, laid out like a state component).  The sweeps blend the
// monotonised parabola with the zone average:  aL <- f*aL + (1-f)*a,  aR <- f*aR + (1-f)*a.
//
// The coefficient contains two yes/no decisions (shock strength > 0.33, converging flow); both are taken
// exactly as the definition takes them (flat_zc), in both builds; the value z of the ramp is continuous.
#pragma once
#include "hydro_device.cuh"

namespace hydro {

__device__ __forceinline__ void flat_blend(double f, double omf, double a, double& aL, double& aR)
{
    aL = f * aL + omf * a;
    aR = f * aR + omf * a;
}

// chi*z of the zone at padded offset z along direction DIR (st = stride of DIR).
// The two yes/no tests are filtered predicates: they are decided with the fast reciprocal when the
// margin is far larger than its error (relative 1e-12 against <= 2 ulp), and only the rare near-ties
// are redone with IEEE division, so the decision is always the definition's; z itself is continuous in
// its inputs and may differ from the definition by rounding.
template <int DIR>
__device__ __forceinline__ double flat_zc(const Geom& g, const double* __restrict__ Ub, long long z, long long st)
{
    auto pres = [&](long long zz) { return dmax(g.gm1 * __ldg(Ub + 5 * g.cstride + zz), g.small_pres); };
    const double pm = pres(z - st), pp = pres(z + st);
    const double adp = fabs(pp - pm);
    const double den = dmax(g.small_pres, fabs(pres(z + 2 * st) - pres(z - 2 * st)));
    const double zeta = ddiv(adp, den);
    const double zr = dmin(1.0, dmax(0.0, 10.0 * (zeta - 0.75)));
    double zc = 0.0;
    if (zr > 0.0) {                                    // only zones inside a steep pressure ramp go on
        const double pmin = dmin(pp, pm);
        const double q = adp * drcp(pmin);
        bool strong;
        if (fabs(q - 0.33) > 1e-12) strong = q > 0.33;
        else strong = __ddiv_rn(adp, pmin) > 0.33;
        if (strong) {
            const double rm = dmax(__ldg(Ub + z - st), g.small_dens), rp = dmax(__ldg(Ub + z + st), g.small_dens);
            const double mm = __ldg(Ub + (1 + DIR) * g.cstride + z - st), mp = __ldg(Ub + (1 + DIR) * g.cstride + z + st);
            const double um = mm * drcp(rm), up = mp * drcp(rp);
            const double d = um - up;
            bool conv;
            if (fabs(d) > 1e-12 * (fabs(um) + fabs(up))) conv = d >= 0.0;
            else conv = __dmul_rn(mm, __drcp_rn(rm)) - __dmul_rn(mp, __drcp_rn(rp)) >= 0.0;
            if (conv) zc = zr;
        }
    }
    return zc;
}

// Blocks of 32 x 4 x 4 zones over the cube lo .. nb+1-lo' of every box:
// grid (ceil(n0/32) * boxes, ceil(n1/4), ceil(n2/4)) with n_d the zones of the cube along d.
constexpr int FLT_BX = 32, FLT_BY = 4, FLT_BZ = 4;
__device__ __forceinline__ bool flat_zone(const Geom& g, int lo, int& b, long long& z)
{
    const int n2 = g.nb[2] - 2 * lo;
    const int xblocks = gridDim.x / g.nboxes;
    b = blockIdx.x / xblocks;
    const int il = (blockIdx.x - b * xblocks) * FLT_BX + threadIdx.x;
    const int jl = blockIdx.y * FLT_BY + threadIdx.y;
    const int kl = blockIdx.z * FLT_BZ + threadIdx.z;
    if (il >= g.nb[0] - 2 * lo || jl >= g.nb[1] - 2 * lo || kl >= n2) return false;
    z = ((long long)(kl + g.ng + lo) * g.nt[1] + (jl + g.ng + lo)) * g.nt[0] + (il + g.ng + lo);
    return true;
}

// pass 1: ZC[d] = chi*z along d, d = 0, 1, 2, on zones -2 .. nb+1 (three padded arrays per box)
__global__ void __launch_bounds__(FLT_BX * FLT_BY * FLT_BZ)
k_flatten_zc(const __grid_constant__ Geom g, const double* __restrict__ U, double* __restrict__ ZC)
{
    int b; long long z;
    if (!flat_zone(g, -2, b, z)) return;
    const double* Ub = U + (long long)b * g.bstride;
    double* Zb = ZC + (long long)b * 3 * g.cstride + z;
    Zb[0] = flat_zc<0>(g, Ub, z, 1);
    Zb[g.cstride] = flat_zc<1>(g, Ub, z, g.nt[0]);
    Zb[2 * g.cstride] = flat_zc<2>(g, Ub, z, (long long)g.nt[0] * g.nt[1]);
}

// pass 2: FL = min over d of 1 - max(zc_d[i], zc_d[i -+ 1]) on zones -1 .. nb; the neighbour is the one
// on the low-pressure side (none when dp == 0, reading F3)
__global__ void __launch_bounds__(FLT_BX * FLT_BY * FLT_BZ)
k_flatten(const __grid_constant__ Geom g, const double* __restrict__ U, const double* __restrict__ ZC,
          double* __restrict__ FL)
{
    int b; long long z;
    if (!flat_zone(g, -1, b, z)) return;
    const double* Pb = U + (long long)b * g.bstride + 5 * g.cstride + z;
    const double* Zb = ZC + (long long)b * 3 * g.cstride + z;
    double f = 1.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const long long st = d == 0 ? 1 : (d == 1 ? (long long)g.nt[0] : (long long)g.nt[0] * g.nt[1]);
        const double* Zd = Zb + d * g.cstride;
        // all five loads are independent (the neighbour is chosen after they return)
        const double pp = __ldg(Pb + st), pm = __ldg(Pb - st);
        const double zm = __ldg(Zd - st), z0 = __ldg(Zd), zp = __ldg(Zd + st);
        const double dp = dmax(g.gm1 * pp, g.small_pres) - dmax(g.gm1 * pm, g.small_pres);
        const double nbr = dp > 0.0 ? zm : (dp < 0.0 ? zp : 0.0);
        f = dmin(f, 1.0 - dmax(z0, nbr));
    }
    FL[(long long)b * g.cstride + z] = f;
}

__global__ void __launch_bounds__(256)
k_fill_value(double* __restrict__ x, long long n, double v)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) x[i] = v;
}

}  // namespace hydro
