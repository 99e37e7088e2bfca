// flatten.cuh -- optional shock flattening (O10): the multi-dimensional
// flattening coefficient of every zone -1 .. nb (one ghost layer in each direction) of every box,
// written to FL (one padded array per box, laid out like a state component).  The sweeps blend the
// monotonised parabola with the zone average:  aL <- f*aL + (1-f)*a,  aR <- f*aR + (1-f)*a.
//
// The coefficient contains two yes/no decisions (shock strength > 0.33, converging flow), so its
// inputs are formed with IEEE division in BOTH builds: p = max((gamma-1)*rho_e, small_pres) and
// u = m * (1/max(rho, small_dens)) are then bit-identical to the definition's, and so is FL.
#pragma once
#include "hydro_device.cuh"

namespace hydro {

__device__ __forceinline__ void flat_blend(double f, double omf, double a, double& aL, double& aR)
{
    aL = f * aL + omf * a;
    aR = f * aR + omf * a;
}

// chi*z and dp of padded zone index m along direction DIR of the line through (i, j, k)
template <int DIR>
__device__ __forceinline__ void flat_zc(const Geom& g, const double* __restrict__ Ub, long long z, long long st,
                                        double& zc, double& dp)
{
    auto pres = [&](long long zz) { return dmax(g.gm1 * __ldg(Ub + 5 * g.cstride + zz), g.small_pres); };
    auto vel = [&](long long zz) {
        const double r = dmax(__ldg(Ub + zz), g.small_dens);
        return __dmul_rn(__ldg(Ub + (1 + DIR) * g.cstride + zz), __drcp_rn(r));
    };
    const double pm = pres(z - st), pp = pres(z + st);
    dp = pp - pm;
    const double den = dmax(g.small_pres, fabs(pres(z + 2 * st) - pres(z - 2 * st)));
    const double zeta = __ddiv_rn(fabs(dp), den);
    const double zr = dmin(1.0, dmax(0.0, 10.0 * (zeta - 0.75)));
    const bool shock = __ddiv_rn(fabs(dp), dmin(pp, pm)) > 0.33 && (vel(z - st) - vel(z + st) >= 0.0);
    zc = shock ? zr : 0.0;
}

template <int DIR>
__device__ __forceinline__ double flat_dir(const Geom& g, const double* __restrict__ Ub, long long z)
{
    const long long st = DIR == 0 ? 1 : (DIR == 1 ? (long long)g.nt[0] : (long long)g.nt[0] * g.nt[1]);
    double zc0, dp0, zcm, zcp, dpx;
    flat_zc<DIR>(g, Ub, z, st, zc0, dp0);
    flat_zc<DIR>(g, Ub, z - st, st, zcm, dpx);
    flat_zc<DIR>(g, Ub, z + st, st, zcp, dpx);
    // neighbour on the low-pressure side: i-1 for dp > 0, i+1 for dp < 0, none for dp == 0
    const double nb = dp0 > 0.0 ? zcm : (dp0 < 0.0 ? zcp : 0.0);
    return 1.0 - dmax(zc0, nb);
}

// grid (ceil((nb0+2)/128) * (nb1+2), nb2+2, boxes), 128 threads: one thread per zone -1 .. nb
__global__ void __launch_bounds__(128)
k_flatten(const __grid_constant__ Geom g, const double* __restrict__ U, double* __restrict__ FL)
{
    const int xblocks = (g.nb[0] + 2 + 127) / 128;
    const int jl = blockIdx.x / xblocks, kl = blockIdx.y;
    const int il = (blockIdx.x - jl * xblocks) * 128 + threadIdx.x;     // 0 .. nb0+1  <->  zone -1 .. nb0
    if (il > g.nb[0] + 1) return;
    const int b = blockIdx.z;
    const long long z = ((long long)(kl + g.ng - 1) * g.nt[1] + (jl + g.ng - 1)) * g.nt[0] + (il + g.ng - 1);
    const double* Ub = U + (long long)b * g.bstride;
    const double f = dmin(flat_dir<0>(g, Ub, z), dmin(flat_dir<1>(g, Ub, z), flat_dir<2>(g, Ub, z)));
    FL[(long long)b * g.cstride + z] = f;
}

__global__ void __launch_bounds__(256)
k_fill_value(double* __restrict__ x, long long n, double v)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) x[i] = v;
}

}  // namespace hydro
