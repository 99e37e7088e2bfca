// amr_fill.cuh -- O13 (second half): two-level ghost fill.  The fine
// level is a rectangular patch of the coarse domain refined by `ratio` (2 or 4), tiled by its own
// boxes; its faces inside the coarse domain are HYDRO_BC_EXTERNAL.  Every fine ghost zone whose index lies across
// such a face in at least one dimension takes its NVAR components from the coarse level by conservative linear
// interpolation: value = Uc + sx*xi_x + sy*xi_y + sz*xi_z, slopes = the limited slope of O3 of the coarse zone
// averages, xi = (child + 0.5)/ratio - 0.5 (readings A1-A5, oracle_fill_from_coarse).  Coarse zones outside the
// coarse domain are the coarse level's own ghost zones (fill them first).
#pragma once
#include "ghost_reduce.cuh"
#include "hydro_device.cuh"

namespace hydro {

struct AmrArgs {
    double* Uf;            // fine state (ghost zones across EXTERNAL faces written)
    const double* Uc;      // coarse state, ghosts filled
    int lo[3];             // coarse zone of the patch's first fine zone
    int ratio;
};

// padded offset inside the coarse state of component 0 of coarse GLOBAL zone (gx, gy, gz), which may lie up to
// ng zones outside the coarse domain (then it is a ghost zone of the nearest box)
__device__ __forceinline__ long long coarse_off(const Geom& gc, int gx, int gy, int gz)
{
    const int gi[3] = {gx, gy, gz};
    int bd[3], l[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        int b = floor_div(gi[d], gc.nb[d]);
        b = b < 0 ? 0 : (b > gc.NB[d] - 1 ? gc.NB[d] - 1 : b);
        bd[d] = b;
        l[d] = gi[d] - b * gc.nb[d] + gc.ng;
    }
    const long long b = ((long long)bd[2] * gc.NB[1] + bd[1]) * gc.NB[0] + bd[0];
    return b * gc.bstride + ((long long)l[2] * gc.nt[1] + l[1]) * gc.nt[0] + l[0];
}

// one thread per padded fine zone of a (k-plane, box): grid (ceil(nt0*nt1 / 256), nt2, fine boxes)
__global__ void __launch_bounds__(256)
k_fill_from_coarse(const __grid_constant__ Geom gf, const __grid_constant__ Geom gc, const __grid_constant__ AmrArgs a)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= gf.nt[0] * gf.nt[1]) return;
    const int jl = t / gf.nt[0], il = t - jl * gf.nt[0], kl = blockIdx.y;
    const int b = blockIdx.z;
    const int bb[3] = {b % gf.NB[0], (b / gf.NB[0]) % gf.NB[1], b / (gf.NB[0] * gf.NB[1])};
    const int ll[3] = {il, jl, kl};
    int cz[3];
    double xi[3];
    bool ext = false;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int g = bb[d] * gf.nb[d] + ll[d] - gf.ng;
        if ((g < 0 && gf.bc_lo[d] == 3) || (g >= gf.ndom[d] && gf.bc_hi[d] == 3)) ext = true;
        const int q = floor_div(g, a.ratio);
        cz[d] = a.lo[d] + q;
        xi[d] = ((double)(g - a.ratio * q) + 0.5) / (double)a.ratio - 0.5;
    }
    if (!ext) return;
    const long long z0 = coarse_off(gc, cz[0], cz[1], cz[2]);
    long long zm[3], zp[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        int m[3] = {cz[0], cz[1], cz[2]}, p[3] = {cz[0], cz[1], cz[2]};
        m[d] -= 1; p[d] += 1;
        zm[d] = coarse_off(gc, m[0], m[1], m[2]);
        zp[d] = coarse_off(gc, p[0], p[1], p[2]);
    }
    double* dst = a.Uf + (long long)b * gf.bstride + ((long long)kl * gf.nt[1] + jl) * gf.nt[0] + il;
    for (int c = 0; c < gf.nvar; ++c) {
        const long long co = (long long)c * gc.cstride;
        const double u0 = __ldg(a.Uc + z0 + co);
        double val = u0;
#pragma unroll
        for (int d = 0; d < 3; ++d)
            val = val + ppm_slope(__ldg(a.Uc + zm[d] + co), u0, __ldg(a.Uc + zp[d] + co)) * xi[d];
        dst[(long long)c * gf.cstride] = val;
    }
}

// restriction (reading A6): coarse valid zone under the patch <- mean of its ratio^3 children, summed k, j, i (i innermost).
// One thread per (coarse zone of the patch, component): grid (ceil(zones / 256), nvar).
__global__ void __launch_bounds__(256)
k_average_down(const __grid_constant__ Geom gc, const __grid_constant__ Geom gf, double* __restrict__ Uc,
               const double* __restrict__ Uf, int lo0, int lo1, int lo2, int ratio)
{
    const int n0 = gf.ndom[0] / ratio, n1 = gf.ndom[1] / ratio, n2 = gf.ndom[2] / ratio;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n0 * n1 * n2) return;
    const int I = (int)(t % n0), J = (int)((t / n0) % n1), K = (int)(t / ((long long)n0 * n1));
    const int c = blockIdx.y;
    const int G[3] = {lo0 + I, lo1 + J, lo2 + K};
    const long long cb = ((long long)(G[2] / gc.nb[2]) * gc.NB[1] + G[1] / gc.nb[1]) * gc.NB[0] + G[0] / gc.nb[0];
    const long long cz = cb * gc.bstride + (long long)c * gc.cstride +
                         ((long long)(G[2] % gc.nb[2] + gc.ng) * gc.nt[1] + (G[1] % gc.nb[1] + gc.ng)) * gc.nt[0] + (G[0] % gc.nb[0] + gc.ng);
    double sum = 0.0;
    for (int kk = 0; kk < ratio; ++kk)
        for (int jj = 0; jj < ratio; ++jj)
            for (int ii = 0; ii < ratio; ++ii) {
                const int g[3] = {I * ratio + ii, J * ratio + jj, K * ratio + kk};
                const long long fb = ((long long)(g[2] / gf.nb[2]) * gf.NB[1] + g[1] / gf.nb[1]) * gf.NB[0] + g[0] / gf.nb[0];
                sum = sum + __ldg(Uf + fb * gf.bstride + (long long)c * gf.cstride +
                                  ((long long)(g[2] % gf.nb[2] + gf.ng) * gf.nt[1] + (g[1] % gf.nb[1] + gf.ng)) * gf.nt[0] + (g[0] % gf.nb[0] + gf.ng));
            }
    Uc[cz] = sum * (1.0 / (double)(ratio * ratio * ratio));
}

}  // namespace hydro
