// ghost_reduce.cuh -- ghost-zone fill (O1), CFL reduction (O8), conservation totals (O9).
#pragma once
#include "hydro_device.cuh"

namespace hydro {

// ---- O1 ----------------------------------------------------------------------------
// Global index along dimension d -> the valid global index that supplies it; flip is set
// when a reflecting wall was crossed.  Returns -1 when the zone lies across an EXTERNAL face
// (bc 3: it belongs to another shard and is filled by hydro_unpack_halo, not here).
__device__ __forceinline__ int map_global(const Geom& g, int d, int gi, bool& flip)
{
    const int n = g.ndom[d];
    flip = false;
    if (gi >= 0 && gi < n) return gi;
    const int bc = gi < 0 ? g.bc_lo[d] : g.bc_hi[d];
    if (bc == 0) return ((gi % n) + n) % n;
    if (bc == 1) return gi < 0 ? 0 : n - 1;
    if (bc == 3) return -1;
    flip = true;
    return gi < 0 ? -1 - gi : 2 * n - 1 - gi;
}

// One CTA per (padded k-plane, box, component): grid (nt2 * boxes, nvar); the plane's ghost zones are enumerated as a
// flat task list so that consecutive threads touch consecutive zones.  A plane in the ghost
// k-range is filled whole; a plane in the valid k-range has 2*ng whole ghost rows plus the
// 2*ng end zones of each valid row.  The k mapping is done once per CTA.  Reads valid zones,
// writes ghost zones: disjoint, so one launch is race free.
__global__ void __launch_bounds__(256)
k_fill_ghosts(const __grid_constant__ Geom g, double* __restrict__ U)
{
    const int b = blockIdx.x / g.nt[2], kl = blockIdx.x - b * g.nt[2], c = blockIdx.y;
    const int bi = b % g.NB[0], bj = (b / g.NB[0]) % g.NB[1], bk = b / (g.NB[0] * g.NB[1]);
    bool fz;
    const int gz = map_global(g, 2, bk * g.nb[2] + kl - g.ng, fz);
    if (gz < 0) return;                                                // plane across an external z face
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
        if (gx < 0 || gy < 0) continue;                                // across an external x or y face
        const int sbi = gx / g.nb[0], sbj = gy / g.nb[1];
        const long long sb = ((long long)sbk * g.NB[1] + sbj) * g.NB[0] + sbi;
        double v = splane[sb * g.bstride + (long long)(gy - sbj * g.nb[1] + g.ng) * g.nt[0] + (gx - sbi * g.nb[0] + g.ng)];
        if ((c == 1 && fx) || (c == 2 && fy) || (c == 3 && fz)) v = -v;
        dplane[(long long)jl * g.nt[0] + il] = v;
    }
}

// ---- O1, split form used inside hydro_step ---------------------------------------------
// The z (FINAL) sweeps write, next to every valid zone, the x-direction ghost images of that
// zone (march_ring.cuh), so that every valid row (j, k valid) of the destination state is a
// complete padded row.  What is left of the ghost fill are the ghost ROWS (j or k in the ghost
// range): whole padded rows, each a copy of the complete padded row that the y/z mapping of O1
// selects (same box column, so the x ends compose exactly as in k_fill_ghosts), with the sign
// of rho*v / rho*w flipped across a reflecting y / z wall.  k_fill_ghost_rows does those copies
// as 16-byte vectors.

__device__ __forceinline__ int floor_div(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

// q-th ghost image (q = 0, 1, ...) along dimension d of valid zone l of box bd: the ghost zone
// of box `dbox` at padded index `p` whose O1 source is this zone.  Returns false when there
// are fewer than q+1 images.  Requires nb[d] >= ng.  Enumeration: the zone's own coordinate
// (ghost of the adjacent boxes), then the coordinates the boundary condition maps onto it.
__device__ __noinline__ bool dim_image(const Geom& g, int d, int bd, int l, int q, int& dbox, int& p, bool& flip)
{
    const int nb = g.nb[d], n = g.ndom[d], ng = g.ng, NB = g.NB[d];
    const int g0 = bd * nb + l;
    int cnt = 0;
    // every box whose ghost range contains virtual coordinate v
    auto visit = [&](int v, bool f) -> bool {
        const int qb = floor_div(v, nb);
        if (qb + 1 >= 0 && qb + 1 < NB && v >= (qb + 1) * nb - ng) {       // low ghosts of box qb+1
            if (cnt == q) { dbox = qb + 1; p = v - (qb + 1) * nb + ng; flip = f; return true; }
            ++cnt;
        }
        if (qb - 1 >= 0 && qb - 1 < NB && v < qb * nb + ng) {              // high ghosts of box qb-1
            if (cnt == q) { dbox = qb - 1; p = v - (qb - 1) * nb + ng; flip = f; return true; }
            ++cnt;
        }
        return false;
    };
    if (visit(g0, false)) return true;
    if (g.bc_lo[d] == 0) {                     // periodic (both sides)
        if (visit(g0 - n, false)) return true;
        if (visit(g0 + n, false)) return true;
        return false;
    }
    if (g.bc_lo[d] == 1 && g0 == 0) {
        for (int v = -1; v >= -ng; --v) if (visit(v, false)) return true;
    } else if (g.bc_lo[d] == 2 && g0 < ng) {
        if (visit(-1 - g0, true)) return true;
    }
    if (g.bc_hi[d] == 1 && g0 == n - 1) {
        for (int v = n; v < n + ng; ++v) if (visit(v, false)) return true;
    } else if (g.bc_hi[d] == 2 && g0 >= n - ng) {
        if (visit(2 * n - 1 - g0, true)) return true;
    }
    return false;
}

// x ghost zones of the VALID rows (j, k valid): the first half of O1 in its split form when no z sweep has
// written them (the caller's state).  One thread per ghost zone; grid (ceil(nb1 * 2ng / 256) * boxes, nb2, nvar).
__global__ void __launch_bounds__(256)
k_fill_xends(const __grid_constant__ Geom g, double* __restrict__ U)
{
    const int ng2 = 2 * g.ng;
    const int xblocks = gridDim.x / g.nboxes;
    const int b = blockIdx.x / xblocks, c = blockIdx.z;
    const int t = (blockIdx.x - b * xblocks) * blockDim.x + threadIdx.x;
    if (t >= g.nb[1] * ng2) return;
    const int j = t / ng2, l = t - j * ng2;
    const int k = blockIdx.y;
    const int bi = b % g.NB[0];
    const int il = l < g.ng ? l : g.nb[0] + l;
    bool fx;
    const int gx = map_global(g, 0, bi * g.nb[0] + il - g.ng, fx);
    const int sbi = gx / g.nb[0];
    const long long row = ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0];
    double v = U[((long long)(b + sbi - bi) * g.nvar + c) * g.cstride + row + (gx - sbi * g.nb[0] + g.ng)];
    if (c == 1 && fx) v = -v;
    U[((long long)b * g.nvar + c) * g.cstride + row + il] = v;
}

constexpr int GR_ROWS = 16;    // ghost rows per CTA of k_fill_ghost_rows

// grid (ceil(nrows / GR_ROWS) * boxes, nvar), 256 threads.  nt[0] must be even (16-byte rows).
__global__ void __launch_bounds__(256)
k_fill_ghost_rows(const __grid_constant__ Geom g, double* __restrict__ U)
{
    __shared__ long long s_src[GR_ROWS], s_dst[GR_ROWS];
    __shared__ double s_sgn[GR_ROWS];
    const int rblocks = gridDim.x / g.nboxes;
    const int b = blockIdx.x / rblocks, c = blockIdx.y;
    const int ng2 = 2 * g.ng;
    const int nrows = g.nt[2] * g.nt[1] - g.nb[2] * g.nb[1];
    const int r0 = (blockIdx.x - b * rblocks) * GR_ROWS;
    if (threadIdx.x < GR_ROWS) {
        const int r = r0 + threadIdx.x;
        long long src = -1, dst = 0;
        double sgn = 1.0;
        if (r < nrows) {
            int kl, jl;
            if (r < ng2 * g.nt[1]) {                                 // the 2*ng whole ghost planes
                const int pz = r / g.nt[1];
                kl = pz < g.ng ? pz : g.nb[2] + pz;
                jl = r - pz * g.nt[1];
            } else {                                                 // ghost rows of the valid planes
                const int rr = r - ng2 * g.nt[1];
                const int kz = rr / ng2, t = rr - kz * ng2;
                kl = g.ng + kz;
                jl = t < g.ng ? t : g.nb[1] + t;
            }
            const int bi = b % g.NB[0], bj = (b / g.NB[0]) % g.NB[1], bk = b / (g.NB[0] * g.NB[1]);
            bool fy, fz;
            const int gy = map_global(g, 1, bj * g.nb[1] + jl - g.ng, fy);
            const int gz = map_global(g, 2, bk * g.nb[2] + kl - g.ng, fz);
            const int sbj = gy / g.nb[1], sbk = gz / g.nb[2];
            const long long sb = ((long long)sbk * g.NB[1] + sbj) * g.NB[0] + bi;
            src = (sb * g.nvar + c) * g.cstride +
                  ((long long)(gz - sbk * g.nb[2] + g.ng) * g.nt[1] + (gy - sbj * g.nb[1] + g.ng)) * g.nt[0];
            dst = ((long long)b * g.nvar + c) * g.cstride + ((long long)kl * g.nt[1] + jl) * g.nt[0];
            if ((c == 2 && fy) || (c == 3 && fz)) sgn = -1.0;
        }
        s_src[threadIdx.x] = src; s_dst[threadIdx.x] = dst; s_sgn[threadIdx.x] = sgn;
    }
    __syncthreads();
    const int vpr = g.nt[0] >> 1;                                    // double2 per row
    for (int e = threadIdx.x; e < GR_ROWS * vpr; e += blockDim.x) {
        const int r = e / vpr, col = e - r * vpr;
        const long long src = s_src[r];
        if (src < 0) continue;
        double2 v = __ldg(reinterpret_cast<const double2*>(U + src) + col);
        const double sg = s_sgn[r];
        v.x *= sg; v.y *= sg;
        reinterpret_cast<double2*>(U + s_dst[r])[col] = v;
    }
}

// ---- O8 ----------------------------------------------------------------------------
// Grid-wide max of the per-thread CFL signal `tmax`: warp shuffle, one atomicMax per CTA on the
// ordered bit pattern; the last CTA to arrive writes dtslot[0] = cfl / max, dtslot[1] = max and
// resets the workspace.  Called by every thread of every CTA; sm = 8+ words of shared scratch
// that no thread still reads.  red[0] = running max (as ordered bits), red[1] = CTAs done.
__device__ __forceinline__ void cfl_reduce_finish(const Geom& g, bool bad, double tmax, unsigned long long* red,
                                                  double* dtslot, unsigned long long* sm)
{
    // t >= 0, so the IEEE bit pattern orders like the value; NaN is mapped above +inf
    unsigned long long bits = bad ? 0x7ff8000000000000ull : (unsigned long long)__double_as_longlong(tmax);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, bits, o);
        bits = other > bits ? other : bits;
    }
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = bits;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int wv = 1; wv < (int)(blockDim.x >> 5); ++wv) bits = sm[wv] > bits ? sm[wv] : bits;
        atomicMax(red, bits);
        __threadfence();
        const unsigned long long nblk = (unsigned long long)gridDim.x * gridDim.y * gridDim.z;
        if (atomicAdd(red + 1, 1ull) == nblk - 1) {
            __threadfence();
            const unsigned long long mx = atomicExch(red, 0ull);   // reset for the next call
            red[1] = 0ull;
            const double tm = __longlong_as_double((long long)mx);
            dtslot[1] = tm;
            dtslot[0] = g.cfl / tm;
        }
    }
}

// red[0] = running max of t (as ordered bits), red[1] = blocks-done counter,
// dtslot[0] = dt, dtslot[1] = max t of the last reduction.
__global__ void __launch_bounds__(256)
k_estimate_dt(const __grid_constant__ Geom g, const double* __restrict__ U, unsigned long long* red,
              double* dtslot)
{
    // a warp takes whole rows (the row index is decoded once per row, not once per zone)
    const long long nrows = (long long)g.nb[1] * g.nb[2] * g.nboxes;
    const int wpb = blockDim.x >> 5, lane = threadIdx.x & 31;
    double tmax = 0.0;
    bool bad = false;
    for (long long row = (long long)blockIdx.x * wpb + (threadIdx.x >> 5); row < nrows; row += (long long)gridDim.x * wpb) {
        long long r = row;
        const int j = (int)(r % g.nb[1]); r /= g.nb[1];
        const int k = (int)(r % g.nb[2]);
        const long long b = r / g.nb[2];
        const double* Ur = U + b * g.bstride + ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0] + g.ng;
        for (int i = lane; i < g.nb[0]; i += 32) {
            const double* Uz = Ur + i;
            double q[5], rinv;
            cons_to_prim(g, ldg(Uz), ldg(Uz + g.cstride), ldg(Uz + 2 * g.cstride), ldg(Uz + 3 * g.cstride),
                         ldg(Uz + 5 * g.cstride), q, rinv);
            const double cs = sqrt(g.gamma * q[4] * rinv);
            const double t = (fabs(q[1]) + cs) * g.dxinv[0] + (fabs(q[2]) + cs) * g.dxinv[1] + (fabs(q[3]) + cs) * g.dxinv[2];
            if (!(t == t)) bad = true;
            if (t > tmax) tmax = t;
        }
    }
    __shared__ unsigned long long sm[8];
    cfl_reduce_finish(g, bad, tmax, red, dtslot, sm);
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
    // a warp takes whole rows (fixed assignment of rows to warps and of zones to lanes: deterministic)
    const long long nrows = (long long)g.nb[1] * g.nb[2] * g.nboxes;
    const int wpb = blockDim.x >> 5, lane = threadIdx.x & 31;
    double hi = 0.0, lo = 0.0;
    for (long long row = (long long)blockIdx.x * wpb + (threadIdx.x >> 5); row < nrows; row += (long long)gridDim.x * wpb) {
        long long r = row;
        const int j = (int)(r % g.nb[1]); r /= g.nb[1];
        const int k = (int)(r % g.nb[2]);
        const long long b = r / g.nb[2];
        const double* Ur = U + b * g.bstride + sc * g.cstride + ((long long)(k + g.ng) * g.nt[1] + (j + g.ng)) * g.nt[0] + g.ng;
        for (int i = lane; i < g.nb[0]; i += 32) dd_add(hi, lo, ldg(Ur + i), 0.0);
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

// ---- halo layers of a sharded MultiFab (paper_2007_05218_b200/sharded.py) ------------------
// A halo of dimension `dim` = the ng layers next to a face, over the FULL padded extent of the other two
// dimensions, of every component of every box on that face: buffer layout [face box][component][t1][t0][layer]
// for dim = 0 and [face box][component][layer][t1][t0] for dim = 1 (t0 = i, t1 = k) and dim = 2 (t0 = i, t1 = j);
// face boxes ordered by their other two box coordinates, lower dimension fastest.  PACK reads the VALID layers
// next to the face, UNPACK writes the GHOST layers beyond it.  One thread per double, grid-stride.
template <bool PACK>
__global__ void __launch_bounds__(256)
k_halo(const __grid_constant__ Geom g, double* __restrict__ U, double* __restrict__ buf, int dim, int side)
{
    const int d0 = dim == 0 ? 1 : 0, d1 = dim == 2 ? 1 : 2;          // the other two dimensions, lower first
    const long long n0 = g.nt[d0], n1 = g.nt[d1], ng = g.ng;
    const long long per_comp = ng * n0 * n1, per_box = per_comp * g.nvar;
    const long long total = per_box * g.NB[d0] * g.NB[d1];
    const int lay0 = PACK ? (side == 0 ? g.ng : g.nb[dim]) : (side == 0 ? 0 : g.nb[dim] + g.ng);
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const long long fb = e / per_box;
        long long r = e - fb * per_box;
        const int c = (int)(r / per_comp);
        r -= c * per_comp;
        int l, t0, t1;
        if (dim == 0) { l = (int)(r % ng); r /= ng; t0 = (int)(r % n0); t1 = (int)(r / n0); }
        else { t0 = (int)(r % n0); r /= n0; t1 = (int)(r % n1); l = (int)(r / n1); }
        int bc[3], pc[3];
        bc[dim] = side == 0 ? 0 : g.NB[dim] - 1;
        bc[d0] = (int)(fb % g.NB[d0]); bc[d1] = (int)(fb / g.NB[d0]);
        pc[dim] = lay0 + l; pc[d0] = t0; pc[d1] = t1;
        const long long b = ((long long)bc[2] * g.NB[1] + bc[1]) * g.NB[0] + bc[0];
        const long long z = (b * g.nvar + c) * g.cstride + ((long long)pc[2] * g.nt[1] + pc[1]) * g.nt[0] + pc[0];
        if (PACK) buf[e] = U[z]; else U[z] = buf[e];
    }
}

}  // namespace hydro
