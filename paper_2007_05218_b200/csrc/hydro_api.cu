// hydro_api.cu -- the C ABI of include/hydro.h: validation, scratch carving and kernel
// launches.  All arithmetic of the path runs in the kernels included below; this file
// only marshals.  sm_100a only; no CPU fallback.
#include "../../include/hydro.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <set>
#include <string>
#include <vector>

#include "ghost_reduce.cuh"
#include "flatten.cuh"
#include "hydro_device.cuh"
#include "sweep_x.cuh"
#include "sweep_xc.cuh"
#include "sweep_yz.cuh"
#include "march_ring.cuh"
#include "march_x.cuh"
#include "ctu.cuh"
#include "amr_fill.cuh"

using namespace hydro;

namespace {

constexpr int RED_BLOCKS = 148 * 8;   // reduction grids: 8 CTAs of 256 threads per SM
constexpr int NS_MAX = 5;             // species per thread in the y/z species kernels: 5 keeps the marching
                                      // kernels at 128 registers = 4 CTAs per SM (measured faster than 7 at 168 / 3)
constexpr int BS = 128;               // threads per CTA of the marching kernels
#ifndef HYDRO_RING_D
#define HYDRO_RING_D 8
#endif
constexpr int RING_D = HYDRO_RING_D;  // depth of the TMA ring of the marching kernels
#ifndef HYDRO_RING_D_SY
#define HYDRO_RING_D_SY 6
#endif
#ifndef HYDRO_RING_D_SZ
#define HYDRO_RING_D_SZ 6
#endif
// depth of the ring of the species kernels, y sweep (not FINAL) and z sweep (FINAL)
constexpr int ring_ds(bool final_) { return final_ ? HYDRO_RING_D_SZ : HYDRO_RING_D_SY; }
#ifndef HYDRO_XM_D
#define HYDRO_XM_D 3
#endif
constexpr int XM_D = HYDRO_XM_D;      // depth of the ring of the x marching kernels (a step is four zones)
#ifndef HYDRO_XS_MODE
#define HYDRO_XS_MODE 1               // x species kernels: 1 = one species per thread, one thread set per species of the
#endif                                // group; 0 = one thread per row marches the whole group
#ifndef HYDRO_XS_ROWS
#define HYDRO_XS_ROWS 32
#endif
constexpr int XS_ROWS = HYDRO_XS_MODE ? HYDRO_XS_ROWS : XBS;   // rows per CTA of the x species kernels

constexpr int DT_SLOTS = 1024;        // (dt, max t) pairs kept on the device: one per step of a hydro_step chunk
constexpr int PROF_EVENTS = 8192;     // event pool of hydro_profile (two per recorded launch)

thread_local std::string g_init_error = "";

struct Carve {
    size_t lacc, frho, part, totals, red, dtslot, flat, zc, total;
};

// tuning switches, read from the environment ONCE per hydro_init (include/hydro.h lists them)
struct Knobs {
    int ring, seglen, nsmax, fuse_dt, split_ghosts, fill_monolithic, xmarch, species_one_launch, xchunk;
};

int env_int(const char *name, int dflt)
{
    const char *e = getenv(name);
    return (e && *e) ? atoi(e) : dflt;
}

// makes the handle's device current for the duration of an entry point
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

}  // namespace

struct hydro_ctx {
    hydro_params p;
    Geom g;
    double *U[2];
    char *scratch;
    Carve cv;
    cudaStream_t stream;
    int device;               // the device the caller's buffers live on; made current by every entry point
    double *pinned;           // max(nflux, 2 * DT_SLOTS) doubles of pinned host memory
    long long launches;
    Knobs kn;
    std::set<const void *> configured;   // kernels whose dynamic shared-memory limit is set on `device`
    int seglen[3];
    int ns_max;
    bool use_ring;            // TMA-ring marching kernels usable for this geometry
    bool split_ghosts;        // hydro_step: x ghost images written by the z sweeps + ghost-row copies
    bool fuse_dt;             // hydro_step: the stage-1 z hydro sweep also reduces the next step's dt
    CUtensorMap maps[2][2][7]; // [state][DIR-1][components per box]: TMA views of the states for the ring kernels
    CUtensorMap fmaps[2];      // [DIR-1]: TMA views of the flattening-coefficient array (flatten == 1)
    bool external;             // some face is HYDRO_BC_EXTERNAL (sharded MultiFab)
    bool use_xmarch;           // x sweep by the marching kernels of march_x.cuh (else k_sweep_xc / k_sweep_x)
    bool use_xchunk;           // x sweep by the chunk-lane kernel of sweep_xc.cuh (else k_sweep_x)
    CUtensorMap xmaps[2][6];   // [state][components per box]: {4 zones, 128 rows} views for the x hydro marching kernel
    CUtensorMap xsmaps[2][6];  // the same with XS_ROWS rows per box, for the x species marching kernels
    CUtensorMap fxmap;         // {4 columns, XS_ROWS rows} view of the face mass-flux array in its x layout (rows of nb0 + 4)
    std::string err;
    // optional per-launch timing (hydro_profile): event pairs from a pool created by hydro_profile(1);
    // nothing is allocated while launches are recorded (when the pool is used up, recording stops)
    bool profiling;
    std::vector<cudaEvent_t> pool;
    size_t pool_used;
    struct Ev { int a, b, klass; };
    std::vector<Ev> events;
    int pending;
};

namespace {

bool make_geom(const hydro_params *p, Geom &g, std::string &why)
{
    if (!p) { why = "null params"; return false; }
    if (p->ng < 3) { why = "ng must be >= 3"; return false; }
    if (p->nspec < 0) { why = "nspec must be >= 0"; return false; }
    if (!(p->gamma > 1.0)) { why = "gamma must be > 1"; return false; }
    if (p->flatten != 0 && p->flatten != 1) { why = "flatten must be 0 or 1"; return false; }
    if (p->flatten == 1 && p->ng < 4) { why = "flattening needs ng >= 4"; return false; }
    if (p->evolve_eint != 0 && p->evolve_eint != 1) { why = "evolve_eint must be 0 or 1"; return false; }
    std::memset(&g, 0, sizeof(g));
    g.flatten = p->flatten;
    g.evolve = p->evolve_eint;
    g.ng = p->ng; g.nspec = p->nspec; g.nvar = 6 + p->nspec; g.nflux = 5 + p->nspec;
    g.nboxes = 1;
    double dx[3];
    for (int d = 0; d < 3; ++d) {
        if (p->ndom[d] <= 0 || p->nbox[d] <= 0 || p->ndom[d] % p->nbox[d] != 0) {
            why = "nbox must be positive and divide ndom"; return false;
        }
        if (p->bc_lo[d] < 0 || p->bc_lo[d] > 3 || p->bc_hi[d] < 0 || p->bc_hi[d] > 3) {
            why = "bc must be 0, 1, 2 or 3"; return false;
        }
        if ((p->bc_lo[d] == HYDRO_BC_PERIODIC) != (p->bc_hi[d] == HYDRO_BC_PERIODIC)) {
            why = "periodic must be set on both sides of a dimension"; return false;
        }
        if ((p->bc_lo[d] == HYDRO_BC_REFLECT || p->bc_hi[d] == HYDRO_BC_REFLECT) && p->ng > p->ndom[d]) {
            why = "ng must not exceed ndom across a reflecting boundary"; return false;
        }
        if (!(p->prob_hi[d] > p->prob_lo[d])) { why = "prob_hi must exceed prob_lo"; return false; }
        g.nb[d] = p->nbox[d]; g.nt[d] = p->nbox[d] + 2 * p->ng; g.NB[d] = p->ndom[d] / p->nbox[d];
        g.ndom[d] = p->ndom[d]; g.bc_lo[d] = p->bc_lo[d]; g.bc_hi[d] = p->bc_hi[d];
        g.nboxes *= g.NB[d];
        if (!(p->dx[d] >= 0.0) || std::isinf(p->dx[d])) { why = "dx must be 0 (derive it from the extent) or a positive finite zone width"; return false; }
        dx[d] = p->dx[d] > 0.0 ? p->dx[d] : (p->prob_hi[d] - p->prob_lo[d]) / p->ndom[d];
        g.dxinv[d] = 1.0 / dx[d];
        g.grav[d] = p->grav[d];
    }
    if (g.nboxes > (1 << 20)) { why = "more than 2^20 boxes"; return false; }
    g.cstride = (long long)g.nt[0] * g.nt[1] * g.nt[2];
    g.bstride = g.cstride * g.nvar;
    g.lcstride = (long long)g.nb[0] * g.nb[1] * g.nb[2];
    // accumulator components per zone: the NFLUX flux differences; with O11 three more (flux of rho*e,
    // div(u_face), rho*E - K of the new state)
    g.lbstride = g.lcstride * (g.nflux + (p->evolve_eint ? 3 : 0));
    // one face mass-flux array serves the three sweeps in turn: y and z faces as (nb+1)-extended arrays, x faces
    // in rows of nb0 + 4 (march_x.cuh)
    g.fbstride = (long long)(g.nb[0] + 1) * (g.nb[1] + 1) * (g.nb[2] + 1);
    const long long fx = (long long)(g.nb[0] + 4) * g.nb[1] * g.nb[2];
    if (fx > g.fbstride) g.fbstride = fx;
    g.fbstride = (g.fbstride + 3) & ~3LL;             // keep every box's face array 32-byte aligned
    g.gamma = p->gamma; g.gm1 = p->gamma - 1.0; g.gm1inv = 1.0 / (p->gamma - 1.0);
    g.small_dens = p->small_dens; g.small_pres = p->small_pres;
    g.floor_rhoe = p->small_pres * g.gm1inv;
    g.cfl = p->cfl;
    g.vol = dx[0] * dx[1] * dx[2];
    g.has_grav = !(p->grav[0] == 0.0 && p->grav[1] == 0.0 && p->grav[2] == 0.0);
    return true;
}

size_t up256(size_t x) { return (x + 255) & ~(size_t)255; }

Carve carve(const Geom &g)
{
    Carve c;
    size_t off = 0;
    c.lacc = off;   off += up256((size_t)g.lbstride * g.nboxes * 8);
    c.frho = off;   off += up256((size_t)g.fbstride * g.nboxes * 8);
    c.part = off;   off += up256((size_t)g.nflux * RED_BLOCKS * 2 * 8);
    c.totals = off; off += up256((size_t)g.nflux * 8);
    c.red = off;    off += 256;
    c.dtslot = off; off += up256((size_t)DT_SLOTS * 16);
    c.flat = off;   if (g.flatten) off += up256((size_t)g.cstride * g.nboxes * 8);   // O10 coefficients
    c.zc = off;     if (g.flatten) off += up256((size_t)g.cstride * g.nboxes * 3 * 8); // O10 chi*z per direction
    c.total = off;
    return c;
}

// TMA view of one state for the ring kernels of direction dir (1: y march, 2: z march): a 5-D
// tensor (i, j, k, component, box) with a box of W zones x R rows x nc components, R counted
// along the transverse dimension (k for the y march, j for the z march).
bool make_ring_map(CUtensorMap *out, double *U, const Geom &g, int dir, int nc, std::string &why,
                   int ncomp_total = -1, long long box_stride = -1)
{
    if (ncomp_total < 0) ncomp_total = g.nvar;
    if (box_stride < 0) box_stride = g.bstride;
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
            why = "cuTensorMapEncodeTiled is not available from the driver";
            return false;
        }
        encode = (encode_fn)fn;
    }
    const int W = g.nb[0] < BS ? g.nb[0] : BS, R = BS / W;
    cuuint64_t dims[5] = {(cuuint64_t)g.nt[0], (cuuint64_t)g.nt[1], (cuuint64_t)g.nt[2], (cuuint64_t)ncomp_total,
                          (cuuint64_t)g.nboxes};
    cuuint64_t strides[4] = {(cuuint64_t)g.nt[0] * 8, (cuuint64_t)g.nt[0] * g.nt[1] * 8, (cuuint64_t)g.cstride * 8,
                             (cuuint64_t)box_stride * 8};
    cuuint32_t box[5] = {(cuuint32_t)W, dir == 2 ? (cuuint32_t)R : 1u, dir == 1 ? (cuuint32_t)R : 1u, (cuuint32_t)nc, 1u};
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, U, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { why = "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")"; return false; }
    return true;
}

// TMA view of one state for the x marching kernels: the same 5-D tensor with a box of XC zones x RJ rows (j) x
// RK rows (k) x nc components; thread t of the CTA reads row t of the box.
bool make_xmarch_map(CUtensorMap *out, double *U, const Geom &g, int nc, int rows, std::string &why)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
        why = "cuTensorMapEncodeTiled is not available from the driver";
        return false;
    }
    const int RJ = g.nb[1] < rows ? g.nb[1] : rows, RK = rows / RJ;
    cuuint64_t dims[5] = {(cuuint64_t)g.nt[0], (cuuint64_t)g.nt[1], (cuuint64_t)g.nt[2], (cuuint64_t)g.nvar,
                          (cuuint64_t)g.nboxes};
    cuuint64_t strides[4] = {(cuuint64_t)g.nt[0] * 8, (cuuint64_t)g.nt[0] * g.nt[1] * 8, (cuuint64_t)g.cstride * 8,
                             (cuuint64_t)g.bstride * 8};
    cuuint32_t box[5] = {(cuuint32_t)XC, (cuuint32_t)RJ, (cuuint32_t)RK, (cuuint32_t)nc, 1u};
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
#ifndef HYDRO_XM_PROMO
#define HYDRO_XM_PROMO CU_TENSOR_MAP_L2_PROMOTION_L2_256B
#endif
    CUresult r = ((encode_fn)fn)(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, U, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                 CU_TENSOR_MAP_SWIZZLE_NONE, HYDRO_XM_PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { why = "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")"; return false; }
    return true;
}

// TMA view of the face mass-flux array in the layout of the x marching kernels: rows of nb0 + 4 columns,
// [box][k][j][column]; box = XC columns x RJ x RK rows.
bool make_fx_map(CUtensorMap *out, double *FX, const Geom &g, int rows, std::string &why)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
        why = "cuTensorMapEncodeTiled is not available from the driver";
        return false;
    }
    const int RJ = g.nb[1] < rows ? g.nb[1] : rows, RK = rows / RJ;
    const cuuint64_t pitch = (cuuint64_t)(g.nb[0] + 4);
    cuuint64_t dims[4] = {pitch, (cuuint64_t)g.nb[1], (cuuint64_t)g.nb[2], (cuuint64_t)g.nboxes};
    cuuint64_t strides[3] = {pitch * 8, pitch * g.nb[1] * 8, (cuuint64_t)g.fbstride * 8};
    cuuint32_t box[4] = {(cuuint32_t)XC, (cuuint32_t)RJ, (cuuint32_t)RK, 1u};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = ((encode_fn)fn)(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, FX, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                 CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { why = "cuTensorMapEncodeTiled (FX) failed (" + std::to_string((int)r) + ")"; return false; }
    return true;
}

int fail(hydro_handle h, int code, const std::string &msg)
{
    if (h) h->err = msg; else g_init_error = msg;
    return code;
}

// kernel classes of hydro_profile_read
enum { K_GHOST = 0, K_DT, K_SWEEP_X, K_HYDRO_Y, K_SPECIES_Y, K_HYDRO_Z, K_SPECIES_Z, K_TOTALS, K_FLATTEN, K_CTU, K_NCLASS };

void prof_begin(hydro_handle h)
{
    h->pending = -1;
    if (!h->profiling || h->pool_used + 2 > h->pool.size()) return;
    h->pending = (int)h->pool_used;
    cudaEventRecord(h->pool[h->pending], h->stream);
}

int check_launch(hydro_handle h, const char *what, int klass)
{
    cudaError_t e = cudaGetLastError();
    h->launches++;
    if (h->profiling && h->pending >= 0 && e == cudaSuccess) {
        hydro_ctx::Ev ev;
        ev.a = h->pending; ev.b = h->pending + 1; ev.klass = klass;
        cudaEventRecord(h->pool[ev.b], h->stream);
        h->pool_used += 2;
        h->events.push_back(ev);          // capacity reserved by hydro_profile(1)
    }
    h->pending = -1;
    if (e != cudaSuccess) return fail(h, HYDRO_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
    return HYDRO_OK;
}

int pick_seglen(const Geom &g, int dir, int forced)
{
    if (forced > 0) return forced < g.nb[dir] ? forced : g.nb[dir];
    // enough pencils to fill 148 SMs several times over? then march the whole box
    const int T = dir == 1 ? 2 : 1;
    long long pencils = (long long)g.nb[0] * g.nb[T] * g.nboxes;
    int nseg = 1;
    while (pencils * nseg < 148LL * 1024 && g.nb[dir] / (nseg * 2) >= 16) nseg *= 2;
    return (g.nb[dir] + nseg - 1) / nseg;
}

// The ring kernels need more than the default 48 KB of dynamic shared memory.  The limit is a per-device
// attribute of a kernel, so it is set once per (handle, kernel): a handle lives on one device.
template <typename K>
void set_smem(hydro_handle h, K kernel, size_t bytes)
{
    if (h->configured.count((const void *)kernel)) return;
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    h->configured.insert((const void *)kernel);
}

// bytes of the accumulator prefetch ring of the species march kernels (march_ring.cuh, RING_LPD)
constexpr size_t lring_bytes(int n, bool final_, int stage)
{
    const int lpd = final_ ? RING_LPD_Z : RING_LPD_Y;
    return lpd ? (size_t)(lpd + 1) * n * ((final_ && stage == 1) ? 2 : 1) * BS * 8 : 0;
}

template <int DIR, bool FINAL, int STAGE, int N, bool FLAT>
void launch_species_ring_n(hydro_handle h, const SweepArgs &a, dim3 grid, const RingMaps &tm)
{
    constexpr int DS = ring_ds(FINAL);
    const size_t sm = (size_t)DS * (1 + N + (FLAT ? 1 : 0)) * BS * 8 + DS * 8 + lring_bytes(N, FINAL, STAGE);
    auto kern = k_march_species<DIR, FINAL, STAGE, N, BS, DS, FLAT>;
    set_smem(h, kern, sm);
    kern<<<grid, BS, sm, h->stream>>>(h->g, a, tm);
}

template <int DIR, bool FINAL, int STAGE, bool FLAT>
void launch_energy_ring(hydro_handle h, const SweepArgs &a, dim3 grid, const RingMaps &tm)
{
    constexpr int DS = ring_ds(FINAL);
    const size_t sm = (size_t)DS * (2 + (FLAT ? 1 : 0)) * BS * 8 + DS * 8 + lring_bytes(1, FINAL, STAGE);
    auto kern = k_march_species<DIR, FINAL, STAGE, 1, BS, DS, FLAT, FINAL>;   // ENERGY terms only in the FINAL sweep
    set_smem(h, kern, sm);
    kern<<<grid, BS, sm, h->stream>>>(h->g, a, tm);
}

// The three launchers below pick a kernel instance by the species per thread; they return false (and launch
// nothing) when no instance exists for that count, which the caller turns into HYDRO_EINVAL.
template <int DIR, bool FINAL, int STAGE>
bool launch_species_ring(hydro_handle h, const SweepArgs &a, int ns, dim3 grid, int state)
{
    RingMaps tm;
    tm.a = h->maps[state][DIR - 1][1];
    tm.b = h->maps[state][DIR - 1][ns];
    tm.f = h->fmaps[DIR - 1];
    const bool flat = h->g.flatten != 0;
    switch (ns) {
#define CASE(N) case N: \
        if (flat) launch_species_ring_n<DIR, FINAL, STAGE, N, true>(h, a, grid, tm); \
        else launch_species_ring_n<DIR, FINAL, STAGE, N, false>(h, a, grid, tm); \
        break;
        CASE(1) CASE(2) CASE(3) CASE(4) CASE(5)
#undef CASE
        default: return false;
    }
    return true;
}

// all species groups of a direction in ONE launch (k_march_species_groups): nsa = species of the larger groups, >= 2
// (with one species per group there is no rho / F_rho row to share that a plain launch per group would not also
// find in L2, and no instance is built for it: sweep_dir launches those groups one by one)
template <int DIR, bool FINAL, int STAGE>
bool launch_species_groups(hydro_handle h, const SweepArgs &a, int nsa, dim3 grid, int state)
{
    RingMaps tm;
    tm.a = h->maps[state][DIR - 1][1];
    tm.b = h->maps[state][DIR - 1][nsa];
    tm.b2 = h->maps[state][DIR - 1][nsa > 1 ? nsa - 1 : 1];
    tm.f = h->fmaps[DIR - 1];
    const bool flat = h->g.flatten != 0;
    constexpr int DS = ring_ds(FINAL);
    const size_t sm = (size_t)DS * (1 + nsa + (flat ? 1 : 0)) * BS * 8 + DS * 8 + lring_bytes(nsa, FINAL, STAGE);
    grid.x *= a.ngroups;
    switch (nsa) {
#define CASE(N) case N: \
        if (flat) { auto kern = k_march_species_groups<DIR, FINAL, STAGE, N, BS, DS, true>; set_smem(h, kern, sm); \
                    kern<<<grid, BS, sm, h->stream>>>(h->g, a, tm); } \
        else { auto kern = k_march_species_groups<DIR, FINAL, STAGE, N, BS, DS, false>; set_smem(h, kern, sm); \
               kern<<<grid, BS, sm, h->stream>>>(h->g, a, tm); } \
        break;
        CASE(2) CASE(3) CASE(4) CASE(5)
#undef CASE
        default: return false;
    }
    return true;
}

template <int DIR, bool FINAL, int STAGE, bool FLAT, bool EVOLVE>
void launch_hydro_ring(hydro_handle h, const SweepArgs &a, dim3 grid, int state)
{
    constexpr int NROW = (FINAL ? 6 : 5) + (FLAT ? 1 : 0);
    const size_t sm = (size_t)RING_D * NROW * BS * 8 + RING_D * 8;
    auto kern = k_march_hydro<DIR, FINAL, STAGE, BS, RING_D, FLAT, EVOLVE>;
    set_smem(h, kern, sm);
    RingMaps tm;
    tm.a = h->maps[state][DIR - 1][FINAL ? 6 : 4];
    tm.b = h->maps[state][DIR - 1][1];
    tm.f = h->fmaps[DIR - 1];
    kern<<<grid, BS, sm, h->stream>>>(h->g, a, tm);
}

template <int DIR, bool FINAL, int STAGE>
bool launch_species(hydro_handle h, const SweepArgs &a, int ns, dim3 grid)
{
    switch (ns) {
#define CASE(N) case N: k_sweep_species<DIR, FINAL, STAGE, N, BS><<<grid, BS, 0, h->stream>>>(h->g, a); break;
        CASE(1) CASE(2) CASE(3) CASE(4) CASE(5)
#undef CASE
        default: return false;
    }
    return true;
}

template <int DIR, bool FINAL, int STAGE>
int sweep_dir(hydro_handle h, SweepArgs a, int state)
{
    const Geom &g = h->g;
    constexpr int T = DIR == 1 ? 2 : 1;
    a.seglen = h->seglen[DIR];
    const int nseg = (g.nb[DIR] + a.seglen - 1) / a.seglen;
    dim3 grid((g.nb[0] * g.nb[T] + BS - 1) / BS, nseg, 1);
    const bool ring = h->use_ring;
    if (ring) {   // CTA = R row segments of W zones; rows may not fill the last CTA
        const int W = g.nb[0] < BS ? g.nb[0] : BS, R = BS / W;
        grid.x = (g.nb[T] * (g.nb[0] / W) + R - 1) / R;
    }
    if ((long long)grid.x * g.nboxes > 2147483647LL || nseg > 65535) return fail(h, HYDRO_EINVAL, "sweep grid too large");
    grid.x *= g.nboxes;   // the box index rides in blockIdx.x
    prof_begin(h);
    if (ring) {
        if (g.flatten && g.evolve) launch_hydro_ring<DIR, FINAL, STAGE, true, true>(h, a, grid, state);
        else if (g.flatten) launch_hydro_ring<DIR, FINAL, STAGE, true, false>(h, a, grid, state);
        else if (g.evolve) launch_hydro_ring<DIR, FINAL, STAGE, false, true>(h, a, grid, state);
        else launch_hydro_ring<DIR, FINAL, STAGE, false, false>(h, a, grid, state);
    } else if (g.evolve)
        k_sweep_hydro<DIR, FINAL, STAGE, BS, true><<<grid, BS, 0, h->stream>>>(g, a);
    else
        k_sweep_hydro<DIR, FINAL, STAGE, BS, false><<<grid, BS, 0, h->stream>>>(g, a);
    int rc = check_launch(h, "k_sweep_hydro", DIR == 1 ? K_HYDRO_Y : K_HYDRO_Z);
    if (rc) return rc;
    const int ngroups = g.nspec > 0 ? (g.nspec + h->ns_max - 1) / h->ns_max : 0;
    const int nsa = ngroups > 0 ? (g.nspec + ngroups - 1) / ngroups : 0;   // species of the larger groups
    if (ring && ngroups >= 2 && nsa >= 2 && (h->kn.species_one_launch & (DIR == 1 ? 1 : 2)) &&
        (long long)grid.x * ngroups <= 2147483647LL) {
        // every group in one launch: sibling CTAs share their rho and F_rho rows through L2
        const int rem = g.nspec % ngroups;
        a.sbase = 0;
        a.lacc_shift = 0;
        a.ngroups = ngroups;
        a.n_hi = rem > 0 ? rem : ngroups;
        prof_begin(h);
        if (!launch_species_groups<DIR, FINAL, STAGE>(h, a, nsa, grid, state))
            return fail(h, HYDRO_EINVAL, "no k_march_species_groups instance for " + std::to_string(nsa) + " species per thread");
        if ((rc = check_launch(h, "k_march_species_groups", DIR == 1 ? K_SPECIES_Y : K_SPECIES_Z))) return rc;
    } else if (g.nspec > 0) {
        const int base = g.nspec / ngroups, rem = g.nspec % ngroups;
        int s0 = 0;
        for (int gr = 0; gr < ngroups; ++gr) {
            const int ns = base + (gr < rem ? 1 : 0);
            a.sbase = s0;
            a.lacc_shift = 0;
            prof_begin(h);
            if (!(ring ? launch_species_ring<DIR, FINAL, STAGE>(h, a, ns, grid, state)
                       : launch_species<DIR, FINAL, STAGE>(h, a, ns, grid)))
                return fail(h, HYDRO_EINVAL, "no species sweep instance for " + std::to_string(ns) + " species per thread");
            if ((rc = check_launch(h, "k_sweep_species", DIR == 1 ? K_SPECIES_Y : K_SPECIES_Z))) return rc;
            s0 += ns;
        }
    }
    if (g.evolve) {   // O11: e = rho*e / rho as one more upwinded scalar (state component 5, accumulator slot nflux)
        a.sbase = -1;
        a.lacc_shift = g.nflux - 4;
        prof_begin(h);
        RingMaps tm;
        tm.a = h->maps[state][DIR - 1][1];
        tm.b = h->maps[state][DIR - 1][1];
        tm.f = h->fmaps[DIR - 1];
        if (!ring) k_sweep_species<DIR, FINAL, STAGE, 1, BS, FINAL><<<grid, BS, 0, h->stream>>>(g, a);
        else if (g.flatten) launch_energy_ring<DIR, FINAL, STAGE, true>(h, a, grid, tm);
        else launch_energy_ring<DIR, FINAL, STAGE, false>(h, a, grid, tm);
        if ((rc = check_launch(h, "k_march_species<energy>", DIR == 1 ? K_SPECIES_Y : K_SPECIES_Z))) return rc;
    }
    return HYDRO_OK;
}

template <int N>
void launch_xmarch_species_n(hydro_handle h, const XArgs &xa, dim3 grid, const XMaps &tm)
{
    const size_t sm = (size_t)XM_D * (2 + N) * XS_ROWS * XC * 8 + (size_t)2 * XS_ROWS * XC * 8 + XM_D * 8;
#if HYDRO_XS_MODE
    auto kern = k_xmarch_species<1, N, XS_ROWS, XM_D>;
    const int threads = XS_ROWS * N;
#else
    auto kern = k_xmarch_species<N, 1, XS_ROWS, XM_D>;
    const int threads = XS_ROWS;
#endif
    set_smem(h, kern, sm);
    kern<<<grid, threads, sm, h->stream>>>(h->g, xa, tm);
}

// x sweep of a stage by the marching kernels: hydro launch (writes the accumulator rows of the five hydro
// variables and F_rho,x), then one species launch per group
int xmarch_stage(hydro_handle h, int state, double *Lacc, double *FX)
{
    const Geom &g = h->g;
    const int RJ = g.nb[1] < XBS ? g.nb[1] : XBS, RK = XBS / RJ;
    const long long tiles = (long long)(g.nb[1] / RJ) * ((g.nb[2] + RK - 1) / RK);
    if (tiles * g.nboxes > 2147483647LL) return fail(h, HYDRO_EINVAL, "x-march grid too large");
    const dim3 grid((unsigned)(tiles * g.nboxes), 1, 1);
    XArgs xa;
    xa.Lacc = Lacc; xa.FX = FX; xa.sbase = 0;
    XMaps tm;
    {
        const size_t sm = (size_t)XM_D * 5 * XBS * XC * 8 + XM_D * 8;
        auto kern = k_xmarch_hydro<XM_D>;
        set_smem(h, kern, sm);
        tm.a = h->xmaps[state][4];
        tm.b = h->xmaps[state][1];
        prof_begin(h);
        kern<<<grid, XBS, sm, h->stream>>>(g, xa, tm);
        int rc = check_launch(h, "k_xmarch_hydro", K_SWEEP_X);
        if (rc) return rc;
    }
    if (g.nspec > 0) {
        const int SJ = g.nb[1] < XS_ROWS ? g.nb[1] : XS_ROWS, SK = XS_ROWS / SJ;
        const dim3 sgrid((unsigned)((long long)(g.nb[1] / SJ) * ((g.nb[2] + SK - 1) / SK) * g.nboxes), 1, 1);
        const int ngroups = (g.nspec + h->ns_max - 1) / h->ns_max;
        const int base = g.nspec / ngroups, rem = g.nspec % ngroups;
        int s0 = 0;
        for (int gr = 0; gr < ngroups; ++gr) {
            const int ns = base + (gr < rem ? 1 : 0);
            xa.sbase = s0;
            tm.a = h->xsmaps[state][1];
            tm.b = h->xsmaps[state][ns];
            tm.fx = h->fxmap;
            prof_begin(h);
            switch (ns) {
                case 1: launch_xmarch_species_n<1>(h, xa, sgrid, tm); break;
                case 2: launch_xmarch_species_n<2>(h, xa, sgrid, tm); break;
                case 3: launch_xmarch_species_n<3>(h, xa, sgrid, tm); break;
                case 4: launch_xmarch_species_n<4>(h, xa, sgrid, tm); break;
                case 5: launch_xmarch_species_n<5>(h, xa, sgrid, tm); break;
                default: return fail(h, HYDRO_EINVAL, "no k_xmarch_species instance for " + std::to_string(ns) + " species per thread");
            }
            int rc = check_launch(h, "k_xmarch_species", K_SWEEP_X);
            if (rc) return rc;
            s0 += ns;
        }
    }
    return HYDRO_OK;
}

int advance_stage_impl(hydro_handle h, int stage, double dt, const double *dt_dev, bool xends = false,
                       double *dt_next = nullptr)
{
    const Geom &g = h->g;
    SweepArgs a;
    std::memset(&a, 0, sizeof(a));
    a.Us = h->U[stage];
    a.Ubase = h->U[0];
    a.Uout = h->U[stage == 0 ? 1 : 0];
    a.Lacc = (double *)(h->scratch + h->cv.lacc);
    a.Frho = (double *)(h->scratch + h->cv.frho);
    a.dt = dt;
    a.dt_dev = dt_dev;
    a.xends = (xends && h->use_ring) ? 1 : 0;
    a.red = (unsigned long long *)(h->scratch + h->cv.red);
    a.dt_next = (stage == 1 && h->use_ring) ? dt_next : nullptr;
    a.FL = nullptr;
    if (g.flatten) {   // O10: flattening coefficients of the stage state (ghosts are filled) before any sweep
        a.FL = (const double *)(h->scratch + h->cv.flat);
        auto fgrid = [&](int lo) {
            return dim3((unsigned)(((g.nb[0] - 2 * lo + FLT_BX - 1) / FLT_BX) * g.nboxes), (g.nb[1] - 2 * lo + FLT_BY - 1) / FLT_BY,
                        (g.nb[2] - 2 * lo + FLT_BZ - 1) / FLT_BZ);
        };
        if ((long long)((g.nb[0] + 4 + FLT_BX - 1) / FLT_BX) * g.nboxes > 2147483647LL || g.nb[1] + 4 > 65535 * FLT_BY ||
            g.nb[2] + 4 > 65535 * FLT_BZ)
            return fail(h, HYDRO_EINVAL, "flattening grid too large");
        double *ZC = (double *)(h->scratch + h->cv.zc);
        prof_begin(h);
        k_flatten_zc<<<fgrid(-2), dim3(FLT_BX, FLT_BY, FLT_BZ), 0, h->stream>>>(g, a.Us, ZC);
        int rc0 = check_launch(h, "k_flatten_zc", K_FLATTEN);
        if (rc0) return rc0;
        prof_begin(h);
        k_flatten<<<fgrid(-1), dim3(FLT_BX, FLT_BY, FLT_BZ), 0, h->stream>>>(g, a.Us, ZC, (double *)(h->scratch + h->cv.flat));
        int rc = check_launch(h, "k_flatten", K_FLATTEN);
        if (rc) return rc;
    }
    if (h->use_xmarch) {   // x sweep: a thread per row, marching (march_x.cuh)
        int rc = xmarch_stage(h, stage, a.Lacc, a.Frho);
        if (rc) return rc;
    } else if (h->use_xchunk) {   // x sweep: a lane per 4-zone chunk of the flattened valid rows (sweep_xc.cuh)
        const long long T = (long long)g.nb[1] * g.nb[2] * (g.nt[0] / 4);
        const long long warps = (T + XC_LANES - 1) / XC_LANES;
        const unsigned gy = g.nboxes < 32768 ? g.nboxes : 32768, gz = (g.nboxes + gy - 1) / gy;
        const dim3 xg((unsigned)((warps + XC_WARPS - 1) / XC_WARPS), gy, gz);
        prof_begin(h);
        if (g.flatten && g.evolve) k_sweep_xc<true, true><<<xg, XC_WARPS * 32, 0, h->stream>>>(g, a.Us, a.Lacc, a.FL);
        else if (g.flatten) k_sweep_xc<true, false><<<xg, XC_WARPS * 32, 0, h->stream>>>(g, a.Us, a.Lacc, a.FL);
        else if (g.evolve) k_sweep_xc<false, true><<<xg, XC_WARPS * 32, 0, h->stream>>>(g, a.Us, a.Lacc, nullptr);
        else k_sweep_xc<false, false><<<xg, XC_WARPS * 32, 0, h->stream>>>(g, a.Us, a.Lacc, nullptr);
        int rc = check_launch(h, "k_sweep_xc", K_SWEEP_X);
        if (rc) return rc;
    } else {   // x sweep: one warp per 26-zone chunk of a row
        constexpr int WARPS = 4;
        const int nchunk = (g.nb[0] + XW_VALID - 1) / XW_VALID;
        const bool fold = g.nboxes > 65535;             // the box index in blockIdx.z when it fits
        const long long gx = (long long)nchunk * ((g.nb[1] + WARPS - 1) / WARPS) * (fold ? g.nboxes : 1);
        if (gx > 2147483647LL || g.nb[2] > 65535) return fail(h, HYDRO_EINVAL, "x-sweep grid too large");
        prof_begin(h);
        const dim3 xg((unsigned)gx, g.nb[2], fold ? 1 : g.nboxes);
#define XSWEEP(FL, EV, PTR) \
        do { if (fold) k_sweep_x<WARPS, FL, EV, true><<<xg, WARPS * 32, 0, h->stream>>>(g, a.Us, a.Lacc, PTR); \
             else k_sweep_x<WARPS, FL, EV, false><<<xg, WARPS * 32, 0, h->stream>>>(g, a.Us, a.Lacc, PTR); } while (0)
        if (g.flatten && g.evolve) XSWEEP(true, true, a.FL);
        else if (g.flatten) XSWEEP(true, false, a.FL);
        else if (g.evolve) XSWEEP(false, true, nullptr);
        else XSWEEP(false, false, nullptr);
#undef XSWEEP
        int rc = check_launch(h, "k_sweep_x", K_SWEEP_X);
        if (rc) return rc;
    }
    int rc = sweep_dir<1, false, 0>(h, a, stage);
    if (rc) return rc;
    if (stage == 0) return sweep_dir<2, true, 0>(h, a, stage);
    return sweep_dir<2, true, 1>(h, a, stage);
}

int fill_ghost_rows_impl(hydro_handle h, int which);

int fill_ghosts_impl(hydro_handle h, int which)
{
    const Geom &g = h->g;
    if (g.nvar > 65535 || (long long)g.nt[2] * g.nboxes > 2147483647LL)
        return fail(h, HYDRO_EINVAL, "ghost-fill grid too large");
    if (h->split_ghosts && g.nb[2] <= 65535 && !h->kn.fill_monolithic) {
        // split form (bit-identical, less index arithmetic and no 32-byte row-end gathers in the plane
        // kernel): x ghost zones of the valid rows, then the ghost rows as whole-row copies
        prof_begin(h);
        k_fill_xends<<<dim3((unsigned)(((g.nb[1] * 2 * g.ng + 255) / 256) * g.nboxes), g.nb[2], g.nvar), 256, 0, h->stream>>>(g, h->U[which]);
        int rc = check_launch(h, "k_fill_xends", K_GHOST);
        if (rc) return rc;
        return fill_ghost_rows_impl(h, which);
    }
    prof_begin(h);
    k_fill_ghosts<<<dim3((unsigned)(g.nt[2] * g.nboxes), g.nvar, 1), 256, 0, h->stream>>>(g, h->U[which]);
    return check_launch(h, "k_fill_ghosts", K_GHOST);
}

// ghost rows of state `which` (the part of O1 left when the z sweeps wrote the x images)
int fill_ghost_rows_impl(hydro_handle h, int which)
{
    const Geom &g = h->g;
    const int nrows = g.nt[2] * g.nt[1] - g.nb[2] * g.nb[1];
    prof_begin(h);
    k_fill_ghost_rows<<<dim3((unsigned)(((nrows + GR_ROWS - 1) / GR_ROWS) * g.nboxes), g.nvar, 1), 256, 0, h->stream>>>(g, h->U[which]);
    return check_launch(h, "k_fill_ghost_rows", K_GHOST);
}

// (dt, max t) slots on the device, one per step of a hydro_step chunk: the dt of step s+1, reduced by the
// last hydro kernel of step s, must not overwrite the dt the rest of step s still reads, and the host
// validates every step's max t after the chunk
double *dt_slot(hydro_handle h, int slot) { return (double *)(h->scratch + h->cv.dtslot) + 2 * (slot % DT_SLOTS); }

int launch_dt(hydro_handle h, int slot = 0, int which = 0)
{
    const long long nrows = (long long)h->g.nb[1] * h->g.nb[2] * h->g.nboxes;
    long long blocks = (nrows + 7) / 8;            // 8 warps per block, one row per warp and trip
    if (blocks > RED_BLOCKS) blocks = RED_BLOCKS;
    prof_begin(h);
    k_estimate_dt<<<(unsigned)blocks, 256, 0, h->stream>>>(h->g, h->U[which],
                                                           (unsigned long long *)(h->scratch + h->cv.red),
                                                           dt_slot(h, slot));
    return check_launch(h, "k_estimate_dt", K_DT);
}

// read back slots 0..n-1, validate every max t, copy the dts to dt_host (may be NULL)
int read_dts(hydro_handle h, double *dt_host, int n)
{
    cudaError_t e = cudaMemcpyAsync(h->pinned, dt_slot(h, 0), (size_t)n * 16, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(h, HYDRO_ECUDA, std::string("dt read-back: ") + cudaGetErrorString(e));
    for (int s = 0; s < n; ++s) {
        const double dt = h->pinned[2 * s], tmax = h->pinned[2 * s + 1];
        if (!(tmax > 0.0) || !std::isfinite(tmax) || !std::isfinite(dt))
            return fail(h, HYDRO_ESTATE, "estimate_dt: max signal speed is not a positive finite number (step " +
                                             std::to_string(s) + " of the call)");
        if (dt_host) dt_host[s] = dt;
    }
    return HYDRO_OK;
}

// one chunk of at most DT_SLOTS steps; step s of the chunk keeps its (dt, max t) in slot s
int step_chunk(hydro_handle h, int nsteps, double *dt_host)
{
    int rc;
    const bool split = h->split_ghosts, fuse = h->fuse_dt;
    for (int s = 0; s < nsteps; ++s) {
        const double *dt_dev = dt_slot(h, s);
        // the caller's U0 gets the dt kernel; later steps use the dt that the stage-1 z sweep of the
        // previous step reduced from the very values it wrote (same formula, same bits)
        if (s == 0 || !fuse) if ((rc = launch_dt(h, s))) return rc;
        // the caller's U0 gets the full fill; after that stage 1 has left every valid row of U0
        // complete (x images written by the z sweeps) and only the ghost rows remain
        if ((rc = (split && s > 0) ? fill_ghost_rows_impl(h, 0) : fill_ghosts_impl(h, 0))) return rc;
        if ((rc = advance_stage_impl(h, 0, 0.0, dt_dev, split))) return rc;
        if ((rc = split ? fill_ghost_rows_impl(h, 1) : fill_ghosts_impl(h, 1))) return rc;
        double *dt_next = (fuse && s + 1 < nsteps) ? dt_slot(h, s + 1) : nullptr;
        if ((rc = advance_stage_impl(h, 1, 0.0, dt_dev, split, dt_next))) return rc;
    }
    return read_dts(h, dt_host, nsteps);
}

// ---- O12: CTU step (ctu.cuh) --------------------------------------------------------------------------------
size_t ctu_box_bytes(const Geom &g) { return (size_t)12 * g.nflux * g.cstride * 8; }

template <int DIR>
int ctu_dir(hydro_handle h, const CtuArgs &a, int phase)
{
    const Geom &g = h->g;
    const int nb[3] = {g.nb[0], g.nb[1], g.nb[2]};
    auto grid = [&](int ext, int face) {
        int n[3] = {nb[0] + 2 * ext, nb[1] + 2 * ext, nb[2] + 2 * ext};
        if (face >= 0) n[face] = nb[face] + 1;
        return dim3((unsigned)(((n[0] + 31) / 32) * a.nbatch), (unsigned)((n[1] + CTU_BY - 1) / CTU_BY), (unsigned)n[2]);
    };
    const dim3 blk(32, CTU_BY);
    int rc = HYDRO_OK;
    const int ns = g.nspec;
    prof_begin(h);
    if (phase == 0) k_ctu_trace_hydro<DIR><<<grid(1, -1), blk, 0, h->stream>>>(g, a);
    else if (phase == 1) k_ctu_flux_hydro<DIR, false><<<grid(1, DIR), blk, 0, h->stream>>>(g, a);
    else k_ctu_flux_hydro<DIR, true><<<grid(0, DIR), blk, 0, h->stream>>>(g, a);
    if ((rc = check_launch(h, "k_ctu hydro", K_CTU))) return rc;
    if (ns > 0) {
        prof_begin(h);
        if (phase == 0) k_ctu_trace_species<DIR><<<grid(1, -1), blk, 0, h->stream>>>(g, a);
        else if (phase == 1) k_ctu_flux_species<DIR, false><<<grid(1, DIR), blk, 0, h->stream>>>(g, a);
        else k_ctu_flux_species<DIR, true><<<grid(0, DIR), blk, 0, h->stream>>>(g, a);
        rc = check_launch(h, "k_ctu species", K_CTU);
    }
    return rc;
}

int ctu_chunk(hydro_handle h, char *scratch, size_t bytes, int nsteps, double *dt_host, int &cur)
{
    const Geom &g = h->g;
    int nbatch_max = (int)(bytes / ctu_box_bytes(g));
    if (nbatch_max > g.nboxes) nbatch_max = g.nboxes;
    int rc;
    for (int s = 0; s < nsteps; ++s) {
        if ((rc = launch_dt(h, s, cur))) return rc;
        if ((rc = fill_ghosts_impl(h, cur))) return rc;
        for (int box0 = 0; box0 < g.nboxes; box0 += nbatch_max) {
            CtuArgs a;
            a.U = h->U[cur]; a.Unew = h->U[cur ^ 1]; a.Q = (double *)scratch; a.dt_dev = dt_slot(h, s);
            a.box0 = box0; a.nbatch = g.nboxes - box0 < nbatch_max ? g.nboxes - box0 : nbatch_max;
            for (int phase = 0; phase < 3; ++phase) {
                if ((rc = ctu_dir<0>(h, a, phase))) return rc;
                if ((rc = ctu_dir<1>(h, a, phase))) return rc;
                if ((rc = ctu_dir<2>(h, a, phase))) return rc;
            }
            prof_begin(h);
            const dim3 ugrid((unsigned)(((g.nb[0] + 31) / 32) * a.nbatch), (unsigned)((g.nb[1] + CTU_BY - 1) / CTU_BY), g.nb[2]);
            k_ctu_update_hydro<<<ugrid, dim3(32, CTU_BY), 0, h->stream>>>(g, a);
            if ((rc = check_launch(h, "k_ctu_update_hydro", K_CTU))) return rc;
            if (g.nspec > 0) {
                prof_begin(h);
                k_ctu_update_species<<<ugrid, dim3(32, CTU_BY), 0, h->stream>>>(g, a);
                if ((rc = check_launch(h, "k_ctu_update_species", K_CTU))) return rc;
            }
        }
        cur ^= 1;
    }
    return read_dts(h, dt_host, nsteps);
}

}  // namespace

extern "C" {

size_t hydro_state_bytes(const hydro_params *p)
{
    Geom g; std::string why;
    if (!make_geom(p, g, why)) return 0;
    return (size_t)g.bstride * g.nboxes * 8;
}

size_t hydro_scratch_bytes(const hydro_params *p)
{
    Geom g; std::string why;
    if (!make_geom(p, g, why)) return 0;
    return carve(g).total;
}

int hydro_init(const hydro_params *p, void *U0_dev, void *U1_dev, void *scratch_dev, size_t scratch_bytes,
               void *cuda_stream, hydro_handle *out)
{
    Geom g; std::string why;
    if (!out) return fail(nullptr, HYDRO_EINVAL, "null out handle");
    *out = nullptr;
    if (!make_geom(p, g, why)) return fail(nullptr, HYDRO_EINVAL, why);
    if (!U0_dev || !U1_dev || !scratch_dev) return fail(nullptr, HYDRO_EINVAL, "null device buffer");
    if (((uintptr_t)U0_dev | (uintptr_t)U1_dev | (uintptr_t)scratch_dev) & 15)
        return fail(nullptr, HYDRO_EINVAL, "device buffers must be 16-byte aligned");
    if (U0_dev == U1_dev) return fail(nullptr, HYDRO_EINVAL, "U0 and U1 must be distinct");
    Carve cv = carve(g);
    if (scratch_bytes < cv.total) return fail(nullptr, HYDRO_ENOMEM, "scratch_bytes too small");
    // the device of the handle = the device the caller's buffers live on (all three on the same one)
    int device = -1;
    {
        void *bufs[3] = {U0_dev, U1_dev, scratch_dev};
        for (void *b : bufs) {
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, b) != cudaSuccess || at.type != cudaMemoryTypeDevice) {
                cudaGetLastError();
                return fail(nullptr, HYDRO_EINVAL, "U0_dev, U1_dev and scratch_dev must be device memory");
            }
            if (device >= 0 && at.device != device)
                return fail(nullptr, HYDRO_EINVAL, "U0_dev, U1_dev and scratch_dev must live on one device");
            device = at.device;
        }
    }
    DeviceGuard guard(device);
    hydro_ctx *h = new (std::nothrow) hydro_ctx();
    if (!h) return fail(nullptr, HYDRO_ENOMEM, "host allocation failed");
    h->p = *p; h->g = g; h->U[0] = (double *)U0_dev; h->U[1] = (double *)U1_dev;
    h->scratch = (char *)scratch_dev; h->cv = cv; h->stream = (cudaStream_t)cuda_stream;
    h->device = device;
    h->launches = 0; h->pinned = nullptr; h->profiling = false; h->pool_used = 0; h->pending = -1;
    // tuning switches (include/hydro.h): read here, once
    h->kn.ring = env_int("HYDRO_RING", 1);
    h->kn.seglen = env_int("HYDRO_SEGLEN", 0);
    h->kn.nsmax = env_int("HYDRO_NSMAX", NS_MAX);
    h->kn.fuse_dt = env_int("HYDRO_FUSE_DT", 1);
    h->kn.split_ghosts = env_int("HYDRO_SPLIT_GHOSTS", 1);
    h->kn.fill_monolithic = env_int("HYDRO_FILL_MONOLITHIC", 0);
    h->kn.xmarch = env_int("HYDRO_XMARCH", 0);
    h->kn.species_one_launch = env_int("HYDRO_SPECIES_ONE_LAUNCH", 1);
    h->kn.xchunk = env_int("HYDRO_XCHUNK", 1);
    h->ns_max = (h->kn.nsmax >= 1 && h->kn.nsmax <= NS_MAX) ? h->kn.nsmax : NS_MAX;
    for (int d = 0; d < 3; ++d) h->seglen[d] = d == 0 ? g.nb[0] : pick_seglen(g, d, h->kn.seglen);
    {   // TMA tensor copies: 16-byte row pitch AND 16-byte aligned box starts (the first valid zone of a row sits
        // ng doubles in, so ng must be even), row segments that tile the CTA exactly
        const int W = g.nb[0] < BS ? g.nb[0] : BS;
        h->use_ring = (g.ng % 2 == 0) && (g.nb[0] % 2 == 0) && (BS % W == 0) && (g.nb[0] % W == 0) && h->kn.ring != 0;
        for (int st = 0; st < 2 && h->use_ring; ++st)
            for (int dir = 1; dir <= 2 && h->use_ring; ++dir)
                for (int nc = 1; nc <= 6 && h->use_ring; ++nc) {
                    if (nc > g.nvar) continue;
                    std::string why2;
                    if (!make_ring_map(&h->maps[st][dir - 1][nc], h->U[st], g, dir, nc, why2)) h->use_ring = false;
                }
    }
    {   // x marching kernels: rows of nb0 in whole 4-zone steps, 128 rows per CTA, zones -4 .. nb0+3 inside the padded
        // row at 16-byte aligned starts; the options O10 / O11 stay with k_sweep_x
        h->use_xmarch = h->kn.xmarch != 0 && g.ng % 2 == 0 && g.ng >= 4 && g.nb[0] % XC == 0 &&
                        (XBS % g.nb[1] == 0 || g.nb[1] % XBS == 0) && (XS_ROWS % g.nb[1] == 0 || g.nb[1] % XS_ROWS == 0) &&
                        !g.flatten && !g.evolve;
        for (int st = 0; st < 2 && h->use_xmarch; ++st)
            for (int nc = 1; nc <= 5 && h->use_xmarch; ++nc) {
                if (nc > g.nvar) continue;
                std::string why2;
                if (!make_xmarch_map(&h->xmaps[st][nc], h->U[st], g, nc, XBS, why2)) h->use_xmarch = false;
                if (!make_xmarch_map(&h->xsmaps[st][nc], h->U[st], g, nc, XS_ROWS, why2)) h->use_xmarch = false;
            }
        if (h->use_xmarch) {
            std::string why2;
            if (!make_fx_map(&h->fxmap, (double *)(h->scratch + cv.frho), g, XS_ROWS, why2)) h->use_xmarch = false;
        }
    }
    // chunk-lane x sweep (sweep_xc.cuh): whole 4-zone chunks (256-bit loads and stores: 32-byte aligned arrays), the
    // flattened chunk sequence of a box in an int
    h->use_xchunk = h->kn.xchunk != 0 && g.ng % 4 == 0 && g.nb[0] % 4 == 0 &&
                    (long long)g.nb[1] * g.nb[2] * (g.nt[0] / 4) < (1LL << 30) &&
                    ((uintptr_t)U0_dev % 32) == 0 && ((uintptr_t)U1_dev % 32) == 0 && ((uintptr_t)(h->scratch + cv.lacc) % 32) == 0 &&
                    (!g.flatten || ((uintptr_t)(h->scratch + cv.flat) % 32) == 0);
    cudaError_t e = cudaSuccess;
    if (g.flatten) {   // coefficient array = 1 (no flattening) outside the zones k_flatten writes
        double *FL = (double *)(h->scratch + cv.flat);
        k_fill_value<<<148 * 8, 256, 0, h->stream>>>(FL, (long long)g.cstride * g.nboxes, 1.0);
        e = cudaGetLastError();
        h->launches++;
        for (int dir = 1; dir <= 2 && h->use_ring; ++dir) {
            std::string why2;
            if (!make_ring_map(&h->fmaps[dir - 1], FL, g, dir, 1, why2, 1, g.cstride)) h->use_ring = false;
        }
    }
    // a face shared with another shard (HYDRO_BC_EXTERNAL): its ghosts come from hydro_unpack_halo; only the
    // one-launch ghost fill knows how to leave them alone, and hydro_step (no exchange between its stages) is refused
    h->external = false;
    for (int d = 0; d < 3; ++d) h->external = h->external || p->bc_lo[d] == HYDRO_BC_EXTERNAL || p->bc_hi[d] == HYDRO_BC_EXTERNAL;
    // split ghost fill inside hydro_step: needs the ring kernels, 16-byte rows and boxes >= ng wide
    h->fuse_dt = h->use_ring && !g.evolve && h->kn.fuse_dt != 0;   // O11: rho*e is final only after the energy kernel
    h->split_ghosts = h->use_ring && (g.nt[0] % 2 == 0) && g.nb[0] >= g.ng && g.nb[1] >= g.ng && g.nb[2] >= g.ng &&
                      h->kn.split_ghosts != 0 && !h->external;
    const size_t npin = (size_t)(g.nflux > 2 * DT_SLOTS ? g.nflux : 2 * DT_SLOTS);
    if (e == cudaSuccess) e = cudaMallocHost((void **)&h->pinned, npin * 8);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->scratch + cv.red, 0, 256, h->stream);
    if (e != cudaSuccess) {
        std::string msg = std::string("hydro_init: ") + cudaGetErrorString(e);
        if (h->pinned) cudaFreeHost(h->pinned);
        delete h;
        return fail(nullptr, HYDRO_ECUDA, msg);
    }
    *out = h;
    return HYDRO_OK;
}

int hydro_fill_ghosts(hydro_handle h, int which)
{
    if (!h) return fail(nullptr, HYDRO_EINVAL, "null handle");
    if (which != 0 && which != 1) return fail(h, HYDRO_EINVAL, "which must be 0 or 1");
    DeviceGuard guard(h->device);
    return fill_ghosts_impl(h, which);
}

int hydro_advance_stage(hydro_handle h, int stage, double dt)
{
    if (!h) return fail(nullptr, HYDRO_EINVAL, "null handle");
    if (stage != 0 && stage != 1) return fail(h, HYDRO_EINVAL, "stage must be 0 or 1");
    DeviceGuard guard(h->device);
    return advance_stage_impl(h, stage, dt, nullptr);
}

int hydro_estimate_dt(hydro_handle h, double *dt_host)
{
    if (!h) return fail(nullptr, HYDRO_EINVAL, "null handle");
    if (!dt_host) return fail(h, HYDRO_EINVAL, "null dt_host");
    DeviceGuard guard(h->device);
    int rc = launch_dt(h);
    if (rc) return rc;
    return read_dts(h, dt_host, 1);
}

int hydro_conserved_totals(hydro_handle h, int which, double *totals_host)
{
    if (!h) return fail(nullptr, HYDRO_EINVAL, "null handle");
    if (which != 0 && which != 1) return fail(h, HYDRO_EINVAL, "which must be 0 or 1");
    if (!totals_host) return fail(h, HYDRO_EINVAL, "null totals_host");
    DeviceGuard guard(h->device);
    const Geom &g = h->g;
    const long long nrows = (long long)g.nb[1] * g.nb[2] * g.nboxes;
    long long blocks = (nrows + 7) / 8;            // 8 warps per block, one row per warp and trip
    if (blocks > RED_BLOCKS) blocks = RED_BLOCKS;
    double *part = (double *)(h->scratch + h->cv.part);
    double *tot = (double *)(h->scratch + h->cv.totals);
    prof_begin(h);
    k_totals_partial<<<dim3((unsigned)blocks, g.nflux), 256, 0, h->stream>>>(g, h->U[which], part);
    int rc = check_launch(h, "k_totals_partial", K_TOTALS);
    if (rc) return rc;
    prof_begin(h);
    k_totals_final<<<g.nflux, 32, 0, h->stream>>>(g, part, (int)blocks, tot);
    if ((rc = check_launch(h, "k_totals_final", K_TOTALS))) return rc;
    cudaError_t e = cudaMemcpyAsync(h->pinned, tot, (size_t)g.nflux * 8, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(h, HYDRO_ECUDA, std::string("totals read-back: ") + cudaGetErrorString(e));
    std::memcpy(totals_host, h->pinned, (size_t)g.nflux * 8);
    return HYDRO_OK;
}

int hydro_step(hydro_handle h, int nsteps, double *dt_host)
{
    if (!h) return fail(nullptr, HYDRO_EINVAL, "null handle");
    if (nsteps < 0) return fail(h, HYDRO_EINVAL, "nsteps must be >= 0");
    if (h->external)
        return fail(h, HYDRO_EINVAL, "hydro_step cannot run on a shard (HYDRO_BC_EXTERNAL faces need a halo exchange "
                                     "between the stages): call the stages one by one");
    DeviceGuard guard(h->device);
    for (int done = 0; done < nsteps; done += DT_SLOTS) {
        const int n = nsteps - done < DT_SLOTS ? nsteps - done : DT_SLOTS;
        int rc = step_chunk(h, n, dt_host ? dt_host + done : nullptr);
        if (rc) return rc;
    }
    return HYDRO_OK;
}

size_t hydro_halo_bytes(const hydro_params *p, int dim)
{
    Geom g; std::string why;
    if (!make_geom(p, g, why) || dim < 0 || dim > 2) return 0;
    const int d0 = dim == 0 ? 1 : 0, d1 = dim == 2 ? 1 : 2;
    return (size_t)g.nvar * g.ng * g.nt[d0] * g.nt[d1] * g.NB[d0] * g.NB[d1] * 8;
}

static int halo_impl(hydro_handle h, int which, int dim, int side, void *buf_dev, bool pack)
{
    if (!h) return fail(nullptr, HYDRO_EINVAL, "null handle");
    if ((which != 0 && which != 1) || dim < 0 || dim > 2 || (side != 0 && side != 1))
        return fail(h, HYDRO_EINVAL, "which and side must be 0 or 1, dim 0..2");
    if (!buf_dev || ((uintptr_t)buf_dev & 7)) return fail(h, HYDRO_EINVAL, "null or misaligned halo buffer");
    if (h->g.nb[dim] < h->g.ng) return fail(h, HYDRO_EINVAL, "boxes narrower than ng cannot supply a halo");
    DeviceGuard guard(h->device);
    prof_begin(h);
    if (pack) k_halo<true><<<RED_BLOCKS, 256, 0, h->stream>>>(h->g, h->U[which], (double *)buf_dev, dim, side);
    else k_halo<false><<<RED_BLOCKS, 256, 0, h->stream>>>(h->g, h->U[which], (double *)buf_dev, dim, side);
    return check_launch(h, pack ? "k_halo<pack>" : "k_halo<unpack>", K_GHOST);
}

int hydro_pack_halo(hydro_handle h, int which, int dim, int side, void *buf_dev) { return halo_impl(h, which, dim, side, buf_dev, true); }

int hydro_unpack_halo(hydro_handle h, int which, int dim, int side, const void *buf_dev)
{
    return halo_impl(h, which, dim, side, const_cast<void *>(buf_dev), false);
}

size_t hydro_ctu_scratch_bytes(const hydro_params *p)
{
    Geom g; std::string why;
    if (!make_geom(p, g, why)) return 0;
    return ctu_box_bytes(g);
}

int hydro_ctu_step(hydro_handle h, void *ctu_scratch_dev, size_t ctu_scratch_bytes, int nsteps, double *dt_host)
{
    if (!h) return fail(nullptr, HYDRO_EINVAL, "null handle");
    if (nsteps < 0) return fail(h, HYDRO_EINVAL, "nsteps must be >= 0");
    const Geom &g = h->g;
    if (g.flatten || g.evolve) return fail(h, HYDRO_EINVAL, "the options flatten / evolve_eint belong to the method-of-lines path");
    if (h->external) return fail(h, HYDRO_EINVAL, "hydro_ctu_step cannot run on a shard (HYDRO_BC_EXTERNAL)");
    if (!ctu_scratch_dev || ((uintptr_t)ctu_scratch_dev & 15)) return fail(h, HYDRO_EINVAL, "null or misaligned CTU scratch");
    if (ctu_scratch_bytes < ctu_box_bytes(g)) return fail(h, HYDRO_ENOMEM, "ctu_scratch_bytes too small (hydro_ctu_scratch_bytes)");
    if (g.nb[2] + 2 > 65535 || (g.nb[1] + 2 + CTU_BY - 1) / CTU_BY > 65535)
        return fail(h, HYDRO_EINVAL, "CTU grid too large (nbox[1] or nbox[2])");
    DeviceGuard guard(h->device);
    int cur = 0, rc = HYDRO_OK;
    for (int done = 0; done < nsteps && rc == HYDRO_OK; done += DT_SLOTS) {
        const int n = nsteps - done < DT_SLOTS ? nsteps - done : DT_SLOTS;
        rc = ctu_chunk(h, (char *)ctu_scratch_dev, ctu_scratch_bytes, n, dt_host ? dt_host + done : nullptr, cur);
    }
    if (cur == 1) {     // an odd number of steps left the result in U1: the contract is "U0 advanced in place"
        cudaError_t e = cudaMemcpyAsync(h->U[0], h->U[1], (size_t)g.bstride * g.nboxes * 8, cudaMemcpyDeviceToDevice, h->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
        if (e != cudaSuccess && rc == HYDRO_OK) rc = fail(h, HYDRO_ECUDA, std::string("CTU copy back: ") + cudaGetErrorString(e));
    }
    return rc;
}

int hydro_fill_from_coarse(hydro_handle fine, int which_fine, hydro_handle coarse, int which_coarse, const int32_t *lo_coarse,
                           int ratio)
{
    if (!fine || !coarse) return fail(nullptr, HYDRO_EINVAL, "null handle");
    hydro_handle h = fine;
    if ((which_fine != 0 && which_fine != 1) || (which_coarse != 0 && which_coarse != 1))
        return fail(h, HYDRO_EINVAL, "which must be 0 or 1");
    if (!lo_coarse) return fail(h, HYDRO_EINVAL, "null lo_coarse");
    if (ratio != 2 && ratio != 4) return fail(h, HYDRO_EINVAL, "ratio must be 2 or 4");
    const Geom &gf = fine->g, &gc = coarse->g;
    if (fine->device != coarse->device) return fail(h, HYDRO_EINVAL, "the two levels must live on one device");
    if (gf.nvar != gc.nvar) return fail(h, HYDRO_EINVAL, "the two levels must carry the same components");
    AmrArgs a;
    for (int d = 0; d < 3; ++d) {
        if (gf.ndom[d] % ratio) return fail(h, HYDRO_EINVAL, "the fine patch must cover whole coarse zones");
        if (lo_coarse[d] < 0 || lo_coarse[d] + gf.ndom[d] / ratio > gc.ndom[d])
            return fail(h, HYDRO_EINVAL, "the fine patch must lie inside the coarse domain");
        // the deepest fine ghost zone needs the coarse zone (ng_f + ratio - 1)/ratio outside the patch, and its slope one more
        if ((gf.ng + ratio - 1) / ratio + 1 > gc.ng) return fail(h, HYDRO_EINVAL, "coarse level has too few ghost zones for this ratio");
        a.lo[d] = lo_coarse[d];
    }
    if (gf.nt[2] > 65535 || gf.nboxes > 65535) return fail(h, HYDRO_EINVAL, "fine level grid too large for the coarse-fine fill");
    a.Uf = fine->U[which_fine]; a.Uc = coarse->U[which_coarse]; a.ratio = ratio;
    DeviceGuard guard(h->device);
    if (coarse->stream != fine->stream) {      // order after the coarse level's work (its ghost fill)
        cudaEvent_t ev;
        if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) return fail(h, HYDRO_ECUDA, "event creation failed");
        cudaEventRecord(ev, coarse->stream);
        cudaStreamWaitEvent(fine->stream, ev, 0);
        cudaEventDestroy(ev);
    }
    prof_begin(h);
    k_fill_from_coarse<<<dim3((gf.nt[0] * gf.nt[1] + 255) / 256, gf.nt[2], gf.nboxes), 256, 0, h->stream>>>(gf, gc, a);
    return check_launch(h, "k_fill_from_coarse", K_GHOST);
}

int hydro_average_down(hydro_handle coarse, int which_coarse, hydro_handle fine, int which_fine, const int32_t *lo_coarse, int ratio)
{
    if (!fine || !coarse) return fail(nullptr, HYDRO_EINVAL, "null handle");
    hydro_handle h = coarse;
    if ((which_fine != 0 && which_fine != 1) || (which_coarse != 0 && which_coarse != 1))
        return fail(h, HYDRO_EINVAL, "which must be 0 or 1");
    if (!lo_coarse) return fail(h, HYDRO_EINVAL, "null lo_coarse");
    if (ratio != 2 && ratio != 4) return fail(h, HYDRO_EINVAL, "ratio must be 2 or 4");
    const Geom &gf = fine->g, &gc = coarse->g;
    if (fine->device != coarse->device) return fail(h, HYDRO_EINVAL, "the two levels must live on one device");
    if (gf.nvar != gc.nvar) return fail(h, HYDRO_EINVAL, "the two levels must carry the same components");
    for (int d = 0; d < 3; ++d) {
        if (gf.ndom[d] % ratio) return fail(h, HYDRO_EINVAL, "the fine patch must cover whole coarse zones");
        if (lo_coarse[d] < 0 || lo_coarse[d] + gf.ndom[d] / ratio > gc.ndom[d])
            return fail(h, HYDRO_EINVAL, "the fine patch must lie inside the coarse domain");
    }
    DeviceGuard guard(h->device);
    if (coarse->stream != fine->stream) {      // order after the fine level's work
        cudaEvent_t ev;
        if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) return fail(h, HYDRO_ECUDA, "event creation failed");
        cudaEventRecord(ev, fine->stream);
        cudaStreamWaitEvent(coarse->stream, ev, 0);
        cudaEventDestroy(ev);
    }
    const long long zones = (long long)(gf.ndom[0] / ratio) * (gf.ndom[1] / ratio) * (gf.ndom[2] / ratio);
    prof_begin(h);
    k_average_down<<<dim3((unsigned)((zones + 255) / 256), gc.nvar), 256, 0, h->stream>>>(gc, gf, coarse->U[which_coarse], fine->U[which_fine],
                                                                                          lo_coarse[0], lo_coarse[1], lo_coarse[2], ratio);
    return check_launch(h, "k_average_down", K_GHOST);
}

int hydro_query(hydro_handle h, int what)
{
    if (!h) return -1;
    switch (what) {
        case 0: return h->use_ring ? 1 : 0;
        case 1: return h->split_ghosts ? 1 : 0;
        case 2: return h->fuse_dt ? 1 : 0;
        case 3: return h->ns_max;
        case 4: return h->use_xmarch ? 1 : 0;
        case 5: return h->use_ring ? (h->kn.species_one_launch & 3) : 0;
        case 6: return (!h->use_xmarch && h->use_xchunk) ? 1 : 0;
        default: return -1;
    }
}

long long hydro_launch_count(hydro_handle h) { return h ? h->launches : 0; }

int hydro_profile(hydro_handle h, int enable)
{
    if (!h) return fail(nullptr, HYDRO_EINVAL, "null handle");
    DeviceGuard guard(h->device);
    if (enable && h->pool.empty()) {      // the event pool is created here, never while launches are recorded
        h->pool.resize(PROF_EVENTS);
        for (auto &ev : h->pool)
            if (cudaEventCreate(&ev) != cudaSuccess) {
                h->pool.clear();
                return fail(h, HYDRO_ECUDA, "hydro_profile: cudaEventCreate failed");
            }
        h->events.reserve(PROF_EVENTS / 2);
    }
    h->profiling = enable != 0;
    return HYDRO_OK;
}

int hydro_profile_read(hydro_handle h, double *ms_host, long long *count_host)
{
    if (!h) return fail(nullptr, HYDRO_EINVAL, "null handle");
    if (!ms_host || !count_host) return fail(h, HYDRO_EINVAL, "null output");
    DeviceGuard guard(h->device);
    for (int c = 0; c < K_NCLASS; ++c) { ms_host[c] = 0.0; count_host[c] = 0; }
    cudaError_t e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(h, HYDRO_ECUDA, std::string("profile_read: ") + cudaGetErrorString(e));
    for (auto &ev : h->events) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, h->pool[ev.a], h->pool[ev.b]) == cudaSuccess) { ms_host[ev.klass] += ms; count_host[ev.klass]++; }
    }
    h->events.clear();
    h->pool_used = 0;
    return HYDRO_OK;
}

int hydro_destroy(hydro_handle h)
{
    if (!h) return HYDRO_OK;
    DeviceGuard guard(h->device);
    cudaStreamSynchronize(h->stream);
    for (auto &ev : h->pool) cudaEventDestroy(ev);
    if (h->pinned) cudaFreeHost(h->pinned);
    delete h;
    return HYDRO_OK;
}

const char *hydro_last_error(hydro_handle h) { return h ? h->err.c_str() : g_init_error.c_str(); }

int hydro_run_host(const hydro_params *p, double *U_host, int nsteps, double *dt_host, double *totals_host)
{
    Geom g; std::string why;
    if (!make_geom(p, g, why)) return fail(nullptr, HYDRO_EINVAL, why);
    if (!U_host || nsteps < 0) return fail(nullptr, HYDRO_EINVAL, "null U_host or negative nsteps");
    const size_t sb = (size_t)g.bstride * g.nboxes * 8, scb = carve(g).total;
    void *U0 = nullptr, *U1 = nullptr, *sc = nullptr;
    hydro_handle h = nullptr;
    int rc = HYDRO_OK;
    cudaError_t e = cudaMalloc(&U0, sb);
    if (e == cudaSuccess) e = cudaMalloc(&U1, sb);
    if (e == cudaSuccess) e = cudaMalloc(&sc, scb);
    if (e != cudaSuccess) { rc = fail(nullptr, HYDRO_ENOMEM, std::string("hydro_run_host: ") + cudaGetErrorString(e)); goto done; }
    e = cudaMemcpy(U0, U_host, sb, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { rc = fail(nullptr, HYDRO_ECUDA, std::string("H2D: ") + cudaGetErrorString(e)); goto done; }
    if ((rc = hydro_init(p, U0, U1, sc, scb, nullptr, &h))) goto done;
    rc = hydro_step(h, nsteps, dt_host);
    if (rc == HYDRO_OK && totals_host) rc = hydro_conserved_totals(h, 0, totals_host);
    if (rc != HYDRO_OK) { g_init_error = h->err; goto done; }
    e = cudaMemcpy(U_host, U0, sb, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) rc = fail(nullptr, HYDRO_ECUDA, std::string("D2H: ") + cudaGetErrorString(e));
done:
    if (h) hydro_destroy(h);
    if (sc) cudaFree(sc);
    if (U1) cudaFree(U1);
    if (U0) cudaFree(U0);
    return rc;
}

}  // extern "C"

// ---- O9 totals for callers that cannot allocate: hydro_conserved_totals_static (include/hydro.h) ----------------
// The two-pass reduction of hydro_conserved_totals needs a place for the per-block partial sums.  Every other entry
// point takes that place from the caller's scratch buffer, which somebody had to cudaMalloc; this one keeps it in
// the library image instead.  The array below is part of the loaded module: each GPU that loads libhydro_b200.so
// carries its own 592 KiB copy from the moment the module is loaded there until the process exits, used or not.
namespace {

constexpr int STATIC_TOTALS_NFLUX = HYDRO_TOTALS_STATIC_MAX_NFLUX;
constexpr size_t STATIC_TOTALS_DOUBLES = (size_t)STATIC_TOTALS_NFLUX * RED_BLOCKS * 2;   // (hi, lo) per block and component

static __device__ __align__(256) double g_static_partials[STATIC_TOTALS_DOUBLES];

// In host code `g_static_partials` is only a stand-in that the runtime maps to the real array; it is NOT a device
// address and must never be handed to a kernel.  The device address differs from GPU to GPU, so it is looked up
// with cudaGetSymbolAddress once per device, with that device current, and remembered here.
constexpr int STATIC_TOTALS_MAX_DEVICES = 64;
std::mutex g_static_mutex;
double *g_static_partials_addr[STATIC_TOTALS_MAX_DEVICES] = {};

}  // namespace

extern "C" int hydro_conserved_totals_static(const hydro_params *p, const void *U_dev, void *totals_dev,
                                             void *cuda_stream)
{
    Geom g; std::string why;
    if (!make_geom(p, g, why)) return fail(nullptr, HYDRO_EINVAL, why);
    if (g.nflux > STATIC_TOTALS_NFLUX) {
        char msg[256];
        snprintf(msg, sizeof msg,
                 "hydro_conserved_totals_static: nspec = %d gives %d conserved components, the built-in scratch holds "
                 "%d (nspec <= %d); use hydro_conserved_totals with a caller-provided scratch buffer instead",
                 g.nspec, g.nflux, STATIC_TOTALS_NFLUX, STATIC_TOTALS_NFLUX - 5);
        return fail(nullptr, HYDRO_ENOMEM, msg);
    }
    if (!U_dev || !totals_dev) return fail(nullptr, HYDRO_EINVAL, "null U_dev or totals_dev");
    if (((uintptr_t)U_dev % 8) != 0 || ((uintptr_t)totals_dev % 8) != 0)
        return fail(nullptr, HYDRO_EINVAL, "U_dev and totals_dev must be 8-byte aligned");
    int device = -1;
    {
        const void *bufs[2] = {U_dev, totals_dev};
        for (const void *b : bufs) {
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, b) != cudaSuccess || at.type != cudaMemoryTypeDevice) {
                cudaGetLastError();
                return fail(nullptr, HYDRO_EINVAL, "U_dev and totals_dev must be device memory");
            }
            if (device >= 0 && at.device != device)
                return fail(nullptr, HYDRO_EINVAL, "U_dev and totals_dev must live on one device");
            device = at.device;
        }
    }
    if (device >= STATIC_TOTALS_MAX_DEVICES) return fail(nullptr, HYDRO_EINVAL, "device ordinal beyond 63");
    DeviceGuard guard(device);
    int current = -1;
    if (cudaGetDevice(&current) != cudaSuccess || current != device)
        return fail(nullptr, HYDRO_ECUDA, "hydro_conserved_totals_static: could not make the buffers' device current");
    double *part = nullptr;
    {   // set-up, on the first call that sees this device (it may load the module there: keep it out of a capture)
        std::lock_guard<std::mutex> lock(g_static_mutex);
        if (!g_static_partials_addr[device]) {
            double *addr = nullptr;
            const cudaError_t e = cudaGetSymbolAddress((void **)&addr, g_static_partials);
            if (e != cudaSuccess || !addr) {
                cudaGetLastError();
                return fail(nullptr, HYDRO_ECUDA, std::string("hydro_conserved_totals_static: cudaGetSymbolAddress: ") +
                                                      cudaGetErrorString(e));
            }
            g_static_partials_addr[device] = addr;
        }
        part = g_static_partials_addr[device];
    }
    // the same launch geometry as hydro_conserved_totals, hence the same reduction tree and the same bits
    const long long nrows = (long long)g.nb[1] * g.nb[2] * g.nboxes;
    long long blocks = (nrows + 7) / 8;
    if (blocks > RED_BLOCKS) blocks = RED_BLOCKS;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // Pass 1 writes partial (component, block) for every block < blocks and every component < nflux; pass 2 reads
    // exactly those.  Whatever an earlier call left in the array is therefore never read, and nothing is cleared.
    k_totals_partial<<<dim3((unsigned)blocks, g.nflux), 256, 0, st>>>(g, (const double *)U_dev, part);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) {
        k_totals_final<<<g.nflux, 32, 0, st>>>(g, part, (int)blocks, (double *)totals_dev);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess)
        return fail(nullptr, HYDRO_ECUDA, std::string("hydro_conserved_totals_static: ") + cudaGetErrorString(e));
    return HYDRO_OK;
}
