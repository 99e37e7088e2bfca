/*
 * hydro.h -- C ABI of libhydro_b200: one explicit compressible-hydro advance (unsplit
 * method of lines: gamma-law EOS, PPM with the Colella-Woodward limiter, HLLC on every
 * x/y/z face, flux divergence + constant gravity, SSP-RK2, intra-GPU ghost fill, CFL
 * reduction) of a Castro-style state on a uniform-level MultiFab of boxes with ghost
 * zones, on ONE NVIDIA B200 (sm_100a).
 *
 * Problem statement: PAPER.md:35 (sec. II: MultiFab = collection of Fabs, a Fab = a
 * contiguous index box with several components, "a four-dimensional array"),
 * PAPER.md:49-57 (sec. III: per-zone parallel hydro kernels, the slope/reconstruction
 * stencil), PAPER.md:71,75 (no allocation inside the step loop; simulation data stay on
 * the device), PAPER.md:83 (nearest-neighbour coupling only).  The paper prints no
 * equations; the scheme is the one BASELINE.json:north_star names, written out step by
 * step in DESIGN.md sec. 2 (O1..O9).
 *
 * Pointers: every pointer named *_dev is DEVICE memory owned by the caller for the whole
 * lifetime of the handle; every pointer named *_host is HOST memory.  No torch types, no
 * C++ types; plain pointers and sizes only.
 *
 * State layout a1: FP64, SoA, one padded 3-D array per (box, component),
 * i fastest:
 *     idx = (((b*NVAR + c)*NZt + k)*NYt + j)*NXt + i,   b = (bk*NBy + bj)*NBx + bi,
 *     NXt = nbox[0] + 2*ng (etc.), valid zone (i,j,k) of a box at (i+ng, j+ng, k+ng).
 * Components c: 0 rho, 1 rho*u, 2 rho*v, 3 rho*w, 4 rho*E, 5 rho*e, 6+k rho*X_k.
 * NVAR = 6 + nspec stored components; NFLUX = 5 + nspec conserved components (all but
 * rho*e, which is re-synchronised from rho*E after every stage).
 *
 * Errors: every int-returning call returns 0 on success or a negative HYDRO_E* code; no
 * exception or abort crosses this boundary.  hydro_last_error() gives a message.
 */
#ifndef HYDRO_B200_H
#define HYDRO_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HYDRO_OK       0
#define HYDRO_EINVAL  -1  /* null pointer, nbox does not divide ndom, ng < 3, stage not 0/1,
                             periodic flag on one side only, buffer not 16-byte aligned      */
#define HYDRO_ENOMEM  -2  /* scratch_bytes too small (or device allocation failed in
                             hydro_run_host)                                                 */
#define HYDRO_ECUDA   -3  /* CUDA launch/runtime error; text via hydro_last_error            */
#define HYDRO_ESTATE  -4  /* a CFL reduction (hydro_estimate_dt, or any step of hydro_step) met a
                             non-finite or non-positive max signal speed                     */

#define HYDRO_BC_PERIODIC 0
#define HYDRO_BC_OUTFLOW  1
#define HYDRO_BC_REFLECT  2
#define HYDRO_BC_EXTERNAL 3  /* the face is shared with another shard of the MultiFab (another handle, usually another
                                GPU): hydro_fill_ghosts leaves the ghost zones across it alone, hydro_unpack_halo
                                fills them (PAPER.md:85-99 the boxes of a level are distributed
                                over ranks that exchange ghost zones) */

typedef struct {
    int32_t ndom[3];            /* zones in the domain (x,y,z)                               */
    int32_t nbox[3];            /* zones per box; must divide ndom (regular tiling)          */
    int32_t ng;                 /* ghost zones per side, >= 3 (the scheme reads 3)           */
    int32_t nspec;              /* passive species, >= 0                                     */
    int32_t bc_lo[3], bc_hi[3]; /* HYDRO_BC_*; periodic must be set on both sides of a dim; ndom, prob_lo and prob_hi
                                   of a shard (EXTERNAL faces) describe the shard's own sub-domain */
    double  prob_lo[3], prob_hi[3]; /* physical domain; dx = (prob_hi-prob_lo)/ndom          */
    double  gamma, cfl;
    double  grav[3];            /* constant acceleration; {0,0,0} disables the source        */
    double  small_dens, small_pres; /* floors (1e-12, 1e-14 in all workloads)                */
    int32_t flatten;            /* 0: off; 1: PPM shock flattening O10, needs ng >= 4 */
    int32_t evolve_eint;        /* 0: rho*e re-synchronised from rho*E after every stage; 1: evolved rho*e with a
                                   dual-energy switch, O11 */
    double  dx[3];              /* 0: zone width = (prob_hi - prob_lo)/ndom.  > 0: THIS zone width, and prob_lo / prob_hi
                                   only have to be ordered.  For a shard or a refined patch, whose extent is a piece of
                                   another handle's domain: the quotient of the piece's own extent can differ from the
                                   parent's zone width by an ulp (non-dyadic spacings), and then the piece no longer gives
                                   the parent's bits.  The drivers sharded.py / amr.py pass the parent's dx (/ ratio) */
} hydro_params;

typedef struct hydro_ctx *hydro_handle;

/* Size queries (host only, no CUDA call).  Return 0 for invalid params.
 * hydro_state_bytes   = nboxes * NVAR * NXt*NYt*NZt * 8   (one state, layout a1)
 * hydro_scratch_bytes = stage-increment accumulator (NFLUX per valid zone), one face
 *                       mass-flux array, and the reduction workspace. */
size_t hydro_state_bytes(const hydro_params *p);
size_t hydro_scratch_bytes(const hydro_params *p);

/* Create a handle.  U0_dev, U1_dev: two states of hydro_state_bytes each; scratch_dev:
 * at least hydro_scratch_bytes; all 16-byte aligned, all caller-owned DEVICE memory on ONE
 * device that must outlive the handle (HYDRO_EINVAL otherwise).  That device is the handle's:
 * every later call on the handle makes it current for its own duration and restores the
 * caller's device before it returns, so handles on several devices can live in one process.
 * cuda_stream: a cudaStream_t of that device (NULL = legacy default stream); every kernel of
 * this handle is enqueued on it.  The library allocates 16 KB of pinned host memory for scalar
 * read-back here and nothing afterwards, hydro_profile(h, 1) excepted.
 * The caller writes the initial state (all NVAR components of the valid zones; ghosts
 * may hold anything) into U0 before the first step, with rho*e consistent with rho*E.
 *
 * Tuning switches, read from the environment ONCE, here (they select among internal code paths
 * that give bit-identical results; defaults in brackets; hydro_query reports what a handle uses):
 *   HYDRO_RING=0            plain-load y/z sweeps instead of the TMA-ring marching kernels   [1]
 *   HYDRO_XCHUNK=0          x sweep by the one-zone-per-lane k_sweep_x (sweep_x.cuh) instead of the chunk-lane
 *                           k_sweep_xc (sweep_xc.cuh: a lane owns a 4-zone chunk; taken where ng and nbox[0]
 *                           are multiples of 4 and the buffers are 32-byte aligned; profiles/r02_xchunk.md)  [1]
 *   HYDRO_XMARCH=1          x sweep by the thread-per-row marching kernels of march_x.cuh instead of either
 *                           (measured equal in time to k_sweep_x, profiles/r02_xmarch.md)    [0]
 *   HYDRO_SEGLEN=n          zones per pencil segment of the y/z sweeps                       [auto]
 *   HYDRO_NSMAX=n           passive species per thread and launch, 1..5                      [5]
 *   HYDRO_SPECIES_ONE_LAUNCH=m  bit 0: the y species sweep, bit 1: the z species sweep launches all species groups
 *                           together (sibling CTAs share rho and F_rho rows through L2) instead of one by one     [1]
 *   HYDRO_FUSE_DT=0         hydro_step runs k_estimate_dt every step                         [1]
 *   HYDRO_SPLIT_GHOSTS=0    hydro_step / hydro_fill_ghosts use the one-launch ghost fill     [1]
 *   HYDRO_FILL_MONOLITHIC=1 hydro_fill_ghosts alone uses the one-launch ghost fill           [0] */
int hydro_init(const hydro_params *p, void *U0_dev, void *U1_dev, void *scratch_dev,
               size_t scratch_bytes, void *cuda_stream, hydro_handle *out);

/* O1 ghost fill: fill every ghost zone (faces, edges, corners) of every box
 * and component of state `which` (0: U0, 1: U1) from the valid zone that owns it:
 * periodic wrap, outflow = nearest valid zone, reflect = mirror with the wall-normal
 * momentum negated.  Asynchronous on the handle's stream. */
int hydro_fill_ghosts(hydro_handle h, int which);

/* O2..O7 one SSP-RK2 stage.  stage 0: reads U0 (ghosts must be filled), writes the valid
 * zones of U1 = U0 + dt*L(U0).  stage 1: reads U1 (ghosts filled) and U0, overwrites the
 * valid zones of U0 = 0.5*U0 + 0.5*(U1 + dt*L(U1)).  rho*e is re-synchronised in the
 * written state.  Does NOT fill ghosts.  Asynchronous on the handle's stream. */
int hydro_advance_stage(hydro_handle h, int stage, double dt);

/* O8 CFL timestep: dt = cfl / max over valid zones of U0 of sum_d (|u_d| + c)/dx_d.
 * Writes *dt_host; synchronises the stream.  HYDRO_ESTATE if the maximum is not a
 * positive finite number. */
int hydro_estimate_dt(hydro_handle h, double *dt_host);

/* O9 totals: totals_host[f] = sum over valid zones of conserved component f times
 * dx*dy*dz, f = 0..NFLUX-1 (rho, rho*u, rho*v, rho*w, rho*E, rho*X_k).  Deterministic
 * (fixed reduction tree, compensated).  Synchronises the stream. */
int hydro_conserved_totals(hydro_handle h, int which, double *totals_host);

/* n whole RK2 steps = n x { estimate_dt; fill(0); stage(0); fill(1); stage(1) } without host round
 * trips (dt stays on the device).  Results are bit-identical to the five separate calls; inside one
 * call the work is arranged differently from the second step on: the z sweeps write
 * the x ghost images of the zones they produce, so a ghost fill shrinks to whole-row copies, and the
 * stage-1 z hydro sweep reduces the next step's dt.  Ghost zones of U0 are unspecified on return, as
 * after the separate calls.
 * dt_host: NULL, or HOST memory for nsteps doubles that receive the dt of every step (a driver that
 * tracks simulation time needs them all).  Every step leaves its (dt, max signal speed) pair on the
 * device; after the last launch the call synchronises the stream, reads the pairs back in one copy and
 * returns HYDRO_ESTATE if ANY step's maximum was not a positive finite number (the state is then
 * unusable), with or without dt_host.  nsteps = 0 is a no-op; nsteps < 0 is HYDRO_EINVAL. */
int hydro_step(hydro_handle h, int nsteps, double *dt_host);

/* O12 (the integrator family behind PAPER.md:79 and :89): n steps of
 * the unsplit corner-transport-upwind update -- PPM, characteristic tracing, transverse flux corrections, ONE
 * conservative flux evaluation per step -- each step = { estimate_dt; fill ghosts; CTU update }, dt kept on the
 * device.  U0 is advanced in place (U1 is work space); dt_host and the HYDRO_ESTATE rule as for hydro_step.
 * ctu_scratch_dev: caller-owned DEVICE memory, 16-byte aligned, of at least hydro_ctu_scratch_bytes (the traced
 * states and fluxes of ONE box: 12 * NFLUX padded arrays); the boxes are worked through in batches of as many
 * boxes as the buffer holds, so a larger buffer means fewer, larger launches.  Not available with the options
 * flatten / evolve_eint or on a shard (HYDRO_EINVAL). */
size_t hydro_ctu_scratch_bytes(const hydro_params *p);
int hydro_ctu_step(hydro_handle h, void *ctu_scratch_dev, size_t ctu_scratch_bytes, int nsteps, double *dt_host);

/* Halo exchange of a sharded MultiFab (driver: paper_2007_05218_b200/sharded.py).
 * A halo of dimension dim (0 x, 1 y, 2 z) is the ng layers next to a face over the FULL padded extent of the
 * other two dimensions, all NVAR components, of every box on that face:
 *   hydro_halo_bytes = NVAR * ng * NTa * NTb * NBa * NBb * 8   (a, b = the other two dimensions).
 * hydro_pack_halo copies the VALID layers next to face (dim, side; side 0 low, 1 high) of state `which` into
 * buf_dev; hydro_unpack_halo copies a buffer packed by the neighbour shard from ITS opposite face into the GHOST
 * layers beyond (dim, side).  Exchanging x, then y, then z after hydro_fill_ghosts fills edges and corners
 * through the earlier dimensions' ghosts.  buf_dev: caller-owned DEVICE memory of hydro_halo_bytes, 8-byte
 * aligned.  Asynchronous on the handle's stream.  A handle with an EXTERNAL face refuses hydro_step (no exchange
 * is possible between its stages): HYDRO_EINVAL. */
size_t hydro_halo_bytes(const hydro_params *p, int dim);
int hydro_pack_halo(hydro_handle h, int which, int dim, int side, void *buf_dev);
int hydro_unpack_halo(hydro_handle h, int which, int dim, int side, const void *buf_dev);

/* O13 two-level ghost fill (second half; PAPER.md:35 a MultiFab lives
 * "at a given level of mesh refinement", PAPER.md:149 refinement by factors of 4).  `fine` is the handle of a
 * rectangular patch of `coarse`'s domain refined by ratio (2 or 4) in every direction: fine ndom = ratio * (patch
 * extent in coarse zones), prob_lo / prob_hi = the patch, its own boxes and ghost zones; the faces of the patch that
 * lie inside the coarse domain are HYDRO_BC_EXTERNAL, the others carry the physical boundary type.  The call fills
 * every ghost zone of fine state `which_fine` whose index lies across an EXTERNAL face in at least one dimension
 * from coarse state `which_coarse` (ghosts filled!) by conservative linear interpolation: value = Uc + sum_d
 * slope_d * xi_d, slope_d = the limited slope of O3 of the coarse zone averages, xi_d = (child + 0.5)/ratio - 0.5
 * (children average to their parent, linear data are reproduced exactly, no new extrema).  The other fine ghost
 * zones are hydro_fill_ghosts's.  lo_coarse[3] (HOST): coarse zone of the patch's first fine zone.  Both handles on
 * one device; the coarse level needs (ng_fine + ratio - 1)/ratio + 1 <= ng_coarse ghost zones.  Asynchronous on the
 * fine handle's stream (ordered after the coarse handle's stream). */
int hydro_fill_from_coarse(hydro_handle fine, int which_fine, hydro_handle coarse, int which_coarse,
                           const int32_t *lo_coarse, int ratio);

/* O13 restriction: every VALID zone of coarse state `which_coarse` that the patch covers becomes the mean of its
 * ratio^3 fine children (all NVAR components; conservative: the children's volumes add up to the parent's).  Same
 * patch description and checks as hydro_fill_from_coarse.  Asynchronous on the coarse handle's stream (ordered after
 * the fine handle's stream). */
int hydro_average_down(hydro_handle coarse, int which_coarse, hydro_handle fine, int which_fine,
                       const int32_t *lo_coarse, int ratio);

/* Which internal paths this handle uses (for bench accounting; they change no result):
 * what = 0: TMA-ring marching kernels (1) or the plain-load fallback (0);
 *        1: hydro_step fills ghosts in two parts (x images written by the z sweeps + ghost-row
 *           copies) instead of one k_fill_ghosts launch per stage;
 *        2: hydro_step reduces the next step's dt inside the stage-1 z hydro sweep;
 *        3: passive species per thread and launch in the species sweeps;
 *        4: the x sweep runs as marching kernels (a thread per row, march_x.cuh; 1) or as a
 *           lane-parallel kernel (0: see 6);
 *        5: which species sweeps launch all species groups together (bit 0: y, bit 1: z);
 *        6: the lane-parallel x sweep is the chunk-lane k_sweep_xc (1) or the one-zone-per-lane k_sweep_x (0).
 * Returns -1 for a NULL handle or an unknown `what`. */
int hydro_query(hydro_handle h, int what);

/* Number of kernel launches this handle has enqueued so far (for bench accounting). */
long long hydro_launch_count(hydro_handle h);

/* Optional per-launch timing for measurement (bench.py's roofline object).  While enabled,
 * every kernel launch of this handle is bracketed by a CUDA event pair on the handle's stream.
 * hydro_profile(h, 1) creates a pool of 8192 events on first use (the only allocation outside
 * hydro_init); recording stops silently when the pool is used up and resumes after the next read.
 * hydro_profile_read synchronises, then writes the summed device time in ms and the launch
 * count of each kernel class into ms_host[HYDRO_NCLASS] / count_host[HYDRO_NCLASS] and clears the record.
 * Classes: 0 ghost fill, 1 dt reduction, 2 x sweep, 3 y hydro sweep, 4 y species sweep,
 * 5 z hydro sweep + update, 6 z species sweep + update, 7 totals, 8 flattening coefficients, 9 CTU kernels. */
#define HYDRO_NCLASS 10
int hydro_profile(hydro_handle h, int enable);
int hydro_profile_read(hydro_handle h, double *ms_host, long long *count_host);

int hydro_destroy(hydro_handle h);

/* Message of the last error on this handle; with h == NULL, of the last failed
 * hydro_init / hydro_run_host on this thread.  Never NULL. */
const char *hydro_last_error(hydro_handle h);

/* End-to-end entry for callers without device buffers: U_host (hydro_state_bytes, layout
 * a1, valid zones filled) is copied to the device, advanced nsteps RK2 steps, and copied
 * back in place; dt_host[0..nsteps-1] (may be NULL) receives the timesteps and
 * totals_host[NFLUX] (may be NULL) the final conserved totals.  Allocates and frees its
 * own device memory (outside the step loop).  Synchronous. */
int hydro_run_host(const hydro_params *p, double *U_host, int nsteps, double *dt_host,
                   double *totals_host);

/* O9 totals (the sums of hydro_conserved_totals, bit for bit) for a caller that has a state on the device but may not
 * allocate anything: no handle, no scratch buffer, no pinned memory.
 *
 * Who that is: the codes of the paper draw all device memory from a pool that is grabbed up front and handed out as
 * sub-buffers, because cudaMalloc inside the timestep loop is "disastrous".  A diagnostics routine, an
 * in-situ monitor or a plug-in that is called from inside such a code is lent a pointer to the state and nothing
 * else: it has no access to the host code's pool, a cudaMalloc of its own may simply fail because the pool has
 * already taken the device's memory, and where it succeeds it stalls the device in the middle of a step.  Such a
 * caller cannot build a handle either (hydro_init wants a scratch buffer and pins host memory).  This call needs
 * neither: the partial sums of the reduction live in an array compiled into the library.
 *
 *   p           HOST: describes the state (ndom, nbox, ng, nspec, prob_lo/hi must be valid; the rest is ignored
 *               beyond the usual validation).
 *   U_dev       DEVICE, read only: one state in layout a1, hydro_state_bytes(p) bytes, 8-byte aligned.
 *   totals_dev  DEVICE, written: NFLUX = 5 + nspec doubles, 8-byte aligned, on the same device as U_dev;
 *               totals_dev[f] = sum over valid zones of conserved component f times dx*dy*dz.
 *   cuda_stream a cudaStream_t of that device (NULL = legacy default stream).  The two kernels are enqueued on it
 *               and the call returns without waiting; read totals_dev after synchronising that stream.
 *
 * Limit: nspec <= HYDRO_TOTALS_STATIC_MAX_NFLUX - 5 = 27.  A larger nspec returns HYDRO_ENOMEM and the message says
 * what the limit is; use hydro_conserved_totals, whose scratch the caller sizes, for those.  The number of zones
 * and boxes is not limited.  The built-in array is 592 KiB (32 components x 1184 blocks x 2 doubles); every GPU on
 * which the library's module is loaded holds its own copy until the process exits, whether or not this call is used.
 *
 * First call on a device: looks up the device address of the built-in array (once per device; it can make the CUDA
 * runtime load the library's module on that device).  Make that first call during start-up, outside any stream
 * capture; later calls only validate their arguments and launch.
 *
 * Sharing: every call on a device uses the same array, on whatever stream it is given.  Two calls that can run on
 * the GPU at the same time (different streams, or different host threads using different streams) overwrite each
 * other's partial sums and both may return wrong totals; order them on one stream or with events.  Calls that run
 * one after the other need no clean-up in between: the first kernel writes every partial sum the second reads, so
 * the contents left by an earlier call, of any shape, are never seen and nothing has to start at zero.
 *
 * Allocates nothing, on the host side of CUDA or on the device: no cudaMalloc / cudaFree / cudaMallocHost, no event
 * or stream creation, no library call that allocates.  Errors as everywhere: 0 or a negative HYDRO_E* code, message
 * via hydro_last_error(NULL). */
#define HYDRO_TOTALS_STATIC_MAX_NFLUX 32
int hydro_conserved_totals_static(const hydro_params *p, const void *U_dev, void *totals_dev, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* HYDRO_B200_H */
