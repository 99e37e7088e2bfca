/*
 * oracle/hydro_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of the hot path that
 * BASELINE.json:north_star names: one unsplit method-of-lines compressible
 * hydro advance (gamma-law EOS, PPM with the Colella-Woodward limiter, HLLC on
 * every x/y/z face, flux divergence + constant gravity, SSP-RK2, ghost fill,
 * CFL reduction) of a Castro-style state on a uniform-level MultiFab of boxes
 * with ghost zones (sec. II, MultiFab/Fab/Box; sec. III,
 * "a slope ... calculated by looking at several zones to the left and right"
 * feeding "a polynomial approximation of the fluid state").
 *
 * The paper prints no equations (SURVEY.md header), so every step follows
 * SURVEY.md sec. 8(c) O1..O9 and readings S1..S22 (restated in DESIGN.md).  Each
 * function below cites the step it implements.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this file.  It shares no code, header, table or
 * helper with paper_2007_05218_b200/csrc (the CUDA path); neither includes the
 * other.
 *
 * Floating-point contract (S18): FP64, every expression evaluated as written,
 * one IEEE operation per operator, no FMA contraction (compile with
 * -ffp-contract=off), constants HALF = 0.5, SIXTH = 1.0/6.0, dxinv = 1.0/dx
 * used as multipliers.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1 free-stream, P2 conservation,
 * P3 Sod exact solution, P4 Sedov radius, P5 PPM worked example (exact
 * rationals), P6 HLLC worked example, P7 axis permutation, P8 decomposition
 * invariance, P9 3-D = 1-D, P10 gravity closed form, P11 dt closed form, P12
 * ghost fill on index-encoded data, P13 order of accuracy; optional flattening O10:
 * tests/test_oracle_flatten.py (worked lines, exact no-op, Sod, symmetry).
 * Optional evolved rho*e O11: tests/test_oracle_evolve.py (bitwise the base scheme where the switch is
 * off, exact free stream where it is on, rounding of rho*E at Mach 1e6, conservation, invariance) and
 * tests/test_oracle_evolve_pins.py (P14: adiabatic compression of a hypersonic linear velocity field,
 * rho*e_1 = rho*e_0 (1 + gamma A dt) after one stage and the Heun closed form after two -- fixes the sign
 * of p_c div(u_face), the state p_c is taken from and every direction's dxinv; P15: a step in e moved by
 * the upwinded mass flux only -- fixes the side F_e takes e from).
 * The CTU update O12 (oracle_ctu_step, readings C1-C9 further down; pins P16-P22 in tests/test_oracle_ctu.py) and the
 * two-level ghost fill / restriction O13 (oracle_fill_from_coarse, oracle_average_down, readings A1-A6; pins in
 * tests/test_oracle_amr.py) carry their readings and pin lists in their own headers below.
 * Parity unpinned: behaviour when the small_dens / small_pres floors trigger
 * (exercised GPU-vs-oracle only).
 *
 * State layout (a1): SoA FP64, idx = (((b*NVAR + c)*NZt + k)*NYt + j)*NXt + i,
 * b = (bk*NBy + bj)*NBx + bi, valid zone (i,j,k) at padded (i+NG, j+NG, k+NG).
 * Components: 0 rho, 1 rho*u, 2 rho*v, 3 rho*w, 4 rho*E, 5 rho*e, 6.. rho*X_k.
 * Flux/conserved components (NFLUX = 5+nspec): the above without rho*e, i.e.
 * flux slot f maps to state component (f < 5 ? f : f+1).
 * Primitives (NQ = 5+nspec): 0 rho, 1 u, 2 v, 3 w, 4 p, 5.. X_k.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define HALF 0.5
static const double SIXTH = 1.0 / 6.0;

typedef struct {
    int32_t ndom[3];
    int32_t nbox[3];
    int32_t ng;
    int32_t nspec;
    int32_t bc_lo[3], bc_hi[3]; /* 0 periodic, 1 outflow, 2 reflect */
    double prob_lo[3], prob_hi[3];
    double gamma, cfl;
    double grav[3];
    double small_dens, small_pres;
    int32_t flatten;            /* 0: off (O1..O9 as in rounds before); 1: shock flattening O10 (needs ng >= 4) */
    int32_t evolve_eint;        /* 0: rho*e re-synchronised from rho*E after every stage (O7); 1: evolved rho*e
                                   with a dual-energy switch, O11 */
} oracle_params;

enum { BC_PERIODIC = 0, BC_OUTFLOW = 1, BC_REFLECT = 2, BC_EXTERNAL = 3 };
/* BC_EXTERNAL: the ghost zones across the face are somebody else's to fill (another shard, or the coarser level:
 * oracle_fill_from_coarse); oracle_fill_ghosts leaves them alone. */

static double dmin(double a, double b) { return a < b ? a : b; }
static double dmax(double a, double b) { return a > b ? a : b; }

/* ---- geometry helpers ---------------------------------------------------- */
typedef struct {
    int nvar, nflux, nq, ng;
    int nb[3];   /* valid zones per box            */
    int nt[3];   /* padded zones per box           */
    int NB[3];   /* boxes per dimension            */
    int nboxes;
    size_t comp_stride; /* doubles per (box, component) */
    size_t box_stride;  /* doubles per box              */
    double dx[3], dxinv[3];
} geom_t;

static int make_geom(const oracle_params *p, geom_t *g)
{
    if (!p) return -1;
    if (p->ng < 3 || p->nspec < 0) return -1;
    if (p->flatten != 0 && (p->flatten != 1 || p->ng < 4)) return -1;
    if (p->evolve_eint != 0 && p->evolve_eint != 1) return -1;
    g->nvar = 6 + p->nspec;
    g->nflux = 5 + p->nspec;
    g->nq = 5 + p->nspec;
    g->ng = p->ng;
    g->nboxes = 1;
    for (int d = 0; d < 3; ++d) {
        if (p->ndom[d] <= 0 || p->nbox[d] <= 0) return -1;
        if (p->ndom[d] % p->nbox[d] != 0) return -1;
        if ((p->bc_lo[d] == BC_PERIODIC) != (p->bc_hi[d] == BC_PERIODIC)) return -1;
        if (p->bc_lo[d] < 0 || p->bc_lo[d] > 3 || p->bc_hi[d] < 0 || p->bc_hi[d] > 3) return -1;
        g->nb[d] = p->nbox[d];
        g->nt[d] = p->nbox[d] + 2 * p->ng;
        g->NB[d] = p->ndom[d] / p->nbox[d];
        g->nboxes *= g->NB[d];
        g->dx[d] = (p->prob_hi[d] - p->prob_lo[d]) / p->ndom[d];
        g->dxinv[d] = 1.0 / g->dx[d];
    }
    g->comp_stride = (size_t)g->nt[0] * g->nt[1] * g->nt[2];
    g->box_stride = g->comp_stride * g->nvar;
    return 0;
}

static size_t zidx(const geom_t *g, int i, int j, int k) /* padded indices */
{
    return ((size_t)k * g->nt[1] + j) * g->nt[0] + i;
}

size_t oracle_state_doubles(const oracle_params *p)
{
    geom_t g;
    if (make_geom(p, &g)) return 0;
    return g.box_stride * (size_t)g.nboxes;
}

/* ---- O1 ghost fill --------------------------------- */
/* Maps a global index along dimension d to the valid global index that
 * supplies it, and reports whether a reflecting wall was crossed. */
static int map_global(const oracle_params *p, int d, int gidx, int *sgn)
{
    int n = p->ndom[d];
    *sgn = 1;
    if (gidx >= 0 && gidx < n) return gidx;
    int bc = gidx < 0 ? p->bc_lo[d] : p->bc_hi[d];
    if (bc == BC_PERIODIC) return ((gidx % n) + n) % n;
    if (bc == BC_OUTFLOW) return gidx < 0 ? 0 : n - 1;
    if (bc == BC_EXTERNAL) return -1;
    /* reflect */
    *sgn = -1;
    return gidx < 0 ? -1 - gidx : 2 * n - 1 - gidx;
}

int oracle_fill_ghosts(const oracle_params *p, double *U)
{
    geom_t g;
    if (make_geom(p, &g) || !U) return -1;
    const int ng = g.ng;
    for (int bk = 0; bk < g.NB[2]; ++bk)
    for (int bj = 0; bj < g.NB[1]; ++bj)
    for (int bi = 0; bi < g.NB[0]; ++bi) {
        size_t b = ((size_t)bk * g.NB[1] + bj) * g.NB[0] + bi;
        for (int kl = 0; kl < g.nt[2]; ++kl)
        for (int jl = 0; jl < g.nt[1]; ++jl)
        for (int il = 0; il < g.nt[0]; ++il) {
            int valid = il >= ng && il < ng + g.nb[0] && jl >= ng && jl < ng + g.nb[1] &&
                        kl >= ng && kl < ng + g.nb[2];
            if (valid) continue;
            int sg[3];
            int gx = map_global(p, 0, bi * g.nb[0] + il - ng, &sg[0]);
            int gy = map_global(p, 1, bj * g.nb[1] + jl - ng, &sg[1]);
            int gz = map_global(p, 2, bk * g.nb[2] + kl - ng, &sg[2]);
            if (gx < 0 || gy < 0 || gz < 0) continue;      /* across an external face: not ours to fill */
            size_t sb = ((size_t)(gz / g.nb[2]) * g.NB[1] + gy / g.nb[1]) * g.NB[0] + gx / g.nb[0];
            size_t sz = zidx(&g, gx % g.nb[0] + ng, gy % g.nb[1] + ng, gz % g.nb[2] + ng);
            size_t dz = zidx(&g, il, jl, kl);
            for (int c = 0; c < g.nvar; ++c) {
                double v = U[sb * g.box_stride + c * g.comp_stride + sz];
                if (c >= 1 && c <= 3 && sg[c - 1] < 0) v = -v;
                U[b * g.box_stride + c * g.comp_stride + dz] = v;
            }
        }
    }
    return 0;
}

/* ---- O2 primitives -------------------------------------- */
/* Uc: NVAR conserved values of one zone; q: NQ primitives out. */
void oracle_cons_to_prim(double gamma, double small_dens, double small_pres, int nspec,
                         const double *Uc, double *q)
{
    double rho = dmax(Uc[0], small_dens);
    double rinv = 1.0 / rho;
    q[0] = rho;
    q[1] = Uc[1] * rinv;
    q[2] = Uc[2] * rinv;
    q[3] = Uc[3] * rinv;
    q[4] = dmax((gamma - 1.0) * Uc[5], small_pres);
    for (int s = 0; s < nspec; ++s) q[5 + s] = Uc[6 + s] * rinv;
}

/* ---- O3 + O4 PPM along one line (CW84 eqs. 1.6-1.8, 1.10) ---------------- */
/* a[0..n-1] zone averages.  Outputs (arrays of length n):
 *   s[i]   limited slope of zone i,                 valid for i = 1..n-2
 *   e[i]   edge value between zones i and i+1,      valid for i = 1..n-3
 *   aL[i], aR[i] monotonised parabola edges of zone i, valid for i = 2..n-3
 * Entries outside the valid ranges are set to 0. */
void oracle_ppm_line(const double *a, int n, double *s, double *e, double *aL, double *aR)
{
    for (int i = 0; i < n; ++i) { s[i] = 0.0; e[i] = 0.0; aL[i] = 0.0; aR[i] = 0.0; }
    for (int i = 1; i <= n - 2; ++i) {
        double dp = a[i + 1] - a[i];
        double dm = a[i] - a[i - 1];
        double dc = HALF * (a[i + 1] - a[i - 1]);
        if (dp * dm > 0.0) {
            double lim = dmin(fabs(dc), dmin(2.0 * fabs(dp), 2.0 * fabs(dm)));
            s[i] = copysign(lim, dc);
        } else {
            s[i] = 0.0;
        }
    }
    for (int i = 1; i <= n - 3; ++i)
        e[i] = a[i] + HALF * (a[i + 1] - a[i]) - SIXTH * (s[i + 1] - s[i]);
    for (int i = 2; i <= n - 3; ++i) {
        double l = e[i - 1], r = e[i], ac = a[i];
        if ((r - ac) * (ac - l) <= 0.0) {
            l = ac;
            r = ac;
        } else {
            double d = r - l;
            double m = ac - HALF * (l + r);
            double t = d * d * SIXTH;
            if (d * m > t) l = 3.0 * ac - 2.0 * r;
            else if (-t > d * m) r = 3.0 * ac - 2.0 * l;
        }
        aL[i] = l;
        aR[i] = r;
    }
}

/* ---- O5 HLLC (Toro star-state form, Davis wave speeds; S6, S7, S8) ------- */
/* dir: 0,1,2.  qL, qR: NQ primitives of the left/right face states.
 * F: NFLUX fluxes out (rho, rho*u, rho*v, rho*w, rho*E, rho*X_k). */
/* O5 + the face-normal velocity of the HLLC fan (O11, reading G2): the contact speed SM between the
 * two acoustic waves, the left / right normal velocity where the whole fan lies on one side. */
void oracle_hllc_u(int dir, double gamma, double small_dens, double small_pres, int nspec,
                   const double *qL, const double *qR, double *F, double *uface)
{
    const double gm1inv = 1.0 / (gamma - 1.0);
    double rK[2], vK[2][3], pK[2], nK[2], rinvK[2], cK[2], EK[2], FK[2][5], UK[2][5];
    const double *q[2] = { qL, qR };
    for (int K = 0; K < 2; ++K) {
        rK[K] = dmax(q[K][0], small_dens);
        pK[K] = dmax(q[K][4], small_pres);
        vK[K][0] = q[K][1]; vK[K][1] = q[K][2]; vK[K][2] = q[K][3];
        nK[K] = vK[K][dir];
        rinvK[K] = 1.0 / rK[K];
        cK[K] = sqrt(gamma * pK[K] * rinvK[K]);
        EK[K] = pK[K] * gm1inv +
                HALF * rK[K] * (vK[K][0] * vK[K][0] + vK[K][1] * vK[K][1] + vK[K][2] * vK[K][2]);
        FK[K][0] = rK[K] * nK[K];
        for (int c = 0; c < 3; ++c) {
            FK[K][1 + c] = rK[K] * nK[K] * vK[K][c];
            if (c == dir) FK[K][1 + c] = FK[K][1 + c] + pK[K];
        }
        FK[K][4] = (EK[K] + pK[K]) * nK[K];
        UK[K][0] = rK[K];
        for (int c = 0; c < 3; ++c) UK[K][1 + c] = rK[K] * vK[K][c];
        UK[K][4] = EK[K];
    }
    double SL = dmin(nK[0] - cK[0], nK[1] - cK[1]);
    double SR = dmax(nK[0] + cK[0], nK[1] + cK[1]);
    if (SL >= 0.0) {
        for (int c = 0; c < 5; ++c) F[c] = FK[0][c];
        *uface = nK[0];
    } else if (SR <= 0.0) {
        for (int c = 0; c < 5; ++c) F[c] = FK[1][c];
        *uface = nK[1];
    } else {
        double mL = rK[0] * (SL - nK[0]);
        double mR = rK[1] * (SR - nK[1]);
        double SM = (pK[1] - pK[0] + mL * nK[0] - mR * nK[1]) / (mL - mR);
        int K = SM >= 0.0 ? 0 : 1;
        double S = K == 0 ? SL : SR;
        double mK = K == 0 ? mL : mR;
        double fac = mK / (S - SM);
        double Us[5];
        Us[0] = fac;
        for (int c = 0; c < 3; ++c) Us[1 + c] = fac * (c == dir ? SM : vK[K][c]);
        Us[4] = fac * (EK[K] * rinvK[K] + (SM - nK[K]) * (SM + pK[K] / mK));
        for (int c = 0; c < 5; ++c) F[c] = FK[K][c] + S * (Us[c] - UK[K][c]);
        *uface = SM;
    }
    for (int s = 0; s < nspec; ++s)
        F[5 + s] = F[0] * (F[0] >= 0.0 ? qL[5 + s] : qR[5 + s]);
}

void oracle_hllc(int dir, double gamma, double small_dens, double small_pres, int nspec,
                 const double *qL, const double *qR, double *F)
{
    double uface;
    oracle_hllc_u(dir, gamma, small_dens, small_pres, nspec, qL, qR, F, &uface);
}

/* ---- O2..O7 one RK stage of one box -------------------------------------- */
/* Us: stage state of this box (ghosts filled), Ubase: U0 of this box (stage 1
 * only), Uout: destination box (valid zones written). */
/* ---- O10 shock flattening (NEXT-1 of SURVEY 8(f), readings F1..F5) ----
 * Colella & Woodward 1984 appendix, in the single-pass form used by Castro-type codes, along one
 * line of n zones with pressure pr[] and the velocity component along the line un[]:
 *   dp   = pr[i+1] - pr[i-1]
 *   zeta = |dp| / max(small_pres, |pr[i+2] - pr[i-2]|)
 *   z    = min(1, max(0, 10*(zeta - 0.75)))                    (ramp from 0.75 to 0.85)
 *   chi  = (|dp| / min(pr[i+1], pr[i-1]) > 0.33  and  un[i-1] - un[i+1] >= 0) ? 1 : 0
 *   flat[i] = 1 - max(chi[i]*z[i], chi[i-s]*z[i-s]),  s = +1 if dp[i] > 0, -1 if dp[i] < 0;
 *             with dp[i] == 0 there is no high-pressure side and no neighbour is consulted (reading
 *             F3: keeps the scheme exactly mirror-symmetric; chi[i]*z[i] is 0 there anyway)
 * z, chi are defined for i = 2 .. n-3 and flat for i = 3 .. n-4; other entries are set to 1
 * (no flattening).  flat = 1 keeps the parabola, flat = 0 replaces it by the zone average. */
void oracle_flatten_line(const double *pr, const double *un, int n, double small_pres, double *flat)
{
    double *zc = (double *)malloc(sizeof(double) * (size_t)n);   /* chi*z */
    double *dpl = (double *)malloc(sizeof(double) * (size_t)n);
    for (int i = 0; i < n; ++i) { zc[i] = 0.0; dpl[i] = 0.0; flat[i] = 1.0; }
    for (int i = 2; i <= n - 3; ++i) {
        double dp = pr[i + 1] - pr[i - 1];
        double den = dmax(small_pres, fabs(pr[i + 2] - pr[i - 2]));
        double zeta = fabs(dp) / den;
        double z = dmin(1.0, dmax(0.0, 10.0 * (zeta - 0.75)));
        double chi = 0.0;
        if (fabs(dp) / dmin(pr[i + 1], pr[i - 1]) > 0.33 && un[i - 1] - un[i + 1] >= 0.0) chi = 1.0;
        zc[i] = chi * z;
        dpl[i] = dp;
    }
    for (int i = 3; i <= n - 4; ++i) {
        double nbr = 0.0;
        if (dpl[i] > 0.0) nbr = zc[i - 1];
        else if (dpl[i] < 0.0) nbr = zc[i + 1];
        flat[i] = 1.0 - dmax(zc[i], nbr);
    }
    free(dpl); free(zc);
}

static void advance_box(const oracle_params *p, const geom_t *g, int stage, double dt,
                        const double *Us, const double *Ubase, double *Uout)
{
    const int ng = g->ng, nq = g->nq, nflux = g->nflux, nvar = g->nvar;
    const int evolve = p->evolve_eint;
    const int nqx = nq + (evolve ? 1 : 0);   /* O11: e = rho*e / rho is one more reconstructed scalar (G1) */
    const size_t cs = g->comp_stride;
    /* O2: primitives on every padded zone */
    double *q = (double *)malloc(sizeof(double) * cs * nqx);
    double *Uc = (double *)malloc(sizeof(double) * nvar);
    double *qz = (double *)malloc(sizeof(double) * nq);
    for (size_t z = 0; z < cs; ++z) {
        for (int c = 0; c < nvar; ++c) Uc[c] = Us[c * cs + z];
        oracle_cons_to_prim(p->gamma, p->small_dens, p->small_pres, p->nspec, Uc, qz);
        for (int c = 0; c < nq; ++c) q[c * cs + z] = qz[c];
        if (evolve) q[nq * cs + z] = Uc[5] * (1.0 / dmax(Uc[0], p->small_dens));
    }
    /* O10 (optional): multi-dimensional flattening coefficient = min over the three directions of
     * the line coefficient, on zones -1 .. nb in every direction (1 elsewhere) */
    double *flatn = NULL;
    if (p->flatten) {
        flatn = (double *)malloc(sizeof(double) * cs);
        for (size_t z = 0; z < cs; ++z) flatn[z] = 1.0;
        int nm = 0;
        for (int d = 0; d < 3; ++d) if (g->nt[d] > nm) nm = g->nt[d];
        double *pl = (double *)malloc(sizeof(double) * nm);
        double *ul = (double *)malloc(sizeof(double) * nm);
        double *fl = (double *)malloc(sizeof(double) * nm);
        for (int d = 0; d < 3; ++d) {
            const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
            for (int t2 = ng - 1; t2 <= ng + g->nb[d2]; ++t2)
            for (int t1 = ng - 1; t1 <= ng + g->nb[d1]; ++t1) {
                int ijk[3];
                ijk[d1] = t1; ijk[d2] = t2;
                for (int m = 0; m < g->nt[d]; ++m) {
                    ijk[d] = m;
                    size_t z = zidx(g, ijk[0], ijk[1], ijk[2]);
                    pl[m] = q[4 * cs + z];
                    ul[m] = q[(1 + d) * cs + z];
                }
                oracle_flatten_line(pl, ul, g->nt[d], p->small_pres, fl);
                for (int m = ng - 1; m <= ng + g->nb[d]; ++m) {
                    ijk[d] = m;
                    size_t z = zidx(g, ijk[0], ijk[1], ijk[2]);
                    flatn[z] = dmin(flatn[z], fl[m]);
                }
            }
        }
        free(fl); free(ul); free(pl);
    }
    /* O3-O5: face fluxes per direction.  F[d] holds NFLUX x (faces of d),
     * face (i,j,k) of direction d = low face of valid zone (i,j,k), with the
     * index along d running 0..nb[d]. */
    double *F[3], *Fe[3], *Uf[3];
    size_t fdim[3][3];
    for (int d = 0; d < 3; ++d) {
        for (int e = 0; e < 3; ++e) fdim[d][e] = g->nb[e] + (e == d ? 1 : 0);
        F[d] = (double *)malloc(sizeof(double) * nflux * fdim[d][0] * fdim[d][1] * fdim[d][2]);
        Fe[d] = (double *)malloc(sizeof(double) * fdim[d][0] * fdim[d][1] * fdim[d][2]);   /* flux of rho*e (O11) */
        Uf[d] = (double *)malloc(sizeof(double) * fdim[d][0] * fdim[d][1] * fdim[d][2]);   /* face-normal velocity */
    }
    int nmax = 0;
    for (int d = 0; d < 3; ++d) if (g->nt[d] > nmax) nmax = g->nt[d];
    double *line = (double *)malloc(sizeof(double) * nmax * nqx);
    double *sl = (double *)malloc(sizeof(double) * nmax);
    double *ed = (double *)malloc(sizeof(double) * nmax);
    double *lL = (double *)malloc(sizeof(double) * nmax * nqx);
    double *lR = (double *)malloc(sizeof(double) * nmax * nqx);
    double *fL = (double *)malloc(sizeof(double) * nq);
    double *fR = (double *)malloc(sizeof(double) * nq);
    double *Ff = (double *)malloc(sizeof(double) * nflux);
    for (int d = 0; d < 3; ++d) {
        const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
        const int n = g->nb[d] + 6; /* zones -3 .. nb+2 along d */
        const size_t fcs = fdim[d][0] * fdim[d][1] * fdim[d][2];
        for (int t2 = 0; t2 < g->nb[d2]; ++t2)
        for (int t1 = 0; t1 < g->nb[d1]; ++t1) {
            int ijk[3];
            ijk[d1] = t1 + ng;
            ijk[d2] = t2 + ng;
            for (int c = 0; c < nqx; ++c) {
                for (int m = 0; m < n; ++m) {
                    ijk[d] = m - 3 + ng;
                    line[c * nmax + m] = q[c * cs + zidx(g, ijk[0], ijk[1], ijk[2])];
                }
                oracle_ppm_line(line + c * nmax, n, sl, ed, lL + c * nmax, lR + c * nmax);
                if (flatn) {   /* O10: blend the monotonised parabola with the zone average */
                    for (int m = 2; m <= n - 3; ++m) {
                        ijk[d] = m - 3 + ng;
                        const double f = flatn[zidx(g, ijk[0], ijk[1], ijk[2])];
                        const double omf = 1.0 - f;
                        lL[c * nmax + m] = f * lL[c * nmax + m] + omf * line[c * nmax + m];
                        lR[c * nmax + m] = f * lR[c * nmax + m] + omf * line[c * nmax + m];
                    }
                }
            }
            /* face f (0..nb[d]) lies between line zones m = f+2 and m = f+3 */
            for (int f = 0; f <= g->nb[d]; ++f) {
                for (int c = 0; c < nq; ++c) {
                    fL[c] = lR[c * nmax + f + 2];
                    fR[c] = lL[c * nmax + f + 3];
                }
                double uface;
                oracle_hllc_u(d, p->gamma, p->small_dens, p->small_pres, p->nspec, fL, fR, Ff, &uface);
                int fi[3];
                fi[d] = f; fi[d1] = t1; fi[d2] = t2;
                size_t fz = ((size_t)fi[2] * fdim[d][1] + fi[1]) * fdim[d][0] + fi[0];
                for (int c = 0; c < nflux; ++c) F[d][c * fcs + fz] = Ff[c];
                if (evolve) {   /* G1: passive upwinding of e with the mass flux, like a species (S7) */
                    const double eL = lR[nq * nmax + f + 2], eR = lL[nq * nmax + f + 3];
                    Fe[d][fz] = Ff[0] * (Ff[0] >= 0.0 ? eL : eR);
                    Uf[d][fz] = uface;
                }
            }
        }
    }
    /* O6 + O7 */
    const int has_grav = !(p->grav[0] == 0.0 && p->grav[1] == 0.0 && p->grav[2] == 0.0);
    const double floor_rhoe = p->small_pres * (1.0 / (p->gamma - 1.0));
    double *L = (double *)malloc(sizeof(double) * nflux);
    for (int k = 0; k < g->nb[2]; ++k)
    for (int j = 0; j < g->nb[1]; ++j)
    for (int i = 0; i < g->nb[0]; ++i) {
        size_t z = zidx(g, i + ng, j + ng, k + ng);
        size_t fx0 = ((size_t)k * fdim[0][1] + j) * fdim[0][0] + i, fx1 = fx0 + 1;
        size_t fy0 = ((size_t)k * fdim[1][1] + j) * fdim[1][0] + i, fy1 = fy0 + fdim[1][0];
        size_t fz0 = ((size_t)k * fdim[2][1] + j) * fdim[2][0] + i, fz1 = fz0 + fdim[2][0] * fdim[2][1];
        size_t fcx = fdim[0][0] * fdim[0][1] * fdim[0][2];
        size_t fcy = fdim[1][0] * fdim[1][1] * fdim[1][2];
        size_t fcz = fdim[2][0] * fdim[2][1] * fdim[2][2];
        for (int c = 0; c < nflux; ++c) {
            L[c] = -(F[0][c * fcx + fx1] - F[0][c * fcx + fx0]) * g->dxinv[0]
                   - (F[1][c * fcy + fy1] - F[1][c * fcy + fy0]) * g->dxinv[1]
                   - (F[2][c * fcz + fz1] - F[2][c * fcz + fz0]) * g->dxinv[2];
        }
        if (has_grav) {
            double rho = Us[0 * cs + z], mx = Us[1 * cs + z], my = Us[2 * cs + z], mz = Us[3 * cs + z];
            L[1] += rho * p->grav[0];
            L[2] += rho * p->grav[1];
            L[3] += rho * p->grav[2];
            L[4] += mx * p->grav[0] + my * p->grav[1] + mz * p->grav[2];
        }
        for (int c = 0; c < nflux; ++c) {
            int sc = c < 5 ? c : c + 1;
            double unew;
            if (stage == 0) unew = Us[sc * cs + z] + dt * L[c];
            else unew = HALF * Ubase[sc * cs + z] + HALF * (Us[sc * cs + z] + dt * L[c]);
            Uout[sc * cs + z] = unew;
        }
        {   /* rho*e re-synchronisation (O7, S2) */
            double rho = Uout[0 * cs + z], mx = Uout[1 * cs + z], my = Uout[2 * cs + z],
                   mz = Uout[3 * cs + z], rE = Uout[4 * cs + z];
            double K = HALF * (mx * mx + my * my + mz * mz) / rho;
            double re = rE - K;
            if (evolve) {
                /* O11 (G3-G5): rho*e advanced by its own equation,
                 *   d(rho e)/dt = -div(F_rho e) - p div(u_face),  p = cell pressure of the stage state,
                 * and used instead of rho*E - K wherever the latter is a small difference of large
                 * numbers: rho*E - K <= eta2 * rho*E, eta2 = 1e-4 (dual-energy switch) */
                double Le = -(Fe[0][fx1] - Fe[0][fx0]) * g->dxinv[0]
                            - (Fe[1][fy1] - Fe[1][fy0]) * g->dxinv[1]
                            - (Fe[2][fz1] - Fe[2][fz0]) * g->dxinv[2];
                double divu = (Uf[0][fx1] - Uf[0][fx0]) * g->dxinv[0]
                              + (Uf[1][fy1] - Uf[1][fy0]) * g->dxinv[1]
                              + (Uf[2][fz1] - Uf[2][fz0]) * g->dxinv[2];
                double pc = dmax((p->gamma - 1.0) * Us[5 * cs + z], p->small_pres);
                Le = Le - pc * divu;
                double rev;
                if (stage == 0) rev = Us[5 * cs + z] + dt * Le;
                else rev = HALF * Ubase[5 * cs + z] + HALF * (Us[5 * cs + z] + dt * Le);
                if (!(re > 1.0e-4 * rE)) re = rev;
            }
            if (re < floor_rhoe) re = floor_rhoe;
            Uout[5 * cs + z] = re;
        }
    }
    free(L);
    free(Ff); free(fR); free(fL); free(lR); free(lL); free(ed); free(sl); free(line);
    for (int d = 0; d < 3; ++d) { free(F[d]); free(Fe[d]); free(Uf[d]); }
    free(flatn);
    free(qz); free(Uc); free(q);
}

/* stage 0: reads U0 (ghosts filled), writes valid zones of U1.
 * stage 1: reads U1 (ghosts filled) and U0, overwrites valid zones of U0. */
int oracle_advance_stage(const oracle_params *p, int stage, double dt, double *U0, double *U1)
{
    geom_t g;
    if (make_geom(p, &g) || !U0 || !U1) return -1;
    if (stage != 0 && stage != 1) return -1;
    /* boxes are independent within a stage; the loop over boxes
     * may run on several host threads without changing any bit of the result */
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < g.nboxes; ++b) {
        size_t off = (size_t)b * g.box_stride;
        if (stage == 0) advance_box(p, &g, 0, dt, U0 + off, NULL, U1 + off);
        else advance_box(p, &g, 1, dt, U1 + off, U0 + off, U0 + off);
    }
    return 0;
}

/* ---- O8 CFL timestep (S9, S10) ------------------------------------------- */
int oracle_estimate_dt(const oracle_params *p, const double *U0, double *dt_out)
{
    geom_t g;
    if (make_geom(p, &g) || !U0 || !dt_out) return -1;
    const int ng = g.ng;
    const size_t cs = g.comp_stride;
    double tmax = 0.0;
    int bad = 0;
    for (int b = 0; b < g.nboxes; ++b) {
        const double *Ub = U0 + (size_t)b * g.box_stride;
        for (int k = 0; k < g.nb[2]; ++k)
        for (int j = 0; j < g.nb[1]; ++j)
        for (int i = 0; i < g.nb[0]; ++i) {
            size_t z = zidx(&g, i + ng, j + ng, k + ng);
            double rho = dmax(Ub[0 * cs + z], p->small_dens);
            double rinv = 1.0 / rho;
            double u = Ub[1 * cs + z] * rinv, v = Ub[2 * cs + z] * rinv, w = Ub[3 * cs + z] * rinv;
            double pr = dmax((p->gamma - 1.0) * Ub[5 * cs + z], p->small_pres);
            double c = sqrt(p->gamma * pr * rinv);
            double t = (fabs(u) + c) * g.dxinv[0] + (fabs(v) + c) * g.dxinv[1] + (fabs(w) + c) * g.dxinv[2];
            if (!(t == t) || isinf(t)) bad = 1;
            if (t > tmax) tmax = t;
        }
    }
    if (bad || !(tmax > 0.0)) return -4;
    *dt_out = p->cfl / tmax;
    return 0;
}

/* ---- O9 conservation totals (Neumaier-compensated sum) ------------------- */
int oracle_conserved_totals(const oracle_params *p, const double *U, double *totals)
{
    geom_t g;
    if (make_geom(p, &g) || !U || !totals) return -1;
    const int ng = g.ng;
    const size_t cs = g.comp_stride;
    const double vol = g.dx[0] * g.dx[1] * g.dx[2];
    for (int c = 0; c < g.nflux; ++c) {
        int sc = c < 5 ? c : c + 1;
        double sum = 0.0, comp = 0.0;
        for (int b = 0; b < g.nboxes; ++b) {
            const double *Ub = U + (size_t)b * g.box_stride + sc * cs;
            for (int k = 0; k < g.nb[2]; ++k)
            for (int j = 0; j < g.nb[1]; ++j)
            for (int i = 0; i < g.nb[0]; ++i) {
                double x = Ub[zidx(&g, i + ng, j + ng, k + ng)];
                double t = sum + x;
                if (fabs(sum) >= fabs(x)) comp += (sum - t) + x;
                else comp += (x - t) + sum;
                sum = t;
            }
        }
        totals[c] = (sum + comp) * vol;
    }
    return 0;
}

/* ---- one RK2 step (S17): estimate_dt; fill(0); stage(0); fill(1); stage(1) */
int oracle_step(const oracle_params *p, double *U0, double *U1, double *dt_out)
{
    double dt;
    int rc = oracle_estimate_dt(p, U0, &dt);
    if (rc) return rc;
    if ((rc = oracle_fill_ghosts(p, U0))) return rc;
    if ((rc = oracle_advance_stage(p, 0, dt, U0, U1))) return rc;
    if ((rc = oracle_fill_ghosts(p, U1))) return rc;
    if ((rc = oracle_advance_stage(p, 1, dt, U0, U1))) return rc;
    if (dt_out) *dt_out = dt;
    return 0;
}

/* Same as oracle_step but with dt supplied by the caller (used for sampled
 * sub-block parity at full size, where dt comes from the whole domain). */
int oracle_step_fixed_dt(const oracle_params *p, double *U0, double *U1, double dt)
{
    int rc;
    if ((rc = oracle_fill_ghosts(p, U0))) return rc;
    if ((rc = oracle_advance_stage(p, 0, dt, U0, U1))) return rc;
    if ((rc = oracle_fill_ghosts(p, U1))) return rc;
    if ((rc = oracle_advance_stage(p, 1, dt, U0, U1))) return rc;
    return 0;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Number of host threads of the loop over boxes from now on (n >= 1); no effect without OpenMP.  Results do
 * not depend on it bit for bit; bench.py uses it to time the oracle on one core as well as on all. */
void oracle_set_threads(int n)
{
#ifdef _OPENMP
    extern void omp_set_num_threads(int);
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* =====================================================================================================
 * O12 (readings C1..C9): the unsplit corner-transport-upwind (CTU)
 * update -- PPM reconstruction, characteristic tracing of the parabolas over the domain of dependence of
 * each wave, transverse flux corrections of the face states, ONE conservative flux evaluation per step.
 * This is the integrator family the paper's throughput numbers were measured with; the
 * paper prints none of it, so every formula below is a reading:
 *
 *  C1  one step, ghosts filled (ng >= 3):  U(n+1) = U(n) + dt * ( -dFx*dxinv - dFy*dyinv - dFz*dzinv + S ),
 *      association as O6; then the rho*e re-synchronisation of O7.  dt is O8's (sum form, S9).
 *  C2  per direction and primitive (rho, u, v, w, p, X_k): the monotonised parabola (aL, aR) of O3/O4, with
 *      da = aR - aL, a6 = 6*(a - 0.5*(aL + aR)).  For a wave of speed lam, sig = fabs(lam)*dt*dxinv:
 *        Ip(lam) = lam > 0 ? aR - 0.5*sig*(da - (1 - (2/3)*sig)*a6) : aR      (average over the part of the
 *        Im(lam) = lam < 0 ? aL + 0.5*sig*(da + (1 - (2/3)*sig)*a6) : aL       zone the wave sweeps; CW84 1.12)
 *      with the three speeds lam = un - c, un, un + c of the ZONE (c = sqrt(gamma*p/rho), zone averages).
 *  C3  state on the HIGH face of a zone (left state of face i+1/2), reference state and characteristic
 *      projection (Miller & Colella 2002 form):  ref = Ip(un + c) of (rho, un, p) if un + c > 0, else the zone
 *      average;  with d*m = ref - Ip(un - c), d*0 = ref - Ip(un), d*p = ref - Ip(un + c):
 *        am = 0.5*(dpm/(rho*c) - dum)*(rho/c),  ap = 0.5*(dpp/(rho*c) + dup)*(rho/c),  a0 = drho0 - dp0/(c*c)
 *        am = un - c > 0 ? -am : 0;  ap = un + c > 0 ? -ap : 0;  a0 = un > 0 ? -a0 : 0   (waves that reach the face)
 *        rho_f = rho_ref + ap + am + a0;  un_f = un_ref + (ap - am)*(c/rho);  p_f = p_ref + (ap + am)*(c*c)
 *      LOW face (right state of face i-1/2): the same with Im, ref = Im(un - c) if un - c < 0 else the zone
 *      average, and the waves kept are those with negative speed.
 *  C4  transverse velocities and mass fractions ride on the un wave: HIGH face Ip(un) if un > 0 else the zone
 *      average; LOW face Im(un) if un < 0 else the zone average.
 *  C5  floors rho >= small_dens, p >= small_pres on every face state (as O5 does inside the solver).
 *  C6  first fluxes F1_d = HLLC (O5) of the traced states on every face of direction d whose two zones lie in
 *      -1 .. nb of every direction.
 *  C7  transverse correction in the 6-solve form (the 2-D CTU of Colella 1990 applied pairwise; no
 *      intermediate corner solves -- Castro's 12-solve corner coupling is the alternative this reading does not
 *      take): the face state of zone z for direction d is turned into conserved variables
 *      (rho, rho*u, rho*v, rho*w, rho*E = p*gm1inv + 0.5*rho*|u|^2, rho*X_k), every d' != d subtracts
 *      0.5*dt*dxinv_d' * (F1_d'[high face of z] - F1_d'[low face of z]), d' in ascending order, and the result
 *      goes back to primitives (rho floored, p = max(gm1*(rho*E - 0.5*|m|^2/rho), small_pres)).
 *  C8  gravity: every face state's velocity gets + 0.5*dt*g after C7;  S_m = rho(n)*g,
 *      S_E = (m(n) + 0.5*dt*rho(n)*g) . g  (time-centred momentum: exact for a uniform state at rest).
 *  C9  final fluxes F_d = HLLC of the corrected states on the faces of the valid zones; update C1.
 *
 * Pins (tests/test_oracle_ctu.py): P16 free stream bitwise; P17 Sod against the exact solution; P18 a linear
 * density profile advected exactly (fails on a wrong sig factor or wave gate); P19 diagonal advection order;
 * P20 conservation 1e-13; P21 decomposition invariance bitwise, axis permutation; P22 gravity closed form.
 * Parity unpinned: behaviour when the floors of C5 / C7 trigger.
 * ===================================================================================================== */
static const double TWO3 = 2.0 / 3.0;

/* conserved (rho, mx, my, mz, rhoE, rhoX_k) <-> primitive (rho, u, v, w, p, X_k), NQ = NFLUX entries */
static void ctu_prim_to_cons(const oracle_params *p, int nspec, const double *q, double *Uc)
{
    const double gm1inv = 1.0 / (p->gamma - 1.0);
    Uc[0] = q[0];
    Uc[1] = q[0] * q[1]; Uc[2] = q[0] * q[2]; Uc[3] = q[0] * q[3];
    Uc[4] = q[4] * gm1inv + HALF * q[0] * (q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int s = 0; s < nspec; ++s) Uc[5 + s] = q[0] * q[5 + s];
}

static void ctu_cons_to_prim(const oracle_params *p, int nspec, const double *Uc, double *q)
{
    double rho = dmax(Uc[0], p->small_dens);
    double rinv = 1.0 / rho;
    q[0] = rho;
    q[1] = Uc[1] * rinv; q[2] = Uc[2] * rinv; q[3] = Uc[3] * rinv;
    double K = HALF * (Uc[1] * Uc[1] + Uc[2] * Uc[2] + Uc[3] * Uc[3]) * rinv;
    q[4] = dmax((p->gamma - 1.0) * (Uc[4] - K), p->small_pres);
    for (int s = 0; s < nspec; ++s) q[5 + s] = Uc[5 + s] * rinv;
}

/* C2: parabola averages over the domain of dependence of a wave */
static double ctu_Ip(double lam, double dtdx, double a, double aL, double aR)
{
    if (!(lam > 0.0)) return aR;
    double sig = fabs(lam) * dtdx;
    double da = aR - aL, a6 = 6.0 * (a - HALF * (aL + aR));
    return aR - HALF * sig * (da - (1.0 - TWO3 * sig) * a6);
}

static double ctu_Im(double lam, double dtdx, double a, double aL, double aR)
{
    if (!(lam < 0.0)) return aL;
    double sig = fabs(lam) * dtdx;
    double da = aR - aL, a6 = 6.0 * (a - HALF * (aL + aR));
    return aL + HALF * sig * (da + (1.0 - TWO3 * sig) * a6);
}

/* C3 + C4 + C5: traced states of ONE zone along direction d.  a, aL, aR: NQ zone averages and parabola edges.
 * qm: state on the low face (right state of face i-1/2), qp: state on the high face (left state of i+1/2). */
void oracle_ctu_trace(int d, double gamma, double small_dens, double small_pres, int nspec, double dtdx,
                      const double *a, const double *aL, const double *aR, double *qm, double *qp)
{
    const int nq = 5 + nspec, in = 1 + d;
    const double rho = a[0], un = a[in], pr = a[4];
    const double c = sqrt(gamma * pr / rho);
    const double lam[3] = { un - c, un, un + c };
    const int hv[3] = { 0, in, 4 };       /* rho, normal velocity, pressure */
    for (int side = 0; side < 2; ++side) {            /* 0: low face (Im), 1: high face (Ip) */
        double I[3][3];                                /* [wave][rho, un, p] */
        for (int w = 0; w < 3; ++w)
            for (int v = 0; v < 3; ++v)
                I[w][v] = side ? ctu_Ip(lam[w], dtdx, a[hv[v]], aL[hv[v]], aR[hv[v]])
                               : ctu_Im(lam[w], dtdx, a[hv[v]], aL[hv[v]], aR[hv[v]]);
        double ref[3];
        const int wr = side ? 2 : 0;                   /* the fastest wave towards this face */
        const int reaches = side ? (lam[2] > 0.0) : (lam[0] < 0.0);
        for (int v = 0; v < 3; ++v) ref[v] = reaches ? I[wr][v] : a[hv[v]];
        double dum = ref[1] - I[0][1], dpm = ref[2] - I[0][2];
        double drho0 = ref[0] - I[1][0], dp0 = ref[2] - I[1][2];
        double dup = ref[1] - I[2][1], dpp = ref[2] - I[2][2];
        double am = HALF * (dpm / (rho * c) - dum) * (rho / c);
        double ap = HALF * (dpp / (rho * c) + dup) * (rho / c);
        double a0 = drho0 - dp0 / (c * c);
        if (side) {
            am = lam[0] > 0.0 ? -am : 0.0; ap = lam[2] > 0.0 ? -ap : 0.0; a0 = lam[1] > 0.0 ? -a0 : 0.0;
        } else {
            am = lam[0] < 0.0 ? -am : 0.0; ap = lam[2] < 0.0 ? -ap : 0.0; a0 = lam[1] < 0.0 ? -a0 : 0.0;
        }
        double *qf = side ? qp : qm;
        qf[0] = dmax(ref[0] + ap + am + a0, small_dens);
        qf[in] = ref[1] + (ap - am) * (c / rho);
        qf[4] = dmax(ref[2] + (ap + am) * (c * c), small_pres);
        for (int v = 1; v < nq; ++v) {                 /* C4: passively advected variables */
            if (v == in || v == 4) continue;
            if (side) qf[v] = lam[1] > 0.0 ? ctu_Ip(lam[1], dtdx, a[v], aL[v], aR[v]) : a[v];
            else qf[v] = lam[1] < 0.0 ? ctu_Im(lam[1], dtdx, a[v], aL[v], aR[v]) : a[v];
        }
    }
}

/* one CTU step of one box: Us = U(n) with ghosts filled, Uout = U(n+1) on the valid zones */
static void ctu_box(const oracle_params *p, const geom_t *g, double dt, const double *Us, double *Uout)
{
    const int ng = g->ng, nq = g->nq, nflux = g->nflux, nvar = g->nvar, nspec = p->nspec;
    const size_t cs = g->comp_stride;
    const long st[3] = { 1, g->nt[0], (long)g->nt[0] * g->nt[1] };    /* padded strides */
    const int has_grav = !(p->grav[0] == 0.0 && p->grav[1] == 0.0 && p->grav[2] == 0.0);
    /* O2 on every padded zone */
    double *q = (double *)malloc(sizeof(double) * cs * nq);
    double *Uc = (double *)malloc(sizeof(double) * nvar);
    double *qz = (double *)malloc(sizeof(double) * nq);
    for (size_t z = 0; z < cs; ++z) {
        for (int c = 0; c < nvar; ++c) Uc[c] = Us[c * cs + z];
        oracle_cons_to_prim(p->gamma, p->small_dens, p->small_pres, nspec, Uc, qz);
        for (int c = 0; c < nq; ++c) q[c * cs + z] = qz[c];
    }
    /* C2-C5: traced face states of every zone -1 .. nb (all three directions), per direction */
    double *qm[3], *qp[3], *F1[3], *F2[3];
    for (int d = 0; d < 3; ++d) {
        qm[d] = (double *)calloc(cs * nq, sizeof(double));
        qp[d] = (double *)calloc(cs * nq, sizeof(double));
        F1[d] = (double *)calloc(cs * nflux, sizeof(double));      /* flux on the LOW face of a zone */
        F2[d] = (double *)calloc(cs * nflux, sizeof(double));
    }
    int nmax = 0;
    for (int d = 0; d < 3; ++d) if (g->nt[d] > nmax) nmax = g->nt[d];
    double *line = (double *)malloc(sizeof(double) * nmax * nq);
    double *sl = (double *)malloc(sizeof(double) * nmax);
    double *ed = (double *)malloc(sizeof(double) * nmax);
    double *lL = (double *)malloc(sizeof(double) * nmax * nq);
    double *lR = (double *)malloc(sizeof(double) * nmax * nq);
    double *za = (double *)malloc(sizeof(double) * nq), *zL = (double *)malloc(sizeof(double) * nq);
    double *zR = (double *)malloc(sizeof(double) * nq), *zm = (double *)malloc(sizeof(double) * nq);
    double *zp = (double *)malloc(sizeof(double) * nq), *Ff = (double *)malloc(sizeof(double) * nflux);
    for (int d = 0; d < 3; ++d) {
        const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
        const int n = g->nb[d] + 6;                                  /* line zones -3 .. nb+2 */
        const double dtdx = dt * g->dxinv[d];
        for (int t2 = -1; t2 <= g->nb[d2]; ++t2)
        for (int t1 = -1; t1 <= g->nb[d1]; ++t1) {
            int ijk[3];
            ijk[d1] = t1 + ng; ijk[d2] = t2 + ng;
            for (int c = 0; c < nq; ++c) {
                for (int m = 0; m < n; ++m) {
                    ijk[d] = m - 3 + ng;
                    line[c * nmax + m] = q[c * cs + zidx(g, ijk[0], ijk[1], ijk[2])];
                }
                oracle_ppm_line(line + c * nmax, n, sl, ed, lL + c * nmax, lR + c * nmax);
            }
            for (int m = 2; m <= n - 3; ++m) {                       /* zones -1 .. nb */
                for (int c = 0; c < nq; ++c) { za[c] = line[c * nmax + m]; zL[c] = lL[c * nmax + m]; zR[c] = lR[c * nmax + m]; }
                oracle_ctu_trace(d, p->gamma, p->small_dens, p->small_pres, nspec, dtdx, za, zL, zR, zm, zp);
                ijk[d] = m - 3 + ng;
                size_t z = zidx(g, ijk[0], ijk[1], ijk[2]);
                for (int c = 0; c < nq; ++c) { qm[d][c * cs + z] = zm[c]; qp[d][c * cs + z] = zp[c]; }
            }
        }
    }
    /* C6: first fluxes on the low face of zones 0 .. nb along d, -1 .. nb across */
    for (int d = 0; d < 3; ++d) {
        const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
        for (int t2 = -1; t2 <= g->nb[d2]; ++t2)
        for (int t1 = -1; t1 <= g->nb[d1]; ++t1)
        for (int m = 0; m <= g->nb[d]; ++m) {
            int ijk[3];
            ijk[d] = m + ng; ijk[d1] = t1 + ng; ijk[d2] = t2 + ng;
            size_t z = zidx(g, ijk[0], ijk[1], ijk[2]);
            for (int c = 0; c < nq; ++c) { zL[c] = qp[d][c * cs + z - st[d]]; zR[c] = qm[d][c * cs + z]; }
            oracle_hllc(d, p->gamma, p->small_dens, p->small_pres, nspec, zL, zR, Ff);
            for (int c = 0; c < nflux; ++c) F1[d][c * cs + z] = Ff[c];
        }
    }
    /* C7-C9: corrected states and final fluxes on the low face of zones 0 .. nb along d, valid across */
    double *Ucf = (double *)malloc(sizeof(double) * nflux);
    for (int d = 0; d < 3; ++d) {
        const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
        for (int t2 = 0; t2 < g->nb[d2]; ++t2)
        for (int t1 = 0; t1 < g->nb[d1]; ++t1)
        for (int m = 0; m <= g->nb[d]; ++m) {
            int ijk[3];
            ijk[d] = m + ng; ijk[d1] = t1 + ng; ijk[d2] = t2 + ng;
            size_t z = zidx(g, ijk[0], ijk[1], ijk[2]);
            for (int side = 0; side < 2; ++side) {                   /* 0: left state (zone m-1), 1: right (zone m) */
                const size_t zz = side ? z : z - st[d];
                const double *src = side ? qm[d] : qp[d];
                double *dst = side ? zR : zL;
                for (int c = 0; c < nq; ++c) za[c] = src[c * cs + zz];
                ctu_prim_to_cons(p, nspec, za, Ucf);
                for (int dd = 0; dd < 3; ++dd) {                     /* ascending d' != d */
                    if (dd == d) continue;
                    for (int c = 0; c < nflux; ++c)
                        Ucf[c] = Ucf[c] - HALF * dt * g->dxinv[dd] * (F1[dd][c * cs + zz + st[dd]] - F1[dd][c * cs + zz]);
                }
                ctu_cons_to_prim(p, nspec, Ucf, dst);
                if (has_grav)
                    for (int e = 0; e < 3; ++e) dst[1 + e] = dst[1 + e] + HALF * dt * p->grav[e];
            }
            oracle_hllc(d, p->gamma, p->small_dens, p->small_pres, nspec, zL, zR, Ff);
            for (int c = 0; c < nflux; ++c) F2[d][c * cs + z] = Ff[c];
        }
    }
    /* C1 + C8 + O7 */
    const double floor_rhoe = p->small_pres * (1.0 / (p->gamma - 1.0));
    double *L = (double *)malloc(sizeof(double) * nflux);
    for (int k = 0; k < g->nb[2]; ++k)
    for (int j = 0; j < g->nb[1]; ++j)
    for (int i = 0; i < g->nb[0]; ++i) {
        size_t z = zidx(g, i + ng, j + ng, k + ng);
        for (int c = 0; c < nflux; ++c)
            L[c] = -(F2[0][c * cs + z + st[0]] - F2[0][c * cs + z]) * g->dxinv[0]
                   - (F2[1][c * cs + z + st[1]] - F2[1][c * cs + z]) * g->dxinv[1]
                   - (F2[2][c * cs + z + st[2]] - F2[2][c * cs + z]) * g->dxinv[2];
        if (has_grav) {
            double rho = Us[0 * cs + z];
            for (int e = 0; e < 3; ++e) {
                L[1 + e] += rho * p->grav[e];
                L[4] += (Us[(1 + e) * cs + z] + HALF * dt * rho * p->grav[e]) * p->grav[e];
            }
        }
        for (int c = 0; c < nflux; ++c) {
            int sc = c < 5 ? c : c + 1;
            Uout[sc * cs + z] = Us[sc * cs + z] + dt * L[c];
        }
        double rho = Uout[0 * cs + z], mx = Uout[1 * cs + z], my = Uout[2 * cs + z], mz = Uout[3 * cs + z];
        double re = Uout[4 * cs + z] - HALF * (mx * mx + my * my + mz * mz) / rho;
        if (re < floor_rhoe) re = floor_rhoe;
        Uout[5 * cs + z] = re;
    }
    free(L); free(Ucf);
    free(Ff); free(zp); free(zm); free(zR); free(zL); free(za);
    free(lR); free(lL); free(ed); free(sl); free(line);
    for (int d = 0; d < 3; ++d) { free(F2[d]); free(F1[d]); free(qp[d]); free(qm[d]); }
    free(qz); free(Uc); free(q);
}

/* U0 <- one CTU step of U0 with the given dt (ghosts are filled here); U1 is work space of the same size */
int oracle_ctu_step_fixed_dt(const oracle_params *p, double *U0, double *U1, double dt)
{
    geom_t g;
    if (make_geom(p, &g) || !U0 || !U1) return -1;
    if (p->flatten || p->evolve_eint) return -1;       /* the options O10 / O11 belong to the method-of-lines path */
    int rc = oracle_fill_ghosts(p, U0);
    if (rc) return rc;
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < g.nboxes; ++b) {
        size_t off = (size_t)b * g.box_stride;
        ctu_box(p, &g, dt, U0 + off, U1 + off);
    }
    /* copy the new valid zones back (ghosts of U0 keep the old values and are refilled by the next step) */
    for (int b = 0; b < g.nboxes; ++b)
        for (int c = 0; c < g.nvar; ++c)
            for (int k = 0; k < g.nb[2]; ++k)
            for (int j = 0; j < g.nb[1]; ++j)
            for (int i = 0; i < g.nb[0]; ++i) {
                size_t z = (size_t)b * g.box_stride + c * g.comp_stride + zidx(&g, i + g.ng, j + g.ng, k + g.ng);
                U0[z] = U1[z];
            }
    return 0;
}

int oracle_ctu_step(const oracle_params *p, double *U0, double *U1, double *dt_out)
{
    double dt;
    int rc = oracle_estimate_dt(p, U0, &dt);
    if (rc) return rc;
    if ((rc = oracle_ctu_step_fixed_dt(p, U0, U1, dt))) return rc;
    if (dt_out) *dt_out = dt;
    return 0;
}

/* =====================================================================================================
 * O13 (second half; "a MultiFab ... at a given level of mesh refinement",
 * PAPER.md:149 refinement by factors of 4): two-level ghost fill.  The FINE level is a rectangular patch of the
 * coarse domain, refined by `ratio` (2 or 4) in every direction and tiled by its own boxes; its faces that lie
 * inside the coarse domain are BC_EXTERNAL.  Every fine ghost zone across such a face takes its NVAR components
 * from the coarse level by conservative linear interpolation.  The paper prints none of this; readings:
 *  A1  the fine global index gf (negative or >= ndom_f across a face) belongs to the coarse zone
 *      gc = lo + floor(gf / ratio), child position r = gf - ratio*floor(gf / ratio) in 0 .. ratio-1;
 *  A2  value = Uc + sx*xi_x + sy*xi_y + sz*xi_z (left to right), xi = (r + 0.5)/ratio - 0.5, per component;
 *  A3  slopes per coarse zone and dimension = the limited slope of O3 (CW84 1.7-1.8) of the coarse zone averages
 *      gc-1, gc, gc+1: monotone, exact for linear data, and the children of a zone average to its value;
 *  A4  coarse zones outside the coarse domain are the coarse level's own ghost zones (its boundary conditions
 *      apply; they must be filled first), looked up in the box nearest to them;
 *  A5  a fine ghost zone is filled here iff its index is across an EXTERNAL face in at least one dimension;
 *      the other fine ghost zones (fine-fine neighbours, physical boundaries of the patch) are O1's.
 * Pins (tests/test_oracle_amr.py): linear data reproduced bit for bit (dyadic coefficients), constants, child
 * means, a local extremum interpolates flat, every EXTERNAL-side ghost zone and no other zone is written, ratio 4.
 * ===================================================================================================== */
static int floor_div_i(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

/* value of component c at coarse GLOBAL zone gidx[3] (may lie up to ng zones outside the domain) */
static int coarse_at(const geom_t *gc, const double *Uc, int c, const int *gidx, double *out)
{
    size_t b = 0;
    int l[3];
    int bd[3];
    for (int d = 0; d < 3; ++d) {
        bd[d] = floor_div_i(gidx[d], gc->nb[d]);
        if (bd[d] < 0) bd[d] = 0;
        if (bd[d] > gc->NB[d] - 1) bd[d] = gc->NB[d] - 1;
        l[d] = gidx[d] - bd[d] * gc->nb[d] + gc->ng;
        if (l[d] < 0 || l[d] >= gc->nt[d]) return -1;
    }
    b = ((size_t)bd[2] * gc->NB[1] + bd[1]) * gc->NB[0] + bd[0];
    *out = Uc[b * gc->box_stride + (size_t)c * gc->comp_stride + zidx(gc, l[0], l[1], l[2])];
    return 0;
}

int oracle_fill_from_coarse(const oracle_params *pf, double *Uf, const oracle_params *pc, const double *Uc,
                            const int32_t *lo, int ratio)
{
    geom_t gf, gc;
    if (make_geom(pf, &gf) || make_geom(pc, &gc) || !Uf || !Uc || !lo) return -1;
    if ((ratio != 2 && ratio != 4) || pf->nspec != pc->nspec) return -1;
    for (int d = 0; d < 3; ++d) {
        if (pf->ndom[d] % ratio) return -1;
        if (lo[d] < 0 || lo[d] + pf->ndom[d] / ratio > pc->ndom[d]) return -1;
    }
    const int ng = gf.ng;
    for (int bk = 0; bk < gf.NB[2]; ++bk)
    for (int bj = 0; bj < gf.NB[1]; ++bj)
    for (int bi = 0; bi < gf.NB[0]; ++bi) {
        size_t b = ((size_t)bk * gf.NB[1] + bj) * gf.NB[0] + bi;
        const int bb[3] = { bi, bj, bk };
        for (int kl = 0; kl < gf.nt[2]; ++kl)
        for (int jl = 0; jl < gf.nt[1]; ++jl)
        for (int il = 0; il < gf.nt[0]; ++il) {
            const int ll[3] = { il, jl, kl };
            int g[3], cz[3], ext = 0;
            double xi[3];
            for (int d = 0; d < 3; ++d) {
                g[d] = bb[d] * gf.nb[d] + ll[d] - ng;
                if ((g[d] < 0 && pf->bc_lo[d] == BC_EXTERNAL) || (g[d] >= pf->ndom[d] && pf->bc_hi[d] == BC_EXTERNAL)) ext = 1;
                int q = floor_div_i(g[d], ratio);
                cz[d] = lo[d] + q;
                xi[d] = ((double)(g[d] - ratio * q) + 0.5) / (double)ratio - 0.5;
            }
            if (!ext) continue;
            size_t dz = b * gf.box_stride + zidx(&gf, il, jl, kl);
            for (int c = 0; c < gf.nvar; ++c) {
                double u0;
                if (coarse_at(&gc, Uc, c, cz, &u0)) return -1;
                double val = u0;
                for (int d = 0; d < 3; ++d) {
                    int cm[3] = { cz[0], cz[1], cz[2] }, cp[3] = { cz[0], cz[1], cz[2] };
                    cm[d] -= 1; cp[d] += 1;
                    double um, up;
                    if (coarse_at(&gc, Uc, c, cm, &um) || coarse_at(&gc, Uc, c, cp, &up)) return -1;
                    double dp = up - u0, dm = u0 - um, dc = HALF * (up - um), sl = 0.0;
                    if (dp * dm > 0.0) sl = copysign(dmin(fabs(dc), dmin(2.0 * fabs(dp), 2.0 * fabs(dm))), dc);
                    val = val + sl * xi[d];
                }
                Uf[dz + (size_t)c * gf.comp_stride] = val;
            }
        }
    }
    return 0;
}

/* O13, restriction (reading A6): every coarse VALID zone covered by the patch becomes the mean of its ratio^3 fine
 * children, summed in the order k, j, i (i innermost) and multiplied by 1/ratio^3 (exact: 1/8 or 1/64), all NVAR
 * components -- the conservative average-down of an AMR hierarchy (volumes of the children add up to the parent's).
 * Pins: constants and dyadic linear fields exact, the coarse total over the patch equals the fine total. */
int oracle_average_down(const oracle_params *pc, double *Uc, const oracle_params *pf, const double *Uf,
                        const int32_t *lo, int ratio)
{
    geom_t gf, gc;
    if (make_geom(pf, &gf) || make_geom(pc, &gc) || !Uf || !Uc || !lo) return -1;
    if ((ratio != 2 && ratio != 4) || pf->nspec != pc->nspec) return -1;
    for (int d = 0; d < 3; ++d) {
        if (pf->ndom[d] % ratio) return -1;
        if (lo[d] < 0 || lo[d] + pf->ndom[d] / ratio > pc->ndom[d]) return -1;
    }
    const double inv = 1.0 / (double)(ratio * ratio * ratio);
    for (int K = 0; K < pf->ndom[2] / ratio; ++K)
    for (int J = 0; J < pf->ndom[1] / ratio; ++J)
    for (int I = 0; I < pf->ndom[0] / ratio; ++I) {
        const int G[3] = { lo[0] + I, lo[1] + J, lo[2] + K };
        size_t cb = ((size_t)(G[2] / gc.nb[2]) * gc.NB[1] + G[1] / gc.nb[1]) * gc.NB[0] + G[0] / gc.nb[0];
        size_t cz = cb * gc.box_stride + zidx(&gc, G[0] % gc.nb[0] + gc.ng, G[1] % gc.nb[1] + gc.ng, G[2] % gc.nb[2] + gc.ng);
        for (int c = 0; c < gc.nvar; ++c) {
            double sum = 0.0;
            for (int kk = 0; kk < ratio; ++kk)
            for (int jj = 0; jj < ratio; ++jj)
            for (int ii = 0; ii < ratio; ++ii) {
                const int g[3] = { I * ratio + ii, J * ratio + jj, K * ratio + kk };
                size_t fb = ((size_t)(g[2] / gf.nb[2]) * gf.NB[1] + g[1] / gf.nb[1]) * gf.NB[0] + g[0] / gf.nb[0];
                sum = sum + Uf[fb * gf.box_stride + (size_t)c * gf.comp_stride +
                               zidx(&gf, g[0] % gf.nb[0] + gf.ng, g[1] % gf.nb[1] + gf.ng, g[2] % gf.nb[2] + gf.ng)];
            }
            Uc[cz + (size_t)c * gc.comp_stride] = sum * inv;
        }
    }
    return 0;
}
