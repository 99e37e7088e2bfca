"""Seeded synthetic workloads (the five BASELINE.json configs) -- input generation ONLY.

This module holds none of the method's arithmetic (no EOS inversion, reconstruction,
Riemann solve, update or reduction): it writes initial conserved states in layout a1 and
is the one module that both the CUDA path's tests/bench and the CPU oracle's tests use,
so that both sides see bit-identical inputs (
sec. 8(d) table of synthetic inputs).  It depends on numpy only.

Layout a1 ("a four-dimensional array" per Fab; BASELINE.json north_star
"SoA FP64 per component per box"):
    U[b, c, k, j, i]  with shape (nboxes, NVAR, nbz+2NG, nby+2NG, nbx+2NG), C-contiguous,
    b = (bk*NBy + bj)*NBx + bi, valid zone (i,j,k) stored at (i+NG, j+NG, k+NG).
Components: 0 rho, 1..3 rho*(u,v,w), 4 rho*E, 5 rho*e, 6.. rho*X_k.

Random numbers (S15): counter based and decomposition independent,
    u64 = splitmix64(seed ^ (stream << 56) ^ global_zone_index),  U = (u64 >> 11) * 2**-53.
"""
from __future__ import annotations

import copy
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np

PERIODIC, OUTFLOW, REFLECT = 0, 1, 2
RHO, MX, MY, MZ, EDEN, EINT, FS = 0, 1, 2, 3, 4, 5, 6


@dataclass
class Workload:
    name: str
    kind: str               # "sod" | "sedov" | "random" | "atmosphere" | "uniform"
    params: dict            # keys of the C struct hydro_params
    steps: int
    seed: int = 0
    extra: dict = field(default_factory=dict)

    # ---- derived layout numbers -------------------------------------------------
    @property
    def nspec(self): return int(self.params["nspec"])
    @property
    def nvar(self): return 6 + self.nspec
    @property
    def nflux(self): return 5 + self.nspec
    @property
    def ng(self): return int(self.params["ng"])
    @property
    def nb(self): return tuple(int(x) for x in self.params["nbox"])
    @property
    def NB(self): return tuple(int(n) // int(b) for n, b in zip(self.params["ndom"], self.params["nbox"]))
    @property
    def nboxes(self): return int(np.prod(self.NB))
    @property
    def nt(self): return tuple(b + 2 * self.ng for b in self.nb)
    @property
    def zones(self): return int(np.prod([int(x) for x in self.params["ndom"]]))
    @property
    def dx(self):
        p = self.params
        return tuple((p["prob_hi"][d] - p["prob_lo"][d]) / p["ndom"][d] for d in range(3))
    @property
    def state_shape(self):
        nt = self.nt
        return (self.nboxes, self.nvar, nt[2], nt[1], nt[0])
    @property
    def state_bytes(self): return int(np.prod(self.state_shape)) * 8


def _params(ndom, nbox, nspec, bc_lo, bc_hi, prob_hi, gamma, cfl, grav=(0.0, 0.0, 0.0), ng=4):
    return dict(ndom=list(ndom), nbox=list(nbox), ng=ng, nspec=nspec, bc_lo=list(bc_lo), bc_hi=list(bc_hi),
                prob_lo=[0.0, 0.0, 0.0], prob_hi=list(prob_hi), gamma=gamma, cfl=cfl, grav=list(grav),
                small_dens=1e-12, small_pres=1e-14)


def config(n: int, ndom=None, nbox=None, nspec=None, steps=None) -> Workload:
    """BASELINE.json configs[n-1] (n = 1..5).  ndom/nbox/nspec/steps override the size for
    reduced parity-test instances of the same recipe (the physical zone size of configs 1, 2
    and 4 follows the zone count so that the recipe stays self-consistent)."""
    if n == 1:      # Sod: 128x4x4, one box, outflow x, periodic y/z, 1 species (S14, S20)
        ndom = list(ndom or (128, 4, 4)); nbox = list(nbox or ndom)
        dx = 1.0 / ndom[0]
        p = _params(ndom, nbox, 1 if nspec is None else nspec, (OUTFLOW, PERIODIC, PERIODIC),
                    (OUTFLOW, PERIODIC, PERIODIC), (1.0, ndom[1] * dx, ndom[2] * dx), 1.4, 0.5)
        return Workload("cfg1_sod", "sod", p, steps or 20)
    if n == 2:      # Sedov: 128^3 in 4 boxes of 64x64x128, outflow (S19)
        ndom = list(ndom or (128, 128, 128)); nbox = list(nbox or (ndom[0] // 2, ndom[1] // 2, ndom[2]))
        p = _params(ndom, nbox, 0 if nspec is None else nspec, (OUTFLOW,) * 3, (OUTFLOW,) * 3,
                    (1.0, 1.0, 1.0), 1.4, 0.5)
        return Workload("cfg2_sedov", "sedov", p, steps or 50, extra=dict(E=1.0, rho0=1.0, p0=1e-5, rhot=3.5))
    if n == 3:      # periodic random flow: 256^3 in 64^3 boxes, 3 species
        ndom = list(ndom or (256,) * 3); nbox = list(nbox or (64,) * 3)
        p = _params(ndom, nbox, 3 if nspec is None else nspec, (PERIODIC,) * 3, (PERIODIC,) * 3,
                    (1.0, 1.0, 1.0), 5.0 / 3.0, 0.4)
        return Workload("cfg3_periodic", "random", p, steps or 10, seed=20070518)
    if n == 4:      # stratified atmosphere: 256x256x512 in 64^3 boxes, g_z = -1, 13 species (S14)
        ndom = list(ndom or (256, 256, 512)); nbox = list(nbox or (64,) * 3)
        Lz = 5.0
        dx = Lz / ndom[2]
        p = _params(ndom, nbox, 13 if nspec is None else nspec, (PERIODIC, PERIODIC, REFLECT),
                    (PERIODIC, PERIODIC, REFLECT), (ndom[0] * dx, ndom[1] * dx, Lz), 5.0 / 3.0, 0.4,
                    grav=(0.0, 0.0, -1.0))
        return Workload("cfg4_atmosphere", "atmosphere", p, steps or 10, seed=20070519)
    if n == 5:      # 512^3 in 128^3 boxes, 13 species, recipe of config 3
        ndom = list(ndom or (512,) * 3); nbox = list(nbox or (128,) * 3)
        p = _params(ndom, nbox, 13 if nspec is None else nspec, (PERIODIC,) * 3, (PERIODIC,) * 3,
                    (1.0, 1.0, 1.0), 5.0 / 3.0, 0.4)
        return Workload("cfg5_scaling", "random", p, steps or 5, seed=20070518)
    raise ValueError("config number must be 1..5")


def uniform(ndom, nbox, nspec, prim, bc=PERIODIC, gamma=1.4, cfl=0.5, grav=(0.0, 0.0, 0.0),
            prob_hi=(1.0, 1.0, 1.0), X=None) -> Workload:
    """Uniform state (rho,u,v,w,p) -- used by the free-stream / gravity / dt pins."""
    bcs = (bc,) * 3 if isinstance(bc, int) else tuple(bc)
    p = _params(ndom, nbox, nspec, bcs, bcs, prob_hi, gamma, cfl, grav)
    return Workload("uniform", "uniform", p, 1, extra=dict(prim=tuple(prim), X=X))


def with_boxes(wl: Workload, nbox) -> Workload:
    """Same problem, different box decomposition (pin P8)."""
    w2 = copy.deepcopy(wl)
    w2.params["nbox"] = list(nbox)
    return w2


# ---- counter-based RNG (S15) --------------------------------------------------------
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = x + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def uniform01(seed: int, stream: int, gidx: np.ndarray) -> np.ndarray:
    key = np.uint64(seed) ^ (np.uint64(stream) << np.uint64(56))
    u = splitmix64(gidx.astype(np.uint64) ^ key)
    return (u >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def _gidx(wl: Workload, lo, shape):
    """Global zone index for the window starting at global (x,y,z)=lo, periodic wrap;
    shape is (nz, ny, nx)."""
    nd = wl.params["ndom"]
    gx = (np.arange(lo[0], lo[0] + shape[2]) % nd[0]).astype(np.int64)
    gy = (np.arange(lo[1], lo[1] + shape[1]) % nd[1]).astype(np.int64)
    gz = (np.arange(lo[2], lo[2] + shape[0]) % nd[2]).astype(np.int64)
    return (gz[:, None, None] * nd[1] + gy[None, :, None]) * nd[0] + gx[None, None, :]


def _normal(wl, s1, s2, gidx, sigma):
    u1 = uniform01(wl.seed, s1, gidx)
    u2 = uniform01(wl.seed, s2, gidx)
    return sigma * np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)


def _dirichlet(wl, gidx, nspec):
    if nspec == 0:
        return np.zeros((0,) + gidx.shape)
    x = np.stack([-np.log(1.0 - uniform01(wl.seed, 8 + k, gidx)) for k in range(nspec)])
    return x / x.sum(axis=0, keepdims=True)


def _filtered_velocity(wl, s1, s2, lo, shape, sigma):
    """N(0, sigma) field smoothed by a separable 3-point box filter with periodic wrap."""
    lo1 = (lo[0] - 1, lo[1] - 1, lo[2] - 1)
    sh1 = (shape[0] + 2, shape[1] + 2, shape[2] + 2)
    v = _normal(wl, s1, s2, _gidx(wl, lo1, sh1), sigma)
    third = 1.0 / 3.0
    v = (v[:, :, :-2] + v[:, :, 1:-1] + v[:, :, 2:]) * third
    v = (v[:, :-2, :] + v[:, 1:-1, :] + v[:, 2:, :]) * third
    v = (v[:-2, :, :] + v[1:-1, :, :] + v[2:, :, :]) * third
    return v


def primitives(wl: Workload, lo, shape):
    """Primitive fields (rho,u,v,w,p) and X[nspec] on the window of valid global zones
    starting at lo=(x,y,z) with shape (nz,ny,nx)."""
    p = wl.params
    nd, dx = p["ndom"], wl.dx
    zeros = np.zeros(shape)
    xc = (np.arange(lo[0], lo[0] + shape[2]) + 0.5) * dx[0] + p["prob_lo"][0]
    yc = (np.arange(lo[1], lo[1] + shape[1]) + 0.5) * dx[1] + p["prob_lo"][1]
    zc = (np.arange(lo[2], lo[2] + shape[0]) + 0.5) * dx[2] + p["prob_lo"][2]
    ns = wl.nspec
    if wl.kind == "uniform":
        r, u, v, w, pr = wl.extra["prim"]
        X = wl.extra.get("X")
        X = np.full(ns, 1.0 / max(ns, 1)) if X is None else np.asarray(X, dtype=np.float64)
        return (zeros + r, zeros + u, zeros + v, zeros + w, zeros + pr,
                np.broadcast_to(X[:, None, None, None], (ns,) + tuple(shape)).copy())
    if wl.kind == "sod":
        gx = np.arange(lo[0], lo[0] + shape[2])
        left = (gx < nd[0] // 2)[None, None, :] & np.ones(shape, dtype=bool)
        rho = np.where(left, 1.0, 0.125)
        pr = np.where(left, 1.0, 0.1)
        X = np.zeros((ns,) + tuple(shape))
        if ns > 0:
            X[0] = np.where(left, 1.0, 0.0)
        return rho, zeros, zeros.copy(), zeros.copy(), pr, X
    if wl.kind == "sedov":
        ex = wl.extra
        # centre = domain centre (a zone corner); r measured in zones from zone centres
        rx = (np.arange(lo[0], lo[0] + shape[2]) + 0.5 - nd[0] / 2.0)
        ry = (np.arange(lo[1], lo[1] + shape[1]) + 0.5 - nd[1] / 2.0)
        rz = (np.arange(lo[2], lo[2] + shape[0]) + 0.5 - nd[2] / 2.0)
        r2 = rz[:, None, None] ** 2 + ry[None, :, None] ** 2 + rx[None, None, :] ** 2
        hot = r2 < ex["rhot"] ** 2
        nhot = sedov_hot_count(ex["rhot"])
        gm1 = p["gamma"] - 1.0
        rhoe_hot = ex["E"] / (nhot * dx[0] * dx[1] * dx[2])
        pr = np.where(hot, gm1 * rhoe_hot, ex["p0"])
        X = np.full((ns,) + tuple(shape), 1.0 / max(ns, 1))
        return zeros + ex["rho0"], zeros, zeros.copy(), zeros.copy(), pr, X
    if wl.kind == "random":
        g = _gidx(wl, lo, shape)
        rho = 1.0 + 0.1 * (2.0 * uniform01(wl.seed, 0, g) - 1.0)
        u = _filtered_velocity(wl, 1, 2, lo, shape, 0.3)
        v = _filtered_velocity(wl, 3, 4, lo, shape, 0.3)
        w = _filtered_velocity(wl, 5, 6, lo, shape, 0.3)
        return rho, u, v, w, zeros + 1.0, _dirichlet(wl, g, ns)
    if wl.kind == "atmosphere":
        g = _gidx(wl, lo, shape)
        Lz = p["prob_hi"][2] - p["prob_lo"][2]
        base = np.exp(-zc)[:, None, None] + zeros          # H = 1 (S14)
        mid = ((zc >= Lz / 3.0) & (zc < 2.0 * Lz / 3.0))[:, None, None]
        pert = 1.0 + 0.01 * (2.0 * uniform01(wl.seed, 0, g) - 1.0)
        rho = np.where(mid, base * pert, base)
        return rho, zeros, zeros.copy(), zeros.copy(), base.copy(), _dirichlet(wl, g, ns)
    raise ValueError(wl.kind)


def sedov_hot_count(rhot: float) -> int:
    """Number of zone centres within rhot zone widths of a zone corner (160 for 3.5)."""
    m = int(np.ceil(rhot)) + 1
    c = np.arange(-m, m) + 0.5
    r2 = c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2
    return int((r2 < rhot ** 2).sum())


def conserved_from_primitives(gamma, rho, u, v, w, pr, X):
    """Initial-condition bookkeeping: (rho,u,v,w,p,X) -> the NVAR stored components, with
    rho*e consistent with rho*E (rho*E = rho*e + 0.5*rho*|u|^2)."""
    out = np.empty((6 + X.shape[0],) + rho.shape)
    out[RHO] = rho
    out[MX], out[MY], out[MZ] = rho * u, rho * v, rho * w
    out[EINT] = pr / (gamma - 1.0)
    out[EDEN] = out[EINT] + 0.5 * rho * (u * u + v * v + w * w)
    for k in range(X.shape[0]):
        out[FS + k] = rho * X[k]
    return out


def fill_box(wl: Workload, b: int, out_box: np.ndarray, ghost_value: float = 0.0):
    """Write box b (shape (NVAR, NZt, NYt, NXt)) of the initial state; ghosts get ghost_value
    (the hot path overwrites them: the caller's ghosts 'may be garbage')."""
    NB, nb, ng = wl.NB, wl.nb, wl.ng
    bi, bj, bk = b % NB[0], (b // NB[0]) % NB[1], b // (NB[0] * NB[1])
    lo = (bi * nb[0], bj * nb[1], bk * nb[2])
    shape = (nb[2], nb[1], nb[0])
    cons = conserved_from_primitives(wl.params["gamma"], *primitives(wl, lo, shape))
    out_box[...] = ghost_value
    out_box[:, ng:ng + nb[2], ng:ng + nb[1], ng:ng + nb[0]] = cons


def initial_state(wl: Workload, out: np.ndarray | None = None, ghost_value: float = 0.0,
                  threads: int = 1) -> np.ndarray:
    """Whole initial state in layout a1 (host numpy).  `out` may be a preallocated (e.g.
    pinned) array of wl.state_shape."""
    if out is None:
        out = np.empty(wl.state_shape, dtype=np.float64)
    assert out.shape == wl.state_shape and out.dtype == np.float64
    if threads <= 1 or wl.nboxes == 1:
        for b in range(wl.nboxes):
            fill_box(wl, b, out[b], ghost_value)
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(lambda b: fill_box(wl, b, out[b], ghost_value), range(wl.nboxes)))
    return out


# ---- layout helpers for tests (no arithmetic) ---------------------------------------
def gather_valid(wl: Workload, U: np.ndarray) -> np.ndarray:
    """(NVAR, nz, ny, nx) global array assembled from the valid zones of every box."""
    NB, nb, ng = wl.NB, wl.nb, wl.ng
    nd = wl.params["ndom"]
    G = np.empty((wl.nvar, nd[2], nd[1], nd[0]))
    U = U.reshape(wl.state_shape)
    for b in range(wl.nboxes):
        bi, bj, bk = b % NB[0], (b // NB[0]) % NB[1], b // (NB[0] * NB[1])
        G[:, bk * nb[2]:(bk + 1) * nb[2], bj * nb[1]:(bj + 1) * nb[1], bi * nb[0]:(bi + 1) * nb[0]] = \
            U[b, :, ng:ng + nb[2], ng:ng + nb[1], ng:ng + nb[0]]
    return G


def scatter_valid(wl: Workload, G: np.ndarray, ghost_value: float = 0.0) -> np.ndarray:
    """Inverse of gather_valid: distribute a global (NVAR,nz,ny,nx) array over the boxes."""
    NB, nb, ng = wl.NB, wl.nb, wl.ng
    U = np.full(wl.state_shape, ghost_value)
    for b in range(wl.nboxes):
        bi, bj, bk = b % NB[0], (b // NB[0]) % NB[1], b // (NB[0] * NB[1])
        U[b, :, ng:ng + nb[2], ng:ng + nb[1], ng:ng + nb[0]] = \
            G[:, bk * nb[2]:(bk + 1) * nb[2], bj * nb[1]:(bj + 1) * nb[1], bi * nb[0]:(bi + 1) * nb[0]]
    return U
