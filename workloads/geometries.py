"""Synthetic vessel geometries and initial fields (inputs only, no LB arithmetic).

Conventions (shared by the oracle and by the library, see include/hlb.h):

* ``site_type`` is a C-contiguous ``uint8`` array of shape ``(nz, ny, nx)``; the linear
  voxel index is ``v = (z*ny + y)*nx + x``.
* 0 = solid, 1 = fluid, 2+k = ghost voxel of iolet ``k`` (never simulated; it only marks
  the links that cross iolet ``k``).
* "canonical site order" = ascending ``v`` over the fluid voxels; every per-site array
  (``rho0``, ``u0``) is in that order.

Recipes follow SURVEY.md §8(d) (BASELINE.json ``configs[0..4]``); the free parameters
the configs leave open are listed in DESIGN.md "Input recipe".
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

SOLID = 0
FLUID = 1
IOLET0 = 2  # ghost voxel of iolet k has type IOLET0 + k

PERIODIC_X, PERIODIC_Y, PERIODIC_Z = 1, 2, 4

CONFIG_NAMES = ("pipe", "cube", "aneurysm", "tree", "bigtree")


@dataclasses.dataclass
class Workload:
    name: str
    site_type: np.ndarray            # uint8 (nz, ny, nx)
    periodic: int                    # bit0 x, bit1 y, bit2 z
    tau: float
    iolet_rho: np.ndarray            # float64 (n_iolets,)
    steps: int                       # step count the config asks for
    rho0: Optional[np.ndarray] = None  # float64 (N,) canonical order, None => 1
    u0: Optional[np.ndarray] = None    # float64 (N, 3) canonical order, None => 0
    iolet_kind: Optional[np.ndarray] = None  # uint8 (n_iolets,): 0 density, 1 Ladd velocity; None => all 0
    iolet_u: Optional[np.ndarray] = None     # float64 (n_iolets, 3) velocities of the velocity iolets
    iolet_normal: Optional[np.ndarray] = None  # float64 (n_iolets, 3): normals of density iolets
    iolet_weight: Optional[np.ndarray] = None  # float64 (N,), canonical order: factor of u_k on the
                                               # velocity-iolet links of each site; None => 1
    wall_distance: Optional[np.ndarray] = None  # float64 (N, 27): BFL wall distances (include/hlb.h)
    scheme: str = "two_lattice"      # "two_lattice" | "aa"  (what the config asks for)
    store: str = "f64"               # "f64" | "f32"
    info: dict = dataclasses.field(default_factory=dict)

    @property
    def shape(self):
        nz, ny, nx = self.site_type.shape
        return nx, ny, nz

    @property
    def n_iolets(self) -> int:
        return int(self.iolet_rho.shape[0])

    def fluid_voxels(self) -> np.ndarray:
        """Canonical site list: ascending linear voxel indices of fluid voxels."""
        return np.flatnonzero(self.site_type.reshape(-1) == FLUID).astype(np.int64)

    @property
    def n_sites(self) -> int:
        return int(np.count_nonzero(self.site_type == FLUID))


# --------------------------------------------------------------------------- config 0
def pipe(radius: int = 8, length: int = 64, tau: float = 0.8, rho_in: float = 1.001,
         rho_out: float = 0.999, steps: int = 200) -> Workload:
    """Straight pipe along z (BASELINE configs[0]).

    Fluid where (x-R)^2 + (y-R)^2 <= R^2 for z = 1..length; z = 0 is the inlet ghost
    slice (type 2), z = length+1 the outlet ghost slice (type 3), on the same disc.
    R = 8, length = 64 gives N = 197*64 = 12,608.
    """
    n = 2 * radius + 1
    y, x = np.mgrid[0:n, 0:n]
    disc = (x - radius) ** 2 + (y - radius) ** 2 <= radius * radius
    st = np.zeros((length + 2, n, n), dtype=np.uint8)
    st[1:length + 1][:, disc] = FLUID
    st[0][disc] = IOLET0
    st[length + 1][disc] = IOLET0 + 1
    return Workload("pipe", st, 0, tau, np.array([rho_in, rho_out], dtype=np.float64), steps,
                    info={"radius": radius, "length": length})


# --------------------------------------------------------------------------- config 1
def periodic_cube(n: int = 128, tau: float = 0.6, u0: float = 0.01, steps: int = 1000,
                  nz: Optional[int] = None, with_state: bool = True) -> Workload:
    """Fully periodic all-fluid box with a z-invariant Taylor-Green vortex
    (BASELINE configs[1]; field: SURVEY.md §8(c) A12).

    u_x = u0 sin(kx) cos(ky), u_y = -u0 cos(kx) sin(ky), u_z = 0, rho = 1, k = 2 pi / n.
    """
    nz = n if nz is None else nz
    st = np.full((nz, n, n), FLUID, dtype=np.uint8)
    k = 2.0 * math.pi / n
    if not with_state:   # geometry only (rest state): the huge cube of the 64-bit-offset runs
        return Workload("cube", st, PERIODIC_X | PERIODIC_Y | PERIODIC_Z, tau,
                        np.zeros(0, dtype=np.float64), steps, info={"n": n, "u0": 0.0, "k": k})
    xs = np.arange(n, dtype=np.float64)
    sx, cx = np.sin(k * xs), np.cos(k * xs)
    ux2d = u0 * np.outer(cx, sx)          # [y, x] -> u0 sin(kx) cos(ky)
    uy2d = -u0 * np.outer(sx, cx)         # [y, x] -> -u0 cos(kx) sin(ky)
    u = np.zeros((nz, n, n, 3), dtype=np.float64)
    u[..., 0] = ux2d[None]
    u[..., 1] = uy2d[None]
    return Workload("cube", st, PERIODIC_X | PERIODIC_Y | PERIODIC_Z, tau,
                    np.zeros(0, dtype=np.float64), steps,
                    rho0=np.ones(nz * n * n, dtype=np.float64), u0=u.reshape(-1, 3),
                    info={"n": n, "u0": u0, "k": k})


# --------------------------------------------------------------------------- painting
def _paint(mask: np.ndarray, lo, hi, inside_fn, value: int, only_solid: bool = False,
           zchunk: int = 64) -> None:
    """Set mask[z,y,x] = value where inside_fn(X, Y, Z) holds, over the integer box
    [lo, hi] (inclusive, xyz order) clipped to the array."""
    nz, ny, nx = mask.shape
    x0, y0, z0 = (max(0, int(math.floor(v))) for v in lo)
    x1 = min(nx - 1, int(math.ceil(hi[0])))
    y1 = min(ny - 1, int(math.ceil(hi[1])))
    z1 = min(nz - 1, int(math.ceil(hi[2])))
    if x1 < x0 or y1 < y0 or z1 < z0:
        return
    X = np.arange(x0, x1 + 1, dtype=np.float64)[None, None, :]
    Y = np.arange(y0, y1 + 1, dtype=np.float64)[None, :, None]
    for za in range(z0, z1 + 1, zchunk):
        zb = min(z1 + 1, za + zchunk)
        Z = np.arange(za, zb, dtype=np.float64)[:, None, None]
        inside = inside_fn(X, Y, Z)
        sub = mask[za:zb, y0:y1 + 1, x0:x1 + 1]
        if only_solid:
            inside = inside & (sub == SOLID)
        sub[inside] = value


def _paint_ball(mask, c, r, value=FLUID, xclip=None):
    cx, cy, cz = c

    def inside(X, Y, Z):
        m = (X - cx) ** 2 + (Y - cy) ** 2 + (Z - cz) ** 2 <= r * r
        if xclip is not None:
            m = m & (X >= xclip[0]) & (X <= xclip[1])
        return m

    _paint(mask, (cx - r, cy - r, cz - r), (cx + r, cy + r, cz + r), inside, value)


def _paint_cylinder(mask, p, d, r, a_lo, a_hi, value=FLUID, only_solid=False, lo_open=False):
    """Voxels whose axial coordinate a = (x - p).d lies in [a_lo, a_hi] (or (a_lo, a_hi]
    when lo_open) and whose distance from the axis is <= r."""
    p = np.asarray(p, dtype=np.float64)
    d = np.asarray(d, dtype=np.float64)
    e0, e1 = p + a_lo * d, p + a_hi * d
    lo = np.minimum(e0, e1) - r
    hi = np.maximum(e0, e1) + r

    def inside(X, Y, Z):
        rx, ry, rz = X - p[0], Y - p[1], Z - p[2]
        a = rx * d[0] + ry * d[1] + rz * d[2]
        rad2 = rx * rx + ry * ry + rz * rz - a * a
        ok_lo = (a > a_lo) if lo_open else (a >= a_lo)
        return ok_lo & (a <= a_hi) & (rad2 <= r * r)

    _paint(mask, lo, hi, inside, value, only_solid=only_solid)


# --------------------------------------------------------------------------- config 2
def aneurysm(scale: float = 1.0, tau: float = 0.55, rho_in: float = 1.0005,
             rho_out: float = 0.9995, steps: int = 2000) -> Workload:
    """Vessel of radius 20 on a sine centreline with a radius-40 sac on the outer bend
    (BASELINE configs[2]; completion of the recipe: SURVEY.md §8(d)).

    Box 480x160x160. Centreline y_c(x) = 50 + 30 sin(pi (x-40)/400), z_c = 80 for
    x in [40, 440], sampled every 0.5 in x; vessel = union of radius-20 balls on the
    samples clipped to 40 <= x <= 439; sac = ball radius 40 at (240, 115, 80). Ghost
    slice x = 39 copies the fluid pattern of x = 40 as type 2 (inlet), x = 440 copies
    x = 439 as type 3 (outlet). ``scale`` multiplies every length (tests use < 1).
    """
    s = float(scale)
    nx, ny, nz = int(round(480 * s)), int(round(160 * s)), int(round(160 * s))
    xa, xb = int(round(40 * s)), int(round(440 * s))      # fluid x in [xa, xb-1]
    r_v, r_s = 20.0 * s, 40.0 * s
    st = np.zeros((nz, ny, nx), dtype=np.uint8)
    n_samp = 2 * (xb - xa) + 1
    for i in range(n_samp):
        x = xa + 0.5 * i
        yc = 50.0 * s + 30.0 * s * math.sin(math.pi * (x - xa) / (xb - xa))
        _paint_ball(st, (x, yc, 80.0 * s), r_v, FLUID, xclip=(xa, xb - 1))
    _paint_ball(st, (240.0 * s, 115.0 * s, 80.0 * s), r_s, FLUID)
    st[:, :, xa - 1][st[:, :, xa] == FLUID] = IOLET0
    st[:, :, xb][st[:, :, xb - 1] == FLUID] = IOLET0 + 1
    return Workload("aneurysm", st, 0, tau, np.array([rho_in, rho_out], dtype=np.float64),
                    steps, info={"scale": s})


# ----------------------------------------------------------------------- configs 3, 4
def _perp_basis(d):
    """(e1, e2) orthonormal and perpendicular to unit d; e2 is the direction
    perpendicular to d that is closest to +z (closest to +x if d is along z)."""
    ref = np.array([0.0, 0.0, 1.0])
    if abs(float(d @ ref)) > 0.999:
        ref = np.array([1.0, 0.0, 0.0])
    e2 = ref - (ref @ d) * d
    e2 /= np.linalg.norm(e2)
    e1 = np.cross(e2, d)
    return e1, e2


def _tree_segments(rng, p0, r0, levels, len_over_r, planar_deg):
    """Depth-first, plus-child-first list of segments and bifurcations."""
    segs, junctions, leaves = [], [], []

    def grow(p, d, g):
        r = r0 * 2.0 ** (-g / 3.0)
        L = len_over_r * r
        segs.append({"p": p, "d": d, "r": r, "L": L, "g": g})
        end = p + L * d
        if g == levels:
            leaves.append(len(segs) - 1)
            return
        th_p = math.radians(rng.uniform(25.0, 45.0))
        th_m = math.radians(rng.uniform(25.0, 45.0))
        uphi = rng.uniform(0.0, 1.0)
        if planar_deg is None:
            phi = 2.0 * math.pi * uphi
        else:  # bifurcation plane within +-planar_deg of the xy-plane
            phi = 0.5 * math.pi + math.radians((2.0 * uphi - 1.0) * planar_deg)
        e1, e2 = _perp_basis(d)
        n = math.cos(phi) * e1 + math.sin(phi) * e2
        t = np.cross(n, d)
        junctions.append({"c": end, "r": r, "n": n})
        grow(end, math.cos(th_p) * d + math.sin(th_p) * t, g + 1)
        grow(end, math.cos(th_m) * d - math.sin(th_m) * t, g + 1)

    grow(np.asarray(p0, dtype=np.float64), np.array([1.0, 0.0, 0.0]), 0)
    return segs, junctions, leaves


def tree(box=(1024, 1024, 1024), r0: float = 32.0, levels: int = 5, seed: int = 190611925,
         len_over_r: float = 8.0, n_sacs: int = 3, planar_deg: Optional[float] = None,
         tau: float = 0.55, rho_in: float = 1.0005, rho_out: float = 0.9995,
         steps: int = 500, scheme: str = "two_lattice", store: str = "f64",
         name: str = "tree", max_tries: int = 256) -> Workload:
    """Binary bifurcation tree of cylinders with spherical sacs (BASELINE configs[3],
    configs[4]; completion of the recipe: SURVEY.md §8(d) "Tree generator").

    Generations g = 0..levels, radius r_g = r0 2^(-g/3), length L_g = len_over_r r_g.
    The root starts at (2, ny/2, nz/2) heading +x with an inlet ghost slab (type 2) at
    x = 0..1. At every bifurcation theta+, theta- ~ U[25,45] deg and one azimuth draw
    fix the two children; a ball of the parent radius is painted at each junction.
    ``n_sacs`` distinct bifurcations get a ball of radius U[1.5,2.5] r_parent centred
    at junction + (R_s - r_parent/2) n. Leaf j gets a 2-voxel ghost slab of type 3+j.
    A seed whose tree leaves [2, n-3] (fluid) or clips a cap is rejected and the next
    seed is tried; the seed finally used is in ``info['seed']``.
    RNG: numpy default_rng(seed); draws: (theta+, theta-, azimuth) per bifurcation in
    depth-first plus-child-first order, then the sac sites (choice without
    replacement), then the sac radius factors.
    """
    nx, ny, nz = box
    n_leaves = 2 ** levels
    if n_leaves + 1 > 254:
        raise ValueError("too many iolets for a uint8 site type")
    for attempt in range(max_tries):
        s = seed + attempt
        rng = np.random.default_rng(s)
        segs, junctions, leaves = _tree_segments(
            rng, (2.0, ny / 2.0, nz / 2.0), r0, levels, len_over_r, planar_deg)
        n_s = min(n_sacs, len(junctions))
        sac_at = rng.choice(len(junctions), size=n_s, replace=False) if n_s else []
        sac_f = rng.uniform(1.5, 2.5, size=n_s)
        sacs = []
        for j, f in zip(sac_at, sac_f):
            J = junctions[int(j)]
            R = float(f) * J["r"]
            sacs.append((J["c"] + (R - 0.5 * J["r"]) * J["n"], R))
        # cheap rejection on bounding extents before painting anything
        ok = True
        lo_lim, hi_lim = np.array([2.0, 2.0, 2.0]), np.array([nx - 3.0, ny - 3.0, nz - 3.0])
        for sg in segs:
            for a in (0.0, sg["L"]):
                c = sg["p"] + a * sg["d"]
                ext = sg["r"] * np.sqrt(np.maximum(0.0, 1.0 - sg["d"] ** 2))
                if np.any(c - ext < lo_lim) or np.any(c + ext > hi_lim):
                    ok = False
        for J in junctions:
            if np.any(J["c"] - J["r"] < lo_lim) or np.any(J["c"] + J["r"] > hi_lim):
                ok = False
        for c, R in sacs:
            if np.any(c - R < lo_lim) or np.any(c + R > hi_lim):
                ok = False
        for li in leaves:
            sg = segs[li]
            c = sg["p"] + (sg["L"] + 2.0) * sg["d"]
            if np.any(c - sg["r"] < 0.0) or np.any(c + sg["r"] > np.array([nx, ny, nz]) - 1.0):
                ok = False
        if not ok:
            continue
        st = np.zeros((nz, ny, nx), dtype=np.uint8)
        for sg in segs:
            _paint_cylinder(st, sg["p"], sg["d"], sg["r"], 0.0, sg["L"], FLUID)
        for J in junctions:
            _paint_ball(st, J["c"], J["r"], FLUID)
        for c, R in sacs:
            _paint_ball(st, c, R, FLUID)
        # the extents test above is exact for cylinders/balls, so fluid is in [2, n-3]
        root = segs[0]
        _paint_cylinder(st, root["p"], root["d"], root["r"], -2.0, 0.0, IOLET0,
                        only_solid=True)
        for j, li in enumerate(leaves):
            sg = segs[li]
            _paint_cylinder(st, sg["p"], sg["d"], sg["r"], sg["L"], sg["L"] + 2.0,
                            IOLET0 + 1 + j, only_solid=True, lo_open=True)
        rho = np.full(1 + n_leaves, rho_out, dtype=np.float64)
        rho[0] = rho_in
        return Workload(name, st, 0, tau, rho, steps, scheme=scheme, store=store,
                        info={"seed": s, "seed_requested": seed, "r0": r0, "levels": levels,
                              "len_over_r": len_over_r, "n_sacs": n_s,
                              "planar_deg": planar_deg})
    raise RuntimeError(f"no seed in [{seed}, {seed + max_tries}) fits the box {box}")


# --------------------------------------------------------------------------- tests
def random_mask(shape=(8, 7, 6), p_fluid: float = 0.6, n_iolets: int = 2, p_iolet: float = 0.05,
                periodic: int = 0, tau: float = 0.7, seed: int = 0, steps: int = 8) -> Workload:
    """Random small mask (nx, ny, nz) with random walls and iolet ghost voxels; used for
    brute-force equivalence tests. Iolet densities are drawn in [0.98, 1.02]."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = shape
    r = rng.random((nz, ny, nx))
    st = np.where(r < p_fluid, FLUID, SOLID).astype(np.uint8)
    if n_iolets:
        io = rng.random((nz, ny, nx)) < p_iolet
        st[io] = (IOLET0 + rng.integers(0, n_iolets, size=(nz, ny, nx)))[io].astype(np.uint8)
    if not np.any(st == FLUID):
        st[0, 0, 0] = FLUID
    n = int(np.count_nonzero(st == FLUID))
    rho0 = 1.0 + 0.02 * (rng.random(n) - 0.5)
    u0 = 0.04 * (rng.random((n, 3)) - 0.5)
    return Workload("random", st, periodic, tau,
                    rng.uniform(0.98, 1.02, size=n_iolets).astype(np.float64), steps,
                    rho0=rho0, u0=u0, info={"seed": seed})


def with_velocity_inlet(wl: Workload, u_in: float = 0.004) -> Workload:
    """The same geometry with iolet 0 turned into a Ladd velocity inlet (the paper's
    "LADDIOLET" configuration) blowing u_in along +x for the vessel
    geometries (their inlet caps face -x) and along +z for the pipe; the other iolets stay
    constant-density outlets."""
    kind = np.zeros(wl.n_iolets, dtype=np.uint8)
    u = np.zeros((wl.n_iolets, 3), dtype=np.float64)
    kind[0] = 1
    u[0, 2 if wl.name == "pipe" else 0] = u_in
    return dataclasses.replace(wl, iolet_kind=kind, iolet_u=u, name=wl.name)


def with_inlet_profile(wl: Workload) -> Workload:
    """Per-site velocity weights for iolet 0 (the paper's USE_VELOCITY_WEIGHTS_FILE build flag,
    PAPER.md line 59; the file itself is not in the paper): a parabolic profile across the inlet
    cap, omega proportional to 1 - r^2 / R^2 and scaled to mean 1 over the cap (so the mean inlet
    velocity stays u_k), r measured from the centroid of the fluid sites that touch a ghost
    voxel of iolet 0 and R = their largest distance + 1/2. Sites
    that do not touch the inlet keep weight 1 (they have no velocity link to weigh)."""
    st = wl.site_type
    nz, ny, nx = st.shape
    v = wl.fluid_voxels()
    x, y, z = v % nx, (v // nx) % ny, v // (nx * ny)
    touch = np.zeros(len(v), dtype=bool)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                xs, ys, zs = x + dx, y + dy, z + dz
                ok = (xs >= 0) & (xs < nx) & (ys >= 0) & (ys < ny) & (zs >= 0) & (zs < nz)
                hit = np.zeros(len(v), dtype=bool)
                hit[ok] = st[zs[ok], ys[ok], xs[ok]] == IOLET0
                touch |= hit
    w = np.ones(len(v), dtype=np.float64)
    if touch.any():
        p = np.stack([x[touch], y[touch], z[touch]], axis=1).astype(np.float64)
        c = p.mean(axis=0)
        r = np.linalg.norm(p - c, axis=1)
        R = r.max() + 0.5
        prof = 1.0 - (r / R) ** 2
        w[touch] = prof / prof.mean()
    return dataclasses.replace(wl, iolet_weight=w)


def pulsatile_waveform(wl: Workload, n_t: int, u_peak: float = 0.006, u_base: float = 0.002,
                       seed: int = 8) -> np.ndarray:
    """A periodic inlet-velocity waveform u[n_t][n_iolets][3] standing in for the paper's inlet
    velocity file (Table I, line 126 Fig. 8 -- the data are not in the paper):
    a cardiac-cycle-like pulse, baseline u_base plus a systolic bump to u_peak over the first
    third of the period and a small seeded dicrotic ripple, along the direction of
    ``wl.iolet_u[0]`` (see with_velocity_inlet) for iolet 0; all other rows are 0 (constant-
    density outlets ignore them). One period = n_t time steps."""
    if wl.iolet_u is None:
        raise ValueError("apply with_velocity_inlet first")
    rng = np.random.default_rng(seed)
    phase = np.arange(n_t, dtype=np.float64) / float(n_t)
    bump = np.where(phase < 1.0 / 3.0, np.sin(3.0 * np.pi * phase) ** 2, 0.0)
    ripple = 0.08 * float(rng.uniform(0.5, 1.0)) * np.sin(2.0 * np.pi * 3.0 * phase + float(rng.uniform(0, 6.28)))
    speed = u_base + (u_peak - u_base) * bump + (u_peak - u_base) * ripple * (phase >= 1.0 / 3.0)
    direction = wl.iolet_u[0] / np.linalg.norm(wl.iolet_u[0])
    u = np.zeros((n_t, wl.n_iolets, 3), dtype=np.float64)
    u[:, 0, :] = speed[:, None] * direction[None, :]
    return u


def wall_distance_by_bisection(wl: Workload, inside_fn, iters: int = 48) -> np.ndarray:
    """Sub-voxel wall distances for interpolated (BFL) walls from the analytic surface the
    voxel mask was painted from: for every fluid voxel and each of the 26 lattice vectors whose
    neighbouring voxel is solid, the fraction d of the link at which ``inside_fn(X, Y, Z)``
    (vectorised, float coordinates -> bool) turns false, found by bisection; entry
    (dz+1)*9 + (dy+1)*3 + (dx+1) of row i (canonical order), 0 where the neighbour is not solid.
    A surface that the link does not cross (staircase corners) gets d = 1/2."""
    st = wl.site_type
    nz, ny, nx = st.shape
    v = wl.fluid_voxels()
    x, y, z = v % nx, (v // nx) % ny, v // (nx * ny)
    out = np.zeros((len(v), 27), dtype=np.float64)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                if dx == dy == dz == 0:
                    continue
                xs, ys, zs = x + dx, y + dy, z + dz
                ok = (xs >= 0) & (xs < nx) & (ys >= 0) & (ys < ny) & (zs >= 0) & (zs < nz)
                solid = np.zeros(len(v), dtype=bool)
                solid[ok] = st[zs[ok], ys[ok], xs[ok]] == SOLID
                sel = np.flatnonzero(solid)
                if sel.size == 0:
                    continue
                px, py, pz = x[sel].astype(float), y[sel].astype(float), z[sel].astype(float)
                lo, hi = np.zeros(sel.size), np.ones(sel.size)
                crosses = inside_fn(px, py, pz) & ~inside_fn(px + dx, py + dy, pz + dz)
                for _ in range(iters):
                    mid = 0.5 * (lo + hi)
                    ins = inside_fn(px + mid * dx, py + mid * dy, pz + mid * dz)
                    lo = np.where(ins, mid, lo)
                    hi = np.where(ins, hi, mid)
                d = np.where(crosses, np.clip(0.5 * (lo + hi), 1e-6, 1.0), 0.5)
                out[sel, (dz + 1) * 9 + (dy + 1) * 3 + (dx + 1)] = d
    return out


def with_bfl_walls(wl: Workload) -> Workload:
    """The pipe or the aneurysm with sub-voxel wall distances from their analytic surfaces."""
    if wl.name == "pipe":
        R = float(wl.info["radius"])

        def inside(X, Y, Z):
            return (X - R) ** 2 + (Y - R) ** 2 <= R * R
    elif wl.name == "aneurysm":
        s = float(wl.info["scale"])
        xa, xb = int(round(40 * s)), int(round(440 * s))
        xs = xa + 0.5 * np.arange(2 * (xb - xa) + 1)
        yc = 50.0 * s + 30.0 * s * np.sin(np.pi * (xs - xa) / (xb - xa))

        def inside(X, Y, Z):
            X, Y, Z = (np.asarray(a, dtype=np.float64) for a in (X, Y, Z))
            d2 = (X[:, None] - xs[None, :]) ** 2 + (Y[:, None] - yc[None, :]) ** 2 + \
                (Z[:, None] - 80.0 * s) ** 2
            tube = (d2.min(axis=1) <= (20.0 * s) ** 2) & (X >= xa) & (X <= xb - 1)
            sac = (X - 240.0 * s) ** 2 + (Y - 115.0 * s) ** 2 + (Z - 80.0 * s) ** 2 <= (40.0 * s) ** 2
            return tube | sac
    else:
        raise KeyError(f"no analytic surface recorded for {wl.name}")
    return dataclasses.replace(wl, wall_distance=wall_distance_by_bisection(wl, inside))


def by_name(name: str, small: bool = False) -> Workload:
    """The five BASELINE.json configs (``small=True``: the scaled-down parity cases)."""
    if name == "pipe":
        return pipe(radius=4, length=16, steps=50) if small else pipe()
    if name == "cube":
        return periodic_cube(n=32, steps=100) if small else periodic_cube()
    if name == "aneurysm":
        return aneurysm(scale=0.2, steps=100) if small else aneurysm()
    if name == "paper_sized":
        # not a BASELINE config: the aneurysm recipe scaled to the site count of the paper's
        # larger subject (296,814 sites, Table II) -- context for its Table III
        return aneurysm(scale=0.2 if small else 0.7375, steps=100 if small else 2000)
    if name == "paper_sized_23":
        # not a BASELINE config: the same recipe at the site count of the paper's smaller subject
        # (132,910 sites, Table II)
        return aneurysm(scale=0.2 if small else 0.5645, steps=100 if small else 2000)
    if name == "tree":
        if small:
            return tree(box=(160, 160, 160), r0=5.0, levels=3, steps=60)
        return tree()
    if name == "cube672":
        # not a BASELINE config: the smallest periodic cube whose Q * N exceeds 2^32 (303.5 M
        # sites), so that the 64-bit flat-offset kernels are the ones that run (include/hlb.h
        # HLB_INDEX64); A-A in place, rest state unless the caller sets one
        w = periodic_cube(n=40 if small else 672, steps=25, with_state=False)
        return dataclasses.replace(w, name="cube672", scheme="aa")
    if name == "bigtree_x":
        # not a BASELINE config: configs[4] at BASELINE's nominal 80-100 M sites. Its generator
        # cannot get there inside the 2048 x 2048 x 1024 box (SURVEY.md section 8(d) caveat: with
        # r0, the radius law and the angles fixed, L / r = 8 is what fits -- the root-to-leaf
        # path is 1862 voxels -- and three sacs on the largest bifurcations would add 34 M at
        # most), so the third knob is turned: the voxel size. Box and r0 scaled by 1.3
        # (77 um voxels instead of 100 um), same seed search, everything else as configs[4].
        if small:
            return tree(box=(248, 248, 124), r0=6.5, levels=3, planar_deg=30.0, tau=0.52,
                        steps=60, scheme="aa", name="bigtree_x")
        return tree(box=(2662, 2662, 1331), r0=83.2, planar_deg=30.0, tau=0.52, steps=200,
                    scheme="aa", name="bigtree_x")
    if name == "bigtree":
        if small:
            return tree(box=(192, 192, 96), r0=5.0, levels=3, planar_deg=30.0, tau=0.52,
                        steps=60, scheme="aa", name="bigtree")
        return tree(box=(2048, 2048, 1024), r0=64.0, planar_deg=30.0, tau=0.52, steps=200,
                    scheme="aa", name="bigtree")
    raise KeyError(name)
