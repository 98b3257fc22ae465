"""ctypes wrapper around the C++ oracle (hlb_oracle.cpp, hlb_oracle_dense.cpp).

TEST INFRASTRUCTURE ONLY -- see the package docstring. Argument marshalling and the g++
build; no arithmetic of the method lives here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_SOURCES = [os.path.join(_HERE, "hlb_oracle.cpp"), os.path.join(_HERE, "hlb_oracle_dense.cpp"),
            os.path.join(_HERE, "render_oracle.cpp")]
_lock = threading.Lock()
_lib = None

VARIANT_SHIFTED, VARIANT_RAW, VARIANT_SHIFTED_LD, VARIANT_RAW_LD = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (no -ffast-math, no -march: plain IEEE double,
    no FMA contraction) into oracle/liboracle.so."""
    newest = max(os.path.getmtime(s) for s in _SOURCES)
    if not force and os.path.exists(_LIB_PATH) and os.path.getmtime(_LIB_PATH) >= newest:
        return _LIB_PATH
    tmp = _LIB_PATH + f".tmp{os.getpid()}"
    cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-Wall", "-Wextra", "-o", tmp] + _SOURCES
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


def _load():
    global _lib
    with _lock:
        if _lib is not None:
            return _lib
        build()
        lib = ctypes.CDLL(_LIB_PATH)
        c_dp = ctypes.POINTER(ctypes.c_double)
        lib.hlbo_create.restype = ctypes.c_void_p
        lib.hlbo_create.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                    ctypes.c_uint, ctypes.c_double, ctypes.c_int, ctypes.c_void_p,
                                    ctypes.c_int]
        lib.hlbo_create_lattice.restype = ctypes.c_void_p
        lib.hlbo_create_lattice.argtypes = lib.hlbo_create.argtypes + [ctypes.c_int]
        lib.hlbo_velocity_set_lattice.restype = ctypes.c_int
        lib.hlbo_velocity_set_lattice.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                                  ctypes.c_void_p]
        lib.hlbo_num_q.restype = ctypes.c_int
        lib.hlbo_num_q.argtypes = [ctypes.c_void_p]
        lib.hlbo_destroy.argtypes = [ctypes.c_void_p]
        lib.hlbo_destroy.restype = None
        for name in ("hlbo_num_sites", "hlbo_steps_done"):
            getattr(lib, name).restype = ctypes.c_int64
            getattr(lib, name).argtypes = [ctypes.c_void_p]
        lib.hlbo_site_voxels.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_set_state.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_set_populations.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_get_populations.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_step.argtypes = [ctypes.c_void_p, ctypes.c_int64]
        lib.hlbo_get_macroscopic.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_velocity_set.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_set_threads.argtypes = [ctypes.c_int]
        lib.hlbo_get_threads.restype = ctypes.c_int
        lib.hlbd_run.restype = ctypes.c_int
        lib.hlbd_run.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                 ctypes.c_uint, ctypes.c_double, ctypes.c_int, ctypes.c_void_p,
                                 ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                                 ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_set_wall_distance.restype = None
        lib.hlbo_set_wall_distance.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_get_wall_shear_stress.restype = None
        lib.hlbo_get_wall_shear_stress.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_get_stress.restype = None
        lib.hlbo_get_stress.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_set_iolet_velocity.restype = None
        lib.hlbo_set_iolet_velocity.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbd_run_ladd.restype = ctypes.c_int
        lib.hlbd_run_ladd.argtypes = lib.hlbd_run.argtypes[:8] + [ctypes.c_void_p, ctypes.c_void_p] + \
            lib.hlbd_run.argtypes[8:] + [ctypes.c_int]
        lib.rendo_sample.restype = ctypes.c_float
        lib.rendo_sample.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_float, ctypes.c_float, ctypes.c_float]
        lib.rendo_render.restype = ctypes.c_int64
        lib.rendo_render.argtypes = [ctypes.c_void_p] + [ctypes.c_int] * 5 + [ctypes.c_void_p] + \
            [ctypes.c_float] * 5 + [ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbo_set_iolet_normal.restype = None
        lib.hlbo_set_iolet_normal.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbd_run_all.restype = ctypes.c_int
        lib.hlbd_run_all.argtypes = lib.hlbd_run.argtypes[:8] + [ctypes.c_void_p] * 4 + \
            lib.hlbd_run.argtypes[8:] + [ctypes.c_int]
        lib.hlbo_set_iolet_weight.restype = None
        lib.hlbo_set_iolet_weight.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.hlbd_run_weights.restype = ctypes.c_int
        lib.hlbd_run_weights.argtypes = lib.hlbd_run.argtypes[:8] + [ctypes.c_void_p] * 5 + \
            lib.hlbd_run.argtypes[8:] + [ctypes.c_int]
        lib.hlbd_run_bfl.restype = ctypes.c_int
        lib.hlbd_run_bfl.argtypes = lib.hlbd_run.argtypes[:8] + [ctypes.c_void_p] * 3 + \
            lib.hlbd_run.argtypes[8:] + [ctypes.c_int]
        lib.hlbd_run_lattice.restype = ctypes.c_int
        lib.hlbd_run_lattice.argtypes = lib.hlbd_run.argtypes + [ctypes.c_int]
        for name in ("hlbo_site_voxels", "hlbo_set_state", "hlbo_set_populations",
                     "hlbo_get_populations", "hlbo_step", "hlbo_get_macroscopic",
                     "hlbo_velocity_set", "hlbo_set_threads"):
            getattr(lib, name).restype = None
        del c_dp
        _lib = lib
        return lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


LATTICE_Q = {"d3q15": 15, "d3q19": 19}


def velocity_set(lattice="d3q15"):
    """(c[Q,3] int32, w[Q] float64, opp[Q] int32) in the oracle's own q order."""
    lib = _load()
    nq = LATTICE_Q[lattice]
    c = np.zeros((nq, 3), dtype=np.int32)
    w = np.zeros(nq, dtype=np.float64)
    opp = np.zeros(nq, dtype=np.int32)
    assert lib.hlbo_velocity_set_lattice(nq, _ptr(c), _ptr(w), _ptr(opp)) == nq
    return c, w, opp


class Oracle:
    """One oracle simulation. Per-site arrays are in canonical order (ascending voxel)."""

    def __init__(self, site_type, periodic=0, tau=1.0, iolet_rho=(), variant=VARIANT_SHIFTED,
                 threads=1, lattice="d3q15"):
        lib = _load()
        st = np.ascontiguousarray(site_type, dtype=np.uint8)
        assert st.ndim == 3
        nz, ny, nx = st.shape
        io = np.ascontiguousarray(np.asarray(iolet_rho, dtype=np.float64))
        lib.hlbo_set_threads(int(threads))
        self._lib = lib
        self.n_q = LATTICE_Q[lattice]
        self._h = lib.hlbo_create_lattice(_ptr(st), nx, ny, nz, int(periodic), float(tau),
                                          int(io.shape[0]), _ptr(io), int(variant), self.n_q)
        if not self._h:
            raise ValueError("hlbo_create rejected its arguments")
        self.n_sites = int(lib.hlbo_num_sites(self._h))
        self.n_iolets = int(io.shape[0])
        self.threads = int(lib.hlbo_get_threads())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.hlbo_destroy(self._h)
            self._h = None

    __del__ = close

    def site_voxels(self):
        v = np.zeros(self.n_sites, dtype=np.int64)
        self._lib.hlbo_site_voxels(self._h, _ptr(v))
        return v

    def set_state(self, rho=None, u=None):
        rho = None if rho is None else np.ascontiguousarray(rho, dtype=np.float64)
        u = None if u is None else np.ascontiguousarray(u, dtype=np.float64)
        if rho is not None:
            assert rho.shape == (self.n_sites,)
        if u is not None:
            assert u.shape == (self.n_sites, 3)
        self._lib.hlbo_set_state(self._h, _ptr(rho), _ptr(u))

    def set_iolet_velocity(self, kind, u):
        """kind [n_iolets]: 0 constant density, 1 Ladd velocity; u [n_iolets, 3]. Takes effect
        from the next step."""
        kind = np.ascontiguousarray(np.asarray(kind, dtype=np.uint8).reshape(-1))
        u = np.ascontiguousarray(np.asarray(u, dtype=np.float64).reshape(-1, 3))
        assert kind.shape == (self.n_iolets,) and u.shape == (self.n_iolets, 3)
        self._lib.hlbo_set_iolet_velocity(self._h, _ptr(kind), _ptr(u))

    def set_iolet_weight(self, weight):
        """weight [N] (canonical order): factor of u_k on the velocity-iolet links of each site
        (a velocity profile across the inlet cap); None removes it."""
        if weight is None:
            self._lib.hlbo_set_iolet_weight(self._h, None)
            return
        w = np.ascontiguousarray(np.asarray(weight, dtype=np.float64).reshape(-1))
        assert w.shape == (self.n_sites,)
        self._lib.hlbo_set_iolet_weight(self._h, _ptr(w))

    def set_iolet_normal(self, normals):
        """Normals [n_iolets, 3] of the constant-density iolets (any length; zero vector or
        None: no projection)."""
        if normals is not None:
            normals = np.ascontiguousarray(np.asarray(normals, dtype=np.float64).reshape(-1, 3))
            assert normals.shape == (self.n_iolets, 3)
        self._lib.hlbo_set_iolet_normal(self._h, _ptr(normals))

    def set_populations(self, f):
        f = np.ascontiguousarray(f, dtype=np.float64)
        assert f.shape == (self.n_sites, self.n_q)
        self._lib.hlbo_set_populations(self._h, _ptr(f))

    def get_populations(self):
        f = np.zeros((self.n_sites, self.n_q), dtype=np.float64)
        self._lib.hlbo_get_populations(self._h, _ptr(f))
        return f

    def step(self, n=1):
        self._lib.hlbo_set_threads(self.threads)
        self._lib.hlbo_step(self._h, int(n))

    def steps_done(self):
        return int(self._lib.hlbo_steps_done(self._h))

    def set_wall_distance(self, d27):
        """BFL wall distances [N, 27] (canonical order; entry (dz+1)*9+(dy+1)*3+(dx+1) = fraction
        of the link along (dx,dy,dz) at which the wall sits, <= 0: none) or None (off)."""
        if d27 is not None:
            d27 = np.ascontiguousarray(d27, dtype=np.float64)
            assert d27.shape == (self.n_sites, 27)
        self._lib.hlbo_set_wall_distance(self._h, _ptr(d27))

    def get_stress(self):
        """Deviatoric stress [N, 6] (xx, yy, zz, xy, xz, yz) of the pre-collision state."""
        sg = np.zeros((self.n_sites, 6), dtype=np.float64)
        self._lib.hlbo_get_stress(self._h, _ptr(sg))
        return sg

    def get_wall_shear_stress(self, normals):
        """|tangential part of sigma n| per site for wall normals [N, 3] (zero vector -> 0)."""
        nrm = np.ascontiguousarray(normals, dtype=np.float64)
        assert nrm.shape == (self.n_sites, 3)
        out = np.zeros(self.n_sites, dtype=np.float64)
        self._lib.hlbo_get_wall_shear_stress(self._h, _ptr(nrm), _ptr(out))
        return out

    def get_macroscopic(self):
        rho = np.zeros(self.n_sites, dtype=np.float64)
        u = np.zeros((self.n_sites, 3), dtype=np.float64)
        self._lib.hlbo_get_macroscopic(self._h, _ptr(rho), _ptr(u))
        return rho, u


def run(workload, steps=None, variant=VARIANT_SHIFTED, threads=1, lattice="d3q15"):
    """Run a workloads.Workload for ``steps`` (default: its own count); returns rho, u."""
    o = Oracle(workload.site_type, workload.periodic, workload.tau, workload.iolet_rho,
               variant=variant, threads=threads, lattice=lattice)
    if workload.rho0 is not None or workload.u0 is not None:
        o.set_state(workload.rho0, workload.u0)
    if getattr(workload, "iolet_kind", None) is not None:
        o.set_iolet_velocity(workload.iolet_kind, workload.iolet_u)
    if getattr(workload, "iolet_normal", None) is not None:
        o.set_iolet_normal(workload.iolet_normal)
    if getattr(workload, "iolet_weight", None) is not None:
        o.set_iolet_weight(workload.iolet_weight)
    if getattr(workload, "wall_distance", None) is not None:
        o.set_wall_distance(workload.wall_distance)
    o.step(workload.steps if steps is None else steps)
    out = o.get_macroscopic()
    o.close()
    return out


def dense_run(site_type, periodic, tau, iolet_rho, steps, rho0_vox=None, u0_vox=None,
              lattice="d3q15", iolet_kind=None, iolet_u=None, wall_d27_vox=None, iolet_normal=None,
              site_weight_vox=None):
    """Dense-grid twin: per-VOXEL rho [nz,ny,nx] and u [nz,ny,nx,3]."""
    lib = _load()
    st = np.ascontiguousarray(site_type, dtype=np.uint8)
    nz, ny, nx = st.shape
    io = np.ascontiguousarray(np.asarray(iolet_rho, dtype=np.float64))
    r0 = None if rho0_vox is None else np.ascontiguousarray(rho0_vox, dtype=np.float64)
    u0 = None if u0_vox is None else np.ascontiguousarray(u0_vox, dtype=np.float64)
    rho = np.zeros((nz, ny, nx), dtype=np.float64)
    u = np.zeros((nz, ny, nx, 3), dtype=np.float64)
    kind = None if iolet_kind is None else \
        np.ascontiguousarray(np.asarray(iolet_kind, dtype=np.uint8).reshape(-1))
    uio = None if iolet_u is None else \
        np.ascontiguousarray(np.asarray(iolet_u, dtype=np.float64).reshape(-1, 3))
    wd = None if wall_d27_vox is None else np.ascontiguousarray(wall_d27_vox, dtype=np.float64)
    if wd is not None:
        assert wd.shape == (nz * ny * nx, 27)
    nio = None if iolet_normal is None else \
        np.ascontiguousarray(np.asarray(iolet_normal, dtype=np.float64).reshape(-1, 3))
    sw = None if site_weight_vox is None else \
        np.ascontiguousarray(np.asarray(site_weight_vox, dtype=np.float64).reshape(-1))
    if sw is not None:
        assert sw.shape == (nz * ny * nx,)
    rc = lib.hlbd_run_weights(_ptr(st), nx, ny, nz, int(periodic), float(tau), int(io.shape[0]),
                              _ptr(io), _ptr(kind), _ptr(uio), _ptr(wd), _ptr(nio), _ptr(sw), _ptr(r0),
                              _ptr(u0), int(steps), _ptr(rho), _ptr(u), LATTICE_Q[lattice])
    if rc != 0:
        raise ValueError("hlbd_run rejected its arguments")
    return rho, u


# ----------------------------------------------------------------------------- renderer oracle
def render_sample(volume, p):
    """One trilinear sample of a float32 volume [nz, ny, nx] at p = (x, y, z)."""
    lib = _load()
    vol = np.ascontiguousarray(volume, dtype=np.float32)
    nz, ny, nx = vol.shape
    return float(lib.rendo_sample(_ptr(vol), nx, ny, nz, float(p[0]), float(p[1]), float(p[2])))


def render(volume, width, height, rot, zoom, step, tf_scale, tf_offset, opacity, lut):
    """Ray-marched image [height, width, 4] float32 of a float32 volume [nz, ny, nx] (see
    render_oracle.cpp for the definition). Returns (image, samples_inside_the_box)."""
    lib = _load()
    vol = np.ascontiguousarray(volume, dtype=np.float32)
    nz, ny, nx = vol.shape
    r = np.ascontiguousarray(np.asarray(rot, dtype=np.float32).reshape(9))
    l = np.ascontiguousarray(np.asarray(lut, dtype=np.float32).reshape(256, 4))
    img = np.zeros((height, width, 4), dtype=np.float32)
    n = lib.rendo_render(_ptr(vol), nx, ny, nz, int(width), int(height), _ptr(r), float(zoom),
                         float(step), float(tf_scale), float(tf_offset), float(opacity), _ptr(l),
                         _ptr(img))
    if n < 0:
        raise ValueError("rendo_render rejected its arguments")
    return img, int(n)
