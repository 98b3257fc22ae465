"""Thin Python binding of include/hlb.h: argument marshalling only.

Same names as the C-ABI entry points. PyTorch supplies device memory (the allocator
callback hands out ``torch.empty`` buffers that live as long as the Geometry object) and
the CUDA stream; every step of the path runs in the kernels of libhlb.so. There is no CPU
fallback: if libhlb.so cannot be built or loaded, importing this module raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

from . import build as _build

HLB_OK, HLB_EINVAL, HLB_ENOFLUID, HLB_ETOOLARGE, HLB_ENOMEM, HLB_ECUDA = 0, -1, -2, -3, -4, -5
HLB_STORE_F64, HLB_STORE_F32 = 0x0, 0x1
HLB_TWO_LATTICE, HLB_AA = 0x0, 0x2
HLB_ORDER_AUTO, HLB_ORDER_MORTON, HLB_ORDER_RASTER, HLB_ORDER_TILED = 0x0, 0x4, 0x8, 0xC
HLB_NO_GRAPH = 0x10
HLB_LINKS_AUTO, HLB_LINKS_TABLE, HLB_LINKS_RECORDS = 0x0, 0x20, 0x40
HLB_NO_PREFETCH = 0x80
HLB_INDEX64 = 0x100
HLB_NO_PDL = 0x400
HLB_NO_RESIDENT = 0x800
HLB_SCHEME_AUTO = 0x1000
HLB_LATTICE_D3Q15, HLB_LATTICE_D3Q19 = 0x0, 0x200

_ALLOC_FN = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)
_FREE_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)


class hlb_params(ctypes.Structure):
    _fields_ = [
        ("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
        ("periodic", ctypes.c_uint32),
        ("tau", ctypes.c_double),
        ("n_iolets", ctypes.c_int32),
        ("iolet_rho", ctypes.c_void_p),
        ("flags", ctypes.c_uint32),
        ("alloc", _ALLOC_FN),
        ("alloc_user", ctypes.c_void_p),
        ("stream", ctypes.c_void_p),
        ("free", _FREE_FN),
        ("copy_stream", ctypes.c_void_p),
    ]


class hlb_view(ctypes.Structure):
    _fields_ = [
        ("width", ctypes.c_int32), ("height", ctypes.c_int32),
        ("rot", ctypes.c_float * 9),
        ("zoom", ctypes.c_float), ("step", ctypes.c_float),
        ("tf_scale", ctypes.c_float), ("tf_offset", ctypes.c_float),
        ("opacity", ctypes.c_float),
        ("field", ctypes.c_int32),
    ]


def make_view(width, height, rot=None, zoom=1.0, step=1.0, tf_scale=1.0, tf_offset=0.0, opacity=1.0,
              field=0) -> "hlb_view":
    v = hlb_view()
    v.width, v.height = int(width), int(height)
    r = np.eye(3, dtype=np.float32) if rot is None else np.asarray(rot, dtype=np.float32).reshape(3, 3)
    v.rot = (ctypes.c_float * 9)(*[float(x) for x in r.reshape(-1)])
    v.zoom, v.step = float(zoom), float(step)
    v.tf_scale, v.tf_offset, v.opacity, v.field = float(tf_scale), float(tf_offset), float(opacity), int(field)
    return v


class HlbError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"hlb error {code}: {msg}")
        self.code = code


def _load() -> ctypes.CDLL:
    path = _build.build()
    lib = ctypes.CDLL(path)
    vp, i64, c_int = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
    sigs = {
        "hlb_geometry_create": (c_int, [vp, ctypes.POINTER(hlb_params), ctypes.POINTER(vp)]),
        "hlb_set_state": (c_int, [vp, vp, vp]),
        "hlb_set_iolet_density": (c_int, [vp, vp]),
        "hlb_set_iolet_velocity": (c_int, [vp, vp, vp]),
        "hlb_set_iolet_waveform": (c_int, [vp, vp, i64]),
        "hlb_set_iolet_weight": (c_int, [vp, vp]),
        "hlb_set_iolet_normal": (c_int, [vp, vp]),
        "hlb_set_wall_distance": (c_int, [vp, vp]),
        "hlb_num_bfl_sites": (i64, [vp]),
        "hlb_step": (c_int, [vp, i64]),
        "hlb_get_macroscopic": (c_int, [vp, vp, vp]),
        "hlb_get_macroscopic_device": (c_int, [vp, vp, vp]),
        "hlb_get_macroscopic_async": (c_int, [vp, vp, vp]),
        "hlb_wait_copies": (c_int, [vp]),
        "hlb_stage_state": (c_int, [vp, vp, vp]),
        "hlb_set_state_staged": (c_int, [vp]),
        "hlb_get_populations": (c_int, [vp, vp]),
        "hlb_get_stress": (c_int, [vp, vp]),
        "hlb_get_stress_device": (c_int, [vp, vp]),
        "hlb_get_wall_shear_stress": (c_int, [vp, vp, vp]),
        "hlb_get_wall_shear_stress_noalloc": (c_int, [vp, vp, vp]),
        "hlb_noalloc_max_sites": (i64, []),
        "hlb_render_volume": (c_int, [vp, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                      ctypes.POINTER(hlb_view), vp, vp, vp]),
        "hlb_render": (c_int, [vp, ctypes.POINTER(hlb_view), vp, vp]),
        "hlb_render_device": (c_int, [vp, ctypes.POINTER(hlb_view), vp, vp]),
        "hlb_set_populations": (c_int, [vp, vp]),
        "hlb_num_sites": (i64, [vp]),
        "hlb_num_q": (c_int, [vp]),
        "hlb_lattice": (c_int, [ctypes.c_uint32, vp, vp, vp]),
        "hlb_steps_done": (i64, [vp]),
        "hlb_get_site_voxels": (c_int, [vp, vp]),
        "hlb_device_bytes": (i64, [vp]),
        "hlb_launch_count": (i64, [vp]),
        "hlb_uses_records": (c_int, [vp]),
        "hlb_uses_aa": (c_int, [vp]),
        "hlb_offset_bits": (c_int, [vp]),
        "hlb_record_sentinel_fraction": (ctypes.c_double, [vp]),
        "hlb_preprocess_records": (c_int, [vp, ctypes.c_int32, i64, vp, ctypes.POINTER(i64)]),
        "hlb_preprocess_bfl": (c_int, [vp, vp, ctypes.c_int32, i64, i64, vp, vp, vp, i64,
                                      ctypes.POINTER(i64), ctypes.POINTER(i64)]),
        "hlb_geometry_destroy": (None, [vp]),
        "hlb_last_error": (ctypes.c_char_p, []),
        "hlb_velocity_set": (None, [vp, vp, vp]),
        "hlb_preprocess_count": (c_int, [vp, ctypes.POINTER(hlb_params), ctypes.POINTER(i64),
                                         ctypes.POINTER(i64)]),
        "hlb_preprocess_tables": (c_int, [vp, ctypes.POINTER(hlb_params), vp, vp, vp]),
    }
    for name, (res, args) in sigs.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    return lib


LIB_PATH = _build.LIB_PATH
_lib = _load()
EXPORTED = ("hlb_geometry_create", "hlb_set_state", "hlb_set_iolet_density",
            "hlb_set_iolet_velocity", "hlb_set_iolet_waveform", "hlb_set_iolet_weight", "hlb_set_iolet_normal", "hlb_set_wall_distance", "hlb_num_bfl_sites", "hlb_step",
            "hlb_get_macroscopic", "hlb_get_macroscopic_device", "hlb_get_macroscopic_async", "hlb_wait_copies", "hlb_stage_state", "hlb_set_state_staged",
            "hlb_get_populations",
            "hlb_get_stress", "hlb_get_stress_device", "hlb_get_wall_shear_stress", "hlb_get_wall_shear_stress_noalloc", "hlb_noalloc_max_sites", "hlb_render_volume", "hlb_render",
            "hlb_render_device",
            "hlb_set_populations", "hlb_num_sites", "hlb_num_q", "hlb_lattice", "hlb_steps_done", "hlb_get_site_voxels",
            "hlb_device_bytes", "hlb_launch_count", "hlb_uses_records", "hlb_uses_aa", "hlb_offset_bits",
            "hlb_record_sentinel_fraction", "hlb_geometry_destroy", "hlb_last_error",
            "hlb_velocity_set", "hlb_preprocess_count", "hlb_preprocess_tables",
            "hlb_preprocess_records", "hlb_preprocess_bfl")


def hlb_last_error() -> str:
    return _lib.hlb_last_error().decode()


def _check(rc: int):
    if rc != HLB_OK:
        raise HlbError(rc, hlb_last_error())


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _host(a, dtype, shape=None):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=dtype)
    if shape is not None and a.shape != shape:
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def hlb_velocity_set():
    c = np.zeros((15, 3), dtype=np.int32)
    w = np.zeros(15, dtype=np.float64)
    opp = np.zeros(15, dtype=np.int32)
    _lib.hlb_velocity_set(_ptr(c), _ptr(w), _ptr(opp))
    return c, w, opp


def hlb_render_volume(volume, view: "hlb_view", lut):
    """Ray-march a host float32 volume [nz, ny, nx]; returns the image [height, width, 4]."""
    import torch
    if not torch.cuda.is_available():
        raise HlbError(HLB_ECUDA, "no CUDA device: the renderer has no CPU fallback")
    vol = np.ascontiguousarray(volume, dtype=np.float32)
    nz, ny, nx = vol.shape
    lut = np.ascontiguousarray(np.asarray(lut, dtype=np.float32).reshape(256, 4))
    img = np.empty((view.height, view.width, 4), dtype=np.float32)
    stream = torch.cuda.current_stream().cuda_stream
    _check(_lib.hlb_render_volume(_ptr(vol), nx, ny, nz, ctypes.byref(view), _ptr(lut), _ptr(img), stream))
    return img


def hlb_noalloc_max_sites() -> int:
    return int(_lib.hlb_noalloc_max_sites())


def hlb_lattice(flags=0):
    """(c[Q,3], w[Q], opp[Q]) of the lattice selected by the HLB_LATTICE_* bits of flags."""
    c = np.zeros((19, 3), dtype=np.int32)
    w = np.zeros(19, dtype=np.float64)
    opp = np.zeros(19, dtype=np.int32)
    q = _lib.hlb_lattice(int(flags), _ptr(c), _ptr(w), _ptr(opp))
    return c[:q].copy(), w[:q].copy(), opp[:q].copy()


def _params(site_type, periodic, tau, iolet_rho, flags):
    st = np.ascontiguousarray(site_type, dtype=np.uint8)
    if st.ndim != 3:
        raise ValueError("site_type must be a (nz, ny, nx) array")
    nz, ny, nx = st.shape
    io = np.ascontiguousarray(np.asarray(iolet_rho, dtype=np.float64).reshape(-1))
    p = hlb_params()
    p.nx, p.ny, p.nz = nx, ny, nz
    p.periodic = int(periodic)
    p.tau = float(tau)
    p.n_iolets = int(io.shape[0])
    p.iolet_rho = io.ctypes.data if io.shape[0] else None
    p.flags = int(flags)
    return st, io, p


def hlb_preprocess(site_type, periodic=0, n_iolets=0, flags=0):
    """Host-only preprocessor: returns dict(N, Ns, voxel_of_site, canon_of_site, nbr[Q-1, Ns])."""
    st, io, p = _params(site_type, periodic, 1.0, np.ones(n_iolets), flags)
    n, ns = ctypes.c_int64(0), ctypes.c_int64(0)
    _check(_lib.hlb_preprocess_count(_ptr(st), ctypes.byref(p), ctypes.byref(n), ctypes.byref(ns)))
    N, Ns = n.value, ns.value
    vox = np.zeros(N, dtype=np.int64)
    canon = np.zeros(N, dtype=np.int32)
    nbr = np.zeros((18 if int(flags) & HLB_LATTICE_D3Q19 else 14, Ns), dtype=np.int32)
    _check(_lib.hlb_preprocess_tables(_ptr(st), ctypes.byref(p), _ptr(vox), _ptr(canon), _ptr(nbr)))
    return {"N": N, "Ns": Ns, "voxel_of_site": vox, "canon_of_site": canon, "nbr": nbr}


def hlb_preprocess_records(nbr):
    """Run-length link records of a [Q-1, Ns] table: (rec [Ns/32, Q-1, 4] uint32, n_sentinel)."""
    nbr = np.ascontiguousarray(nbr, dtype=np.int32)
    if nbr.ndim != 2 or nbr.shape[0] not in (14, 18):
        raise ValueError("nbr must be [14, Ns] or [18, Ns]")
    nl, ns = nbr.shape
    rec = np.zeros((max(ns // 32, 0), nl, 4), dtype=np.uint32)
    n = ctypes.c_int64(0)
    _check(_lib.hlb_preprocess_records(_ptr(nbr), nl, ns, _ptr(rec), ctypes.byref(n)))
    return rec, n.value


def hlb_preprocess_bfl(nbr, canon_of_site, d27):
    """Site form of the interpolated-wall tables (host only): dict(index [Ns/32, 2] uint32,
    coef [n_flagged, row] float64, n_flagged, n_interpolated); see include/hlb.h."""
    nbr = np.ascontiguousarray(nbr, dtype=np.int32)
    canon = np.ascontiguousarray(canon_of_site, dtype=np.int32)
    d27 = np.ascontiguousarray(d27, dtype=np.float64)
    if nbr.ndim != 2 or nbr.shape[0] not in (14, 18):
        raise ValueError("nbr must be [14, Ns] or [18, Ns]")
    nl, ns = nbr.shape
    n = canon.shape[0]
    if d27.shape != (n, 27):
        raise ValueError("d27 must be [N, 27]")
    nf, ni = ctypes.c_int64(0), ctypes.c_int64(0)
    index = np.zeros((ns // 32, 2), dtype=np.uint32)
    _check(_lib.hlb_preprocess_bfl(_ptr(nbr), _ptr(canon), nl, n, ns, _ptr(d27), _ptr(index), None, 0,
                                   ctypes.byref(nf), ctypes.byref(ni)))
    row = ((nl // 2 + 2) // 2) * 2
    coef = np.zeros((max(nf.value, 1), row), dtype=np.float64)
    _check(_lib.hlb_preprocess_bfl(_ptr(nbr), _ptr(canon), nl, n, ns, _ptr(d27), None, _ptr(coef), coef.shape[0],
                                   None, None))
    return {"index": index, "coef": coef[:nf.value], "n_flagged": nf.value, "n_interpolated": ni.value}


class Geometry:
    """Owner of one hlb_geometry handle and of the torch buffers behind it."""

    def __init__(self, site_type, periodic=0, tau=1.0, iolet_rho=(), flags=0, device=None,
                 stream=None, copy_stream=None):
        import torch
        if not torch.cuda.is_available():
            raise HlbError(HLB_ECUDA, "no CUDA device: the site update has no CPU fallback")
        self._torch = torch
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None \
            else torch.device(device)
        self._buffers = []
        self._h = ctypes.c_void_p(None)
        st, io, p = _params(site_type, periodic, tau, iolet_rho, flags)

        def _alloc(nbytes, _user):
            try:
                t = torch.empty(max(int(nbytes), 1), dtype=torch.uint8, device=self.device)
            except Exception:  # OOM -> NULL -> HLB_ENOMEM
                return None
            self._buffers.append(t)
            return t.data_ptr()

        def _free(ptr, _user):
            for k, t in enumerate(self._buffers):
                if t.data_ptr() == ptr:
                    del self._buffers[k]
                    return

        self._alloc_cb = _ALLOC_FN(_alloc)     # keep the callback objects alive
        self._free_cb = _FREE_FN(_free)
        p.alloc = self._alloc_cb
        p.free = self._free_cb
        p.alloc_user = None
        with torch.cuda.device(self.device):
            self.stream = torch.cuda.current_stream() if stream is None else stream
            p.stream = self.stream.cuda_stream
            self.copy_stream = copy_stream     # a torch.cuda.Stream for hlb_get_macroscopic_async
            p.copy_stream = copy_stream.cuda_stream if copy_stream is not None else None
            _check(_lib.hlb_geometry_create(_ptr(st), ctypes.byref(p), ctypes.byref(self._h)))
        self.n_sites = int(_lib.hlb_num_sites(self._h))
        self.n_q = int(_lib.hlb_num_q(self._h))
        self.n_iolets = int(p.n_iolets)
        self.flags = int(flags)

    def _call(self, fn, *args):
        """Every library call runs with the geometry's device current: the library itself never
        calls cudaSetDevice, and its launches go to whatever device is current."""
        with self._torch.cuda.device(self.device):
            return fn(self._h, *args)

    # -- the C-ABI calls, same names -------------------------------------------------
    def hlb_set_state(self, rho=None, u=None):
        n = self.n_sites
        rho, u = _host(rho, np.float64, (n,)), _host(u, np.float64, (n, 3))
        _check(self._call(_lib.hlb_set_state, _ptr(rho), _ptr(u)))

    def hlb_set_iolet_density(self, iolet_rho):
        io = _host(np.asarray(iolet_rho).reshape(-1), np.float64, (self.n_iolets,))
        _check(self._call(_lib.hlb_set_iolet_density, _ptr(io)))

    def hlb_set_iolet_velocity(self, kind, u=None):
        kind = None if kind is None else _host(np.asarray(kind).reshape(-1), np.uint8, (self.n_iolets,))
        u = None if u is None else _host(np.asarray(u, dtype=np.float64).reshape(-1, 3), np.float64,
                                         (self.n_iolets, 3))
        _check(self._call(_lib.hlb_set_iolet_velocity, _ptr(kind), _ptr(u)))

    def hlb_set_iolet_weight(self, weight):
        w = None if weight is None else _host(np.asarray(weight, dtype=np.float64).reshape(-1),
                                              np.float64, (self.n_sites,))
        _check(self._call(_lib.hlb_set_iolet_weight, _ptr(w)))

    def hlb_set_iolet_waveform(self, u):
        """u: [n_t][n_iolets][3] (or None to remove the waveform)."""
        if u is None:
            _check(self._call(_lib.hlb_set_iolet_waveform, None, 0))
            return
        u = _host(np.asarray(u, dtype=np.float64), np.float64)
        if u.ndim != 3 or u.shape[2] != 3:
            raise ValueError("waveform must have shape [n_t][n_iolets][3]")
        if u.shape[1] != self.n_iolets:
            raise ValueError(f"waveform has {u.shape[1]} iolets, the geometry {self.n_iolets}")
        _check(self._call(_lib.hlb_set_iolet_waveform, _ptr(u), int(u.shape[0])))

    def hlb_set_iolet_normal(self, normals):
        n = None if normals is None else _host(np.asarray(normals, dtype=np.float64).reshape(-1, 3), np.float64,
                                               (self.n_iolets, 3))
        _check(self._call(_lib.hlb_set_iolet_normal, _ptr(n)))

    def hlb_set_wall_distance(self, d27):
        d27 = None if d27 is None else _host(d27, np.float64, (self.n_sites, 27))
        _check(self._call(_lib.hlb_set_wall_distance, _ptr(d27)))

    def hlb_num_bfl_sites(self) -> int:
        return int(self._call(_lib.hlb_num_bfl_sites))

    def hlb_step(self, n: int = 1):
        _check(self._call(_lib.hlb_step, int(n)))

    def hlb_get_macroscopic(self, rho_out=None, u_out=None):
        """Host results (numpy); pass preallocated (e.g. pinned) arrays to reuse them."""
        n = self.n_sites
        rho = np.empty(n, dtype=np.float64) if rho_out is None else rho_out
        u = np.empty((n, 3), dtype=np.float64) if u_out is None else u_out
        for a, shape in ((rho, (n,)), (u, (n, 3))):
            if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.shape == shape
                    and a.flags.c_contiguous and a.flags.writeable):
                raise ValueError(f"output array must be a writable C-contiguous float64 array of shape {shape}")
        _check(self._call(_lib.hlb_get_macroscopic, _ptr(rho), _ptr(u)))
        return rho, u

    def hlb_get_macroscopic_async(self, rho_out, u_out):
        """Read-out into caller-owned PINNED host arrays without waiting (needs copy_stream);
        valid after hlb_wait_copies()."""
        n = self.n_sites
        for a, shape in ((rho_out, (n,)), (u_out, (n, 3))):
            if a is not None and not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.shape == shape
                                      and a.flags.c_contiguous and a.flags.writeable):
                raise ValueError(f"output array must be a writable C-contiguous float64 array of shape {shape}")
        _check(self._call(_lib.hlb_get_macroscopic_async, _ptr(rho_out), _ptr(u_out)))

    def hlb_stage_state(self, rho=None, u=None):
        """Upload rho [N] / u [N, 3] (PINNED float64 numpy arrays, kept alive and unchanged by the
        caller until hlb_wait_copies()) into the staging buffer on the copy stream; no effect on
        the simulation until hlb_set_state_staged()."""
        n = self.n_sites
        for a, shape in ((rho, (n,)), (u, (n, 3))):
            if a is not None and not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.shape == shape
                                      and a.flags.c_contiguous):
                raise ValueError(f"expected a C-contiguous float64 array of shape {shape}")
        _check(self._call(_lib.hlb_stage_state, _ptr(rho), _ptr(u)))

    def hlb_set_state_staged(self):
        _check(self._call(_lib.hlb_set_state_staged))

    def hlb_wait_copies(self):
        _check(self._call(_lib.hlb_wait_copies))

    def hlb_get_macroscopic_device(self):
        """rho [N], u [N,3] as torch cuda tensors (canonical order), stream-ordered."""
        torch = self._torch
        rho = torch.empty(self.n_sites, dtype=torch.float64, device=self.device)
        u = torch.empty((self.n_sites, 3), dtype=torch.float64, device=self.device)
        _check(self._call(_lib.hlb_get_macroscopic_device, rho.data_ptr(), u.data_ptr()))
        return rho, u

    def hlb_get_stress(self):
        """Deviatoric stress [N, 6] (xx, yy, zz, xy, xz, yz), host."""
        sg = np.empty((self.n_sites, 6), dtype=np.float64)
        _check(self._call(_lib.hlb_get_stress, _ptr(sg)))
        return sg

    def hlb_get_wall_shear_stress(self, normals):
        nrm = _host(normals, np.float64, (self.n_sites, 3))
        out = np.empty(self.n_sites, dtype=np.float64)
        _check(self._call(_lib.hlb_get_wall_shear_stress, _ptr(nrm), _ptr(out)))
        return out

    def hlb_get_wall_shear_stress_noalloc(self, normals_dev, wss_dev):
        """No-allocation variant (include/hlb.h): normals_dev [N, 3] and wss_dev [N] are the
        caller's float64 CUDA tensors on this geometry's device; nothing is allocated, nothing
        synchronised; N <= hlb_noalloc_max_sites()."""
        torch = self._torch
        for t, shape in ((normals_dev, (self.n_sites, 3)), (wss_dev, (self.n_sites,))):
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.device == self.device and
                    t.dtype == torch.float64 and tuple(t.shape) == shape and t.is_contiguous()):
                raise ValueError(f"expected a contiguous float64 CUDA tensor of shape {shape} on {self.device}")
        _check(self._call(_lib.hlb_get_wall_shear_stress_noalloc, normals_dev.data_ptr(), wss_dev.data_ptr()))

    def hlb_get_stress_device(self):
        torch = self._torch
        sg = torch.empty((self.n_sites, 6), dtype=torch.float64, device=self.device)
        _check(self._call(_lib.hlb_get_stress_device, sg.data_ptr()))
        return sg

    def hlb_render(self, view: "hlb_view", lut):
        """Image [height, width, 4] float32 (host) of the current state."""
        lut = np.ascontiguousarray(np.asarray(lut, dtype=np.float32).reshape(256, 4))
        img = np.empty((view.height, view.width, 4), dtype=np.float32)
        _check(self._call(_lib.hlb_render, ctypes.byref(view), _ptr(lut), _ptr(img)))
        return img

    def hlb_render_device(self, view: "hlb_view", lut):
        torch = self._torch
        lut = np.ascontiguousarray(np.asarray(lut, dtype=np.float32).reshape(256, 4))
        img = torch.empty((view.height, view.width, 4), dtype=torch.float32, device=self.device)
        _check(self._call(_lib.hlb_render_device, ctypes.byref(view), _ptr(lut), img.data_ptr()))
        return img

    def hlb_get_populations(self):
        f = np.empty((self.n_sites, self.n_q), dtype=np.float64)
        _check(self._call(_lib.hlb_get_populations, _ptr(f)))
        return f

    def hlb_set_populations(self, f):
        f = _host(f, np.float64, (self.n_sites, self.n_q))
        _check(self._call(_lib.hlb_set_populations, _ptr(f)))

    def hlb_num_q(self) -> int:
        return int(self._call(_lib.hlb_num_q))

    def hlb_num_sites(self) -> int:
        return int(self._call(_lib.hlb_num_sites))

    def hlb_steps_done(self) -> int:
        return int(self._call(_lib.hlb_steps_done))

    def hlb_get_site_voxels(self):
        v = np.empty(self.n_sites, dtype=np.int64)
        _check(self._call(_lib.hlb_get_site_voxels, _ptr(v)))
        return v

    def hlb_device_bytes(self) -> int:
        return int(self._call(_lib.hlb_device_bytes))

    def hlb_launch_count(self) -> int:
        return int(self._call(_lib.hlb_launch_count))

    def hlb_offset_bits(self) -> int:
        return int(self._call(_lib.hlb_offset_bits))

    def hlb_uses_aa(self) -> bool:
        return bool(self._call(_lib.hlb_uses_aa))

    def hlb_uses_records(self) -> bool:
        return bool(self._call(_lib.hlb_uses_records))

    def hlb_record_sentinel_fraction(self) -> float:
        return float(self._call(_lib.hlb_record_sentinel_fraction))

    def hlb_geometry_destroy(self):
        if self._h:
            self._torch.cuda.synchronize(self.device)
            self._call(_lib.hlb_geometry_destroy)
            self._h = ctypes.c_void_p(None)
            self._buffers.clear()

    close = hlb_geometry_destroy

    def __del__(self):
        try:
            self.hlb_geometry_destroy()
        except Exception:
            pass


def hlb_geometry_create(site_type, periodic=0, tau=1.0, iolet_rho=(), flags=0, **kw) -> Geometry:
    return Geometry(site_type, periodic, tau, iolet_rho, flags, **kw)
