"""Thin Python binding of libtpmc.so (include/tpmc.h): argument marshalling only.

Every step of the hot path (seed, LBVH build, trace, reflect, accumulate, reduce) runs in the
hand-written CUDA kernels of csrc/; PyTorch is used here for device buffers and streams.
There is no CPU fallback and this package never imports ``oracle``: if the library is missing
or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtpmc.so")

TPMC_OK, TPMC_EINVAL, TPMC_ENOMEM, TPMC_ECUDA, TPMC_ECAPACITY = 0, -1, -2, -3, -4
TPMC_STATIC_MAX_FACETS = 8388608
TPMC_MEM_HOST, TPMC_MEM_DEVICE = 0, 1
TPMC_MAX_SPECIES = 8
TPMC_MAX_BOUNCES = 0x0FFFFFFF
TPMC_FLAG_NO_PRECULL, TPMC_FLAG_NO_HORIZON, TPMC_FLAG_ALIGN_OFF, TPMC_FLAG_ALIGN_ON = 0x01, 0x02, 0x04, 0x08
TPMC_FLAG_EXACT_TRACE, TPMC_FLAG_SORT_RAYS, TPMC_FLAG_NO_AGGREGATION, TPMC_FLAG_SERIAL_SEED = 0x10, 0x20, 0x40, 0x80
TPMC_CV_SPHERE, TPMC_CV_BOX, TPMC_CV_BOX_UNWEIGHTED = 0, 1, 2
TPMC_MESH_NO_HORIZON = 0x1

EXPORTS = ["tpmc_mesh_create", "tpmc_mesh_destroy", "tpmc_mesh_info", "tpmc_mesh_copy_bvh", "tpmc_run",
           "tpmc_mesh_copy_horizon", "tpmc_run_host", "tpmc_seed", "tpmc_trace", "tpmc_strerror", "tpmc_last_cuda_error", "tpmc_version",
           "tpmc_measure_peaks", "tpmc_mesh_set_surface", "tpmc_run_sweep", "tpmc_mesh_copy_wide", "tpmc_facet_sum_static",
           "tpmc_mesh_create_ex", "tpmc_mesh_build_horizon"]


class TpmcError(RuntimeError):
    pass


class tpmc_mesh_info_t(C.Structure):
    _fields_ = [("centre", C.c_double * 3), ("bounding_radius", C.c_double), ("aabb_lo", C.c_float * 3),
                ("aabb_hi", C.c_float * 3), ("nt", C.c_int64), ("n_nodes", C.c_int64), ("build_ms", C.c_double),
                ("horizon_ms", C.c_double)]


class tpmc_params(C.Structure):
    _fields_ = [("n", C.c_double), ("T_inf", C.c_double), ("T_W", C.c_double), ("V", C.c_double * 3),
                ("accommodation", C.c_double), ("n_species", C.c_int32),
                ("m", C.POINTER(C.c_double)), ("x", C.POINTER(C.c_double)),
                ("cv_radius_factor", C.c_double), ("N", C.c_uint64), ("first", C.c_uint64),
                ("count", C.c_uint64), ("seed", C.c_uint64), ("max_bounces", C.c_uint32),
                ("x_ref", C.c_double * 3), ("energy_accommodation", C.c_double), ("wave_particles", C.c_uint64),
                ("chunk_particles", C.c_uint64), ("flags", C.c_uint32), ("control_volume", C.c_int32)]


class tpmc_stats(C.Structure):
    _fields_ = [("hits", C.c_uint64), ("segments", C.c_uint64), ("escaped", C.c_uint64), ("truncated", C.c_uint64),
                ("culled", C.c_uint64), ("tri_tests", C.c_uint64), ("node_visits", C.c_uint64),
                ("kernel_launches", C.c_uint64), ("ms", C.c_double), ("ms_seed", C.c_double), ("ms_trace", C.c_double),
                ("ms_reflect", C.c_double), ("ms_finish", C.c_double), ("timed_waves", C.c_uint64),
                ("trace_launches", C.c_uint64), ("traced_rays", C.c_uint64),
                ("ret_precull_a", C.c_uint64), ("ret_precull_b", C.c_uint64), ("ret_seed", C.c_uint64),
                ("ret_trace", C.c_uint64), ("ret_resolve", C.c_uint64), ("ret_horizon", C.c_uint64),
                ("ret_finish", C.c_uint64), ("queued_primaries", C.c_uint64), ("queued_reflected", C.c_uint64),
                ("overflow_rays", C.c_uint64), ("final_stragglers", C.c_uint64), ("finish_segments", C.c_uint64),
                ("ms_sort", C.c_double), ("precull_uncertified", C.c_uint64)]


class tpmc_peaks(C.Structure):
    _fields_ = [("sms", C.c_int32), ("sm_clock_mhz_nominal", C.c_double), ("sm_clock_mhz_fp32", C.c_double),
                ("fp32_lane_ops_per_s", C.c_double), ("fp64_fma_per_s", C.c_double), ("gather32_bytes_per_s", C.c_double),
                ("gather32_dependent_bytes_per_s", C.c_double), ("gather_array_bytes", C.c_double),
                ("red_f64_per_s", C.c_double * 3), ("red_f64_addresses", C.c_double * 3),
                ("gather64_bytes_per_s", C.c_double)]


class tpmc_debug(C.Structure):
    _fields_ = [("hash", C.c_void_p), ("bounces", C.c_void_p), ("first_facet", C.c_void_p)]


_lib = None


def lib():
    """Load libtpmc.so (built in-tree by build.py).  Raises if it is missing: no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise TpmcError(f"{LIB_PATH} not found: run `python -m paper_1312_3691_b200.build` "
                            "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.tpmc_mesh_create.restype = C.c_int
        L.tpmc_mesh_create.argtypes = [vp, C.c_int64, vp, C.c_int64, vp, C.c_int, vp, C.POINTER(vp)]
        L.tpmc_mesh_create_ex.restype = C.c_int
        L.tpmc_mesh_create_ex.argtypes = [vp, C.c_int64, vp, C.c_int64, vp, C.c_int, C.c_uint32, vp, C.POINTER(vp)]
        L.tpmc_mesh_build_horizon.restype = C.c_int
        L.tpmc_mesh_build_horizon.argtypes = [vp, vp]
        L.tpmc_mesh_destroy.restype = None
        L.tpmc_mesh_destroy.argtypes = [vp]
        L.tpmc_mesh_info.restype = C.c_int
        L.tpmc_mesh_info.argtypes = [vp, C.POINTER(tpmc_mesh_info_t)]
        L.tpmc_mesh_set_surface.restype = C.c_int
        L.tpmc_mesh_set_surface.argtypes = [vp, vp, vp, C.c_int, vp]
        L.tpmc_mesh_copy_wide.restype = C.c_int
        L.tpmc_mesh_copy_wide.argtypes = [vp, vp, vp, vp]
        L.tpmc_mesh_copy_bvh.restype = C.c_int
        L.tpmc_mesh_copy_bvh.argtypes = [vp, vp, vp]
        L.tpmc_mesh_copy_horizon.restype = C.c_int
        L.tpmc_mesh_copy_horizon.argtypes = [vp, vp]
        L.tpmc_run.restype = C.c_int
        L.tpmc_run.argtypes = [vp, C.POINTER(tpmc_params), vp, vp, vp, vp, C.POINTER(tpmc_stats), C.POINTER(tpmc_debug)]
        L.tpmc_run_sweep.restype = C.c_int
        L.tpmc_run_sweep.argtypes = [vp, C.POINTER(tpmc_params), C.c_int32, vp, vp, vp, vp, vp, vp]
        L.tpmc_run_host.restype = C.c_int
        L.tpmc_run_host.argtypes = [vp, C.POINTER(tpmc_params), vp, vp, vp, vp, C.POINTER(tpmc_stats)]
        L.tpmc_seed.restype = C.c_int
        L.tpmc_seed.argtypes = [vp, C.POINTER(tpmc_params), vp, vp, vp, vp]
        L.tpmc_trace.restype = C.c_int
        L.tpmc_trace.argtypes = [vp, vp, vp, vp, C.c_int64, vp, vp, vp, vp]
        L.tpmc_facet_sum_static.restype = C.c_int
        L.tpmc_facet_sum_static.argtypes = [vp, C.c_int64, vp, vp]
        L.tpmc_measure_peaks.restype = C.c_int
        L.tpmc_measure_peaks.argtypes = [C.POINTER(tpmc_peaks), vp]
        for n in ("tpmc_strerror", "tpmc_last_cuda_error", "tpmc_version"):
            getattr(L, n).restype = C.c_char_p
        L.tpmc_strerror.argtypes = [C.c_int]
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != TPMC_OK:
        L = lib()
        msg = L.tpmc_strerror(rc).decode()
        if rc in (TPMC_ECUDA, TPMC_ECAPACITY):
            msg += ": " + L.tpmc_last_cuda_error().decode()
        raise TpmcError(f"{what} failed ({rc}): {msg}")


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise TpmcError("no CUDA device: the TPMC hot path has no CPU fallback")
    return torch


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        return _torch().cuda.current_stream().cuda_stream or None
    return getattr(stream, "cuda_stream", stream) or None


def make_params(cfg, first=None, count=None, N=None, flags=0, wave_particles=0, chunk_particles=0):
    """Marshal a parameter record (anything with the tpmc_params field names, e.g.
    tpmc_inputs.RunConfig) into a C struct.  Returns (struct, keepalive)."""
    p = tpmc_params()
    p.n, p.T_inf, p.T_W = float(cfg.n), float(cfg.T_inf), float(cfg.T_W)
    p.V = (C.c_double * 3)(*[float(a) for a in cfg.V])
    p.accommodation = float(cfg.accommodation)
    m = np.ascontiguousarray(cfg.m, dtype=np.float64)
    x = np.ascontiguousarray(cfg.x, dtype=np.float64)
    p.n_species = int(m.size)
    p.m = m.ctypes.data_as(C.POINTER(C.c_double))
    p.x = x.ctypes.data_as(C.POINTER(C.c_double))
    p.cv_radius_factor = float(cfg.cv_radius_factor)
    p.N = int(cfg.N if N is None else N)
    p.first = int(0 if first is None else first)
    p.count = int(p.N - p.first if count is None else count)
    p.seed = int(cfg.seed)
    p.max_bounces = int(cfg.max_bounces)
    p.x_ref = (C.c_double * 3)(*[float(a) for a in cfg.x_ref])
    p.energy_accommodation = float(getattr(cfg, "energy_accommodation", 1.0))
    p.wave_particles = int(wave_particles)
    p.chunk_particles = int(chunk_particles)
    p.flags = int(flags)
    p.control_volume = int(getattr(cfg, "control_volume", TPMC_CV_SPHERE))
    return p, (m, x)


@dataclass
class RunResult:
    force: "object"                 # torch [3] float64, device
    torque: "object"                # torch [3] float64, device
    facet_momentum: "object"        # torch [nt,3] float64 device, or None
    stats: Optional[dict]
    hash: "object" = None           # torch [count] int64 (bit pattern of the u64 hash), device
    bounces: "object" = None        # torch [count] int32
    first_facet: "object" = None    # torch [count] int32


class Mesh:
    """Owns a tpmc_mesh handle (triangulation + on-device LBVH)."""

    def __init__(self, vertices, indices, flags=None, stream=None, mesh_flags=0):
        """mesh_flags: TPMC_MESH_* (0 = tpmc_mesh_create's behaviour; else tpmc_mesh_create_ex)."""
        L = lib()
        torch = _torch()
        self._h = C.c_void_p()
        if isinstance(vertices, np.ndarray) or not hasattr(vertices, "is_cuda"):
            v = np.ascontiguousarray(vertices, dtype=np.float32)
            i = np.ascontiguousarray(indices, dtype=np.int32)
            f = None if flags is None else np.ascontiguousarray(flags, dtype=np.uint8)
            nv, nt = v.shape[0], i.shape[0]
            args = (v.ctypes.data, nv, i.ctypes.data, nt, None if f is None else f.ctypes.data, TPMC_MEM_HOST)
        else:
            v = vertices.to(dtype=torch.float32).contiguous()
            i = indices.to(dtype=torch.int32).contiguous()
            f = None if flags is None else flags.to(dtype=torch.uint8).contiguous()
            if not (v.is_cuda and i.is_cuda and (f is None or f.is_cuda)):
                raise TpmcError("device meshes need CUDA tensors")
            nv, nt = v.shape[0], i.shape[0]
            args = (v.data_ptr(), nv, i.data_ptr(), nt, None if f is None else f.data_ptr(), TPMC_MEM_DEVICE)
        if mesh_flags:
            _check(L.tpmc_mesh_create_ex(*args, int(mesh_flags), _stream_ptr(stream), C.byref(self._h)), "tpmc_mesh_create_ex")
        else:
            _check(L.tpmc_mesh_create(*args, _stream_ptr(stream), C.byref(self._h)), "tpmc_mesh_create")
        self.nt = int(nt)
        self.nv = int(nv)

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().tpmc_mesh_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self) -> dict:
        out = tpmc_mesh_info_t()
        _check(lib().tpmc_mesh_info(self._h, C.byref(out)), "tpmc_mesh_info")
        return {"centre": np.array(list(out.centre)), "bounding_radius": out.bounding_radius,
                "aabb_lo": np.array(list(out.aabb_lo)), "aabb_hi": np.array(list(out.aabb_hi)),
                "nt": int(out.nt), "n_nodes": int(out.n_nodes), "build_ms": out.build_ms, "horizon_ms": out.horizon_ms}

    def set_surface(self, T_W=None, sigma=None, stream=None):
        """Per-facet wall temperature / accommodation (tpmc_mesh_set_surface); None restores the run's scalar.
        Host arrays, or CUDA float64 tensors (then both must be CUDA tensors or None)."""
        on_dev = [a is not None and hasattr(a, "is_cuda") and a.is_cuda for a in (T_W, sigma)]
        if any(on_dev):
            torch = _torch()
            if not all(d or a is None for d, a in zip(on_dev, (T_W, sigma))):
                raise TpmcError("surface arrays must live in one memory space")
            tw = None if T_W is None else T_W.to(torch.float64).contiguous()
            sg = None if sigma is None else sigma.to(torch.float64).contiguous()
            ptr = lambda a: None if a is None else a.data_ptr()
            space = TPMC_MEM_DEVICE
        else:
            tw = None if T_W is None else np.ascontiguousarray(T_W, dtype=np.float64)
            sg = None if sigma is None else np.ascontiguousarray(sigma, dtype=np.float64)
            ptr = lambda a: None if a is None else a.ctypes.data
            space = TPMC_MEM_HOST
        for a in (tw, sg):
            if a is not None and tuple(a.shape) != (self.nt,):
                raise TpmcError("surface arrays must have one entry per facet")
        _check(lib().tpmc_mesh_set_surface(self._h, ptr(tw), ptr(sg), space, _stream_ptr(stream)), "tpmc_mesh_set_surface")

    def build_horizon(self, stream=None):
        """Add the escape horizons to a mesh created with TPMC_MESH_NO_HORIZON (tpmc_mesh_build_horizon)."""
        _check(lib().tpmc_mesh_build_horizon(self._h, _stream_ptr(stream)), "tpmc_mesh_build_horizon")

    def copy_bvh(self):
        n_nodes = self.info()["n_nodes"]
        nodes = np.zeros((n_nodes, 16), dtype=np.float32)
        leaf = np.zeros(self.nt, dtype=np.int32)
        _check(lib().tpmc_mesh_copy_bvh(self._h, nodes.ctypes.data, leaf.ctypes.data), "tpmc_mesh_copy_bvh")
        return nodes, leaf

    def copy_wide(self):
        n = C.c_int64(0)
        _check(lib().tpmc_mesh_copy_wide(self._h, C.byref(n), None, None), "tpmc_mesh_copy_wide")
        wn = np.zeros((n.value, 16), dtype=np.uint32)
        grid = np.zeros(6, dtype=np.float32)
        _check(lib().tpmc_mesh_copy_wide(self._h, C.byref(n), wn.ctypes.data, grid.ctypes.data), "tpmc_mesh_copy_wide")
        return wn, grid

    def copy_horizon(self):
        hz = np.zeros((self.nt, 16), dtype=np.uint8)
        _check(lib().tpmc_mesh_copy_horizon(self._h, hz.ctypes.data), "tpmc_mesh_copy_horizon")
        return hz

    # ------------------------------------------------------------------ the hot path
    def run(self, cfg, first=None, count=None, N=None, facets=True, debug=False, stats=True, stream=None,
            flags=0, wave_particles=0, chunk_particles=0) -> RunResult:
        torch = _torch()
        p, keep = make_params(cfg, first, count, N, flags, wave_particles, chunk_particles)
        dev = torch.device("cuda", torch.cuda.current_device())
        force = torch.empty(3, dtype=torch.float64, device=dev)
        torque = torch.empty(3, dtype=torch.float64, device=dev)
        fm = torch.empty((self.nt, 3), dtype=torch.float64, device=dev) if facets else None
        dbg, hs, nb, ff = None, None, None, None
        if debug:
            cnt = int(p.count)
            hs = torch.empty(cnt, dtype=torch.int64, device=dev)
            nb = torch.empty(cnt, dtype=torch.int32, device=dev)
            ff = torch.empty(cnt, dtype=torch.int32, device=dev)
            dbg = tpmc_debug(hs.data_ptr() or None, nb.data_ptr() or None, ff.data_ptr() or None)
        st = tpmc_stats() if stats else None
        rc = lib().tpmc_run(self._h, C.byref(p), _stream_ptr(stream), force.data_ptr(), torque.data_ptr(),
                            None if fm is None else fm.data_ptr(), None if st is None else C.byref(st),
                            None if dbg is None else C.byref(dbg))
        _check(rc, "tpmc_run")
        sd = None if st is None else {k: getattr(st, k) for k, _ in tpmc_stats._fields_}
        return RunResult(force, torque, fm, sd, hs, nb, ff)

    def sweep(self, cfg, velocities, facets=False, stats=False, stream=None, flags=0):
        """tpmc_run_sweep: one run per row of `velocities` [K,3]; returns (force [K,3], torque [K,3], facet momentum
        [K,nt,3] or None, list of stats dicts or None), device tensors."""
        torch = _torch()
        p, keep = make_params(cfg, flags=flags)
        V = np.ascontiguousarray(velocities, dtype=np.float64).reshape(-1, 3)
        K = int(V.shape[0])
        dev = torch.device("cuda", torch.cuda.current_device())
        force = torch.empty((K, 3), dtype=torch.float64, device=dev)
        torque = torch.empty((K, 3), dtype=torch.float64, device=dev)
        fm = torch.empty((K, self.nt, 3), dtype=torch.float64, device=dev) if facets else None
        st = (tpmc_stats * K)() if stats else None
        rc = lib().tpmc_run_sweep(self._h, C.byref(p), K, V.ctypes.data, _stream_ptr(stream), force.data_ptr() or None,
                                  torque.data_ptr() or None, None if fm is None else fm.data_ptr(),
                                  None if st is None else C.cast(st, C.c_void_p))
        _check(rc, "tpmc_run_sweep")
        sd = None if st is None else [{k: getattr(s, k) for k, _ in tpmc_stats._fields_} for s in st]
        return force, torque, fm, sd

    def run_host(self, cfg, first=None, count=None, N=None, facets=True, stats=True, stream=None,
                 out_facets: Optional[np.ndarray] = None, flags=0):
        """tpmc_run_host: results land in HOST numpy buffers (D2H copies inside the call)."""
        _torch()
        p, keep = make_params(cfg, first, count, N, flags)
        force = np.empty(3, dtype=np.float64)
        torque = np.empty(3, dtype=np.float64)
        fm = None
        if facets:
            fm = out_facets if out_facets is not None else np.empty((self.nt, 3), dtype=np.float64)
        st = tpmc_stats() if stats else None
        rc = lib().tpmc_run_host(self._h, C.byref(p), _stream_ptr(stream), force.ctypes.data, torque.ctypes.data,
                                 None if fm is None else fm.ctypes.data, None if st is None else C.byref(st))
        _check(rc, "tpmc_run_host")
        sd = None if st is None else {k: getattr(st, k) for k, _ in tpmc_stats._fields_}
        return force, torque, fm, sd

    def seed(self, cfg, first=None, count=None, N=None, stream=None):
        """fp64 (x, v, species) of particles [first, first+count) before the fp32 rounding (tpmc_seed)."""
        torch = _torch()
        p, keep = make_params(cfg, first, count, N)
        dev = torch.device("cuda", torch.cuda.current_device())
        cnt = int(p.count)
        x = torch.empty((cnt, 3), dtype=torch.float64, device=dev)
        v = torch.empty((cnt, 3), dtype=torch.float64, device=dev)
        s = torch.empty(cnt, dtype=torch.int32, device=dev)
        _check(lib().tpmc_seed(self._h, C.byref(p), _stream_ptr(stream), x.data_ptr() or None, v.data_ptr() or None,
                               s.data_ptr() or None), "tpmc_seed")
        return x, v, s

    def trace(self, o, d, f_prev=None, stream=None, align_V=None):
        """Closest hit of rays o + tau d (tpmc_trace).  o, d: [n,3] float32 (numpy or CUDA tensors); align_V: walk
        the hierarchy refitted in the stream frame of this bulk velocity instead of the body-frame one."""
        torch = _torch()
        dev = torch.device("cuda", torch.cuda.current_device())
        o = torch.as_tensor(np.ascontiguousarray(o, dtype=np.float32) if isinstance(o, np.ndarray) else o).to(dev, torch.float32).contiguous()
        d = torch.as_tensor(np.ascontiguousarray(d, dtype=np.float32) if isinstance(d, np.ndarray) else d).to(dev, torch.float32).contiguous()
        n = int(o.shape[0])
        fp = None
        if f_prev is not None:
            fp = torch.as_tensor(f_prev).to(dev, torch.int32).contiguous()
        facet = torch.empty(n, dtype=torch.int32, device=dev)
        tau = torch.empty(n, dtype=torch.float64, device=dev)
        av = None if align_V is None else (C.c_double * 3)(*[float(a) for a in align_V])
        _check(lib().tpmc_trace(self._h, o.data_ptr() or None, d.data_ptr() or None, None if fp is None else fp.data_ptr(),
                                n, av, _stream_ptr(stream), facet.data_ptr() or None, tau.data_ptr() or None), "tpmc_trace")
        return facet, tau


# C-ABI names, as plain functions -------------------------------------------------------------------
def tpmc_mesh_create(vertices, indices, flags=None, stream=None) -> Mesh:
    return Mesh(vertices, indices, flags, stream)


def tpmc_mesh_create_ex(vertices, indices, flags=None, mesh_flags=0, stream=None) -> Mesh:
    return Mesh(vertices, indices, flags, stream, mesh_flags)


def tpmc_mesh_build_horizon(mesh: Mesh, **kw) -> None:
    mesh.build_horizon(**kw)


def tpmc_mesh_destroy(mesh: Mesh) -> None:
    mesh.close()


def tpmc_mesh_info(mesh: Mesh) -> dict:
    return mesh.info()


def tpmc_mesh_set_surface(mesh: Mesh, T_W=None, sigma=None, **kw) -> None:
    mesh.set_surface(T_W, sigma, **kw)


def tpmc_mesh_copy_bvh(mesh: Mesh):
    return mesh.copy_bvh()


def tpmc_mesh_copy_wide(mesh: Mesh):
    return mesh.copy_wide()


def tpmc_mesh_copy_horizon(mesh: Mesh):
    return mesh.copy_horizon()


def tpmc_run(mesh: Mesh, cfg, **kw) -> RunResult:
    return mesh.run(cfg, **kw)


def tpmc_run_sweep(mesh: Mesh, cfg, velocities, **kw):
    return mesh.sweep(cfg, velocities, **kw)


def tpmc_run_host(mesh: Mesh, cfg, **kw):
    return mesh.run_host(cfg, **kw)


def tpmc_seed(mesh: Mesh, cfg, **kw):
    return mesh.seed(cfg, **kw)


def tpmc_trace(mesh: Mesh, o, d, f_prev=None, **kw):
    return mesh.trace(o, d, f_prev, **kw)


def tpmc_facet_sum_static(facet_momentum, out=None, stream=None):
    """Sum a device [nt,3] float64 facet-momentum tensor into a device [3] force with tpmc_facet_sum_static, the entry
    point that allocates no device memory (its scratch is a fixed array inside libtpmc.so; see include/tpmc.h for who
    needs that and what it costs: at most TPMC_STATIC_MAX_FACETS facets, one call at a time per GPU).  Pass `out` (device
    [3] float64) to keep this wrapper from allocating the result too; without it a torch tensor is made for convenience."""
    torch = _torch()
    fm = facet_momentum
    if not (fm.is_cuda and fm.dtype == torch.float64 and fm.is_contiguous() and fm.dim() == 2 and fm.shape[1] == 3):
        raise TpmcError("facet_momentum must be a contiguous CUDA float64 tensor [nt, 3]")
    if out is None:
        out = torch.empty(3, dtype=torch.float64, device=fm.device)
    elif not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 3):
        raise TpmcError("out must be a contiguous CUDA float64 tensor of 3 elements")
    with torch.cuda.device(fm.device):
        _check(lib().tpmc_facet_sum_static(fm.data_ptr() or None, int(fm.shape[0]), _stream_ptr(stream), out.data_ptr()),
               "tpmc_facet_sum_static")
    return out


def tpmc_measure_peaks(stream=None) -> dict:
    """Measured peaks of the binding units (tpmc_measure_peaks): plain dict of the C struct's fields."""
    _torch()
    out = tpmc_peaks()
    _check(lib().tpmc_measure_peaks(C.byref(out), _stream_ptr(stream)), "tpmc_measure_peaks")
    d = {k: getattr(out, k) for k, _ in tpmc_peaks._fields_}
    d["red_f64_per_s"] = list(out.red_f64_per_s)
    d["red_f64_addresses"] = list(out.red_f64_addresses)
    return d


def tpmc_version() -> str:
    return lib().tpmc_version().decode()
