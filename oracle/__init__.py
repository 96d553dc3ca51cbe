"""ctypes view of the CPU oracle (oracle/tpmc_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It never
imports paper_1312_3691_b200 and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpmc_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_tpmc.so")


def build_sanitized(path: str) -> str:
    """The same source with -fsanitize=address,undefined (tests/test_oracle_pins.py runs a few workloads through it)."""
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-o", path, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return path


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (strict IEEE evaluation: no contraction, no fast-math).
    TPMC_ORACLE_LIB names an already built library to load instead (the sanitizer test)."""
    if os.environ.get("TPMC_ORACLE_LIB"):
        return os.environ["TPMC_ORACLE_LIB"]
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Params(C.Structure):
    _fields_ = [("n", C.c_double), ("T_inf", C.c_double), ("T_W", C.c_double), ("V", C.c_double * 3),
                ("accommodation", C.c_double), ("n_species", C.c_int32),
                ("m", C.POINTER(C.c_double)), ("x", C.POINTER(C.c_double)),
                ("cv_radius_factor", C.c_double), ("N", C.c_uint64), ("first", C.c_uint64),
                ("count", C.c_uint64), ("seed", C.c_uint64), ("max_bounces", C.c_uint32),
                ("x_ref", C.c_double * 3), ("energy_accommodation", C.c_double),
                ("control_volume", C.c_int32), ("pad_", C.c_int32)]


class _Stats(C.Structure):
    _fields_ = [("hits", C.c_uint64), ("segments", C.c_uint64), ("escaped", C.c_uint64), ("truncated", C.c_uint64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, vp = C.POINTER(C.c_double), C.c_void_p
        L.oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.oracle_flux_bracket.restype = C.c_double
        L.oracle_flux_bracket.argtypes = [C.c_double]
        L.oracle_flux.restype = C.c_double
        L.oracle_flux.argtypes = [C.c_double] * 4
        for name in ("oracle_position_cdf", "oracle_position_inv", "oracle_vn_cdf", "oracle_vn_inv", "oracle_vn_unweighted_inv"):
            getattr(L, name).restype = C.c_double
            getattr(L, name).argtypes = [C.c_double, C.c_double]
        L.oracle_rotation.argtypes = [dp, dp]
        L.oracle_mesh_create.restype = vp
        L.oracle_mesh_create.argtypes = [vp, C.c_int64, vp, C.c_int64, vp]
        L.oracle_mesh_destroy.argtypes = [vp]
        L.oracle_mesh_bounds.argtypes = [vp, dp, dp]
        L.oracle_mesh_set_surface.argtypes = [vp, vp, vp]
        L.oracle_closest_hit.restype = C.c_int32
        L.oracle_closest_hit.argtypes = [vp, vp, vp, C.c_int32, C.c_int, dp]
        L.oracle_seed.restype = C.c_int
        L.oracle_seed.argtypes = [vp, C.POINTER(_Params), C.c_uint64, dp, dp]
        L.oracle_reflect.argtypes = [vp, C.POINTER(_Params), C.c_int32, vp, C.c_uint64, C.c_uint32, C.c_int, dp]
        L.oracle_run.restype = C.c_int
        L.oracle_run.argtypes = [vp, C.POINTER(_Params), C.c_int, dp, dp, vp, dp, C.POINTER(_Stats), vp, vp, vp]
        _lib = L
    return _lib


# ------------------------------------------------------------------ scalar building blocks (pins)
def philox4x32_10(key, ctr):
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(k, c, o)
    return [int(v) for v in o]


def flux_bracket(S):
    return lib().oracle_flux_bracket(float(S))


def flux(S, c, n, r):
    return lib().oracle_flux(float(S), float(c), float(n), float(r))


def position_cdf(t, S):
    return lib().oracle_position_cdf(float(t), float(S))


def position_inv(u, S):
    return lib().oracle_position_inv(float(u), float(S))


def vn_cdf(x, s):
    return lib().oracle_vn_cdf(float(x), float(s))


def vn_inv(u, s):
    return lib().oracle_vn_inv(float(u), float(s))


def vn_unweighted_inv(u, s):
    return lib().oracle_vn_unweighted_inv(float(u), float(s))


def rotation(V):
    v = (C.c_double * 3)(*[float(a) for a in V])
    r = (C.c_double * 9)()
    lib().oracle_rotation(v, r)
    return np.array(list(r)).reshape(3, 3)


# ------------------------------------------------------------------ mesh + runs
@dataclass
class Result:
    force: np.ndarray
    torque: np.ndarray
    facet_momentum: np.ndarray | None
    force_sq: np.ndarray
    hits: int
    segments: int
    escaped: int
    truncated: int
    hash: np.ndarray | None
    bounces: np.ndarray | None
    first_facet: np.ndarray | None

    def force_stderr(self, count: int) -> np.ndarray:
        """Standard error of the total force of this slice (O14)."""
        var = np.maximum(self.force_sq - self.force ** 2 / max(count, 1), 0.0)
        return np.sqrt(var * count / max(count - 1, 1))


class OracleMesh:
    def __init__(self, vertices, indices, flags=None):
        self.v = np.ascontiguousarray(vertices, dtype=np.float32)
        self.idx = np.ascontiguousarray(indices, dtype=np.int32)
        self.flags = None if flags is None else np.ascontiguousarray(flags, dtype=np.uint8)
        self.nt = int(self.idx.shape[0])
        self._h = lib().oracle_mesh_create(self.v.ctypes.data, self.v.shape[0], self.idx.ctypes.data, self.nt,
                                           None if self.flags is None else self.flags.ctypes.data)
        if not self._h:
            raise ValueError("oracle_mesh_create failed")

    def __del__(self):
        try:
            if getattr(self, "_h", None):
                lib().oracle_mesh_destroy(self._h)
                self._h = None
        except Exception:
            pass

    def set_surface(self, T_W=None, sigma=None):
        """Per-facet wall temperature and accommodation (A23); None = the run's scalar."""
        tw = None if T_W is None else np.ascontiguousarray(T_W, dtype=np.float64)
        sg = None if sigma is None else np.ascontiguousarray(sigma, dtype=np.float64)
        assert tw is None or tw.shape == (self.nt,)
        assert sg is None or sg.shape == (self.nt,)
        lib().oracle_mesh_set_surface(self._h, None if tw is None else tw.ctypes.data, None if sg is None else sg.ctypes.data)

    def bounds(self):
        c = (C.c_double * 3)()
        r = C.c_double()
        lib().oracle_mesh_bounds(self._h, c, C.byref(r))
        return np.array(list(c)), r.value

    def closest_hit(self, o, d, f_prev=-1, use_bvh=True):
        o = np.ascontiguousarray(o, dtype=np.float32)
        d = np.ascontiguousarray(d, dtype=np.float32)
        tau = C.c_double()
        f = lib().oracle_closest_hit(self._h, o.ctypes.data, d.ctypes.data, int(f_prev), int(use_bvh), C.byref(tau))
        return int(f), tau.value

    def _params(self, cfg, first=None, count=None, N=None):
        p = _Params()
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
        p.control_volume = int(getattr(cfg, "control_volume", 0))
        return p, (m, x)

    def seed(self, cfg, i, N=None):
        """(x, v, species) of particle i in fp64, before the fp32 rounding of O9."""
        p, keep = self._params(cfg, 0, 0, N)
        x = (C.c_double * 3)()
        v = (C.c_double * 3)()
        s = lib().oracle_seed(self._h, C.byref(p), int(i), x, v)
        return np.array(list(x)), np.array(list(v)), int(s)

    def reflect(self, cfg, facet, v_in, i, k, species=0):
        p, keep = self._params(cfg, 0, 0)
        vin = np.ascontiguousarray(v_in, dtype=np.float32)
        out = (C.c_double * 3)()
        lib().oracle_reflect(self._h, C.byref(p), int(facet), vin.ctypes.data, int(i), int(k), int(species), out)
        return np.array(list(out))

    def run(self, cfg, first=None, count=None, N=None, use_bvh=True, debug=True, facets=True) -> Result:
        p, keep = self._params(cfg, first, count, N)
        cnt = int(p.count)
        force = (C.c_double * 3)()
        torque = (C.c_double * 3)()
        fsq = (C.c_double * 3)()
        st = _Stats()
        fm = np.zeros((self.nt, 3), dtype=np.float64) if facets else None
        hs = np.zeros(cnt, dtype=np.uint64) if debug else None
        nb = np.zeros(cnt, dtype=np.uint32) if debug else None
        ff = np.zeros(cnt, dtype=np.int32) if debug else None
        rc = lib().oracle_run(self._h, C.byref(p), int(use_bvh), force, torque,
                              None if fm is None else fm.ctypes.data, fsq, C.byref(st),
                              None if hs is None else hs.ctypes.data,
                              None if nb is None else nb.ctypes.data,
                              None if ff is None else ff.ctypes.data)
        if rc != 0:
            raise ValueError(f"oracle_run failed ({rc})")
        return Result(np.array(list(force)), np.array(list(torque)), fm, np.array(list(fsq)),
                      int(st.hits), int(st.segments), int(st.escaped), int(st.truncated), hs, nb, ff)
