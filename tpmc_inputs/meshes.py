"""Seeded procedural triangle meshes for the five BASELINE.json configs.

Geometry only (numpy): vertices are float32 [nv,3] (metres, body frame), indices
int32 [nt,3] counter-clockwise seen from outside, flags uint8 [nt] with
bit0 = two-sided facet.  Closed solids are outward oriented and welded so
that shared vertices are bit-identical.  Nothing here knows about gases,
random particle streams or ray tracing.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

TWO_SIDED = 1


@dataclass
class Mesh:
    vertices: np.ndarray  # float32 [nv,3]
    indices: np.ndarray   # int32   [nt,3]
    flags: np.ndarray     # uint8   [nt]
    name: str = "mesh"

    @property
    def nt(self) -> int:
        return int(self.indices.shape[0])

    @property
    def nv(self) -> int:
        return int(self.vertices.shape[0])

    def triangles(self) -> np.ndarray:
        """float64 [nt,3,3] corner coordinates (exact widening of the fp32 data)."""
        return self.vertices.astype(np.float64)[self.indices]

    def transformed(self, R: np.ndarray, shift=(0.0, 0.0, 0.0)) -> "Mesh":
        v = self.vertices.astype(np.float64) @ np.asarray(R, dtype=np.float64).T + np.asarray(shift)
        return Mesh(v.astype(np.float32), self.indices.copy(), self.flags.copy(), self.name + "_xf")


def _finish(verts64: np.ndarray, tris: np.ndarray, flags=None, name="mesh", weld=True) -> Mesh:
    """Weld coincident vertices (after fp32 rounding), drop unreferenced ones."""
    v32 = np.ascontiguousarray(verts64, dtype=np.float32)
    tris = np.asarray(tris, dtype=np.int64)
    if weld:
        # positions that agree to 2^-20 m are the same vertex; keep the first one's fp32 value
        key = np.round(v32.astype(np.float64) * float(1 << 20)).astype(np.int64)
        _, first, inv = np.unique(key, axis=0, return_index=True, return_inverse=True)
        inv = inv.reshape(-1)
        v32 = v32[first]
        tris = inv[tris]
    used = np.zeros(v32.shape[0], dtype=bool)
    used[tris.reshape(-1)] = True
    remap = np.cumsum(used) - 1
    v32 = v32[used]
    tris = remap[tris]
    # drop triangles that welding made degenerate
    ok = (tris[:, 0] != tris[:, 1]) & (tris[:, 1] != tris[:, 2]) & (tris[:, 0] != tris[:, 2])
    tris = tris[ok]
    if flags is None:
        flags = np.zeros(tris.shape[0], dtype=np.uint8)
    else:
        flags = np.asarray(flags, dtype=np.uint8)[ok]
    return Mesh(np.ascontiguousarray(v32), np.ascontiguousarray(tris.astype(np.int32)),
                np.ascontiguousarray(flags), name)


# ----------------------------------------------------------------------------- plate (config 1)
def plate(alpha_deg: float = 30.0, size: float = 1.0) -> Mesh:
    """Unit square, two triangles, two-sided; normal (cos a, sin a, 0)."""
    a = np.deg2rad(alpha_deg)
    ea = np.array([-np.sin(a), np.cos(a), 0.0])
    eb = np.array([0.0, 0.0, 1.0])
    h = 0.5 * size
    c00, c10, c11, c01 = (-h * ea - h * eb, h * ea - h * eb, h * ea + h * eb, -h * ea + h * eb)
    v = np.stack([c00, c10, c11, c01])
    t = np.array([[0, 1, 2], [0, 2, 3]])
    return _finish(v, t, np.full(2, TWO_SIDED, np.uint8), f"plate{alpha_deg:g}", weld=False)


# ----------------------------------------------------------------------------- geodesic sphere
def _icosahedron():
    p = (1.0 + np.sqrt(5.0)) / 2.0
    v = np.array([[-1, p, 0], [1, p, 0], [-1, -p, 0], [1, -p, 0],
                  [0, -1, p], [0, 1, p], [0, -1, -p], [0, 1, -p],
                  [p, 0, -1], [p, 0, 1], [-p, 0, -1], [-p, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
                  [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
                  [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
                  [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]])
    # make every face counter-clockwise seen from outside
    a, b, c = v[f[:, 0]], v[f[:, 1]], v[f[:, 2]]
    flip = np.einsum("ij,ij->i", np.cross(b - a, c - a), a + b + c) < 0
    f[flip] = f[flip][:, [0, 2, 1]]
    return v, f


def geodesic_sphere(freq: int = 32, radius: float = 1.0, radial=None, name=None) -> Mesh:
    """Class-I geodesic sphere: each icosahedron face split into freq^2 triangles
    (20*freq^2 facets; freq=32 is 'subdivision level 5' = 20480).  ``radial`` is an
    optional callable unit-directions[n,3] -> radius[n] (star-shaped displacement)."""
    iv, ifc = _icosahedron()
    f = int(freq)
    ii, jj = np.meshgrid(np.arange(f + 1), np.arange(f + 1), indexing="ij")
    keep = (ii + jj) <= f
    ii, jj = ii[keep], jj[keep]
    lid = -np.ones((f + 1, f + 1), dtype=np.int64)
    lid[ii, jj] = np.arange(ii.size)
    w0 = (f - ii - jj)[:, None] / f
    w1 = ii[:, None] / f
    w2 = jj[:, None] / f
    # local triangles
    ui, uj = np.meshgrid(np.arange(f), np.arange(f), indexing="ij")
    m_up = (ui + uj) <= f - 1
    up = np.stack([lid[ui[m_up], uj[m_up]], lid[ui[m_up] + 1, uj[m_up]], lid[ui[m_up], uj[m_up] + 1]], 1)
    m_dn = (ui + uj) <= f - 2
    dn = np.stack([lid[ui[m_dn] + 1, uj[m_dn]], lid[ui[m_dn] + 1, uj[m_dn] + 1], lid[ui[m_dn], uj[m_dn] + 1]], 1)
    loc = np.concatenate([up, dn], 0)
    verts, tris = [], []
    npf = ii.size
    for k, (a, b, c) in enumerate(ifc):
        p = w0 * iv[a] + w1 * iv[b] + w2 * iv[c]
        p /= np.linalg.norm(p, axis=1, keepdims=True)
        verts.append(p)
        tris.append(loc + k * npf)
    verts = np.concatenate(verts, 0)
    tris = np.concatenate(tris, 0)
    # weld on the unit sphere first so displaced shared vertices stay identical
    key = np.round(verts * float(1 << 24)).astype(np.int64)
    _, first, inv = np.unique(key, axis=0, return_index=True, return_inverse=True)
    inv = inv.reshape(-1)
    verts = verts[first]
    tris = inv[tris]
    r = radius if radial is None else np.asarray(radial(verts), dtype=np.float64)[:, None]
    return _finish(verts * r, tris, name=name or f"geodesic{f}", weld=False)


# ----------------------------------------------------------------------------- cylinder (config 3)
def cylinder(radius: float = 0.5, length: float = 2.0, nseg: int = 256, nbands: int = 3) -> Mesh:
    """Capped right circular cylinder along z: nseg*nbands*2 side + 2*nseg cap facets."""
    th = 2.0 * np.pi * np.arange(nseg) / nseg
    ring = np.stack([radius * np.cos(th), radius * np.sin(th)], 1)
    zs = np.linspace(-0.5 * length, 0.5 * length, nbands + 1)
    verts = [np.concatenate([ring, np.full((nseg, 1), z)], 1) for z in zs]
    verts = np.concatenate(verts + [np.array([[0, 0, zs[0]], [0, 0, zs[-1]]])], 0)
    cb, ct = nseg * (nbands + 1), nseg * (nbands + 1) + 1
    tris = []
    for b in range(nbands):
        for s in range(nseg):
            s1 = (s + 1) % nseg
            a0, a1 = b * nseg + s, b * nseg + s1
            b0, b1 = (b + 1) * nseg + s, (b + 1) * nseg + s1
            tris.append([a0, a1, b1])
            tris.append([a0, b1, b0])
    top = nbands * nseg
    for s in range(nseg):
        s1 = (s + 1) % nseg
        tris.append([cb, s1, s])              # bottom cap, normal -z
        tris.append([ct, top + s, top + s1])  # top cap, normal +z
    return _finish(verts, np.array(tris), name=f"cylinder{nseg}x{nbands}", weld=False)


# ----------------------------------------------------------------------------- gridded patches / boxes
def _patch(origin, eu, ev, nu, nv, rng=None, jitter=0.0, hole=None):
    """Planar grid patch, normal eu x ev.  Interior grid points may be jittered in-plane;
    points on the outer boundary or on the hole boundary stay put (they are shared)."""
    origin, eu, ev = (np.asarray(x, dtype=np.float64) for x in (origin, eu, ev))
    ii, jj = np.meshgrid(np.arange(nu + 1), np.arange(nv + 1), indexing="ij")
    fu = ii / nu
    fv = jj / nv
    if rng is not None and jitter > 0.0:
        free = (ii > 0) & (ii < nu) & (jj > 0) & (jj < nv)
        if hole is not None:
            i0, i1, j0, j1 = hole
            free &= ~((ii >= i0) & (ii <= i1) & (jj >= j0) & (jj <= j1))
        du = rng.uniform(-jitter, jitter, size=ii.shape) / nu
        dv = rng.uniform(-jitter, jitter, size=ii.shape) / nv
        fu = fu + np.where(free, du, 0.0)
        fv = fv + np.where(free, dv, 0.0)
    p = origin + fu[..., None] * eu + fv[..., None] * ev
    vid = (ii * (nv + 1) + jj)
    ci, cj = np.meshgrid(np.arange(nu), np.arange(nv), indexing="ij")
    keep = np.ones(ci.shape, dtype=bool)
    if hole is not None:
        i0, i1, j0, j1 = hole
        keep = ~((ci >= i0) & (ci < i1) & (cj >= j0) & (cj < j1))
    ci, cj = ci[keep], cj[keep]
    a = vid[ci, cj]
    b = vid[ci + 1, cj]
    c = vid[ci + 1, cj + 1]
    d = vid[ci, cj + 1]
    tris = np.concatenate([np.stack([a, b, c], 1), np.stack([a, c, d], 1)], 0)
    return p.reshape(-1, 3), tris


def _box_patches(center, axes, half, h, rng=None, jitter=0.0, top_hole=None):
    """Six outward-facing gridded faces of an oriented box. axes: 3x3 with unit columns."""
    c = np.asarray(center, dtype=np.float64)
    X, Y, Z = (np.asarray(axes, dtype=np.float64)[:, k] for k in range(3))
    a, b, cc = half
    na, nb, nc = (max(1, int(round(2 * s / h))) for s in (a, b, cc))
    out = []
    out.append(_patch(c + a * X - b * Y - cc * Z, 2 * b * Y, 2 * cc * Z, nb, nc, rng, jitter))   # +X
    out.append(_patch(c - a * X - b * Y - cc * Z, 2 * cc * Z, 2 * b * Y, nc, nb, rng, jitter))   # -X
    out.append(_patch(c + b * Y - a * X - cc * Z, 2 * cc * Z, 2 * a * X, nc, na, rng, jitter))   # +Y
    out.append(_patch(c - b * Y - a * X - cc * Z, 2 * a * X, 2 * cc * Z, na, nc, rng, jitter))   # -Y
    out.append(_patch(c + cc * Z - a * X - b * Y, 2 * a * X, 2 * b * Y, na, nb, rng, jitter, top_hole))  # +Z
    out.append(_patch(c - cc * Z - a * X - b * Y, 2 * b * Y, 2 * a * X, nb, na, rng, jitter))   # -Z
    return out


def _merge(patches):
    verts, tris, off = [], [], 0
    for p, t in patches:
        verts.append(p)
        tris.append(t + off)
        off += p.shape[0]
    return np.concatenate(verts, 0), np.concatenate(tris, 0)


def box(center=(0, 0, 0), half=(0.5, 0.5, 0.5), h=0.25, axes=None, seed=None, jitter=0.0) -> Mesh:
    rng = None if seed is None else np.random.default_rng(seed)
    axes = np.eye(3) if axes is None else np.asarray(axes, dtype=np.float64)
    v, t = _merge(_box_patches(center, axes, half, h, rng, jitter))
    return _finish(v, t, name="box")


# ----------------------------------------------------------------------------- satellite (config 4)
def satellite(seed: int = 4, h: float = 1.0 / 30.0, jitter: float = 0.25) -> Mesh:
    """Concave synthetic satellite: 1x1x2 m bus with a 0.6x0.6x0.5 m open pocket in its +z
    face, and two 4x1x0.02 m slab panels along +-y canted 45 deg about y.  All parts are
    closed outward-oriented solids; faces are gridded at cell size h (default ~5e4 facets)
    with seeded in-plane jitter of interior grid points."""
    rng = np.random.default_rng(seed)
    patches = []
    a, b, c = 0.5, 0.5, 1.0
    na, nb = int(round(2 * a / h)), int(round(2 * b / h))
    hw = int(round(0.3 / h))            # pocket half-width in cells
    i0, i1 = na // 2 - hw, na // 2 + hw
    j0, j1 = nb // 2 - hw, nb // 2 + hw
    patches += _box_patches((0, 0, 0), np.eye(3), (a, b, c), h, rng, jitter, top_hole=(i0, i1, j0, j1))
    x0, x1 = -a + 2 * a * i0 / na, -a + 2 * a * i1 / na
    y0, y1 = -b + 2 * b * j0 / nb, -b + 2 * b * j1 / nb
    depth = 0.5
    zt, zf = c, c - depth
    nd = max(1, int(round(depth / h)))
    nx, ny = i1 - i0, j1 - j0
    X, Y, Z = np.eye(3)
    patches.append(_patch((x0, y0, zf), (y1 - y0) * Y, (zt - zf) * Z, ny, nd, rng, jitter))   # wall facing +X
    patches.append(_patch((x1, y0, zf), (zt - zf) * Z, (y1 - y0) * Y, nd, ny, rng, jitter))   # wall facing -X
    patches.append(_patch((x0, y0, zf), (zt - zf) * Z, (x1 - x0) * X, nd, nx, rng, jitter))   # wall facing +Y
    patches.append(_patch((x0, y1, zf), (x1 - x0) * X, (zt - zf) * Z, nx, nd, rng, jitter))   # wall facing -Y
    patches.append(_patch((x0, y0, zf), (x1 - x0) * X, (y1 - y0) * Y, nx, ny, rng, jitter))   # floor facing +Z
    s = np.sqrt(0.5)
    # panel axes (columns): long side along y, width along (s,0,s), thickness along (s,0,-s)
    pax = np.array([[0.0, s, s], [1.0, 0.0, 0.0], [0.0, s, -s]])
    for sign in (+1.0, -1.0):
        patches += _box_patches((0.0, sign * (b + 0.1 + 2.0), 0.0), pax, (2.0, 0.5, 0.01), h, rng, jitter)
    v, t = _merge(patches)
    return _finish(v, t, name=f"satellite_s{seed}")


# ----------------------------------------------------------------------------- gradient noise
class _GradientNoise:
    """Seeded lattice gradient noise (my own restatement of the classic improved-noise idea)."""

    def __init__(self, seed: int):
        rng = np.random.default_rng(seed)
        self.perm = np.concatenate([rng.permutation(256)] * 2).astype(np.int64)
        g = rng.normal(size=(256, 3))
        self.grad = g / np.linalg.norm(g, axis=1, keepdims=True)

    def __call__(self, p: np.ndarray) -> np.ndarray:
        pi = np.floor(p).astype(np.int64)
        pf = p - pi
        w = pf * pf * pf * (pf * (pf * 6.0 - 15.0) + 10.0)
        out = np.zeros(p.shape[0])
        for dx in (0, 1):
            for dy in (0, 1):
                for dz in (0, 1):
                    hx = self.perm[(pi[:, 0] + dx) & 255]
                    hy = self.perm[(hx + pi[:, 1] + dy) & 255]
                    hz = self.perm[(hy + pi[:, 2] + dz) & 255]
                    g = self.grad[hz]
                    d = pf - np.array([dx, dy, dz], dtype=np.float64)
                    wx = w[:, 0] if dx else 1.0 - w[:, 0]
                    wy = w[:, 1] if dy else 1.0 - w[:, 1]
                    wz = w[:, 2] if dz else 1.0 - w[:, 2]
                    out += wx * wy * wz * np.einsum("ij,ij->i", g, d)
        return out


def _fbm(noise, p, octaves=4, base=2.0):
    tot, amp, f, norm = np.zeros(p.shape[0]), 1.0, base, 0.0
    for _ in range(octaves):
        tot += amp * noise(p * f + 17.0)
        norm += amp
        amp *= 0.5
        f *= 2.0
    return tot / norm


# ----------------------------------------------------------------------------- large body (config 5)
def large_body(seed: int = 5, freq: int = 224, amplitude: float = 0.05,
               panel_len: float = 1.0, panel_w: float = 0.5, panel_h: float = 0.02) -> Mesh:
    """Geodesic sphere (20*freq^2 facets, ~1.0e6 at freq=224) displaced radially by seeded
    4-octave gradient noise (star-shaped, +-~amplitude), plus 6 slab panels along +-x,+-y,+-z
    whose bases are embedded in the body."""
    noise = _GradientNoise(seed)

    def radial(d):
        return 1.0 + 2.0 * amplitude * _fbm(noise, d)

    body = geodesic_sphere(freq, 1.0, radial, name="body")
    rng = np.random.default_rng(seed + 1)
    patches = []
    r0 = 0.9
    for k in range(3):
        for sign in (+1.0, -1.0):
            ax = np.zeros((3, 3))
            ax[k, 0] = sign                       # radial (long) axis
            ax[(k + 1) % 3, 1] = 1.0              # width axis
            ax[:, 2] = np.cross(ax[:, 0], ax[:, 1])
            ctr = ax[:, 0] * (r0 + 0.5 * panel_len)
            patches += _box_patches(ctr, ax, (0.5 * panel_len, 0.5 * panel_w, 0.5 * panel_h),
                                    panel_h, rng, 0.2)
    pv, pt = _merge(patches)
    panels = _finish(pv, pt, name="panels")
    v = np.concatenate([body.vertices, panels.vertices], 0)
    t = np.concatenate([body.indices, panels.indices + body.nv], 0)
    return Mesh(np.ascontiguousarray(v), np.ascontiguousarray(t.astype(np.int32)),
                np.zeros(t.shape[0], np.uint8), f"large_body_s{seed}_f{freq}")


# ----------------------------------------------------------------------------- extras for tests
def hemisphere_shell(freq: int = 16, radius: float = 1.0) -> Mesh:
    """Open two-sided hemispherical shell, concave side towards +x."""
    s = geodesic_sphere(freq, radius)
    cen = s.vertices.astype(np.float64)[s.indices].mean(1)
    keep = cen[:, 0] < 0.0
    m = _finish(s.vertices.astype(np.float64), s.indices[keep], np.full(int(keep.sum()), TWO_SIDED, np.uint8),
                f"hemishell{freq}", weld=False)
    return m


def random_blob(seed: int = 0, freq: int = 2, amplitude: float = 0.15) -> Mesh:
    """Small closed star-shaped test mesh (20*freq^2 facets)."""
    noise = _GradientNoise(seed)
    return geodesic_sphere(freq, 1.0, lambda d: 1.0 + 2.0 * amplitude * _fbm(noise, d, 2, 1.5),
                           name=f"blob{seed}")


def lobster_pot(hole: float = 0.5, h: float = 0.25) -> Mesh:
    """Hollow unit cube of two-sided sheets with a square opening of side `hole` in its +x face: a particle that
    enters bounces many times before it finds the opening again (long reflection chains, a full reflected-ray
    region with a small wave)."""
    n = max(2, int(round(1.0 / h)))
    k = max(1, int(round(hole / 2.0 * n)))
    X, Y, Z = np.eye(3)
    c = np.zeros(3)
    a = 0.5
    patches = [
        _patch(c + a * X - a * Y - a * Z, 2 * a * Y, 2 * a * Z, n, n, hole=(n // 2 - k, n // 2 + k, n // 2 - k, n // 2 + k)),
        _patch(c - a * X - a * Y - a * Z, 2 * a * Z, 2 * a * Y, n, n),
        _patch(c + a * Y - a * X - a * Z, 2 * a * Z, 2 * a * X, n, n),
        _patch(c - a * Y - a * X - a * Z, 2 * a * X, 2 * a * Z, n, n),
        _patch(c + a * Z - a * X - a * Y, 2 * a * X, 2 * a * Y, n, n),
        _patch(c - a * Z - a * X - a * Y, 2 * a * Y, 2 * a * X, n, n),
    ]
    v, t = _merge(patches)
    return _finish(v, t, np.full(t.shape[0], TWO_SIDED, np.uint8), name="lobster_pot")


def stacked_duplicates(copies: int = 6) -> Mesh:
    """A unit square (two triangles, normal +x) stored `copies` times over: every hit is a tie between `copies`
    coincident facets (rule A12: the smallest facet index wins) -- more candidates than a short list holds."""
    v = np.array([[0, -0.5, -0.5], [0, 0.5, -0.5], [0, 0.5, 0.5], [0, -0.5, 0.5]], dtype=np.float64)
    t = np.array([[0, 1, 2], [0, 2, 3]] * copies)
    return _finish(v, t, np.full(t.shape[0], TWO_SIDED, np.uint8), name=f"stack{copies}", weld=False)


def deep_chain(levels: int = 21, cluster: int = 64) -> Mesh:
    """Parallel two-sided unit squares normal to x at x = 2^-i (i < levels) plus `cluster` more packed below
    2^-(levels+1): centroid Morton codes with one leading bit each, so a radix-tree hierarchy over them is a chain
    about levels + log2(cluster) deep, and a ray along +x overlaps every box of it (deeper than a short
    traversal stack)."""
    xs = [2.0 ** -i for i in range(levels)] + [2.0 ** -(levels + 1) * (j + 1) / (cluster + 1) for j in range(cluster)]
    verts, tris = [], []
    for x in xs:
        o = len(verts)
        verts += [[x, -0.5, -0.5], [x, 0.5, -0.5], [x, 0.5, 0.5], [x, -0.5, 0.5]]
        tris += [[o, o + 1, o + 2], [o, o + 2, o + 3]]
    t = np.array(tris)
    return _finish(np.array(verts, dtype=np.float64), t, np.full(t.shape[0], TWO_SIDED, np.uint8), name="deep_chain", weld=False)
