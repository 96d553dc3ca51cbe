"""Parity of the CUDA path (through the C ABI) with the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): integer/index work bit-exact -- Philox
stream, closest-hit facet and, since both sides evaluate O10 in the same fp64 order, tau;
per-particle hit-facet sequences equal on >= 99.99 % of particles; total force within 1e-4
relative; per-facet momentum within 1e-3 relative on facets untouched by a mismatched particle
(reading A18); seeding within 1e-12 relative before the fp32 rounding."""
import numpy as np
import pytest

import tpmc_inputs as ti

pytestmark = pytest.mark.gpu

SEQ_AGREE = 0.9999     # >= 99.99 % identical hit sequences
FORCE_RTOL = 1e-4
FACET_RTOL = 1e-3
SEED_RTOL = 1e-12


@pytest.fixture(scope="module")
def T():
    import paper_1312_3691_b200 as t
    return t


@pytest.fixture(scope="module")
def O():
    import oracle
    return oracle


_mesh_cache = {}


def meshes(T, O, cfg):
    key = cfg.name + cfg.mesh().name
    if key not in _mesh_cache:
        m = cfg.mesh()
        _mesh_cache[key] = (T.Mesh(m.vertices, m.indices, m.flags), O.OracleMesh(m.vertices, m.indices, m.flags))
    return _mesh_cache[key]


def check_conservation(st, count, exact=False):
    """tpmc_stats counts every event where it happens (include/tpmc.h): a particle lost or duplicated between the
    pre-cull lists, the two queue regions, the hit list, the overflow lists and the straggler kernel breaks these."""
    retired = (st["truncated"] + st["ret_precull_a"] + st["ret_precull_b"] + st["ret_seed"] + st["ret_trace"]
               + st["ret_resolve"] + st["ret_horizon"] + st["ret_finish"])
    assert retired == count, (retired, count, st)
    assert st["escaped"] == count - st["truncated"]
    assert st["segments"] == count + st["hits"] - st["truncated"], st
    assert st["culled"] == st["ret_precull_a"] + st["ret_precull_b"] + st["ret_seed"]
    assert st["queued_primaries"] == count - st["culled"]
    if exact:
        assert st["traced_rays"] == 0 and st["overflow_rays"] == st["queued_primaries"]
    else:
        assert st["traced_rays"] + st["final_stragglers"] == st["queued_primaries"] + st["queued_reflected"], st


def compare_run(T, O, cfg, first, count, use_bvh=True, pair=None, **run_kw):
    gm, om = pair if pair is not None else meshes(T, O, cfg)
    g = gm.run(cfg, first=first, count=count, debug=True, **run_kw)
    check_conservation(g.stats, count, exact=bool(run_kw.get("flags", 0) & T.TPMC_FLAG_EXACT_TRACE))
    o = om.run(cfg, first=first, count=count, use_bvh=use_bvh)
    gh = g.hash.cpu().numpy().view(np.uint64)
    same = gh == o.hash
    frac = same.mean() if count else 1.0
    assert frac >= SEQ_AGREE, f"{cfg.label}: only {frac:.6f} of hit sequences agree"
    gb = g.bounces.cpu().numpy().astype(np.uint32)
    assert np.array_equal(gb[same], o.bounces[same])
    assert np.array_equal(g.first_facet.cpu().numpy()[same], o.first_facet[same])
    F = g.force.cpu().numpy()
    assert np.linalg.norm(F - o.force) <= FORCE_RTOL * np.linalg.norm(o.force), (cfg.label, F, o.force)
    Tq = g.torque.cpu().numpy()
    assert np.linalg.norm(Tq - o.torque) <= FORCE_RTOL * max(np.linalg.norm(o.torque), 1e-3 * np.linalg.norm(o.force))
    fm = g.facet_momentum.cpu().numpy()
    if same.all():
        assert g.stats["hits"] == o.hits and g.stats["segments"] == o.segments
        assert g.stats["truncated"] == o.truncated and g.stats["escaped"] == o.escaped
        nrm = np.linalg.norm(o.facet_momentum, axis=1)
        err = np.linalg.norm(fm - o.facet_momentum, axis=1)
        assert np.all(err <= FACET_RTOL * nrm + 1e-300), (cfg.label, float((err / np.maximum(nrm, 1e-300)).max()))
        assert np.array_equal(nrm == 0, np.linalg.norm(fm, axis=1) == 0)       # untouched facets stay exactly zero
    # a7: F = sum_f P_f, to the rounding of an fp64 sum of these terms (1e-12 of sum |P_f|: a component that
    # cancels to ~0, like the side force of an axisymmetric body, has no relative accuracy of its own)
    assert np.all(np.abs(fm.sum(0) - F) <= 1e-12 * np.abs(fm).sum(0) + 1e-30)
    return g, o, frac


# ------------------------------------------------------------------ a2: seeding
@pytest.mark.parametrize("name,idx,first,N", [("C1", 0, 0, 100_000), ("C2", 0, 123_456, 10_000_000),
                                               ("C3", 1, 99_990_000, 100_000_000),
                                               ("C5", 7, 6_000_000_000, 10_000_000_000)])
def test_seed_parity(T, O, name, idx, first, N):
    cfg = ti.config(name)[idx]
    if name == "C5":
        cfg = cfg.with_(mesh_fn=lambda: ti.large_body(5, 16))
        cfg._mesh_cache = []
    gm, om = meshes(T, O, cfg)
    cnt = 3000
    x, v, s = gm.seed(cfg, first=first, count=cnt, N=N)
    x, v, s = x.cpu().numpy(), v.cpu().numpy(), s.cpu().numpy()
    xs = np.abs(x).max()
    for j in range(cnt):
        xo, vo, so = om.seed(cfg, first + j, N=N)
        assert so == s[j]
        assert np.abs(x[j] - xo).max() <= SEED_RTOL * xs
        assert np.abs(v[j] - vo).max() <= SEED_RTOL * np.abs(vo).max() + 1e-9
    info = gm.info()
    ctr, Rb = om.bounds()
    assert np.array_equal(info["centre"], ctr) and info["bounding_radius"] == Rb     # O1 bit-exact


def test_seed_equilibrium_and_tiny_speed_ratio(T, O):
    base = ti.RunConfig("eq", lambda: ti.box(h=0.5), T_inf=500.0, T_W=500.0, V=(0.0, 0.0, 0.0), N=5000)
    for V in ((0.0, 0.0, 0.0), (0.0, 1e-3, 0.0), (0.02, 0.0, 0.01)):
        cfg = base.with_(V=V)
        gm, om = meshes(T, O, cfg)
        x, v, s = (a.cpu().numpy() for a in gm.seed(cfg))
        for j in range(0, cfg.N, 7):
            xo, vo, _ = om.seed(cfg, j)
            assert np.abs(x[j] - xo).max() <= 1e-11 and np.abs(v[j] - vo).max() <= 1e-9


# ------------------------------------------------------------------ a0: LBVH
@pytest.mark.parametrize("mesh_fn", [lambda: ti.plate(30.0), lambda: ti.box(h=1.0), lambda: ti.geodesic_sphere(8),
                                      lambda: ti.satellite(4, 0.125), lambda: ti.cylinder(0.5, 2.0, 256, 3),
                                      lambda: ti.large_body(5, 24)])
def test_lbvh_topology_and_boxes(T, mesh_fn):
    m = mesh_fn()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    nodes, leaf = gm.copy_bvh()
    nt = m.nt
    assert sorted(leaf.tolist()) == list(range(nt))                     # every facet in exactly one slot
    kids = nodes[:, 12:14].copy().view(np.int32)
    n_int = max(nt - 1, 1)
    assert nodes.shape[0] == n_int
    tri = m.vertices[m.indices[leaf]]                                   # [slot,3,3] fp32
    tlo, thi = tri.min(1), tri.max(1)
    seen_leaf = np.zeros(nt, int)
    seen_node = np.zeros(n_int, int)
    seen_node[0] = 1

    def child_box(i, k):
        b = nodes[i, 6 * k:6 * k + 6]
        return b[:3], b[3:]

    # bottom-up exact boxes
    order, stack = [], [0]
    while stack:
        i = stack.pop()
        order.append(i)
        for k in range(2):
            c = kids[i, k]
            if c >= 0:
                seen_node[c] += 1
                stack.append(c)
            elif nt > 1 or k == 0:
                seen_leaf[~c] += 1
    assert np.all(seen_leaf == 1) and np.all(seen_node == 1)           # a tree: each leaf/node reached once
    lo = np.zeros((n_int, 3), np.float32)
    hi = np.zeros((n_int, 3), np.float32)
    for i in reversed(order):
        l, h = [], []
        for k in range(2):
            c = kids[i, k]
            if nt == 1 and k == 1:
                continue
            bl, bh = (lo[c], hi[c]) if c >= 0 else (tlo[~c], thi[~c])
            cl, ch = child_box(i, k)
            assert np.array_equal(cl, bl) and np.array_equal(ch, bh)   # stored child box = exact fp32 bounds
            l.append(bl); h.append(bh)
        lo[i], hi[i] = np.min(l, 0), np.max(h, 0)
    info = gm.info()
    assert np.array_equal(lo[0], info["aabb_lo"].astype(np.float32)) or nt == 1
    assert info["build_ms"] > 0


@pytest.mark.parametrize("mesh_fn", [lambda: ti.plate(30.0), lambda: ti.box(h=1.0), lambda: ti.meshes.Mesh(np.float32([[0, 0, 0], [1, 0, 0], [0, 1, 0]]), np.int32([[0, 1, 2]]), np.zeros(1, np.uint8), "one"),
                                      lambda: ti.satellite(4, 0.125), lambda: ti.deep_chain(), lambda: ti.large_body(5, 24)])
def test_wide_hierarchy_topology_and_boxes(T, mesh_fn):
    """The 4-ary hierarchy the wavefront traversal walks (tpmc_mesh_copy_wide): a tree over the same sorted facets as the
    radix tree, every facet in exactly one leaf, every node reached once from the root, and every stored child box --
    16-bit grid coordinates, decoded as the traversal decodes them -- contains the exact fp32 bounds of everything below it."""
    m = mesh_fn()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    _, leaf = gm.copy_bvh()
    wn, grid = gm.copy_wide()
    nt, nw = m.nt, wn.shape[0]
    assert 1 <= nw <= max(nt - 1, 1)
    refs = wn[:, 12:16].view(np.int32)
    q = wn[:, :12].reshape(nw, 4, 3)
    qlo, qhi = (q & 0xFFFF).astype(np.float64), (q >> 16).astype(np.float64)
    org, step = grid[:3].astype(np.float64), grid[3:].astype(np.float64)
    blo, bhi = org + qlo * step, org + qhi * step                       # decoded boxes [node, child, axis]
    empty = (qlo == 65535).all(2) & (qhi == 0).all(2)
    tri = m.vertices[m.indices[leaf]].astype(np.float64)                # [slot,3,3]
    tlo, thi = tri.min(1), tri.max(1)
    seen_leaf, seen_node = np.zeros(nt, int), np.zeros(nw, int)
    seen_node[0] = 1
    order, stack = [], [0]
    while stack:
        i = stack.pop()
        order.append(i)
        assert not empty[i, 0]
        for k in range(4):
            if empty[i, k]:
                assert refs[i, k] == refs[i, 0]                           # an empty slot repeats the first ref
                continue
            c = refs[i, k]
            if c >= 0:
                assert c < nw and c > i                                   # breadth-first numbering
                seen_node[c] += 1
                stack.append(c)
            else:
                seen_leaf[~c] += 1
    assert np.all(seen_leaf == 1) and np.all(seen_node == 1)
    lo, hi = np.zeros((nw, 3)), np.zeros((nw, 3))
    tol = 1e-9 * np.abs(grid[:3]).max() + 1e-12                           # the fp64 quotient of the quantisation (see k_compact_wide)
    for i in reversed(order):
        l, h = [], []
        for k in range(4):
            if empty[i, k]:
                continue
            c = refs[i, k]
            el, eh = (lo[c], hi[c]) if c >= 0 else (tlo[~c], thi[~c])
            assert np.all(blo[i, k] <= el + tol) and np.all(bhi[i, k] >= eh - tol)
            assert np.all(el - blo[i, k] <= 1.001 * step + tol) and np.all(bhi[i, k] - eh <= 1.001 * step + tol)   # and is tight: < 1 step
            l.append(el); h.append(eh)
        lo[i], hi[i] = np.min(l, 0), np.max(h, 0)
    gm.close()


def test_mesh_create_from_device_tensors_and_errors(T):
    import torch
    m = ti.geodesic_sphere(4)
    a = T.Mesh(m.vertices, m.indices, m.flags)
    b = T.Mesh(torch.tensor(m.vertices).cuda(), torch.tensor(m.indices).cuda(), torch.tensor(m.flags).cuda())
    na, la = a.copy_bvh()
    nb, lb = b.copy_bvh()
    assert np.array_equal(na.view(np.int32), nb.view(np.int32)) and np.array_equal(la, lb)
    bad = m.indices.copy()
    bad[3, 1] = m.nv + 5
    with pytest.raises(T.TpmcError):
        T.Mesh(m.vertices, bad)
    with pytest.raises(T.TpmcError):
        T.Mesh(m.vertices * np.float32("nan"), m.indices)
    cfg = ti.RunConfig("bad", None)
    for kw in (dict(T_inf=-1.0), dict(accommodation=1.5), dict(cv_radius_factor=0.5), dict(max_bounces=0),
               dict(x=(0.5,)), dict(N=10, seed=1)):
        c = cfg.with_(**kw)
        if "N" in kw:
            with pytest.raises(T.TpmcError):
                a.run(c, first=5, count=6)
        else:
            with pytest.raises(T.TpmcError):
                a.run(c)
    good = ti.config("C2")[0].with_(N=1000)
    for flags in (0x100, T.TPMC_FLAG_ALIGN_OFF | T.TPMC_FLAG_ALIGN_ON):      # unknown bit; contradictory pair
        with pytest.raises(T.TpmcError):
            a.run(good, flags=flags)
    a.run(good, flags=T.TPMC_FLAG_SERIAL_SEED | T.TPMC_FLAG_NO_AGGREGATION)  # every defined bit is accepted


def test_mesh_without_escape_horizons_and_late_build(T):
    """tpmc_mesh_create_ex(TPMC_MESH_NO_HORIZON): no horizon pass at creation, runs trace every re-emitted ray and give
    the same hit sequences; tpmc_mesh_build_horizon adds the same horizons tpmc_mesh_create would have built."""
    import torch
    cfg = ti.config("C4")[3].with_(N=2_000_000)
    m = cfg.mesh()
    ref_mesh = T.Mesh(m.vertices, m.indices, m.flags)
    lean = T.tpmc_mesh_create_ex(m.vertices, m.indices, m.flags, mesh_flags=T.TPMC_MESH_NO_HORIZON)
    assert lean.info()["horizon_ms"] == 0.0 and ref_mesh.info()["horizon_ms"] > 0.0
    with pytest.raises(T.TpmcError):
        lean.copy_horizon()
    ref = ref_mesh.run(cfg, debug=True)
    a = lean.run(cfg, debug=True)
    check_conservation(a.stats, cfg.N)
    assert a.stats["ret_horizon"] == 0 and ref.stats["ret_horizon"] > 0
    assert a.stats["hits"] == ref.stats["hits"] and torch.equal(a.hash, ref.hash) and torch.equal(a.bounces, ref.bounces)
    assert np.linalg.norm((a.force - ref.force).cpu().numpy()) <= 1e-12 * np.linalg.norm(ref.force.cpu().numpy())
    lean.build_horizon()
    lean.build_horizon()                                                     # a second call is a no-op
    assert lean.info()["horizon_ms"] > 0.0
    assert np.array_equal(lean.copy_horizon(), ref_mesh.copy_horizon())
    b = lean.run(cfg, debug=True)
    assert b.stats["ret_horizon"] == ref.stats["ret_horizon"] and torch.equal(b.hash, ref.hash)
    with pytest.raises(T.TpmcError):
        T.tpmc_mesh_create_ex(m.vertices, m.indices, m.flags, mesh_flags=0x80)   # unknown option bit
    lean.close()
    ref_mesh.close()


# ------------------------------------------------------------------ a3: closest hit, bit-exact
def crafted_rays(m, om, rng, n_random=400):
    V = m.vertices.astype(np.float64)
    tri = m.triangles()
    ctr, Rb = om.bounds()
    tg = np.concatenate([V[:300], 0.5 * (tri[:300, 0] + tri[:300, 1]), 0.5 * (tri[:300, 1] + tri[:300, 2]),
                         tri[:300].mean(1), ctr + rng.normal(size=(n_random, 3)) * Rb * 0.6])
    dirs = rng.normal(size=tg.shape)
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    o = (ctr + 2.5 * Rb * dirs).astype(np.float32)
    d = (tg - o.astype(np.float64)).astype(np.float32)
    # axis-parallel rays: zero direction components
    cen = tri.mean(1)[:60]
    for ax in range(3):
        oo = cen.copy(); oo[:, ax] += 3 * Rb
        dd = np.zeros_like(cen); dd[:, ax] = -1.0
        o = np.concatenate([o, oo.astype(np.float32)]); d = np.concatenate([d, dd.astype(np.float32)])
    # rays starting ON the surface (secondary-ray situation), leaving and grazing
    st = tri.mean(1)[:200]
    dd = rng.normal(size=st.shape)
    o = np.concatenate([o, st.astype(np.float32)]); d = np.concatenate([d, dd.astype(np.float32)])
    fprev = np.full(o.shape[0], -1, np.int32)
    fprev[-st.shape[0]:] = np.arange(st.shape[0])
    return o, d, fprev


@pytest.mark.parametrize("mesh_fn,bvh", [(lambda: ti.plate(30.0), False), (lambda: ti.box(h=0.5), False),
                                          (lambda: ti.random_blob(1, 3), False), (lambda: ti.satellite(4, 0.125), True),
                                          (lambda: ti.geodesic_sphere(32), True), (lambda: ti.large_body(5, 40), True)])
def test_trace_parity_bit_exact(T, O, mesh_fn, bvh):
    m = mesh_fn()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    om = O.OracleMesh(m.vertices, m.indices, m.flags)
    o, d, fprev = crafted_rays(m, om, np.random.default_rng(5))
    facet, tau = gm.trace(o, d, fprev)
    facet, tau = facet.cpu().numpy(), tau.cpu().numpy()
    nh = 0
    for r in range(o.shape[0]):
        fo, to = om.closest_hit(o[r], d[r], int(fprev[r]), use_bvh=bvh)
        assert facet[r] == fo, (r, facet[r], fo)
        if fo >= 0:
            assert tau[r] == to                                           # same fp64 operations, same bits
            nh += 1
        else:
            assert np.isinf(tau[r])
    assert nh > 100
    # the same rays on the hierarchy refitted in a stream frame (what tpmc_run walks at oblique attitudes): the
    # boxes differ, the answers must not
    for V in ((-3000.0, 5200.0, -4100.0), (100.0, -7000.0, 2500.0)):
        fa, ta = gm.trace(o, d, fprev, align_V=V)
        assert np.array_equal(fa.cpu().numpy(), facet) and np.array_equal(ta.cpu().numpy(), tau)


def test_trace_tie_and_sidedness_rules(T):
    pl = ti.plate(0.0)
    gm = T.Mesh(pl.vertices, pl.indices, pl.flags)
    o = np.float32([[2, 0, 0], [2, 0, 0], [-2, 0.1, 0.2]])
    d = np.float32([[-1, 0, 0], [-1, 0, 0], [1, 0, 0]])
    f, tau = gm.trace(o, d, np.int32([-1, 0, -1]))
    f = f.cpu().numpy()
    assert f[0] == 0 and f[1] == 1 and f[2] >= 0           # A12 tie -> smallest index; A11 source excluded; two-sided
    bx = ti.box(h=1.0)
    gb = T.Mesh(bx.vertices, bx.indices, bx.flags)
    f, _ = gb.trace(np.float32([[0, 0, 0]]), np.float32([[1, 0.1, 0.2]]))
    assert f.cpu().numpy()[0] == -1                         # one-sided facets are invisible from behind
    one = T.Mesh(np.float32([[0, 0, 0], [1, 0, 0], [0, 1, 0]]), np.int32([[0, 1, 2]]))   # single-triangle mesh
    f, tau = one.trace(np.float32([[0.2, 0.2, 1], [0.2, 0.2, -1], [2, 2, 1]]), np.float32([[0, 0, -1], [0, 0, 1], [0, 0, -1]]))
    assert f.cpu().numpy().tolist() == [0, -1, -1] and tau.cpu().numpy()[0] == 1.0


def test_trace_every_ray_hits_with_the_queue_filled_to_capacity(T, O):
    """The hit list holds one entry per ray that ends with a candidate facet and is sized from the queue capacity plus a
    fixed slack (run.cu: ensure_scratch, kHitSlack).  Worst case for it: a queue filled to the last slot (tpmc_trace on a
    fresh handle sizes the queue to exactly n rays) in which EVERY ray hits, at a size where any slot a warp reserved
    and then left unused would add up to more than the slack (2^25 rays against 2^19 slots of slack)."""
    import torch
    m = ti.geodesic_sphere(32)
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    om = O.OracleMesh(m.vertices, m.indices, m.flags)
    n = 1 << 25
    g = torch.Generator(device="cuda").manual_seed(11)
    u = torch.randn((n, 3), generator=g, device="cuda", dtype=torch.float32)
    o = 3.0 * u / u.norm(dim=1, keepdim=True)
    t = torch.randn((n, 3), generator=g, device="cuda", dtype=torch.float32)
    t = 0.9 * t / t.norm(dim=1, keepdim=True) * torch.rand((n, 1), generator=g, device="cuda") ** (1.0 / 3.0)
    d = t - o                                                            # aimed at a point well inside the body
    facet, tau = gm.trace(o, d)
    assert int((facet < 0).sum()) == 0 and bool(torch.isfinite(tau).all())
    hit = o.double() + tau[:, None] * d.double()
    rad = hit.norm(dim=1)
    assert float(rad.min()) > 0.995 and float(rad.max()) <= 1.0 + 1e-6     # on the faceted unit sphere, first crossing
    assert bool(((hit * o.double()).sum(1) > 0).all())                      # ... on the side the ray came from
    idx = np.random.default_rng(3).integers(0, n, 300)
    oc, dc = o[idx].cpu().numpy(), d[idx].cpu().numpy()
    fc, tc = facet[idx].cpu().numpy(), tau[idx].cpu().numpy()
    for k in range(idx.size):
        fo, to = om.closest_hit(oc[k], dc[k], -1, use_bvh=True)
        assert fc[k] == fo and tc[k] == to
    gm.close()


# ------------------------------------------------------------------ whole path on the five configs
def test_run_parity_c1_plate_all_particles(T, O):
    cfg = ti.config("C1")[0]
    g, o, frac = compare_run(T, O, cfg, 0, cfg.N, use_bvh=False)
    assert frac == 1.0
    # and the physics: C_D within 4 sigma of the (corrected) Sentman value
    F = g.force.cpu().numpy() / cfg.q_inf
    se = o.force_stderr(cfg.N) / cfg.q_inf
    assert abs(-F[0] - 1.847023) < 4 * se[0] and abs(-F[1] - 0.066379) < 4 * se[1]


@pytest.mark.parametrize("idx", [0, 1, 2])
def test_run_parity_c2_sphere(T, O, idx):
    cfg = ti.config("C2")[idx]
    compare_run(T, O, cfg, 1_000_000 * idx, 150_000)


@pytest.mark.parametrize("idx", [0, 1, 2])
def test_run_parity_c3_cylinder_maxwell(T, O, idx):
    cfg = ti.config("C3")[idx]
    g, o, _ = compare_run(T, O, cfg, 50_000_000, 150_000)
    if idx == 0:                                             # config 3's invariant: zero lateral force at 0 deg
        se = o.force_stderr(150_000)
        F = g.force.cpu().numpy()
        assert abs(F[0]) < 4 * se[0] and abs(F[1]) < 4 * se[1]


@pytest.mark.parametrize("idx", [0, 5, 10, 15])
def test_run_parity_c4_satellite_multiple_reflections(T, O, idx):
    cfg = ti.config("C4")[idx]
    g, o, _ = compare_run(T, O, cfg, 6_000_000 * idx, 200_000)
    assert int(o.bounces.max()) >= 3 and o.truncated == 0


@pytest.mark.parametrize("idx,first,count", [(0, 0, 200_000), (21, 500_000_000, 100_000), (63, 999_900_000, 100_000)])
def test_run_parity_c5_large_body_full_size_stream(T, O, idx, first, count):
    """Slices of the N = 1e9 stream on the ~1.0e6-facet body, in the configuration bench.py times."""
    cfg = ti.config("C5")[idx]
    g, o, _ = compare_run(T, O, cfg, first, count)
    assert g.stats["truncated"] == 0


def test_slices_are_additive_and_runs_repeat(T, O):
    cfg = ti.config("C4")[3].with_(N=400_000)
    gm, _ = meshes(T, O, cfg)
    full = gm.run(cfg)
    a = gm.run(cfg, first=0, count=150_000)
    b = gm.run(cfg, first=150_000, count=250_000)
    F = full.force.cpu().numpy()
    assert np.allclose(a.force.cpu().numpy() + b.force.cpu().numpy(), F, rtol=1e-11)
    assert np.allclose((a.facet_momentum + b.facet_momentum).cpu().numpy(), full.facet_momentum.cpu().numpy(), rtol=1e-9, atol=1e-25)
    assert a.stats["hits"] + b.stats["hits"] == full.stats["hits"]
    again = gm.run(cfg, debug=True)
    assert np.allclose(again.force.cpu().numpy(), F, rtol=1e-12)        # fp64 atomic order only (A20)
    # wave boundaries do not matter: a run spanning several waves equals its one-wave slices
    for r, n in ((full, cfg.N), (a, 150_000), (b, 250_000), (again, cfg.N)):
        check_conservation(r.stats, n)


def test_two_slices_on_two_handles_and_streams_sum_to_the_full_run(T):
    """SURVEY 8(e), the particle-range split as bench.py --split slices runs it on N GPUs, here with both "ranks" on one
    device: two mesh handles, two streams, the two halves of one stream of particles in flight at the same time (handles
    are independent, include/tpmc.h), outputs summed.  Equal to the undivided run: hits exactly, sums to the order of the
    fp64 additions."""
    import torch
    import bench
    cfg = ti.config("C4")[7].with_(N=6_000_001)
    m = cfg.mesh()
    handles = [T.Mesh(m.vertices, m.indices, m.flags) for _ in range(2)]
    full = handles[0].run(cfg)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    parts = []
    for rank in range(2):
        att, first, count = bench.split_plan("slices", 7, rank, 2, 16, cfg.N)
        assert att == 7 and (first, count) == ((0, 3_000_000) if rank == 0 else (3_000_000, 3_000_001))
        with torch.cuda.stream(streams[rank]):
            parts.append(handles[rank].run(cfg, first=first, count=count, stats=False, stream=streams[rank]))
    torch.cuda.synchronize()
    for name in ("force", "torque", "facet_momentum"):
        tot = getattr(parts[0], name) + getattr(parts[1], name)
        ref = getattr(full, name)
        assert float((tot - ref).abs().max()) <= 1e-12 * float(ref.abs().max()) + 1e-30, name
    again = [handles[r].run(cfg, first=r * 3_000_000, count=3_000_000 + r) for r in range(2)]
    assert again[0].stats["hits"] + again[1].stats["hits"] == full.stats["hits"]
    for h in handles:
        h.close()


def test_edge_cases_empty_truncated_host_buffers(T, O):
    cfg = ti.config("C4")[0].with_(N=100_000)
    gm, om = meshes(T, O, cfg)
    z = gm.run(cfg, first=10, count=0, debug=True)
    assert np.all(z.force.cpu().numpy() == 0) and z.stats["hits"] == 0 and z.stats["segments"] == 0
    # bounce cap: particles cut off are counted, and both sides agree on them
    c1 = cfg.with_(max_bounces=1)
    g = gm.run(c1, debug=True)
    o = om.run(c1)
    assert g.stats["truncated"] == o.truncated > 0 and g.stats["hits"] == o.hits and g.stats["segments"] == o.segments
    assert np.array_equal(g.hash.cpu().numpy().view(np.uint64), o.hash)
    # host-buffer entry point gives the same numbers as the device one
    d = gm.run(cfg)
    F, Tq, fm, st = gm.run_host(cfg)
    assert np.allclose(F, d.force.cpu().numpy(), rtol=1e-12) and np.allclose(Tq, d.torque.cpu().numpy(), rtol=1e-10, atol=1e-30)
    assert np.allclose(fm, d.facet_momentum.cpu().numpy(), rtol=1e-9, atol=1e-25) and st["hits"] == d.stats["hits"]
    # no per-facet buffer requested
    nf = gm.run(cfg, facets=False)
    assert np.allclose(nf.force.cpu().numpy(), d.force.cpu().numpy(), rtol=1e-12)


def test_specular_and_mixture_parity(T, O):
    cfg = ti.config("C3")[1].with_(accommodation=0.0, N=1_000_000)
    compare_run(T, O, cfg, 0, 100_000)
    mix = ti.config("C5")[9].with_(mesh_fn=lambda: ti.large_body(5, 24), N=1_000_000)
    mix._mesh_cache = []
    compare_run(T, O, mix, 300_000, 100_000)


def test_run_on_side_stream(T, O):
    import torch
    cfg = ti.config("C2")[1].with_(N=200_000)
    gm, _ = meshes(T, O, cfg)
    ref = gm.run(cfg).force.cpu().numpy()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        r = gm.run(cfg, stream=s)
    s.synchronize()
    assert np.allclose(r.force.cpu().numpy(), ref, rtol=1e-12)


# ------------------------------------------------------------------ a2: the fp32 pre-cull pass drops only misses
@pytest.mark.parametrize("name,idx,count", [("C1", 0, 100_000), ("C2", 0, 3_000_000), ("C2", 2, 3_000_000),
                                             ("C3", 1, 3_000_000), ("C4", 5, 3_000_000), ("C5", 3, 20_000_000)])
def test_precull_pass_changes_nothing(T, name, idx, count):
    """The pre-cull pass may only drop particles whose first segment misses the body: with the pass switched
    off (TPMC_FLAG_NO_PRECULL, every particle through the fp64 sampler) hits, hashes and per-facet sums are identical."""
    cfg = ti.config(name)[idx]
    m = cfg.mesh()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    first = min(cfg.N - count, 777_777)
    a = gm.run(cfg, first=first, count=count, debug=True)
    b = gm.run(cfg, first=first, count=count, debug=True, flags=T.TPMC_FLAG_NO_PRECULL)
    check_conservation(a.stats, count)
    check_conservation(b.stats, count)
    assert b.stats["ret_precull_a"] == 0 and b.stats["ret_precull_b"] == 0
    assert a.stats["hits"] == b.stats["hits"] and a.stats["hits"] > 0
    assert a.stats["kernel_launches"] > b.stats["kernel_launches"]          # the pass really ran in `a` only
    assert bool((a.hash == b.hash).all()) and bool((a.first_facet == b.first_facet).all())
    Fa, Fb = a.force.cpu().numpy(), b.force.cpu().numpy()
    assert np.linalg.norm(Fa - Fb) <= 1e-12 * np.linalg.norm(Fb)
    assert a.stats["culled"] >= b.stats["culled"]     # the grown bounding sphere also drops rays the boxes keep
    gm.close()


# ------------------------------------------------------------------ a4: the escape-horizon test skips only escapes
@pytest.mark.parametrize("name,idx,count", [("C1", 0, 100_000), ("C2", 1, 3_000_000), ("C3", 1, 3_000_000),
                                             ("C4", 0, 3_000_000), ("C4", 9, 3_000_000), ("C5", 3, 20_000_000),
                                             ("C5", 40, 20_000_000)])
def test_escape_horizon_changes_nothing(T, name, idx, count):
    """A re-emitted ray above its facet's escape horizon (k_horizon, lbvh.cu) is not traced: with the test
    switched off (TPMC_FLAG_NO_HORIZON, every reflected ray traced) hits, hashes, bounce counts and forces are
    identical, and with it on fewer rays reach the traversal."""
    cfg = ti.config(name)[idx]
    m = cfg.mesh()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    first = min(cfg.N - count, 1_234_567)
    a = gm.run(cfg, first=first, count=count, debug=True)
    b = gm.run(cfg, first=first, count=count, debug=True, flags=T.TPMC_FLAG_NO_HORIZON)
    check_conservation(a.stats, count)
    check_conservation(b.stats, count)
    assert b.stats["ret_horizon"] == 0
    assert a.stats["hits"] == b.stats["hits"] and a.stats["hits"] > 0
    assert bool((a.hash == b.hash).all()) and bool((a.bounces == b.bounces).all())
    Fa, Fb = a.force.cpu().numpy(), b.force.cpu().numpy()
    assert np.linalg.norm(Fa - Fb) <= 1e-12 * np.linalg.norm(Fb)
    assert a.stats["traced_rays"] <= b.stats["traced_rays"]
    if name in ("C2", "C5"):                           # smooth bodies: most re-emitted rays are above the horizon
        assert a.stats["traced_rays"] < b.stats["traced_rays"] - a.stats["hits"] // 4
    elif name != "C1":                                 # C1 is two-sided (no horizon); facets at sharp edges have none either
        assert a.stats["traced_rays"] < b.stats["traced_rays"]
    gm.close()


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5small"])
def test_rays_above_the_escape_horizon_hit_nothing(T, O, name):
    """Direct check of what the horizon promises (include/tpmc.h, tpmc_mesh_copy_horizon): a ray that leaves a
    point of a one-sided facet above the stored bound of its azimuth sector has no hit in the ORACLE's closest-hit
    search (brute force on the small meshes).  Also: smooth closed bodies do get bounds (the test is not vacuous)."""
    if name == "C5small":
        m = ti.large_body(5, 24)            # same recipe as C5, ~1.2e4 facets: displaced sphere + panels
    else:
        m = ti.config(name)[0].mesh()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    om = O.OracleMesh(m.vertices, m.indices, m.flags)
    hz = gm.copy_horizon()
    _, leaf = gm.copy_bvh()
    rng = np.random.default_rng(7)
    V = m.vertices.astype(np.float64)
    tested = 0
    for slot in rng.integers(0, m.nt, 1500):
        f = int(leaf[slot])
        a0, a1, a2 = (V[m.indices[f, k]] for k in range(3))
        n = np.cross(a1 - a0, a2 - a0)
        n /= np.linalg.norm(n)
        e1 = (a1 - a0) / np.linalg.norm(a1 - a0)
        e2 = np.cross(n, e1)
        k = int(rng.integers(0, 16))
        b = int(hz[slot, k])
        if b == 255:
            continue
        w = rng.dirichlet([1.0, 1.0, 1.0])
        p = (w[0] * a0 + w[1] * a1 + w[2] * a2).astype(np.float32)
        phi = -np.pi + (k + rng.uniform(0.02, 0.98)) * (2 * np.pi / 16)
        s_lo = b / 254.0
        sin_e = min(s_lo + rng.uniform(1e-4, 1.0) ** 3 * (1.0 - s_lo) + 1e-5, 1.0)
        cos_e = np.sqrt(max(1.0 - sin_e ** 2, 0.0))
        d = (500.0 * (cos_e * (np.cos(phi) * e1 + np.sin(phi) * e2) + sin_e * n)).astype(np.float32)
        dd = d.astype(np.float64)
        if not (dd @ n / np.linalg.norm(dd) > s_lo + 1e-6):
            continue
        facet, tau = om.closest_hit(p, d, f_prev=f, use_bvh=(m.nt > 30000))
        assert facet == -1, (name, slot, f, k, b, sin_e, facet, tau)
        tested += 1
    assert tested > 300
    if name in ("C2", "C5small"):
        assert (hz < 128).mean() > 0.5
    gm.close()


def test_c5_whole_stream_in_one_run_sampled_against_the_oracle(T, O):
    """The launch configuration bench.py times: ONE tpmc_run of all N = 1e9 particles of a C5 attitude (15 waves of
    2^26 particles, cross-wave queues, escape horizons, pre-cull), with the per-particle outputs kept (16 GB).
    Windows of the stream are compared particle by particle with the oracle; properties that hold at any size
    (F = sum of P_f, segment count, slices summing to the whole) are checked on the whole run."""
    import torch
    cfg = ti.config("C5")[7]
    gm, om = meshes(T, O, cfg)
    g = gm.run(cfg, debug=True)
    st = g.stats
    check_conservation(st, cfg.N)
    assert st["truncated"] == 0 and st["segments"] == cfg.N + st["hits"]
    assert 0.15 * cfg.N < st["hits"] < 0.20 * cfg.N
    fm = g.facet_momentum
    F = g.force.cpu().numpy()
    assert np.allclose(fm.sum(0).cpu().numpy(), F, rtol=1e-10)
    assert int((g.bounces > 0).sum().item()) <= st["hits"] and int(g.bounces.sum(dtype=torch.int64).item()) == st["hits"]
    worst = 1.0
    for first, count in ((0, 100_000), (67_108_864 - 50_000, 100_000), (523_456_789, 100_000), (999_900_000, 100_000)):
        o = om.run(cfg, first=first, count=count, facets=False)
        gh = g.hash[first:first + count].cpu().numpy().view(np.uint64)
        same = gh == o.hash
        worst = min(worst, same.mean())
        assert same.mean() >= SEQ_AGREE
        assert np.array_equal(g.bounces[first:first + count].cpu().numpy().astype(np.uint32)[same], o.bounces[same])
        assert np.array_equal(g.first_facet[first:first + count].cpu().numpy()[same], o.first_facet[same])
    del g
    torch.cuda.empty_cache()
    # the whole run equals the sum of its quarters (different wave boundaries, different queue contents)
    Fq, hq = np.zeros(3), 0
    for k in range(4):
        r = gm.run(cfg, first=k * 250_000_000, count=250_000_000, facets=False)
        Fq += r.force.cpu().numpy()
        hq += r.stats["hits"]
    assert hq == st["hits"]
    assert np.linalg.norm(Fq - F) <= 1e-11 * np.linalg.norm(F)


@pytest.mark.parametrize("S", [5.0, 40.0])
def test_run_parity_concave_shell(T, O, S):
    """NEXT-2 workload: two-sided hemispherical shell, concave to the stream, at the paper's
    verification temperatures; 0.7 hits per particle, two-sided facets (no escape horizon), hits from both sides."""
    m = ti.hemisphere_shell(16)
    mO = 16 * ti.AMU
    speed = S * np.sqrt(2 * ti.K_B * 922.0 / mO)
    cfg = ti.RunConfig("shell", lambda: m, T_inf=922.0, T_W=300.0, V=(-speed, 0.0, 0.0), N=300_000,
                       A_ref=float(np.pi), seed=14, label=f"concave shell S={S:g}")
    g, o, _ = compare_run(T, O, cfg, 0, 300_000)
    assert g.stats["hits"] == o.hits > 0.6 * cfg.N


def test_repeated_multi_wave_runs_agree(T, O):
    """Several waves of 2^26 particles through the staged pre-cull pass, the cross-wave queues and the side streams,
    four times over: integer outputs must repeat exactly, sums to the order of the fp64 atomics (A20).  (A barrier
    race in the pre-cull kernel once changed the survivor lists of about one run in 180.)"""
    cfg = ti.config("C5")[11]
    gm, _ = meshes(T, O, cfg)
    ref = None
    for _ in range(4):
        r = gm.run(cfg, first=100_000_000, count=200_000_000, facets=False)
        check_conservation(r.stats, 200_000_000)
        cur = (r.stats["hits"], r.stats["segments"], r.stats["truncated"], r.force.cpu().numpy(), r.torque.cpu().numpy())
        if ref is None:
            ref = cur
            continue
        assert cur[:3] == ref[:3]
        assert np.linalg.norm(cur[3] - ref[3]) <= 1e-12 * np.linalg.norm(ref[3])
        assert np.linalg.norm(cur[4] - ref[4]) <= 1e-11 * max(np.linalg.norm(ref[4]), 1e-3 * np.linalg.norm(ref[3]))


# ------------------------------------------------------------------ the flow-aligned hierarchy changes nothing
def thin_plate_cfg():
    """A two-sided plate whose normal lies along an oblique stream: in the stream frame the body has (almost) no
    extent along z', the case in which the rotation error of the traversal's slab margin, a length in metres, is
    thousands of steps of that axis' quantisation grid (trace.cuh, grid_ray)."""
    n = np.array([0.48, -0.62, 0.62])
    n /= np.linalg.norm(n)
    a = np.cross(n, [0.0, 0.0, 1.0]); a /= np.linalg.norm(a)
    b = np.cross(n, a)
    c = np.array([3.0, -2.0, 1.5])              # far from the origin: large |o|_1
    v = np.array([c - 0.5 * a - 0.5 * b, c + 0.5 * a - 0.5 * b, c + 0.5 * a + 0.5 * b, c - 0.5 * a + 0.5 * b])
    m = ti.Mesh(v.astype(np.float32), np.int32([[0, 1, 2], [0, 2, 3]]), np.uint8([1, 1]), "oblique_plate")
    return ti.RunConfig("thin", lambda: m, V=tuple(-7500.0 * n), N=400_000, seed=31, label="plate normal to an oblique stream")


@pytest.mark.parametrize("name,idx,count", [("C1", 0, 100_000), ("thin", 0, 400_000), ("C2", 1, 2_000_000), ("C3", 1, 2_000_000),
                                             ("C4", 6, 3_000_000), ("C4", 15, 3_000_000), ("C5", 3, 10_000_000),
                                             ("C5", 30, 10_000_000)])
def test_flow_alignment_changes_nothing(T, O, name, idx, count):
    """tpmc_run walks either the body-frame hierarchy or its refit in the stream frame (heuristic on the attitude);
    forced one way and the other (TPMC_FLAG_ALIGN_OFF / _ON), hashes, bounce counts and forces are identical."""
    cfg = thin_plate_cfg() if name == "thin" else ti.config(name)[idx]
    m = cfg.mesh()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    first = min(cfg.N - count, 2_345_678)
    a = gm.run(cfg, first=first, count=count, debug=True, flags=T.TPMC_FLAG_ALIGN_OFF)
    b = gm.run(cfg, first=first, count=count, debug=True, flags=T.TPMC_FLAG_ALIGN_ON)
    check_conservation(a.stats, count)
    check_conservation(b.stats, count)
    assert a.stats["hits"] == b.stats["hits"] > 0
    assert b.stats["kernel_launches"] > a.stats["kernel_launches"]          # the refit really ran in `b` only
    assert bool((a.hash == b.hash).all()) and bool((a.bounces == b.bounces).all()) and bool((a.first_facet == b.first_facet).all())
    Fa, Fb = a.force.cpu().numpy(), b.force.cpu().numpy()
    assert np.linalg.norm(Fa - Fb) <= 1e-12 * np.linalg.norm(Fb)
    if name == "thin":                          # and against the oracle, on the aligned hierarchy
        compare_run(T, O, cfg, 0, 100_000, use_bvh=False, flags=T.TPMC_FLAG_ALIGN_ON)
    gm.close()


# ------------------------------------------------------------------ the fp32 filter + candidate lists change nothing
@pytest.mark.parametrize("name,idx,count", [("C1", 0, 100_000), ("C2", 2, 2_000_000), ("C3", 2, 2_000_000), ("C4", 3, 2_000_000),
                                             ("C5", 17, 4_000_000)])
def test_exact_trace_arm_changes_nothing(T, name, idx, count):
    """TPMC_FLAG_EXACT_TRACE sends every segment through the fp64 closest-hit search of the straggler kernel (no
    wavefront traversal, no fp32 classification, no candidate lists): same hashes, bounces, forces."""
    cfg = ti.config(name)[idx]
    m = cfg.mesh()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    first = min(cfg.N - count, 3_456_789)
    a = gm.run(cfg, first=first, count=count, debug=True)
    b = gm.run(cfg, first=first, count=count, debug=True, flags=T.TPMC_FLAG_EXACT_TRACE)
    check_conservation(a.stats, count)
    check_conservation(b.stats, count, exact=True)
    assert a.stats["hits"] == b.stats["hits"] > 0
    assert bool((a.hash == b.hash).all()) and bool((a.bounces == b.bounces).all()) and bool((a.first_facet == b.first_facet).all())
    Fa, Fb = a.force.cpu().numpy(), b.force.cpu().numpy()
    assert np.linalg.norm(Fa - Fb) <= 1e-12 * np.linalg.norm(Fb)
    gm.close()


# ------------------------------------------------------------------ rare paths of tpmc_run, each forced
def test_candidate_overflow_inside_a_run(T, O):
    """Six coincident copies of every facet: each hit is a six-way tie, the traversal's three-slot candidate list
    overflows, the ray goes to the overflow list and the straggler kernel resolves it (A12: smallest index)."""
    cfg = ti.RunConfig("dup", lambda: ti.stacked_duplicates(6), N=200_000, seed=41, label="six coincident copies")
    g, o, frac = compare_run(T, O, cfg, 0, cfg.N, use_bvh=False)
    assert frac == 1.0 and g.stats["overflow_rays"] >= o.hits // 2 > 1000
    assert set(np.unique(o.first_facet)) <= {-1, 0, 1}


def test_traversal_stack_overflow_inside_a_run(T, O):
    """A hierarchy about 28 levels deep whose boxes a ray along +x all overlaps: the shared-memory stack of the wavefront
    traversal (24 entries of the 4-wide hierarchy) gives up and the straggler kernel (deep stack) takes the ray."""
    cfg = ti.RunConfig("chain", lambda: ti.deep_chain(), V=(7500.0, 0.0, 0.0), N=100_000, seed=42, label="deep chain")
    g, o, frac = compare_run(T, O, cfg, 0, cfg.N, use_bvh=False)
    assert frac == 1.0 and g.stats["overflow_rays"] > 1000
    assert g.stats["truncated"] == o.truncated


def test_full_reflected_region_tiny_waves_and_untimed_iterations(T, O):
    """A hollow box with a small opening keeps particles bouncing (chains of > 100 reflections): with waves of 256
    particles the reflected rays outgrow region A of the queue (write-back into the ray's own slot + overflow list),
    and the run has more iterations than the per-kernel timing events cover."""
    cfg = ti.RunConfig("pot", lambda: ti.lobster_pot(), N=300_000, seed=43, label="lobster pot")
    g, o, frac = compare_run(T, O, cfg, 0, cfg.N, wave_particles=256)
    assert frac == 1.0 and int(o.bounces.max()) > 100
    assert g.stats["overflow_rays"] > 0 and g.stats["trace_launches"] == 1024 and g.stats["timed_waves"] == 1024
    big = meshes(T, O, cfg)[0].run(cfg, debug=True)                       # one wave: same answers
    assert bool((big.hash == g.hash).all()) and big.stats["overflow_rays"] == 0


def test_index_chunks(T, O):
    """Queues carry 32-bit particle offsets into a chunk of the slice; with a small chunk_particles the chunk loop
    of tpmc_run (otherwise reached only beyond 4.0e9 particles) runs several times."""
    cfg = ti.config("C4")[7].with_(N=1_000_000)
    g, o, frac = compare_run(T, O, cfg, 123_456, 250_000, chunk_particles=100_000, wave_particles=40_000)
    assert frac == 1.0


def test_torque_about_an_off_centre_reference_point(T, O):
    """A14 on the GPU: x_ref != 0 against the oracle (whose torque is pinned by P16), and the shift identity."""
    cfg = ti.config("C4")[9].with_(N=400_000, x_ref=(0.3, -0.2, 0.5))
    g, o, _ = compare_run(T, O, cfg, 0, 200_000)
    assert np.linalg.norm(o.torque) > 1e-2 * np.linalg.norm(o.force)
    gm, _ = meshes(T, O, cfg)
    z = gm.run(cfg.with_(x_ref=(0.0, 0.0, 0.0)), first=0, count=200_000)
    F, t0, t1 = g.force.cpu().numpy(), z.torque.cpu().numpy(), g.torque.cpu().numpy()
    assert np.linalg.norm(t1 - (t0 - np.cross(cfg.x_ref, F))) <= 1e-10 * (np.linalg.norm(t0) + np.linalg.norm(F))


def test_equilibrium_through_the_whole_path(T, O):
    """P10 through tpmc_run: V = 0, T_W = T_inf on the pocket satellite (S = 0: the series branch of the position
    CDF, no certified pre-cull, degenerate rotation and alignment).  Parity with the oracle on the same stream, and
    the physics on a GPU-sized sample: zero net force on a closed solid, P_f = -n k_B T A_f n_f inside the pocket."""
    mfn = lambda: ti.satellite(seed=2, h=0.25)
    cfg = ti.RunConfig("eq", mfn, T_inf=500.0, T_W=500.0, V=(0.0, 0.0, 0.0), N=20_000_000, seed=5, cv_radius_factor=1.05,
                       label="equilibrium")
    g, o, frac = compare_run(T, O, cfg, 0, 150_000)
    assert frac >= SEQ_AGREE and int(o.bounces.max()) >= 3
    gm, _ = meshes(T, O, cfg)
    per = cfg.N // 8
    runs = [gm.run(cfg, first=k * per, count=per) for k in range(8)]
    Fs = np.array([r.force.cpu().numpy() for r in runs]) * 8
    m = cfg.mesh()
    tri = m.triangles()
    Ng = np.cross(tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0])
    A = 0.5 * np.linalg.norm(Ng, axis=1)
    nh = Ng / (2 * A)[:, None]
    p = cfg.n * ti.K_B * cfg.T_inf
    scale = p * A.sum()
    assert np.all(np.abs(Fs.mean(0)) < 4 * Fs.std(0, ddof=1) / np.sqrt(8) + 1e-9 * scale)
    cen = tri.mean(1)
    floor = (np.abs(cen[:, 2] - 0.5) < 1e-6) & (np.abs(cen[:, 0]) < 0.31) & (np.abs(cen[:, 1]) < 0.31)
    vals = np.array([np.einsum("ij,ij->", r.facet_momentum.cpu().numpy()[floor], nh[floor]) * 8 for r in runs])
    want = -p * A[floor].sum()
    se = vals.std(ddof=1) / np.sqrt(8)
    assert abs(vals.mean() - want) < 4 * se and se < 0.02 * abs(want)


# ------------------------------------------------------------------ exhaustive on/off checks at timing size
def _arms(T):
    return [("no pre-cull", T.TPMC_FLAG_NO_PRECULL), ("no horizon", T.TPMC_FLAG_NO_HORIZON),
            ("body-frame boxes", T.TPMC_FLAG_ALIGN_OFF), ("flow-aligned boxes", T.TPMC_FLAG_ALIGN_ON),
            ("rays sorted by key", T.TPMC_FLAG_SORT_RAYS), ("seed kernels behind the traversal", T.TPMC_FLAG_SERIAL_SEED),
            ("fp64 search, nothing skipped", T.TPMC_FLAG_EXACT_TRACE | T.TPMC_FLAG_NO_PRECULL | T.TPMC_FLAG_NO_HORIZON)]


def _full_size_arms(T, cfg, arms):
    import torch
    m = cfg.mesh()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    ref = gm.run(cfg, debug=True, facets=False)
    check_conservation(ref.stats, cfg.N)
    assert ref.stats["truncated"] == 0
    F = ref.force.cpu().numpy()
    for label, flags in arms:
        r = gm.run(cfg, debug=True, facets=False, flags=flags)
        check_conservation(r.stats, cfg.N, exact=bool(flags & T.TPMC_FLAG_EXACT_TRACE))
        assert r.stats["hits"] == ref.stats["hits"], label
        assert torch.equal(r.hash, ref.hash), label                       # every particle of the stream
        assert torch.equal(r.bounces, ref.bounces) and torch.equal(r.first_facet, ref.first_facet), label
        assert np.linalg.norm(r.force.cpu().numpy() - F) <= 1e-11 * np.linalg.norm(F), label
        del r
        torch.cuda.empty_cache()
    gm.close()


@pytest.mark.parametrize("att", [0, 21, 40])
def test_c5_every_shortcut_off_at_full_size(T, att):
    """Every "exact" shortcut switched off in turn on ALL 1e9 particles of a C5 attitude (axis-near, oblique, and
    the diagonal-most of the sweep), in the launch configuration bench.py times: the per-particle hashes, bounce
    counts and first facets of the whole stream are compared on the device.  The last arm runs every segment
    through the fp64 search with the pre-cull and the horizon off as well."""
    cfg = ti.config("C5")[att]
    arms = _arms(T)
    if att != 21:
        arms = arms[:-1]            # the thread-per-particle fp64 arm on 1e9 particles once only
    _full_size_arms(T, cfg, arms)


@pytest.mark.parametrize("name,idx", [("C2", 0), ("C3", 1), ("C4", 8)])
def test_c2_c3_c4_every_shortcut_off_at_timing_size(T, name, idx):
    """The same at the timing sizes of SURVEY 8(d): C2 N = 1e7, C3 N = 1e8, C4 N = 1e8."""
    _full_size_arms(T, ti.config(name)[idx], _arms(T))


def test_c5_precull_and_horizon_off_on_every_attitude_of_the_sweep(T):
    """The two shortcuts whose exactness rests on a margin rather than on a proof carried by the code (the fp32 pre-cull's
    grown volumes and the per-facet escape horizons) switched off together on ALL 1e9 particles of
    ALL 64 attitudes of the C5 sweep -- the three attitudes of the test above leave 61 directions of the stream, and with
    them most of the facets' horizon sectors, unvisited.  Per attitude: same hits, same hash / bounce count / first facet
    for every particle, same force to the order of the fp64 additions."""
    import torch
    cfgs = ti.config("C5")
    m = cfgs[0].mesh()
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    off = T.TPMC_FLAG_NO_PRECULL | T.TPMC_FLAG_NO_HORIZON
    for k, cfg in enumerate(cfgs):
        a = gm.run(cfg, debug=True, facets=False)
        b = gm.run(cfg, debug=True, facets=False, flags=off)
        check_conservation(a.stats, cfg.N)
        check_conservation(b.stats, cfg.N)
        assert b.stats["ret_precull_a"] + b.stats["ret_precull_b"] + b.stats["ret_horizon"] == 0
        assert a.stats["ret_precull_a"] + a.stats["ret_precull_b"] > 0 and a.stats["ret_horizon"] > 0
        assert a.stats["hits"] == b.stats["hits"] > 0, k
        assert torch.equal(a.hash, b.hash), k
        assert torch.equal(a.bounces, b.bounces) and torch.equal(a.first_facet, b.first_facet), k
        Fa, Fb = a.force.cpu().numpy(), b.force.cpu().numpy()
        assert np.linalg.norm(Fa - Fb) <= 1e-11 * np.linalg.norm(Fb), k
        del a, b
    gm.close()


@pytest.mark.parametrize("S", [0.1, 0.3, 1.0])
def test_precull_and_horizon_off_at_low_speed_ratio_all_particles(T, S):
    """The same two switches where the thermal spread is largest: speed ratio S of the heavier species 0.1, 0.3, 1 (the
    lighter one at half of that), 1e8 particles on the concave satellite.  At these S the particles arrive from all
    round the control sphere and the pre-cull's certified-miss test works with wide velocity cones; every config of the
    sweep tests runs at S >= 2."""
    base = ti.config("C4")[5]
    c_mp = np.sqrt(2.0 * ti.K_B * base.T_inf / (16.0 * ti.AMU))
    vhat = np.array(base.V) / np.linalg.norm(base.V)
    cfg = base.with_(N=100_000_000, V=tuple(S * c_mp * vhat), m=(16.0 * ti.AMU, 4.0 * ti.AMU), x=(0.7, 0.3))
    _full_size_arms(T, cfg, [("no pre-cull", T.TPMC_FLAG_NO_PRECULL), ("no horizon", T.TPMC_FLAG_NO_HORIZON)])


# ------------------------------------------------------------------ NEXT-3: surface models beyond one global T_W, sigma
def test_per_facet_surface_and_energy_accommodation_parity(T, O):
    """Readings A22 / A23 against the oracle (whose versions are pinned by P17): wall temperature and accommodation
    per facet, partial energy accommodation, both together on a concave body with a gas mixture; and alpha_E = 1 with
    uniform arrays equal to the scalars reproduces the scalar run."""
    m = ti.satellite(4, 0.1)
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    om = O.OracleMesh(m.vertices, m.indices, m.flags)
    cen = m.triangles().mean(1)
    TW = np.where(cen[:, 1] > 0, 200.0, 1500.0) + 50.0 * np.sin(7.0 * cen[:, 0])
    sg = np.where(cen[:, 2] > 0, 1.0, 0.5)
    base = ti.config("C4")[6].with_(N=1_000_000, mesh_fn=lambda: m, m=(16.0 * ti.AMU, 4.0 * ti.AMU), x=(0.6, 0.4))
    base._mesh_cache = [m]
    ref = gm.run(base, first=0, count=150_000, debug=True)
    # (1) alpha_E < 1, scalar surface
    g1, o1, _ = compare_run(T, O, base.with_(energy_accommodation=0.4), 0, 150_000, pair=(gm, om))
    assert not np.allclose(g1.force.cpu().numpy(), ref.force.cpu().numpy(), rtol=1e-3)        # the model does act
    # (2) per-facet arrays, alpha_E = 1
    gm.set_surface(TW, sg)
    om.set_surface(TW, sg)
    g2, o2, _ = compare_run(T, O, base, 0, 150_000, pair=(gm, om))
    assert not np.allclose(g2.force.cpu().numpy(), ref.force.cpu().numpy(), rtol=1e-3)
    # (3) both
    compare_run(T, O, base.with_(energy_accommodation=0.7), 300_000, 150_000, pair=(gm, om))
    # (4) only sigma per facet; T_W from the run
    gm.set_surface(None, sg)
    om.set_surface(None, sg)
    compare_run(T, O, base, 0, 100_000, pair=(gm, om))
    # (5) uniform arrays equal to the run's scalars: the scalar run again (same hashes; sums to the atomics' order)
    gm.set_surface(np.full(m.nt, base.T_W), np.full(m.nt, base.accommodation))
    u = gm.run(base, first=0, count=150_000, debug=True)
    assert bool((u.hash == ref.hash).all())
    assert np.linalg.norm(u.force.cpu().numpy() - ref.force.cpu().numpy()) <= 1e-12 * np.linalg.norm(ref.force.cpu().numpy())
    gm.set_surface(None, None)
    z = gm.run(base, first=0, count=150_000, debug=True)
    assert bool((z.hash == ref.hash).all())
    with pytest.raises(T.TpmcError):
        gm.set_surface(np.full(m.nt, -1.0), None)
    # (6) arrays handed over in DEVICE memory: the same run as from host arrays, and the same checks -- a wall
    # temperature <= 0 or NaN, or an accommodation outside [0, 1], anywhere in the array, is refused and changes nothing
    import torch
    TWd, sgd = torch.as_tensor(TW, device="cuda"), torch.as_tensor(sg, device="cuda")
    gm.set_surface(TWd, sgd)
    d2 = gm.run(base, first=0, count=150_000, debug=True)
    assert bool((d2.hash == g2.hash).all())
    assert np.linalg.norm(d2.force.cpu().numpy() - g2.force.cpu().numpy()) <= 1e-12 * np.linalg.norm(g2.force.cpu().numpy())
    for k, val in ((0, 0.0), (m.nt // 2, float("nan")), (m.nt - 1, -5.0), (3, float("inf"))):
        bad = TWd.clone(); bad[k] = val
        with pytest.raises(T.TpmcError):
            gm.set_surface(bad, sgd)
    for k, val in ((1, 1.0 + 1e-9), (m.nt - 1, float("nan")), (7, -0.1)):
        bad = sgd.clone(); bad[k] = val
        with pytest.raises(T.TpmcError):
            gm.set_surface(TWd, bad)
        with pytest.raises(T.TpmcError):
            gm.set_surface(None, bad)
    d3 = gm.run(base, first=0, count=150_000, debug=True)                # the refused calls left the surface as it was
    assert bool((d3.hash == g2.hash).all()) and bool(torch.isfinite(d3.force).all())
    with pytest.raises(T.TpmcError):
        gm.run(base.with_(energy_accommodation=1.5))
    gm.close()


def test_warp_aggregated_accumulation_changes_nothing(T, O):
    """a5: on bodies with few facets the reflect step sums the lanes of a warp that hit the same facet before its fp64
    atomics; with TPMC_FLAG_NO_AGGREGATION every hit issues its own.  Same per-facet sums to the order of the additions."""
    for name, idx, count in (("C1", 0, 100_000), ("C3", 1, 3_000_000)):
        cfg = ti.config(name)[idx]
        gm, om = meshes(T, O, cfg)
        a = gm.run(cfg, first=0, count=count, debug=True)
        b = gm.run(cfg, first=0, count=count, debug=True, flags=T.TPMC_FLAG_NO_AGGREGATION)
        assert a.stats["hits"] == b.stats["hits"] > 0 and bool((a.hash == b.hash).all())
        fa, fb = a.facet_momentum.cpu().numpy(), b.facet_momentum.cpu().numpy()
        assert np.all(np.abs(fa - fb) <= 1e-11 * np.abs(fb).max(0))
        assert np.array_equal(np.linalg.norm(fa, axis=1) == 0, np.linalg.norm(fb, axis=1) == 0)


# ------------------------------------------------------------------ NEXT-4: rectangular control volume, sweeps, moment maps
@pytest.mark.parametrize("cv", [1, 2])
def test_box_control_volume_parity(T, O, cv):
    """The rectangular scheme the paper replaces (readings A24 / A25; oracle pins P18), flux-weighted and as the
    unweighted negative control: seeding within 1e-12 of the oracle, then the whole path on a concave body."""
    cfg = ti.config("C4")[4].with_(N=600_000, mesh_fn=lambda: ti.satellite(4, 0.1), control_volume=cv, seed=71,
                                   m=(16.0 * ti.AMU, 4.0 * ti.AMU), x=(0.5, 0.5))
    cfg._mesh_cache = []
    gm, om = meshes(T, O, cfg)
    x, v, s = (a.cpu().numpy() for a in gm.seed(cfg, first=1000, count=2000))
    for j in range(0, 2000, 3):
        xo, vo, so = om.seed(cfg, 1000 + j)
        assert so == s[j] and np.abs(x[j] - xo).max() <= 1e-12 * np.abs(xo).max() + 1e-300
        assert np.abs(v[j] - vo).max() <= SEED_RTOL * np.abs(vo).max() + 1e-9
    g, o, frac = compare_run(T, O, cfg, 100_000, 200_000)
    assert g.stats["ret_precull_a"] == 0 and g.stats["ret_precull_b"] == 0      # the fp32 pre-cull is the sphere scheme's


def test_box_scheme_agrees_with_sphere_scheme_and_its_negative_control_does_not(T):
    """Fig. 1 of the paper on the GPU: sphere drag at 2e7 particles per point.  The spherical scheme and
    the flux-weighted box agree at both attitudes; the unweighted box is off by ~2 % at 45 deg to the box."""
    m = ti.geodesic_sphere(16)
    gm = T.Mesh(m.vertices, m.indices, m.flags)
    N, nb = 24_000_000, 8
    cd = {}
    for ang in (0.0, 45.0):
        a = np.deg2rad(ang)
        V = (-7500.0 * np.cos(a), -7500.0 * np.sin(a), 0.0)
        up = -np.array(V) / 7500.0
        for cv in (0, 1, 2):
            cfg = ti.RunConfig("fig1", None, V=V, N=N, seed=72, control_volume=cv)
            Fs = np.array([gm.run(cfg, first=k * (N // nb), count=N // nb, facets=False, stats=False).force.cpu().numpy()
                           for k in range(nb)])
            d = (Fs @ (-up)) * nb / cfg.q_inf / np.pi
            cd[(ang, cv)] = (d.mean(), d.std(ddof=1) / np.sqrt(nb))
    for ang in (0.0, 45.0):
        s, b, u = cd[(ang, 0)], cd[(ang, 1)], cd[(ang, 2)]
        assert abs(s[0] - b[0]) < 4 * np.hypot(s[1], b[1]), (ang, s, b)
    s, u = cd[(45.0, 0)], cd[(45.0, 2)]
    assert abs(u[0] - s[0]) > 10 * np.hypot(s[1], u[1]) and abs(u[0] / s[0] - 1.0) > 0.01
    assert abs(cd[(0.0, 0)][0] - cd[(45.0, 0)][0]) < 4 * np.hypot(cd[(0.0, 0)][1], cd[(45.0, 0)][1])   # sphere scheme: no attitude dependence
    gm.close()


def test_attitude_sweep_in_one_call_and_moment_map(T, O):
    """tpmc_run_sweep: K attitudes in one call equal K separate runs, and the pitching-moment map about a reference
    point (Figs. 8-9) agrees with the oracle's at the sampled pitch angles."""
    cfgs = [c.with_(N=200_000, x_ref=(0.0, 0.0, -0.5), mesh_fn=lambda: ti.satellite(4, 0.1)) for c in ti.config("C4")[::5]]
    for c in cfgs:
        c._mesh_cache = cfgs[0]._mesh_cache
    gm, om = meshes(T, O, cfgs[0])
    V = np.array([c.V for c in cfgs])
    F, Tq, fm, st = gm.sweep(cfgs[0], V, facets=True, stats=True)
    F, Tq = F.cpu().numpy(), Tq.cpu().numpy()
    assert F.shape == (len(cfgs), 3) and fm.shape == (len(cfgs), gm.nt, 3)
    for k, c in enumerate(cfgs):
        one = gm.run(c)
        assert np.allclose(one.force.cpu().numpy(), F[k], rtol=1e-11) and st[k]["hits"] == one.stats["hits"]
        assert np.allclose(fm[k].sum(0).cpu().numpy(), F[k], rtol=1e-9)
        o = om.run(c, debug=False, facets=False)
        q = c.q_inf
        cm_gpu, cm_cpu = Tq[k, 1] / (q * 1.0 * 2.0), o.torque[1] / (q * 1.0 * 2.0)      # pitch axis y, A_ref 1 m^2, L_ref 2 m
        assert abs(cm_gpu - cm_cpu) <= 1e-4 * max(abs(cm_cpu), 1e-3 * np.linalg.norm(o.force) / q)
    assert np.ptp(Tq[:, 1]) > 0.0                                     # the map is not flat
