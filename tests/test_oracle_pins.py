"""Pins of the CPU oracle: the oracle against what the paper and the
mathematics fix -- published Philox vectors, quadrature of the paper's integrals, closed forms,
invariants, brute force.  None of these compare the oracle with itself or with the CUDA path."""
import numpy as np
import pytest
from scipy import stats

import closed_forms as cf
import oracle
import tpmc_inputs as ti

S1, SW1 = 7.356804, 13.431624


def omesh(m):
    return oracle.OracleMesh(m.vertices, m.indices, m.flags)


def batch_sigma(om, cfg, nb=8):
    """Total force and its standard error from nb disjoint slices of the same stream."""
    per = cfg.N // nb
    Fs = np.array([om.run(cfg, first=k * per, count=per, debug=False).force for k in range(nb)])
    F = Fs.sum(0) * (cfg.N / (per * nb))
    return F, Fs.std(0, ddof=1) * np.sqrt(nb) * (cfg.N / (per * nb))


# ------------------------------------------------------------------ P1
def test_p1_philox_known_answers():
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        w = [int(x, 16) for x in r]
        assert oracle.philox4x32_10(w[4:6], w[0:4]) == w[6:10]


# ------------------------------------------------------------------ P2
@pytest.mark.parametrize("S", [1e-6, 5e-5, 1e-3, 0.3, 2.0, 5.0, 8.0, 30.0])
def test_p2_flux_vs_quadrature(S):
    assert oracle.flux_bracket(S) == pytest.approx(cf.flux_bracket_quadrature(S), rel=1e-11)


def test_p2_flux_limits_and_scaling():
    assert oracle.flux(0.0, 3.0, 2.0, 5.0) == pytest.approx(2 * np.sqrt(np.pi) * 3 * 2 * 25, rel=1e-14)
    c, n, r = 1000.0, 1e15, 1.5
    assert oracle.flux(80.0, c, n, r) == pytest.approx(np.pi * r * r * n * 80.0 * c, rel=1e-4)
    for S, v in cf.golden("flux_bracket").items():
        assert oracle.flux_bracket(S) == pytest.approx(v, rel=1e-11)


# ------------------------------------------------------------------ P3
@pytest.mark.parametrize("S", [0.05, 2.0, 5.0, 8.0])
def test_p3_position_inverse_vs_quadrature_of_eq11(S):
    # H^{-1} inverts the quadrature CDF of eq. (11) as printed
    for t in (-0.95, -0.5, -0.1, 0.0, 0.2, 0.6, 0.9, 0.999):
        u = cf.phi_cdf_quadrature(np.arcsin(t), S)
        if u < 1e-9:
            continue  # below the resolution the quadrature reference can give
        assert oracle.position_inv(u, S) == pytest.approx(t, abs=2e-9 / max(u, 1e-3) ** 0 + 1e-9)
    if S in cf.golden("p_lee"):
        assert oracle.position_cdf(0.0, S) == pytest.approx(cf.golden("p_lee")[S], rel=2e-6)


def test_p3_ks_and_limits():
    rng = np.random.default_rng(1)
    S = 5.0
    u = (rng.integers(0, 2 ** 32, 40000) + 0.5) / 2 ** 32
    t = np.array([oracle.position_inv(x, S) for x in u])
    grid = np.linspace(-1, 1, 801)
    cdf = np.array([cf.phi_cdf_quadrature(np.arcsin(g), S) for g in grid])
    ks = stats.kstest(t, lambda x: np.interp(x, grid, cdf))
    assert ks.pvalue > 1e-3
    # eq. (12): S->0 gives g = cos(phi)/2, i.e. t uniform on [-1,1]
    for x in (0.01, 0.3, 0.77):
        assert oracle.position_inv(x, 1e-6) == pytest.approx(2 * x - 1, abs=1e-5)
        assert oracle.position_inv(x, 2e-4) == pytest.approx(oracle.position_inv(x, 0.99e-4), abs=2e-4)
    # eq. (13): S->inf gives sin(2 phi) on phi>=0, i.e. CDF t^2
    for x in (0.04, 0.25, 0.81):
        assert oracle.position_inv(x, 60.0) == pytest.approx(np.sqrt(x), abs=2e-3)


# ------------------------------------------------------------------ P4
@pytest.mark.parametrize("s", [-5.0, -2.0, 0.0, 2.0, 8.0])
def test_p4_normal_speed_inverse_vs_quadrature_of_eq14a(s):
    for x in (0.02, 0.3, 1.0, 2.5):
        xx = x + max(s, 0.0) - (1.0 if s > 1 else 0.0)
        u = cf.vn_cdf_quadrature(xx, s)
        if not (1e-9 < u < 1 - 1e-9):
            continue
        assert oracle.vn_inv(u, s) == pytest.approx(xx, rel=1e-7, abs=1e-9)
    # mean of eq. (14a): sample mean over a stratified set of uniforms
    u = (np.arange(20000) + 0.5) / 20000
    xs = np.array([oracle.vn_inv(x, s) for x in u])
    assert xs.mean() == pytest.approx(cf.vn_mean(s), rel=2e-4)
    assert np.all(np.diff(xs) > 0)


def test_p4_printed_means():
    assert cf.vn_mean(0.0) == pytest.approx(0.886227, abs=1e-6)
    assert cf.vn_mean(5.0) == pytest.approx(5.100000, abs=1e-6)
    assert cf.vn_mean(-2.0) == pytest.approx(0.391425, abs=1e-6)


# ------------------------------------------------------------------ rotation O8
def test_rotation_maps_z_to_upstream():
    rng = np.random.default_rng(3)
    for V in list(rng.normal(size=(20, 3))) + [np.array([0, 0, -2.0]), np.array([0, 0, 3.0]), np.array([-7500.0, 0, 0])]:
        R = oracle.rotation(V)
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-14)
        assert np.linalg.det(R) == pytest.approx(1.0, abs=1e-14)
        assert np.allclose(R @ [0, 0, 1], -V / np.linalg.norm(V), atol=1e-14)
    assert np.allclose(oracle.rotation([0, 0, 0]), np.eye(3))


# ------------------------------------------------------------------ P5, P6: seeding, jointly
@pytest.mark.parametrize("S", [0.0, 2.0, 8.0])
def test_p5_p6_first_hit_counts_on_convex_mesh(S):
    m = ti.geodesic_sphere(3)          # 180 facets, convex
    om = omesh(m)
    mO = 16 * ti.AMU
    N = 120000
    T = 1000.0
    V = S * cf.thermal_speed(T, mO)
    cfg = ti.RunConfig("t", None, T_inf=T, V=(-V * 0.6, 0.0, -V * 0.8), N=N, seed=11)
    r = om.run(cfg, use_bvh=False)
    ctr, Rb = om.bounds()
    rcv = 1.5 * Rb
    if S == 0.0:
        flux = 0.5 * np.linalg.norm(np.cross(*(m.triangles()[:, k] - m.triangles()[:, 0] for k in (1, 2))), axis=1) / (2 * np.sqrt(np.pi))
        expect = N * flux / (2 * np.sqrt(np.pi) * rcv ** 2)
    else:
        _, flux, _ = cf.panel_sum(m.triangles(), m.flags, -np.array(cfg.V) / V, S, 10.0)
        expect = N * flux / (cf.flux_bracket_quadrature(S) * rcv ** 2)
    counts = np.bincount(r.first_facet[r.first_facet >= 0], minlength=m.nt)
    # total hit fraction: binomial 4 sigma (P5: = projected-area ratio, (R/r)^2 for a sphere)
    ptot = expect.sum() / N
    assert abs(counts.sum() - N * ptot) < 4 * np.sqrt(N * ptot * (1 - ptot))
    # per-facet chi^2 (merge cells with small expectation)
    big = expect > 20
    chi2 = ((counts[big] - expect[big]) ** 2 / expect[big]).sum()
    dof = int(big.sum())
    assert stats.chi2.sf(chi2, dof) > 1e-4
    # convex body: one hit per hitting particle
    assert r.hits == counts.sum() and r.truncated == 0 and r.segments == N + r.hits


# ------------------------------------------------------------------ P7, P8, P9: forces on convex bodies
def test_p8_config1_plate_vs_sentman():
    cfg = ti.config("C1")[0].with_(N=240000)
    om = omesh(cfg.mesh())
    r = om.run(cfg, use_bvh=False)
    se = r.force_stderr(cfg.N) / cfg.q_inf
    F = r.force / cfg.q_inf
    a = np.deg2rad(30)
    assert abs(-F[0] - cf.plate_cd(S1, SW1, a)) < 4 * se[0]
    assert abs(-F[1] - cf.plate_cl(S1, SW1, a)) < 4 * se[1]
    assert abs(F[2]) < 4 * se[2]                                   # P9
    assert abs(-F[0] - cf.plate_cd(S1, SW1, a, halved=False)) > 8 * se[0]   # G1: the printed eq. (3) is excluded
    assert se[0] / cf.plate_cd(S1, SW1, a) < 0.01
    assert r.hits / cfg.N == pytest.approx(0.242792, abs=4 * np.sqrt(0.2428 * 0.7572 / cfg.N))   # P6


@pytest.mark.parametrize("S", [2.0, 5.0, 8.0])
def test_p7_p8_sphere_vs_panel_sum_and_eq4(S):
    idx = [2.0, 5.0, 8.0].index(S)
    cfg = ti.config("C2")[idx].with_(N=100000, mesh_fn=lambda: ti.geodesic_sphere(8))
    cfg._mesh_cache = []
    m = cfg.mesh()
    om = omesh(m)
    r = om.run(cfg)
    se = r.force_stderr(cfg.N) / cfg.q_inf
    F = r.force / cfg.q_inf
    Fp, _, _ = cf.panel_sum(m.triangles(), m.flags, [1, 0, 0], S, SW1)
    assert np.all(np.abs(F - Fp) < 4 * se)                          # P7 (+ P9: lateral components)
    assert -Fp[0] / np.pi == pytest.approx(cf.sphere_cd(S, SW1), rel=0.03)   # faceted f=8 vs smooth eq. (4)
    assert abs(-F[0] / np.pi - cf.sphere_cd(S, SW1)) < 4 * se[0] / np.pi + 0.03 * cf.sphere_cd(S, SW1)


@pytest.mark.parametrize("ang", [0.0, 45.0, 90.0])
def test_p7_cylinder_maxwell_mix_vs_panel_sum(ang):
    idx = [0.0, 45.0, 90.0].index(ang)
    cfg = ti.config("C3")[idx].with_(N=100000, mesh_fn=lambda: ti.cylinder(0.5, 2.0, 24, 1))
    cfg._mesh_cache = []
    m = cfg.mesh()
    om = omesh(m)
    r = om.run(cfg, use_bvh=False)
    se = r.force_stderr(cfg.N) / cfg.q_inf
    F = r.force / cfg.q_inf
    up = -np.array(cfg.V) / cfg.speed
    Fp, _, _ = cf.panel_sum(m.triangles(), m.flags, up, S1, SW1, sigma=0.8)
    assert np.all(np.abs(F - Fp) < 4 * se)
    if ang == 0.0:                                                  # config 3's invariant
        assert abs(F[0]) < 4 * se[0] and abs(F[1]) < 4 * se[1]


def test_p7_mixture_on_convex_body():
    # A8: species by number fraction, weight m_s Gamma_s / N
    base = ti.config("C5")[3]
    cfg = base.with_(N=100000, mesh_fn=lambda: ti.geodesic_sphere(4))
    cfg._mesh_cache = []
    m = cfg.mesh()
    om = omesh(m)
    r = om.run(cfg)
    se = r.force_stderr(cfg.N)
    up = -np.array(cfg.V) / cfg.speed
    Fexp = np.zeros(3)
    for ms, xs in zip(cfg.m, cfg.x):
        S = cfg.speed / cf.thermal_speed(cfg.T_inf, ms)
        SW = cfg.speed / cf.thermal_speed(cfg.T_W, ms)
        Fp, _, _ = cf.panel_sum(m.triangles(), m.flags, up, S, SW)
        Fexp += Fp * 0.5 * cfg.n * xs * ms * cfg.speed ** 2
    assert np.all(np.abs(r.force - Fexp) < 4 * se)


# ------------------------------------------------------------------ P15: the standard error itself
def test_p15_standard_error_against_batch_scatter_and_the_papers_figure():
    """Every 4-sigma pin above leans on force_stderr (O14, from the sum of squared per-particle forces).  Pin it to
    something it is not computed from: the scatter of the forces of disjoint batches of the same stream.  With B batches
    of n particles the total is the sum of the batch forces, so its variance is B x the sample variance of those; the
    estimate from 64 batches has a relative standard deviation of 1/sqrt(2 x 63) = 9 %, and 25 % is asked for.  And the
    paper's own number: 'a particle count of 10 million (providing a statistical scatter of approximately 0.07 % for the
    comparison with the flat-plate analytical solution': scaled to 1e7 particles by 1/sqrt(N)."""
    B, n = 64, 12_500
    cfg = ti.config("C1")[0].with_(N=B * n)
    om = omesh(cfg.mesh())
    parts = [om.run(cfg, first=b * n, count=n, use_bvh=False, debug=False, facets=False) for b in range(B)]
    Fb = np.array([r.force for r in parts])
    F = Fb.sum(0)
    se_batches = np.sqrt(B * Fb.var(axis=0, ddof=1))
    whole = parts[0]
    fsq = sum(r.force_sq for r in parts)
    var = fsq - F ** 2 / cfg.N                                     # Result.force_stderr, written out for the summed slices
    se = np.sqrt(var * cfg.N / (cfg.N - 1))
    full = om.run(cfg, use_bvh=False, debug=False, facets=False)
    assert np.allclose(full.force, F, rtol=1e-12) and np.allclose(full.force_stderr(cfg.N), se, rtol=1e-9)
    for a in (0, 1):                                               # drag and lift; the third component is pure noise too:
        assert abs(se[a] / se_batches[a] - 1.0) < 0.25, (a, se[a], se_batches[a])
    assert abs(se[2] / se_batches[2] - 1.0) < 0.25
    rel_1e7 = se[0] / abs(F[0]) * np.sqrt(cfg.N / 1e7)
    assert 0.03e-2 < rel_1e7 < 0.15e-2, rel_1e7                    # the paper: ~0.07 %
    assert whole.hits > 0


# ------------------------------------------------------------------ P10: equilibrium, through multiple reflections
def test_p10_equilibrium_pressure_inside_cavity():
    m = ti.satellite(seed=2, h=0.25)        # coarse concave satellite with the open pocket
    om = omesh(m)
    T = 500.0
    cfg = ti.RunConfig("eq", None, T_inf=T, T_W=T, V=(0.0, 0.0, 0.0), N=480000, seed=5, cv_radius_factor=1.05)
    per = cfg.N // 8
    runs = [om.run(cfg, first=k * per, count=per) for k in range(8)]
    assert sum(r.truncated for r in runs) == 0
    assert max(int(r.bounces.max()) for r in runs) >= 3            # the pocket does give multiple reflections
    tri = m.triangles()
    Ng = np.cross(tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0])
    A = 0.5 * np.linalg.norm(Ng, axis=1)
    nh = Ng / (2 * A)[:, None]
    p = cfg.n * cf.K_B * T
    expect = -p * A[:, None] * nh                                   # P_f = -n k_B T A_f n_f on EVERY exposed facet
    cen = tri.mean(1)
    groups = {
        "pocket_floor": (np.abs(cen[:, 2] - 0.5) < 1e-6) & (np.abs(cen[:, 0]) < 0.31) & (np.abs(cen[:, 1]) < 0.31),
        "pocket_walls": (cen[:, 2] > 0.5) & (cen[:, 2] < 1.0) & (np.abs(cen[:, 0]) < 0.31) & (np.abs(cen[:, 1]) < 0.31)
                        & (np.abs(nh[:, 2]) < 0.5),
        "bus_bottom": np.abs(cen[:, 2] + 1.0) < 1e-6,
        "panel_faces": (np.abs(cen[:, 1]) > 0.55) & (np.abs(nh[:, 1]) < 0.5),
    }
    for name, g in groups.items():
        assert g.sum() > 0, name
        # signed normal force of the group, batch by batch
        vals = np.array([np.einsum("ij,ij->", r.facet_momentum[g], nh[g]) * 8 for r in runs])
        want = np.einsum("ij,ij->", expect[g], nh[g])
        se = vals.std(ddof=1) / np.sqrt(8)
        assert abs(vals.mean() - want) < 4 * se, (name, vals.mean(), want, se)
        assert se < 0.15 * abs(want), (name, se, want)
    Fs = np.array([r.force for r in runs]) * 8
    Ts = np.array([r.torque for r in runs]) * 8
    assert np.all(np.abs(Fs.mean(0)) < 4 * Fs.std(0, ddof=1) / np.sqrt(8))      # closed solid: zero net force
    assert np.all(np.abs(Ts.mean(0)) < 4 * Ts.std(0, ddof=1) / np.sqrt(8))      # and torque


# ------------------------------------------------------------------ P11: invariance
def test_p11_control_volume_and_rotation_invariance():
    m = ti.random_blob(3, 3)
    om = omesh(m)
    base = ti.RunConfig("inv", None, T_inf=1500.0, V=(-4000.0, 2000.0, 1000.0), N=160000, seed=9)
    ref, se_ref = batch_sigma(om, base)
    for fac in (1.2, 3.0):
        F, se = batch_sigma(om, base.with_(cv_radius_factor=fac))
        assert np.all(np.abs(F - ref) < 4 * np.hypot(se, se_ref)), fac
    # shifted mesh (centre moves with it) and rotated mesh + V
    sh = ti.Mesh(m.vertices + np.float32([0.5, -0.25, 0.125]), m.indices, m.flags)
    F, se = batch_sigma(omesh(sh), base)
    assert np.all(np.abs(F - ref) < 4 * np.hypot(se, se_ref))
    th = 0.7
    Rz = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1.0]])
    Rx = np.array([[1, 0, 0], [0, np.cos(1.1), -np.sin(1.1)], [0, np.sin(1.1), np.cos(1.1)]])
    Rot = Rz @ Rx
    F, se = batch_sigma(omesh(m.transformed(Rot)), base.with_(V=tuple(Rot @ np.array(base.V))))
    assert np.all(np.abs(Rot.T @ F - ref) < 4 * np.hypot(np.abs(Rot.T) @ se, se_ref) + 1e-30)


# ------------------------------------------------------------------ P12: BVH == brute force
@pytest.mark.parametrize("mesh_fn", [lambda: ti.plate(30.0), lambda: ti.random_blob(1, 2), lambda: ti.box(h=0.5),
                                      lambda: ti.satellite(1, 0.5), lambda: ti.cylinder(0.5, 2.0, 16, 2)])
def test_p12_bvh_equals_brute_force_including_edges_and_vertices(mesh_fn):
    m = mesh_fn()
    om = omesh(m)
    rng = np.random.default_rng(7)
    V = m.vertices.astype(np.float64)
    tri = m.triangles()
    ctr, Rb = om.bounds()
    targets = [V, 0.5 * (tri[:, 0] + tri[:, 1]), 0.5 * (tri[:, 1] + tri[:, 2]), tri.mean(1),
               ctr + rng.normal(size=(200, 3)) * Rb * 0.7]
    nhit = 0
    for T in targets:
        for tg in T[:150]:
            o = (ctr + 2.5 * Rb * (lambda d: d / np.linalg.norm(d))(rng.normal(size=3))).astype(np.float32)
            d = (tg - o.astype(np.float64)).astype(np.float32)
            for fprev in (-1, int(rng.integers(0, m.nt))):
                a = om.closest_hit(o, d, fprev, use_bvh=False)
                b = om.closest_hit(o, d, fprev, use_bvh=True)
                assert a == b
                nhit += a[0] >= 0
    # axis-parallel rays (zero direction components)
    for ax in range(3):
        for tg in tri.mean(1)[:50]:
            o = tg.copy(); o[ax] += 3 * Rb
            d = np.zeros(3); d[ax] = -1.0
            assert om.closest_hit(o, d, -1, False) == om.closest_hit(o, d, -1, True)
    assert nhit > 50


def test_p12_stream_rays_and_tie_rule():
    cfg = ti.config("C4")[5].with_(N=3000, mesh_fn=lambda: ti.satellite(4, 0.125))
    cfg._mesh_cache = []
    om = omesh(cfg.mesh())
    a = om.run(cfg, use_bvh=False)
    b = om.run(cfg, use_bvh=True)
    assert np.array_equal(a.hash, b.hash) and np.array_equal(a.bounces, b.bounces)
    assert np.array_equal(a.facet_momentum, b.facet_momentum)
    # A12: a ray through a shared edge of two coplanar facets reports the smaller facet index
    pl = ti.plate(0.0)
    op = omesh(pl)
    f, tau = op.closest_hit([2.0, 0.0, 0.0], [-1.0, 0.0, 0.0], -1, False)   # plate centre lies on the shared diagonal
    assert f == 0 and tau == pytest.approx(2.0)
    assert op.closest_hit([2.0, 0.0, 0.0], [-1.0, 0.0, 0.0], -1, True) == (f, tau)
    assert op.closest_hit([2.0, 0.0, 0.0], [-1.0, 0.0, 0.0], 0, False)[0] == 1    # source facet excluded (A11)
    # one-sided facets are invisible from behind; two-sided ones are not
    bx = omesh(ti.box(h=1.0))
    assert bx.closest_hit([0, 0, 0], [1, 0.1, 0.2], -1, False)[0] == -1
    assert op.closest_hit([-2.0, 0.1, 0.2], [1.0, 0.0, 0.0], -1, False)[0] >= 0


# ------------------------------------------------------------------ O11: surface interaction
def test_reflection_laws():
    m = ti.plate(0.0)                     # normal +x
    om = omesh(m)
    cfg = ti.RunConfig("r", None, accommodation=0.0)
    v = np.float32([-3.0, 1.0, 2.0])
    assert np.allclose(om.reflect(cfg, 0, v, 0, 0), [3.0, 1.0, 2.0])          # specular, front
    assert np.allclose(om.reflect(cfg, 0, -v, 0, 0), [-3.0, -1.0, -2.0])      # specular, back of a two-sided facet
    cfg = ti.RunConfig("r", None, accommodation=1.0, T_W=300.0)
    cw = cf.thermal_speed(300.0, cfg.m[0])
    out = np.array([om.reflect(cfg, 0, v, i, 0) for i in range(40000)]) / cw
    assert np.all(out[:, 0] > 0)
    # flux-weighted half-Maxwellian (A6): <v_n> = sqrt(pi)/2 c_W, <v_n^2> = c_W^2, tangentials N(0, 1/2)
    assert out[:, 0].mean() == pytest.approx(np.sqrt(np.pi) / 2, abs=4 * np.sqrt((1 - np.pi / 4) / 40000))
    assert (out[:, 0] ** 2).mean() == pytest.approx(1.0, abs=0.03)
    for k in (1, 2):
        assert out[:, k].mean() == pytest.approx(0.0, abs=4 * np.sqrt(0.5 / 40000))
        assert out[:, k].var() == pytest.approx(0.5, abs=0.02)
    assert stats.kstest(out[:, 0] ** 2, "expon").pvalue > 1e-3
    # from the back side the emission is into -x
    assert om.reflect(cfg, 0, -v, 1, 0)[0] < 0


# ------------------------------------------------------------------ P13: specular limits
def test_p13_specular_sphere_and_plate():
    mO = 16 * ti.AMU
    S = 50.0
    T = mO * (7500.0 / S) ** 2 / (2 * cf.K_B)
    cfg = ti.RunConfig("sp", lambda: ti.geodesic_sphere(8), T_inf=T, accommodation=0.0, N=60000, seed=2)
    m = cfg.mesh()
    r = omesh(m).run(cfg)
    se = r.force_stderr(cfg.N) / cfg.q_inf
    Fp, _, _ = cf.panel_sum(m.triangles(), m.flags, [1, 0, 0], S, S * np.sqrt(T / 300.0), sigma=0.0)
    assert np.all(np.abs(r.force / cfg.q_inf - Fp) < 4 * se)
    assert -Fp[0] / np.pi == pytest.approx(2.0, rel=0.03)
    cfgp = ti.RunConfig("pp", lambda: ti.plate(0.0), T_inf=T, accommodation=0.0, N=60000, seed=3)
    rp = omesh(cfgp.mesh()).run(cfgp, use_bvh=False)
    sep = rp.force_stderr(cfgp.N) / cfgp.q_inf
    assert abs(-rp.force[0] / cfgp.q_inf - 4.0) < 4 * sep[0] + 0.01   # broadside specular plate: C_D -> 4


def test_p14_concave_hemisphere_approaches_pratt():
    """NEXT-2 / P14: the paper's own multi-reflection check (Fig. 6).  A two-sided
    hemispherical shell, concave side to the stream, at the paper's verification temperatures (922 K / 300 K,
    PAPER.md:223): C_D approaches eq. (5) "asymptotically" as S grows.  Re-emitted molecules hit the shell again
    (0.70 hits per particle against a hit fraction of 0.44): a wrong reflection loop or re-emission law moves the
    re-emission term eps_D sqrt(pi)/S sqrt(T_W/T_inf), which is 5 % of C_D at S = 10."""
    m = ti.hemisphere_shell(16)
    om = omesh(m)
    mO, T_inf, T_W, N = 16 * ti.AMU, 922.0, 300.0, 300_000
    dev = {}
    for S in (10.0, 20.0, 40.0):
        speed = S * cf.thermal_speed(T_inf, mO)
        cfg = ti.RunConfig("shell", lambda: m, T_inf=T_inf, T_W=T_W, V=(-speed, 0.0, 0.0), N=N, A_ref=float(np.pi), seed=14)
        r = om.run(cfg, facets=False)
        q = cfg.q_inf * np.pi
        cd, se = -r.force[0] / q, r.force_stderr(N)[0] / q
        ref = cf.pratt_hemisphere_cd(S, T_W / T_inf)
        dev[S] = (cd - ref, se)
        assert r.truncated == 0 and r.hits > 0.6 * N                 # multiple reflections do happen
        assert abs(r.force[1]) < 4 * r.force_stderr(N)[1] + 1e-3 * abs(r.force[0])   # axisymmetric: no side force
        assert abs(cd - ref) < 4 * se + (0.012 if S < 15 else 0.006) * ref
    # the thermal excess over the hyperthermal asymptote shrinks with S
    assert dev[10.0][0] > dev[40.0][0] - 4 * (dev[10.0][1] + dev[40.0][1])
    assert dev[10.0][0] > 0.0


# ------------------------------------------------------------------ O12 / A14: torque and its reference point
def _batched_torque(om, cfg, nb=8):
    """Force and torque of the whole stream with the standard error of the torque from nb disjoint slices."""
    per = cfg.N // nb
    rs = [om.run(cfg, first=k * per, count=per, debug=False, facets=False) for k in range(nb)]
    Ts = np.array([r.torque for r in rs])
    Fs = np.array([r.force for r in rs])
    return Fs.sum(0), Ts.sum(0), Ts.std(0, ddof=1) * np.sqrt(nb)


@pytest.mark.parametrize("body", ["sphere", "plate"])
def test_p16_torque_about_an_off_centre_point_vs_panel_sum(body):
    """O12: tau = sum (p - x_ref) x dp with p the HIT point (moments about a reference point).  On a
    convex mesh every facet sees a uniform incident flux and a uniform re-emission, so the expected torque is
    sum_f (centroid_f - x_ref) x F_f with F_f the panel force of the facet -- non-zero here because x_ref is off
    the line of action.  A swapped cross product, the segment origin in place of the hit point, or an ignored
    x_ref all move the result by many sigma."""
    x_ref = np.array([0.3, -0.2, 0.5])
    if body == "sphere":
        m = ti.geodesic_sphere(4)
        cfg = ti.RunConfig("tq", None, T_inf=1200.0, V=(-5200.0, 3100.0, -4300.0), N=160_000, seed=21,
                           x_ref=tuple(x_ref))
    else:
        m = ti.plate(30.0)               # two-sided canted plate; reference point like a quarter-chord point, off the plate
        cfg = ti.config("C1")[0].with_(N=240_000, seed=22, x_ref=tuple(x_ref))
    om = omesh(m)
    F, Tq, seT = _batched_torque(om, cfg)
    up = -np.array(cfg.V) / cfg.speed
    S = cfg.speed / cf.thermal_speed(cfg.T_inf, cfg.m[0])
    SW = cfg.speed / cf.thermal_speed(cfg.T_W, cfg.m[0])
    _, _, Fpf = cf.panel_sum(m.triangles(), m.flags, up, S, SW)
    cen = m.triangles().mean(1)
    want = np.cross(cen - x_ref, Fpf * cfg.q_inf).sum(0)
    assert np.all(np.abs(Tq - want) < 4 * seT), (Tq, want, seT)
    assert np.linalg.norm(want) > 30 * np.linalg.norm(seT)          # the pin has teeth: the expected torque is far from 0
    # the mistakes it must catch, each evaluated from the same expectation
    assert np.linalg.norm(-want - Tq) > 8 * np.linalg.norm(seT)                                   # dp x r
    about_origin = np.cross(cen, Fpf * cfg.q_inf).sum(0)
    assert np.linalg.norm(about_origin - Tq) > 8 * np.linalg.norm(seT)                            # x_ref ignored


def test_a14_moving_the_reference_point():
    """A14: tau(x_ref + dx) = tau(x_ref) - dx x F on the same particle stream, to rounding; per-facet momentum and
    force do not depend on x_ref."""
    m = ti.satellite(seed=2, h=0.25)
    om = omesh(m)
    base = ti.RunConfig("a14", None, T_inf=900.0, V=(-4000.0, 1500.0, -6000.0), N=40_000, seed=23)
    a = om.run(base)
    dx = np.array([0.7, -1.1, 0.4])
    b = om.run(base.with_(x_ref=tuple(dx)))
    assert np.array_equal(a.force, b.force) and np.array_equal(a.facet_momentum, b.facet_momentum)
    scale = np.linalg.norm(dx) * np.linalg.norm(a.force) + np.linalg.norm(a.torque)
    assert np.linalg.norm(b.torque - (a.torque - np.cross(dx, a.force))) <= 1e-11 * scale
    assert np.linalg.norm(np.cross(dx, a.force)) > 1e-3 * scale       # the shift is not a no-op


# ------------------------------------------------------------------ P17: surface models beyond one global T_W, sigma (NEXT-3)
def test_p17_quadrature_reduces_to_the_panel_term():
    # the reference of the alpha_E pin is itself pinned: alpha_E = 1 must give chi(s) / (2 S S_W)
    for S, SW, g in ((7.356804, 13.431624, 0.8660254), (2.0, 5.0, 0.3), (5.0, 9.0, -0.2)):
        want = float(cf.chi(S * g)) / (2 * S * SW)
        assert cf.reemission_pressure_alpha_e(S, SW, g, 1.0) == pytest.approx(want, rel=1e-9)


def test_p17_per_facet_wall_temperature_and_accommodation_vs_panel_sum():
    """A23: T_W and sigma per facet.  On a convex body the expectation is still the panel sum, now with S_W,f and
    sigma_f per facet; hot/cold halves give a side force that a global T_W cannot."""
    m = ti.geodesic_sphere(4)
    cen = m.triangles().mean(1)
    TW = np.where(cen[:, 1] > 0, 200.0, 1500.0)
    sg = np.where(cen[:, 2] > 0, 1.0, 0.5)
    om = omesh(m)
    om.set_surface(TW, sg)
    cfg = ti.RunConfig("surf", None, T_inf=1000.0, T_W=300.0, accommodation=1.0, N=200_000, seed=51)
    r = om.run(cfg, use_bvh=False)
    se = r.force_stderr(cfg.N) / cfg.q_inf
    F = r.force / cfg.q_inf
    S = cfg.speed / cf.thermal_speed(cfg.T_inf, cfg.m[0])
    SWf = cfg.speed / cf.thermal_speed(TW, cfg.m[0])
    Fp, _, _ = cf.panel_sum(m.triangles(), m.flags, [1, 0, 0], S, SWf, sigma=sg)
    assert np.all(np.abs(F - Fp) < 4 * se), (F, Fp, se)
    Fu, _, _ = cf.panel_sum(m.triangles(), m.flags, [1, 0, 0], S, cfg.speed / cf.thermal_speed(300.0, cfg.m[0]), sigma=1.0)
    assert abs(Fp[1] - Fu[1]) > 8 * se[1] and abs(Fp[2] - Fu[2]) > 8 * se[2]     # the arrays matter: side forces appear
    # NULL arrays fall back to the run's scalars; uniform arrays equal to the scalars change nothing, bit for bit
    om.set_surface(None, None)
    a = om.run(cfg.with_(N=20_000), use_bvh=False)
    om.set_surface(np.full(m.nt, 300.0), np.full(m.nt, 1.0))
    b = om.run(cfg.with_(N=20_000), use_bvh=False)
    assert np.array_equal(a.force, b.force) and np.array_equal(a.hash, b.hash) and np.array_equal(a.facet_momentum, b.facet_momentum)


@pytest.mark.parametrize("alpha_e", [0.5, 0.0])
def test_p17_energy_accommodation_vs_quadrature(alpha_e):
    """A22: re-emission at T_r = alpha_E T_W + (1 - alpha_E) m v_in^2 / (3 k_B), per particle.  On the C1 plate the
    expected force is the incident part of the panel sum plus the re-emission pressure integrated over the incident
    flux (closed_forms.reemission_pressure_alpha_e); full accommodation (the paper's case) is many sigma away."""
    cfg = ti.config("C1")[0].with_(N=240_000, seed=52, energy_accommodation=alpha_e)
    m = cfg.mesh()
    r = omesh(m).run(cfg, use_bvh=False)
    se = r.force_stderr(cfg.N) / cfg.q_inf
    F = r.force / cfg.q_inf
    up = -np.array(cfg.V) / cfg.speed
    tri = m.triangles()
    Ng = np.cross(tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0])
    A = 0.5 * np.linalg.norm(Ng, axis=1)
    n0 = Ng / (2 * A)[:, None]
    Finc, _, _ = cf.panel_sum(tri, m.flags, up, S1, 1e30)              # incident momentum only (no re-emission term)
    want = Finc.copy()
    for side in (+1.0, -1.0):                                          # two-sided sheet: both faces re-emit
        for f in range(m.nt):
            g = float(side * n0[f] @ up)
            want += -A[f] * cf.reemission_pressure_alpha_e(S1, SW1, g, alpha_e) * side * n0[f]
    assert np.all(np.abs(F - want) < 4 * se), (F, want, se)
    Ffull, _, _ = cf.panel_sum(tri, m.flags, up, S1, SW1)
    assert abs(want[0] - Ffull[0]) > 30 * se[0]
    # alpha_E = 1 is the scalar model, bit for bit
    a = omesh(m).run(cfg.with_(N=20_000, energy_accommodation=1.0), use_bvh=False)
    b = omesh(m).run(ti.config("C1")[0].with_(N=20_000, seed=52), use_bvh=False)
    assert np.array_equal(a.force, b.force) and np.array_equal(a.hash, b.hash)


def test_p17_equilibrium_with_per_facet_arrays():
    """P10 again with the wall temperature given per facet (all equal to T_inf) and alpha_E = 1: per-facet pressure
    -n k_B T A_f n_f on the pocket floor and zero net force, through any number of reflections."""
    m = ti.satellite(seed=2, h=0.25)
    om = omesh(m)
    T = 500.0
    om.set_surface(np.full(m.nt, T), np.ones(m.nt))
    cfg = ti.RunConfig("eq", None, T_inf=T, T_W=123.0, accommodation=0.3, V=(0.0, 0.0, 0.0), N=240_000, seed=5, cv_radius_factor=1.05)
    per = cfg.N // 8
    runs = [om.run(cfg, first=k * per, count=per) for k in range(8)]
    tri = m.triangles()
    Ng = np.cross(tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0])
    A = 0.5 * np.linalg.norm(Ng, axis=1)
    nh = Ng / (2 * A)[:, None]
    cen = tri.mean(1)
    g = (np.abs(cen[:, 2] - 0.5) < 1e-6) & (np.abs(cen[:, 0]) < 0.31) & (np.abs(cen[:, 1]) < 0.31)
    vals = np.array([np.einsum("ij,ij->", r.facet_momentum[g], nh[g]) * 8 for r in runs])
    want = -cfg.n * cf.K_B * T * A[g].sum()
    se = vals.std(ddof=1) / np.sqrt(8)
    assert abs(vals.mean() - want) < 4 * se and se < 0.2 * abs(want)
    Fs = np.array([r.force for r in runs]) * 8
    assert np.all(np.abs(Fs.mean(0)) < 4 * Fs.std(0, ddof=1) / np.sqrt(8))


# ------------------------------------------------------------------ P18: rectangular control volume (NEXT-4)
def test_p18_unweighted_normal_speed_inverse():
    from scipy import special
    for s in (-3.0, -0.5, 0.0, 1.0, 7.4):
        for u in (1e-6, 0.01, 0.3, 0.77, 0.999):
            want = s + special.erfcinv((1.0 - u) * special.erfc(-s))
            assert oracle.vn_unweighted_inv(u, s) == pytest.approx(want, rel=1e-9, abs=1e-12)


def _drag_over_q(om, cfg):
    r = om.run(cfg, use_bvh=True, facets=False)
    up = -np.array(cfg.V) / cfg.speed
    return r, (r.force / cfg.q_inf) @ (-up), np.linalg.norm(r.force_stderr(cfg.N) / cfg.q_inf)


def test_p18_box_control_volume_exact_and_negative_control():
    """The scheme the paper replaces: uniform seeding on the six faces of a box, the share of each face from the
    flat-plate flux.  Done consistently (inward speed from the flux-weighted law (14a), reading A24) it is exact: the
    force on a convex body is the panel sum at any attitude, the hit count is N Gamma_body / Gamma_box, and it agrees
    with the spherical scheme.  With the inward speed drawn WITHOUT the flux weight (reading A25, the negative
    control) the drag depends on the attitude of the stream to the box, as in the paper's Fig. 1."""
    m = ti.geodesic_sphere(4)
    om = omesh(m)
    dev = {}
    for ang in (0.0, 45.0):
        a = np.deg2rad(ang)
        V = (-7500.0 * np.cos(a), -7500.0 * np.sin(a), 0.0)
        up = -np.array(V) / 7500.0
        Fp, flux, _ = cf.panel_sum(m.triangles(), m.flags, up, S1, SW1)
        want = Fp @ (-up)
        cfg = ti.RunConfig("box", None, V=V, N=400_000, seed=61, control_volume=1)
        r, drag, se = _drag_over_q(om, cfg)
        assert abs(drag - want) < 4 * se, (ang, drag, want, se)
        # share of the box flux that reaches the body: sum_f Gamma_f / Gamma_box (every hit is a first hit: convex)
        h = 1.5 * 0.5 * (m.vertices.max(0) - m.vertices.min(0)).astype(np.float64)
        gbox = 0.0
        for ax in range(3):
            area = 4.0 * h[(ax + 1) % 3] * h[(ax + 2) % 3]
            for sgn in (+1.0, -1.0):
                gbox += area * float(cf.chi(S1 * sgn * V[ax] / 7500.0)) / (2 * np.sqrt(np.pi))
        pin = flux.sum() / gbox
        assert abs(r.hits - cfg.N * pin) < 4 * np.sqrt(cfg.N * pin * (1 - pin))
        rs, drag_s, se_s = _drag_over_q(om, cfg.with_(control_volume=0))
        assert abs(drag - drag_s) < 4 * np.hypot(se, se_s)               # box and sphere schemes agree
        ru, drag_u, se_u = _drag_over_q(om, cfg.with_(control_volume=2))
        dev[ang] = ((drag_u - want) / want, se_u / want)
    # negative control: biased at 45 deg by several sigma, and the bias changes with the attitude
    assert abs(dev[45.0][0]) > 5 * dev[45.0][1]
    assert abs(dev[45.0][0] - dev[0.0][0]) > 4 * np.hypot(dev[45.0][1], dev[0.0][1])


# ------------------------------------------------------------------ the oracle under AddressSanitizer + UBSan
def test_oracle_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """oracle/tpmc_oracle.c rebuilt with -fsanitize=address,undefined -fno-sanitize-recover=all and run, in a child
    process with the sanitizer runtime preloaded, through every entry point on small workloads (plate, two-sided shell
    with multiple reflections, mixture, per-facet surface arrays, both box schemes, brute force and BVH): any
    out-of-bounds access, use after free, signed overflow, misaligned access or invalid shift aborts the child."""
    import subprocess, sys, os, textwrap
    import oracle as orc
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("no libasan in this toolchain")
    lib = orc.build_sanitized(str(tmp_path / "liboracle_san.so"))
    code = textwrap.dedent("""
        import numpy as np, oracle, tpmc_inputs as ti
        assert oracle.philox4x32_10((1, 2), (3, 4, 5, 6))
        oracle.flux_bracket(5.0); oracle.position_inv(0.3, 7.0); oracle.vn_inv(0.9, -1.5); oracle.vn_unweighted_inv(0.2, 2.0)
        oracle.rotation((1.0, 2.0, -3.0))
        cases = [ti.config("C1")[0].with_(N=4000),
                 ti.RunConfig("shell", lambda: ti.hemisphere_shell(4), N=4000, seed=3, label="shell"),
                 ti.config("C5")[5].with_(N=3000, mesh_fn=lambda: ti.large_body(5, 6)),
                 ti.config("C4")[3].with_(N=3000, mesh_fn=lambda: ti.satellite(4, 0.25), control_volume=1),
                 ti.config("C2")[0].with_(N=3000, mesh_fn=lambda: ti.geodesic_sphere(3), control_volume=2, energy_accommodation=0.5)]
        for k, cfg in enumerate(cases):
            cfg._mesh_cache = []
            m = cfg.mesh()
            om = oracle.OracleMesh(m.vertices, m.indices, m.flags)
            if k == 4:
                om.set_surface(np.full(m.nt, 350.0), np.linspace(0.0, 1.0, m.nt))
            a = om.run(cfg, first=0, count=cfg.N, use_bvh=True)
            b = om.run(cfg, first=0, count=cfg.N, use_bvh=False)
            assert a.hits == b.hits and np.array_equal(a.hash, b.hash)
            om.seed(cfg, 0, 16)
            del om
        print("sanitized ok")
    """)
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1",
               TPMC_ORACLE_LIB=lib, PYTHONPATH=os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0 and "sanitized ok" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
