"""The closed forms in tests/closed_forms.py against the numbers the paper's formulas give
(tests/golden/closed_form_values.txt) and against one another -- so that the references used
to pin the oracle are themselves pinned.  Pure numpy/scipy; no oracle, no GPU."""
import numpy as np
import pytest

import closed_forms as cf
import tpmc_inputs as ti

S1, SW1 = 7.356804, 13.431624   # config 1: O at 1000 K / 300 K, 7500 m/s


def test_config1_speed_ratios():
    m = 16 * ti.AMU
    assert 7500 / cf.thermal_speed(1000.0, m) == pytest.approx(S1, rel=1e-6)
    assert 7500 / cf.thermal_speed(300.0, m) == pytest.approx(SW1, rel=1e-6)


def test_flux_bracket_golden_and_limits():
    for S, v in cf.golden("flux_bracket").items():
        assert cf.flux_bracket_quadrature(S) == pytest.approx(v, rel=1e-10)
    # limits of eq. (10): S->0: 2 sqrt(pi); S->inf: pi S
    assert cf.flux_bracket_quadrature(1e-6) == pytest.approx(2 * np.sqrt(np.pi), rel=1e-6)
    assert cf.flux_bracket_quadrature(60.0) / (np.pi * 60.0) == pytest.approx(1.0, rel=2e-4)


def test_eq11_normalised_and_lee_side_mass():
    for S, v in cf.golden("p_lee").items():
        assert cf.phi_cdf_quadrature(np.pi / 2, S) == pytest.approx(1.0, abs=1e-10)
        assert cf.phi_cdf_quadrature(0.0, S) == pytest.approx(v, rel=2e-6)


def test_plate_golden_and_g1():
    a = np.deg2rad(30)
    assert cf.plate_cd(S1, SW1, a) == pytest.approx(cf.golden("plate_CD")[30], abs=2e-6)
    assert cf.plate_cl(S1, SW1, a) == pytest.approx(cf.golden("plate_CL")[30], abs=2e-6)
    assert cf.plate_cd(S1, SW1, a, halved=False) == pytest.approx(cf.golden("plate_CD_printed_eq3")[30], abs=2e-6)
    # G1: hyperthermal plate normal to the stream must give 2 + sqrt(pi)/S_W
    assert cf.plate_cd(200.0, 50.0, 0.0) == pytest.approx(2 + np.sqrt(np.pi) / 50.0, rel=1e-4)


def test_sphere_golden():
    m = 16 * ti.AMU
    for S, v in cf.golden("sphere_CD").items():
        assert cf.sphere_cd(S, SW1) == pytest.approx(v, abs=2e-6)
        T = ti.config("C2")[[2.0, 5.0, 8.0].index(S)].T_inf
        assert 7500 / cf.thermal_speed(T, m) == pytest.approx(S, rel=1e-12)


def test_panel_sum_reproduces_plate_sphere_cylinder():
    a = np.deg2rad(30)
    pl = ti.plate(30.0)
    F, flux, _ = cf.panel_sum(pl.triangles(), pl.flags, [1, 0, 0], S1, SW1)
    assert -F[0] == pytest.approx(cf.plate_cd(S1, SW1, a), rel=1e-6)
    assert -F[1] == pytest.approx(cf.plate_cl(S1, SW1, a), rel=1e-5)
    assert abs(F[2]) < 1e-12
    # eq. (4) is eq. (3) integrated over the sphere: fine mesh -> smooth value
    sp = ti.geodesic_sphere(48)
    for S in (2.0, 5.0, 8.0):
        F, _, _ = cf.panel_sum(sp.triangles(), sp.flags, [0, 0, 1], S, SW1)
        assert -F[2] / np.pi == pytest.approx(cf.sphere_cd(S, SW1), rel=1.5e-3)   # faceting ~ 1/freq^2
    # smooth capped cylinder values of BASELINE.md (config 3, sigma = 0.8)
    cy = ti.cylinder(0.5, 2.0, 2048, 1)
    for ang, want in cf.golden("cyl_drag").items():
        an = np.deg2rad(ang)
        up = np.array([np.sin(an), 0.0, np.cos(an)])
        F, _, _ = cf.panel_sum(cy.triangles(), cy.flags, up, S1, SW1, sigma=0.8)
        assert -F @ up == pytest.approx(want, rel=2e-5)
        side = np.linalg.norm(F - (F @ up) * up)
        assert side == pytest.approx(cf.golden("cyl_side").get(ang, 0.0), abs=3e-5)


def test_cylinder_crossflow_closed_form():
    # side facets only of a long cylinder in cross-flow, A_ref = 2 R L
    cy = ti.cylinder(0.5, 2.0, 4096, 1)
    tri = cy.triangles()
    n = np.cross(tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0])
    side = np.abs(n[:, 2]) < 1e-9 * np.linalg.norm(n, axis=1)
    for S in (2.0, S1):
        F, _, _ = cf.panel_sum(tri[side], cy.flags[side], [1, 0, 0], S, SW1)
        assert -F[0] / 2.0 == pytest.approx(cf.cylinder_crossflow_cd(S, SW1), rel=1e-5)


def test_pratt_concave_hemisphere_golden():
    for S, v in cf.golden("shell_CD").items():
        assert cf.pratt_hemisphere_cd(S, 300.0 / 922.0) == pytest.approx(v, abs=2e-6)
    assert cf.pratt_hemisphere_cd(1e9, 0.3) == pytest.approx(2.0, abs=1e-8)
