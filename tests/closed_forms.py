"""Free-molecular closed forms used to pin the oracle (independent of oracle/ and of the CUDA path).

Sources: PAPER.md eq. (3) :85 (Sentman plate; third term halved, reading G1), eq. (4) :93
(sphere), eq. (8) :141-143 / eq. (10) :151-154 (flux), eq. (11) :158, eq. (14a) :194; the
standard flat-element ("panel") coefficients of free-molecular theory (Sentman 1961;
Schaaf & Chambre 1961), written out in SURVEY.md 8(c) "What pins the oracle".
"""
from __future__ import annotations

import os

import numpy as np
from scipy import integrate, special

SQRTPI = np.sqrt(np.pi)
K_B = 1.380649e-23


def golden(name):
    """Rows of tests/golden/closed_form_values.txt for one name -> {key: value}."""
    out = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "closed_form_values.txt")
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        n, k, v = line.split()
        if n == name:
            out[float(k)] = float(v)
    return out


def chi(s):
    """Bracket of eq. (8): e^{-s^2} + sqrt(pi) s (1 + erf s)."""
    s = np.asarray(s, dtype=np.float64)
    return np.exp(-s * s) + SQRTPI * s * special.erfc(-s)


# ------------------------------------------------------------------ eq. (8)/(10): flux into the sphere
def flux_bracket_quadrature(S):
    """Gamma/(c n r^2) by direct quadrature of eq. (8) over the sphere."""
    # Gamma = n/(c^2 pi)^{3/2} * int (1/2) c^2 pi (c^2 e^{-u^2/c^2} + sqrt(pi) u c [1+erf(u/c)]) r^2 cos(phi) dtheta dphi
    # => Gamma/(c n r^2) = (1/(2 sqrt(pi))) * 2 pi * int_{-pi/2}^{pi/2} chi(S sin phi) cos(phi) dphi
    val, _ = integrate.quad(lambda ph: float(chi(S * np.sin(ph))) * np.cos(ph), -np.pi / 2, np.pi / 2,
                            epsabs=1e-13, epsrel=1e-13, limit=200)
    return SQRTPI * val


# ------------------------------------------------------------------ eq. (11): incidence-angle likelihood
def g_phi(phi, S):
    """eq. (11) exactly as printed (with 1+erf)."""
    num = np.cos(phi) * (np.exp(-(S * np.sin(phi)) ** 2) + S * SQRTPI * np.sin(phi) * (1 + special.erf(S * np.sin(phi))))
    den = np.exp(-S * S) + SQRTPI * (1 + 2 * S * S) * special.erf(S) / (2 * S)
    return num / den


def phi_cdf_quadrature(phi, S):
    val, _ = integrate.quad(lambda p: float(g_phi(p, S)), -np.pi / 2, phi, epsabs=1e-13, epsrel=1e-12, limit=200)
    return val


# ------------------------------------------------------------------ eq. (14a): inward normal speed (in x = v_n/c)
def pvn(x, s):
    return 2 * x * np.exp(-(x - s) ** 2) / float(chi(s))


def vn_cdf_quadrature(x, s):
    val, _ = integrate.quad(lambda y: float(pvn(y, s)), 0.0, x, epsabs=1e-14, epsrel=1e-12, limit=200)
    return val


def vn_mean(s):
    """E[x_n] of eq. (14a)."""
    return (s * np.exp(-s * s) + SQRTPI * (0.5 + s * s) * special.erfc(-s)) / float(chi(s))


# ------------------------------------------------------------------ eqs. (3), (4) and friends
def plate_cd(S, S_W, alpha, halved=True):
    """eq. (3) (double-sided plate, A_ref = plate area); halved=True is reading G1."""
    ca = np.cos(alpha)
    third = (np.pi * S / S_W) * ca * ca * (0.5 if halved else 1.0)
    return (2 / (SQRTPI * S)) * (np.exp(-(S * ca) ** 2) + SQRTPI * S * ca * (1 + 1 / (2 * S * S)) * special.erf(S * ca) + third)


def plate_cl(S, S_W, alpha):
    return np.sin(alpha) * (special.erf(S * np.cos(alpha)) / S ** 2 + SQRTPI * np.cos(alpha) / S_W)


def sphere_cd(S, S_W):
    """eq. (4), A_ref = pi R^2."""
    return (np.exp(-S * S) / (SQRTPI * S ** 3) * (1 + 2 * S * S) + (4 * S ** 4 + 4 * S * S - 1) / (2 * S ** 4) * special.erf(S)
            + 2 * SQRTPI / (3 * S_W))


def pratt_hemisphere_cd(S, Tw_over_Tinf, eps_d=1.05349):
    """Concave hemispherical shell in hyperthermal flow, eq. (5) PAPER.md:100 with eps_D(90 deg) = 1.05349
    (PAPER.md:103); A_ref = pi R^2.  An asymptote for S -> inf."""
    return 2.0 + eps_d * np.sqrt(np.pi) / S * np.sqrt(Tw_over_Tinf)


def cylinder_crossflow_cd(S, S_W):
    """Infinite cylinder normal to the stream, diffuse, A_ref = 2 R L (Schaaf & Chambre form)."""
    h = 0.5 * S * S
    return (SQRTPI / S) * np.exp(-h) * ((S * S + 1.5) * special.iv(0, h) + (S * S + 0.5) * special.iv(1, h)) + np.pi ** 1.5 / (4 * S_W)


# ------------------------------------------------------------------ panel sum (exact expectation for convex bodies)
def panel_sum(tri, flags, upstream, S, S_W, sigma=1.0):
    """F/q [m^2] and per-facet expected incident number flux / (n c) [m^2] for a convex mesh.

    tri: [nt,3,3] corner coordinates; flags bit0 = two-sided; upstream: unit vector z~ = -V/|V|.
    Per one-sided element with outward normal n, gamma = n.z~, s = S gamma, in units of q = rho V^2/2:
      p_i = [s e^{-s^2}/sqrt(pi) + (1/2+s^2) erfc(-s)]/S^2, tau_i = sqrt(1-gamma^2) chi(s)/(sqrt(pi) S),
      p_r = chi(s)/(2 S S_W); Maxwell mix: pressure sigma(p_i+p_r) + (1-sigma) 2 p_i, shear sigma tau_i.
    """
    tri = np.asarray(tri, dtype=np.float64)
    z = np.asarray(upstream, dtype=np.float64)
    z = z / np.linalg.norm(z)
    Ng = np.cross(tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0])
    A = 0.5 * np.linalg.norm(Ng, axis=1)
    n0 = Ng / (2 * A)[:, None]
    F = np.zeros(3)
    flux = np.zeros(tri.shape[0])
    Fpf = np.zeros((tri.shape[0], 3))
    for side in (+1.0, -1.0):
        n = side * n0
        act = np.ones(tri.shape[0], dtype=bool) if side > 0 else (np.asarray(flags) & 1).astype(bool)
        gamma = n @ z
        s = S * gamma
        c = chi(s)
        p_i = (s * np.exp(-s * s) / SQRTPI + (0.5 + s * s) * special.erfc(-s)) / S ** 2
        tau_i = np.sqrt(np.maximum(0.0, 1 - gamma ** 2)) * c / (SQRTPI * S)
        p_r = c / (2 * S * S_W)
        pres = sigma * (p_i + p_r) + (1 - sigma) * 2 * p_i
        shear = sigma * tau_i
        vhat = -z
        tvec = vhat[None, :] + gamma[:, None] * n          # V^ - (V^.n) n, V^.n = -gamma
        tn = np.linalg.norm(tvec, axis=1)
        that = np.where(tn[:, None] > 1e-300, tvec / np.maximum(tn, 1e-300)[:, None], 0.0)
        f = A[:, None] * (-pres[:, None] * n + shear[:, None] * that)
        f[~act] = 0.0
        Fpf += f
        F += f.sum(0)
        flux += np.where(act, A * c / (2 * SQRTPI), 0.0)
    return F, flux, Fpf


def thermal_speed(T, m):
    return np.sqrt(2 * K_B * T / m)


# ------------------------------------------------------------------ partial energy accommodation (reading A22)
def reemission_pressure_alpha_e(S, S_W, gamma, alpha_e):
    """Normal momentum flux of diffuse re-emission from a one-sided flat element, in units of q = rho V^2 / 2, when a
    molecule arriving with velocity v leaves as a flux-weighted half-Maxwellian at
        T_r = alpha_E T_W + (1 - alpha_E) m |v|^2 / (3 k_B)        (reading A22 of DESIGN.md).
    With x = v / c_mp:  c_r(x)^2 / c_mp^2 = alpha_E (S/S_W)^2 + (1 - alpha_E) (2/3) |x|^2,  each re-emitted molecule
    carries the mean normal momentum m (sqrt(pi)/2) c_r, and the incident flux density is n c_mp x_n f(x):
        p_r = (sqrt(pi) / S^2) int_{x_n > 0} x_n pi^{-3/2} exp(-|x - S_vec|^2) (c_r(x) / c_mp) d^3x .
    alpha_E = 1 gives chi(s) / (2 S S_W), the standard panel term.  Gauss-Hermite in the two tangential components,
    adaptive quadrature in the normal one."""
    s, st = S * gamma, S * np.sqrt(max(0.0, 1.0 - gamma * gamma))
    xh, wh = np.polynomial.hermite.hermgauss(64)          # int e^{-x^2} g(x) dx ~ sum w g(x)
    T1, T2 = np.meshgrid(xh + st, xh, indexing="ij")
    W = np.outer(wh, wh)
    r2t = T1 ** 2 + T2 ** 2

    def inner(xn):
        cr = np.sqrt(alpha_e * (S / S_W) ** 2 + (1.0 - alpha_e) * (2.0 / 3.0) * (xn * xn + r2t))
        return xn * np.exp(-(xn - s) ** 2) * float((W * cr).sum())

    lo = max(0.0, s - 7.0)
    val, _ = integrate.quad(inner, lo, max(s, 0.0) + 7.0, epsabs=1e-13, epsrel=1e-11, limit=200)
    return SQRTPI / S ** 2 * np.pi ** -1.5 * val
