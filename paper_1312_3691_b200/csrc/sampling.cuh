// sampling.cuh -- step a2: consistent particle seeding on the spherical control volume
// (eqs. 10, 11, 14a-c, 15; definitions O3-O8 of DESIGN.md).  Device code, fp64.
//
// Both random variates that the paper gives only as densities are drawn by INVERSE CDF (readings
// A2/A3): one uniform per variate keeps the Philox counter layout fixed, and the result is a
// mathematically defined function of the uniform, so any convergent root-finder gives the same value.
#pragma once

#include "common.cuh"

// chi(s) = e^{-s^2} + sqrt(pi) s erfc(-s): bracket of eq. (8) P:143 written without cancellation (A4)
TPMC_HD double chi_fn(double s) { return exp(-s * s) + TPMC_SQRTPI * s * erfc(-s); }

// Position (eq. 11).  With t = sin(phi), y = S t:  dP ~ chi(y) dy, antiderivative
//   Gt(y) = (sqrt(pi)/4)(1 + 2 y^2) erfc(-y) + (y/2) e^{-y^2},   Gt' = chi > 0,  Gt'' = sqrt(pi) erfc(-y) > 0.
// Solve Gt(y) = Gt(-S) + u [Gt(S) - Gt(-S)].  Gt is convex and increasing, so Newton from any point is
// to the right of the root after one step and then decreases monotonically: no bracket is needed.
TPMC_HD double sample_sin_phi(double u, const SpeciesConst& sc) {
  const double S = sc.S;
  if (S < 1e-4) {
    // A19: chi(s) = 1 + sqrt(pi) s + s^2 + O(s^4):  H(t) = [(t+1) + sqrt(pi) S (t^2-1)/2 + S^2 (t^3+1)/3] / (2 + 2S^2/3)
    const double rhs = u * (2.0 + 2.0 * S * S / 3.0);
    double t = 2.0 * u - 1.0;
    for (int it = 0; it < 8; ++it) {
      const double f = (t + 1.0) + 0.5 * TPMC_SQRTPI * S * (t * t - 1.0) + S * S * (t * t * t + 1.0) / 3.0 - rhs;
      const double d = 1.0 + TPMC_SQRTPI * S * t + S * S * t * t;
      t -= f / d;
    }
    return fmin(1.0, fmax(-1.0, t));
  }
  const double target = sc.g0 + u * sc.gI;
  // large-y asymptote Gt ~ sqrt(pi) (y^2 + 1/2) as first guess; anything works (see above)
  double y = sqrt(fmax(target / TPMC_SQRTPI - 0.5, 0.0));
  y = fmin(y, S);
  for (int it = 0; it < 64; ++it) {
    const double e = exp(-y * y);
    const double ec = erfc(-y);
    const double g = 0.25 * TPMC_SQRTPI * (1.0 + 2.0 * y * y) * ec + 0.5 * y * e;
    const double d = e + TPMC_SQRTPI * y * ec;
    double yn = y - (g - target) / d;
    yn = fmin(S, fmax(-S, yn));
    const double step = fabs(yn - y);
    y = yn;
    if (step <= 4e-16 * fmax(1.0, fabs(y))) break;
  }
  return fmin(1.0, fmax(-1.0, y / S));
}

// Inward normal speed (eq. 14a, read in x = v_n / c_mp, G2): density 2x e^{-(x-s)^2} / chi(s), x >= 0.
// Survival form (A4):  1 - F(x) = Q(x)/chi(s),  Q(x) = e^{-(x-s)^2} + sqrt(pi) s erfc(x-s),  Q' = -2x e^{-(x-s)^2}.
// F is convex left of the mode x* = (s + sqrt(s^2+2))/2 and concave right of it, so Newton started at the
// mode converges monotonically from either side.
TPMC_HD double sample_normal_speed(double u, double s) {
  const double target = (1.0 - u) * chi_fn(s);
  const double xm = 0.5 * (s + sqrt(s * s + 2.0));
  double x = xm;
  {  // cheap improvement of the start on the low side, where F ~ x^2 e^{-s^2}/chi(s): stays right of the root
    const double q0 = chi_fn(s) - target;            // = u chi(s)
    const double xs = sqrt(q0) * exp(0.5 * s * s);   // root of the leading term
    if (xs < 0.25 * xm) x = fmin(xm, 2.0 * xs);
  }
  for (int it = 0; it < 96; ++it) {
    const double z = x - s;
    const double e = exp(-z * z);
    const double q = e + TPMC_SQRTPI * s * erfc(z);
    const double d = -2.0 * x * e;
    double xn = x - (q - target) / d;
    if (!(xn > 0.0)) xn = 0.5 * x;
    const double step = fabs(xn - x);
    x = xn;
    if (step <= 4e-16 * (1.0 + x)) break;
  }
  return x;
}

// ---- fast path: fp32 Newton to ~1e-7, one fp64 Halley step, convergence check -------------------------
// Root-finding in fp64 costs ~150 instructions per step and its iteration count differs from lane to
// lane.  The first digits are therefore found in fp32 (erfcf/expf, a fixed number of steps), then one
// cubically convergent fp64 step cubes the error.  If that step is longer than 3e-6 (ill-conditioned
// tails, a poor start: 1-6 % of the variates) fp64 Newton continues from the current point until a step
// falls below 1e-8: the result is the same root either way.
#define TPMC_SQRTPI_F 1.7724538509055160f

TPMC_HD double sample_sin_phi_fast(double u, const SpeciesConst& sc) {
  const double S = sc.S;
  if (S < 1e-4) return sample_sin_phi(u, sc);
  const double target = sc.g0 + u * sc.gI;
  const float T = (float)target, Sf = (float)S;
  float y;
  if (T >= 2.0f) {
    y = sqrtf(T * (1.0f / TPMC_SQRTPI_F) - 0.5f);            // Gt ~ sqrt(pi)(y^2 + 1/2)
  } else if (T >= 0.004f) {
    y = T - 0.4431135f;                                      // tangent at y = 0 (Gt(0) = sqrt(pi)/4, Gt' = 1)
  } else {
    const float L = -logf(4.0f * fmaxf(T, 1e-37f));          // Gt ~ e^{-y^2} / (4 |y|^3) for y << 0
    y = -sqrtf(fmaxf(L - 1.5f * logf(L), 0.25f));
  }
  y = fminf(Sf, fmaxf(-Sf, y));
#pragma unroll
  for (int it = 0; it < 5; ++it) {
    const float e = expf(-y * y);
    const float ec = erfcf(-y);
    const float g = 0.25f * TPMC_SQRTPI_F * (1.0f + 2.0f * y * y) * ec + 0.5f * y * e;
    const float d = e + TPMC_SQRTPI_F * y * ec;
    y = fminf(Sf, fmaxf(-Sf, y - (g - T) / d));
  }
  // one fp64 Halley step (cubic): from an fp32-converged start (error ~1e-7) it lands at rounding level.
  // The step length measures the start error; if it is not small the Newton loop below finishes the job.
  double yd = (double)y;
  {
    const double e = exp(-yd * yd);
    const double ec = erfc(-yd);
    const double f = 0.25 * TPMC_SQRTPI * (1.0 + 2.0 * yd * yd) * ec + 0.5 * yd * e - target;
    const double d1 = e + TPMC_SQRTPI * yd * ec;       // G' = chi
    const double d2 = TPMC_SQRTPI * ec;                // G''
    const double yn = fmin(S, fmax(-S, yd - 2.0 * f * d1 / (2.0 * d1 * d1 - f * d2)));
    const double step = fabs(yn - yd);
    yd = yn;
    if (step <= 3e-6 * fmax(1.0, fabs(yd))) return fmin(1.0, fmax(-1.0, yd / S));
  }
  for (int it = 0; it < 64; ++it) {   // general solver, continued from yd; a step below 1e-8 squares to < 1e-16
    const double e = exp(-yd * yd);
    const double ec = erfc(-yd);
    const double g = 0.25 * TPMC_SQRTPI * (1.0 + 2.0 * yd * yd) * ec + 0.5 * yd * e;
    const double d = e + TPMC_SQRTPI * yd * ec;
    const double yn = fmin(S, fmax(-S, yd - (g - target) / d));
    const double step = fabs(yn - yd);
    yd = yn;
    if (step <= 1e-8 * fmax(1.0, fabs(yd))) break;
  }
  return fmin(1.0, fmax(-1.0, yd / S));
}

TPMC_HD double sample_normal_speed_fast(double u, double s) {
  const double chis = chi_fn(s);
  const double target = (1.0 - u) * chis;
  const float sf = (float)s, T = (float)target;
  const float xm = 0.5f * (sf + sqrtf(sf * sf + 2.0f));
  float x = xm;
  if (sf >= 1.0f) {
    // Q / (sqrt(pi) s) = erfc(z) + e^{-z^2} / (sqrt(pi) s), z = x - s: start from the erfc part alone
    const float tau = fminf(fmaxf(T / (TPMC_SQRTPI_F * sf), 1e-30f), 1.9999f);
    x = sf + erfcinvf(tau) + 0.5f / sf;
  }
  {
    const float q0 = (float)(u * chis);
    const float xs = sqrtf(q0) * expf(0.5f * sf * sf);       // root of the leading term of F near x = 0
    if (xs < 0.25f * xm || !(x > 0.0f)) x = fminf(xm, 2.0f * xs);
  }
#pragma unroll
  for (int it = 0; it < 5; ++it) {
    const float z = x - sf;
    const float e = expf(-z * z);
    const float q = e + TPMC_SQRTPI_F * sf * erfcf(z);
    float xn = x + (q - T) / (2.0f * x * e);
    if (!(xn > 0.0f)) xn = 0.5f * x;
    x = xn;
  }
  double xd = (double)x;
  {  // one fp64 Halley step, as above: f = Q - target, f' = -2x e^{-z^2}, f'' = -2 e^{-z^2} (1 - 2 x z)
    const double z = xd - s;
    const double e = exp(-z * z);
    const double f = e + TPMC_SQRTPI * s * erfc(z) - target;
    const double d1 = -2.0 * xd * e;
    const double d2 = -2.0 * e * (1.0 - 2.0 * xd * z);
    double xn = xd - 2.0 * f * d1 / (2.0 * d1 * d1 - f * d2);
    if (!(xn > 0.0) || !(xn < 1e300)) xn = 0.5 * xd;
    const double step = fabs(xn - xd);
    xd = xn;
    if (step <= 3e-6 * (1.0 + xd)) return xd;
  }
  for (int it = 0; it < 96; ++it) {   // general solver, continued from xd
    const double z = xd - s;
    const double e = exp(-z * z);
    const double q = e + TPMC_SQRTPI * s * erfc(z);
    double xn = xd + (q - target) / (2.0 * xd * e);
    if (!(xn > 0.0) || !(xn < 1e300)) xn = (xn > 0.0) ? 0.5 * (s > 0.0 ? s : 0.0) + 0.35 : 0.5 * xd;
    const double step = fabs(xn - xd);
    xd = xn;
    if (step <= 1e-8 * (1.0 + xd)) break;
  }
  return xd;
}

struct SeedState {
  double x[3];
  double v[3];
  int species;
};

// O3-O8 for particle i.  Uniform usage: block 0 = (species, sin phi, theta, v_n), block 1 = (rho, angle, -, -).
TPMC_HD SeedState seed_particle(const RunConst& rc, unsigned long long i) {
  const uint4 b0 = particle_block(rc, i, 0u);
  const uint4 b1 = particle_block(rc, i, 1u);
  SeedState out;
  // A8: species by number fraction
  const double u0 = u01(b0.x);
  int s = 0;
  while (s < rc.n_species - 1 && u0 >= rc.sp[s].cumx) ++s;
  out.species = s;
  const SpeciesConst& sc = rc.sp[s];
  // O5: position on the unit sphere, stream frame (pole = upstream, A1)
  const double t = sample_sin_phi_fast(u01(b0.y), sc);
  const double cphi = sqrt(1.0 - t * t);
  double st, ct;
  sincospi(2.0 * u01(b0.z), &st, &ct);
  const double xh[3] = {cphi * ct, cphi * st, t};
  // O6: local frame: n = -xhat inward, t1 meridional (downstream), t2 = t1 x n
  const double t1[3] = {t * ct, t * st, -cphi};
  const double t2[3] = {-st, ct, 0.0};
  // O7: velocity components in units of c_mp (eqs. 14a-c)
  const double xn = sample_normal_speed_fast(u01(b0.w), sc.S * t);
  const double rho = sqrt(-log(u01(b1.x)));
  double sa, ca;
  sincospi(2.0 * u01(b1.y), &sa, &ca);
  const double xt1 = sc.S * cphi + rho * ca;
  const double xt2 = rho * sa;
  double vl[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) vl[k] = (xn * -xh[k] + xt1 * t1[k]) + xt2 * t2[k];
  // O8: rotate to the body frame (eq. 15), scale
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const double rx = (rc.R[3 * k] * xh[0] + rc.R[3 * k + 1] * xh[1]) + rc.R[3 * k + 2] * xh[2];
    const double rv = (rc.R[3 * k] * vl[0] + rc.R[3 * k + 1] * vl[1]) + rc.R[3 * k + 2] * vl[2];
    out.x[k] = rc.centre[k] + rc.r * rx;
    out.v[k] = sc.c * rv;
  }
  return out;
}
