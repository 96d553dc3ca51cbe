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

// fp64 finish of the position root from an fp32-accurate start y0 (target = g0 + u gI)
TPMC_HD double polish_sin_phi(double target, double S, double y0) {
  // one fp64 Halley step (cubic): from an fp32-converged start (error ~1e-7) it lands at rounding level.
  // The step length measures the start error; if it is not small the Newton loop below finishes the job.
  double yd = y0;
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
  return polish_sin_phi(target, S, (double)y);
}

// fp64 finish of the normal-speed root from an fp32-accurate start x0 (target = (1 - u) chi(s))
TPMC_HD double polish_normal_speed(double target, double s, double x0) {
  double xd = x0;
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
  return polish_normal_speed(target, s, (double)x);
}

struct SeedState {
  double x[3];
  double v[3];
  int species;
};

// O3-O8 for particle i.  Uniform usage: block 0 = (species, sin phi, theta, v_n), block 1 = (rho, angle, -, -).
// hint != nullptr: fp32-converged roots (y = S sin phi, x_n) handed over by the pre-cull pass; they replace the
// fp32 starts above, the fp64 finish is the same.
TPMC_HD SeedState seed_particle(const RunConst& rc, unsigned long long i, const float* hint = nullptr) {
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
  const double t = hint ? polish_sin_phi(sc.g0 + u01(b0.y) * sc.gI, sc.S, (double)hint[0])
                        : sample_sin_phi_fast(u01(b0.y), sc);
  const double cphi = sqrt(1.0 - t * t);
  double st, ct;
  sincospi(2.0 * u01(b0.z), &st, &ct);
  const double xh[3] = {cphi * ct, cphi * st, t};
  // O6: local frame: n = -xhat inward, t1 meridional (downstream), t2 = t1 x n
  const double t1[3] = {t * ct, t * st, -cphi};
  const double t2[3] = {-st, ct, 0.0};
  // O7: velocity components in units of c_mp (eqs. 14a-c)
  const double xn = hint ? polish_normal_speed((1.0 - u01(b0.w)) * chi_fn(sc.S * t), sc.S * t, (double)hint[1])
                         : sample_normal_speed_fast(u01(b0.w), sc.S * t);
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

// ---- rectangular control volume (readings A24, A25) ------------------------------------------
// The scheme the paper replaces, as a cross-check (TPMC_CV_BOX: exact) and as a negative control
// (TPMC_CV_BOX_UNWEIGHTED: inward speed without the flux weight).  Face k = 2 axis + side (side 0 at -h with inward
// normal +e_axis).  Uniforms: block 0 = (species, face, position, position), block 1 = (v_n, rho, angle, -).
TPMC_HD SeedState seed_particle_box(const RunConst& rc, unsigned long long i) {
  const uint4 b0 = particle_block(rc, i, 0u);
  const uint4 b1 = particle_block(rc, i, 1u);
  SeedState out;
  const double u0 = u01(b0.x);
  int s = 0;
  while (s < rc.n_species - 1 && u0 >= rc.sp[s].cumx) ++s;
  out.species = s;
  const SpeciesConst& sc = rc.sp[s];
  const double uf = u01(b0.y) * sc.bcum[5];
  int k = 0;
  while (k < 5 && uf >= sc.bcum[k]) ++k;
  const int a = k >> 1, side = k & 1, e1 = (a + 1) % 3, e2 = (a + 2) % 3;
  const double sn = sc.bsn[k];
  double xn;
  if (rc.control_volume == TPMC_CV_BOX_UNWEIGHTED) xn = sn + erfcinv((1.0 - u01(b1.x)) * erfc(-sn));
  else xn = sample_normal_speed_fast(u01(b1.x), sn);
  const double rho = sqrt(-log(u01(b1.y)));
  double sa, ca;
  sincospi(2.0 * u01(b1.z), &sa, &ca);
  double x[3], v[3];
  x[a] = rc.centre[a] + (side ? rc.box_h[a] : -rc.box_h[a]);
  x[e1] = rc.centre[e1] + (2.0 * u01(b0.z) - 1.0) * rc.box_h[e1];
  x[e2] = rc.centre[e2] + (2.0 * u01(b0.w) - 1.0) * rc.box_h[e2];
  v[a] = sc.c * (side ? -xn : xn);
  v[e1] = sc.c * (rc.V[e1] / sc.c + rho * ca);
  v[e2] = sc.c * (rc.V[e2] / sc.c + rho * sa);
#pragma unroll
  for (int j = 0; j < 3; ++j) { out.x[j] = x[j]; out.v[j] = v[j]; }
  return out;
}

// ---- a2, pre-cull pass: fp32 ESTIMATE of the seeded ray ------------------------------------------------
// Most particles of the spherical control volume never come near the body (hit fraction of the bounding
// sphere = (R_b/r)^2, P5), and a particle whose first segment misses the body contributes nothing (O10:
// it escapes).  The pre-cull pass evaluates O3-O8 in fp32 -- same Philox words, same inverse-CDF roots,
// three fp32 Newton steps with a convergence check, no data-dependent branch -- and tests the estimated ray
// against the mesh AABB and bounding sphere grown by kPrecullMargin * R_b.  Only a ray that misses them with
// a certified estimate is dropped; everything else goes through the fp64 sampler above (which starts from
// the fp32 roots found here).  Error budget of a certified estimate: sin(phi) to ~1e-6 => position and local
// frame to <= sqrt(2e-6) ~ 1.5e-3 rad near the poles (where cos(phi) = sqrt(1-t^2) is ill-conditioned),
// velocity components to ~1e-4 relative => the estimated ray stays within
// (1.5e-3 * 1.5 + 1.5e-3 * 2.5 + 3e-4) R_b < 7e-3 R_b of the exact one anywhere inside the bounding sphere
// (measured over 3e9 particles, S = 0.3 .. 20: <= 6.2e-4 R_b); the margin is 2e-2 R_b.
// tests/test_gpu_parity.py checks that runs with and without this pass give identical results.
struct SpeciesF {
  float S, c, g0, gI;
  unsigned long long thr;   // word >= thr  <=>  u01(word) >= cumx, exactly (thr = ceil(cumx 2^32 - 1/2))
};
struct SeedConstF {
  SpeciesF sp[TPMC_MAX_SPECIES];
  int n_species;
  float R[9], centre[3], r;
  float lo[3], hi[3];  // grown mesh AABB
  float Rg2;           // (grown bounding radius)^2
  float cot_g;         // cot(theta), sin(theta) = (grown bounding radius) / r: stage-A threshold
  // two-level cull volume (k_reach_hist / k_outlier_boxes in lbvh.cu): every facet lies in the sphere of radius
  // R_in about the centre or in one of n_box boxes; both grown like the AABB.  n_box < 0: not used.
  float Rin2;
  int n_box;
  float blo[8][3], bhi[8][3];
};

__device__ __forceinline__ float u01f(uint32_t w) { return ((float)w + 0.5f) * 2.3283064365386963e-10f; }
// square root and reciprocal to ~2 ulp without the range checks and fix-up steps of sqrtf / __frcp_rn (one MUFU + one
// multiply): the estimate's own error budget is 1e-4 and its margin 2e-2 R_b.  sqrt_fast(0) = 0; arguments are >= 0.
__device__ __forceinline__ float sqrt_fast(float x) { return x * rsqrtf(fmaxf(x, 1e-36f)); }
__device__ __forceinline__ float rcp_fast(float x) { return __fdividef(1.0f, x); }
// sin and cos of 2 pi u, u in (0, 1), by the hardware approximations on an argument folded into [-pi, pi) (absolute
// error ~5e-7: as good as the estimate needs; sincospif costs six times as many instructions)
__device__ __forceinline__ void sincos_2pi_fast(float u, float& s, float& c) {
  const float x = 6.2831853071795865f * (u - (u >= 0.5f ? 1.0f : 0.0f));
  s = __sinf(x);
  c = __cosf(x);
}

// erfc(x) with fractional error ~2e-7 in ~20 instructions (the library erfcf costs ~45): the classical
// Chebyshev fit erfc(z) = t exp(-z^2 + P(t)), t = 1/(1 + z/2), z >= 0 (Numerical Recipes' erfcc coefficients),
// erfc(-z) = 2 - erfc(z).  Used by the pre-cull estimate only; its tolerances (1e-5, 1e-4) are far above this.
__device__ __forceinline__ float erfc_fast(float x) {
  const float z = fabsf(x);
  const float t = __fdividef(1.0f, fmaf(0.5f, z, 1.0f));
  float p = 0.17087277f;
  p = fmaf(p, t, -0.82215223f);
  p = fmaf(p, t, 1.48851587f);
  p = fmaf(p, t, -1.13520398f);
  p = fmaf(p, t, 0.27886807f);
  p = fmaf(p, t, -0.18628806f);
  p = fmaf(p, t, 0.09678418f);
  p = fmaf(p, t, 0.37409196f);
  p = fmaf(p, t, 1.00002368f);
  p = fmaf(p, t, -1.26551223f);
  const float r = t * __expf(fmaf(-z, z, p));
  return x >= 0.0f ? r : 2.0f - r;
}

// y = S sin(phi) to ~1e-6 relative, ok = certified.  Start: the large-y form Gt ~ sqrt(pi)(y^2 + 1/2) for T >= 5
// (y > 1.55: relative error < 1e-2), else a degree-6 polynomial in ln T fitted to Gt^-1 on y in [-2.05, 1.6]
// (T in [2.6e-4, 5.4], error < 2e-3).  Two Newton steps from there land at fp32 resolution and the second step's
// length certifies it (Gt is convex and increasing: from the right of the root the iteration is monotone); the
// old start (tangent at y = 0 below T = 2) needed three steps and left 1.3 % (S = 8) to 5 % (S = 4) of the
// particles uncertified -- every one of those goes through the fp64 sampler whatever its ray does.
__device__ __forceinline__ float approx_y(float u, const SpeciesF& sc, bool& ok) {
  const float S = sc.S;
  const float T = fmaf(u, sc.gI, sc.g0);
  const float L = __logf(fmaxf(T, 2.7e-4f));
  float pl = 6.191523802e-06f;
  pl = fmaf(pl, L, 1.690018055e-04f);
  pl = fmaf(pl, L, 1.939014817e-03f);
  pl = fmaf(pl, L, 1.328511861e-02f);
  pl = fmaf(pl, L, 7.322245522e-02f);
  pl = fmaf(pl, L, 5.387478773e-01f);
  pl = fmaf(pl, L, 3.962664050e-01f);
  float y = (T >= 5.0f) ? sqrt_fast(fmaf(T, 1.0f / TPMC_SQRTPI_F, -0.5f)) : pl;
  y = fminf(S, fmaxf(-S, y));
  float step = 1.0f;
#pragma unroll
  for (int it = 0; it < 2; ++it) {
    const float e = __expf(-y * y);
    const float ec = erfc_fast(-y);
    const float g = 0.25f * TPMC_SQRTPI_F * fmaf(2.0f * y, y, 1.0f) * ec + 0.5f * y * e;
    const float d = fmaf(TPMC_SQRTPI_F * y, ec, e);
    const float yn = fminf(S, fmaxf(-S, y - __fdividef(g - T, d)));
    step = fabsf(yn - y);
    y = yn;
  }
  // S -> 0 (series, A19) and the far lee-side tail go to the fp64 path
  ok = (S >= 0.05f) && (T >= 0.004f) && (step <= 1e-5f * fmaxf(1.0f, fabsf(y)));
  return y;
}

// x_n = v_n / c_mp to ~1e-4 relative, ok = certified.  omu = 1 - u
__device__ __forceinline__ float approx_normal_speed(float omu, float s, float chis, bool& ok) {
  const float T = omu * chis;
  const float xm = 0.5f * (s + sqrt_fast(fmaf(s, s, 2.0f)));
  const float tau = fminf(fmaxf(__fdividef(T, TPMC_SQRTPI_F * s), 1e-30f), 1.9999f);
  const float xa = s + erfcinvf(tau) + __fdividef(0.5f, s);
  float x = (s >= 1.0f) ? xa : xm;
  const float xs = sqrt_fast(fmaxf(chis - T, 0.0f)) * __expf(0.5f * s * s);   // chis - T = u chi(s)
  x = (xs < 0.25f * xm || !(x > 0.0f)) ? fminf(xm, 2.0f * xs) : x;
  float step = 1.0f, q = 0.0f, e = 0.0f;
#pragma unroll
  for (int it = 0; it < 3; ++it) {
    const float z = x - s;
    e = __expf(-z * z);
    q = fmaf(TPMC_SQRTPI_F * s, erfc_fast(z), e);
    float xn = x + __fdividef(q - T, 2.0f * x * e);
    xn = (xn > 0.0f) ? xn : 0.5f * x;
    step = fabsf(xn - x);
    x = xn;
  }
  // chi(s) cancels in fp32 for s << 0.  Conditioning: an evaluation error eps*Q moves the root by eps*Q/|Q'|;
  // certify only where that stays below ~5e-5 (1 + x) for eps ~ 1e-6 (the low tail x << s of a fast stream is
  // flat in this form).  Every comparison is false on NaN.
  ok = (s > -2.0f) && (x > 0.0f) && (step <= 1e-4f * (1.0f + x)) && (q <= 100.0f * x * e * (1.0f + x));
  return x;
}

// ---- the estimate in two stages (k_seed_precull) -------------------------------------------------------------
// Stage A stops before the normal speed: with everything else known, the ray reaches the grown bounding sphere
// iff its inward normal speed exceeds a threshold, x_n >= x_req = cot(theta) |x_t| with sin(theta) = R_g / r, and
// x_n = F^-1(u) is increasing in u, so that is  1 - u <= Q(x_req) / chi(s)  -- ONE evaluation of the survival
// function of eq. (14a) instead of its inversion.  Only particles that pass (44 % at r = 1.5 R_b) go on to
// stage B (inversion, ray, cull volumes).  A particle is dropped here only when the comparison is certain:
// Q and chi are evaluated to ~1e-5 relative under the conditions checked below, the slack is 2e-3, and x_req is
// taken for the sphere grown by kPrecullMargin (a 3 % shift of x_req, against ~1e-4 of estimate error).
struct PrecullA {
  float y, t, cphi, xt1, xt2, s;   // S sin(phi), sin(phi), cos(phi), tangential speeds / c, S_n
  float chis;                       // chi(S_n)
  unsigned int w2, w3;              // Philox words of the azimuth theta (needed from stage B on) and of the normal speed
  bool ok_t;
};

__device__ __forceinline__ bool precull_stage_a(const SeedConstF& sf, unsigned int seed_lo, unsigned int seed_hi,
                                                unsigned long long i, PrecullA& a) {
  const uint4 b0 = philox4x32_10(seed_lo, seed_hi, (uint32_t)i, (uint32_t)(i >> 32), 0u, 0u);
  const uint4 b1 = philox4x32_10(seed_lo, seed_hi, (uint32_t)i, (uint32_t)(i >> 32), 1u, 0u);
  SpeciesF sc = sf.sp[0];
  for (int s = 1; s < sf.n_species; ++s)
    if ((unsigned long long)b0.x >= sf.sp[s - 1].thr) sc = sf.sp[s];   // cumx is non-decreasing: the last hit wins
  a.y = approx_y(u01f(b0.y), sc, a.ok_t);
  a.t = fminf(1.0f, fmaxf(-1.0f, __fdividef(a.y, sc.S)));
  a.cphi = sqrt_fast(fmaxf((1.0f - a.t) * (1.0f + a.t), 0.0f));
  a.w2 = b0.z;
  const float rho = sqrt_fast(-__logf(u01f(b1.x)));
  float sa, ca;
  sincos_2pi_fast(u01f(b1.y), sa, ca);
  a.xt1 = fmaf(sc.S, a.cphi, rho * ca);
  a.xt2 = rho * sa;
  a.s = sc.S * a.t;
  a.w3 = b0.w;
  // threshold on the normal speed for the grown bounding sphere
  const float xr = sf.cot_g * sqrt_fast(fmaf(a.xt1, a.xt1, a.xt2 * a.xt2));
  const float s = a.s, z = xr - s;
  const float e = __expf(-z * z);
  const float q = fmaf(TPMC_SQRTPI_F * s, erfc_fast(z), e);                        // Q(x_req)
  const float chis = fmaf(TPMC_SQRTPI_F * s, erfc_fast(-s), __expf(-s * s));       // chi(s)
  const float omu = u01f(~b0.w);                                                   // 1 - u
  a.chis = chis;
  // certain only without heavy cancellation in Q or chi (lee side) and away from under/overflow
  const bool sure = a.ok_t && (s > -2.0f) && (q >= 1e-3f * e) && (chis > 1e-30f) && (q == q);
  const bool miss = sure && (omu * chis > q * 1.002f + 1e-37f);
  return !miss;
}

// Stage B: the normal speed, the estimated ray, the fp32 roots.  Returns false when the estimate is not certified.
__device__ __forceinline__ bool precull_stage_b(const SeedConstF& sf, const PrecullA& a, float o[3], float v[3],
                                                float root[2]) {
  bool ok_x;
  const float xn = approx_normal_speed(u01f(~a.w3), a.s, a.chis, ok_x);
  float st, ct;
  sincos_2pi_fast(u01f(a.w2), st, ct);
  const float xh[3] = {a.cphi * ct, a.cphi * st, a.t};
  const float t1[3] = {a.t * ct, a.t * st, -a.cphi};
  const float t2[3] = {-st, ct, 0.0f};
  float vl[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) vl[k] = fmaf(a.xt2, t2[k], fmaf(a.xt1, t1[k], -xn * xh[k]));
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const float rx = fmaf(sf.R[3 * k + 2], xh[2], fmaf(sf.R[3 * k + 1], xh[1], sf.R[3 * k] * xh[0]));
    const float rv = fmaf(sf.R[3 * k + 2], vl[2], fmaf(sf.R[3 * k + 1], vl[1], sf.R[3 * k] * vl[0]));
    o[k] = fmaf(sf.r, rx, sf.centre[k]);
    v[k] = rv;
  }
  root[0] = a.y;
  root[1] = xn;
  return a.ok_t && ok_x;
}

// Can the estimated ray touch the grown bounding sphere and the grown AABB?  (branch-free)
__device__ __forceinline__ bool precull_touch(const SeedConstF& sf, const float o[3], const float v[3]) {
  const float oc[3] = {o[0] - sf.centre[0], o[1] - sf.centre[1], o[2] - sf.centre[2]};
  const float b = fmaf(oc[2], v[2], fmaf(oc[1], v[1], oc[0] * v[0]));
  const float vv = fmaf(v[2], v[2], fmaf(v[1], v[1], v[0] * v[0]));
  const float cc = fmaf(oc[2], oc[2], fmaf(oc[1], oc[1], oc[0] * oc[0])) - sf.Rg2;
  // closest approach to the centre: |oc|^2 - b^2/|v|^2 <= Rg^2, approached (b < 0); 1e-3 relative slack on the
  // cancelling difference (the terms are ~2.25 R_b^2, their rounding ~1e-7 of that)
  const bool sphere = (b < 0.0f) && (b * b >= vv * (cc - 1e-3f * sf.Rg2));
  // plane distances as fma(plane, 1/v, -o/v): one instruction each.  The absolute error u |o/v| of this form is,
  // relative to the width of a slab in t, u |o| / extent < 1e-5 -- far inside the growth of the volumes.
  // (a direction component below 1e-30 is replaced by 1e-30: no inf - inf; the ray stays parallel to the slab)
  const float vs[3] = {fabsf(v[0]) < 1e-30f ? 1e-30f : v[0], fabsf(v[1]) < 1e-30f ? 1e-30f : v[1],
                       fabsf(v[2]) < 1e-30f ? 1e-30f : v[2]};
  const float id[3] = {rcp_fast(vs[0]), rcp_fast(vs[1]), rcp_fast(vs[2])};
  const float oi[3] = {-o[0] * id[0], -o[1] * id[1], -o[2] * id[2]};
  float ax[3], bx[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    ax[k] = fmaf(sf.lo[k], id[k], oi[k]);
    bx[k] = fmaf(sf.hi[k], id[k], oi[k]);
  }
  const float tn = fmaxf(fmaxf(fminf(ax[0], bx[0]), fminf(ax[1], bx[1])), fminf(ax[2], bx[2]));
  const float tf = fminf(fminf(fmaxf(ax[0], bx[0]), fmaxf(ax[1], bx[1])), fmaxf(ax[2], bx[2]));
  const bool box = fmaxf(tn, 0.0f) * 0.999999f <= tf * 1.000001f;   // NaN planes (0 * inf) are dropped by min/max
  if (sf.n_box >= 0) {   // uniform branch: the inner sphere (same slack as above) or any of the outlier boxes
    const float cin = fmaf(oc[2], oc[2], fmaf(oc[1], oc[1], oc[0] * oc[0])) - sf.Rin2;
    bool any = (b < 0.0f) && (b * b >= vv * (cin - 1e-3f * sf.Rg2));
    for (int j = 0; j < sf.n_box; ++j) {
      float a2[3], b2[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        a2[k] = fmaf(sf.blo[j][k], id[k], oi[k]);
        b2[k] = fmaf(sf.bhi[j][k], id[k], oi[k]);
      }
      const float un = fmaxf(fmaxf(fminf(a2[0], b2[0]), fminf(a2[1], b2[1])), fminf(a2[2], b2[2]));
      const float uf = fminf(fminf(fmaxf(a2[0], b2[0]), fmaxf(a2[1], b2[1])), fmaxf(a2[2], b2[2]));
      any = any || (fmaxf(un, 0.0f) * 0.999999f <= uf * 1.000001f);
    }
    return sphere && box && any;
  }
  return sphere && box;
}
