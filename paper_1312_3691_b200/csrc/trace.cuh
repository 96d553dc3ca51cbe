// trace.cuh -- steps a3/a4 device code: closest-hit traversal of the LBVH and the surface interaction.
//
// Precision contract (reading A9): the mesh and the ray (o, d) are fp32 VALUES; which facet
// is hit is decided as in exact arithmetic on those values (concretely: by the fp64 edge functions of
// O10, evaluated with separately rounded multiplies and adds so that the function of a shared edge is
// exactly antisymmetric for the two facets that share it -- the test is watertight).
//
// The wavefront traversal never evaluates fp64.  It walks the hierarchy with fp32 slab tests made
// conservative by an explicit rounding-error margin, and classifies each facet it reaches with an fp32
// version of the same edge functions carrying a forward error bound:
//     MISS       -- some pair of edge functions has provably opposite signs, or the facet is provably
//                   back-facing / behind the origin: the exact test would reject it too;
//     HIT        -- all three edge functions provably share a sign (and det, tau are provably admissible):
//                   the exact test accepts it; its tau lies in [tlo, thi];
//     UNCERTAIN  -- anything inside the error band.
// HITs shrink the search interval (tmax = min thi); every HIT or UNCERTAIN facet whose tlo <= tmax stays
// in a short candidate list.  The resolve step (k_reflect) evaluates the exact fp64 test on the
// candidates only, and picks the smallest tau, ties to the smallest facet index (A12).
#pragma once

#include "common.cuh"

#ifndef TPMC_STACK_SMEM
#define TPMC_STACK_SMEM 24      // stack entries per thread kept in shared memory (+ 3 rows of headroom in the wavefront kernel)
#endif
#define TPMC_STACK_LOCAL 80     // overflow entries (a Karras tree over 64-bit keys + index is <= 97 deep)
#define TPMC_SENTINEL ((int)0x7FFFFFFF)
#ifndef TPMC_MAX_CAND
#define TPMC_MAX_CAND 3      // candidate slots per ray (1..4); more candidates send the ray to the fp64 search
#endif
#define TPMC_CAND_OVERFLOW ((int)0x7FFFFFFE)   // in cand.w: more candidates than slots -> full fp64 traversal

// 256-bit read-only load (sm_100: LDG.E.256): one L1 sector per lane per instruction instead of half a
// sector -- the traversal is bound by L1 tag lookups of divergent 64-byte node fetches.
__device__ __forceinline__ void ldg256(const float4* p, float4& a, float4& b) {
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w)
               : "l"(p));
}

struct Hit {
  double tau;   // +inf: no hit
  int facet;    // original facet id, -1: no hit
  int slot;     // sorted triangle slot
};

struct TraceCounters {
  unsigned int nodes, tris;
};

// ---- O10: facet test in fp64, exactly in this order ------------------------------------------------
//   a=p0-o, b=p1-o, c=p2-o;  Ng=(p1-p0)x(p2-p0);  det=d.Ng  (one-sided: det<0, two-sided: det!=0)
//   w0=d.(b x c), w1=d.(c x a), w2=d.(a x b);  inside iff all >=0 or all <=0;  tau=(a.Ng)/det > 0
//   cross(x,y) = (x1 y2 - x2 y1, x2 y0 - x0 y2, x0 y1 - x1 y0),  dot(x,y) = (x0 y0 + x1 y1) + x2 y2
__device__ __forceinline__ double nc_mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double nc_sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double nc_add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double dot_nc(const double x[3], const double y[3]) {
  return nc_add(nc_add(nc_mul(x[0], y[0]), nc_mul(x[1], y[1])), nc_mul(x[2], y[2]));
}
__device__ __forceinline__ void cross_nc(const double x[3], const double y[3], double z[3]) {
  z[0] = nc_sub(nc_mul(x[1], y[2]), nc_mul(x[2], y[1]));
  z[1] = nc_sub(nc_mul(x[2], y[0]), nc_mul(x[0], y[2]));
  z[2] = nc_sub(nc_mul(x[0], y[1]), nc_mul(x[1], y[0]));
}

__device__ __forceinline__ bool facet_test(const float4 q0, const float4 q1, const float4 q2, const float of[3],
                                           const float df[3], double& tau) {
  const double o[3] = {(double)of[0], (double)of[1], (double)of[2]};
  const double d[3] = {(double)df[0], (double)df[1], (double)df[2]};
  const double p0[3] = {(double)q0.x, (double)q0.y, (double)q0.z};
  const double p1[3] = {(double)q1.x, (double)q1.y, (double)q1.z};
  const double p2[3] = {(double)q2.x, (double)q2.y, (double)q2.z};
  double a[3], b[3], c[3], e1[3], e2[3], Ng[3], t[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    a[k] = nc_sub(p0[k], o[k]); b[k] = nc_sub(p1[k], o[k]); c[k] = nc_sub(p2[k], o[k]);
    e1[k] = nc_sub(p1[k], p0[k]); e2[k] = nc_sub(p2[k], p0[k]);
  }
  cross_nc(e1, e2, Ng);
  const double det = dot_nc(d, Ng);
  const bool two_sided = (__float_as_uint(q1.w) & TPMC_FACET_TWO_SIDED) != 0u;
  if (two_sided ? (det == 0.0) : !(det < 0.0)) return false;
  cross_nc(b, c, t);
  const double w0 = dot_nc(d, t);
  cross_nc(c, a, t);
  const double w1 = dot_nc(d, t);
  cross_nc(a, b, t);
  const double w2 = dot_nc(d, t);
  const bool allpos = (w0 >= 0.0) && (w1 >= 0.0) && (w2 >= 0.0);
  const bool allneg = (w0 <= 0.0) && (w1 <= 0.0) && (w2 <= 0.0);
  if (!(allpos || allneg)) return false;
  const double tt = __ddiv_rn(dot_nc(a, Ng), det);
  if (!(tt > 0.0)) return false;
  tau = tt;
  return true;
}

// ---- fp32 classification of the same test, with forward error bounds --------------------------------
// The edge functions d.(b x c) with b = p1 - o, c = p2 - o do not change when the origin slides along the ray
// (exact arithmetic: d.((b - t d) x (c - t d)) = d.(b x c)), but their fp32 evaluation does: with the origin on the
// control sphere, metres away, the rounding band 10u * sum|d_i b_j c_k| is as wide as a millimetre-sized facet and
// nothing is ever certain.  So the origin is first moved next to the facet, o' = fl(o + t0 d) with t0 the
// parameter of the ray point closest to p0 (any t0 is valid; this one makes |p - o'| facet-sized for a hit), and
// the rounding of that move is carried as a perturbation of the inputs:
//   x = o + t0 d exactly;  o'_k = fma(t0, d_k, o_k) = x_k + e,  |e| <= u |o'_k|         (one rounding)
//   a'_k = fl(p0_k - o'_k) = (p0_k - x_k) + eps_k,  |eps_k| <= u |o'_k| + u |a'_k| <= eta    (likewise b', c')
//   eta  = u (1 + 2^-10) max_k (|o'_k| + max(|a'_k|, |b'_k|, |c'_k|))
//   d.(b' x c') - d.(B x C) = d.(eps_b x c') + d.(b' x eps_c) - d.(eps_b x eps_c),  and
//   |d.(e x c)| = |e.(c x d)| <= |e|_inf |c x d|_1 <= |e|_inf |c|_1 |d|_1,  so the perturbation is bounded by
//   P(b', c') = eta |d|_1 (|b'|_1 + |c'|_1 + 3 eta).
// On top of it the evaluation itself: every monomial d_i b'_j c'_k passes through at most 5 roundings (product,
// difference, product with d, two sums; 7 for det and the numerator, whose edge vectors are rounded differences of
// corners): |computed - exact| <= ((1+u)^7 - 1) M with M the sum of the absolute monomials, itself computed in fp32:
// band 10u M.  The bounds are sums of positive terms evaluated in fp32 (relative error < 1e-6): a factor 1.0001
// covers that.  tau: the shifted ray hits at tau - t0 = (A.Ng)/det with A = p0 - x; the numerator's perturbation is
// |eps_a.(e1 x e2)| <= eta |e1 x e2|_1 <= eta sum|e1_j e2_k|; quotient and sum are rounded outwards by directed
// roundings.  Magnitudes in this application (metres, m/s) are far from the fp32 under/overflow range; a NaN (zero
// direction) fails every comparison and ends as UNCERTAIN.
enum { TRI_MISS = 0, TRI_HIT = 1, TRI_UNCERTAIN = 2 };
__device__ __forceinline__ float rcp_approx(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

__device__ __forceinline__ void triple_f32(const float d[3], const float x[3], const float y[3], float& w, float& M) {
  const float p0 = x[1] * y[2], p1 = x[2] * y[1];
  const float p2 = x[2] * y[0], p3 = x[0] * y[2];
  const float p4 = x[0] * y[1], p5 = x[1] * y[0];
  w = fmaf(d[2], p4 - p5, fmaf(d[1], p2 - p3, d[0] * (p0 - p1)));
  M = fmaf(fabsf(d[2]), fabsf(p4) + fabsf(p5), fmaf(fabsf(d[1]), fabsf(p2) + fabsf(p3), fabsf(d[0]) * (fabsf(p0) + fabsf(p1))));
}
__device__ __forceinline__ float norm1(const float x[3]) { return fabsf(x[0]) + fabsf(x[1]) + fabsf(x[2]); }

__device__ __forceinline__ int tri_filter(const float4 q0, const float4 q1, const float4 q2, const float o[3],
                                          const float d[3], float& tlo, float& thi) {
  const float EPS = 5.9604645e-07f;   // 10 * 2^-24
  const float e1[3] = {q1.x - q0.x, q1.y - q0.y, q1.z - q0.z};
  const float e2[3] = {q2.x - q0.x, q2.y - q0.y, q2.z - q0.z};
  float det, Mdet;
  triple_f32(d, e1, e2, det, Mdet);               // d . (e1 x e2)
  const float Edet = EPS * Mdet;
  const bool two_sided = (__float_as_uint(q1.w) & TPMC_FACET_TWO_SIDED) != 0u;
  if (!two_sided && det > Edet) return TRI_MISS;  // provably back-facing
  // origin moved next to the facet
  const float dd = fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
  const float t0 = fmaf(q0.z - o[2], d[2], fmaf(q0.y - o[1], d[1], (q0.x - o[0]) * d[0])) * rcp_approx(dd);   // (any t0 is valid)
  const float os[3] = {fmaf(t0, d[0], o[0]), fmaf(t0, d[1], o[1]), fmaf(t0, d[2], o[2])};
  const float a[3] = {q0.x - os[0], q0.y - os[1], q0.z - os[2]};
  const float b[3] = {q1.x - os[0], q1.y - os[1], q1.z - os[2]};
  const float c[3] = {q2.x - os[0], q2.y - os[1], q2.z - os[2]};
  float eta = 0.0f;
#pragma unroll
  for (int k = 0; k < 3; ++k) eta = fmaxf(eta, fabsf(os[k]) + fmaxf(fabsf(a[k]), fmaxf(fabsf(b[k]), fabsf(c[k]))));
  eta *= 5.9662852e-08f;                          // u (1 + 2^-10)
  const float d1 = norm1(d) * 1.0001f, na = norm1(a), nb = norm1(b), nc = norm1(c), e3 = 3.0f * eta;
  float w0, M0, w1, M1, w2, M2;
  triple_f32(d, b, c, w0, M0);
  triple_f32(d, c, a, w1, M1);
  triple_f32(d, a, b, w2, M2);
  const float pd = eta * d1;
  const float E0 = fmaf(EPS, M0, pd * (nb + nc + e3)), E1 = fmaf(EPS, M1, pd * (nc + na + e3)), E2 = fmaf(EPS, M2, pd * (na + nb + e3));
  const bool anypos = (w0 > E0) || (w1 > E1) || (w2 > E2);
  const bool anyneg = (w0 < -E0) || (w1 < -E1) || (w2 < -E2);
  if (anypos && anyneg) return TRI_MISS;          // two edge functions of provably opposite sign
  float num, Mn;
  triple_f32(a, e1, e2, num, Mn);                 // a' . (e1 x e2) = (tau - t0) det, up to the bands
  const float Mx = (fabsf(e1[1] * e2[2]) + fabsf(e1[2] * e2[1])) + (fabsf(e1[2] * e2[0]) + fabsf(e1[0] * e2[2])) +
                   (fabsf(e1[0] * e2[1]) + fabsf(e1[1] * e2[0]));
  const float En = fmaf(EPS, Mn, 1.0001f * eta * Mx);
  const float ad = fabsf(det);
  const bool det_ok = ad > Edet;                  // sign of det is certain
  tlo = 0.0f;
  thi = INFINITY;
  if (!det_ok) return TRI_UNCERTAIN;
  // tau - t0 = N / |det| with N = sign(det) num in [nl, nh], |det| in [dl, dh]: quotient and sum rounded outwards
  const float ns = det < 0.0f ? -num : num;
  const float nl = __fadd_rd(ns, -En), nh = __fadd_ru(ns, En);
  const float dl = __fadd_rd(ad, -Edet), dh = __fadd_ru(ad, Edet);
  // quotients as numerator x approximate reciprocal (1 ulp + the product's rounding; a denormal denominator flushes to an
  // infinite or NaN quotient, which never shrinks tmax), pushed outwards by 4 ulp and a denormal's worth: still directed
  // bounds, at a tenth of the instructions of __fdiv_rd/ru
  const float qa = nl * rcp_approx(nl >= 0.0f ? dh : dl), qb = nh * rcp_approx(nh >= 0.0f ? dl : dh);
  const float ql = fmaf(-2.4e-7f, fabsf(qa), qa) - 1e-37f, qh = fmaf(2.4e-7f, fabsf(qb), qb) + 1e-37f;
  const float tl = __fadd_rd(t0, ql), th = __fadd_ru(t0, qh);
  if (th < 0.0f) return TRI_MISS;                 // provably behind the origin
  tlo = fmaxf(tl, 0.0f);
  const bool allpos = (w0 > E0) && (w1 > E1) && (w2 > E2);
  const bool allneg = (w0 < -E0) && (w1 < -E1) && (w2 < -E2);
  if ((allpos || allneg) && tl > 0.0f) {          // (one-sided: det < -Edet follows from det_ok)
    thi = th;
    return TRI_HIT;
  }
  return TRI_UNCERTAIN;
}

// ---- conservative fp32 slab test -------------------------------------------------------------------
// Each plane distance (lo - o) * (1/d) carries three roundings: relative error <= 3 * 2^-24.  min/max are
// exact and x -> x -+ 4u|x| is monotone, so one margin on the entry and one on the exit make the test
// conservative.  NaN (0 * inf when d = 0 and o on the plane) is dropped by fminf/fmaxf.
// (The one-FMA form fma(l, 1/d, -o/d) was tried and rejected: its error is absolute, ~u|o/d|, so a ray
// with one tiny direction component needs a margin that inflates every box and walks thousands of nodes.
// Carrying the entry distance on the stack to skip stale entries was tried too: no fewer node visits.)
__device__ __forceinline__ bool slab(float lx, float ly, float lz, float hx, float hy, float hz, const float o[3],
                                     const float id[3], float tmax, float& tnear) {
  const float u4 = 2.384185791015625e-07f;  // 4 * 2^-24
  const float ax = (lx - o[0]) * id[0], bx = (hx - o[0]) * id[0];
  const float ay = (ly - o[1]) * id[1], by = (hy - o[1]) * id[1];
  const float az = (lz - o[2]) * id[2], bz = (hz - o[2]) * id[2];
  float tn = fmaxf(fmaxf(fminf(ax, bx), fminf(ay, by)), fminf(az, bz));
  float tf = fminf(fminf(fmaxf(ax, bx), fmaxf(ay, by)), fmaxf(az, bz));
  tn = fmaf(-u4, fabsf(tn), tn);
  tf = fmaf(u4, fabsf(tf), tf);
  tnear = tn;
  return fmaxf(tn, 0.0f) <= fminf(tf, tmax);
}

// ---- the same test on a box of the compact hierarchy (grid coordinates, see k_compact_nodes) ----------
// The ray is carried in grid coordinates: o' = (o - origin) * inv_scale, d' = d * inv_scale; the ray
// parameter t is unchanged.  A plane q (unsigned 16-bit grid coordinate) is crossed at
//     t = (q - o') / d' = P * id - O * id,     P = 2^23 + q,  O = 2^23 + o',  id = 1 / d'.
// P comes out of the node word by ONE byte permute (the float 0x4B00qqqq is exactly 2^23 + q), and the ray's
// octant decides per axis which half of the word is the near plane and which the far one (sel_n, sel_f are
// permute selectors fixed per ray), so a plane distance costs one PRMT and one FFMA and the slab test needs
// no per-axis min/max:      t_near_k = fma(P_near, id_k, ncn_k),   t_far_k = fma(P_far, id_k, ncf_k).
// ncn_k = -(O id) - G |id|,  ncf_k = -(O id) + G |id|: every error of this evaluation is bounded by a growth
// of the box by G_k grid steps along axis k, so the test is conservative for the fp32 box the node encodes:
//   * o' carries three roundings (difference, rounded inv_scale, product): <= 3u |o'| steps;
//   * O = fl(2^23 + o') and the rounding of fma(-O, id, -+G|id|): <= u |O| steps each;
//   * id = 1/d' carries <= 5u relative (rounded inv_scale, product, 2-ulp reciprocal), which scales the
//     distance |P - O| <= |o'| + 2^16 steps; the final FFMA rounds once more, u relative;
//   * the rounded inv_scale moves a plane by <= u q <= 0.004 steps.
// Sum <= 2u|O| + 9u|o'| + 0.03, plus the rotation into an aligned frame (see grid_ray), which is an error in METRES
// and therefore enters per axis as E_rot * inv_scale_k steps (large in steps, tiny in metres, on an axis along which
// the body is thin);  G_k = 2.5u|O| + 10u|o'| + 0.25 + E_rot * inv_scale_k (about 1.5 steps of the 16-bit grid for an
// origin inside or near the grid; it scales with the origin for a ray that starts far outside, e.g. on a flat axis).
// A zero direction component gives id = inf and NaN plane distances, which fminf/fmaxf drop: the axis then
// does not constrain the ray (conservative).
__device__ __forceinline__ float q_plane(unsigned int w, unsigned int sel) {
  unsigned int r;   // prmt.b32 directly: __byte_perm masks the selector first (one LOP3 per use)
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(w), "r"(0x4B000000u), "r"(sel));
  return __uint_as_float(r);
}

__device__ __forceinline__ void ldg256u(const uint4* p, uint4& a, uint4& b) {
  asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w)
               : "l"(p));
}

// Per-ray constants of the grid-coordinate slab test (see above): 1/d', the two offsets and the permute selectors.
struct GridRay {
  float id[3], ncn[3], ncf[3];
  unsigned int sn[3], sf[3];
};
__device__ __forceinline__ void grid_ray(GridRay& r, const QuantGrid& g, const float o[3], const float d[3]) {
  // into the frame of the grid (x' = R x; R = identity for the body-frame hierarchy, where this is exact: g.rot_* = 0).
  // The fp32 rotation adds an absolute error of <= 3u |o|_1 to each component of o' and <= 3u |d|_1 to each of d'.  At
  // parameter t the rotated ray is therefore within 3u (|o|_1 + t |d|_1) METRES of the exact one along every axis, and
  // while the ray is inside the root box t |d|_1 <= sqrt(3) t |d| <= sqrt(3) (|o| + reach), reach = the largest |x| in
  // the box: E_rot <= 3u (1 + sqrt 3) |o|_1 + 3 sqrt(3) u reach < 9u |o|_1 + 6u reach = g.rot_o |o|_1 + g.rot_c.  A box
  // that the exact ray enters at t is entered at t by the rotated ray once grown by E_rot: in grid steps of axis k that
  // is E_rot * inv_scale_k, whatever the extent of the body along that axis.
  float og[3], dg[3];
  const float e_rot = fmaf(g.rot_o, fabsf(o[0]) + fabsf(o[1]) + fabsf(o[2]), g.rot_c) * 1.000001f;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    og[k] = fmaf(g.R[3 * k + 2], o[2], fmaf(g.R[3 * k + 1], o[1], g.R[3 * k] * o[0]));
    dg[k] = fmaf(g.R[3 * k + 2], d[2], fmaf(g.R[3 * k + 1], d[1], g.R[3 * k] * d[0]));
  }
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const float dq = dg[k] * g.inv_scale[k];
    const float idk = __fdividef(1.0f, dq);                  // 2 ulp
    const float oq = (og[k] - g.origin[k]) * g.inv_scale[k];
    const float O = 8388608.0f + oq;
    const float G = fmaf(1.4901161e-07f, fabsf(O), fmaf(5.9604645e-07f, fabsf(oq), fmaf(e_rot, g.inv_scale[k], 0.25f)));   // 2.5u|O| + 10u|o'| + 0.25 + E_rot
    const float mg = G * fabsf(idk);
    r.id[k] = idk;
    r.ncn[k] = fmaf(-O, idk, -mg);
    r.ncf[k] = fmaf(-O, idk, mg);
    const bool neg = dq < 0.0f;
    r.sn[k] = neg ? 0x7632u : 0x7610u;
    r.sf[k] = neg ? 0x7610u : 0x7632u;
  }
}
// entry and exit distance of the box stored in words (wx, wy, wz) of a compact node
__device__ __forceinline__ void grid_slab(const GridRay& r, unsigned int wx, unsigned int wy, unsigned int wz, float& tn,
                                          float& tf) {
  tn = fmaxf(fmaxf(fmaf(q_plane(wx, r.sn[0]), r.id[0], r.ncn[0]), fmaf(q_plane(wy, r.sn[1]), r.id[1], r.ncn[1])),
             fmaf(q_plane(wz, r.sn[2]), r.id[2], r.ncn[2]));
  tf = fminf(fminf(fmaf(q_plane(wx, r.sf[0]), r.id[0], r.ncf[0]), fmaf(q_plane(wy, r.sf[1]), r.id[1], r.ncf[1])),
             fmaf(q_plane(wz, r.sf[2]), r.id[2], r.ncf[2]));
}

// ---- per-ray traversal state of the wavefront kernel -------------------------------------------------
struct Walk {
  GridRay g;           // the ray in grid coordinates
  float tmax;          // min over provable hits of their thi
  int f_prev;
  int cur;             // node to visit next (>= 0 internal, < 0 leaf ~slot), TPMC_SENTINEL when the stack is empty
  int stash;           // leaf put aside for the next leaf phase (< 0), 0 = none
  int sp;
  int cs[TPMC_MAX_CAND];     // candidate slots
  float cl[TPMC_MAX_CAND];   // their tlo
  int nc;              // number of candidates; TPMC_MAX_CAND+1 = overflow
};

// start of a walk: everything but the ray in grid coordinates (w.g, set up when the warp fetched its chunk of rays)
__device__ __forceinline__ void walk_reset(Walk& w, int f_prev) {
  w.tmax = INFINITY;
  w.f_prev = f_prev;
  w.cur = 0;
  w.stash = 0;
  w.sp = 0;
  w.nc = 0;
#pragma unroll
  for (int k = 0; k < TPMC_MAX_CAND; ++k) { w.cs[k] = -1; w.cl[k] = 0.0f; }
}

// ---- seed-time cull on the compact copy of the top of the hierarchy (k_build_cull): can the ray touch any
// cut-off subtree?  Any-hit: true as soon as a box whose child ref is cut off (< 0) is touched.  Conservative
// like the traversal (same slab test); a walk deeper than the stack keeps the ray.
__device__ __forceinline__ bool cull_touch_q(const uint4* __restrict__ cc, const QuantGrid& g, const float o[3],
                                             const float d[3]) {
  GridRay r;
  grid_ray(r, g, o, d);
  int stack[16];
  int sp = 0, node = 0;
  for (;;) {
    uint4 a, b;
    ldg256u(cc + 2 * (size_t)node, a, b);
    float n0, f0, n1, f1;
    grid_slab(r, a.x, a.y, a.z, n0, f0);
    grid_slab(r, a.w, b.x, b.y, n1, f1);
    const bool h0 = !(fmaxf(n0, 0.0f) > f0), h1 = !(fmaxf(n1, 0.0f) > f1);
    const int c0 = (int)b.z, c1 = (int)b.w;
    if ((h0 && c0 < 0) || (h1 && c1 < 0)) return true;
    if (h0 && h1) {
      if (sp >= 16) return true;
      stack[sp++] = c1;
      node = c0;
    } else if (h0 || h1) {
      node = h0 ? c0 : c1;
    } else {
      if (sp == 0) return false;
      node = stack[--sp];
    }
  }
}

// Stack: TPMC_STACK_SMEM entries per thread in shared memory, [level][thread], above two guard entries that
// hold TPMC_SENTINEL (`stk` points at level 0; levels -1 and -2 are the guards, so popping an empty stack needs
// no test).  A ray that needs more gives up and is flagged for the full fp64 traversal of the resolve step
// (which has a deep stack), like a ray with too many candidates.
__device__ __forceinline__ int walk_pop(Walk& w, const int* stk, int sstride) {
  const int v = stk[(w.sp - 1) * sstride];
  w.sp = max(w.sp - 1, 0);
  return v;
}

__device__ __forceinline__ void walk_abort(Walk& w) {
  w.nc = TPMC_MAX_CAND + 1;
  w.cur = TPMC_SENTINEL;
  w.stash = 0;
  w.sp = 0;
}

// Candidate list: up to TPMC_MAX_CAND live entries in any of the slots (cs[k] < 0: free), w.nc of them; a provable hit
// that shrinks tmax frees the entries that start beyond it.  (Kept short: this runs with the few lanes whose facet was
// not a miss, and every instruction there costs the warp a full issue slot.)
__device__ __forceinline__ void walk_add_candidate(Walk& w, int slot, int cls, float tlo, float thi) {
  if (cls == TRI_HIT && thi < w.tmax) {
    w.tmax = thi;
    if (w.nc <= TPMC_MAX_CAND) {   // (an overflowed list stays overflowed)
#pragma unroll
      for (int k = 0; k < TPMC_MAX_CAND; ++k)
        if (w.cs[k] >= 0 && w.cl[k] > thi) { w.cs[k] = -1; --w.nc; }
    }
  }
  if (tlo > w.tmax) return;
  if (w.nc >= TPMC_MAX_CAND) { w.nc = TPMC_MAX_CAND + 1; return; }
  bool placed = false;
#pragma unroll
  for (int k = 0; k < TPMC_MAX_CAND; ++k)
    if (!placed && w.cs[k] < 0) { w.cs[k] = slot; w.cl[k] = tlo; placed = true; }
  ++w.nc;
}

// One step at a wide node (four slab tests; the children the ray enters are taken nearest first) -- requires
// w.cur >= 0 and != SENTINEL.  Node words (k_compact_wide, lbvh.cu): 3k .. 3k+2 = box of child k (x, y, z), each
// lo | hi << 16; 12-15 = the four child refs.
__device__ __forceinline__ void ce_sort(float& ka, int& ra, float& kb, int& rb) {   // compare-exchange: ka <= kb after
  const bool sw = kb < ka;
  const float k0 = fminf(ka, kb), k1 = fmaxf(ka, kb);
  const int r0 = sw ? rb : ra, r1 = sw ? ra : rb;
  ka = k0; kb = k1; ra = r0; rb = r1;
}
__device__ __forceinline__ void walk_node(Walk& w, const uint4* __restrict__ wnodes, int* stk, int sstride,
                                          TraceCounters& cnt) {
  uint4 a, b, c, d;
  ldg256u(wnodes + 4 * (size_t)w.cur, a, b);
  ldg256u(wnodes + 4 * (size_t)w.cur + 2, c, d);
  ++cnt.nodes;
  float n0, f0, n1, f1, n2, f2, n3, f3;
  grid_slab(w.g, a.x, a.y, a.z, n0, f0);
  grid_slab(w.g, a.w, b.x, b.y, n1, f1);
  grid_slab(w.g, b.z, b.w, c.x, n2, f2);
  grid_slab(w.g, c.y, c.z, c.w, n3, f3);
  // entered iff !(max(near, 0) > min(far, tmax)); the clamps also drop a NaN that survived three NaN plane distances
  // (zero direction).  Sort key: the entry distance (finite) of an entered child, +inf of a missed one.
  // (Whatever the keys, each of the four refs is safe to visit: a box at infinity sorted among the missed ones costs work, not a hit.)
  const float INF = __int_as_float(0x7F800000);
  float k0 = fmaxf(n0, 0.0f), k1 = fmaxf(n1, 0.0f), k2 = fmaxf(n2, 0.0f), k3 = fmaxf(n3, 0.0f);
  const bool h0 = !(k0 > fminf(f0, w.tmax)), h1 = !(k1 > fminf(f1, w.tmax)), h2 = !(k2 > fminf(f2, w.tmax)),
             h3 = !(k3 > fminf(f3, w.tmax));
  k0 = h0 ? k0 : INF; k1 = h1 ? k1 : INF; k2 = h2 ? k2 : INF; k3 = h3 ? k3 : INF;
  const int cnt_h = (int)h0 + (int)h1 + (int)h2 + (int)h3;
  int r0 = (int)d.x, r1 = (int)d.y, r2 = (int)d.z, r3 = (int)d.w;
  ce_sort(k0, r0, k1, r1);
  ce_sort(k2, r2, k3, r3);
  ce_sort(k0, r0, k2, r2);
  ce_sort(k1, r1, k3, r3);
  ce_sort(k1, r1, k2, r2);
  // Branch-free stack traffic.  The virtual sequence of what comes next is [r0 .. r_{cnt-1}, top, top2, ...]: the
  // entered children nearest first, then the stack.  Its first entry is next; if that is a leaf and no leaf is put
  // aside it is put aside (speculation: it is tested in the next leaf phase) and the second entry is next.  Children
  // r1 .. r_{cnt-1} are written above the top of the stack, the farthest lowest; the two entries below the top are
  // always read.  The stack has TPMC_STACK_SMEM + 3 rows above the two guard rows.
  const int sp = w.sp;
  if (sp > TPMC_STACK_SMEM) { walk_abort(w); return; }   // rare; three rows of headroom above TPMC_STACK_SMEM
  const int top = stk[(sp - 1) * sstride], top2 = stk[(sp - 2) * sstride];
  // r_j (j = 1..3) goes to row sp + ((cnt - 1 - j) & 3): an entered child lands at sp + cnt - 1 - j, a missed one
  // (j >= cnt) above the new top, where it is never read -- three unconditional stores, no branch (predicated stores
  // were measured: 4 % slower)
  stk[(sp + ((cnt_h - 2) & 3)) * sstride] = r1;
  stk[(sp + ((cnt_h - 3) & 3)) * sstride] = r2;
  stk[(sp + (cnt_h & 3)) * sstride] = r3;
  const int e0 = cnt_h >= 1 ? r0 : top;
  const int e1 = cnt_h >= 2 ? r1 : (cnt_h == 1 ? top : top2);
  const bool take = e0 < 0 && w.stash == 0;
  if (take) w.stash = e0;
  w.cur = take ? e1 : e0;
  w.sp = max(sp + cnt_h - (take ? 2 : 1), 0);
}

// One leaf step (fp32 facet classification of the leaf put aside), then the next leaf, if the walk stands at
// one, is put aside in turn.
__device__ __forceinline__ void walk_leaf(Walk& w, const float4* __restrict__ tris, const float o[3], const float d[3],
                                          int* stk, int sstride, TraceCounters& cnt) {
  const int slot = ~w.stash;
  // all three loads at once (the source facet is rare: waiting for q0 before asking for q1, q2 cost a second round trip)
  const float4 q0 = __ldg(tris + 3 * (size_t)slot + 0);
  const float4 q1 = __ldg(tris + 3 * (size_t)slot + 1);
  const float4 q2 = __ldg(tris + 3 * (size_t)slot + 2);
  if (__float_as_int(q0.w) != w.f_prev) {
    ++cnt.tris;
    float tlo, thi;
    const int cls = tri_filter(q0, q1, q2, o, d, tlo, thi);
    if (cls != TRI_MISS) walk_add_candidate(w, slot, cls, tlo, thi);
  }
  w.stash = 0;
  if (w.cur < 0) {
    w.stash = w.cur;
    w.cur = walk_pop(w, stk, sstride);
  }
}

// ---- exact closest hit by a full fp64 traversal (stragglers, candidate overflow) ----------------------
// Closest hit ("the closest intersection point to the initial position becomes the first
// collision"), ties to the smallest facet index (A12), source facet excluded (A11).
__device__ __forceinline__ Hit closest_hit(const float4* __restrict__ nodes, const float4* __restrict__ tris,
                                           const float of[3], const float df[3], int f_prev, int* sstack,
                                           int sstride, TraceCounters& cnt) {
  Hit best;
  best.tau = INFINITY; best.facet = -1; best.slot = -1;
  const float id[3] = {1.0f / df[0], 1.0f / df[1], 1.0f / df[2]};
  float tmax = INFINITY;
  int lstack[TPMC_STACK_LOCAL];
  int sp = 0;
  int node = 0;
  for (;;) {
    const float4 n0 = __ldg(nodes + 4 * (size_t)node + 0);
    const float4 n1 = __ldg(nodes + 4 * (size_t)node + 1);
    const float4 n2 = __ldg(nodes + 4 * (size_t)node + 2);
    const float4 n3 = __ldg(nodes + 4 * (size_t)node + 3);
    ++cnt.nodes;
    float t0, t1;
    const bool h0 = slab(n0.x, n0.y, n0.z, n0.w, n1.x, n1.y, of, id, tmax, t0);
    const bool h1 = slab(n1.z, n1.w, n2.x, n2.y, n2.z, n2.w, of, id, tmax, t1);
    int c0 = __float_as_int(n3.x), c1 = __float_as_int(n3.y);
    int next;
    if (h0 && h1) {
      if (t1 < t0) { const int t = c0; c0 = c1; c1 = t; }
      if (sp < TPMC_STACK_SMEM) sstack[sp * sstride] = c1; else lstack[sp - TPMC_STACK_SMEM] = c1;
      ++sp;
      next = c0;
    } else if (h0) {
      next = c0;
    } else if (h1) {
      next = c1;
    } else {
      if (sp == 0) break;
      --sp;
      next = (sp < TPMC_STACK_SMEM) ? sstack[sp * sstride] : lstack[sp - TPMC_STACK_SMEM];
    }
    bool done = false;
    while (next < 0) {
      const int slot = ~next;
      const float4 q0 = __ldg(tris + 3 * (size_t)slot + 0);
      const int facet = __float_as_int(q0.w);
      if (facet != f_prev) {
        const float4 q1 = __ldg(tris + 3 * (size_t)slot + 1);
        const float4 q2 = __ldg(tris + 3 * (size_t)slot + 2);
        ++cnt.tris;
        double tau;
        if (facet_test(q0, q1, q2, of, df, tau) && (tau < best.tau || (tau == best.tau && facet < best.facet))) {
          best.tau = tau; best.facet = facet; best.slot = slot;
          tmax = __double2float_ru(tau);
        }
      }
      if (sp == 0) { done = true; break; }
      --sp;
      next = (sp < TPMC_STACK_SMEM) ? sstack[sp * sstride] : lstack[sp - TPMC_STACK_SMEM];
    }
    if (done) break;
    node = next;
  }
  return best;
}

// Resolve a candidate list with the exact test: smallest tau, ties to the smallest facet index.
__device__ __forceinline__ Hit resolve_candidates(const float4* __restrict__ tris, const int4 cand, const float of[3],
                                                  const float df[3], unsigned int& ntests) {
  Hit best;
  best.tau = INFINITY; best.facet = -1; best.slot = -1;
  const int cs[4] = {cand.x, cand.y, cand.z, cand.w};
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int slot = cs[k];
    if (slot < 0) continue;
    const float4 q0 = __ldg(tris + 3 * (size_t)slot + 0), q1 = __ldg(tris + 3 * (size_t)slot + 1),
                 q2 = __ldg(tris + 3 * (size_t)slot + 2);
    const int facet = __float_as_int(q0.w);
    double tau;
    ++ntests;
    if (facet_test(q0, q1, q2, of, df, tau) && (tau < best.tau || (tau == best.tau && facet < best.facet))) {
      best.tau = tau; best.facet = facet; best.slot = slot;
    }
  }
  return best;
}

// ---- O11: surface interaction (P:73 diffuse re-emission at T_W; P:53 specular; Maxwell mix A7) ------
// w: the four words of Philox block 2+k.  Returns v_out in fp64 (the caller rounds it to fp32, O9).
// sin_e, phi: elevation (sin) above the facet plane and azimuth in the frame (e1, n_eff x e1) of fp32(v_out), for
// the comparison with the facet's escape horizon (k_horizon, lbvh.cu); fp32 accuracy is enough (the stored
// horizon carries a safety factor of 1e-4 and an azimuth margin of 2e-3 rad).
__device__ __forceinline__ void reflect(const float4 q0, const float4 q1, const float4 q2, const float vf[3],
                                        double sigma, double cW, const uint4 w, double vout[3], float& sin_e, float& phi) {
  const double p0[3] = {(double)q0.x, (double)q0.y, (double)q0.z};
  double e1[3], e2[3], Ng[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) { e1[k] = (double)(&q1.x)[k] - p0[k]; e2[k] = (double)(&q2.x)[k] - p0[k]; }
  Ng[0] = e1[1] * e2[2] - e1[2] * e2[1];
  Ng[1] = e1[2] * e2[0] - e1[0] * e2[2];
  Ng[2] = e1[0] * e2[1] - e1[1] * e2[0];
  const double nl = sqrt((Ng[0] * Ng[0] + Ng[1] * Ng[1]) + Ng[2] * Ng[2]);
  const double v[3] = {(double)vf[0], (double)vf[1], (double)vf[2]};
  const double inl = 1.0 / nl;   // one division per frame vector (the unit vectors are within 1 ulp either way)
  double ne[3] = {Ng[0] * inl, Ng[1] * inl, Ng[2] * inl};
  const double vn = (v[0] * ne[0] + v[1] * ne[1]) + v[2] * ne[2];
  if (!(vn < 0.0)) { ne[0] = -ne[0]; ne[1] = -ne[1]; ne[2] = -ne[2]; }   // n_eff faces the incoming particle
  const double el = sqrt((e1[0] * e1[0] + e1[1] * e1[1]) + e1[2] * e1[2]);
  const double iel = 1.0 / el;
  const double t1[3] = {e1[0] * iel, e1[1] * iel, e1[2] * iel};
  const double t2[3] = {ne[1] * t1[2] - ne[2] * t1[1], ne[2] * t1[0] - ne[0] * t1[2], ne[0] * t1[1] - ne[1] * t1[0]};
  if (u01(w.x) < sigma) {
    // diffuse, fully accommodated: flux-weighted half-Maxwellian at T_W (A6); tangent basis A17
    const double an = sqrt(-log(u01(w.y)));
    const double at = sqrt(-log(u01(w.z)));
    double sa, ca;
    sincospi(2.0 * u01(w.w), &sa, &ca);
#pragma unroll
    for (int k = 0; k < 3; ++k) vout[k] = cW * (an * ne[k] + at * (ca * t1[k] + sa * t2[k]));
  } else {
    const double vne = (v[0] * ne[0] + v[1] * ne[1]) + v[2] * ne[2];
#pragma unroll
    for (int k = 0; k < 3; ++k) vout[k] = v[k] - 2.0 * vne * ne[k];
  }
  const float r[3] = {(float)vout[0], (float)vout[1], (float)vout[2]};
  const float rn = r[0] * (float)ne[0] + r[1] * (float)ne[1] + r[2] * (float)ne[2];
  const float r1 = r[0] * (float)t1[0] + r[1] * (float)t1[1] + r[2] * (float)t1[2];
  const float r2 = r[0] * (float)t2[0] + r[1] * (float)t2[1] + r[2] * (float)t2[2];
  sin_e = rn * rsqrtf(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);   // NaN for a zero velocity: never above a horizon
  phi = atan2f(r2, r1);
}

__device__ __forceinline__ unsigned long long fnv1a_facet(unsigned long long h, int facet) {
  const unsigned int w = (unsigned int)facet;
#pragma unroll
  for (int b = 0; b < 4; ++b) {
    h ^= (unsigned long long)((w >> (8 * b)) & 0xFFu);
    h *= 0x100000001B3ull;
  }
  return h;
}
