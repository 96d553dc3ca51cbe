// trace.cuh -- steps a3/a4 device code: closest-hit traversal of the LBVH and the surface interaction.
//
// Precision contract (reading A9): the mesh and the ray (o, d) are fp32 VALUES; which facet
// is hit is decided as in exact arithmetic on those values.  The hierarchy is walked with fp32 slab
// tests made conservative by an explicit rounding-error margin (a box is never wrongly skipped), and
// every facet whose box the ray touches is decided by the fp64 edge functions below, evaluated with
// separately rounded multiplies and adds (no FMA contraction): that keeps the shared-edge function of
// two neighbouring facets exactly antisymmetric, i.e. the test watertight, and equal to DESIGN.md O10.
#pragma once

#include "common.cuh"

#define TPMC_STACK_SMEM 24      // stack entries per thread kept in shared memory
#define TPMC_STACK_LOCAL 80     // overflow entries (a Karras tree over 64-bit keys + index is <= 97 deep)
#define TPMC_SENTINEL ((int)0x80000000)

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

__device__ __forceinline__ bool facet_test(const float4 q0, const float4 q1, const float4 q2, const double o[3],
                                           const double d[3], double& tau) {
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

// ---- conservative fp32 slab test -------------------------------------------------------------------
// Each plane distance (lo - o) * (1/d) carries three roundings: relative error <= 3 * 2^-24.  min/max are
// exact and x -> x -+ 4u|x| is monotone, so one margin on the entry and one on the exit make the test
// conservative.  NaN (0 * inf when d = 0 and o on the plane) is dropped by fminf/fmaxf.
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

// Closest hit ("the closest intersection point to the initial position becomes the first
// collision"), ties to the smallest facet index (A12), source facet excluded (A11).
// `sstack` points at this thread's column of the shared-memory stack (stride = blockDim.x).
__device__ __forceinline__ Hit closest_hit(const float4* __restrict__ nodes, const float4* __restrict__ tris,
                                           const float of[3], const float df[3], int f_prev, int* sstack,
                                           int sstride, TraceCounters& cnt) {
  Hit best;
  best.tau = INFINITY; best.facet = -1; best.slot = -1;
  const double o[3] = {(double)of[0], (double)of[1], (double)of[2]};
  const double d[3] = {(double)df[0], (double)df[1], (double)df[2]};
  const float id[3] = {1.0f / df[0], 1.0f / df[1], 1.0f / df[2]};
  float tmax = INFINITY;
  int lstack[TPMC_STACK_LOCAL];
  int sp = 0;
  int node = 0;
  for (;;) {
    // ---- internal node: test both child boxes
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
    // ---- leaves
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
        if (facet_test(q0, q1, q2, o, d, tau) && (tau < best.tau || (tau == best.tau && facet < best.facet))) {
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

// ---- O11: surface interaction (P:73 diffuse re-emission at T_W; P:53 specular; Maxwell mix A7) ------
// u: the four uniforms of Philox block 2+k.  Returns v_out in fp64 (the caller rounds it to fp32, O9).
__device__ __forceinline__ void reflect(const float4 q0, const float4 q1, const float4 q2, const float vf[3],
                                        double sigma, double cW, const uint4 w, double vout[3]) {
  const double p0[3] = {(double)q0.x, (double)q0.y, (double)q0.z};
  double e1[3], e2[3], Ng[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) { e1[k] = (double)(&q1.x)[k] - p0[k]; e2[k] = (double)(&q2.x)[k] - p0[k]; }
  Ng[0] = e1[1] * e2[2] - e1[2] * e2[1];
  Ng[1] = e1[2] * e2[0] - e1[0] * e2[2];
  Ng[2] = e1[0] * e2[1] - e1[1] * e2[0];
  const double nl = sqrt((Ng[0] * Ng[0] + Ng[1] * Ng[1]) + Ng[2] * Ng[2]);
  const double v[3] = {(double)vf[0], (double)vf[1], (double)vf[2]};
  double ne[3] = {Ng[0] / nl, Ng[1] / nl, Ng[2] / nl};
  const double vn = (v[0] * ne[0] + v[1] * ne[1]) + v[2] * ne[2];
  if (!(vn < 0.0)) { ne[0] = -ne[0]; ne[1] = -ne[1]; ne[2] = -ne[2]; }   // n_eff faces the incoming particle
  if (u01(w.x) < sigma) {
    // diffuse, fully accommodated: flux-weighted half-Maxwellian at T_W (A6); tangent basis A17
    const double el = sqrt((e1[0] * e1[0] + e1[1] * e1[1]) + e1[2] * e1[2]);
    const double t1[3] = {e1[0] / el, e1[1] / el, e1[2] / el};
    const double t2[3] = {ne[1] * t1[2] - ne[2] * t1[1], ne[2] * t1[0] - ne[0] * t1[2], ne[0] * t1[1] - ne[1] * t1[0]};
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
