/*
 * tpmc_oracle.c -- CPU ORACLE for the TPMC hot path of arXiv 1312.3691.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may load it.  It shares no code,
 * header, table or helper with the CUDA path (paper_1312_3691_b200/csrc); the two
 * share only data (mesh arrays, parameters) and the definitions written in DESIGN.md.
 *
 * Plain C, one thread, fp64 throughout, the algorithm step by step in the paper's
 * order (seed -> closest hit -> surface interaction -> accumulate -> repeat).  Each
 * function cites the passage of /root/reference/PAPER.md it follows ("P:<line>") and
 * the reading of SURVEY.md 8(c) / DESIGN.md it takes ("O<n>", "A<n>", "G<n>").
 * Compile with -O2 -ffp-contract=off (no -ffast-math): arithmetic is evaluated as written.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): Philox known answers (P1), flux
 * integral vs quadrature (P2), sampler CDFs by KS test and printed limits (P3,P4),
 * hit fraction (R/r)^2 (P5), facet counts (P6), convex-body force = panel sum (P7),
 * Sentman / sphere / cylinder closed forms (P8), symmetry (P9), equilibrium (P10),
 * control-volume invariance and rotation covariance (P11), BVH == brute force (P12),
 * specular limits (P13), Pratt's concave hemisphere (P14), torque about an off-centre
 * reference point = panel sum of (centroid - x_ref) x F_f, and the A14 shift identity (P16).
 * Per-facet wall temperature / accommodation and partial energy accommodation (NEXT-3, readings A22/A23 of
 * DESIGN.md): panel sum with per-facet S_W and sigma, quadrature of the re-emission momentum flux with
 * T_r = alpha_E T_W + (1 - alpha_E) m v_in^2 / (3 k_B), and alpha_E = 1 / uniform arrays reproducing the scalar run (P17).
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_KB 1.380649e-23 /* J/K */
#define SQRTPI 1.7724538509055160272981674833411
#define TWOPI 6.2831853071795864769252867665590

/* ------------------------------------------------------------------ O3: random stream */
/* Philox4x32-10 (Salmon et al. 2011).  key=(seed_lo,seed_hi), counter=(i_lo,i_hi,block,0). */
void oracle_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* word -> uniform in (0,1), A16: u = (w + 0.5) * 2^-32 */
static double u01(uint32_t w) { return ((double)w + 0.5) * (1.0 / 4294967296.0); }

static void particle_block(uint64_t seed, uint64_t i, uint32_t block, double u[4]) {
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t ctr[4] = {(uint32_t)i, (uint32_t)(i >> 32), block, 0u};
  uint32_t w[4];
  oracle_philox4x32_10(key, ctr, w);
  for (int k = 0; k < 4; ++k) u[k] = u01(w[k]);
}

/* ------------------------------------------------------------------ O2: flux, eq. (10) */
/* chi(s) = e^{-s^2} + sqrt(pi) s (1+erf s), the bracket of eq. (8), with 1+erf = erfc(-s) (A4) */
static double chi(double s) { return exp(-s * s) + SQRTPI * s * erfc(-s); }

/* Gamma/(c n r^2) = sqrt(pi) e^{-S^2} + (pi/(2S) + pi S) erf S ; S<1e-4: erf(S)/S series (A19) */
double oracle_flux_bracket(double S) {
  const double pi = 3.14159265358979323846;
  double erf_over_S = (S < 1e-4) ? (2.0 / SQRTPI) * (1.0 - S * S / 3.0) : erf(S) / S;
  return SQRTPI * exp(-S * S) + 0.5 * pi * erf_over_S + pi * S * erf(S);
}
double oracle_flux(double S, double c, double n, double r) { return oracle_flux_bracket(S) * c * n * r * r; }

/* ------------------------------------------------------------------ O5: position, eq. (11) */
/* Antiderivative of chi:  Gt(y) = (sqrt(pi)/4)(1+2y^2) erfc(-y) + (y/2) e^{-y^2}  (Gt' = chi).
 * In t = sin(phi):  dP = g(phi) dphi = chi(S t) dt / I,  so  H(t) = [Gt(St) - Gt(-S)] / [Gt(S) - Gt(-S)]. */
static double Gt(double y) { return 0.25 * SQRTPI * (1.0 + 2.0 * y * y) * erfc(-y) + 0.5 * y * exp(-y * y); }

double oracle_position_cdf(double t, double S) {
  if (S < 1e-4) { /* A19: chi(s) = 1 + sqrt(pi) s + s^2 + O(s^4) integrated in closed form */
    double num = (t + 1.0) + 0.5 * SQRTPI * S * (t * t - 1.0) + S * S * (t * t * t + 1.0) / 3.0;
    return num / (2.0 + 2.0 * S * S / 3.0);
  }
  double g0 = Gt(-S);
  return (Gt(S * t) - g0) / (Gt(S) - g0);
}
static double position_pdf(double t, double S) { /* dH/dt */
  if (S < 1e-4) return (1.0 + SQRTPI * S * t + S * S * t * t) / (2.0 + 2.0 * S * S / 3.0);
  return S * chi(S * t) / (Gt(S) - Gt(-S));
}
/* A2: t = H^{-1}(u) by bracketed Newton (bisection whenever Newton leaves the bracket) */
double oracle_position_inv(double u, double S) {
  double lo = -1.0, hi = 1.0, t = 0.0;
  for (int it = 0; it < 400; ++it) {
    double f = oracle_position_cdf(t, S) - u;
    if (f > 0.0) hi = t; else lo = t;
    double d = position_pdf(t, S);
    double tn = (d > 0.0) ? t - f / d : 0.5 * (lo + hi);
    if (!(tn > lo && tn < hi)) tn = 0.5 * (lo + hi);
    if (fabs(tn - t) <= 2e-16 || hi - lo <= 2e-16) { t = tn; break; }
    t = tn;
  }
  return t;
}

/* ------------------------------------------------------------------ O7: normal speed, eq. (14a) P:194 (G2) */
/* x = v_n/c >= 0, density 2x e^{-(x-s)^2}/chi(s).  Survival 1-F(x|s) = Q(x)/chi(s),
 * Q(x) = e^{-(x-s)^2} + sqrt(pi) s erfc(x-s)  (Q(0) = chi(s), Q' = -2x e^{-(x-s)^2}). */
static double Qsurv(double x, double s) { double z = x - s; return exp(-z * z) + SQRTPI * s * erfc(z); }
double oracle_vn_cdf(double x, double s) { return 1.0 - Qsurv(x, s) / chi(s); }
double oracle_vn_inv(double u, double s) {
  double target = (1.0 - u) * chi(s);
  double lo = 0.0, hi = (s > 0.0 ? s : 0.0) + 8.0;
  double x = (s > 0.0 ? s : 0.0) + 0.7;
  for (int it = 0; it < 400; ++it) {
    double f = Qsurv(x, s) - target; /* decreasing in x */
    if (f > 0.0) lo = x; else hi = x;
    double z = x - s;
    double d = -2.0 * x * exp(-z * z);
    double xn = (d < 0.0) ? x - f / d : 0.5 * (lo + hi);
    if (!(xn > lo && xn < hi)) xn = 0.5 * (lo + hi);
    if (fabs(xn - x) <= 1e-16 * (1.0 + x) || hi - lo <= 1e-16 * (1.0 + x)) { x = xn; break; }
    x = xn;
  }
  return x;
}

/* ------------------------------------------------------------------ O8: rotation, eq. (15) P:207-209 (A5) */
/* R zhat = ztilde, ztilde = -V/|V| (upstream, A1).  Rodrigues about u = (zhat x ztilde)/|.|,
 * cos(beta) = zhat.ztilde, sin(beta) = |zhat x ztilde|.  Row-major R[9]. */
void oracle_rotation(const double V[3], double R[9]) {
  double sp = sqrt(V[0] * V[0] + V[1] * V[1] + V[2] * V[2]);
  double zt[3] = {0.0, 0.0, 1.0};
  if (sp > 0.0) { zt[0] = -V[0] / sp; zt[1] = -V[1] / sp; zt[2] = -V[2] / sp; }
  double ax = -zt[1], ay = zt[0]; /* zhat x ztilde = (-zt.y, zt.x, 0) */
  double sb = sqrt(ax * ax + ay * ay), cb = zt[2];
  memset(R, 0, 9 * sizeof(double));
  if (sb < 1e-12) {
    R[0] = 1.0;
    R[4] = (cb > 0.0) ? 1.0 : -1.0;
    R[8] = (cb > 0.0) ? 1.0 : -1.0;
    return;
  }
  double ux = ax / sb, uy = ay / sb, uz = 0.0, omc = 1.0 - cb;
  R[0] = cb + ux * ux * omc;      R[1] = ux * uy * omc - uz * sb; R[2] = ux * uz * omc + uy * sb;
  R[3] = uy * ux * omc + uz * sb; R[4] = cb + uy * uy * omc;      R[5] = uy * uz * omc - ux * sb;
  R[6] = uz * ux * omc - uy * sb; R[7] = uz * uy * omc + ux * sb; R[8] = cb + uz * uz * omc;
}

/* ------------------------------------------------------------------ mesh */
typedef struct {
  double lo[3], hi[3];
  int32_t left, right; /* children, or -1 */
  int32_t first, count; /* leaf range in perm[] */
} bvh_node;

typedef struct oracle_mesh {
  int64_t nv, nt;
  float* v;       /* [nv][3] */
  int32_t* idx;   /* [nt][3] */
  uint8_t* flags; /* [nt] */
  double centre[3], Rb;
  double lo[3], hi[3]; /* AABB of the vertices */
  bvh_node* nodes;
  int32_t n_nodes;
  int32_t* perm;
  double* surf_TW;    /* [nt] wall temperature per facet, or NULL: the run's T_W (A23) */
  double* surf_sigma; /* [nt] accommodation per facet, or NULL: the run's sigma (A23) */
} oracle_mesh;

static void tri_corner(const oracle_mesh* m, int64_t f, int k, double p[3]) {
  const float* q = m->v + 3 * (int64_t)m->idx[3 * f + k];
  p[0] = (double)q[0]; p[1] = (double)q[1]; p[2] = (double)q[2];
}

static int32_t bvh_build(oracle_mesh* m, double* cen, int32_t first, int32_t count) {
  int32_t me = m->n_nodes++;
  bvh_node* nd = &m->nodes[me];
  for (int a = 0; a < 3; ++a) { nd->lo[a] = INFINITY; nd->hi[a] = -INFINITY; }
  double clo[3] = {INFINITY, INFINITY, INFINITY}, chi_[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int32_t i = first; i < first + count; ++i) {
    int32_t f = m->perm[i];
    for (int k = 0; k < 3; ++k) {
      double p[3];
      tri_corner(m, f, k, p);
      for (int a = 0; a < 3; ++a) { if (p[a] < nd->lo[a]) nd->lo[a] = p[a]; if (p[a] > nd->hi[a]) nd->hi[a] = p[a]; }
    }
    for (int a = 0; a < 3; ++a) { double c = cen[3 * f + a]; if (c < clo[a]) clo[a] = c; if (c > chi_[a]) chi_[a] = c; }
  }
  for (int a = 0; a < 3; ++a) { /* generous padding: the BVH only has to be conservative (P12) */
    double pad = 1e-9 * (1.0 + fabs(nd->lo[a]) + fabs(nd->hi[a]));
    nd->lo[a] -= pad; nd->hi[a] += pad;
  }
  nd->left = nd->right = -1; nd->first = first; nd->count = count;
  if (count <= 4) return me;
  int axis = 0;
  if (chi_[1] - clo[1] > chi_[axis] - clo[axis]) axis = 1;
  if (chi_[2] - clo[2] > chi_[axis] - clo[axis]) axis = 2;
  if (!(chi_[axis] - clo[axis] > 0.0)) return me; /* all centroids equal: keep as a leaf */
  /* median split by nth_element-style partial sort (simple insertion of a quickselect) */
  int32_t lo = first, hi = first + count - 1, mid = first + count / 2;
  while (lo < hi) {
    double pv = cen[3 * m->perm[(lo + hi) / 2] + axis];
    int32_t i = lo, j = hi;
    while (i <= j) {
      while (cen[3 * m->perm[i] + axis] < pv) ++i;
      while (cen[3 * m->perm[j] + axis] > pv) --j;
      if (i <= j) { int32_t t = m->perm[i]; m->perm[i] = m->perm[j]; m->perm[j] = t; ++i; --j; }
    }
    if (mid <= j) hi = j; else if (mid >= i) lo = i; else break;
  }
  int32_t l = bvh_build(m, cen, first, mid - first);
  int32_t r = bvh_build(m, cen, mid, first + count - mid);
  m->nodes[me].left = l; m->nodes[me].right = r;
  return me;
}

oracle_mesh* oracle_mesh_create(const float* v, int64_t nv, const int32_t* idx, int64_t nt, const uint8_t* flags) {
  if (!v || !idx || nv < 3 || nt < 1) return NULL;
  oracle_mesh* m = (oracle_mesh*)calloc(1, sizeof(oracle_mesh));
  m->nv = nv; m->nt = nt;
  m->v = (float*)malloc(sizeof(float) * 3 * nv); memcpy(m->v, v, sizeof(float) * 3 * nv);
  m->idx = (int32_t*)malloc(sizeof(int32_t) * 3 * nt); memcpy(m->idx, idx, sizeof(int32_t) * 3 * nt);
  m->flags = (uint8_t*)calloc(nt, 1);
  if (flags) memcpy(m->flags, flags, nt);
  /* O1/A10: control-sphere centre = centre of the AABB of the vertices, R_b = max distance to it */
  double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int64_t i = 0; i < nv; ++i)
    for (int a = 0; a < 3; ++a) { double p = (double)v[3 * i + a]; if (p < lo[a]) lo[a] = p; if (p > hi[a]) hi[a] = p; }
  for (int a = 0; a < 3; ++a) { m->centre[a] = 0.5 * (lo[a] + hi[a]); m->lo[a] = lo[a]; m->hi[a] = hi[a]; }
  double r2 = 0.0;
  for (int64_t i = 0; i < nv; ++i) {
    double dx = (double)v[3 * i] - m->centre[0], dy = (double)v[3 * i + 1] - m->centre[1], dz = (double)v[3 * i + 2] - m->centre[2];
    double d2 = (dx * dx + dy * dy) + dz * dz;
    if (d2 > r2) r2 = d2;
  }
  m->Rb = sqrt(r2);
  /* the oracle's own simple median-split BVH (validated against brute force, P12) */
  double* cen = (double*)malloc(sizeof(double) * 3 * nt);
  m->perm = (int32_t*)malloc(sizeof(int32_t) * nt);
  for (int64_t f = 0; f < nt; ++f) {
    m->perm[f] = (int32_t)f;
    double p0[3], p1[3], p2[3];
    tri_corner(m, f, 0, p0); tri_corner(m, f, 1, p1); tri_corner(m, f, 2, p2);
    for (int a = 0; a < 3; ++a) cen[3 * f + a] = (p0[a] + p1[a] + p2[a]) / 3.0;
  }
  m->nodes = (bvh_node*)malloc(sizeof(bvh_node) * (size_t)(2 * nt + 1));
  m->n_nodes = 0;
  bvh_build(m, cen, 0, (int32_t)nt);
  free(cen);
  return m;
}
void oracle_mesh_destroy(oracle_mesh* m) {
  if (!m) return;
  free(m->v); free(m->idx); free(m->flags); free(m->nodes); free(m->perm); free(m->surf_TW); free(m->surf_sigma); free(m);
}
/* A23: surface properties per facet ("arbitrary surface interaction"; re-emission "determined by the satellite
 * surface temperature").  Either array may be NULL (back to the run's scalar). */
void oracle_mesh_set_surface(oracle_mesh* m, const double* T_W, const double* sigma) {
  free(m->surf_TW); free(m->surf_sigma);
  m->surf_TW = NULL; m->surf_sigma = NULL;
  if (T_W) { m->surf_TW = (double*)malloc(sizeof(double) * (size_t)m->nt); memcpy(m->surf_TW, T_W, sizeof(double) * (size_t)m->nt); }
  if (sigma) { m->surf_sigma = (double*)malloc(sizeof(double) * (size_t)m->nt); memcpy(m->surf_sigma, sigma, sizeof(double) * (size_t)m->nt); }
}
void oracle_mesh_bounds(const oracle_mesh* m, double centre[3], double* Rb) {
  for (int a = 0; a < 3; ++a) centre[a] = m->centre[a];
  *Rb = m->Rb;
}

/* ------------------------------------------------------------------ O10: closest hit P:71 (A11, A12) */
/* Ray o + tau d (o, d = fp32 values widened exactly).  Facet f with corners p0,p1,p2:
 *   a=p0-o, b=p1-o, c=p2-o ; edge functions w0=[d,b,c], w1=[d,c,a], w2=[d,a,b] (scalar triple products)
 *   Ng=(p1-p0)x(p2-p0) ; det=d.Ng ; one-sided facets need det<0 (front face), two-sided det!=0
 *   inside iff all w>=0 or all w<=0 (watertight rule: zeros count as inside)
 *   tau=(a.Ng)/det, need tau>0.
 * Returns 1 and *tau on a hit. */
static double dot3(const double x[3], const double y[3]) { return (x[0] * y[0] + x[1] * y[1]) + x[2] * y[2]; }
static void cross3(const double x[3], const double y[3], double z[3]) {
  z[0] = x[1] * y[2] - x[2] * y[1];
  z[1] = x[2] * y[0] - x[0] * y[2];
  z[2] = x[0] * y[1] - x[1] * y[0];
}
static int facet_test(const oracle_mesh* m, int64_t f, const double o[3], const double d[3], double* tau) {
  double p0[3], p1[3], p2[3], a[3], b[3], c[3], e1[3], e2[3], Ng[3], bc[3], ca[3], ab[3];
  tri_corner(m, f, 0, p0); tri_corner(m, f, 1, p1); tri_corner(m, f, 2, p2);
  for (int k = 0; k < 3; ++k) { a[k] = p0[k] - o[k]; b[k] = p1[k] - o[k]; c[k] = p2[k] - o[k]; e1[k] = p1[k] - p0[k]; e2[k] = p2[k] - p0[k]; }
  cross3(e1, e2, Ng);
  double det = dot3(d, Ng);
  if (m->flags[f] & 1) { if (det == 0.0) return 0; }
  else if (!(det < 0.0)) return 0;
  cross3(b, c, bc); cross3(c, a, ca); cross3(a, b, ab);
  double w0 = dot3(d, bc), w1 = dot3(d, ca), w2 = dot3(d, ab);
  int allpos = (w0 >= 0.0) && (w1 >= 0.0) && (w2 >= 0.0);
  int allneg = (w0 <= 0.0) && (w1 <= 0.0) && (w2 <= 0.0);
  if (!(allpos || allneg)) return 0;
  double t = dot3(a, Ng) / det;
  if (!(t > 0.0)) return 0;
  *tau = t;
  return 1;
}

static int32_t closest_brute(const oracle_mesh* m, const double o[3], const double d[3], int32_t f_prev, double* tau_out) {
  int32_t best = -1; double bt = INFINITY;
  for (int64_t f = 0; f < m->nt; ++f) {
    if (f == f_prev) continue;
    double t;
    if (facet_test(m, f, o, d, &t) && t < bt) { bt = t; best = (int32_t)f; } /* ascending f: ties keep the smallest index */
  }
  *tau_out = bt;
  return best;
}

static int slab(const bvh_node* nd, const double o[3], const double d[3], double tmax) {
  double t0 = 0.0, t1 = tmax;
  for (int a = 0; a < 3; ++a) {
    if (d[a] == 0.0) { if (o[a] < nd->lo[a] || o[a] > nd->hi[a]) return 0; continue; }
    double ta = (nd->lo[a] - o[a]) / d[a], tb = (nd->hi[a] - o[a]) / d[a];
    if (ta > tb) { double s = ta; ta = tb; tb = s; }
    ta -= 1e-12 * fabs(ta); tb += 1e-12 * fabs(tb);
    if (ta > t0) t0 = ta;
    if (tb < t1) t1 = tb;
    if (t0 > t1) return 0;
  }
  return 1;
}

static int32_t closest_bvh(const oracle_mesh* m, const double o[3], const double d[3], int32_t f_prev, double* tau_out) {
  int32_t best = -1; double bt = INFINITY;
  int32_t stack[256]; int sp = 0;
  stack[sp++] = 0;
  while (sp > 0) {
    const bvh_node* nd = &m->nodes[stack[--sp]];
    if (!slab(nd, o, d, bt * (1.0 + 1e-12))) continue;
    if (nd->left < 0) {
      for (int32_t i = nd->first; i < nd->first + nd->count; ++i) {
        int32_t f = m->perm[i];
        if (f == f_prev) continue;
        double t;
        if (facet_test(m, f, o, d, &t) && (t < bt || (t == bt && f < best))) { bt = t; best = f; }
      }
    } else {
      if (sp + 2 > 256) return -2;
      stack[sp++] = nd->left; stack[sp++] = nd->right;
    }
  }
  *tau_out = bt;
  return best;
}

int32_t oracle_closest_hit(const oracle_mesh* m, const float o32[3], const float d32[3], int32_t f_prev, int use_bvh, double* tau) {
  double o[3] = {(double)o32[0], (double)o32[1], (double)o32[2]};
  double d[3] = {(double)d32[0], (double)d32[1], (double)d32[2]};
  return use_bvh ? closest_bvh(m, o, d, f_prev, tau) : closest_brute(m, o, d, f_prev, tau);
}

/* ------------------------------------------------------------------ parameters */
typedef struct {
  double n, T_inf, T_W;
  double V[3];
  double accommodation;
  int32_t n_species;
  const double* m;
  const double* x;
  double cv_radius_factor;
  uint64_t N, first, count, seed;
  uint32_t max_bounces;
  double x_ref[3];
  double energy_accommodation; /* alpha_E (A22); 1 = full accommodation to T_W */
  int32_t control_volume;      /* 0 sphere (the paper's scheme); 1 box, flux-weighted; 2 box, inward speed NOT flux-weighted (A24, A25) */
  int32_t pad_;
} oracle_params;

typedef struct { uint64_t hits, segments, escaped, truncated; } oracle_stats;

/* ------------------------------------------------------------------ rectangular control volume (A24, A25) */
/* "placing particles with a random uniform distribution on the six faces of a rectangular control volume.  The number
 * of particles to cross each face derives from the analytical molecular flux across a flat plate with given normal
 * velocity component of the free stream".  Box: the AABB of the vertices scaled by cv_radius_factor about its
 * centre (half-extent at least 0.05 R_b per axis).  Face k = 2a + side: side 0 at -h_a with inward normal +e_a, side 1
 * at +h_a with inward normal -e_a.  Flux through a face with inward bulk component s_k = V.n_k / c:
 * Gamma_k = A_k n c chi(s_k) / (2 sqrt(pi))  (the integrand of eq. (8) on a plane). */
typedef struct { double h[3], area[6], sn[6], cum[6], total; } box_cv;
static void box_setup(const oracle_mesh* mesh, const oracle_params* p, int s, box_cv* b) {
  double c = sqrt(2.0 * ORACLE_KB * p->T_inf / p->m[s]);
  for (int a = 0; a < 3; ++a) {
    double h = 0.5 * (mesh->hi[a] - mesh->lo[a]);
    if (h < 0.05 * mesh->Rb) h = 0.05 * mesh->Rb;
    b->h[a] = p->cv_radius_factor * h;
  }
  double acc = 0.0;
  for (int k = 0; k < 6; ++k) {
    int a = k / 2, side = k % 2;
    b->area[k] = 4.0 * b->h[(a + 1) % 3] * b->h[(a + 2) % 3];
    b->sn[k] = (side ? -p->V[a] : p->V[a]) / c;
    acc += b->area[k] * chi(b->sn[k]);
    b->cum[k] = acc;
  }
  b->total = acc; /* Gamma / (n c / (2 sqrt(pi))) */
}
double oracle_box_flux(const oracle_mesh* mesh, const oracle_params* p, int s) {
  box_cv b;
  box_setup(mesh, p, s, &b);
  double c = sqrt(2.0 * ORACLE_KB * p->T_inf / p->m[s]);
  return b.total * p->n * c / (2.0 * SQRTPI);
}
/* A25 (negative control): inward speed from the half-range Maxwellian WITHOUT the flux weight, density
 * ~ e^{-(x-s)^2} on x > 0: survival 1 - F = erfc(x - s) / erfc(-s).  Bracketed Newton like the other inverses. */
double oracle_vn_unweighted_inv(double u, double s) {
  double target = (1.0 - u) * erfc(-s);
  double lo = 0.0, hi = (s > 0.0 ? s : 0.0) + 8.0, x = (s > 0.0 ? s : 0.0) + 0.5;
  for (int it = 0; it < 400; ++it) {
    double f = erfc(x - s) - target; /* decreasing in x */
    if (f > 0.0) lo = x; else hi = x;
    double z = x - s;
    double d = -2.0 / SQRTPI * exp(-z * z);
    double xn = (d < 0.0) ? x - f / d : 0.5 * (lo + hi);
    if (!(xn > lo && xn < hi)) xn = 0.5 * (lo + hi);
    if (fabs(xn - x) <= 1e-16 * (1.0 + x) || hi - lo <= 1e-16 * (1.0 + x)) { x = xn; break; }
    x = xn;
  }
  return x;
}
static int seed_box(const oracle_mesh* mesh, const oracle_params* p, uint64_t i, double x[3], double v[3]) {
  double ub0[4], ub1[4];
  particle_block(p->seed, i, 0u, ub0);
  particle_block(p->seed, i, 1u, ub1);
  int s = 0; double acc = p->x[0];
  while (s < p->n_species - 1 && ub0[0] >= acc) { ++s; acc += p->x[s]; }
  double c = sqrt(2.0 * ORACLE_KB * p->T_inf / p->m[s]);
  box_cv b;
  box_setup(mesh, p, s, &b);
  int k = 0;
  while (k < 5 && ub0[1] * b.total >= b.cum[k]) ++k;   /* face with probability Gamma_k / Gamma */
  int a = k / 2, side = k % 2, e1 = (a + 1) % 3, e2 = (a + 2) % 3;
  x[a] = mesh->centre[a] + (side ? b.h[a] : -b.h[a]);
  x[e1] = mesh->centre[e1] + (2.0 * ub0[2] - 1.0) * b.h[e1];     /* uniform on the face */
  x[e2] = mesh->centre[e2] + (2.0 * ub0[3] - 1.0) * b.h[e2];
  double xn = (p->control_volume == 2) ? oracle_vn_unweighted_inv(ub1[0], b.sn[k]) : oracle_vn_inv(ub1[0], b.sn[k]);
  double rho = sqrt(-log(ub1[1]));
  double ang = TWOPI * ub1[2];
  v[a] = c * (side ? -xn : xn);                                   /* inward */
  v[e1] = c * (p->V[e1] / c + rho * cos(ang));                    /* Maxwellian about the bulk tangential components */
  v[e2] = c * (p->V[e2] / c + rho * sin(ang));
  return s;
}

/* ------------------------------------------------------------------ O4-O8: seed one particle */
/* Returns the species; x[3], v[3] are the fp64 values BEFORE the fp32 rounding of O9. */
int oracle_seed(const oracle_mesh* mesh, const oracle_params* p, uint64_t i, double x[3], double v[3]) {
  if (p->control_volume != 0) return seed_box(mesh, p, i, x, v);
  double ub0[4], ub1[4];
  particle_block(p->seed, i, 0u, ub0);
  particle_block(p->seed, i, 1u, ub1);
  /* A8: species by number fraction */
  int s = 0; double acc = p->x[0];
  while (s < p->n_species - 1 && ub0[0] >= acc) { ++s; acc += p->x[s]; }
  double speed = sqrt((p->V[0] * p->V[0] + p->V[1] * p->V[1]) + p->V[2] * p->V[2]);
  double c = sqrt(2.0 * ORACLE_KB * p->T_inf / p->m[s]);
  double S = speed / c;
  double r = p->cv_radius_factor * mesh->Rb;             /* A10 */
  double R[9];
  oracle_rotation(p->V, R);
  /* O5: position. t = sin(phi) = H^{-1}(u1), theta = 2 pi u2 */
  double t = oracle_position_inv(ub0[1], S);
  double cphi = sqrt(1.0 - t * t);
  double th = TWOPI * ub0[2];
  double ct = cos(th), st = sin(th);
  double xh[3] = {cphi * ct, cphi * st, t};
  /* O6: local frame: n = -xhat (inward), t1 meridional pointing downstream, t2 = t1 x n */
  double nh[3] = {-xh[0], -xh[1], -xh[2]};
  double t1[3] = {t * ct, t * st, -cphi};
  double t2[3] = {-st, ct, 0.0};
  /* O7: velocity in units of c */
  double sn = S * t;
  double xn = oracle_vn_inv(ub0[3], sn);
  double rho = sqrt(-log(ub1[0]));
  double ang = TWOPI * ub1[1];
  double xt1 = S * cphi + rho * cos(ang);
  double xt2 = rho * sin(ang);
  double vl[3];
  for (int k = 0; k < 3; ++k) vl[k] = (xn * nh[k] + xt1 * t1[k]) + xt2 * t2[k];
  for (int k = 0; k < 3; ++k) {
    double rx = (R[3 * k] * xh[0] + R[3 * k + 1] * xh[1]) + R[3 * k + 2] * xh[2];
    double rv = (R[3 * k] * vl[0] + R[3 * k + 1] * vl[1]) + R[3 * k + 2] * vl[2];
    x[k] = mesh->centre[k] + r * rx;
    v[k] = c * rv;
  }
  return s;
}

/* ------------------------------------------------------------------ O11: surface interaction P:73, P:53 (A6, A7, A17) */
void oracle_reflect(const oracle_mesh* mesh, const oracle_params* p, int32_t f, const float vin32[3],
                    uint64_t i, uint32_t k, int species, double vout[3]) {
  double u[4];
  particle_block(p->seed, i, 2u + k, u);
  double p0[3], p1[3], p2[3], e1[3], e2[3], Ng[3], v[3];
  tri_corner(mesh, f, 0, p0); tri_corner(mesh, f, 1, p1); tri_corner(mesh, f, 2, p2);
  for (int a = 0; a < 3; ++a) { e1[a] = p1[a] - p0[a]; e2[a] = p2[a] - p0[a]; v[a] = (double)vin32[a]; }
  cross3(e1, e2, Ng);
  double nl = sqrt(dot3(Ng, Ng));
  double nf[3] = {Ng[0] / nl, Ng[1] / nl, Ng[2] / nl};
  double vn = dot3(v, nf);
  double sgn = (vn < 0.0) ? 1.0 : -1.0;
  double ne[3] = {sgn * nf[0], sgn * nf[1], sgn * nf[2]}; /* n_eff faces the incoming particle */
  double sigma = mesh->surf_sigma ? mesh->surf_sigma[f] : p->accommodation; /* A23 */
  if (u[0] < sigma) {
    /* diffuse: flux-weighted half-Maxwellian (A6) at the re-emission temperature
     *   T_r = alpha_E T_W + (1 - alpha_E) T_k,i,   T_k,i = m v_in^2 / (3 k_B)   (A22; alpha_E = 1: T_r = T_W exactly) */
    double TW = mesh->surf_TW ? mesh->surf_TW[f] : p->T_W;
    double aE = p->energy_accommodation;
    double Tki = p->m[species] * dot3(v, v) / (3.0 * ORACLE_KB);
    double Tr = aE * TW + (1.0 - aE) * Tki;
    double cw = sqrt(2.0 * ORACLE_KB * Tr / p->m[species]);
    double el = sqrt(dot3(e1, e1));
    double t1[3] = {e1[0] / el, e1[1] / el, e1[2] / el};
    double t2[3];
    cross3(ne, t1, t2);
    double an = sqrt(-log(u[1]));
    double at = sqrt(-log(u[2]));
    double ang = TWOPI * u[3];
    double ca = cos(ang), sa = sin(ang);
    for (int a = 0; a < 3; ++a) vout[a] = cw * (an * ne[a] + at * (ca * t1[a] + sa * t2[a]));
  } else {
    double vne = dot3(v, ne);
    for (int a = 0; a < 3; ++a) vout[a] = v[a] - 2.0 * vne * ne[a];
  }
}

/* ------------------------------------------------------------------ O1-O14: the whole path */
static uint64_t fnv1a_facet(uint64_t h, int32_t f) {
  uint32_t w = (uint32_t)f;
  for (int b = 0; b < 4; ++b) { h ^= (uint64_t)((w >> (8 * b)) & 0xFFu); h *= 0x100000001B3ull; }
  return h;
}

int oracle_run(const oracle_mesh* mesh, const oracle_params* p, int use_bvh,
               double force[3], double torque[3], double* facet_momentum /* [nt][3] or NULL */,
               double force_sq[3] /* sum over particles of (per-particle force)^2, or NULL */,
               oracle_stats* stats, uint64_t* hash, uint32_t* bounces, int32_t* first_facet) {
  if (!mesh || !p || p->n_species < 1 || !p->m || !p->x || !(p->T_inf > 0.0) || !(p->T_W > 0.0) || p->N == 0) return -1;
  if (p->first + p->count > p->N) return -1;
  int64_t nt = mesh->nt;
  double* P = (double*)calloc((size_t)(3 * nt), sizeof(double));
  double tq[3] = {0, 0, 0}, fsq[3] = {0, 0, 0};
  oracle_stats st = {0, 0, 0, 0};
  double speed = sqrt((p->V[0] * p->V[0] + p->V[1] * p->V[1]) + p->V[2] * p->V[2]);
  double r = p->cv_radius_factor * mesh->Rb;
  for (uint64_t j = 0; j < p->count; ++j) {
    uint64_t i = p->first + j;
    double x64[3], v64[3];
    int s = oracle_seed(mesh, p, i, x64, v64);
    /* O2: weight w_s = m_s Gamma_s / N ("effective mass") */
    double c = sqrt(2.0 * ORACLE_KB * p->T_inf / p->m[s]);
    double flux = (p->control_volume != 0) ? oracle_box_flux(mesh, p, s) : oracle_flux(speed / c, c, p->n, r);
    double w = p->m[s] * flux / (double)p->N;
    /* O9: the particle IS the ray defined by these fp32 values */
    float o[3] = {(float)x64[0], (float)x64[1], (float)x64[2]};
    float v[3] = {(float)v64[0], (float)v64[1], (float)v64[2]};
    int32_t f_prev = -1, ff = -1;
    uint32_t k = 0;
    uint64_t h = 0xCBF29CE484222325ull;
    double fp[3] = {0, 0, 0};
    for (;;) {
      double tau;
      int32_t f = oracle_closest_hit(mesh, o, v, f_prev, use_bvh, &tau);
      st.segments++;
      if (f < 0) { st.escaped++; break; }
      st.hits++;
      if (k == 0) ff = f;
      h = fnv1a_facet(h, f);
      double vout[3];
      oracle_reflect(mesh, p, f, v, i, k, s, vout);
      float vo32[3] = {(float)vout[0], (float)vout[1], (float)vout[2]};
      /* O12: dp = w (v_in - v_out), both as their fp32 values; torque about x_ref at the hit point */
      double hp[3], dp[3];
      for (int a = 0; a < 3; ++a) {
        hp[a] = (double)o[a] + tau * (double)v[a];
        dp[a] = w * ((double)v[a] - (double)vo32[a]);
        P[3 * f + a] += dp[a];
        fp[a] += dp[a];
      }
      double rr[3] = {hp[0] - p->x_ref[0], hp[1] - p->x_ref[1], hp[2] - p->x_ref[2]}, cr[3];
      cross3(rr, dp, cr);
      for (int a = 0; a < 3; ++a) tq[a] += cr[a];
      /* O13: next segment */
      for (int a = 0; a < 3; ++a) { o[a] = (float)hp[a]; v[a] = vo32[a]; }
      f_prev = f;
      ++k;
      if (k >= p->max_bounces) { st.truncated++; break; }
    }
    for (int a = 0; a < 3; ++a) fsq[a] += fp[a] * fp[a];
    if (hash) hash[j] = h;
    if (bounces) bounces[j] = k;
    if (first_facet) first_facet[j] = ff;
  }
  /* O14: F = sum_f P_f in facet order */
  double F[3] = {0, 0, 0};
  for (int64_t f = 0; f < nt; ++f) for (int a = 0; a < 3; ++a) F[a] += P[3 * f + a];
  for (int a = 0; a < 3; ++a) { force[a] = F[a]; torque[a] = tq[a]; if (force_sq) force_sq[a] = fsq[a]; }
  if (facet_momentum) memcpy(facet_momentum, P, sizeof(double) * 3 * (size_t)nt);
  if (stats) *stats = st;
  free(P);
  return 0;
}
