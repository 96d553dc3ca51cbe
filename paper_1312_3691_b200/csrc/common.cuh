// common.cuh -- shared declarations of libtpmc (CUDA path only; nothing here is used by oracle/).
#pragma once

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/tpmc.h"

#define TPMC_SQRTPI 1.7724538509055160272981674833411
#define TPMC_KB 1.380649e-23  // J/K

extern thread_local char g_tpmc_cuda_error[512];

#define TPMC_CUDA_TRY(expr)                                                                        \
  do {                                                                                             \
    cudaError_t _e = (expr);                                                                       \
    if (_e != cudaSuccess) {                                                                       \
      snprintf(g_tpmc_cuda_error, sizeof(g_tpmc_cuda_error), "%s:%d: %s: %s", __FILE__, __LINE__,  \
               #expr, cudaGetErrorString(_e));                                                     \
      cudaGetLastError();                                                                          \
      return (_e == cudaErrorMemoryAllocation) ? TPMC_ENOMEM : TPMC_ECUDA;                         \
    }                                                                                              \
  } while (0)

// ---------------------------------------------------------------------------------------------
// One wave pipeline: queues, hit list, counters, its two streams and the events that order them.
// Waves are dealt round-robin to kPipes pipelines that run concurrently: every kernel of the path is
// latency bound on its own, so a second, independent chain of kernels fills the idle issue slots.
constexpr int kPipes = 1;   // two concurrent pipelines were measured: no gain once seeding overlaps trace/reflect
struct Pipe {
  float4* q_o[2];                  // ray queues (ping-pong between iterations), regions A|B of wave_cap rays each
  float4* q_v[2];
  int* q_f[2];
  unsigned int* q_key[2];          // sort key of every queued ray (sort.cuh)
  unsigned int* hist[2];           // [kSortBins] histogram of the keys of queue p, then their offsets
  unsigned int* order;             // [2*wave_cap] queue slots in key order
  unsigned int* hit_ray;           // [2*wave_cap] queue slot of every ray that ended with candidate facets
  int4* hit_cand;                  // [2*wave_cap] its candidate triangle slots
  unsigned int* ctr;               // [kCtrWords] device counters (queue sizes, fetch head, hit count, survivors)
  unsigned int* ovf;               // [2][2*wave_cap] queue slots of rays left to the straggler kernel (overflow lists)
  unsigned int* surv;              // [3][wave_cap] survivors of the fp32 pre-cull pass: wave offset, fp32 roots
  cudaStream_t main, seed, side;   // trace/reflect chain (pipe 0: the caller's); next wave's seed kernels; stragglers
  cudaEvent_t ev_reset[4], ev_seeded[4], ev_done, ev_f0, ev_f1;
  cudaEvent_t ev_refl[2], ev_ovf[2];   // reflect step done / its overflow list processed (iteration parity)
  unsigned long long last_iter;
  cudaEvent_t* wave_ev;            // [kEvPerWave*kMaxTimedWaves] per-kernel timing, created on first use
  unsigned long long iters, seed_iters;   // of the last run: iterations / seeded iterations with timing events
};

// ---------------------------------------------------------------------------------------------
// Device-resident body.  nodes: 4 float4 per internal node (two child boxes + two child refs);
// tris: 3 float4 per triangle in Morton order: (p0, facet id), (p1, flags), (p2, 0).
struct QuantGrid;
struct tpmc_mesh {
  int64_t nv, nt;
  int64_t n_nodes;
  float4* nodes;
  float4* tris;
  // flow-aligned copy of the compact hierarchy, refitted per run (tpmc_mesh_align in lbvh.cu)
  int2* kids;                      // [nt-1] children of every internal node (topology of the LBVH)
  int* parent;                     // [nt-1 | nt] parent of every internal node and leaf
  int* arrive;                     // [nt-1] refit counters
  float* rbox;                     // [(nt-1) + nt][6] boxes in the aligned frame
  // wide (4-ary) hierarchy of the wavefront traversal: the binary tree collapsed breadth-first (k_wide_*), 64 B per node
  int64_t n_wide;                  // wide nodes
  int4* wkids_bin;                 // [n_wide] children as refs of the BINARY tree (>= 0 internal node, < 0 leaf ~slot, TPMC_WIDE_EMPTY)
  int4* wkids;                     // [n_wide] the same children as refs of the WIDE tree (>= 0 wide node, < 0 leaf ~slot)
  uint4* wnodes;                   // [n_wide][4] body-frame boxes on the 16-bit grid + refs (k_compact_wide)
  uint4* wnodes_r;                 // [n_wide][4] the flow-aligned copy, refitted per run
  double* align_R;                 // [9] rotation of the current alignment, [6] its grid origin and scale (device)
  QuantGrid* grid_dev;             // [2] device copies of the grids the traversal reads: body frame, aligned
  uint4* cnodes;                   // compact copy of `nodes` for the wavefront traversal: 2 uint4 = 32 B per node
  float q_origin[3], q_scale[3];   // its quantisation grid: x = q_origin + q * q_scale, q in [0, 65535]
  double* surf_TW;                 // [nt] by facet id: wall temperature per facet, or nullptr (tpmc_mesh_set_surface, A23)
  double* surf_sigma;              // [nt] by facet id: accommodation per facet, or nullptr
  uint4* horizon;                  // [nt] by sorted slot: escape horizon of each facet, 16 azimuth sectors x 1 byte (k_horizon, lbvh.cu)
  double horizon_ms;
  uint4* cull_c;                   // top of the hierarchy (<= kCullNodes nodes, breadth-first) in the compact format of `cnodes`: seed-time cull
  int n_cull;
  // two-level cull volume of the pre-cull pass: all facets lie within cull_rin of the centre or in a box
  float cull_rin;
  int cull_nbox;                   // -1: not used (no gain over the bounding sphere)
  float cull_box[8][6];            // lo.xyz, hi.xyz
  double centre[3];
  double Rb;
  float aabb_lo[3], aabb_hi[3];
  double build_ms;
  int device;
  // per-run scratch, cached in the handle (one run at a time per handle)
  size_t wave_cap;
  Pipe pipe[kPipes];
  double* facet_scratch;           // [nt][3] when the caller passes no per-facet buffer
  double* partials;                // reduction partials
  unsigned long long* stats;       // [ST_COUNT] device counters (enum below), one per tpmc_stats event
  double* totals;                  // [3] torque accumulators
  double* ft_dev;                  // [6] force | torque of tpmc_run_host
  cudaEvent_t ev0, ev1, ev_fork;
  unsigned long long last_launches;
  bool in_run;                     // tpmc_run has enqueued work and not yet returned TPMC_OK (see its error path)
  bool poisoned;                   // a failed run could not be drained: every later run on this handle returns TPMC_ECUDA
};

constexpr int kMaxTimedWaves = 1024;  // iterations covered by the per-kernel event times
#ifndef TPMC_DRAIN
#define TPMC_DRAIN 3
#endif
constexpr int kDrain = TPMC_DRAIN;    // trace/reflect iterations after the last wave, before the straggler kernel
constexpr int kEvPerWave = 8;         // seed start/end (seed stream), iteration start, after trace, after reflect, straggler start/end (side stream), after sort
constexpr int kCtrWords = 16;
constexpr int kCullNodes = 64;        // 4 KB: stays in L1 next to the shared-memory carve-out
constexpr float kPrecullMargin = 2e-2f;   // box growth of the pre-cull pass, in bounding radii (sampling.cuh)

// Quantisation grid of the compact nodes, as the traversal kernel uses it (fp32).
struct QuantGrid {
  float origin[3];
  float inv_scale[3];   // fp32(1 / q_scale)
  float R[9];           // frame of the grid: x' = R x (identity for the body-frame hierarchy, see tpmc_mesh_align)
  float rot_o, rot_c;   // rotation-error terms of the slab margin (trace.cuh, grid_ray): 0 for the identity frame, else
                        // 9u (factor of |o|_1) and 6u * reach, reach = largest |x| over the root box, in metres
};

// Per-run constants (a1: host, fp64), passed to kernels by value.
struct SpeciesConst {
  double m;      // molecular mass, kg
  double c;      // c_mp = sqrt(2 k_B T_inf / m)
  double S;      // speed ratio |V| / c_mp
  double cW;     // sqrt(2 k_B T_W / m)
  double w;      // particle weight m Gamma / N  [kg/s]     (eq. 10)
  double g0;     // Gt(-S)                                  (position CDF constants, O5)
  double gI;     // Gt(S) - Gt(-S)
  double cumx;   // cumulative number fraction
  // rectangular control volume (A24): per face k = 2 axis + side, inward bulk component / c, cumulative A_k chi(s_k)
  double bsn[6], bcum[6];
};

struct RunConst {
  SpeciesConst sp[TPMC_MAX_SPECIES];
  int n_species;
  double R[9];          // stream frame -> body frame, eq. (15)
  double centre[3];
  double r;             // control-sphere radius
  double sigma;
  double T_W, alpha_E;              // wall temperature and energy accommodation of the run (A22)
  const double* surf_TW;            // per-facet overrides by facet id, or nullptr (A23)
  const double* surf_sigma;
  int simple_surface;               // alpha_E == 1 and no per-facet T_W: c_W is the per-species constant
  double x_ref[3];
  float aabb_lo[3], aabb_hi[3];
  unsigned long long first, count;
  unsigned int seed_lo, seed_hi;
  unsigned int max_bounces;
  float key_c[3], key_r2;   // sort key of a ray (sort.cuh): body centre, (radius of the key sphere)^2
  int control_volume;       // TPMC_CV_*
  double box_h[3];          // half-extents of the rectangular control volume (A24)
  double V[3];              // bulk velocity (the box scheme needs its components, not only the stream frame)
};

// Device counters of a run (tpmc_stats: every one is counted where the event happens).
enum { ST_HITS = 0, ST_TRUNC, ST_TRIS, ST_NODES, ST_TRACED, ST_RET_PA, ST_RET_PB, ST_RET_SEED, ST_RET_TRACE,
       ST_RET_RESOLVE, ST_RET_HORIZON, ST_RET_FINISH, ST_Q_PRIM, ST_Q_REFL, ST_OVF_RETRACE, ST_OVF_PENDING, ST_DIVERTED,
       ST_STRAGGLERS, ST_FIN_SEGS, ST_UNCERT, ST_COUNT = 24 };

int tpmc_mesh_align(tpmc_mesh* m, const double R[9], cudaStream_t st, const QuantGrid** grid_out, const uint4** wnodes_out);
#define TPMC_WIDE_EMPTY ((int)0x7FFFFFFD)   // wkids_bin: no child in this slot

#define TPMC_HD __host__ __device__ __forceinline__

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011), counter-based, keyed by particle index (O3).
TPMC_HD uint32_t mulhi32(uint32_t a, uint32_t b) {
#ifdef __CUDA_ARCH__
  return __umulhi(a, b);
#else
  return (uint32_t)(((uint64_t)a * (uint64_t)b) >> 32);
#endif
}

TPMC_HD uint4 philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = mulhi32(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = mulhi32(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return make_uint4(c0, c1, c2, c3);
}

// word -> uniform in (0,1): (w + 1/2) 2^-32, exact in fp64 (A16)
TPMC_HD double u01(uint32_t w) { return ((double)w + 0.5) * (1.0 / 4294967296.0); }

TPMC_HD uint4 particle_block(const RunConst& rc, unsigned long long i, uint32_t block) {
  return philox4x32_10(rc.seed_lo, rc.seed_hi, (uint32_t)i, (uint32_t)(i >> 32), block, 0u);
}
