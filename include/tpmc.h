/*
 * tpmc.h -- C ABI of libtpmc.so: the data-parallel hot path of the test-particle Monte Carlo
 * (TPMC) free-molecular method of arXiv 1312.3691 (Parham & Barba, "Finding the Force"),
 * hand-written CUDA for sm_100a (B200).
 *
 * Citations "P:<line>" are lines of the paper text; "O<n>/A<n>/G<n>" are the
 * step definitions and readings listed in DESIGN.md (taken from SURVEY.md section 8(c)).
 *
 * Conventions (every entry point):
 *   - returns TPMC_OK (0) or a negative TPMC_E* code; never aborts, never throws across the ABI;
 *     tpmc_strerror() names a code, tpmc_last_cuda_error() gives the CUDA text after TPMC_ECUDA.
 *   - "host"/"device" says where a pointer must live.  The library never frees caller buffers.
 *   - work is enqueued on the caller's CUDA stream (cudaStream_t passed as void*, NULL = default
 *     stream); device outputs are valid once the caller has synchronised that stream.
 *   - a mesh handle caches per-run scratch (ray queues, lists, counters, the flow-aligned copy of the
 *     hierarchy): tpmc_run / tpmc_run_host / tpmc_trace take it non-const, and all calls on one handle must
 *     be ordered on ONE stream (or separated by a synchronisation); two handles are independent.
 *   - behaviour is selected by the parameter struct only; the library reads no environment variable.
 *   - there is no CPU fallback: without a CUDA device every compute call returns TPMC_ECUDA.
 */
#ifndef TPMC_H
#define TPMC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TPMC_OK 0
#define TPMC_EINVAL (-1) /* bad argument / degenerate mesh / bad parameter */
#define TPMC_ENOMEM (-2) /* host or device allocation failed */
#define TPMC_ECUDA (-3)  /* a CUDA call failed; see tpmc_last_cuda_error() */
#define TPMC_ECAPACITY (-4) /* input larger than a fixed-capacity entry point takes; tpmc_last_cuda_error() has the numbers */

#define TPMC_MEM_HOST 0
#define TPMC_MEM_DEVICE 1

#define TPMC_MAX_SPECIES 8
#define TPMC_FACET_TWO_SIDED 1u /* facet_flags bit0 */
#define TPMC_MAX_BOUNCES 0x0FFFFFFFu /* largest max_bounces (the bounce count shares a word with the species) */

/* tpmc_params.flags.  Each switches off, forces or adds a step that must not change the physics: the parity tests run
 * with and without them and require the same hit sequence for every particle and sums equal to the order of the fp64
 * additions (1e-12 relative).  "Same" is not "bit for bit" in one respect: the fp64 sampler stops its root searches on a
 * step tolerance, and under NO_PRECULL it starts them from its own guess instead of the pre-cull's, so a seeded
 * coordinate may differ in the last ulp of its fp64 value.  After the fp32 rounding of O9 that moves a ray with
 * probability ~1e-9 per coordinate -- a few particles in 1e9, far inside the 99.99 % bar.  The defaults are all zero. */
#define TPMC_FLAG_NO_PRECULL 0x01u  /* every particle through the fp64 sampler (no fp32 pre-cull pass) */
#define TPMC_FLAG_NO_HORIZON 0x02u  /* every re-emitted ray is traced (no escape-horizon test) */
#define TPMC_FLAG_ALIGN_OFF 0x04u   /* traversal on the body-frame hierarchy, whatever the attitude */
#define TPMC_FLAG_ALIGN_ON 0x08u    /* traversal on the flow-aligned refit, whatever the attitude */
#define TPMC_FLAG_EXACT_TRACE 0x10u /* every segment by the fp64 closest-hit search (no fp32 filter, no candidate lists) */
#define TPMC_FLAG_NO_AGGREGATION 0x40u /* one fp64 atomic per hit and component even on bodies with few facets */
#define TPMC_FLAG_SORT_RAYS 0x20u   /* rays traced in the order of a spatial key (counting sort before the traversal) */
#define TPMC_FLAG_SERIAL_SEED 0x80u /* the seed kernels of the next wave run on the caller's stream, behind trace/reflect, not beside
                                      * them: the per-kernel times of tpmc_stats are then each kernel's own (measurement aid) */

/* tpmc_params.control_volume */
#define TPMC_CV_SPHERE 0 /* the paper's scheme: spherical control volume, eqs. (10)-(15) */
#define TPMC_CV_BOX 1    /* rectangular control volume, flux-weighted per face: cross-check */
#define TPMC_CV_BOX_UNWEIGHTED 2 /* the same with the inward speed drawn WITHOUT flux weighting: negative control */

/* Opaque triangulated body + its on-device LBVH ("Satellite surfaces are represented by a
 * triangulation, allowing the use of well-known ray-tracing methods").  Owns its device memory. */
typedef struct tpmc_mesh tpmc_mesh;

typedef struct {
  double centre[3];        /* centre of the vertex AABB = centre of the control sphere (O1, A10) */
  double bounding_radius;  /* R_b = max |vertex - centre| */
  float aabb_lo[3], aabb_hi[3];
  int64_t nt;              /* facets */
  int64_t n_nodes;         /* LBVH internal nodes (max(nt-1,1)), 64 B each */
  double build_ms;         /* device time of the LBVH build (Morton, sort, hierarchy, refit) */
  double horizon_ms;       /* device time of the per-facet escape-horizon pass that follows it */
} tpmc_mesh_info_t;

/* Gas, control volume and run selection (Table 1). */
typedef struct {
  double n;                /* number density, 1/m^3 */
  double T_inf, T_W;       /* free-stream and wall temperature, K */
  double V[3];             /* free-stream bulk velocity in the body frame, m/s (sweeps rotate V, not the mesh) */
  double accommodation;    /* sigma in [0,1]: P(diffuse re-emission fully accommodated to T_W); else specular (A7) */
  int32_t n_species;       /* 1..TPMC_MAX_SPECIES */
  const double* m;         /* host [n_species] molecular mass, kg */
  const double* x;         /* host [n_species] number fraction, sum 1 (species drawn per particle, A8) */
  double cv_radius_factor; /* control-sphere radius / bounding radius (> 1; the configs use 1.5) */
  uint64_t N;              /* particles of the whole stream; the particle weight is m Gamma / N */
  uint64_t first, count;   /* run only particles [first, first+count) of that stream (slices, multi-GPU) */
  uint64_t seed;           /* Philox4x32-10 key; counter = (particle index, block) (O3) */
  uint32_t max_bounces;    /* cap on reflections per particle, 1..TPMC_MAX_BOUNCES; cut-off particles are counted (A13) */
  double x_ref[3];         /* torque reference point, body frame (A14) */
  double energy_accommodation; /* alpha_E in [0,1]: re-emission temperature T_r = alpha_E T_W + (1 - alpha_E) T_k,i with
                              T_k,i = m v_in^2 / (3 k_B) (reading A22); 1.0 = the paper's full accommodation */
  uint64_t wave_particles; /* particles seeded per pipeline iteration; 0 = default (2^26).  Results do not depend on it */
  uint64_t chunk_particles;/* particles per 32-bit index chunk; 0 = default (0xF0000000).  Results do not depend on it */
  uint32_t flags;          /* TPMC_FLAG_* */
  int32_t control_volume;  /* TPMC_CV_* */
} tpmc_params;

/* Every number below is COUNTED on the device where the event happens (none is derived from another), so
 *   count == truncated + ret_precull_a + ret_precull_b + ret_seed + ret_trace + ret_resolve + ret_horizon + ret_finish
 *   segments == count + hits - truncated,   escaped == count - truncated
 * are checks of the pipeline's bookkeeping (a particle lost or duplicated between two lists breaks them). */
typedef struct {
  uint64_t hits;           /* surface interactions ("bounces") */
  uint64_t segments;       /* segments answered: by a cull (1 per culled particle), the traversal, the escape horizon, the straggler kernel */
  uint64_t escaped;        /* particles that left without (further) hit = all retirements except truncated */
  uint64_t truncated;      /* particles stopped by max_bounces */
  uint64_t culled;         /* particles whose first segment was answered before the traversal = ret_precull_a + ret_precull_b + ret_seed */
  uint64_t tri_tests;      /* fp64 ray-triangle evaluations */
  uint64_t node_visits;    /* 64-byte BVH nodes fetched */
  uint64_t kernel_launches;/* kernels this run enqueued */
  double ms;               /* device time of this run, CUDA events on the caller's stream */
  double ms_seed;          /* summed device time of the seed-kernel launches (events around each launch) */
  double ms_trace;         /* ... of the wavefront traversal kernel launches */
  double ms_reflect;       /* ... of the resolve/reflect/accumulate kernel launches */
  double ms_finish;        /* ... of the straggler kernel launches */
  uint64_t timed_waves;    /* waves covered by the per-kernel times (the first 1024 of the first index chunk) */
  uint64_t trace_launches; /* traversal-kernel launches covered by ms_trace */
  uint64_t traced_rays;    /* rays the traversal kernel processed (all launches) */
  /* where each particle retired (see the identities above) */
  uint64_t ret_precull_a;  /* certain miss of the bounding sphere, pre-cull stage A */
  uint64_t ret_precull_b;  /* certified miss of the cull volumes, pre-cull stage B */
  uint64_t ret_seed;       /* exact fp32 ray misses the mesh AABB / the top of the hierarchy, seed kernel */
  uint64_t ret_trace;      /* traversal ended without a candidate facet */
  uint64_t ret_resolve;    /* all candidates rejected by the exact test */
  uint64_t ret_horizon;    /* re-emitted above the facet's escape horizon */
  uint64_t ret_finish;     /* no hit in the straggler kernel's fp64 search */
  /* flows between the steps */
  uint64_t queued_primaries; /* rays the seed kernel appended to the queue */
  uint64_t queued_reflected; /* rays the reflect step appended to the next queue */
  uint64_t overflow_rays;    /* rays handed to the straggler kernel by an overflow list (candidate overflow, stack abort, full region) */
  uint64_t final_stragglers; /* rays still queued after the drain iterations (followed by the straggler kernel, not traced) */
  uint64_t finish_segments;  /* closest-hit searches of the straggler kernel */
  double ms_sort;          /* summed device time of the ray-sort launches */
  uint64_t precull_uncertified; /* particles whose fp32 pre-cull estimate was not certified (they take the fp64 sampler whatever their ray does) */
} tpmc_stats;

/* Optional per-particle outputs for parity checks; each pointer is device [count] or NULL. */
typedef struct {
  uint64_t* hash;          /* FNV-1a 64 over the little-endian bytes of the hit facet ids, in order (O12) */
  uint32_t* bounces;       /* number of surface interactions */
  int32_t* first_facet;    /* first facet hit, or -1 */
} tpmc_debug;

/* Build a body: copies the triangulation to the device, computes centre / bounding radius (O1) and
 * builds the LBVH there (63-bit Morton codes of centroids -> radix sort -> Karras hierarchy ->
 * bottom-up AABB refit).  There is no host build path.
 *   vertices   [nv][3] fp32, metres, body frame; indices [nt][3] int32, counter-clockwise seen from
 *              outside for one-sided facets; facet_flags [nt] or NULL (bit0 = two-sided, A11);
 *              all three live where mem_space says.  nt >= 1, nv >= 3, indices in range.
 * Synchronises `stream` before returning.  *out is valid only on TPMC_OK. */
int tpmc_mesh_create(const float* vertices, int64_t nv, const int32_t* indices, int64_t nt,
                     const uint8_t* facet_flags, int mem_space, void* cuda_stream, tpmc_mesh** out);
/* The same with options.  mesh_flags: TPMC_MESH_NO_HORIZON skips the per-facet escape-horizon pass that follows the
 * LBVH build.  That pass is 26x the build itself on the 1M-facet body (0.37 s against 14 ms) and pays only when many runs
 * share the handle (4 % of a 64-attitude sweep); without it every run behaves as with TPMC_FLAG_NO_HORIZON -- the same
 * results, every re-emitted ray traced -- so a caller who wants one attitude gets a first result three times sooner.
 * tpmc_mesh_build_horizon adds the horizons later (no-op if present; synchronises the stream; call it between runs, not
 * while one is in flight); tpmc_mesh_copy_horizon returns TPMC_EINVAL while there are none.  Unknown bits: TPMC_EINVAL. */
#define TPMC_MESH_NO_HORIZON 0x1u
int tpmc_mesh_create_ex(const float* vertices, int64_t nv, const int32_t* indices, int64_t nt, const uint8_t* facet_flags,
                        int mem_space, uint32_t mesh_flags, void* cuda_stream, tpmc_mesh** out);
int tpmc_mesh_build_horizon(tpmc_mesh* mesh, void* cuda_stream);
void tpmc_mesh_destroy(tpmc_mesh* mesh);
int tpmc_mesh_info(const tpmc_mesh* mesh, tpmc_mesh_info_t* out /* host */);

/* Surface properties per facet (reading A23; "arbitrary surface interaction"; re-emission "determined by the
 * satellite surface temperature"): T_W [nt] wall temperature (K, > 0) and sigma [nt] accommodation in [0,1],
 * indexed by facet id as in `indices`, both where mem_space says; either may be NULL, which restores the run's scalar
 * (tpmc_params.T_W / .accommodation).  The arrays are copied; they apply to every later run on this handle.
 * Host and device arrays alike are checked first (a value outside those ranges, or a NaN: TPMC_EINVAL, nothing changed).
 * Waits for the whole device before replacing arrays a run may still read, and synchronises the stream after the copy. */
int tpmc_mesh_set_surface(tpmc_mesh* mesh, const double* T_W, const double* sigma, int mem_space, void* cuda_stream);

/* Copy the built hierarchy to the host for inspection: nodes [n_nodes][16] floats
 * (lo0.xyz hi0.xyz lo1.xyz hi1.xyz, then child0, child1 as int32 bit patterns, 2 pad words;
 * child >= 0: internal node, child < 0: leaf holding sorted triangle ~child),
 * leaf_facet [nt] = facet id stored in each sorted triangle slot.  Either pointer may be NULL. */
int tpmc_mesh_copy_bvh(const tpmc_mesh* mesh, float* h_nodes, int32_t* h_leaf_facet);

/* Copy the wide (4-ary) hierarchy the wavefront traversal walks, body frame, to the host for inspection.
 * *n_wide = number of wide nodes (always written); h_wnodes [n_wide][16] uint32 or NULL: words 3k .. 3k+2 = box of child
 * k (x, y, z), each lo | hi << 16 in unsigned 16-bit grid coordinates (lo rounded down, hi up; an empty slot has
 * lo = 65535, hi = 0), words 12-15 = the child refs (>= 0: wide node, < 0: leaf holding sorted triangle ~ref);
 * h_grid [6] float or NULL: origin xyz and step xyz of the grid, x = origin + q * step.  The radix tree is collapsed
 * breadth-first (wide node 0 is the root): every sorted triangle is a leaf of exactly one wide node. */
int tpmc_mesh_copy_wide(const tpmc_mesh* mesh, int64_t* n_wide, uint32_t* h_wnodes, float* h_grid);

/* Copy the escape horizons to the host for inspection: h_horizon [nt][16] bytes, indexed by sorted triangle
 * slot (see leaf_facet above) and azimuth sector.  For a one-sided facet with unit normal n, first edge
 * direction e1 and e2 = n x e1, a ray leaving the facet in direction d with azimuth atan2(d.e2, d.e1) in
 * sector k = floor((azimuth + pi) * 16 / (2 pi)) and elevation sin E = d.n / |d| > byte / 254 cannot hit any
 * facet (O10 finds no hit): the reflect step does not trace it.  255 = no such bound (two-sided facets, facets
 * at sharp concave or convex edges).  Built on the device by tpmc_mesh_create after the LBVH. */
int tpmc_mesh_copy_horizon(const tpmc_mesh* mesh, uint8_t* h_horizon);

/* The hot path: seed particles [first, first+count) on the spherical control
 * volume from the drifting-Maxwellian number flux (eq. 10, 11, 14a-c, 15), trace each against the
 * body (closest hit), apply the surface interaction, follow reflections until
 * escape, and accumulate momentum transfer and torque.
 *   d_force [3], d_torque [3]   device, overwritten: force (N) and torque about x_ref (N m) of this slice
 *   d_facet_momentum [nt][3]    device or NULL, overwritten: momentum-transfer rate per facet (N)
 *   h_stats                     host or NULL; if given the call synchronises the stream and fills it
 *   debug                       host struct of device pointers, or NULL
 * Slices are additive: summing the outputs of disjoint [first,count) slices of one N gives the full run. */
int tpmc_run(tpmc_mesh* mesh, const tpmc_params* params, void* cuda_stream, double* d_force,
             double* d_torque, double* d_facet_momentum, tpmc_stats* h_stats, const tpmc_debug* debug);

/* An attitude sweep in one call (the paper's application: force and moment coefficients over a range of attitudes,
 * P:243, Figs. 8-9): run k (k < n_attitudes) is `params` with V replaced by h_V[k] (host [n_attitudes][3];
 * sweeps rotate V, not the mesh).  d_force, d_torque device [n_attitudes][3]; d_facet_momentum device
 * [n_attitudes][nt][3] or NULL; h_stats host [n_attitudes] or NULL (when given, the stream is synchronised after every
 * attitude).  Stops at the first failing attitude and returns its code. */
int tpmc_run_sweep(tpmc_mesh* mesh, const tpmc_params* params, int32_t n_attitudes, const double* h_V, void* cuda_stream,
                   double* d_force, double* d_torque, double* d_facet_momentum, tpmc_stats* h_stats);

/* Same run with HOST result buffers (h_facet_momentum may be NULL): device results are copied back
 * inside the call and the stream is synchronised before returning. */
int tpmc_run_host(tpmc_mesh* mesh, const tpmc_params* params, void* cuda_stream, double* h_force,
                  double* h_torque, double* h_facet_momentum, tpmc_stats* h_stats);

/* Seeding step alone (O3-O8), for parity checks: fp64 position and velocity of particles
 * [first, first+count) BEFORE the fp32 rounding of O9.  d_x, d_v device [count][3]; d_species device
 * [count] or NULL.  Runs the same device code as tpmc_run's seed kernel. */
int tpmc_seed(const tpmc_mesh* mesh, const tpmc_params* params, void* cuda_stream, double* d_x, double* d_v,
              int32_t* d_species);

/* Closest-hit step alone (O10), for parity checks: rays o + tau d with fp32 origin/direction,
 * d_o, d_d device [n][3]; d_f_prev device [n] (facet to exclude, -1 for none) or NULL;
 * h_align_V host [3] or NULL: when given, the traversal walks the hierarchy refitted in the stream frame of that
 * bulk velocity (what tpmc_run does for oblique attitudes) instead of the body-frame one -- same results;
 * outputs d_facet [n] (-1 = no hit) and d_tau [n] (fp64, +inf when no hit).  Runs the production traversal
 * kernel and the exact resolve; synchronises the stream. */
int tpmc_trace(tpmc_mesh* mesh, const float* d_o, const float* d_d, const int32_t* d_f_prev, int64_t n,
               const double* h_align_V, void* cuda_stream, int32_t* d_facet, double* d_tau);

/* Measured peaks of the units that bound the kernels of the path (roofline denominators are measured,
 * not nominal).  Hand-written micro-kernels, each timed once after a warm-up launch (about 0.1 s in all):
 *   fp32 FFMA lane-instruction rate at full occupancy; fp64 FMA rate; 32-byte read-only gathers (one 256-bit load per
 *   lane, every lane its own record) over an 83 MB array with the traversal kernel's residency (8 blocks of 128
 *   threads per SM), with independent addresses and as a pointer chase -- both with ONE load in flight per lane, i.e.
 *   resident lanes x 32 B / latency; the same array read as 64-byte records the way the traversal kernel reads a wide
 *   node, several loads in flight per lane (the throughput of the gather path); fp64 red.global.add at 1, 2048 and 1e6
 *   accumulators laid out like the per-facet momentum.  out: host.  Synchronises the stream. */
typedef struct {
  int32_t sms;
  double sm_clock_mhz_nominal;      /* cudaDevAttrClockRate */
  double sm_clock_mhz_fp32;         /* fp32_lane_ops_per_s / (sms * 128): the clock if every lane issued every cycle */
  double fp32_lane_ops_per_s;       /* FFMA lane-instructions per second (1 FFMA = 1 op here, 2 flops) */
  double fp64_fma_per_s;            /* DFMA lane-instructions per second */
  double gather32_bytes_per_s;      /* independent 32-byte gathers */
  double gather32_dependent_bytes_per_s; /* pointer chase, same residency */
  double gather_array_bytes;
  double red_f64_per_s[3];          /* fp64 atomic adds per second ... */
  double red_f64_addresses[3];      /* ... over this many accumulators */
  double gather64_bytes_per_s;      /* 64-byte records as two 32-byte loads of one line, two records in flight per lane,
                                       7 blocks of 128 threads per SM: the traversal kernel's access shape and residency */
} tpmc_peaks;
int tpmc_measure_peaks(tpmc_peaks* out, void* cuda_stream);

/* F = sum over facets of the per-facet momentum-transfer rate (the last step of tpmc_run), as a
 * call of its own that ALLOCATES NOTHING.  It is meant for callers that must not, or cannot, obtain device memory at the
 * time of the call: a program that gave all of the GPU's memory to its own pool (a cudaMalloc from inside a library would
 * fail or break its budget), a loop with a deadline (cudaMalloc and cudaFree take driver locks and may wait for the
 * device to drain), code running while another thread holds a global-mode stream capture open (the runtime refuses
 * cudaMalloc then).  Such a caller sums a facet-momentum array it already holds -- one written by tpmc_run, or the sum
 * of several slices -- without libtpmc touching an allocator: no cudaMalloc, cudaFree or allocating library routine is
 * called, on any path.
 *   d_facet_momentum  device [nt][3] fp64, read only (may be NULL when nt == 0)
 *   nt                0 .. TPMC_STATIC_MAX_FACETS; more returns TPMC_ECAPACITY and enqueues nothing (the call does not
 *                     split or fall back to allocating)
 *   d_force           device [3], overwritten (zeros for nt == 0); valid once `cuda_stream` has been synchronised
 * The partial sums live in a fixed array inside the library image (49 408 bytes; every GPU that loads libtpmc.so holds
 * its copy until the process exits).  Consequences the caller must know:
 *   - one array per GPU, shared by all calls, threads and streams: two calls that may overlap on the same GPU race on
 *     it and give wrong sums.  Order them on one stream or with events.  Calls on different GPUs are independent.
 *   - the array keeps what the previous call left; the call clears the one word that has to start at zero itself
 *     (a 4-byte cudaMemsetAsync on `cuda_stream` ahead of the kernel), so nothing needs resetting between calls.
 *   - the first call on each GPU looks up that GPU's address of the array (cudaGetSymbolAddress, with the caller's
 *     current device; this can make the runtime load the library's device code).  Make that first call during set-up,
 *     with the right device current and before any stream capture begins; later calls on that GPU only enqueue.
 * The result depends on (d_facet_momentum, nt) only: a fixed tree of 4096-facet parts.  Its summation order differs from
 * tpmc_run's, so the two agree to rounding (a few ulp of sum |P_f|), not bit for bit. */
#define TPMC_STATIC_MAX_FACETS 8388608LL
int tpmc_facet_sum_static(const double* d_facet_momentum, int64_t nt, void* cuda_stream, double* d_force);

const char* tpmc_strerror(int code);
const char* tpmc_last_cuda_error(void);
const char* tpmc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TPMC_H */
