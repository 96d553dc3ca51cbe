// run.cu -- the hot path behind tpmc_run: seed -> trace -> reflect -> accumulate -> reduce
// (steps a1-a7 of DESIGN.md).
#include <algorithm>
#include <cstdlib>
#include <new>

#include "common.cuh"
#include "sampling.cuh"
#include "sort.cuh"
#include "trace.cuh"

namespace {

constexpr int kSeedBlock = 128;
constexpr int kPrecullBlock = 256;
constexpr int kTraceBlock = 128;
constexpr int kReduceBlock = 256;
constexpr int kReduceParts = 296;   // 2 per SM

// sum of a per-thread count over the warp, added to a device counter by lane 0 (all lanes must call)
__device__ __forceinline__ void warp_count(unsigned long long* __restrict__ ctr, unsigned int v) {
  v = __reduce_add_sync(0xFFFFFFFFu, v);
  if ((threadIdx.x & 31) == 0 && v) atomicAdd(ctr, (unsigned long long)v);
}

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// ------------------------------------------------------------------------------------------------
__global__ void k_init_debug(tpmc_debug dbg, unsigned long long count) {
  const unsigned long long j = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x;
  if (j >= count) return;
  if (dbg.hash) dbg.hash[j] = 0xCBF29CE484222325ull;
  if (dbg.bounces) dbg.bounces[j] = 0u;
  if (dbg.first_facet) dbg.first_facet[j] = -1;
}

// Ray queue: region A [0, cap) holds rays reflected in the previous iteration (any earlier wave), region B
// [cap, 2 cap) the primaries of the current wave.  Record: o.xyz | particle index within the chunk,
// v.xyz | (species | bounce << 4), source facet.
struct RayQueue {
  float4* o;
  float4* v;
  int* f;
  unsigned int* key;    // sort key (sort.cuh)
  unsigned int* hist;   // histogram of the keys of this queue, or nullptr (no sort)
};

// Per-iteration device counters: ctr[2p] = rays in region A of queue p, ctr[2p+1] = rays in region B,
// ctr[4] = fetch head of the trace kernel, ctr[5] = hit-list length, ctr[6..7] = survivors of the pre-cull
// pass (seed stream), ctr[8 + b] = length of the overflow list of iterations of parity b.
__global__ void k_iter_begin(unsigned int* __restrict__ ctr, int out_parity, int iter_parity) {
  if (threadIdx.x == 0) {
    ctr[2 * out_parity] = 0u;
    ctr[2 * out_parity + 1] = 0u;
    ctr[4] = 0u;
    ctr[5] = 0u;
    ctr[8 + iter_parity] = 0u;
  }
}

// a2, pre-cull pass (sampling.cuh): fp32 estimate of every particle's ray against the grown cull volumes, in two
// stages with a compaction inside the block (precull_stage_a/b): stage A (everything but the normal speed, and a
// threshold test against the bounding sphere) for every particle of the block's share, survivors queued in
// shared memory; whenever a full block of them is waiting, stage B (normal speed, ray, cull volumes) runs
// densely on those.  Survivor records (wave offset, fp32 roots) of certified estimates fill `surv` from the
// front, particles whose estimate is not certified from the back; n_surv[0], n_surv[1] count them.
// surv = [3][cap] words, written with streaming stores (evict-first) like every list and queue of the path: the
// hierarchy and the facets (83 MB at C5) should stay in L2 while ~2 GB of lists and queues pass through it.
constexpr int kPrecullQ = 2 * kPrecullBlock;
__global__ void __launch_bounds__(kPrecullBlock) k_seed_precull(const SeedConstF sf, unsigned int seed_lo,
                                                                 unsigned int seed_hi, unsigned long long first,
                                                                 unsigned int wave_n, unsigned int cap,
                                                                 unsigned int* __restrict__ surv,
                                                                 unsigned int* __restrict__ n_surv,
                                                                 unsigned long long* __restrict__ stats) {
  __shared__ float qf[7][kPrecullQ];
  __shared__ unsigned int qj[kPrecullQ], qw[kPrecullQ], qw2[kPrecullQ];
  __shared__ unsigned char qok[kPrecullQ];
  __shared__ unsigned int q_n, s_cnt[2][kPrecullBlock / 32], s_base[2];
  const unsigned int per = (((wave_n + gridDim.x - 1) / gridDim.x) + kPrecullBlock - 1) / kPrecullBlock * kPrecullBlock;
  const unsigned long long b64 = (unsigned long long)blockIdx.x * per;
  const unsigned int begin = (unsigned int)min(b64, (unsigned long long)wave_n);
  const unsigned int end = (unsigned int)min(b64 + per, (unsigned long long)wave_n);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x == 0) q_n = 0u;
  __syncthreads();
  unsigned int base = begin, drop_a = 0u, drop_b = 0u;   // particles retired here (counted, not inferred)
  for (;;) {
    const bool more = base < end;
    if (more) {
      const unsigned int j = base + threadIdx.x;
      PrecullA a;
      const bool reach = precull_stage_a(sf, seed_lo, seed_hi, first + j, a);
      const bool pass = reach && (j < end);
      drop_a += (!reach && j < end) ? 1u : 0u;
      const unsigned m = __ballot_sync(0xFFFFFFFFu, pass);
      unsigned int pos = 0;
      if (lane == 0 && m) pos = atomicAdd(&q_n, (unsigned)__popc(m));
      pos = __shfl_sync(0xFFFFFFFFu, pos, 0);
      if (pass) {
        const unsigned int sl = pos + __popc(m & lanemask_lt());
        qf[0][sl] = a.y; qf[1][sl] = a.t; qf[2][sl] = a.cphi;
        qf[3][sl] = a.xt1; qf[4][sl] = a.xt2; qf[5][sl] = a.s; qf[6][sl] = a.chis;
        qj[sl] = j; qw[sl] = a.w3; qw2[sl] = a.w2; qok[sl] = a.ok_t ? 1 : 0;
      }
      base += kPrecullBlock;
      __syncthreads();
    }
    const unsigned int n = q_n;
    __syncthreads();   // every warp has read q_n before any warp's next stage A (or stage B) changes it
    if (n >= (unsigned)kPrecullBlock || (!more && n > 0u)) {
      const unsigned int take = min(n, (unsigned)kPrecullBlock);
      const bool active = threadIdx.x < take;
      const unsigned int sl = n - take + (active ? threadIdx.x : 0u);
      PrecullA a;
      a.y = qf[0][sl]; a.t = qf[1][sl]; a.cphi = qf[2][sl];
      a.xt1 = qf[3][sl]; a.xt2 = qf[4][sl]; a.s = qf[5][sl]; a.chis = qf[6][sl];
      a.w3 = qw[sl]; a.w2 = qw2[sl]; a.ok_t = qok[sl] != 0;
      const unsigned int j = qj[sl];
      float o[3], v[3], root[2];
      const bool ok = precull_stage_b(sf, a, o, v, root);
      const bool touch = precull_touch(sf, o, v);
      const bool keep_c = active && ok && touch, keep_u = active && !ok;
      drop_b += (active && ok && !touch) ? 1u : 0u;
      const unsigned mcert = __ballot_sync(0xFFFFFFFFu, keep_c);
      const unsigned munc = __ballot_sync(0xFFFFFFFFu, keep_u);
      if (lane == 0) { s_cnt[0][wid] = __popc(mcert); s_cnt[1][wid] = __popc(munc); }
      __syncthreads();                      // also: every read of the queue entries above is done
      if (threadIdx.x == 0) q_n = n - take;
      if (threadIdx.x < 2) {
        unsigned int tot = 0;
        for (int k = 0; k < kPrecullBlock / 32; ++k) { const unsigned int c = s_cnt[threadIdx.x][k]; s_cnt[threadIdx.x][k] = tot; tot += c; }
        s_base[threadIdx.x] = tot ? atomicAdd(&n_surv[threadIdx.x], tot) : 0u;
      }
      __syncthreads();
      if (keep_c) {
        const unsigned slot = s_base[0] + s_cnt[0][wid] + __popc(mcert & lanemask_lt());
        __stcs(surv + slot, j);
        __stcs(surv + cap + slot, __float_as_uint(root[0]));
        __stcs(surv + 2 * cap + slot, __float_as_uint(root[1]));
      }
      if (keep_u) __stcs(surv + (cap - 1u - (s_base[1] + s_cnt[1][wid] + __popc(munc & lanemask_lt()))), j);
      __syncthreads();
    } else if (!more) {
      break;
    }
  }
  warp_count(&stats[ST_RET_PA], drop_a);
  warp_count(&stats[ST_RET_PB], drop_b);
}

// a2: seed particles of one wave in fp64, round the state to fp32 (O9), drop the rays that cannot touch the
// mesh AABB or any box of the top of the hierarchy (their single segment is an escape; same conservative
// slab test as the traversal) and append the rest to the ray queue.
// surv != nullptr: dense over the survivors of the pre-cull pass; else over all wave_n particles.
__global__ void __launch_bounds__(kSeedBlock) k_seed(const RunConst rc, unsigned int wave_first,
                                                     unsigned int wave_n, const unsigned int* __restrict__ surv,
                                                     unsigned int cap_s, const unsigned int* __restrict__ n_surv,
                                                     const uint4* __restrict__ cull_c, const QuantGrid grid, int walk,
                                                     const RayQueue q, unsigned int region_b,
                                                     unsigned int* __restrict__ qcount,
                                                     unsigned long long* __restrict__ stats) {
  const unsigned int n1 = surv ? n_surv[0] : 0u;                 // certified survivors: fp32 roots available
  const unsigned int n = surv ? n1 + n_surv[1] : wave_n;
  if (surv && blockIdx.x == 0 && threadIdx.x == 0 && n_surv[1]) atomicAdd(&stats[ST_UNCERT], (unsigned long long)n_surv[1]);
  const unsigned int stride = gridDim.x * blockDim.x;
  const unsigned int nround = ((n + stride - 1) / stride) * stride;   // keep warps converged for the ballots
  for (unsigned int kk = blockIdx.x * blockDim.x + threadIdx.x; kk < nround; kk += stride) {
  const bool active = kk < n;
  const bool hinted = kk < n1;
  const unsigned int sl = hinted ? kk : cap_s - 1u - (kk - n1);
  const unsigned int j = active ? (surv ? __ldcs(surv + sl) : kk) : 0u;
  bool keep = false;
  float o[3] = {0, 0, 0}, v[3] = {1, 1, 1};
  int species = 0;
  if (active) {
    float hint[2] = {0.0f, 0.0f};
    if (hinted) { hint[0] = __uint_as_float(__ldcs(surv + cap_s + sl)); hint[1] = __uint_as_float(__ldcs(surv + 2 * cap_s + sl)); }
    const SeedState s = rc.control_volume == TPMC_CV_SPHERE ? seed_particle(rc, rc.first + wave_first + j, hinted ? hint : nullptr)
                                                            : seed_particle_box(rc, rc.first + wave_first + j);
    species = s.species;
#pragma unroll
    for (int k = 0; k < 3; ++k) { o[k] = (float)s.x[k]; v[k] = (float)s.v[k]; }
    const float id[3] = {1.0f / v[0], 1.0f / v[1], 1.0f / v[2]};
    float tn;
    keep = slab(rc.aabb_lo[0], rc.aabb_lo[1], rc.aabb_lo[2], rc.aabb_hi[0], rc.aabb_hi[1], rc.aabb_hi[2], o, id,
                INFINITY, tn) && (!walk || cull_touch_q(cull_c, grid, o, v));
  }
  const unsigned m = __ballot_sync(0xFFFFFFFFu, keep);
  const unsigned mc = __ballot_sync(0xFFFFFFFFu, active && !keep);
  const int lane = threadIdx.x & 31;
  unsigned base = 0;
  if (lane == 0) {
    if (m) { base = atomicAdd(qcount, (unsigned)__popc(m)); atomicAdd(&stats[ST_Q_PRIM], (unsigned long long)__popc(m)); }
    if (mc) atomicAdd(&stats[ST_RET_SEED], (unsigned long long)__popc(mc));
  }
  base = __shfl_sync(0xFFFFFFFFu, base, 0);
  if (keep) {
    const unsigned slot = region_b + base + __popc(m & lanemask_lt());
    __stcs(q.o + slot, make_float4(o[0], o[1], o[2], __uint_as_float(wave_first + j)));
    __stcs(q.v + slot, make_float4(v[0], v[1], v[2], __uint_as_float((unsigned int)species)));   // bounce 0
    __stcs(q.f + slot, -1);
    if (q.hist) {
      const SortKeyConst kc = {{rc.key_c[0], rc.key_c[1], rc.key_c[2]}, rc.key_r2};
      const unsigned int key = primary_key(kc, o, v);
      __stcs(q.key + slot, key);
      atomicAdd(q.hist + key, 1u);
    }
  }
  }
}


// a3: wavefront traversal.  Persistent warps, one ray per lane, fp32 only (see trace.cuh).
//  * node phase: lanes standing at an internal node step together (two steps per warp vote, branch-free
//    child selection).  A lane that reaches a leaf puts it aside and walks on speculatively; it waits only
//    when it reaches a second leaf or its stack is empty;
//  * leaf phase: once fewer than kNodeMin lanes can still step, every lane with a leaf put aside classifies
//    its facet (the ~120-instruction facet code then runs with many lanes active, not one);
//  * a lane whose ray has finished takes the next ray of the queue as soon as kRefillIdle lanes are idle
//    (one warp-aggregated atomic), so rays of very different length do not idle the warp.
// Rays that end with at least one candidate facet are appended to the hit list for k_reflect.
#ifndef TPMC_NODE_MIN
#define TPMC_NODE_MIN 20
#endif
#ifndef TPMC_REFILL_IDLE
#define TPMC_REFILL_IDLE 4
#endif
#ifndef TPMC_TRACE_MIN_BLOCKS
#define TPMC_TRACE_MIN_BLOCKS 7   // 72 registers: the wide node step spills at 64 (measured: 7 x 72 is 1.6 % faster than 8 x 64)
#endif
#ifndef TPMC_NODE_STEPS
#define TPMC_NODE_STEPS 2   // wide-node steps per warp vote (a loop over one copy of the step: the votes are 8 % of the issue slots at 1)
#endif
#ifndef TPMC_SRAY
#define TPMC_SRAY 1
#endif
struct TraceTune { int node_min, refill_idle; };
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const unsigned int sa = (unsigned int)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
constexpr int kFetchChunk = 32;   // rays a warp reserves per atomic on the queue head: one per lane (set up together, see k_trace_wf)
constexpr int kHitBlock = 64;     // hit-list slots a warp reserves per atomic
constexpr unsigned int kNoRay = 0xFFFFFFFFu;   // hit_ray: reserved slot without a ray
constexpr size_t kHitSlack = (size_t)1 << 19;   // >= resident warps x kHitBlock: slots reserved but not used
constexpr int kChunkWords = 11;   // per ray of the chunk: 1/d', the two slab offsets per axis, the octant, the queue slot

__global__ void __launch_bounds__(kTraceBlock, TPMC_TRACE_MIN_BLOCKS) k_trace_wf(const uint4* __restrict__ wnodes,
                                                             const QuantGrid* __restrict__ gridp,
                                                             const float4* __restrict__ tris, const RayQueue q,
                                                             const unsigned int* __restrict__ order,
                                                             unsigned int cap, const unsigned int* __restrict__ n_rays,
                                                             unsigned int* __restrict__ next_ray,
                                                             unsigned int* __restrict__ hit_ray,
                                                             int4* __restrict__ hit_cand,
                                                             unsigned int* __restrict__ n_hits,
                                                             unsigned long long* __restrict__ stats,
                                                             const TraceTune tune) {
  const int kNodeMin = tune.node_min, kRefillIdle = tune.refill_idle;
  __shared__ int sstack[(TPMC_STACK_SMEM + 6) * kTraceBlock];      // two guard rows, TPMC_STACK_SMEM rows, four of headroom
  __shared__ unsigned int schunk[kChunkWords][kTraceBlock];        // the warp's current chunk of rays, set up for the walk
#if TPMC_SRAY
  __shared__ float4 sray[2][kTraceBlock];                          // the lane's ray (o | index, d | species) for the leaf phases
#endif
  int* stk = sstack + 2 * kTraceBlock + threadIdx.x;   // level 0; levels -1, -2 are the guard entries (walk_pop)
  stk[-kTraceBlock] = TPMC_SENTINEL;
  stk[-2 * kTraceBlock] = TPMC_SENTINEL;
  const unsigned int na = min(n_rays[0], cap), n = na + n_rays[1];   // region A (reflected), region B (primaries)
  const int lane = threadIdx.x & 31, wbase = threadIdx.x & ~31;
  const unsigned FULL = 0xFFFFFFFFu;
  bool has = false, exhausted = false, fin = false;
  unsigned int r = 0, pool_next = 0, pool_end = 0, hpool_next = 0, hpool_end = 0;
  Walk w;
  w.cur = TPMC_SENTINEL; w.stash = 0; w.sp = 0; w.nc = 0; w.tmax = 0.0f; w.f_prev = -1;
  TraceCounters cnt;
  cnt.nodes = 0; cnt.tris = 0;
  unsigned int n_escaped = 0u;   // rays that ended without a candidate facet: these particles retire here
  for (;;) {
    // ---- refill idle lanes from the warp's chunk of the queue.  A chunk is kFetchChunk = 32 consecutive rays (one
    // atomic on the queue head); when a warp takes one, ALL its lanes set up one ray each for the walk (rotation into the
    // grid's frame, reciprocal direction, slab offsets: grid_ray) and park the result in shared memory, so that the
    // ~150 instructions of set-up run with 32 lanes active instead of the handful that happen to be idle; a lane that
    // runs out of work later picks its ray up from there.
    const unsigned idle = __ballot_sync(FULL, !has && !exhausted);
    const unsigned busy0 = __ballot_sync(FULL, has);
    if (idle && (__popc(idle) >= kRefillIdle || busy0 == 0u)) {
      if (pool_next == pool_end) {
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(next_ray, (unsigned)kFetchChunk);
        pool_next = __shfl_sync(FULL, base, 0);
        pool_end = pool_next + kFetchChunk;
        const unsigned int rr = pool_next + lane;
        if (rr < n) {
          const unsigned int phys = order ? __ldcs(order + rr) : ((rr < na) ? rr : cap + (rr - na));   // physical slot (in key order when sorted)
          const float4 ro = __ldcs(q.o + phys), rv = __ldcs(q.v + phys);
          const float o[3] = {ro.x, ro.y, ro.z}, d[3] = {rv.x, rv.y, rv.z};
          GridRay g;
          grid_ray(g, *gridp, o, d);
          unsigned int* c = &schunk[0][wbase + lane];
#pragma unroll
          for (int k = 0; k < 3; ++k) {
            c[k * kTraceBlock] = __float_as_uint(g.id[k]);
            c[(3 + k) * kTraceBlock] = __float_as_uint(g.ncn[k]);
            c[(6 + k) * kTraceBlock] = __float_as_uint(g.ncf[k]);
          }
          c[9 * kTraceBlock] = (g.sn[0] == 0x7632u ? 1u : 0u) | (g.sn[1] == 0x7632u ? 2u : 0u) | (g.sn[2] == 0x7632u ? 4u : 0u);
          c[10 * kTraceBlock] = phys;
        }
        __syncwarp();
      }
      const unsigned avail = pool_end - pool_next, rank = __popc(idle & lanemask_lt());
      if (!has && !exhausted) {
        if (pool_next >= n) {
          exhausted = true;
        } else if (rank < avail && pool_next + rank < n) {
          const unsigned int* c = &schunk[0][wbase + (kFetchChunk - avail) + rank];
#pragma unroll
          for (int k = 0; k < 3; ++k) {
            w.g.id[k] = __uint_as_float(c[k * kTraceBlock]);
            w.g.ncn[k] = __uint_as_float(c[(3 + k) * kTraceBlock]);
            w.g.ncf[k] = __uint_as_float(c[(6 + k) * kTraceBlock]);
          }
          const unsigned int oct = c[9 * kTraceBlock];
#pragma unroll
          for (int k = 0; k < 3; ++k) {
            const bool neg = (oct >> k) & 1u;
            w.g.sn[k] = neg ? 0x7632u : 0x7610u;
            w.g.sf[k] = neg ? 0x7610u : 0x7632u;
          }
          r = c[10 * kTraceBlock];
          walk_reset(w, __ldcs(q.f + r));
#if TPMC_SRAY
          // asynchronous copies global -> shared (the records were just read by the lane that set the ray up): the lane
          // does not wait for them here; the first leaf phase does (cp.async.wait_all), long after they have landed
          asm volatile("cp.async.wait_all;" ::: "memory");   // (a previous ray's copy that was never waited for must not land after this one)
          cp_async16(&sray[0][threadIdx.x], q.o + r);
          cp_async16(&sray[1][threadIdx.x], q.v + r);
#endif
          has = true;
        }
      }
      pool_next += min((unsigned)__popc(idle), avail);
      __syncwarp();   // every read of the chunk is done before a later iteration may replace it
    }
    if (__ballot_sync(FULL, has) == 0u) break;
    // ---- node phase: two node steps per vote
    for (;;) {
      const bool at_node = has && (unsigned)w.cur < (unsigned)TPMC_SENTINEL;
      const unsigned mn = __ballot_sync(FULL, at_node);
      if (__popc(mn) < kNodeMin) {
        const unsigned ml = __ballot_sync(FULL, has && w.stash != 0);
        if (mn == 0u || ml != 0u) break;
      }
#if TPMC_NODE_STEPS > 1
#pragma unroll 1
      for (int rep = 0; rep < TPMC_NODE_STEPS; ++rep)   // (one copy of the step's code: unrolled, it spills)
        if (has && (unsigned)w.cur < (unsigned)TPMC_SENTINEL) walk_node(w, wnodes, stk, kTraceBlock, cnt);
#else
      if (at_node) walk_node(w, wnodes, stk, kTraceBlock, cnt);
#endif
    }
    // ---- leaf phase: every lane that put a leaf aside classifies it
    if (has && w.stash != 0) {
#if TPMC_SRAY
      // the ray lives in shared memory: six registers stay free during the node phase
      asm volatile("cp.async.wait_all;" ::: "memory");
      const float4 ro = sray[0][threadIdx.x], rv = sray[1][threadIdx.x];
      const float o[3] = {ro.x, ro.y, ro.z}, d[3] = {rv.x, rv.y, rv.z};
#else
      const float4 ro = q.o[r], rv = q.v[r];   // re-read (cache-resident): keeps six registers free during the node phase
      const float o[3] = {ro.x, ro.y, ro.z}, d[3] = {rv.x, rv.y, rv.z};
#endif
      walk_leaf(w, tris, o, d, stk, kTraceBlock, cnt);
    }
    if (has && w.cur == TPMC_SENTINEL && w.stash == 0) { has = false; fin = w.nc > 0; n_escaped += fin ? 0u : 1u; }
    // ---- finished rays with candidates -> hit list.  A warp reserves hit-list slots kHitBlock at a time (one atomic per
    // block instead of one per finish event of ~5 rays, and no round trip to the counter on the common path).  Finishing
    // lanes that do not fit the rest of the warp's block fill that rest first and go on in a fresh block, so every slot
    // of every block but a warp's last is used: slots handed out <= hits + warps * kHitBlock <= 2 * wave_cap + kHitSlack,
    // the size of hit_ray / hit_cand (ensure_scratch; the grid is clamped so that warps * kHitBlock <= kHitSlack).
    // The unused tail of a warp's last block is marked empty (kNoRay) and skipped by the reflect step.
    const unsigned fm = __ballot_sync(FULL, fin);
    if (fm) {
      const unsigned nf = __popc(fm), rest = hpool_end - hpool_next;   // nf <= 32 < kHitBlock
      unsigned nbase = hpool_next;
      if (nf > rest) {
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(n_hits, (unsigned)kHitBlock);
        nbase = __shfl_sync(FULL, base, 0) - rest;   // slot of rank k >= rest: (new block) + k - rest
      }
      if (fin) {
        const unsigned rk = __popc(fm & lanemask_lt());
        const unsigned h = (rk < rest ? hpool_next : nbase) + rk;
        __stcs(hit_ray + h, r);
        int4 cd = make_int4(-1, -1, -1, -1);
        cd.x = w.cs[0];
        if (TPMC_MAX_CAND > 1) cd.y = w.cs[TPMC_MAX_CAND > 1 ? 1 : 0];
        if (TPMC_MAX_CAND > 2) cd.z = w.cs[TPMC_MAX_CAND > 2 ? 2 : 0];
        if (TPMC_MAX_CAND > 3) cd.w = w.cs[TPMC_MAX_CAND > 3 ? 3 : 0];
        __stcs(hit_cand + h, (w.nc > TPMC_MAX_CAND) ? make_int4(-1, -1, -1, TPMC_CAND_OVERFLOW) : cd);
        fin = false;
      }
      if (nf > rest) { hpool_next = nbase + nf; hpool_end = nbase + rest + kHitBlock; }
      else hpool_next += nf;
    }
  }
  for (unsigned int h = hpool_next + lane; h < hpool_end; h += 32u) __stcs(hit_ray + h, kNoRay);   // the unused rest of the last block
  // counters: one atomic per warp
  unsigned long long cn = cnt.nodes, ct = cnt.tris;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    cn += __shfl_down_sync(FULL, cn, off);
    ct += __shfl_down_sync(FULL, ct, off);
  }
  if (lane == 0) {
    if (cn) atomicAdd(&stats[ST_NODES], cn);
    if (ct) atomicAdd(&stats[ST_TRIS], ct);
  }
  warp_count(&stats[ST_RET_TRACE], n_escaped);
  if (blockIdx.x == 0 && threadIdx.x == 0 && n) atomicAdd(&stats[ST_TRACED], (unsigned long long)n);
}

// Block-level sum of per-thread torque and counters, one atomic per block and quantity.
// c[k] is added to stats[c_flush_idx[which][k]], k < kFlushCounters (which: 0 = k_reflect, 1 = k_finish).
constexpr int kFlushCounters = 10;
enum { FC_HITS = 0, FC_TRUNC, FC_TRIS, FC_NODES, FC_HORIZON, FC_NOHIT, FC_QUEUED, FC_RETRACE, FC_PENDING, FC_SEGS };
__constant__ int c_flush_idx[2][kFlushCounters] = {
    {ST_HITS, ST_TRUNC, ST_TRIS, ST_NODES, ST_RET_HORIZON, ST_RET_RESOLVE, ST_Q_REFL, ST_OVF_RETRACE, ST_OVF_PENDING, ST_FIN_SEGS},
    {ST_HITS, ST_TRUNC, ST_TRIS, ST_NODES, ST_RET_HORIZON, ST_RET_FINISH, ST_Q_REFL, ST_OVF_RETRACE, ST_OVF_PENDING, ST_FIN_SEGS}};
struct FlushShared {
  double red[3][8];
  unsigned int cnt[kFlushCounters][8];
};
__device__ __forceinline__ void block_flush(double tq[3], const unsigned int c[kFlushCounters], int which,
                                            double* __restrict__ torque, unsigned long long* __restrict__ stats,
                                            FlushShared& sh) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
    for (int a = 0; a < 3; ++a) tq[a] += __shfl_down_sync(0xFFFFFFFFu, tq[a], off);
  }
#pragma unroll
  for (int a = 0; a < kFlushCounters; ++a) {
    const unsigned int v = __reduce_add_sync(0xFFFFFFFFu, c[a]);
    if (lane == 0) sh.cnt[a][wid] = v;
  }
  if (lane == 0)
    for (int a = 0; a < 3; ++a) sh.red[a][wid] = tq[a];
  __syncthreads();
  if (threadIdx.x == 0) {
    double t3[3] = {0, 0, 0};
    for (int wv = 0; wv < nw; ++wv)
      for (int a = 0; a < 3; ++a) t3[a] += sh.red[a][wv];
    for (int a = 0; a < 3; ++a) if (t3[a] != 0.0) atomicAdd(&torque[a], t3[a]);
  }
  if (threadIdx.x < kFlushCounters) {
    unsigned long long tot = 0;
    for (int wv = 0; wv < nw; ++wv) tot += sh.cnt[threadIdx.x][wv];
    if (tot) atomicAdd(&stats[c_flush_idx[which][threadIdx.x]], tot);
  }
}

// One surface interaction (O11-O13) of a particle whose closest hit is known: momentum and torque
// accumulation, debug records, and the state of the next segment.  Returns GO_ON, or why the particle retires here.
enum { GO_ON = 0, END_TRUNCATED = 1, END_HORIZON = 2 };
struct Particle {
  float o[3], v[3];
  unsigned long long j;   // index within the chunk (rc.first = first particle of the chunk)
  int species;
  unsigned int k;         // reflections so far
  int f_prev;
};

// P != nullptr: dp goes straight to the facet's accumulators (fp64 atomics); else the caller adds dp_out (a5).
__device__ __forceinline__ int interact(const RunConst& rc, const float4* __restrict__ tris, Particle& p, const Hit& hit,
                                        double* __restrict__ P, double tq[3], const tpmc_debug& dbg,
                                        const uint4* __restrict__ horizon, double dp_out[3] = nullptr) {
  const float4 q0 = __ldg(tris + 3 * (size_t)hit.slot), q1 = __ldg(tris + 3 * (size_t)hit.slot + 1),
               q2 = __ldg(tris + 3 * (size_t)hit.slot + 2);
  const double w = rc.sp[p.species].w;
  // A23: accommodation and wall temperature of the facet hit; A22: re-emission temperature of this particle,
  // T_r = alpha_E T_W + (1 - alpha_E) m v_in^2 / (3 k_B), every operation rounded separately (the definition fixes the order)
  const double sigma = rc.surf_sigma ? __ldg(rc.surf_sigma + hit.facet) : rc.sigma;
  double cW = rc.sp[p.species].cW;
  if (!rc.simple_surface) {
    const double ms = rc.sp[p.species].m;
    const double TW = rc.surf_TW ? __ldg(rc.surf_TW + hit.facet) : rc.T_W;
    const double vx = (double)p.v[0], vy = (double)p.v[1], vz = (double)p.v[2];
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(vx, vx), __dmul_rn(vy, vy)), __dmul_rn(vz, vz));
    const double Tki = __ddiv_rn(__dmul_rn(ms, v2), __dmul_rn(3.0, TPMC_KB));
    const double Tr = __dadd_rn(__dmul_rn(rc.alpha_E, TW), __dmul_rn(__dsub_rn(1.0, rc.alpha_E), Tki));
    cW = sqrt(__ddiv_rn(__dmul_rn(__dmul_rn(2.0, TPMC_KB), Tr), ms));
  }
  double vout[3];
  float sin_e, phi;
  reflect(q0, q1, q2, p.v, sigma, cW, particle_block(rc, rc.first + p.j, 2u + p.k), vout, sin_e, phi);
  // O12: dp = w (v_in - v_out) on the fp32 values; hit point o + tau v in fp64
  double hp[3], dp[3];
  float vo[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    vo[a] = (float)vout[a];
    hp[a] = __dadd_rn((double)p.o[a], __dmul_rn(hit.tau, (double)p.v[a]));
    dp[a] = w * ((double)p.v[a] - (double)vo[a]);
    if (P) atomicAdd(&P[3 * (size_t)hit.facet + a], dp[a]);
    else dp_out[a] = dp[a];
  }
  const double rx = hp[0] - rc.x_ref[0], ry = hp[1] - rc.x_ref[1], rz = hp[2] - rc.x_ref[2];
  tq[0] += ry * dp[2] - rz * dp[1];
  tq[1] += rz * dp[0] - rx * dp[2];
  tq[2] += rx * dp[1] - ry * dp[0];
  if (dbg.hash) dbg.hash[p.j] = fnv1a_facet(dbg.hash[p.j], hit.facet);
  if (dbg.bounces) dbg.bounces[p.j] = p.k + 1u;
  if (dbg.first_facet && p.k == 0u) dbg.first_facet[p.j] = hit.facet;
  // O13: next segment starts at the fp32-rounded hit point
#pragma unroll
  for (int a = 0; a < 3; ++a) { p.o[a] = (float)hp[a]; p.v[a] = vo[a]; }
  p.f_prev = hit.facet;
  ++p.k;
  if (p.k >= rc.max_bounces) return END_TRUNCATED;
  // escape horizon of the facet (k_horizon, lbvh.cu): above it the next segment cannot hit anything
  if (horizon) {
    const int sector = min(max((int)floorf((phi + 3.14159265f) * 2.54647909f), 0), 15);   // 16 / (2 pi)
    const unsigned int b = __ldg((const unsigned char*)horizon + 16 * (size_t)hit.slot + sector);
    if (b < 255u && sin_e > (float)b * (1.0f / 254.0f)) return END_HORIZON;
  }
  return GO_ON;
}

// a5: per-facet momentum, warp-aggregated.  Lanes of a (converged) warp that hit the same facet are summed with
// shuffles and their leader issues one fp64 atomic per component: one loop iteration per DISTINCT facet among the
// warp's hits.  That pays when a body has few facets (C1: 2, C3: 2048 -- many lanes per facet, hot accumulators)
// and costs when every lane has its own (C5), so the caller decides per run (aggregate = nt <= kAggregateMaxFacets).
constexpr long long kAggregateMaxFacets = 4096;
__device__ __forceinline__ void accumulate_warp(double* __restrict__ P, bool is_hit, int facet, const double dp[3],
                                                bool aggregate) {
  const unsigned FULL = 0xFFFFFFFFu;
  if (!aggregate) {
    if (is_hit)
      for (int a = 0; a < 3; ++a) atomicAdd(&P[3 * (size_t)facet + a], dp[a]);
    return;
  }
  const int lane = threadIdx.x & 31;
  unsigned todo = __ballot_sync(FULL, is_hit);
  while (todo) {
    const int src = __ffs(todo) - 1;
    const int f = __shfl_sync(FULL, facet, src);
    const bool mine = is_hit && facet == f;
    const unsigned grp = __ballot_sync(FULL, mine);
    double s0 = mine ? dp[0] : 0.0, s1 = mine ? dp[1] : 0.0, s2 = mine ? dp[2] : 0.0;
    if (grp != (1u << src)) {   // more than one lane on this facet: butterfly sum (zeros elsewhere)
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) {
        s0 += __shfl_xor_sync(FULL, s0, off);
        s1 += __shfl_xor_sync(FULL, s1, off);
        s2 += __shfl_xor_sync(FULL, s2, off);
      }
    }
    if (lane == src) {
      atomicAdd(&P[3 * (size_t)f], s0);
      atomicAdd(&P[3 * (size_t)f + 1], s1);
      atomicAdd(&P[3 * (size_t)f + 2], s2);
    }
    todo &= ~grp;
  }
}

#ifndef TPMC_REFLECT_MIN_BLOCKS
#define TPMC_REFLECT_MIN_BLOCKS 6
#endif
// a4-a6: resolve the candidates of every hit ray with the exact fp64 test, apply the surface interaction,
// accumulate, and queue the reflected ray for the next wavefront round (compacted, warp-aggregated).
// Rays the traversal gave up on (too many candidates, stack too deep) and rays whose reflected successor
// finds region A of the next queue full go, untouched, to the overflow list: k_finish follows them to escape
// with the full fp64 traversal, densely, instead of one lane doing so here while its warp waits.
#ifndef TPMC_REFLECT_PREFETCH
#define TPMC_REFLECT_PREFETCH 0   // 1, 2: software-prefetch variants, measured slower or equal
#endif
__global__ void __launch_bounds__(kTraceBlock, TPMC_REFLECT_MIN_BLOCKS) k_reflect(const RunConst rc, unsigned int cap,
                                                         const float4* __restrict__ tris, const RayQueue qin,
                                                         const unsigned int* __restrict__ hit_ray,
                                                         const int4* __restrict__ hit_cand,
                                                         const unsigned int* __restrict__ n_hits, const RayQueue qout,
                                                         unsigned int* __restrict__ n_out,
                                                         unsigned int* __restrict__ ovf, unsigned int* __restrict__ n_ovf,
                                                         double* __restrict__ P, double* __restrict__ torque,
                                                         unsigned long long* __restrict__ stats, tpmc_debug dbg,
                                                         const uint4* __restrict__ horizon, int aggregate) {
  __shared__ FlushShared fsh;
  const unsigned int n = *n_hits;
  const int lane = threadIdx.x & 31;
  const unsigned FULL = 0xFFFFFFFFu;
  double tq[3] = {0.0, 0.0, 0.0};
  unsigned int c[kFlushCounters] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
  const unsigned int stride = gridDim.x * blockDim.x;
  const unsigned int nround = ((n + stride - 1) / stride) * stride;   // keep warps converged for the ballots
#if TPMC_REFLECT_PREFETCH
  // The chain hit list -> ray record -> facet -> horizon -> accumulators is a sequence of dependent scattered loads, and
  // the kernel is bound by their latency (ncu: 7 long-scoreboard stalls per issue, no unit above 45 %).  The list entry of
  // the thread's NEXT hit is therefore read one iteration ahead, and the lines it points to (ray record, first candidate
  // facet) are prefetched while the current hit is worked on.
  unsigned int h0 = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned int r_nx = h0 < n ? __ldcs(hit_ray + h0) : kNoRay;
#if TPMC_REFLECT_PREFETCH == 1
  int4 c_nx = h0 < n ? __ldcs(hit_cand + h0) : make_int4(-1, -1, -1, -1);
#endif
#endif
  for (unsigned int h = blockIdx.x * blockDim.x + threadIdx.x; h < nround; h += stride) {
    bool spill = false, is_hit = false;
    unsigned int r = 0;
    Particle p;
    Hit hit;
    hit.facet = -1;
#if TPMC_REFLECT_PREFETCH
    r = h < n ? r_nx : 0u;
#if TPMC_REFLECT_PREFETCH == 1
    const int4 cand_cur = c_nx;
#endif
    {
      const unsigned int hn = h + stride;
      r_nx = hn < n ? __ldcs(hit_ray + hn) : kNoRay;
#if TPMC_REFLECT_PREFETCH == 1
      c_nx = hn < n ? __ldcs(hit_cand + hn) : make_int4(-1, -1, -1, -1);
#endif
    }
#else
    if (h < n) r = __ldcs(hit_ray + h);
#endif
    if (h < n && r != kNoRay) {
#if TPMC_REFLECT_PREFETCH == 1
      const int4 cand = cand_cur;
#else
      const int4 cand = __ldcs(hit_cand + h);
#endif
      if (cand.w == TPMC_CAND_OVERFLOW) {
        spill = true;
        ++c[FC_RETRACE];
      } else {
        const float4 ro = __ldcs(qin.o + r), rv = __ldcs(qin.v + r);
        p.o[0] = ro.x; p.o[1] = ro.y; p.o[2] = ro.z;
        p.v[0] = rv.x; p.v[1] = rv.y; p.v[2] = rv.z;
        p.j = __float_as_uint(ro.w);
        const unsigned int pk = __float_as_uint(rv.w);
        p.species = (int)(pk & 15u);
        p.k = pk >> 4;
        p.f_prev = __ldcs(qin.f + r);
        hit = resolve_candidates(tris, cand, p.o, p.v, c[FC_TRIS]);
        is_hit = hit.facet >= 0;
        c[FC_NOHIT] += is_hit ? 0u : 1u;
      }
    }
#if TPMC_REFLECT_PREFETCH == 2
    if (r_nx != kNoRay) {
      asm volatile("prefetch.global.L2 [%0];" ::"l"(qin.o + r_nx));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(qin.v + r_nx));
    }
#endif
#if TPMC_REFLECT_PREFETCH == 1
    if (r_nx != kNoRay) {   // (by now the next list entry has arrived)
      asm volatile("prefetch.global.L1 [%0];" ::"l"(qin.o + r_nx));
      asm volatile("prefetch.global.L1 [%0];" ::"l"(qin.v + r_nx));
      asm volatile("prefetch.global.L1 [%0];" ::"l"(qin.f + r_nx));
      if (c_nx.x >= 0) {
        const float4* tp = tris + 3 * (size_t)c_nx.x;
        asm volatile("prefetch.global.L1 [%0];" ::"l"(tp));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(tp + 2));
      }
    }
#endif
    // surface interaction, then a queue slot for every particle that goes on (warp-aggregated).  A particle
    // that finds region A of the next queue full writes its new state back into its own slot of this queue
    // and goes to the overflow list, like one the traversal gave up on.
    bool go_on = false;
    double dp[3] = {0.0, 0.0, 0.0};
    if (is_hit) {
      ++c[FC_HITS];
      const int end = interact(rc, tris, p, hit, nullptr, tq, dbg, horizon, dp);
      go_on = end == GO_ON;
      c[FC_TRUNC] += end == END_TRUNCATED ? 1u : 0u;
      c[FC_HORIZON] += end == END_HORIZON ? 1u : 0u;
    }
    accumulate_warp(P, is_hit, hit.facet, dp, aggregate != 0);
    const unsigned em = __ballot_sync(FULL, go_on);
    if (em) {
      const int leader = __ffs(em) - 1;
      unsigned base = 0;
      if (lane == leader) base = atomicAdd(n_out, (unsigned)__popc(em));
      base = __shfl_sync(FULL, base, leader);
      if (go_on) {
        const unsigned s = base + __popc(em & lanemask_lt());
        const RayQueue& qd = (s >= cap) ? qin : qout;
        const unsigned sd = (s >= cap) ? r : s;
        spill = s >= cap;
        c[FC_PENDING] += spill ? 1u : 0u;
        c[FC_QUEUED] += spill ? 0u : 1u;
        __stcs(qd.o + sd, make_float4(p.o[0], p.o[1], p.o[2], __uint_as_float((unsigned int)p.j)));
        __stcs(qd.v + sd, make_float4(p.v[0], p.v[1], p.v[2], __uint_as_float((unsigned int)p.species | (p.k << 4))));
        __stcs(qd.f + sd, p.f_prev);
        if (qout.hist && !spill) {
          const SortKeyConst kc = {{rc.key_c[0], rc.key_c[1], rc.key_c[2]}, rc.key_r2};
          const unsigned int key = origin_key(kc, p.o);
          __stcs(qout.key + s, key);
          atomicAdd(qout.hist + key, 1u);
        }
      }
    }
    const unsigned sm = __ballot_sync(FULL, spill);
    if (sm) {
      const int leader = __ffs(sm) - 1;
      unsigned base = 0;
      if (lane == leader) base = atomicAdd(n_ovf, (unsigned)__popc(sm));
      base = __shfl_sync(FULL, base, leader);
      if (spill) ovf[base + __popc(sm & lanemask_lt())] = r;
    }
  }
  block_flush(tq, c, 0, torque, stats, fsh);
}

// Particles followed to escape thread by thread (full fp64 traversal per segment): the overflow list of an
// iteration (list != nullptr: queue slots) and, after the wavefront rounds, the stragglers still in the
// queue.  Few particles get here; long multi-bounce paths live here.
__global__ void __launch_bounds__(kTraceBlock) k_finish(const RunConst rc, unsigned int cap,
                                                        const float4* __restrict__ nodes,
                                                        const float4* __restrict__ tris, const RayQueue q,
                                                        const unsigned int* __restrict__ list,
                                                        const unsigned int* __restrict__ n_rays,
                                                        double* __restrict__ P, double* __restrict__ torque,
                                                        unsigned long long* __restrict__ stats, tpmc_debug dbg,
                                                        const uint4* __restrict__ horizon) {
  __shared__ int sstack[TPMC_STACK_SMEM * kTraceBlock];
  __shared__ FlushShared fsh;
  const unsigned int n = list ? *n_rays : min(*n_rays, cap);
  if (!list && blockIdx.x == 0 && threadIdx.x == 0 && n) atomicAdd(&stats[ST_STRAGGLERS], (unsigned long long)n);
  double tq[3] = {0.0, 0.0, 0.0};
  unsigned int c[kFlushCounters] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
  TraceCounters cnt;
  cnt.nodes = 0; cnt.tris = 0;
  for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const unsigned int r = list ? list[i] : i;
    const float4 ro = q.o[r], rv = q.v[r];
    Particle p;
    p.o[0] = ro.x; p.o[1] = ro.y; p.o[2] = ro.z;
    p.v[0] = rv.x; p.v[1] = rv.y; p.v[2] = rv.z;
    p.j = __float_as_uint(ro.w);
    const unsigned int pk = __float_as_uint(rv.w);
    p.species = (int)(pk & 15u);
    p.k = pk >> 4;
    p.f_prev = q.f[r];
    for (;;) {
      const Hit hit = closest_hit(nodes, tris, p.o, p.v, p.f_prev, sstack + threadIdx.x, kTraceBlock, cnt);
      ++c[FC_SEGS];
      if (hit.facet < 0) { ++c[FC_NOHIT]; break; }
      ++c[FC_HITS];
      const int end = interact(rc, tris, p, hit, P, tq, dbg, horizon);
      c[FC_TRUNC] += end == END_TRUNCATED ? 1u : 0u;
      c[FC_HORIZON] += end == END_HORIZON ? 1u : 0u;
      if (end != GO_ON) break;
    }
  }
  c[FC_TRIS] = cnt.tris;
  c[FC_NODES] = cnt.nodes;
  block_flush(tq, c, 1, torque, stats, fsh);
}

// TPMC_FLAG_EXACT_TRACE: every queued ray goes to the overflow list (the straggler kernel follows it to escape with
// the fp64 closest-hit search); the traversal and reflect kernels then see an empty queue.
__global__ void k_divert(unsigned int cap, unsigned int* __restrict__ n_rays, unsigned int* __restrict__ ovf,
                         unsigned int* __restrict__ n_ovf, unsigned long long* __restrict__ stats) {
  const unsigned int na = min(n_rays[0], cap), n = na + n_rays[1];
  for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    ovf[i] = (i < na) ? i : cap + (i - na);
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    *n_ovf = n;
    if (n) atomicAdd(&stats[ST_DIVERTED], (unsigned long long)n);
  }
}


// a7: F = sum_f P_f by a fixed-shape tree (deterministic for given P): parts -> one block.
__global__ void __launch_bounds__(kReduceBlock) k_reduce_parts(const double* __restrict__ P, long long nt,
                                                               double* __restrict__ parts) {
  __shared__ double s[3][kReduceBlock];
  const long long chunk = (nt + gridDim.x - 1) / gridDim.x;
  const long long b = (long long)blockIdx.x * chunk, e = min(nt, b + chunk);
  double acc[3] = {0, 0, 0};
  for (long long f = b + threadIdx.x; f < e; f += kReduceBlock)
    for (int a = 0; a < 3; ++a) acc[a] += P[3 * f + a];
  for (int a = 0; a < 3; ++a) s[a][threadIdx.x] = acc[a];
  __syncthreads();
  for (int st = kReduceBlock / 2; st > 0; st >>= 1) {
    if ((int)threadIdx.x < st)
      for (int a = 0; a < 3; ++a) s[a][threadIdx.x] += s[a][threadIdx.x + st];
    __syncthreads();
  }
  if (threadIdx.x < 3) parts[3 * blockIdx.x + threadIdx.x] = s[threadIdx.x][0];
}

__global__ void k_reduce_final(const double* __restrict__ parts, int nparts, const double* __restrict__ torque_acc,
                               double* __restrict__ force, double* __restrict__ torque) {
  const int a = threadIdx.x;
  if (a < 3) {
    double f = 0.0;
    for (int p = 0; p < nparts; ++p) f += parts[3 * p + a];
    force[a] = f;
    torque[a] = torque_acc[a];
  }
}

// ---- stand-alone steps for parity checks -----------------------------------------------------------
__global__ void k_seed_only(const RunConst rc, double* __restrict__ x, double* __restrict__ v,
                            int32_t* __restrict__ species) {
  const unsigned long long j = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x;
  if (j >= rc.count) return;
  const SeedState s = rc.control_volume == TPMC_CV_SPHERE ? seed_particle(rc, rc.first + j) : seed_particle_box(rc, rc.first + j);
  for (int k = 0; k < 3; ++k) { x[3 * j + k] = s.x[k]; v[3 * j + k] = s.v[k]; }
  if (species) species[j] = s.species;
}

// tpmc_trace: user rays -> queue records; candidates -> (facet, tau)
__global__ void k_pack_rays(const float* __restrict__ o, const float* __restrict__ d, const int32_t* __restrict__ f_prev,
                            unsigned int n, RayQueue q, int32_t* __restrict__ facet, double* __restrict__ tau) {
  const unsigned int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  q.o[r] = make_float4(o[3 * (size_t)r], o[3 * (size_t)r + 1], o[3 * (size_t)r + 2], __uint_as_float(r));
  q.v[r] = make_float4(d[3 * (size_t)r], d[3 * (size_t)r + 1], d[3 * (size_t)r + 2], 0.0f);
  q.f[r] = f_prev ? f_prev[r] : -1;
  facet[r] = -1;
  tau[r] = INFINITY;
}

__global__ void __launch_bounds__(kTraceBlock) k_resolve_only(const float4* __restrict__ nodes,
                                                              const float4* __restrict__ tris, const RayQueue q,
                                                              const unsigned int* __restrict__ hit_ray,
                                                              const int4* __restrict__ hit_cand,
                                                              const unsigned int* __restrict__ n_hits,
                                                              int32_t* __restrict__ facet, double* __restrict__ tau) {
  const unsigned int n = *n_hits;
  TraceCounters cnt;
  cnt.nodes = 0; cnt.tris = 0;
  unsigned int nt = 0;
  for (unsigned int h = blockIdx.x * blockDim.x + threadIdx.x; h < n; h += gridDim.x * blockDim.x) {
    const unsigned int r = hit_ray[h];
    if (r == kNoRay) continue;
    const int4 cand = hit_cand[h];
    const float4 ro = q.o[r], rv = q.v[r];
    const float of[3] = {ro.x, ro.y, ro.z}, df[3] = {rv.x, rv.y, rv.z};
    Hit hit;
    if (cand.w == TPMC_CAND_OVERFLOW) {
      int tmp[TPMC_STACK_SMEM];
      hit = closest_hit(nodes, tris, of, df, q.f[r], tmp, 1, cnt);
    } else {
      hit = resolve_candidates(tris, cand, of, df, nt);
    }
    facet[r] = hit.facet;
    tau[r] = hit.tau;
  }
}

// ---- a1: per-run constants on the host, fp64 -------------------------------------------------------
double host_Gt(double y) { return 0.25 * TPMC_SQRTPI * (1.0 + 2.0 * y * y) * erfc(-y) + 0.5 * y * exp(-y * y); }

// Gamma / (c n r^2), eq. (10); erf(S)/S by series below 1e-4 (A19)
double host_flux_bracket(double S) {
  const double pi = 3.14159265358979323846;
  const double erf_over_S = (S < 1e-4) ? (2.0 / TPMC_SQRTPI) * (1.0 - S * S / 3.0) : erf(S) / S;
  return TPMC_SQRTPI * exp(-S * S) + 0.5 * pi * erf_over_S + pi * S * erf(S);
}

// eq. (15) P:207-209 (A5): R zhat = ztilde = -V/|V|, Rodrigues about (zhat x ztilde)/|.|
void host_rotation(const double V[3], double R[9]) {
  const double sp = sqrt(V[0] * V[0] + V[1] * V[1] + V[2] * V[2]);
  double zt[3] = {0.0, 0.0, 1.0};
  if (sp > 0.0) { zt[0] = -V[0] / sp; zt[1] = -V[1] / sp; zt[2] = -V[2] / sp; }
  const double ax = -zt[1], ay = zt[0];
  const double sb = sqrt(ax * ax + ay * ay), cb = zt[2];
  for (int k = 0; k < 9; ++k) R[k] = 0.0;
  if (sb < 1e-12) {
    R[0] = 1.0;
    R[4] = R[8] = (cb > 0.0) ? 1.0 : -1.0;
    return;
  }
  const double ux = ax / sb, uy = ay / sb, uz = 0.0, omc = 1.0 - cb;
  R[0] = cb + ux * ux * omc;      R[1] = ux * uy * omc - uz * sb; R[2] = ux * uz * omc + uy * sb;
  R[3] = uy * ux * omc + uz * sb; R[4] = cb + uy * uy * omc;      R[5] = uy * uz * omc - ux * sb;
  R[6] = uz * ux * omc - uy * sb; R[7] = uz * uy * omc + ux * sb; R[8] = cb + uz * uz * omc;
}

int make_run_const(const tpmc_mesh* m, const tpmc_params* p, RunConst* rc) {
  if (!m || !p || !p->m || !p->x) return TPMC_EINVAL;
  if (p->n_species < 1 || p->n_species > TPMC_MAX_SPECIES) return TPMC_EINVAL;
  if (!(p->T_inf > 0.0) || !(p->T_W > 0.0) || !(p->n >= 0.0) || !isfinite(p->n)) return TPMC_EINVAL;
  if (!(p->accommodation >= 0.0 && p->accommodation <= 1.0)) return TPMC_EINVAL;
  if (!(p->cv_radius_factor >= 1.0) || !isfinite(p->cv_radius_factor)) return TPMC_EINVAL;
  if (p->N == 0 || p->first > p->N || p->count > p->N - p->first) return TPMC_EINVAL;
  if (p->max_bounces < 1 || p->max_bounces > TPMC_MAX_BOUNCES) return TPMC_EINVAL;
  if (!(p->energy_accommodation >= 0.0 && p->energy_accommodation <= 1.0)) return TPMC_EINVAL;
  if ((p->flags & TPMC_FLAG_ALIGN_OFF) && (p->flags & TPMC_FLAG_ALIGN_ON)) return TPMC_EINVAL;
  if (p->flags & ~0xFFu) return TPMC_EINVAL;
  if (p->wave_particles && (p->wave_particles < 256 || p->wave_particles > (1ull << 28))) return TPMC_EINVAL;
  if (p->chunk_particles > 0xF0000000ull) return TPMC_EINVAL;
  if (p->control_volume < TPMC_CV_SPHERE || p->control_volume > TPMC_CV_BOX_UNWEIGHTED) return TPMC_EINVAL;
  double xs = 0.0;
  for (int s = 0; s < p->n_species; ++s) {
    if (!(p->m[s] > 0.0) || !(p->x[s] >= 0.0)) return TPMC_EINVAL;
    xs += p->x[s];
  }
  if (fabs(xs - 1.0) > 1e-9) return TPMC_EINVAL;
  for (int a = 0; a < 3; ++a)
    if (!isfinite(p->V[a]) || !isfinite(p->x_ref[a])) return TPMC_EINVAL;
  memset(rc, 0, sizeof(*rc));
  const double speed = sqrt((p->V[0] * p->V[0] + p->V[1] * p->V[1]) + p->V[2] * p->V[2]);
  const double r = p->cv_radius_factor * m->Rb;
  rc->control_volume = p->control_volume;
  for (int a = 0; a < 3; ++a) {   // A24: the vertex AABB scaled about its centre, at least 0.05 R_b per axis
    const double h = std::max(0.5 * ((double)m->aabb_hi[a] - (double)m->aabb_lo[a]), 0.05 * m->Rb);
    rc->box_h[a] = p->cv_radius_factor * h;
    rc->V[a] = p->V[a];
  }
  double acc = 0.0;
  for (int s = 0; s < p->n_species; ++s) {
    SpeciesConst& sc = rc->sp[s];
    sc.m = p->m[s];
    sc.c = sqrt(2.0 * TPMC_KB * p->T_inf / p->m[s]);
    sc.S = speed / sc.c;
    sc.cW = sqrt(2.0 * TPMC_KB * p->T_W / p->m[s]);
    double flux = host_flux_bracket(sc.S) * sc.c * p->n * r * r;   // eq. (10)
    {
      double bacc = 0.0;
      for (int k = 0; k < 6; ++k) {
        const int a = k / 2, side = k % 2;
        const double area = 4.0 * rc->box_h[(a + 1) % 3] * rc->box_h[(a + 2) % 3];
        sc.bsn[k] = (side ? -p->V[a] : p->V[a]) / sc.c;
        bacc += area * (exp(-sc.bsn[k] * sc.bsn[k]) + TPMC_SQRTPI * sc.bsn[k] * erfc(-sc.bsn[k]));
        sc.bcum[k] = bacc;
      }
      if (p->control_volume != TPMC_CV_SPHERE) flux = bacc * p->n * sc.c / (2.0 * TPMC_SQRTPI);   // sum of the face fluxes
    }
    sc.w = p->m[s] * flux / (double)p->N;
    sc.g0 = host_Gt(-sc.S);
    sc.gI = host_Gt(sc.S) - sc.g0;
    acc += p->x[s];
    sc.cumx = acc;
  }
  rc->n_species = p->n_species;
  host_rotation(p->V, rc->R);
  for (int a = 0; a < 3; ++a) {
    rc->centre[a] = m->centre[a];
    rc->x_ref[a] = p->x_ref[a];
    rc->aabb_lo[a] = m->aabb_lo[a];
    rc->aabb_hi[a] = m->aabb_hi[a];
  }
  rc->r = r;
  for (int a = 0; a < 3; ++a) rc->key_c[a] = (float)m->centre[a];
  {
    const float rk = m->cull_nbox >= 0 ? m->cull_rin : (float)m->Rb;
    rc->key_r2 = rk * rk;
  }
  rc->sigma = p->accommodation;
  rc->T_W = p->T_W;
  rc->alpha_E = p->energy_accommodation;
  rc->surf_TW = m->surf_TW;
  rc->surf_sigma = m->surf_sigma;
  rc->simple_surface = (p->energy_accommodation == 1.0 && !m->surf_TW) ? 1 : 0;
  rc->first = p->first;
  rc->count = p->count;
  rc->seed_lo = (unsigned int)p->seed;
  rc->seed_hi = (unsigned int)(p->seed >> 32);
  rc->max_bounces = p->max_bounces;
  return TPMC_OK;
}

// fp32 image of the per-run constants for the pre-cull pass
void make_seed_const_f(const tpmc_mesh* m, const RunConst& rc, SeedConstF* sf) {
  memset(sf, 0, sizeof(*sf));
  sf->n_species = rc.n_species;
  for (int s = 0; s < rc.n_species; ++s) {
    SpeciesF& f = sf->sp[s];
    f.S = (float)rc.sp[s].S; f.c = (float)rc.sp[s].c; f.g0 = (float)rc.sp[s].g0; f.gI = (float)rc.sp[s].gI;
    // u01(w) = (w + 1/2) 2^-32 >= cumx  <=>  w >= cumx 2^32 - 1/2; all steps exact in fp64
    const double t = ceil(rc.sp[s].cumx * 4294967296.0 - 0.5);
    f.thr = t <= 0.0 ? 0ull : (t >= 4294967296.0 ? 4294967296ull : (unsigned long long)t);
  }
  const float mg = kPrecullMargin * (float)m->Rb;
  for (int k = 0; k < 9; ++k) sf->R[k] = (float)rc.R[k];
  for (int a = 0; a < 3; ++a) {
    sf->centre[a] = (float)rc.centre[a];
    sf->lo[a] = m->aabb_lo[a] - mg;
    sf->hi[a] = m->aabb_hi[a] + mg;
  }
  sf->r = (float)rc.r;
  const float Rg = (float)m->Rb * (1.0f + kPrecullMargin);
  sf->Rg2 = Rg * Rg;
  {
    const double sg = std::min(0.999999, (double)Rg / rc.r);   // sin(theta)
    sf->cot_g = (float)(sqrt(1.0 - sg * sg) / sg * (1.0 - 1e-6));
  }
  sf->n_box = m->cull_nbox;
  if (sf->n_box >= 0) {
    const float Ri = m->cull_rin + mg;
    sf->Rin2 = Ri * Ri;
    for (int j = 0; j < sf->n_box; ++j)
      for (int a = 0; a < 3; ++a) {
        sf->blo[j][a] = m->cull_box[j][a] - mg;
        sf->bhi[j][a] = m->cull_box[j][3 + a] + mg;
      }
  }
}

TraceTune trace_tune() { return TraceTune{TPMC_NODE_MIN, TPMC_REFILL_IDLE}; }

QuantGrid quant_grid(const tpmc_mesh* m) {   // the body-frame hierarchy
  QuantGrid g;
  for (int a = 0; a < 3; ++a) { g.origin[a] = m->q_origin[a]; g.inv_scale[a] = (float)(1.0 / (double)m->q_scale[a]); }
  for (int k = 0; k < 9; ++k) g.R[k] = (k % 4 == 0) ? 1.0f : 0.0f;
  g.rot_o = g.rot_c = 0.0f;
  return g;
}

constexpr size_t kDefaultWave = (size_t)1 << 26;   // particles per pipeline iteration (tpmc_params.wave_particles = 0)

int ensure_scratch(tpmc_mesh* m, size_t wave, bool need_facets) {
  if (!m->stats) {
    TPMC_CUDA_TRY(cudaMalloc((void**)&m->stats, ST_COUNT * sizeof(unsigned long long)));
    TPMC_CUDA_TRY(cudaMalloc((void**)&m->totals, 4 * sizeof(double)));
    TPMC_CUDA_TRY(cudaMalloc((void**)&m->ft_dev, 6 * sizeof(double)));
    TPMC_CUDA_TRY(cudaMalloc((void**)&m->partials, 3 * kReduceParts * sizeof(double)));
    TPMC_CUDA_TRY(cudaEventCreateWithFlags(&m->ev_fork, cudaEventDisableTiming));
    for (int pi = 0; pi < kPipes; ++pi) {
      Pipe& pp = m->pipe[pi];
      if (pi > 0) TPMC_CUDA_TRY(cudaStreamCreateWithFlags(&pp.main, cudaStreamNonBlocking));
      TPMC_CUDA_TRY(cudaStreamCreateWithFlags(&pp.seed, cudaStreamNonBlocking));
      TPMC_CUDA_TRY(cudaStreamCreateWithFlags(&pp.side, cudaStreamNonBlocking));
      for (int k = 0; k < 2; ++k) {
        TPMC_CUDA_TRY(cudaEventCreateWithFlags(&pp.ev_refl[k], cudaEventDisableTiming));
        TPMC_CUDA_TRY(cudaEventCreateWithFlags(&pp.ev_ovf[k], cudaEventDisableTiming));
      }
      for (int k = 0; k < 4; ++k) {
        TPMC_CUDA_TRY(cudaEventCreateWithFlags(&pp.ev_reset[k], cudaEventDisableTiming));
        TPMC_CUDA_TRY(cudaEventCreateWithFlags(&pp.ev_seeded[k], cudaEventDisableTiming));
      }
      TPMC_CUDA_TRY(cudaEventCreateWithFlags(&pp.ev_done, cudaEventDisableTiming));
      TPMC_CUDA_TRY(cudaEventCreate(&pp.ev_f0));
      TPMC_CUDA_TRY(cudaEventCreate(&pp.ev_f1));
      TPMC_CUDA_TRY(cudaMalloc((void**)&pp.ctr, kCtrWords * sizeof(unsigned int)));
      for (int k = 0; k < 2; ++k) TPMC_CUDA_TRY(cudaMalloc((void**)&pp.hist[k], kSortBins * sizeof(unsigned int)));
    }
  }
  if (m->wave_cap < wave) {
    for (int pi = 0; pi < kPipes; ++pi) {
      Pipe& pp = m->pipe[pi];
      for (int k = 0; k < 2; ++k) {
        cudaFree(pp.q_o[k]); cudaFree(pp.q_v[k]); cudaFree(pp.q_f[k]); cudaFree(pp.q_key[k]);
        pp.q_o[k] = pp.q_v[k] = nullptr; pp.q_f[k] = nullptr; pp.q_key[k] = nullptr;
      }
      cudaFree(pp.hit_ray); cudaFree(pp.hit_cand); cudaFree(pp.surv); cudaFree(pp.ovf); cudaFree(pp.order);
      pp.hit_ray = nullptr; pp.hit_cand = nullptr; pp.surv = nullptr; pp.ovf = nullptr; pp.order = nullptr;
    }
    m->wave_cap = 0;
    for (int pi = 0; pi < kPipes; ++pi) {
      Pipe& pp = m->pipe[pi];
      for (int k = 0; k < 2; ++k) {
        TPMC_CUDA_TRY(cudaMalloc((void**)&pp.q_o[k], 2 * wave * sizeof(float4)));   // regions A and B
        TPMC_CUDA_TRY(cudaMalloc((void**)&pp.q_v[k], 2 * wave * sizeof(float4)));
        TPMC_CUDA_TRY(cudaMalloc((void**)&pp.q_f[k], 2 * wave * sizeof(int)));
        TPMC_CUDA_TRY(cudaMalloc((void**)&pp.q_key[k], 2 * wave * sizeof(unsigned int)));
      }
      TPMC_CUDA_TRY(cudaMalloc((void**)&pp.order, 2 * wave * sizeof(unsigned int)));
      TPMC_CUDA_TRY(cudaMalloc((void**)&pp.hit_ray, (2 * wave + kHitSlack) * sizeof(unsigned int)));
      TPMC_CUDA_TRY(cudaMalloc((void**)&pp.hit_cand, (2 * wave + kHitSlack) * sizeof(int4)));
      TPMC_CUDA_TRY(cudaMalloc((void**)&pp.surv, 3 * wave * sizeof(unsigned int)));
      TPMC_CUDA_TRY(cudaMalloc((void**)&pp.ovf, 4 * wave * sizeof(unsigned int)));   // two lists (iteration parity)
    }
    m->wave_cap = wave;
  }
  if (need_facets && !m->facet_scratch)
    TPMC_CUDA_TRY(cudaMalloc((void**)&m->facet_scratch, 3 * sizeof(double) * (size_t)m->nt));
  return TPMC_OK;
}

struct Grids { int trace, reflect, finish, pipes, seed, precull, scatter; };
const Grids& grids() {
  static Grids g = {0, 0, 0, 0, 0, 0, 0};
  if (!g.trace) {
    int dev = 0, sms = 148, per = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    g.pipes = kPipes;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k_trace_wf, kTraceBlock, 0) != cudaSuccess || per < 1) per = 4;
    // resident trace CTAs per SM over all pipelines (measured: leaving room for the seed kernel does not pay)
    g.trace = sms * std::max(1, per / g.pipes);
    g.trace = std::min<int>(g.trace, (int)(kHitSlack / ((kTraceBlock / 32) * kHitBlock)));   // every warp may leave a hit-list block partly unused
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k_reflect, kTraceBlock, 0) != cudaSuccess || per < 1) per = 4;
    g.reflect = sms * std::max(1, per / g.pipes);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k_finish, kTraceBlock, 0) != cudaSuccess || per < 1) per = 4;
    g.finish = sms * per;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k_seed, kSeedBlock, 0) != cudaSuccess || per < 1) per = 4;
    g.seed = sms * per;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k_seed_precull, kPrecullBlock, 0) != cudaSuccess || per < 1) per = 4;
    g.precull = sms * per * 4;   // four shares per resident block (evens out the tail)
    g.scatter = sms * 8;
  }
  return g;
}

int fill_stats(tpmc_mesh* m, const tpmc_params* params, tpmc_stats* h_stats) {
  unsigned long long hs[ST_COUNT];
  TPMC_CUDA_TRY(cudaMemcpy(hs, m->stats, sizeof(hs), cudaMemcpyDeviceToHost));
  float ms = 0.0f;
  TPMC_CUDA_TRY(cudaEventElapsedTime(&ms, m->ev0, m->ev1));
  (void)params;
  memset(h_stats, 0, sizeof(*h_stats));
  h_stats->hits = hs[ST_HITS];
  h_stats->truncated = hs[ST_TRUNC];
  h_stats->tri_tests = hs[ST_TRIS];
  h_stats->node_visits = hs[ST_NODES];
  h_stats->ret_precull_a = hs[ST_RET_PA];
  h_stats->ret_precull_b = hs[ST_RET_PB];
  h_stats->ret_seed = hs[ST_RET_SEED];
  h_stats->ret_trace = hs[ST_RET_TRACE];
  h_stats->ret_resolve = hs[ST_RET_RESOLVE];
  h_stats->ret_horizon = hs[ST_RET_HORIZON];
  h_stats->ret_finish = hs[ST_RET_FINISH];
  h_stats->queued_primaries = hs[ST_Q_PRIM];
  h_stats->queued_reflected = hs[ST_Q_REFL];
  h_stats->overflow_rays = hs[ST_OVF_RETRACE] + hs[ST_OVF_PENDING] + hs[ST_DIVERTED];
  h_stats->final_stragglers = hs[ST_STRAGGLERS];
  h_stats->finish_segments = hs[ST_FIN_SEGS];
  h_stats->precull_uncertified = hs[ST_UNCERT];
  h_stats->traced_rays = hs[ST_TRACED];
  // sums of counted events (the identities of tpmc.h hold only if no particle was lost or duplicated on the way)
  h_stats->culled = hs[ST_RET_PA] + hs[ST_RET_PB] + hs[ST_RET_SEED];
  h_stats->escaped = h_stats->culled + hs[ST_RET_TRACE] + hs[ST_RET_RESOLVE] + hs[ST_RET_HORIZON] + hs[ST_RET_FINISH];
  // one segment per culled particle, per traced ray whose answer stood (a ray handed on after a candidate overflow is
  // searched again by the straggler kernel), per horizon escape and per search of the straggler kernel
  h_stats->segments = h_stats->culled + (hs[ST_TRACED] - hs[ST_OVF_RETRACE]) + hs[ST_RET_HORIZON] + hs[ST_FIN_SEGS];
  h_stats->kernel_launches = m->last_launches;
  h_stats->ms = ms;
  // Kernels of different streams overlap: these are sums of per-launch durations, not a partition of `ms`.
  for (int pi = 0; pi < kPipes; ++pi) {
    const Pipe& pp = m->pipe[pi];
    for (unsigned long long w = 0; w < pp.iters; ++w) {
      const cudaEvent_t* ev = pp.wave_ev + kEvPerWave * w;
      float t = 0.0f;
      if (w < pp.seed_iters) {
        TPMC_CUDA_TRY(cudaEventElapsedTime(&t, ev[0], ev[1]));
        h_stats->ms_seed += t;
      }
      TPMC_CUDA_TRY(cudaEventElapsedTime(&t, ev[2], ev[7]));
      h_stats->ms_sort += t;
      TPMC_CUDA_TRY(cudaEventElapsedTime(&t, ev[7], ev[3]));
      h_stats->ms_trace += t;
      TPMC_CUDA_TRY(cudaEventElapsedTime(&t, ev[3], ev[4]));
      h_stats->ms_reflect += t;
    }
    h_stats->timed_waves += pp.seed_iters;
    h_stats->trace_launches += pp.iters;
    if (pp.iters) {
      float t = 0.0f;
      TPMC_CUDA_TRY(cudaEventElapsedTime(&t, pp.ev_f0, pp.ev_f1));
      h_stats->ms_finish += t;
    }
  }
  return TPMC_OK;
}

// The flow-aligned refit pays for oblique attitudes only: bodies are usually modelled along their own axes (thin
// panels, flat faces), and a box refitted in a tilted frame is loose around such parts; with the stream within ~25 deg
// of a body axis the body-frame boxes are as good or better (measured on C5).  Both hierarchies give the same results.
bool want_alignment(const tpmc_params* p) {
  if (p->flags & TPMC_FLAG_ALIGN_OFF) return false;
  if (p->flags & TPMC_FLAG_ALIGN_ON) return true;
  const double vmax = std::max(std::fabs(p->V[0]), std::max(std::fabs(p->V[1]), std::fabs(p->V[2])));
  const double vabs = std::sqrt(p->V[0] * p->V[0] + p->V[1] * p->V[1] + p->V[2] * p->V[2]);
  return vabs > 0.0 && vmax < 0.9 * vabs;
}

int run_enqueue(tpmc_mesh* m, const tpmc_params* params, void* cuda_stream, double* d_force, double* d_torque,
                double* d_facet_momentum, tpmc_stats* h_stats, const tpmc_debug* debug);

}  // namespace

// The run itself is run_enqueue below.  A failure after its first enqueue (a CUDA error, a failed refit) would leave
// kernels queued on the handle's seed and side streams that nothing joins, with counters half-way: the next call on the
// handle -- the next attitude of a sweep -- would race with them.  So a failed run is drained here before its code is
// returned, and if even that fails (a sticky CUDA error) the handle is marked unusable instead of being trusted again.
extern "C" int tpmc_run(tpmc_mesh* m, const tpmc_params* params, void* cuda_stream, double* d_force,
                        double* d_torque, double* d_facet_momentum, tpmc_stats* h_stats, const tpmc_debug* debug) {
  if (!m || !params || !d_force || !d_torque) return TPMC_EINVAL;
  if (m->poisoned) {
    snprintf(g_tpmc_cuda_error, sizeof(g_tpmc_cuda_error),
             "tpmc_run: an earlier run on this mesh handle failed and could not be drained; destroy the handle");
    return TPMC_ECUDA;
  }
  const int rcode = run_enqueue(m, params, cuda_stream, d_force, d_torque, d_facet_momentum, h_stats, debug);
  if (rcode != TPMC_OK && m->in_run) {
    char first_error[sizeof(g_tpmc_cuda_error)];
    memcpy(first_error, g_tpmc_cuda_error, sizeof(first_error));   // the caller wants the error that failed the run
    bool drained = true;
    for (int pi = 0; pi < kPipes; ++pi) {
      Pipe& pp = m->pipe[pi];
      cudaStream_t ss[3] = {pp.seed, pp.side, pi > 0 ? pp.main : (cudaStream_t)cuda_stream};
      for (cudaStream_t s : ss)
        if (cudaStreamSynchronize(s) != cudaSuccess) drained = false;
    }
    cudaGetLastError();
    if (!drained) m->poisoned = true;
    memcpy(g_tpmc_cuda_error, first_error, sizeof(first_error));
  }
  m->in_run = false;
  return rcode;
}

namespace {
int run_enqueue(tpmc_mesh* m, const tpmc_params* params, void* cuda_stream, double* d_force, double* d_torque,
                double* d_facet_momentum, tpmc_stats* h_stats, const tpmc_debug* debug) {
  RunConst rc;
  int rcode = make_run_const(m, params, &rc);
  if (rcode != TPMC_OK) return rcode;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t wave_req = params->wave_particles ? (size_t)params->wave_particles : kDefaultWave;
  const size_t wave = std::min<unsigned long long>(std::max<unsigned long long>(params->count, 256), wave_req);
  rcode = ensure_scratch(m, wave, d_facet_momentum == nullptr);
  if (rcode != TPMC_OK) return rcode;
  const unsigned int cap = (unsigned int)wave;   // region size of the queues (<= the allocated m->wave_cap)
  double* P = d_facet_momentum ? d_facet_momentum : m->facet_scratch;
  tpmc_debug dbg0 = {nullptr, nullptr, nullptr};
  if (debug) dbg0 = *debug;
  const bool any_dbg = dbg0.hash || dbg0.bounces || dbg0.first_facet;
  const Grids& g = grids();
  const int K = g.pipes;
  const bool timed = (h_stats != nullptr);   // per-kernel events only when the caller will read them
  const bool precull = !(params->flags & TPMC_FLAG_NO_PRECULL) && params->control_volume == TPMC_CV_SPHERE;
  const bool use_horizon = !(params->flags & TPMC_FLAG_NO_HORIZON) && m->horizon != nullptr;   // (mesh built without: same results)
  const bool exact = (params->flags & TPMC_FLAG_EXACT_TRACE) != 0;
  const bool sorted = !exact && (params->flags & TPMC_FLAG_SORT_RAYS);
  const int aggregate = (m->nt <= kAggregateMaxFacets && !(params->flags & TPMC_FLAG_NO_AGGREGATION)) ? 1 : 0;
  // seed-time walk of the top of the hierarchy: pays only while the pre-cull pass has no two-level cull volume
  // (with it the pass is already tighter than the 64-node tree)
  const int seed_walk = m->cull_nbox < 0;
  SeedConstF sf;
  make_seed_const_f(m, rc, &sf);
  const QuantGrid qg = quant_grid(m);   // seed-time cull (body frame)
  m->in_run = true;   // from here on a failure leaves work enqueued: tpmc_run drains it
  TPMC_CUDA_TRY(cudaEventRecord(m->ev0, st));
  // the traversal's hierarchy: body frame, or refitted in the stream frame of this run (x' = R^T x: z' along the stream)
  const QuantGrid* qg_t = m->grid_dev;
  const uint4* wnodes_t = m->wnodes;
  if (!exact && want_alignment(params)) {
    double Rt[9];
    for (int a = 0; a < 3; ++a)
      for (int b2 = 0; b2 < 3; ++b2) Rt[3 * a + b2] = rc.R[3 * b2 + a];
    rcode = tpmc_mesh_align(m, Rt, st, &qg_t, &wnodes_t);
    if (rcode != TPMC_OK) return rcode;
  }
  m->pipe[0].main = st;
  for (int pi = 0; pi < kPipes; ++pi) {
    Pipe& pp = m->pipe[pi];
    pp.iters = pp.seed_iters = 0;
    if (timed && !pp.wave_ev) {
      pp.wave_ev = new (std::nothrow) cudaEvent_t[kEvPerWave * kMaxTimedWaves];
      if (!pp.wave_ev) return TPMC_ENOMEM;
      for (int i = 0; i < kEvPerWave * kMaxTimedWaves; ++i) TPMC_CUDA_TRY(cudaEventCreate(&pp.wave_ev[i]));
    }
  }

  TPMC_CUDA_TRY(cudaMemsetAsync(P, 0, 3 * sizeof(double) * (size_t)m->nt, st));
  TPMC_CUDA_TRY(cudaMemsetAsync(m->stats, 0, ST_COUNT * sizeof(unsigned long long), st));
  TPMC_CUDA_TRY(cudaMemsetAsync(m->totals, 0, 4 * sizeof(double), st));
  if (any_dbg && params->count)
    k_init_debug<<<(unsigned)((params->count + 255) / 256), 256, 0, st>>>(dbg0, params->count);
  unsigned long long launches = ((any_dbg && params->count) ? 1 : 0) + (wnodes_t != m->wnodes ? 4 : 0);   // + the refit kernels

  // Particle indices inside the queues are 32-bit offsets into a chunk of the slice.
  const unsigned long long kChunk = params->chunk_particles ? params->chunk_particles : 0xF0000000ull;
  for (unsigned long long c0 = 0; c0 < params->count; c0 += kChunk) {
    const unsigned long long cn = std::min<unsigned long long>(kChunk, params->count - c0);
    RunConst rcc = rc;
    rcc.first = rc.first + c0;
    rcc.count = cn;
    tpmc_debug dbg = dbg0;
    if (dbg.hash) dbg.hash += c0;
    if (dbg.bounces) dbg.bounces += c0;
    if (dbg.first_facet) dbg.first_facet += c0;
    // fork: the other pipelines' streams start after everything enqueued so far on the caller's stream
    TPMC_CUDA_TRY(cudaEventRecord(m->ev_fork, st));
    for (int pi = 0; pi < K; ++pi) {
      Pipe& pp = m->pipe[pi];
      if (pi > 0) TPMC_CUDA_TRY(cudaStreamWaitEvent(pp.main, m->ev_fork, 0));
      // a chunk starts from empty queues; the side streams of the previous chunk have been joined
      TPMC_CUDA_TRY(cudaMemsetAsync(pp.ctr, 0, kCtrWords * sizeof(unsigned int), pp.main));
      if (sorted)
        for (int k = 0; k < 2; ++k) TPMC_CUDA_TRY(cudaMemsetAsync(pp.hist[k], 0, kSortBins * sizeof(unsigned int), pp.main));
      TPMC_CUDA_TRY(cudaEventRecord(pp.ev_reset[0], pp.main));
    }
    // Waves are dealt round-robin to the pipelines.  In a pipeline, one iteration per wave: seed the wave
    // into region B of queue p (region A already holds the rays reflected in the previous iteration),
    // trace the whole queue, reflect the hits into region A of the other queue; particles that keep
    // bouncing ride along with the following waves.  The seed kernel of the pipeline's next wave runs on
    // its second stream beside trace/reflect: it only touches region B of the other queue and its counter,
    // which k_iter_begin has reset (ev_reset / ev_seeded order the two streams).
    const unsigned long long n_waves = (cn + wave - 1) / wave;
    for (unsigned long long wv = 0; wv < n_waves + (unsigned long long)K * kDrain; ++wv) {
      Pipe& pp = m->pipe[wv % K];
      const unsigned long long li = wv / K;            // iteration index within the pipeline
      const int p = (int)(li & 1);
      cudaStream_t s1 = pp.main, s2 = (params->flags & TPMC_FLAG_SERIAL_SEED) ? pp.main : pp.seed, s3 = pp.side;
      const int b = (int)(li & 1);
      unsigned int* ovf = pp.ovf + (size_t)b * 2 * m->wave_cap;
      RayQueue Q[2] = {{pp.q_o[0], pp.q_v[0], pp.q_f[0], pp.q_key[0], sorted ? pp.hist[0] : nullptr},
                       {pp.q_o[1], pp.q_v[1], pp.q_f[1], pp.q_key[1], sorted ? pp.hist[1] : nullptr}};
      const bool tw = timed && c0 == 0 && li < (unsigned long long)kMaxTimedWaves;
      cudaEvent_t* ev = tw ? pp.wave_ev + kEvPerWave * li : nullptr;
      if (wv < n_waves) {
        const unsigned int w0 = (unsigned int)(wv * wave);
        const unsigned int wn = (unsigned int)std::min<unsigned long long>(wave, cn - wv * wave);
        TPMC_CUDA_TRY(cudaStreamWaitEvent(s2, pp.ev_reset[li & 3], 0));
        // region B of this queue may still be read by the straggler kernel of iteration li - 2
        if (li >= 2) TPMC_CUDA_TRY(cudaStreamWaitEvent(s2, pp.ev_ovf[b], 0));
        if (tw) TPMC_CUDA_TRY(cudaEventRecord(ev[0], s2));
        const unsigned int gfull = (wn + kSeedBlock - 1) / kSeedBlock;
        if (precull) {
          TPMC_CUDA_TRY(cudaMemsetAsync(pp.ctr + 6, 0, 2 * sizeof(unsigned int), s2));
          k_seed_precull<<<std::min<unsigned int>((wn + kPrecullBlock - 1) / kPrecullBlock, (unsigned int)g.precull),
                           kPrecullBlock, 0, s2>>>(sf, rcc.seed_lo, rcc.seed_hi, rcc.first + w0, wn, cap, pp.surv, pp.ctr + 6,
                                                   m->stats);
          ++launches;
        }
        k_seed<<<std::min<unsigned int>(gfull, (unsigned int)g.seed), kSeedBlock, 0, s2>>>(
            rcc, w0, wn, precull ? pp.surv : nullptr, cap, pp.ctr + 6, m->cull_c, qg, seed_walk, Q[p], cap, pp.ctr + 2 * p + 1,
            m->stats);
        if (tw) TPMC_CUDA_TRY(cudaEventRecord(ev[1], s2));
        TPMC_CUDA_TRY(cudaEventRecord(pp.ev_seeded[li & 3], s2));
        if (tw) pp.seed_iters = li + 1;
        ++launches;
      }
      // (without a reflect step nothing else orders this iteration behind the straggler kernel that still reads list b)
      if (exact && li >= 2) TPMC_CUDA_TRY(cudaStreamWaitEvent(s1, pp.ev_ovf[b], 0));
      // the histogram of the OTHER queue (offsets of the previous iteration's sort by now) starts from zero: the seed
      // kernel of the next wave and this iteration's reflect step both count into it
      if (sorted && li >= 1) TPMC_CUDA_TRY(cudaMemsetAsync(pp.hist[p ^ 1], 0, kSortBins * sizeof(unsigned int), s1));
      k_iter_begin<<<1, 32, 0, s1>>>(pp.ctr, p ^ 1, b);
      TPMC_CUDA_TRY(cudaEventRecord(pp.ev_reset[(li + 1) & 3], s1));
      if (wv < n_waves) TPMC_CUDA_TRY(cudaStreamWaitEvent(s1, pp.ev_seeded[li & 3], 0));
      if (tw) TPMC_CUDA_TRY(cudaEventRecord(ev[2], s1));
      if (sorted) {   // counting sort of the queue by key (sort.cuh)
        k_sort_scan<<<1, kScanBlock, 0, s1>>>(pp.hist[p]);
        k_sort_scatter<<<g.scatter, 256, 0, s1>>>(pp.q_key[p], cap, pp.ctr + 2 * p, pp.hist[p], pp.order);
        launches += 2;
      }
      if (tw) TPMC_CUDA_TRY(cudaEventRecord(ev[7], s1));
      if (!exact) {
        k_trace_wf<<<g.trace, kTraceBlock, 0, s1>>>(wnodes_t, qg_t, m->tris, Q[p], sorted ? pp.order : nullptr, cap,
                                                    pp.ctr + 2 * p, pp.ctr + 4, pp.hit_ray,
                                                    pp.hit_cand, pp.ctr + 5, m->stats, trace_tune());
        if (tw) TPMC_CUDA_TRY(cudaEventRecord(ev[3], s1));
        // the straggler kernel of the previous iteration reads the queue this reflect step writes
        if (li >= 1) TPMC_CUDA_TRY(cudaStreamWaitEvent(s1, pp.ev_ovf[b ^ 1], 0));
        k_reflect<<<g.reflect, kTraceBlock, 0, s1>>>(rcc, cap, m->tris, Q[p], pp.hit_ray, pp.hit_cand, pp.ctr + 5, Q[p ^ 1],
                                                     pp.ctr + 2 * (p ^ 1), ovf, pp.ctr + 8 + b, P, m->totals, m->stats, dbg,
                                                     use_horizon ? m->horizon : nullptr, aggregate);
        launches += 2;
      } else {
        if (tw) TPMC_CUDA_TRY(cudaEventRecord(ev[3], s1));
        k_divert<<<296, 256, 0, s1>>>(cap, pp.ctr + 2 * p, ovf, pp.ctr + 8 + b, m->stats);
        ++launches;
      }
      if (tw) TPMC_CUDA_TRY(cudaEventRecord(ev[4], s1));
      // overflow list of this iteration: followed to escape on the side stream, beside the next traversal
      TPMC_CUDA_TRY(cudaEventRecord(pp.ev_refl[b], s1));
      TPMC_CUDA_TRY(cudaStreamWaitEvent(s3, pp.ev_refl[b], 0));
      if (tw) TPMC_CUDA_TRY(cudaEventRecord(ev[5], s3));
      k_finish<<<exact ? g.finish : g.finish / 4, kTraceBlock, 0, s3>>>(rcc, cap, m->nodes, m->tris, Q[p], ovf, pp.ctr + 8 + b, P,
                                                                        m->totals, m->stats, dbg, use_horizon ? m->horizon : nullptr);
      if (tw) TPMC_CUDA_TRY(cudaEventRecord(ev[6], s3));
      TPMC_CUDA_TRY(cudaEventRecord(pp.ev_ovf[b], s3));
      pp.last_iter = li;
      if (tw) pp.iters = li + 1;
      launches += 2;
    }
    // whatever still bounces after the drain iterations is followed to escape thread by thread; then join
    for (int pi = 0; pi < K; ++pi) {
      Pipe& pp = m->pipe[pi];
      const unsigned long long its = (n_waves + (unsigned long long)K * kDrain - pi + K - 1) / K;   // iterations it ran
      const int p = (int)(its & 1);
      RayQueue q = {pp.q_o[p], pp.q_v[p], pp.q_f[p], pp.q_key[p], nullptr};
      TPMC_CUDA_TRY(cudaStreamWaitEvent(pp.main, pp.ev_ovf[0], 0));   // join the side stream
      TPMC_CUDA_TRY(cudaStreamWaitEvent(pp.main, pp.ev_ovf[1], 0));
      if (timed) TPMC_CUDA_TRY(cudaEventRecord(pp.ev_f0, pp.main));
      k_finish<<<g.finish, kTraceBlock, 0, pp.main>>>(rcc, cap, m->nodes, m->tris, q, nullptr, pp.ctr + 2 * p, P, m->totals,
                                                     m->stats, dbg, use_horizon ? m->horizon : nullptr);
      if (timed) TPMC_CUDA_TRY(cudaEventRecord(pp.ev_f1, pp.main));
      ++launches;
      if (pi > 0) {
        TPMC_CUDA_TRY(cudaEventRecord(pp.ev_done, pp.main));
        TPMC_CUDA_TRY(cudaStreamWaitEvent(st, pp.ev_done, 0));
      }
    }
  }
  k_reduce_parts<<<kReduceParts, kReduceBlock, 0, st>>>(P, (long long)m->nt, m->partials);
  k_reduce_final<<<1, 32, 0, st>>>(m->partials, kReduceParts, m->totals, d_force, d_torque);
  launches += 2;
  m->last_launches = launches;
  TPMC_CUDA_TRY(cudaGetLastError());
  TPMC_CUDA_TRY(cudaEventRecord(m->ev1, st));
  if (h_stats) {
    TPMC_CUDA_TRY(cudaStreamSynchronize(st));
    return fill_stats(m, params, h_stats);
  }
  return TPMC_OK;
}
}  // namespace

// K attitudes of a sweep in one call: run k is `params` with V = h_V[k].  The handle's scratch, streams and events are
// shared by all of them; nothing is read back between attitudes unless statistics are asked for.
extern "C" int tpmc_run_sweep(tpmc_mesh* m, const tpmc_params* params, int32_t n_attitudes, const double* h_V,
                              void* cuda_stream, double* d_force, double* d_torque, double* d_facet_momentum,
                              tpmc_stats* h_stats) {
  if (!m || !params || !h_V || !d_force || !d_torque || n_attitudes < 0) return TPMC_EINVAL;
  for (int32_t k = 0; k < n_attitudes; ++k) {
    tpmc_params p = *params;
    for (int a = 0; a < 3; ++a) p.V[a] = h_V[3 * (size_t)k + a];
    const int rc = tpmc_run(m, &p, cuda_stream, d_force + 3 * (size_t)k, d_torque + 3 * (size_t)k,
                            d_facet_momentum ? d_facet_momentum + 3 * (size_t)m->nt * (size_t)k : nullptr,
                            h_stats ? h_stats + k : nullptr, nullptr);
    if (rc != TPMC_OK) return rc;
  }
  return TPMC_OK;
}

extern "C" int tpmc_run_host(tpmc_mesh* m, const tpmc_params* params, void* cuda_stream, double* h_force,
                             double* h_torque, double* h_facet_momentum, tpmc_stats* h_stats) {
  if (!m || !params || !h_force || !h_torque) return TPMC_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_scratch(m, std::max<size_t>(m->wave_cap, 256), h_facet_momentum != nullptr);   // allocates ft_dev, facet_scratch
  if (rc != TPMC_OK) return rc;
  tpmc_stats tmp_stats;
  rc = tpmc_run(m, params, cuda_stream, m->ft_dev, m->ft_dev + 3, h_facet_momentum ? m->facet_scratch : nullptr,
                h_stats ? &tmp_stats : nullptr, nullptr);
  if (rc != TPMC_OK) return rc;
  double ft[6];
  TPMC_CUDA_TRY(cudaMemcpyAsync(ft, m->ft_dev, sizeof(ft), cudaMemcpyDeviceToHost, st));
  if (h_facet_momentum)
    TPMC_CUDA_TRY(cudaMemcpyAsync(h_facet_momentum, m->facet_scratch, 3 * sizeof(double) * (size_t)m->nt,
                                  cudaMemcpyDeviceToHost, st));
  TPMC_CUDA_TRY(cudaStreamSynchronize(st));
  for (int a = 0; a < 3; ++a) { h_force[a] = ft[a]; h_torque[a] = ft[3 + a]; }
  if (h_stats) *h_stats = tmp_stats;
  return TPMC_OK;
}


extern "C" int tpmc_seed(const tpmc_mesh* mesh, const tpmc_params* params, void* cuda_stream, double* d_x, double* d_v,
                         int32_t* d_species) {
  if (!mesh || !params || !d_x || !d_v) return TPMC_EINVAL;
  RunConst rc;
  const int rcode = make_run_const(mesh, params, &rc);
  if (rcode != TPMC_OK) return rcode;
  if (params->count == 0) return TPMC_OK;
  k_seed_only<<<(unsigned)((params->count + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(rc, d_x, d_v, d_species);
  TPMC_CUDA_TRY(cudaGetLastError());
  return TPMC_OK;
}

extern "C" int tpmc_trace(tpmc_mesh* m, const float* d_o, const float* d_d, const int32_t* d_f_prev, int64_t n,
                          const double* h_align_V, void* cuda_stream, int32_t* d_facet, double* d_tau) {
  if (!m || !d_o || !d_d || !d_facet || !d_tau || n < 0 || n > 0x7FFFFFFF) return TPMC_EINVAL;
  if (n == 0) return TPMC_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rcode = ensure_scratch(m, std::max<size_t>(((size_t)n + 1) / 2, std::max<size_t>(m->wave_cap, 256)), false);
  if (rcode != TPMC_OK) return rcode;
  const Grids& g = grids();
  Pipe& pp = m->pipe[0];
  RayQueue q = {pp.q_o[0], pp.q_v[0], pp.q_f[0], pp.q_key[0], nullptr};
  const unsigned int un = (unsigned int)n;
  const QuantGrid* qg_t = m->grid_dev;
  const uint4* wnodes_t = m->wnodes;
  if (h_align_V) {   // the hierarchy refitted in the stream frame of this velocity, as tpmc_run uses it
    double R[9], Rt[9];
    host_rotation(h_align_V, R);
    for (int a = 0; a < 3; ++a)
      for (int b2 = 0; b2 < 3; ++b2) Rt[3 * a + b2] = R[3 * b2 + a];
    rcode = tpmc_mesh_align(m, Rt, st, &qg_t, &wnodes_t);
    if (rcode != TPMC_OK) return rcode;
  }
  TPMC_CUDA_TRY(cudaMemsetAsync(pp.ctr, 0, kCtrWords * sizeof(unsigned int), st));
  TPMC_CUDA_TRY(cudaMemcpyAsync(pp.ctr, &un, sizeof(un), cudaMemcpyHostToDevice, st));   // region A holds the rays
  TPMC_CUDA_TRY(cudaMemsetAsync(m->stats, 0, ST_COUNT * sizeof(unsigned long long), st));
  k_pack_rays<<<(un + 255) / 256, 256, 0, st>>>(d_o, d_d, d_f_prev, un, q, d_facet, d_tau);
  // the production traversal (fp32 wavefront + candidate lists), then the exact fp64 resolve
  k_trace_wf<<<g.trace, kTraceBlock, 0, st>>>(wnodes_t, qg_t, m->tris, q, nullptr, (unsigned int)(2 * m->wave_cap), pp.ctr, pp.ctr + 4,
                                              pp.hit_ray, pp.hit_cand, pp.ctr + 5, m->stats, trace_tune());
  k_resolve_only<<<g.reflect, kTraceBlock, 0, st>>>(m->nodes, m->tris, q, pp.hit_ray, pp.hit_cand, pp.ctr + 5, d_facet,
                                                    d_tau);
  TPMC_CUDA_TRY(cudaGetLastError());
  TPMC_CUDA_TRY(cudaStreamSynchronize(st));   // &un must outlive the copy
  return TPMC_OK;
}
