// lbvh.cu -- tpmc_mesh_*: triangulation ingest and on-device LBVH build (step a0 of DESIGN.md).
//
// "Satellite surfaces are represented by a triangulation, allowing the use of well-known
// ray-tracing methods"; the paper names no acceleration structure.  Here: 63-bit Morton
// codes of facet centroids -> radix sort (radix.cuh) -> Karras (2012) binary radix tree -> bottom-up refit.
// Everything runs on the device; there is no host build path.
#include <algorithm>
#include <cstdlib>

#include "common.cuh"
#include "radix.cuh"

thread_local char g_tpmc_cuda_error[512] = "";

namespace {

constexpr int kBlock = 256;

// ---- vertex AABB (fp32 min/max are exact) and bounding radius about its centre (O1, A10) ----
__global__ void k_vertex_aabb(const float* __restrict__ v, int64_t nv, float* __restrict__ out) {
  __shared__ float s[6][1024];
  float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int64_t i = threadIdx.x; i < nv; i += blockDim.x)
    for (int a = 0; a < 3; ++a) {
      const float p = v[3 * i + a];
      lo[a] = fminf(lo[a], p);
      hi[a] = fmaxf(hi[a], p);
    }
  for (int a = 0; a < 3; ++a) { s[a][threadIdx.x] = lo[a]; s[3 + a][threadIdx.x] = hi[a]; }
  __syncthreads();
  for (int st = blockDim.x / 2; st > 0; st >>= 1) {
    if ((int)threadIdx.x < st)
      for (int a = 0; a < 3; ++a) {
        s[a][threadIdx.x] = fminf(s[a][threadIdx.x], s[a][threadIdx.x + st]);
        s[3 + a][threadIdx.x] = fmaxf(s[3 + a][threadIdx.x], s[3 + a][threadIdx.x + st]);
      }
    __syncthreads();
  }
  if (threadIdx.x < 6) out[threadIdx.x] = s[threadIdx.x][0];
}

__global__ void k_vertex_r2(const float* __restrict__ v, int64_t nv, double cx, double cy, double cz,
                            double* __restrict__ out) {
  __shared__ double s[1024];
  double r2 = 0.0;
  for (int64_t i = threadIdx.x; i < nv; i += blockDim.x) {
    const double dx = __dsub_rn((double)v[3 * i], cx), dy = __dsub_rn((double)v[3 * i + 1], cy),
                 dz = __dsub_rn((double)v[3 * i + 2], cz);
    // (dx*dx + dy*dy) + dz*dz without contraction: the bounding radius is a definition (O1)
    const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    r2 = fmax(r2, d2);
  }
  s[threadIdx.x] = r2;
  __syncthreads();
  for (int st = blockDim.x / 2; st > 0; st >>= 1) {
    if ((int)threadIdx.x < st) s[threadIdx.x] = fmax(s[threadIdx.x], s[threadIdx.x + st]);
    __syncthreads();
  }
  if (threadIdx.x == 0) out[0] = s[0];
}

__global__ void k_check_indices(const int32_t* __restrict__ idx, int64_t n3, int64_t nv, int* __restrict__ bad) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n3 && (idx[i] < 0 || idx[i] >= nv)) atomicExch(bad, 1);
}

// ---- Morton codes ----
__device__ __forceinline__ uint64_t spread21(uint64_t x) {  // 21 bits -> every third bit
  x &= 0x1FFFFFull;
  x = (x | (x << 32)) & 0x1F00000000FFFFull;
  x = (x | (x << 16)) & 0x1F0000FF0000FFull;
  x = (x | (x << 8)) & 0x100F00F00F00F00Full;
  x = (x | (x << 4)) & 0x10C30C30C30C30C3ull;
  x = (x | (x << 2)) & 0x1249249249249249ull;
  return x;
}

__global__ void k_morton(const float* __restrict__ v, const int32_t* __restrict__ idx, int64_t nt, float3 lo,
                         float3 inv_ext, uint64_t* __restrict__ keys, int32_t* __restrict__ ids) {
  const int64_t f = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (f >= nt) return;
  const int32_t i0 = idx[3 * f], i1 = idx[3 * f + 1], i2 = idx[3 * f + 2];
  const float cx = (v[3 * i0] + v[3 * i1] + v[3 * i2]) * (1.0f / 3.0f);
  const float cy = (v[3 * i0 + 1] + v[3 * i1 + 1] + v[3 * i2 + 1]) * (1.0f / 3.0f);
  const float cz = (v[3 * i0 + 2] + v[3 * i1 + 2] + v[3 * i2 + 2]) * (1.0f / 3.0f);
  const float s = 2097152.0f;  // 2^21
  const uint64_t qx = (uint64_t)fminf(fmaxf((cx - lo.x) * inv_ext.x * s, 0.0f), s - 1.0f);
  const uint64_t qy = (uint64_t)fminf(fmaxf((cy - lo.y) * inv_ext.y * s, 0.0f), s - 1.0f);
  const uint64_t qz = (uint64_t)fminf(fmaxf((cz - lo.z) * inv_ext.z * s, 0.0f), s - 1.0f);
  keys[f] = (spread21(qx) << 2) | (spread21(qy) << 1) | spread21(qz);
  ids[f] = (int32_t)f;
}

// ---- sorted triangle records + leaf boxes ----
__global__ void k_gather(const float* __restrict__ v, const int32_t* __restrict__ idx,
                         const uint8_t* __restrict__ flags, const int32_t* __restrict__ sorted_ids, int64_t nt,
                         float4* __restrict__ tris, float* __restrict__ box /* [(n_int + nt)][6] */, int64_t n_int) {
  const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (s >= nt) return;
  const int32_t f = sorted_ids[s];
  float p[3][3];
  for (int k = 0; k < 3; ++k) {
    const int32_t vi = idx[3 * (int64_t)f + k];
    for (int a = 0; a < 3; ++a) p[k][a] = v[3 * (int64_t)vi + a];
  }
  const uint32_t fl = flags ? (uint32_t)flags[f] : 0u;
  tris[3 * s + 0] = make_float4(p[0][0], p[0][1], p[0][2], __int_as_float(f));
  tris[3 * s + 1] = make_float4(p[1][0], p[1][1], p[1][2], __uint_as_float(fl));
  tris[3 * s + 2] = make_float4(p[2][0], p[2][1], p[2][2], 0.0f);
  float* b = box + 6 * (n_int + s);
  for (int a = 0; a < 3; ++a) {
    b[a] = fminf(p[0][a], fminf(p[1][a], p[2][a]));      // exact: corners are fp32
    b[3 + a] = fmaxf(p[0][a], fmaxf(p[1][a], p[2][a]));
  }
}

// ---- Karras 2012: one thread per internal node ----
__device__ __forceinline__ int delta(const uint64_t* __restrict__ k, int n, int i, int j) {
  if (j < 0 || j >= n) return -1;
  const uint64_t a = k[i], b = k[j];
  if (a == b) return 64 + __clz(i ^ j);   // duplicate codes: fall back to the position
  return __clzll((long long)(a ^ b));
}

__global__ void k_hierarchy(const uint64_t* __restrict__ keys, int n, int2* __restrict__ children,
                            int* __restrict__ parent /* [n-1 internal | n leaves] */, int* __restrict__ nsize /* [n-1] leaves below, or null */) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n - 1) return;
  const int d = (delta(keys, n, i, i + 1) - delta(keys, n, i, i - 1)) >= 0 ? 1 : -1;
  const int dmin = delta(keys, n, i, i - d);
  int lmax = 2;
  while (delta(keys, n, i, i + lmax * d) > dmin) lmax <<= 1;
  int l = 0;
  for (int t = lmax >> 1; t >= 1; t >>= 1)
    if (delta(keys, n, i, i + (l + t) * d) > dmin) l += t;
  const int j = i + l * d;
  const int dnode = delta(keys, n, i, j);
  int s = 0, t = l;
  do {
    t = (t + 1) >> 1;
    if (delta(keys, n, i, i + (s + t) * d) > dnode) s += t;
  } while (t > 1);
  const int gamma = i + s * d + min(d, 0);
  const int lo = min(i, j), hi = max(i, j);
  const int left = (lo == gamma) ? ~gamma : gamma;              // ~x = leaf holding sorted triangle x
  const int right = (hi == gamma + 1) ? ~(gamma + 1) : gamma + 1;
  children[i] = make_int2(left, right);
  if (nsize) nsize[i] = hi - lo + 1;
  parent[left >= 0 ? left : (n - 1) + ~left] = i;
  parent[right >= 0 ? right : (n - 1) + ~right] = i;
  if (i == 0) parent[0] = -1;
}

// ---- bottom-up refit: the second thread to arrive at a node owns it ----
__global__ void k_refit(int n, const int2* __restrict__ children, const int* __restrict__ parent,
                        float* __restrict__ box, int* __restrict__ arrive, float4* __restrict__ nodes) {
  const int leaf = blockIdx.x * blockDim.x + threadIdx.x;
  if (leaf >= n) return;
  int cur = parent[(n - 1) + leaf];
  while (cur >= 0) {
    __threadfence();
    if (atomicAdd(&arrive[cur], 1) == 0) return;
    const int2 ch = children[cur];
    const volatile float* b0 = box + 6 * (size_t)(ch.x >= 0 ? ch.x : (n - 1) + ~ch.x);
    const volatile float* b1 = box + 6 * (size_t)(ch.y >= 0 ? ch.y : (n - 1) + ~ch.y);
    float l0[3], h0[3], l1[3], h1[3];
    for (int a = 0; a < 3; ++a) { l0[a] = b0[a]; h0[a] = b0[3 + a]; l1[a] = b1[a]; h1[a] = b1[3 + a]; }
    float* b = box + 6 * (size_t)cur;
    for (int a = 0; a < 3; ++a) { b[a] = fminf(l0[a], l1[a]); b[3 + a] = fmaxf(h0[a], h1[a]); }
    if (nodes) {   // (the per-run refit in the stream frame only needs the boxes)
      nodes[4 * (size_t)cur + 0] = make_float4(l0[0], l0[1], l0[2], h0[0]);
      nodes[4 * (size_t)cur + 1] = make_float4(h0[1], h0[2], l1[0], l1[1]);
      nodes[4 * (size_t)cur + 2] = make_float4(l1[2], h1[0], h1[1], h1[2]);
      nodes[4 * (size_t)cur + 3] = make_float4(__int_as_float(ch.x), __int_as_float(ch.y), 0.0f, 0.0f);
    }
    cur = parent[cur];
  }
}

// single-triangle mesh: one node whose second child is an empty box
__global__ void k_single(const float* __restrict__ box_leaf, float4* __restrict__ nodes) {
  const float big = 3.0e38f;
  nodes[0] = make_float4(box_leaf[0], box_leaf[1], box_leaf[2], box_leaf[3]);
  nodes[1] = make_float4(box_leaf[4], box_leaf[5], big, big);
  nodes[2] = make_float4(big, -big, -big, -big);
  nodes[3] = make_float4(__int_as_float(~0), __int_as_float(~0), 0.0f, 0.0f);
}

// Compact copy of the hierarchy for the wavefront traversal: 32 B per node = one 256-bit load.
//   words 0-2: child 0 box, words 3-5: child 1 box, one word per axis: lo | hi << 16 as unsigned 16-bit grid
//   coordinates (so that one byte permute yields the near or the far plane of an axis, see trace.cuh);
//   words 6-7: the two child refs.
// Grid: x = origin + q * scale per axis.  lo is rounded down and hi up: the decoded box contains the fp32 box.
// (The quotient is evaluated in fp64: a box corner within 1e-11 steps of a grid plane may land on the wrong
// side of it, which the slack of the traversal's margin G covers.  The clamps below never act on a box of the
// hierarchy: quant_step keeps every plane inside steps 0 .. 65535.)
__global__ void k_compact_nodes(const float4* __restrict__ nodes, int64_t n_nodes, double ox, double oy, double oz,
                                double sx, double sy, double sz, uint4* __restrict__ cnodes,
                                const double* __restrict__ dev_grid = nullptr) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n_nodes) return;
  if (dev_grid) { ox = dev_grid[0]; oy = dev_grid[1]; oz = dev_grid[2]; sx = dev_grid[3]; sy = dev_grid[4]; sz = dev_grid[5]; }
  const float4 n0 = nodes[4 * i], n1 = nodes[4 * i + 1], n2 = nodes[4 * i + 2], n3 = nodes[4 * i + 3];
  const float lo[2][3] = {{n0.x, n0.y, n0.z}, {n1.z, n1.w, n2.x}};
  const float hi[2][3] = {{n0.w, n1.x, n1.y}, {n2.y, n2.z, n2.w}};
  const double o[3] = {ox, oy, oz}, sc[3] = {sx, sy, sz};
  unsigned int w[6];
  for (int c = 0; c < 2; ++c)
    for (int a = 0; a < 3; ++a) {
      unsigned int ql = 65535u, qh = 0u;   // empty box (single-triangle mesh): near plane beyond the far plane
      if (lo[c][a] <= hi[c][a]) {
        const double l = floor(((double)lo[c][a] - o[a]) / sc[a]), h = ceil(((double)hi[c][a] - o[a]) / sc[a]);
        ql = (unsigned int)fmin(fmax(l, 0.0), 65535.0);
        qh = (unsigned int)fmin(fmax(h, 0.0), 65535.0);
      }
      w[3 * c + a] = ql | (qh << 16);
    }
  cnodes[2 * i] = make_uint4(w[0], w[1], w[2], w[3]);
  cnodes[2 * i + 1] = make_uint4(w[4], w[5], __float_as_uint(n3.x), __float_as_uint(n3.y));
}

// Top of the tree, breadth-first, cut at a node budget: child refs >= 0 index this array, -1 marks a
// subtree (or triangle) that was cut off.  A ray that touches no cut-off box cannot hit the mesh.
// Nodes in the compact 32-byte format of k_compact_nodes (what the seed kernel walks).
__global__ void k_build_cull(const float4* __restrict__ nodes, const uint4* __restrict__ cnodes,
                             uint4* __restrict__ cull_c, int* __restrict__ queue, int budget, int* __restrict__ out_count) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  int tail = 1;
  queue[0] = 0;
  for (int head = 0; head < tail; ++head) {
    const float4* np = nodes + 4 * (size_t)queue[head];
    const float4 n3 = np[3];
    int ref[2] = {__float_as_int(n3.x), __float_as_int(n3.y)};
    for (int k = 0; k < 2; ++k) {
      if (ref[k] >= 0 && tail < budget) { queue[tail] = ref[k]; ref[k] = tail++; }
      else ref[k] = -1;
    }
    const uint4 ca = cnodes[2 * (size_t)queue[head]], cb = cnodes[2 * (size_t)queue[head] + 1];
    cull_c[2 * head] = ca;
    cull_c[2 * head + 1] = make_uint4(cb.x, cb.y, (unsigned int)ref[0], (unsigned int)ref[1]);
  }
  *out_count = tail;
}

// ---- wide (4-ary) hierarchy for the wavefront traversal --------------------------------------------------------
// The binary radix tree is collapsed breadth-first: a wide node starts from the two children of a binary node and
// replaces, up to twice, its internal child with the largest box surface by that child's two children (greedy by
// area; a child whose subtree holds <= 4 facets is opened only if it fits into this node's free slots entirely, so small
// subtrees become full nodes instead of fragments of two; TPMC_WIDE_GREEDY=0 opens the two original children instead:
// every second level of the binary tree).  A ray
// then fetches one 64-byte node where it fetched two or three 32-byte nodes one after the other: the chain of
// dependent loads per ray, which bounds the traversal kernel, gets about half as long.  Topology only (which binary
// nodes/leaves are the children of each wide node, and the breadth-first numbering); the boxes are filled in per
// frame by k_compact_wide from the per-node boxes of the refit.  Numbering is deterministic: per level an expand
// pass, a one-block exclusive scan of the internal-child counts, and an assign pass.
#ifndef TPMC_WIDE_GREEDY
#define TPMC_WIDE_GREEDY 2   // 2: by area, small subtrees kept whole (13 % fewer nodes than 1, same steps per ray); 0: every second level
#endif
constexpr int kWideLevels = 100;   // >= depth of a Karras tree over 63-bit keys with a 30-bit index tie-break
__device__ __forceinline__ float box_half_area(const float* __restrict__ b) {
  const float ex = b[3] - b[0], ey = b[4] - b[1], ez = b[5] - b[2];
  return ex * ey + ey * ez + ez * ex;
}
// lvl[0], lvl[1]: wide nodes [begin, end) of the current level; lvl[2]: internal children found on it
__global__ void k_wide_expand(const int2* __restrict__ kids, const float* __restrict__ box, const int* __restrict__ nsize,
                              const int* __restrict__ lvl, const int* __restrict__ wroot, int4* __restrict__ wkids_bin,
                              unsigned int* __restrict__ cnt) {
  const int begin = lvl[0], end = lvl[1];
  for (int w = begin + blockIdx.x * blockDim.x + threadIdx.x; w < end; w += gridDim.x * blockDim.x) {
    const int2 k0 = kids[wroot[w]];
    int c[4] = {k0.x, k0.y, TPMC_WIDE_EMPTY, TPMC_WIDE_EMPTY};
    int nc = 2;
#if TPMC_WIDE_GREEDY
    for (int round = 0; round < 2; ++round) {
      int best = -1;
      float ba = -1.0f;
      for (int j = 0; j < nc; ++j)
        if (c[j] >= 0) {
#if TPMC_WIDE_GREEDY == 2
          // open a child only if its subtree does not fit one wide node anyway (> 4 facets) or fits into the free slots
          // of this one entirely: small subtrees stay whole and become full nodes instead of fragments of 2
          const int sz = nsize[c[j]];
          if (!(sz > 4 || sz <= (4 - nc) + 1)) continue;
#endif
          const float a = box_half_area(box + 6 * (size_t)c[j]);
          if (a > ba) { ba = a; best = j; }
        }
      if (best < 0) break;
      const int2 kk = kids[c[best]];
      for (int j = nc; j > best + 1; --j) c[j] = c[j - 1];   // keep the children in Morton order
      c[best] = kk.x;
      c[best + 1] = kk.y;
      ++nc;
    }
#else
    if (k0.y >= 0) { const int2 kk = kids[k0.y]; c[1] = kk.x; c[2] = kk.y; nc = 3; }
    if (k0.x >= 0) { const int2 kk = kids[k0.x]; for (int j = nc; j > 1; --j) c[j] = c[j - 1]; c[0] = kk.x; c[1] = kk.y; ++nc; }
#endif
    unsigned int ni = 0u;
    for (int j = 0; j < 4; ++j) ni += (c[j] >= 0 && c[j] != TPMC_WIDE_EMPTY) ? 1u : 0u;
    wkids_bin[w] = make_int4(c[0], c[1], c[2], c[3]);
    cnt[w] = ni;
  }
}
// exclusive scan of cnt[begin, end) in place by one block; lvl[2] = total
__global__ void __launch_bounds__(1024) k_wide_scan(unsigned int* __restrict__ cnt, int* __restrict__ lvl) {
  __shared__ unsigned int wsum[32];
  __shared__ unsigned int carry;
  const int begin = lvl[0], end = lvl[1];
  if (threadIdx.x == 0) carry = 0u;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int c0 = begin; c0 < end; c0 += 1024) {
    const int i = c0 + threadIdx.x;
    const unsigned int v = i < end ? cnt[i] : 0u;
    unsigned int inc = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const unsigned int t = __shfl_up_sync(0xFFFFFFFFu, inc, off);
      if (lane >= off) inc += t;
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      unsigned int x = wsum[lane];
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const unsigned int t = __shfl_up_sync(0xFFFFFFFFu, x, off);
        if (lane >= off) x += t;
      }
      wsum[lane] = x;
    }
    __syncthreads();
    const unsigned int before = carry + (wid ? wsum[wid - 1] : 0u);
    if (i < end) cnt[i] = before + inc - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry = before + inc;
    __syncthreads();
  }
  if (threadIdx.x == 0) lvl[2] = (int)carry;
}
__global__ void k_wide_assign(const int* __restrict__ lvl, const int4* __restrict__ wkids_bin, const unsigned int* __restrict__ off,
                              int* __restrict__ wroot, int4* __restrict__ wkids) {
  const int begin = lvl[0], end = lvl[1];
  for (int w = begin + blockIdx.x * blockDim.x + threadIdx.x; w < end; w += gridDim.x * blockDim.x) {
    const int4 kb = wkids_bin[w];
    const int c[4] = {kb.x, kb.y, kb.z, kb.w};
    int r[4];
    int next = end + (int)off[w];
    for (int j = 0; j < 4; ++j) {
      r[j] = c[j];                                    // leaf (< 0) or empty: unchanged
      if (c[j] >= 0 && c[j] != TPMC_WIDE_EMPTY) { wroot[next] = c[j]; r[j] = next++; }
    }
    wkids[w] = make_int4(r[0], r[1], r[2], r[3]);
  }
}
__global__ void k_wide_next(int* __restrict__ lvl) {
  if (blockIdx.x == 0 && threadIdx.x == 0) { lvl[0] = lvl[1]; lvl[1] += lvl[2]; lvl[2] = 0; }
}
__global__ void k_wide_init(int* __restrict__ lvl, int* __restrict__ wroot, int4* __restrict__ wkids_bin, int4* __restrict__ wkids, int single) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  if (single) {   // one triangle: one wide node holding the leaf
    wkids_bin[0] = make_int4(~0, TPMC_WIDE_EMPTY, TPMC_WIDE_EMPTY, TPMC_WIDE_EMPTY);
    wkids[0] = wkids_bin[0];
    lvl[0] = 1; lvl[1] = 1; lvl[2] = 0;
  } else {
    wroot[0] = 0;
    lvl[0] = 0; lvl[1] = 1; lvl[2] = 0;
  }
}

// Boxes of the wide nodes in one frame: 64 B per node = two 256-bit loads.
//   words 3k .. 3k+2: box of child k (x, y, z), one word per axis: lo | hi << 16 as unsigned 16-bit grid coordinates
//   (one byte permute yields the near or the far plane of an axis, see trace.cuh); words 12-15: the four child refs
//   (>= 0: wide node, < 0: leaf holding sorted triangle ~ref).  An empty slot has the box lo = 65535, hi = 0 on every
//   axis, which no ray enters (near plane 65535 steps beyond the far plane), and repeats the ref of child 0, so that
//   even a margin of absurd size (a ray far outside along a flat axis) would only repeat work, never read a bad ref.
// Grid: x = origin + q * scale per axis.  lo is rounded down and hi up: the decoded box contains the fp32 box.
// (The quotient is evaluated in fp64: a box corner within 1e-11 steps of a grid plane may land on the wrong side of it,
// which the slack of the traversal's margin G covers.  The clamps never act: quant_step keeps every plane inside
// steps 0 .. 65535.)  box: [(n_int + nt)][6], the per-node boxes of the refit in this frame.
__global__ void k_compact_wide(const float* __restrict__ box, int64_t n_int, const int4* __restrict__ wkids_bin,
                               const int4* __restrict__ wkids, int64_t n_wide, double ox, double oy, double oz, double sx,
                               double sy, double sz, uint4* __restrict__ wnodes, const double* __restrict__ dev_grid = nullptr) {
  const int64_t w = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (w >= n_wide) return;
  if (dev_grid) { ox = dev_grid[0]; oy = dev_grid[1]; oz = dev_grid[2]; sx = dev_grid[3]; sy = dev_grid[4]; sz = dev_grid[5]; }
  const double o[3] = {ox, oy, oz}, sc[3] = {sx, sy, sz};
  const int4 kb = wkids_bin[w], kw = wkids[w];
  const int cb[4] = {kb.x, kb.y, kb.z, kb.w};
  unsigned int ref[4] = {(unsigned int)kw.x, (unsigned int)kw.y, (unsigned int)kw.z, (unsigned int)kw.w};
  unsigned int q[12];
  for (int k = 0; k < 4; ++k) {
    if (cb[k] == TPMC_WIDE_EMPTY) {
      q[3 * k] = q[3 * k + 1] = q[3 * k + 2] = 0x0000FFFFu;
      ref[k] = ref[0];
      continue;
    }
    const float* b = box + 6 * (size_t)(cb[k] >= 0 ? (int64_t)cb[k] : n_int + (int64_t)~cb[k]);
    for (int a = 0; a < 3; ++a) {
      const double l = floor(((double)b[a] - o[a]) / sc[a]), h = ceil(((double)b[3 + a] - o[a]) / sc[a]);
      const unsigned int ql = (unsigned int)fmin(fmax(l, 0.0), 65535.0), qh = (unsigned int)fmin(fmax(h, 0.0), 65535.0);
      q[3 * k + a] = ql | (qh << 16);
    }
  }
  wnodes[4 * w + 0] = make_uint4(q[0], q[1], q[2], q[3]);
  wnodes[4 * w + 1] = make_uint4(q[4], q[5], q[6], q[7]);
  wnodes[4 * w + 2] = make_uint4(q[8], q[9], q[10], q[11]);
  wnodes[4 * w + 3] = make_uint4(ref[0], ref[1], ref[2], ref[3]);
}

// ---- flow-aligned compact hierarchy (per run) ------------------------------------------------------------------
// An axis-aligned box shows its smallest face to a ray that runs along one of its axes and up to sqrt(3) times
// that area to a diagonal one, and nearly all primaries of a run travel along the free stream (S = 4..8).  So
// each run refits the boxes of the SAME tree (topology, facet order, everything by slot unchanged) in a frame
// whose z axis is the stream direction and hands that compact copy to the wavefront traversal (44 instead of up
// to 75 node visits per ray on C5, whatever the attitude).  Leaf boxes are the bounds of the rotated corners,
// evaluated in fp64 and rounded outwards; the traversal rotates the ray into the same frame (walk_init).
__global__ void k_leaf_boxes_rot(const float4* __restrict__ tris, int64_t nt, int64_t n_int, const double* __restrict__ R,
                                 float* __restrict__ box) {
  const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (s >= nt) return;
  double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
  for (int k = 0; k < 3; ++k) {
    const float4 q = tris[3 * s + k];
    for (int a = 0; a < 3; ++a) {
      const double x = (R[3 * a] * (double)q.x + R[3 * a + 1] * (double)q.y) + R[3 * a + 2] * (double)q.z;
      lo[a] = fmin(lo[a], x);
      hi[a] = fmax(hi[a], x);
    }
  }
  float* b = box + 6 * (n_int + s);
  for (int a = 0; a < 3; ++a) {   // fp64 rounding of the rotation: 1e-15 relative, far below one fp32 ulp
    b[a] = __double2float_rd(lo[a] - 1e-14 * fabs(lo[a]));
    b[3 + a] = __double2float_ru(hi[a] + 1e-14 * fabs(hi[a]));
  }
}

// Grid step of one axis: the root box spans steps 100 .. 65100.  Lower bounds: 1e-6 of the largest extent (flat axes),
// and 4u max|coordinate|, so that the 100-step pad below the box always exceeds the fp32 rounding of the grid origin
// (u |lo|): no plane of the hierarchy ever falls below step 0 or above step 65535, where k_compact_nodes would have to
// clamp it inwards.
__host__ __device__ inline double quant_step(double ext, double emax, double lo, double hi) {
  const double cmax = fmax(fabs(lo), fabs(hi));
  return fmax(fmax(ext, 1e-6 * emax) / 65000.0, fmax(4.0 * 5.9604645e-08 * cmax, 1e-30));
}

// Quantisation grid of the aligned hierarchy from the root box of the refit (device side: no host round trip).
// out_d: origin xyz, scale xyz (fp32 values held as doubles, for k_compact_nodes); out_g: what the traversal reads.
__global__ void k_align_grid(const float* __restrict__ root_box, const double* __restrict__ R, double* __restrict__ out_d,
                             QuantGrid* __restrict__ out_g) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  double ext[3], emax = 0.0, reach2 = 0.0;
  for (int a = 0; a < 3; ++a) {
    ext[a] = (double)root_box[3 + a] - (double)root_box[a];
    emax = fmax(emax, ext[a]);
    const double c = fmax(fabs((double)root_box[a]), fabs((double)root_box[3 + a]));
    reach2 += c * c;
  }
  for (int a = 0; a < 3; ++a) {
    const float qs = (float)quant_step(ext[a], emax, (double)root_box[a], (double)root_box[3 + a]);
    const float qo = (float)((double)root_box[a] - 100.0 * (double)qs);
    out_d[a] = (double)qo;
    out_d[3 + a] = (double)qs;
    out_g->origin[a] = qo;
    out_g->inv_scale[a] = (float)(1.0 / (double)qs);
  }
  for (int k = 0; k < 9; ++k) out_g->R[k] = (float)R[k];
  // rotation-error terms of the traversal's slab margin (trace.cuh, grid_ray): 9u |o|_1 + 6u reach metres
  out_g->rot_o = 9.0f * 5.9604645e-08f;
  out_g->rot_c = (float)(6.0 * 5.9604645e-08 * sqrt(reach2) * 1.0001);
}

// ---- escape horizon of every one-sided facet (a0, read by the reflect step) ------------------------------
// A particle re-emitted from facet f leaves a point p of f with a direction d above f's plane.  In the facet
// frame (e1 = first edge, e2 = n x e1, n = unit normal) let sin E = d.n / |d| be its elevation and
// phi = atan2(d.e2, d.e1) its azimuth.  horizon[slot][k], k = 0..15, is an upper bound of sin E over every ray
// from f with azimuth in sector k (22.5 deg each) that can hit the front of another facet: a ray above it
// escapes (O10 finds no hit) and its traversal is skipped.  Stored as a byte b, bound = b / 254; 255 = never
// skip.  Bounds used, all conservative, per other facet g or box B of the hierarchy:
//   * orientation (facets): a front-face hit needs d.n_g < 0.  With gamma = angle(n, n_g) <= 90 deg,
//     d.n_g >= |d| sin(E - gamma), so E >= gamma rules g out whatever the origin: sin E <= sin gamma.
//     (Two-sided or degenerate g: no bound from this argument.)
//   * position: a hit at x = p + tau d has sin E = n.(x - p) / |x - p|.  With c, rho the centre and radius
//     of f's bounding sphere, for x in B:  n.(x - p) <= h(B) = max_B n.(x - a0) + delta  and
//     |x - p| >= dist(c, B) - rho - delta,  delta covering the fp32 rounding of the ray origin (O13).
//     h(B) <= 0: B lies below f's plane and cannot be reached.  For a facet g, h is taken over its corners.
//   * azimuth: x - p lies in the ball of radius R = r_B + rho + delta about w = centre(B) - c, so d is within
//     alpha = asin(R / |w|) of w; if that cone does not contain the pole its azimuths lie within
//     asin(sin alpha / sin theta) of w's, theta = angle(w, n).  Otherwise, or when |w| <= R, all sectors.
// The hierarchy is walked nearest child first; a subtree is skipped when its position bound is not above the
// current value of any sector it can touch.  At a leaf the bound is the smaller of position and orientation.
constexpr int kHorizonStack = 96;
constexpr double kHorizonAzMargin = 2e-3;   // rad, covers the fp32 azimuth of the reflect step

struct HorizonFacet {
  double n[3], e1[3], e2[3], a0[3], c[3], rho, delta;
};

// position bound of a box, its distance from c, and the mask of azimuth sectors it can touch
__device__ __forceinline__ unsigned int horizon_quant(double b);
// (min_all: the smallest of the 16 sector bounds so far -- a box that cannot raise even that one is skipped before its
// azimuth range is worked out)
__device__ __forceinline__ double horizon_box(const HorizonFacet& f, const float lo[3], const float hi[3], double& dist,
                                              unsigned int& mask, unsigned int min_all) {
  double h = f.delta, d2 = 0.0, w[3], r2 = 0.0;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    h += fmax(f.n[k] * ((double)lo[k] - f.a0[k]), f.n[k] * ((double)hi[k] - f.a0[k]));
    const double e = fmax(fmax((double)lo[k] - f.c[k], f.c[k] - (double)hi[k]), 0.0);
    d2 += e * e;
    w[k] = 0.5 * ((double)lo[k] + (double)hi[k]) - f.c[k];
    const double hw = 0.5 * ((double)hi[k] - (double)lo[k]);
    r2 += hw * hw;
  }
  dist = sqrt(d2);
  mask = 0xFFFFu;
  if (!(h > 0.0)) return -1.0;                      // below the plane; empty boxes (lo > hi) end here as well
  const double den = dist * (1.0 - 1e-12) - f.rho - f.delta;
  const double bound = den > 0.0 ? h / den : INFINITY;
  if (horizon_quant(bound) <= min_all) return -1.0;
  const double R = (sqrt(r2) + f.rho + f.delta) * (1.0 + 1e-9);
  const double L = sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
  if (L > R) {
    const double x = w[0] * f.e1[0] + w[1] * f.e1[1] + w[2] * f.e1[2], y = w[0] * f.e2[0] + w[1] * f.e2[1] + w[2] * f.e2[2];
    const double st = sqrt(x * x + y * y) / L, sa = R / L;
    if (sa < st * (1.0 - 1e-6)) {
      // the two angles in fp32 (asinf, atan2f: a few ulp; the argument's rounding moves asin by at most 1e-7 / sqrt(2e-6));
      // 2e-4 rad on top of the margin covers both
      const float dphi = asinf(fminf((float)(sa / st), 1.0f)) + (float)kHorizonAzMargin + 2e-4f, phi = atan2f((float)y, (float)x);
      if (dphi < 3.0f) {
        const float q = 2.5464790894703255f;   // 16 / (2 pi)
        const int k0 = (int)floorf((phi - dphi + 3.14159265f) * q - 1e-4f), k1 = (int)floorf((phi + dphi + 3.14159265f) * q + 1e-4f);
        unsigned int m = 0u;
        for (int k = k0; k <= k1; ++k) m |= 1u << ((k + 16) & 15);
        mask = m;
      }
    }
  }
  return bound;
}

// 16 sector bounds packed as bytes in four words
__device__ __forceinline__ unsigned int nibble_bytes(unsigned int nib) { return (((nib & 15u) * 0x00204081u) & 0x01010101u) * 0xFFu; }
__device__ __forceinline__ unsigned int horizon_min(const unsigned int cur[4], unsigned int mask) {
  unsigned int m = 0xFFFFFFFFu;
#pragma unroll
  for (int j = 0; j < 4; ++j) m = __vminu4(m, cur[j] | ~nibble_bytes(mask >> (4 * j)));
  m = min(min(m & 0xFFu, (m >> 8) & 0xFFu), min((m >> 16) & 0xFFu, m >> 24));
  return m;
}
__device__ __forceinline__ unsigned int horizon_quant(double b) {   // byte >= 254 b (with the safety factor), 255 = never skip
  const double s = b * (1.0 + 1e-4) + 1e-4;
  return s < 1.0 ? (unsigned int)ceil(s * 254.0) : 255u;
}

__global__ void __launch_bounds__(128) k_horizon(const float4* __restrict__ nodes, const float4* __restrict__ tris,
                                                 int64_t nt, uint4* __restrict__ horizon) {
  const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (s >= nt) return;
  const float4 q0 = tris[3 * s], q1 = tris[3 * s + 1], q2 = tris[3 * s + 2];
  unsigned int cur[4] = {0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu};
  const bool two_sided = (__float_as_uint(q1.w) & TPMC_FACET_TWO_SIDED) != 0u;
  HorizonFacet f;
  const double a1[3] = {q1.x, q1.y, q1.z}, a2[3] = {q2.x, q2.y, q2.z};
  f.a0[0] = q0.x; f.a0[1] = q0.y; f.a0[2] = q0.z;
  double e2v[3];
  for (int k = 0; k < 3; ++k) { f.e1[k] = a1[k] - f.a0[k]; e2v[k] = a2[k] - f.a0[k]; f.c[k] = (f.a0[k] + a1[k] + a2[k]) / 3.0; }
  f.n[0] = f.e1[1] * e2v[2] - f.e1[2] * e2v[1];
  f.n[1] = f.e1[2] * e2v[0] - f.e1[0] * e2v[2];
  f.n[2] = f.e1[0] * e2v[1] - f.e1[1] * e2v[0];
  const double nl = sqrt(f.n[0] * f.n[0] + f.n[1] * f.n[1] + f.n[2] * f.n[2]);
  const double el = sqrt(f.e1[0] * f.e1[0] + f.e1[1] * f.e1[1] + f.e1[2] * f.e1[2]);
  if (!two_sided && nl > 0.0 && el > 0.0 && nt > 1) {
    double amax = 0.0;
    f.rho = 0.0;
    for (int k = 0; k < 3; ++k) {
      f.n[k] /= nl;
      f.e1[k] /= el;
      amax = fmax(amax, fmax(fabs(f.a0[k]), fmax(fabs(a1[k]), fabs(a2[k]))));
    }
    f.e2[0] = f.n[1] * f.e1[2] - f.n[2] * f.e1[1];
    f.e2[1] = f.n[2] * f.e1[0] - f.n[0] * f.e1[2];
    f.e2[2] = f.n[0] * f.e1[1] - f.n[1] * f.e1[0];
    for (int j = 0; j < 3; ++j) {
      const double* a = j == 0 ? f.a0 : (j == 1 ? a1 : a2);
      f.rho = fmax(f.rho, sqrt((a[0] - f.c[0]) * (a[0] - f.c[0]) + (a[1] - f.c[1]) * (a[1] - f.c[1]) + (a[2] - f.c[2]) * (a[2] - f.c[2])));
    }
    f.rho *= 1.0 + 1e-12;
    f.delta = 4e-7 * amax + 1e-30;   // > sqrt(3) * 2^-24 * |coordinate|: rounding of the hit point to fp32
    cur[0] = cur[1] = cur[2] = cur[3] = 0u;
    int stack[kHorizonStack];
    int sp = 0, node = 0;
    bool give_up = false;
    for (;;) {
      const float4 n0 = __ldg(nodes + 4 * (size_t)node), n1 = __ldg(nodes + 4 * (size_t)node + 1),
                   n2 = __ldg(nodes + 4 * (size_t)node + 2), n3 = __ldg(nodes + 4 * (size_t)node + 3);
      const float lo[2][3] = {{n0.x, n0.y, n0.z}, {n1.z, n1.w, n2.x}};
      const float hi[2][3] = {{n0.w, n1.x, n1.y}, {n2.y, n2.z, n2.w}};
      const int ref[2] = {__float_as_int(n3.x), __float_as_int(n3.y)};
      double dist[2];
      bool go[2];
      for (int ch = 0; ch < 2; ++ch) {
        unsigned int mask;
        const double bnd = horizon_box(f, lo[ch], hi[ch], dist[ch], mask, horizon_min(cur, 0xFFFFu));
        go[ch] = bnd > 0.0 && horizon_quant(bnd) > horizon_min(cur, mask);
        if (go[ch] && ref[ch] < 0) {        // leaf: the facet in it
          go[ch] = false;
          const int64_t g = ~ref[ch];
          if (g == s) continue;
          const float4 g0 = __ldg(tris + 3 * g), g1 = __ldg(tris + 3 * g + 1), g2 = __ldg(tris + 3 * g + 2);
          // height of the facet itself (a linear function: its maximum is at a corner), not of its box
          const double hv = f.delta + fmax(fmax(f.n[0] * ((double)g0.x - f.a0[0]) + f.n[1] * ((double)g0.y - f.a0[1]) + f.n[2] * ((double)g0.z - f.a0[2]),
                                               f.n[0] * ((double)g1.x - f.a0[0]) + f.n[1] * ((double)g1.y - f.a0[1]) + f.n[2] * ((double)g1.z - f.a0[2])),
                                          f.n[0] * ((double)g2.x - f.a0[0]) + f.n[1] * ((double)g2.y - f.a0[1]) + f.n[2] * ((double)g2.z - f.a0[2]));
          if (!(hv > 0.0)) continue;                 // wholly below the plane of f
          const double den = dist[ch] * (1.0 - 1e-12) - f.rho - f.delta;
          double b = den > 0.0 ? fmin(bnd, hv / den) : bnd;
          if ((__float_as_uint(g1.w) & TPMC_FACET_TWO_SIDED) == 0u) {
            const double f1[3] = {(double)g1.x - g0.x, (double)g1.y - g0.y, (double)g1.z - g0.z};
            const double f2[3] = {(double)g2.x - g0.x, (double)g2.y - g0.y, (double)g2.z - g0.z};
            const double m[3] = {f1[1] * f2[2] - f1[2] * f2[1], f1[2] * f2[0] - f1[0] * f2[2], f1[0] * f2[1] - f1[1] * f2[0]};
            const double ml = sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
            if (ml > 0.0) {
              const double cg = (f.n[0] * m[0] + f.n[1] * m[1] + f.n[2] * m[2]) / ml;
              if (cg > 0.0) b = fmin(b, sqrt(fmax(1.0 - cg * cg, 0.0)) + 1e-9);
            }
          }
          const unsigned int qb = horizon_quant(b) * 0x01010101u;
#pragma unroll
          for (int j = 0; j < 4; ++j) cur[j] = __vmaxu4(cur[j], qb & nibble_bytes(mask >> (4 * j)));
        }
      }
      if (go[0] && go[1]) {
        const bool sw = dist[1] < dist[0];
        if (sp >= kHorizonStack) { give_up = true; break; }
        stack[sp++] = sw ? ref[0] : ref[1];
        node = sw ? ref[1] : ref[0];
      } else if (go[0] || go[1]) {
        node = go[0] ? ref[0] : ref[1];
      } else {
        if (sp == 0) break;
        node = stack[--sp];
      }
    }
    if (give_up) cur[0] = cur[1] = cur[2] = cur[3] = 0xFFFFFFFFu;
  }
  horizon[s] = make_uint4(cur[0], cur[1], cur[2], cur[3]);
}

// ---- two-level cull volume for the pre-cull pass (a0) --------------------------------------------------------
// A body with a compact core and a few far-reaching parts (panels, booms) fills little of its bounding sphere or
// box.  Every facet is put either in the sphere of radius R_in about the centre (its farthest corner is within
// R_in) or, as an "outlier", in one of at most 8 boxes; a ray that misses the sphere and all boxes misses the
// mesh.  R_in is chosen among quantiles of the facets' reach, the outliers are binned into 4^3 cells of the AABB
// and the cell boxes merged greedily (smallest growth of surface area) on the host; the choice with the smallest
// mean projected area wins, and the volume is not used when it is no better than the bounding sphere.
constexpr int kReachBins = 1024;
__device__ __forceinline__ float facet_reach(const float4* __restrict__ tris, int64_t s, float cx, float cy, float cz) {
  float d2 = 0.0f;
  for (int k = 0; k < 3; ++k) {
    const float4 q = tris[3 * s + k];
    const float dx = q.x - cx, dy = q.y - cy, dz = q.z - cz;
    d2 = fmaxf(d2, __fadd_ru(__fadd_ru(__fmul_ru(dx, dx), __fmul_ru(dy, dy)), __fmul_ru(dz, dz)));
  }
  return __fsqrt_ru(d2) * 1.000001f;   // >= the true distance (the centre is rounded to fp32: 1e-6 covers it)
}
__global__ void k_reach_hist(const float4* __restrict__ tris, int64_t nt, float cx, float cy, float cz, float inv_bin,
                             unsigned int* __restrict__ hist) {
  const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (s >= nt) return;
  const int b = min(kReachBins - 1, (int)(facet_reach(tris, s, cx, cy, cz) * inv_bin));
  atomicAdd(&hist[b], 1u);
}
__device__ __forceinline__ unsigned int float_order(float f) {   // monotone map float -> unsigned
  const unsigned int u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
// boxes [64][6] as ordered unsigned: lo.xyz (atomicMin), hi.xyz (atomicMax) of the facets with reach > r_in
__global__ void k_outlier_boxes(const float4* __restrict__ tris, int64_t nt, float cx, float cy, float cz,
                                const float* __restrict__ r_in_dev, float3 lo, float3 inv_ext, unsigned int* __restrict__ boxes) {
  const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (s >= nt) return;
  const float r_in = *r_in_dev;
  if (!(r_in >= 0.0f) || !(facet_reach(tris, s, cx, cy, cz) > r_in)) return;   // r_in < 0: candidate not in use
  const float4 a = tris[3 * s], b = tris[3 * s + 1], c = tris[3 * s + 2];
  const int ix = min(3, max(0, (int)(((a.x + b.x + c.x) * (1.0f / 3.0f) - lo.x) * inv_ext.x * 4.0f)));
  const int iy = min(3, max(0, (int)(((a.y + b.y + c.y) * (1.0f / 3.0f) - lo.y) * inv_ext.y * 4.0f)));
  const int iz = min(3, max(0, (int)(((a.z + b.z + c.z) * (1.0f / 3.0f) - lo.z) * inv_ext.z * 4.0f)));
  unsigned int* bx = boxes + 6 * (16 * ix + 4 * iy + iz);
  atomicMin(bx + 0, float_order(fminf(a.x, fminf(b.x, c.x))));
  atomicMin(bx + 1, float_order(fminf(a.y, fminf(b.y, c.y))));
  atomicMin(bx + 2, float_order(fminf(a.z, fminf(b.z, c.z))));
  atomicMax(bx + 3, float_order(fmaxf(a.x, fmaxf(b.x, c.x))));
  atomicMax(bx + 4, float_order(fmaxf(a.y, fmaxf(b.y, c.y))));
  atomicMax(bx + 5, float_order(fmaxf(a.z, fmaxf(b.z, c.z))));
}

// The choice itself, on the device: candidate radii from the histogram, then per candidate a greedy merge of the
// outlier cells (<= 64 boxes: one thread) and the comparison of mean projected areas.
constexpr int kCullCandidates = 7;
struct CullChoice {
  float r_in[kCullCandidates];   // candidate inner radii, < 0: not in use
  double best;                   // smallest proxy so far (2 x mean projected area)
  float rin;
  int nbox;                      // -1: the bounding sphere stays
  float box[8][6];
};
__device__ __forceinline__ float float_unorder(unsigned int u) {
  return __uint_as_float((u & 0x80000000u) ? (u & 0x7FFFFFFFu) : ~u);
}
__global__ void k_cull_candidates(const unsigned int* __restrict__ hist, int64_t nt, float bin, double Rg, CullChoice* __restrict__ ch) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  const double quantiles[kCullCandidates] = {0.80, 0.90, 0.95, 0.97, 0.98, 0.99, 0.995};
  int last_bin = -1;
  for (int q = 0; q < kCullCandidates; ++q) {
    unsigned long long acc = 0;
    int b = 0;
    for (; b < kReachBins; ++b) { acc += hist[b]; if ((double)acc >= quantiles[q] * (double)nt) break; }
    const bool use = !(b >= kReachBins - 1 || b == last_bin);
    if (use) last_bin = b;
    ch->r_in[q] = use ? (float)(b + 1) * bin : -1.0f;
  }
  ch->best = 0.8 * 2.0 * 3.14159265358979323846 * Rg * Rg;   // must beat the bounding sphere (2 x projected area) by 20 %
  ch->nbox = -1;
  ch->rin = 0.0f;
}
__global__ void k_cull_init(unsigned int* __restrict__ boxes) {
  const int i = threadIdx.x;
  if (i < 64 * 6) boxes[i] = (i % 6) < 3 ? 0xFFFFFFFFu : 0u;
}
struct HBox { float lo[3], hi[3]; };
__device__ __forceinline__ double half_area(const HBox& b, double g) {
  const double e0 = (double)b.hi[0] - b.lo[0] + 2 * g, e1 = (double)b.hi[1] - b.lo[1] + 2 * g, e2 = (double)b.hi[2] - b.lo[2] + 2 * g;
  return e0 * e1 + e1 * e2 + e0 * e2;   // = 2 x the mean projected area of a box (Cauchy: surface / 4)
}
__device__ __forceinline__ HBox merged(const HBox& a, const HBox& b) {
  HBox m;
  for (int k = 0; k < 3; ++k) { m.lo[k] = fminf(a.lo[k], b.lo[k]); m.hi[k] = fmaxf(a.hi[k], b.hi[k]); }
  return m;
}
__global__ void k_cull_merge(const unsigned int* __restrict__ raw, int q, double g, CullChoice* __restrict__ ch) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  const float r_in = ch->r_in[q];
  if (!(r_in >= 0.0f)) return;
  HBox bx[64];
  int nb = 0;
  for (int i = 0; i < 64; ++i) {
    if (raw[6 * i] == 0xFFFFFFFFu) continue;   // empty cell
    for (int k = 0; k < 3; ++k) { bx[nb].lo[k] = float_unorder(raw[6 * i + k]); bx[nb].hi[k] = float_unorder(raw[6 * i + 3 + k]); }
    ++nb;
  }
  while (nb > 8) {   // greedy merge: the pair whose union adds the least area
    int bi = 0, bj = 1;
    double bc = 1e300;
    for (int i = 0; i < nb; ++i)
      for (int j = i + 1; j < nb; ++j) {
        const double c = half_area(merged(bx[i], bx[j]), g) - half_area(bx[i], g) - half_area(bx[j], g);
        if (c < bc) { bc = c; bi = i; bj = j; }
      }
    bx[bi] = merged(bx[bi], bx[bj]);
    bx[bj] = bx[--nb];
  }
  const double ri = (double)r_in + g;
  double proxy = 2.0 * 3.14159265358979323846 * ri * ri;
  for (int i = 0; i < nb; ++i) proxy += half_area(bx[i], g);
  if (proxy < ch->best) {
    ch->best = proxy;
    ch->rin = r_in;
    ch->nbox = nb;
    for (int i = 0; i < nb; ++i)
      for (int k = 0; k < 3; ++k) { ch->box[i][k] = bx[i].lo[k]; ch->box[i][3 + k] = bx[i].hi[k]; }
  }
}

struct DevBuf {  // frees on scope exit
  void* p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
  template <class T> T* as() { return (T*)p; }
};

// Choose the two-level cull volume (see k_reach_hist).  Leaves m->cull_nbox = -1 when it does not pay.  Everything is
// computed on the device; the host reads the chosen volume once (the per-run constants are assembled there).
int build_cull_volume(tpmc_mesh* m, cudaStream_t st) {
  m->cull_nbox = -1;
  m->cull_rin = (float)m->Rb;
  const int64_t nt = m->nt;
  if (nt < 64) return TPMC_OK;
  DevBuf hist, boxes, choice;
  TPMC_CUDA_TRY(cudaMalloc(&hist.p, sizeof(unsigned int) * kReachBins));
  TPMC_CUDA_TRY(cudaMalloc(&boxes.p, sizeof(unsigned int) * 64 * 6));
  TPMC_CUDA_TRY(cudaMalloc(&choice.p, sizeof(CullChoice)));
  TPMC_CUDA_TRY(cudaMemsetAsync(hist.p, 0, sizeof(unsigned int) * kReachBins, st));
  const float cx = (float)m->centre[0], cy = (float)m->centre[1], cz = (float)m->centre[2];
  const float bin = (float)(m->Rb * 1.0001 / kReachBins);
  const unsigned gt = (unsigned)((nt + kBlock - 1) / kBlock);
  const double g = (double)kPrecullMargin * m->Rb;
  k_reach_hist<<<gt, kBlock, 0, st>>>(m->tris, nt, cx, cy, cz, 1.0f / bin, hist.as<unsigned int>());
  k_cull_candidates<<<1, 32, 0, st>>>(hist.as<unsigned int>(), nt, bin, m->Rb + g, choice.as<CullChoice>());
  float3 lo = make_float3(m->aabb_lo[0], m->aabb_lo[1], m->aabb_lo[2]);
  float3 ie;
  ie.x = m->aabb_hi[0] > m->aabb_lo[0] ? 1.0f / (m->aabb_hi[0] - m->aabb_lo[0]) : 0.0f;
  ie.y = m->aabb_hi[1] > m->aabb_lo[1] ? 1.0f / (m->aabb_hi[1] - m->aabb_lo[1]) : 0.0f;
  ie.z = m->aabb_hi[2] > m->aabb_lo[2] ? 1.0f / (m->aabb_hi[2] - m->aabb_lo[2]) : 0.0f;
  for (int q = 0; q < kCullCandidates; ++q) {
    k_cull_init<<<1, 384, 0, st>>>(boxes.as<unsigned int>());
    k_outlier_boxes<<<gt, kBlock, 0, st>>>(m->tris, nt, cx, cy, cz, choice.as<CullChoice>()->r_in + q, lo, ie, boxes.as<unsigned int>());
    k_cull_merge<<<1, 32, 0, st>>>(boxes.as<unsigned int>(), q, g, choice.as<CullChoice>());
  }
  CullChoice h;
  TPMC_CUDA_TRY(cudaMemcpyAsync(&h, choice.p, sizeof(h), cudaMemcpyDeviceToHost, st));
  TPMC_CUDA_TRY(cudaStreamSynchronize(st));
  if (h.nbox >= 0) {
    m->cull_rin = h.rin;
    m->cull_nbox = h.nbox;
    for (int i = 0; i < h.nbox; ++i)
      for (int k = 0; k < 6; ++k) m->cull_box[i][k] = h.box[i][k];
  }
  return TPMC_OK;
}

}  // namespace

// The escape-horizon pass on its own (tpmc_mesh_create runs it unless told not to; tpmc_mesh_build_horizon runs it later).
static int build_horizon(tpmc_mesh* m, cudaStream_t st) {
  if (m->horizon) return TPMC_OK;
  uint4* hz = nullptr;
  cudaEvent_t h0 = nullptr, h1 = nullptr;
  TPMC_CUDA_TRY(cudaMalloc((void**)&hz, sizeof(uint4) * m->nt));
  cudaError_t e = cudaEventCreate(&h0);
  if (e == cudaSuccess) e = cudaEventCreate(&h1);
  if (e == cudaSuccess) e = cudaEventRecord(h0, st);
  if (e == cudaSuccess) {
    k_horizon<<<(unsigned)((m->nt + 127) / 128), 128, 0, st>>>(m->nodes, m->tris, m->nt, hz);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaEventRecord(h1, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  float ms = 0.0f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, h0, h1);
  if (h0) cudaEventDestroy(h0);
  if (h1) cudaEventDestroy(h1);
  if (e != cudaSuccess) cudaFree(hz);
  TPMC_CUDA_TRY(e);
  m->horizon = hz;   // runs enqueued from now on use it
  m->horizon_ms = ms;
  return TPMC_OK;
}

extern "C" int tpmc_mesh_build_horizon(tpmc_mesh* m, void* cuda_stream) {
  if (!m) return TPMC_EINVAL;
  return build_horizon(m, (cudaStream_t)cuda_stream);
}

static int mesh_create_impl(const float* vertices, int64_t nv, const int32_t* indices, int64_t nt, const uint8_t* facet_flags,
                            int mem_space, uint32_t mesh_flags, void* cuda_stream, tpmc_mesh** out);

extern "C" int tpmc_mesh_create(const float* vertices, int64_t nv, const int32_t* indices, int64_t nt,
                                const uint8_t* facet_flags, int mem_space, void* cuda_stream, tpmc_mesh** out) {
  return mesh_create_impl(vertices, nv, indices, nt, facet_flags, mem_space, 0u, cuda_stream, out);
}

extern "C" int tpmc_mesh_create_ex(const float* vertices, int64_t nv, const int32_t* indices, int64_t nt,
                                   const uint8_t* facet_flags, int mem_space, uint32_t mesh_flags, void* cuda_stream,
                                   tpmc_mesh** out) {
  if (out) *out = nullptr;
  if (mesh_flags & ~(uint32_t)TPMC_MESH_NO_HORIZON) return TPMC_EINVAL;
  return mesh_create_impl(vertices, nv, indices, nt, facet_flags, mem_space, mesh_flags, cuda_stream, out);
}

static int mesh_create_impl(const float* vertices, int64_t nv, const int32_t* indices, int64_t nt, const uint8_t* facet_flags,
                            int mem_space, uint32_t mesh_flags, void* cuda_stream, tpmc_mesh** out) {
  if (!out) return TPMC_EINVAL;
  *out = nullptr;
  if (!vertices || !indices || nv < 3 || nt < 1 || nt > 0x3FFFFFFF || nv > 0x7FFFFFFF) return TPMC_EINVAL;
  if (mem_space != TPMC_MEM_HOST && mem_space != TPMC_MEM_DEVICE) return TPMC_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0;
  TPMC_CUDA_TRY(cudaGetDevice(&dev));

  DevBuf dv, di, df;
  const float* d_v = vertices;
  const int32_t* d_i = indices;
  const uint8_t* d_f = facet_flags;
  if (mem_space == TPMC_MEM_HOST) {
    TPMC_CUDA_TRY(cudaMalloc(&dv.p, sizeof(float) * 3 * nv));
    TPMC_CUDA_TRY(cudaMalloc(&di.p, sizeof(int32_t) * 3 * nt));
    TPMC_CUDA_TRY(cudaMemcpyAsync(dv.p, vertices, sizeof(float) * 3 * nv, cudaMemcpyHostToDevice, st));
    TPMC_CUDA_TRY(cudaMemcpyAsync(di.p, indices, sizeof(int32_t) * 3 * nt, cudaMemcpyHostToDevice, st));
    d_v = dv.as<float>();
    d_i = di.as<int32_t>();
    if (facet_flags) {
      TPMC_CUDA_TRY(cudaMalloc(&df.p, nt));
      TPMC_CUDA_TRY(cudaMemcpyAsync(df.p, facet_flags, nt, cudaMemcpyHostToDevice, st));
      d_f = df.as<uint8_t>();
    }
  }

  cudaEvent_t e0, e1;
  TPMC_CUDA_TRY(cudaEventCreate(&e0));
  TPMC_CUDA_TRY(cudaEventCreate(&e1));
  TPMC_CUDA_TRY(cudaEventRecord(e0, st));

  // validate indices, bounds (O1)
  DevBuf small;
  TPMC_CUDA_TRY(cudaMalloc(&small.p, 64));
  TPMC_CUDA_TRY(cudaMemsetAsync(small.p, 0, 64, st));
  int* d_bad = small.as<int>();
  float* d_aabb = small.as<float>() + 2;
  double* d_r2 = (double*)((char*)small.p + 32);
  k_check_indices<<<(unsigned)((3 * nt + kBlock - 1) / kBlock), kBlock, 0, st>>>(d_i, 3 * nt, nv, d_bad);
  k_vertex_aabb<<<1, 1024, 0, st>>>(d_v, nv, d_aabb);
  struct { int bad; int pad; float aabb[6]; double r2; } h;
  TPMC_CUDA_TRY(cudaMemcpyAsync(&h, small.p, 32, cudaMemcpyDeviceToHost, st));
  TPMC_CUDA_TRY(cudaStreamSynchronize(st));
  if (h.bad) { cudaEventDestroy(e0); cudaEventDestroy(e1); return TPMC_EINVAL; }
  for (int a = 0; a < 6; ++a)
    if (!isfinite(h.aabb[a])) { cudaEventDestroy(e0); cudaEventDestroy(e1); return TPMC_EINVAL; }
  double centre[3];
  for (int a = 0; a < 3; ++a) centre[a] = 0.5 * ((double)h.aabb[a] + (double)h.aabb[3 + a]);
  k_vertex_r2<<<1, 1024, 0, st>>>(d_v, nv, centre[0], centre[1], centre[2], d_r2);
  TPMC_CUDA_TRY(cudaMemcpyAsync(&h.r2, d_r2, 8, cudaMemcpyDeviceToHost, st));
  TPMC_CUDA_TRY(cudaStreamSynchronize(st));
  if (!(h.r2 > 0.0)) { cudaEventDestroy(e0); cudaEventDestroy(e1); return TPMC_EINVAL; }

  tpmc_mesh* m = new (std::nothrow) tpmc_mesh();
  if (!m) return TPMC_ENOMEM;
  memset(m, 0, sizeof(*m));
  m->nv = nv; m->nt = nt; m->device = dev;
  m->n_nodes = nt > 1 ? nt - 1 : 1;
  for (int a = 0; a < 3; ++a) { m->centre[a] = centre[a]; m->aabb_lo[a] = h.aabb[a]; m->aabb_hi[a] = h.aabb[3 + a]; }
  m->Rb = sqrt(h.r2);
  m->ev0 = e0; m->ev1 = e1;

#define MESH_TRY(expr)                       \
  do {                                       \
    int _rc = [&]() -> int { TPMC_CUDA_TRY(expr); return TPMC_OK; }(); \
    if (_rc != TPMC_OK) { tpmc_mesh_destroy(m); return _rc; }          \
  } while (0)

  MESH_TRY(cudaMalloc((void**)&m->nodes, sizeof(float4) * 4 * m->n_nodes));
  MESH_TRY(cudaMalloc((void**)&m->tris, sizeof(float4) * 3 * nt));

  DevBuf keys, keys2, ids, ids2, tmp, box, nsize;
  const int64_t n_int = nt - 1;
  MESH_TRY(cudaMalloc(&keys.p, sizeof(uint64_t) * nt));
  MESH_TRY(cudaMalloc(&keys2.p, sizeof(uint64_t) * nt));
  MESH_TRY(cudaMalloc(&ids.p, sizeof(int32_t) * nt));
  MESH_TRY(cudaMalloc(&ids2.p, sizeof(int32_t) * nt));
  MESH_TRY(cudaMalloc(&box.p, sizeof(float) * 6 * (size_t)(n_int + nt)));
  const unsigned gt = (unsigned)((nt + kBlock - 1) / kBlock);
  float3 lo = make_float3(h.aabb[0], h.aabb[1], h.aabb[2]);
  float3 ie;
  ie.x = h.aabb[3] > h.aabb[0] ? 1.0f / (h.aabb[3] - h.aabb[0]) : 0.0f;
  ie.y = h.aabb[4] > h.aabb[1] ? 1.0f / (h.aabb[4] - h.aabb[1]) : 0.0f;
  ie.z = h.aabb[5] > h.aabb[2] ? 1.0f / (h.aabb[5] - h.aabb[2]) : 0.0f;
  k_morton<<<gt, kBlock, 0, st>>>(d_v, d_i, nt, lo, ie, keys.as<uint64_t>(), ids.as<int32_t>());
  MESH_TRY(cudaMalloc(&tmp.p, radix::scratch_bytes(nt)));
  // 63-bit codes: 16 passes of 4 bits, stable, so equal codes keep the facet order (the hierarchy's tie-break)
  const int where = radix::sort_pairs(keys.as<uint64_t>(), ids.as<int32_t>(), keys2.as<uint64_t>(), ids2.as<int32_t>(), nt, 64,
                                      tmp.as<unsigned int>(), st);
  const uint64_t* keys_sorted = where ? keys2.as<uint64_t>() : keys.as<uint64_t>();
  const int32_t* ids_sorted = where ? ids2.as<int32_t>() : ids.as<int32_t>();
  k_gather<<<gt, kBlock, 0, st>>>(d_v, d_i, d_f, ids_sorted, nt, m->tris, box.as<float>(), n_int);
  if (nt == 1) {
    k_single<<<1, 1, 0, st>>>(box.as<float>(), m->nodes);
  } else {
    MESH_TRY(cudaMalloc((void**)&m->kids, sizeof(int2) * n_int));
    MESH_TRY(cudaMalloc((void**)&m->parent, sizeof(int) * (size_t)(n_int + nt)));
    MESH_TRY(cudaMalloc((void**)&m->arrive, sizeof(int) * n_int));
    MESH_TRY(cudaMalloc((void**)&m->rbox, sizeof(float) * 6 * (size_t)(n_int + nt)));
    MESH_TRY(cudaMalloc((void**)&m->align_R, sizeof(double) * 16));
    MESH_TRY(cudaMemsetAsync(m->arrive, 0, sizeof(int) * n_int, st));
    MESH_TRY(cudaMalloc(&nsize.p, sizeof(int) * n_int));
    k_hierarchy<<<(unsigned)((n_int + kBlock - 1) / kBlock), kBlock, 0, st>>>(keys_sorted, (int)nt, m->kids, m->parent, nsize.as<int>());
    k_refit<<<gt, kBlock, 0, st>>>((int)nt, m->kids, m->parent, box.as<float>(), m->arrive, m->nodes);
  }
  {
    // quantisation grid: the vertex AABB spans steps 100 .. 65100 of each axis (flat axes get a tiny step)
    double ext[3], emax = 0.0;
    for (int a = 0; a < 3; ++a) { ext[a] = (double)h.aabb[3 + a] - (double)h.aabb[a]; emax = std::max(emax, ext[a]); }
    for (int a = 0; a < 3; ++a) {
      m->q_scale[a] = (float)quant_step(ext[a], emax, (double)h.aabb[a], (double)h.aabb[3 + a]);
      m->q_origin[a] = (float)((double)h.aabb[a] - 100.0 * (double)m->q_scale[a]);
    }
    MESH_TRY(cudaMalloc((void**)&m->cnodes, sizeof(uint4) * 2 * m->n_nodes));
    k_compact_nodes<<<(unsigned)((m->n_nodes + kBlock - 1) / kBlock), kBlock, 0, st>>>(
        m->nodes, m->n_nodes, (double)m->q_origin[0], (double)m->q_origin[1], (double)m->q_origin[2],
        (double)m->q_scale[0], (double)m->q_scale[1], (double)m->q_scale[2], m->cnodes);
    QuantGrid hg;
    for (int a = 0; a < 3; ++a) { hg.origin[a] = m->q_origin[a]; hg.inv_scale[a] = (float)(1.0 / (double)m->q_scale[a]); }
    for (int k = 0; k < 9; ++k) hg.R[k] = (k % 4 == 0) ? 1.0f : 0.0f;
    hg.rot_o = hg.rot_c = 0.0f;   // the identity frame is exact
    MESH_TRY(cudaMalloc((void**)&m->grid_dev, 2 * sizeof(QuantGrid)));
    MESH_TRY(cudaMemcpyAsync(m->grid_dev, &hg, sizeof(hg), cudaMemcpyHostToDevice, st));
    MESH_TRY(cudaMemcpyAsync(m->grid_dev + 1, &hg, sizeof(hg), cudaMemcpyHostToDevice, st));
  }
  {
    // wide hierarchy of the traversal: topology breadth-first (k_wide_*), then the body-frame boxes
    DevBuf lvl, wroot, wcnt;
    const int64_t cap_w = std::max<int64_t>(n_int, 1);
    MESH_TRY(cudaMalloc((void**)&m->wkids_bin, sizeof(int4) * cap_w));
    MESH_TRY(cudaMalloc((void**)&m->wkids, sizeof(int4) * cap_w));
    MESH_TRY(cudaMalloc(&wroot.p, sizeof(int) * cap_w));
    MESH_TRY(cudaMalloc(&wcnt.p, sizeof(unsigned int) * cap_w));
    MESH_TRY(cudaMalloc(&lvl.p, sizeof(int) * 4));
    k_wide_init<<<1, 32, 0, st>>>(lvl.as<int>(), wroot.as<int>(), m->wkids_bin, m->wkids, nt == 1 ? 1 : 0);
    int hl[4] = {0, 0, 0, 0};
    const unsigned gw = (unsigned)std::min<int64_t>((cap_w + kBlock - 1) / kBlock, 592);
    for (int L = 0; L < kWideLevels; L += 8) {   // eight levels per read-back of the frontier (a 1e6-facet body has ~12)
      if (nt > 1)
        for (int l8 = 0; l8 < 8; ++l8) {
          k_wide_expand<<<gw, kBlock, 0, st>>>(m->kids, box.as<float>(), nsize.as<int>(), lvl.as<int>(), wroot.as<int>(), m->wkids_bin, wcnt.as<unsigned int>());
          k_wide_scan<<<1, 1024, 0, st>>>(wcnt.as<unsigned int>(), lvl.as<int>());
          k_wide_assign<<<gw, kBlock, 0, st>>>(lvl.as<int>(), m->wkids_bin, wcnt.as<unsigned int>(), wroot.as<int>(), m->wkids);
          k_wide_next<<<1, 32, 0, st>>>(lvl.as<int>());
        }
      MESH_TRY(cudaMemcpyAsync(hl, lvl.p, sizeof(hl), cudaMemcpyDeviceToHost, st));
      MESH_TRY(cudaStreamSynchronize(st));
      if (hl[0] == hl[1]) break;   // the frontier is empty
    }
    if (hl[0] != hl[1] || hl[1] < 1 || hl[1] > cap_w) { tpmc_mesh_destroy(m); return TPMC_ECUDA; }   // the frontier must be empty
    m->n_wide = hl[1];
    MESH_TRY(cudaMalloc((void**)&m->wnodes, sizeof(uint4) * 4 * m->n_wide));
    if (nt > 1) MESH_TRY(cudaMalloc((void**)&m->wnodes_r, sizeof(uint4) * 4 * m->n_wide));
    k_compact_wide<<<(unsigned)((m->n_wide + kBlock - 1) / kBlock), kBlock, 0, st>>>(
        box.as<float>(), n_int, m->wkids_bin, m->wkids, m->n_wide, (double)m->q_origin[0], (double)m->q_origin[1],
        (double)m->q_origin[2], (double)m->q_scale[0], (double)m->q_scale[1], (double)m->q_scale[2], m->wnodes);
  }
  DevBuf cq;
  MESH_TRY(cudaMalloc((void**)&m->cull_c, sizeof(uint4) * 2 * kCullNodes));
  MESH_TRY(cudaMalloc(&cq.p, sizeof(int) * (kCullNodes + 1)));
  k_build_cull<<<1, 32, 0, st>>>(m->nodes, m->cnodes, m->cull_c, cq.as<int>(), kCullNodes, cq.as<int>() + kCullNodes);
  MESH_TRY(cudaMemcpyAsync(&m->n_cull, cq.as<int>() + kCullNodes, sizeof(int), cudaMemcpyDeviceToHost, st));
  {
    const int rcv = build_cull_volume(m, st);
    if (rcv != TPMC_OK) { tpmc_mesh_destroy(m); return rcv; }
  }
  MESH_TRY(cudaGetLastError());
  MESH_TRY(cudaEventRecord(e1, st));
  {
    const cudaError_t es = cudaStreamSynchronize(st);
    float ms = 0.0f;
    if (es == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
    MESH_TRY(es);   // (e0, e1 belong to the handle from here on: m->ev0, m->ev1)
    m->build_ms = ms;
  }
  // escape horizons (timed apart from the hierarchy build; skipped on request: runs then trace every re-emitted ray)
  if (!(mesh_flags & TPMC_MESH_NO_HORIZON)) {
    const int rch = build_horizon(m, st);
    if (rch != TPMC_OK) { tpmc_mesh_destroy(m); return rch; }
  }
#undef MESH_TRY
  *out = m;
  return TPMC_OK;
}


// Refit the compact hierarchy in the frame x' = R x (row-major 3x3, orthonormal) on `stream`; fills *grid.
// Called by tpmc_run with the stream frame of the run.  nt == 1: the body-frame hierarchy is used.
int tpmc_mesh_align(tpmc_mesh* m, const double R[9], cudaStream_t st, const QuantGrid** grid_out, const uint4** wnodes_out) {
  *grid_out = m->grid_dev;   // [0]: the body-frame grid, [1]: the aligned one
  *wnodes_out = m->wnodes;
  if (m->nt < 2 || !m->kids) return TPMC_OK;
  const int64_t nt = m->nt, n_int = nt - 1;
  const unsigned gt = (unsigned)((nt + kBlock - 1) / kBlock);
  TPMC_CUDA_TRY(cudaMemcpyAsync(m->align_R, R, 9 * sizeof(double), cudaMemcpyHostToDevice, st));
  TPMC_CUDA_TRY(cudaMemsetAsync(m->arrive, 0, sizeof(int) * n_int, st));
  k_leaf_boxes_rot<<<gt, kBlock, 0, st>>>(m->tris, nt, n_int, m->align_R, m->rbox);
  k_refit<<<gt, kBlock, 0, st>>>((int)nt, m->kids, m->parent, m->rbox, m->arrive, nullptr);
  k_align_grid<<<1, 32, 0, st>>>(m->rbox, m->align_R, m->align_R + 9, m->grid_dev + 1);
  k_compact_wide<<<(unsigned)((m->n_wide + kBlock - 1) / kBlock), kBlock, 0, st>>>(m->rbox, n_int, m->wkids_bin, m->wkids, m->n_wide, 0, 0,
                                                                                   0, 1, 1, 1, m->wnodes_r, m->align_R + 9);
  TPMC_CUDA_TRY(cudaGetLastError());
  *wnodes_out = m->wnodes_r;
  *grid_out = m->grid_dev + 1;
  return TPMC_OK;
}

extern "C" void tpmc_mesh_destroy(tpmc_mesh* m) {
  if (!m) return;
  cudaFree(m->nodes); cudaFree(m->tris); cudaFree(m->cull_c); cudaFree(m->kids); cudaFree(m->parent); cudaFree(m->arrive); cudaFree(m->rbox); cudaFree(m->wkids_bin); cudaFree(m->wkids); cudaFree(m->wnodes); cudaFree(m->wnodes_r); cudaFree(m->align_R); cudaFree(m->grid_dev); cudaFree(m->cnodes); cudaFree(m->horizon); cudaFree(m->surf_TW); cudaFree(m->surf_sigma);
  for (int pi = 0; pi < kPipes; ++pi) {
    Pipe& pp = m->pipe[pi];
    for (int k = 0; k < 2; ++k) { cudaFree(pp.q_o[k]); cudaFree(pp.q_v[k]); cudaFree(pp.q_f[k]); cudaFree(pp.q_key[k]); cudaFree(pp.hist[k]); }
    cudaFree(pp.hit_ray); cudaFree(pp.hit_cand); cudaFree(pp.ctr); cudaFree(pp.surv); cudaFree(pp.ovf); cudaFree(pp.order);
    if (pi > 0 && pp.main) cudaStreamDestroy(pp.main);
    if (pp.seed) cudaStreamDestroy(pp.seed);
    if (pp.side) cudaStreamDestroy(pp.side);
    for (int k = 0; k < 2; ++k) {
      if (pp.ev_refl[k]) cudaEventDestroy(pp.ev_refl[k]);
      if (pp.ev_ovf[k]) cudaEventDestroy(pp.ev_ovf[k]);
    }
    for (int k = 0; k < 4; ++k) {
      if (pp.ev_reset[k]) cudaEventDestroy(pp.ev_reset[k]);
      if (pp.ev_seeded[k]) cudaEventDestroy(pp.ev_seeded[k]);
    }
    if (pp.ev_done) cudaEventDestroy(pp.ev_done);
    if (pp.ev_f0) cudaEventDestroy(pp.ev_f0);
    if (pp.ev_f1) cudaEventDestroy(pp.ev_f1);
    if (pp.wave_ev) {
      for (int i = 0; i < kEvPerWave * kMaxTimedWaves; ++i) cudaEventDestroy(pp.wave_ev[i]);
      delete[] pp.wave_ev;
    }
  }
  cudaFree(m->facet_scratch); cudaFree(m->partials); cudaFree(m->stats); cudaFree(m->totals); cudaFree(m->ft_dev);
  if (m->ev0) cudaEventDestroy(m->ev0);
  if (m->ev1) cudaEventDestroy(m->ev1);
  if (m->ev_fork) cudaEventDestroy(m->ev_fork);
  delete m;
}

// A23: per-facet wall temperature and accommodation, by facet id; either may be NULL (the run's scalar is used).
namespace {
// counts the entries a run could not use: T_W must be finite and > 0 (c_W = sqrt(2 k T_W / m)), sigma in [0, 1]
__global__ void k_check_surface(const double* __restrict__ T_W, const double* __restrict__ sigma, int64_t nt,
                                unsigned int* __restrict__ bad) {
  const int64_t f = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  bool b = false;
  if (f < nt) {
    if (T_W) { const double t = T_W[f]; b = !(t > 0.0 && isfinite(t)); }
    if (sigma) { const double g = sigma[f]; b = b || !(g >= 0.0 && g <= 1.0); }
  }
  if (__syncthreads_or(b) && threadIdx.x == 0) atomicAdd(bad, 1u);
}
}  // namespace

extern "C" int tpmc_mesh_set_surface(tpmc_mesh* m, const double* T_W, const double* sigma, int mem_space, void* cuda_stream) {
  if (!m || (mem_space != TPMC_MEM_HOST && mem_space != TPMC_MEM_DEVICE)) return TPMC_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t bytes = sizeof(double) * (size_t)m->nt;
  const cudaMemcpyKind kind = mem_space == TPMC_MEM_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
  // validate before anything is replaced: T_W > 0 and finite, 0 <= sigma <= 1 (a NaN passes neither)
  if (mem_space == TPMC_MEM_HOST) {
    for (int64_t f = 0; f < m->nt; ++f) {
      if (T_W && !(T_W[f] > 0.0 && isfinite(T_W[f]))) return TPMC_EINVAL;
      if (sigma && !(sigma[f] >= 0.0 && sigma[f] <= 1.0)) return TPMC_EINVAL;
    }
  } else if (T_W || sigma) {   // device arrays: the same test by a kernel, one word read back
    unsigned int* d_bad = nullptr;
    unsigned int h_bad = 0;
    TPMC_CUDA_TRY(cudaMalloc((void**)&d_bad, sizeof(unsigned int)));
    cudaError_t e = cudaMemsetAsync(d_bad, 0, sizeof(unsigned int), st);
    if (e == cudaSuccess) {
      k_check_surface<<<(unsigned)((m->nt + 255) / 256), 256, 0, st>>>(T_W, sigma, m->nt, d_bad);
      e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h_bad, d_bad, sizeof(unsigned int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_bad);
    TPMC_CUDA_TRY(e);
    if (h_bad) return TPMC_EINVAL;
  }
  // No run may still read the arrays being replaced or freed.  The header asks for all calls on a handle to share one
  // stream, but nothing enforces it and this is a set-up call: wait for the whole device, not just for `st`.
  TPMC_CUDA_TRY(cudaDeviceSynchronize());
  const double* src[2] = {T_W, sigma};
  double** dst[2] = {&m->surf_TW, &m->surf_sigma};
  for (int k = 0; k < 2; ++k) {
    if (!src[k]) { cudaFree(*dst[k]); *dst[k] = nullptr; continue; }
    if (!*dst[k]) TPMC_CUDA_TRY(cudaMalloc((void**)dst[k], bytes));
    TPMC_CUDA_TRY(cudaMemcpyAsync(*dst[k], src[k], bytes, kind, st));
  }
  TPMC_CUDA_TRY(cudaStreamSynchronize(st));
  return TPMC_OK;
}

extern "C" int tpmc_mesh_info(const tpmc_mesh* m, tpmc_mesh_info_t* out) {
  if (!m || !out) return TPMC_EINVAL;
  for (int a = 0; a < 3; ++a) { out->centre[a] = m->centre[a]; out->aabb_lo[a] = m->aabb_lo[a]; out->aabb_hi[a] = m->aabb_hi[a]; }
  out->bounding_radius = m->Rb;
  out->nt = m->nt;
  out->n_nodes = m->n_nodes;
  out->build_ms = m->build_ms;
  out->horizon_ms = m->horizon_ms;
  return TPMC_OK;
}

namespace {
__global__ void k_leaf_facets(const float4* __restrict__ tris, int64_t nt, int32_t* __restrict__ out) {
  const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (s < nt) out[s] = __float_as_int(tris[3 * s].w);
}
}  // namespace

extern "C" int tpmc_mesh_copy_bvh(const tpmc_mesh* m, float* h_nodes, int32_t* h_leaf_facet) {
  if (!m) return TPMC_EINVAL;
  if (h_nodes) TPMC_CUDA_TRY(cudaMemcpy(h_nodes, m->nodes, sizeof(float4) * 4 * m->n_nodes, cudaMemcpyDeviceToHost));
  if (h_leaf_facet) {
    DevBuf t;
    TPMC_CUDA_TRY(cudaMalloc(&t.p, sizeof(int32_t) * m->nt));
    k_leaf_facets<<<(unsigned)((m->nt + kBlock - 1) / kBlock), kBlock>>>(m->tris, m->nt, t.as<int32_t>());
    TPMC_CUDA_TRY(cudaMemcpy(h_leaf_facet, t.p, sizeof(int32_t) * m->nt, cudaMemcpyDeviceToHost));
  }
  return TPMC_OK;
}

extern "C" int tpmc_mesh_copy_wide(const tpmc_mesh* m, int64_t* n_wide, uint32_t* h_wnodes, float* h_grid) {
  if (!m || !n_wide) return TPMC_EINVAL;
  *n_wide = m->n_wide;
  if (h_wnodes) TPMC_CUDA_TRY(cudaMemcpy(h_wnodes, m->wnodes, sizeof(uint4) * 4 * m->n_wide, cudaMemcpyDeviceToHost));
  if (h_grid)
    for (int a = 0; a < 3; ++a) { h_grid[a] = m->q_origin[a]; h_grid[3 + a] = m->q_scale[a]; }
  return TPMC_OK;
}

extern "C" int tpmc_mesh_copy_horizon(const tpmc_mesh* m, uint8_t* h_horizon) {
  if (!m || !h_horizon || !m->horizon) return TPMC_EINVAL;   // (no horizons: created with TPMC_MESH_NO_HORIZON)
  TPMC_CUDA_TRY(cudaMemcpy(h_horizon, m->horizon, sizeof(uint4) * m->nt, cudaMemcpyDeviceToHost));
  return TPMC_OK;
}

extern "C" const char* tpmc_strerror(int code) {
  switch (code) {
    case TPMC_OK: return "ok";
    case TPMC_EINVAL: return "invalid argument";
    case TPMC_ENOMEM: return "out of memory";
    case TPMC_ECUDA: return "CUDA error";
    case TPMC_ECAPACITY: return "input exceeds the fixed capacity of this entry point";
    default: return "unknown error";
  }
}
extern "C" const char* tpmc_last_cuda_error(void) { return g_tpmc_cuda_error; }
extern "C" const char* tpmc_version(void) { return "tpmc-b200 0.1 (sm_100a)"; }
