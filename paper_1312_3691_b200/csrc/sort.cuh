// sort.cuh -- spatial ordering of the ray queue before the wavefront traversal (step a3).
//
// Particles are keyed by index (Philox), so consecutive queue slots hold rays from all over the control sphere:
// the 32 lanes of a traversal warp walk 32 unrelated paths (32 cache lines per node fetch, lanes finishing at
// very different times).  The path computes nothing order-dependent (sums are fp64 atomics), so the queue may be
// traced in any order: every ray gets a small key that says WHERE on the body it is heading, and the traversal
// fetches rays in key order, so that a warp's rays share the top of the hierarchy and most of their node fetches.
//   key      = cell of the octahedral map of the direction (E - centre) from the body centre, kSortBits bits
//              (two coordinates, Morton-interleaved), E = where a primary enters the key sphere (or comes
//              closest to it), or the origin of a reflected ray;
//   sort     = one counting-sort pass: the seed and reflect kernels bump the key's histogram bin as they append
//              a ray, k_sort_scan turns the histogram into offsets, k_sort_scatter writes queue slots in key order.
// Rays with equal keys land in arbitrary order (an atomic): nothing depends on it.
#pragma once

#include "common.cuh"

constexpr int kSortBits = 18;                       // 2 x 9 bits: 512 x 512 cells over the sphere of directions
constexpr unsigned int kSortBins = 1u << kSortBits;
constexpr int kScanBlock = 1024;

__device__ __forceinline__ unsigned int spread_bits(unsigned int x) {   // 0000abcd... -> 0a0b0c0d (16 -> 32 bits)
  x &= 0xFFFFu;
  x = (x | (x << 8)) & 0x00FF00FFu;
  x = (x | (x << 4)) & 0x0F0F0F0Fu;
  x = (x | (x << 2)) & 0x33333333u;
  x = (x | (x << 1)) & 0x55555555u;
  return x;
}

// cell of the direction (x, y, z) (any length) in the octahedral map of the sphere, Morton-interleaved
__device__ __forceinline__ unsigned int direction_key(float x, float y, float z) {
  const float s = fabsf(x) + fabsf(y) + fabsf(z);
  const float inv = __fdividef(1.0f, fmaxf(s, 1e-30f));
  float px = x * inv, py = y * inv;
  if (z < 0.0f) {                                   // lower hemisphere folds over the outer triangles of the square
    const float qx = (1.0f - fabsf(py)) * (px >= 0.0f ? 1.0f : -1.0f);
    const float qy = (1.0f - fabsf(px)) * (py >= 0.0f ? 1.0f : -1.0f);
    px = qx; py = qy;
  }
  const int n = 1 << (kSortBits / 2);
  const int iu = min(n - 1, max(0, (int)(fmaf(px, 0.5f, 0.5f) * (float)n)));   // (int)NaN = 0
  const int iv = min(n - 1, max(0, (int)(fmaf(py, 0.5f, 0.5f) * (float)n)));
  return spread_bits((unsigned int)iu) | (spread_bits((unsigned int)iv) << 1);
}

struct SortKeyConst {
  float c[3];    // body centre
  float r2;      // (radius of the key sphere)^2
};

// primary ray o + t v: where it enters the key sphere, else its point of closest approach to the centre
__device__ __forceinline__ unsigned int primary_key(const SortKeyConst& k, const float o[3], const float v[3]) {
  const float x = o[0] - k.c[0], y = o[1] - k.c[1], z = o[2] - k.c[2];
  const float b = fmaf(z, v[2], fmaf(y, v[1], x * v[0]));
  const float vv = fmaf(v[2], v[2], fmaf(v[1], v[1], v[0] * v[0]));
  const float cc = fmaf(z, z, fmaf(y, y, x * x)) - k.r2;
  const float disc = fmaf(b, b, -vv * cc);
  const float t = __fdividef(-b - sqrtf(fmaxf(disc, 0.0f)), fmaxf(vv, 1e-30f));
  return direction_key(fmaf(t, v[0], x), fmaf(t, v[1], y), fmaf(t, v[2], z));
}
__device__ __forceinline__ unsigned int origin_key(const SortKeyConst& k, const float o[3]) {
  return direction_key(o[0] - k.c[0], o[1] - k.c[1], o[2] - k.c[2]);
}

// histogram -> exclusive offsets, in place: one block, kSortBins / kScanBlock consecutive bins per thread
__global__ void __launch_bounds__(kScanBlock) k_sort_scan(unsigned int* __restrict__ hist) {
  constexpr int kPer = kSortBins / kScanBlock;
  __shared__ unsigned int wsum[kScanBlock / 32];
  unsigned int tot = 0u;
  uint4* h4 = (uint4*)(hist + (size_t)threadIdx.x * kPer);
  for (int k = 0; k < kPer / 4; ++k) {
    const uint4 q = h4[k];
    tot += q.x + q.y + q.z + q.w;
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  unsigned int inc = tot;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const unsigned int n = __shfl_up_sync(0xFFFFFFFFu, inc, off);
    if (lane >= off) inc += n;
  }
  if (lane == 31) wsum[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    unsigned int w = wsum[lane];
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const unsigned int n = __shfl_up_sync(0xFFFFFFFFu, w, off);
      if (lane >= off) w += n;
    }
    wsum[lane] = w;
  }
  __syncthreads();
  unsigned int run = inc - tot + (wid ? wsum[wid - 1] : 0u);
  for (int k = 0; k < kPer / 4; ++k) {   // second read of the thread's own bins (cache-resident)
    const uint4 v = h4[k];
    uint4 q;
    q.x = run; run += v.x;
    q.y = run; run += v.y;
    q.z = run; run += v.z;
    q.w = run; run += v.w;
    h4[k] = q;
  }
}

// queue slots in key order: order[offset[key]++] = slot, over region A [0, na) and region B [cap, cap + nb)
__global__ void __launch_bounds__(256) k_sort_scatter(const unsigned int* __restrict__ keys, unsigned int cap,
                                                     const unsigned int* __restrict__ n_rays, unsigned int* __restrict__ offs,
                                                     unsigned int* __restrict__ order) {
  const unsigned int na = min(n_rays[0], cap), n = na + n_rays[1];
  for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const unsigned int slot = (i < na) ? i : cap + (i - na);
    const unsigned int key = __ldcs(keys + slot);
    const unsigned int pos = atomicAdd(offs + key, 1u);
    __stcs(order + pos, slot);
  }
}
