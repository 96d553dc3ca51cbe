// radix.cuh -- stable LSD radix sort of (64-bit key, 32-bit value) pairs on the device, 4 bits per pass.
// Used once per mesh by the LBVH build (Morton codes of the facet centroids -> sorted facet order, lbvh.cu); about a
// million pairs, far from the timed path, so the layout favours plainness: per pass a digit histogram per block,
// one exclusive scan over the (digit, block) table, and a scatter in which every block ranks its elements stably
// (rounds of one element per thread in index order; within a round, warp ballots per digit and a prefix over the warps).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace radix {

constexpr int kBits = 4, kDigits = 1 << kBits;
constexpr int kBlock = 256, kItems = 8, kTile = kBlock * kItems;

__global__ void __launch_bounds__(kBlock) k_hist(const uint64_t* __restrict__ keys, int64_t n, int shift, int nblocks,
                                                 unsigned int* __restrict__ counts /* [kDigits][nblocks] */) {
  __shared__ unsigned int h[kDigits];
  if (threadIdx.x < kDigits) h[threadIdx.x] = 0u;
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * kTile;
  for (int r = 0; r < kItems; ++r) {
    const int64_t i = base + (int64_t)r * kBlock + threadIdx.x;
    if (i < n) atomicAdd(&h[(unsigned int)(keys[i] >> shift) & (kDigits - 1)], 1u);
  }
  __syncthreads();
  if (threadIdx.x < kDigits) counts[(size_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

// exclusive scan of a table of `len` counts, in place, by one block (chunks of 1024 with a running total)
__global__ void __launch_bounds__(1024) k_scan(unsigned int* __restrict__ a, int64_t len) {
  __shared__ unsigned int wsum[32];
  __shared__ unsigned int carry;
  if (threadIdx.x == 0) carry = 0u;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int64_t c0 = 0; c0 < len; c0 += 1024) {
    const int64_t i = c0 + threadIdx.x;
    const unsigned int v = i < len ? a[i] : 0u;
    unsigned int inc = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const unsigned int t = __shfl_up_sync(0xFFFFFFFFu, inc, off);
      if (lane >= off) inc += t;
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      unsigned int w = wsum[lane];
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const unsigned int t = __shfl_up_sync(0xFFFFFFFFu, w, off);
        if (lane >= off) w += t;
      }
      wsum[lane] = w;
    }
    __syncthreads();
    const unsigned int before = carry + (wid ? wsum[wid - 1] : 0u);
    if (i < len) a[i] = before + inc - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry = before + inc;
    __syncthreads();
  }
}

__global__ void __launch_bounds__(kBlock) k_scatter(const uint64_t* __restrict__ keys, const int32_t* __restrict__ vals,
                                                    int64_t n, int shift, int nblocks, const unsigned int* __restrict__ offs,
                                                    uint64_t* __restrict__ keys_out, int32_t* __restrict__ vals_out) {
  __shared__ unsigned int wc[kBlock / 32][kDigits];   // digit counts of each warp in this round
  __shared__ unsigned int run[kDigits];               // where the block's next element of each digit goes
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x < kDigits) run[threadIdx.x] = offs[(size_t)threadIdx.x * nblocks + blockIdx.x];
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * kTile;
  for (int r = 0; r < kItems; ++r) {
    const int64_t i = base + (int64_t)r * kBlock + threadIdx.x;
    const bool live = i < n;
    const uint64_t key = live ? keys[i] : 0ull;
    const int32_t val = live ? vals[i] : 0;
    const int d = live ? (int)((unsigned int)(key >> shift) & (kDigits - 1)) : -1;
    unsigned int rank = 0u;
#pragma unroll
    for (int k = 0; k < kDigits; ++k) {
      const unsigned int m = __ballot_sync(0xFFFFFFFFu, d == k);
      if (d == k) rank = __popc(m & ((1u << lane) - 1u));
      if (lane == 0) wc[wid][k] = __popc(m);
    }
    __syncthreads();
    if (live) {
      unsigned int before = run[d];
      for (int w = 0; w < wid; ++w) before += wc[w][d];
      keys_out[before + rank] = key;
      vals_out[before + rank] = val;
    }
    __syncthreads();
    if (threadIdx.x < kDigits) {
      unsigned int t = 0u;
      for (int w = 0; w < kBlock / 32; ++w) t += wc[w][threadIdx.x];
      run[threadIdx.x] += t;
    }
    __syncthreads();
  }
}

inline size_t scratch_bytes(int64_t n) {
  const int64_t nblocks = (n + kTile - 1) / kTile;
  return sizeof(unsigned int) * (size_t)kDigits * (size_t)(nblocks > 0 ? nblocks : 1);
}

// Sorts by bits [0, key_bits) of the keys (key_bits rounded up to a multiple of 4).  The pairs ping-pong between
// (keys_a, vals_a) and (keys_b, vals_b); returns 0 if the sorted pairs end in the `a` buffers, 1 if in `b`.
inline int sort_pairs(uint64_t* keys_a, int32_t* vals_a, uint64_t* keys_b, int32_t* vals_b, int64_t n, int key_bits,
                      unsigned int* scratch, cudaStream_t st) {
  const int nblocks = (int)((n + kTile - 1) / kTile);
  int cur = 0;
  for (int shift = 0; shift < key_bits; shift += kBits) {
    const uint64_t* kin = cur ? keys_b : keys_a;
    const int32_t* vin = cur ? vals_b : vals_a;
    uint64_t* kout = cur ? keys_a : keys_b;
    int32_t* vout = cur ? vals_a : vals_b;
    k_hist<<<nblocks, kBlock, 0, st>>>(kin, n, shift, nblocks, scratch);
    k_scan<<<1, 1024, 0, st>>>(scratch, (int64_t)kDigits * nblocks);
    k_scatter<<<nblocks, kBlock, 0, st>>>(kin, vin, n, shift, nblocks, scratch, kout, vout);
    cur ^= 1;
  }
  return cur;
}

}  // namespace radix
